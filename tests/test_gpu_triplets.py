"""Next row (triplet part): triplet building on the GPU vs the oracle.
Integer work in one fixed order: every array must be bit-equal when both sides cut on the same fp32 scores."""
import numpy as np
import pytest
import torch

from conftest import oracle_path
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth

pytestmark = pytest.mark.gpu
KINDS = ("articulation", "left_elbow", "right_elbow")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def device_graph(B, etx, n_hits, src, dst):
    """The two CSR structures of a given edge list (source-sorted), laid out as etx_build_graph leaves them."""
    E = len(src)
    g = B.DeviceGraph(n_hits, max(E, 1), etx.device)
    rp = np.zeros(n_hits + 1, np.int32); np.cumsum(np.bincount(src, minlength=n_hits), out=rp[1:])
    ip = np.zeros(n_hits + 1, np.int32); np.cumsum(np.bincount(dst, minlength=n_hits), out=ip[1:])
    g.row_ptr.copy_(torch.from_numpy(rp)); g.in_ptr.copy_(torch.from_numpy(ip))
    if E:
        g.src[:E].copy_(torch.from_numpy(np.ascontiguousarray(src, np.int32)))
        g.dst[:E].copy_(torch.from_numpy(np.ascontiguousarray(dst, np.int32)))
        g.in_perm[:E].copy_(torch.from_numpy(np.lexsort((np.arange(E), dst)).astype(np.int32)))
    g.c.n_edges = E
    return g


def check(B, etx, db, g, n_hits, src, dst, scores, s_min, capacity=None):
    sc = torch.from_numpy(np.ascontiguousarray(scores, np.float32)).to(etx.device) if len(src) else torch.zeros(1, device=etx.device)
    got = etx.etx_build_triplets(db, g, sc, s_min, capacity=capacity)
    torch.cuda.synchronize()
    want = orc.triplets(n_hits, src, dst, scores, s_min)
    shared = {"articulation": lambda t: dst[t[:, 0]], "left_elbow": lambda t: src[t[:, 0]], "right_elbow": lambda t: dst[t[:, 0]]}
    ptr = got["ptr"].cpu().numpy()
    for k, name in enumerate(KINDS):
        np.testing.assert_array_equal(got[name].cpu().numpy(), want[name])
        off = np.zeros(n_hits + 1, np.int64)
        np.cumsum(np.bincount(shared[name](want[name]), minlength=n_hits), out=off[1:])
        np.testing.assert_array_equal(ptr[k], off)                  # CSR by shared hit
    return {name: want[name] for name in KINDS}


def test_triplets_match_oracle_c1(B, c1, c1_oracle):
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    db = B.DeviceBatch(batch, etx.device)
    n = db.n_hits
    # the graph the GPU builds from the oracle's embeddings (bit-equal to the oracle's), the oracle's scores
    g = B.DeviceGraph(n, len(c1_oracle["src"]) + 8, etx.device)
    etx.ensure_workspace(db.n_events, n, g.c.edge_capacity)
    E = etx.etx_build_graph(db, torch.from_numpy(c1_oracle["emb"]).to(etx.device), synth.r2_max(cfg), cfg.max_plane_gap, g)
    src, dst, s = c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"]
    assert E == len(src)
    sizes = []
    for s_min in (0.0, float(np.median(s)), float(np.quantile(s, 0.9)), 2.0):
        t = check(B, etx, db, g, n, src, dst, s, s_min)
        sizes.append(sum(len(t[k]) for k in KINDS))
    assert sizes[0] > sizes[1] > sizes[2] > sizes[3] == 0
    assert etx.launch_count() > 0


def test_triplets_multi_event_ragged_and_determinism(B):
    cfg = synth.CONFIGS["c2"]
    ids = [3, 11, 200, 512, 999]
    batch = synth.generate_events(cfg, ids)
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    db = B.DeviceBatch(batch, etx.device)
    n = db.n_hits
    etx.ensure_workspace(db.n_events, n, len(ora["src"]) + 8)
    g = device_graph(B, etx, n, ora["src"], ora["dst"])
    s_min = float(np.quantile(ora["scores"], 0.5))
    t = check(B, etx, db, g, n, ora["src"], ora["dst"], ora["scores"], s_min)
    t2 = check(B, etx, db, g, n, ora["src"], ora["dst"], ora["scores"], s_min, capacity=sum(len(t[k]) for k in KINDS) + 5)
    ev = np.repeat(np.arange(len(ids)), np.diff(batch["event_ptr"]))
    for k in KINDS:
        np.testing.assert_array_equal(t[k], t2[k])
        assert len(t[k]) % 256 != 0 and n % 256 != 0
        assert np.array_equal(ev[ora["src"][t[k][:, 0]]], ev[ora["dst"][t[k][:, 1]]])      # never across events


def test_triplets_hand_built_capacity_and_empty(B, c0):
    cfg, batch, blob = c0
    etx = B.Etx(B.make_desc(cfg), blob)
    db = B.DeviceBatch(batch, etx.device)
    n = db.n_hits
    etx.ensure_workspace(db.n_events, n, 64)
    # the oracle test's hand-built graph on hits 0..4 of the event (the call only reads the CSR structures)
    src = np.array([0, 0, 1, 1, 2, 3], np.int32)                    # source-sorted: 0->2, 0->3, 1->2, 1->3, 2->4, 3->4
    dst = np.array([2, 3, 2, 3, 4, 4], np.int32)
    sc = np.array([0.9, 0.8, 0.7, 0.1, 0.9, 0.6], np.float32)
    g = device_graph(B, etx, n, src, dst)
    t = check(B, etx, db, g, n, src, dst, sc, 0.5)
    np.testing.assert_array_equal(t["articulation"], [[0, 4], [2, 4], [1, 5]])
    np.testing.assert_array_equal(t["left_elbow"], [[0, 1]])
    np.testing.assert_array_equal(t["right_elbow"], [[0, 2], [4, 5]])
    check(B, etx, db, g, n, src, dst, sc, 0.1)                      # inclusive cut keeps edge 3
    with pytest.raises(B.EtxError) as ei:                           # 6 rows needed
        etx.etx_build_triplets(db, g, torch.from_numpy(sc).to(etx.device), 0.5, capacity=5)
    assert ei.value.status == B.ETX_ERR_CAPACITY and "6 rows" in str(ei.value)
    # no edges at all, and an empty batch
    g0 = device_graph(B, etx, n, src[:0], dst[:0])
    t0 = check(B, etx, db, g0, n, src[:0], dst[:0], sc[:0], 0.5)
    assert all(len(t0[k]) == 0 for k in KINDS)
    empty = synth.generate_events(cfg, [])
    dbe = B.DeviceBatch(empty, etx.device)
    ge = device_graph(B, etx, 0, src[:0], dst[:0])
    out = etx.etx_build_triplets(dbe, ge, torch.zeros(1, device=etx.device), 0.5)
    assert all(out[k].shape == (0, 2) for k in KINDS) and out["ptr"].shape == (3, 1)
