"""etx_build_triplets_static (include/etx.h): the triplet build whose scan scratch is a fixed device array inside the
library, for callers that may not allocate.  Checked against the existing path (etx_build_triplets, scratch in the
registered workspace): integer work in one fixed order, so every array must be bit-equal.  Two calls in a row on
different inputs (the second smaller, so stale scratch of the first would show), from a context that has NO workspace.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu
KINDS = ("articulation", "left_elbow", "right_elbow")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def random_case(n_hits, n_edges, seed):
    """One event of n_hits hits on two planes and a random source-sorted edge list plane 0 -> plane 1 with scores."""
    rng = np.random.default_rng(seed)
    half = n_hits // 2
    batch = {"event_ptr": np.array([0, n_hits], np.int32),
             "plane": np.r_[np.zeros(half), np.ones(n_hits - half)].astype(np.uint8)}
    for k in ("r", "phi", "z", "x", "y"):
        batch[k] = rng.normal(size=n_hits).astype(np.float32)
    pairs = np.unique(np.stack([rng.integers(0, half, n_edges), rng.integers(half, n_hits, n_edges)], 1), axis=0)
    src, dst = pairs[:, 0].astype(np.int32), pairs[:, 1].astype(np.int32)          # unique rows come out (src, dst)-sorted
    return batch, src, dst, rng.random(len(src)).astype(np.float32)


def device_graph(B, device, n_hits, src, dst):
    E = len(src)
    g = B.DeviceGraph(n_hits, max(E, 1), device)
    rp = np.zeros(n_hits + 1, np.int32); np.cumsum(np.bincount(src, minlength=n_hits), out=rp[1:])
    ip = np.zeros(n_hits + 1, np.int32); np.cumsum(np.bincount(dst, minlength=n_hits), out=ip[1:])
    g.row_ptr.copy_(torch.from_numpy(rp)); g.in_ptr.copy_(torch.from_numpy(ip))
    if E:
        g.src[:E].copy_(torch.from_numpy(src)); g.dst[:E].copy_(torch.from_numpy(dst))
        g.in_perm[:E].copy_(torch.from_numpy(np.lexsort((np.arange(E), dst)).astype(np.int32)))
    g.c.n_edges = E
    return g


def test_static_scratch_triplets_equal_the_workspace_path_twice_in_a_row(B, c0):
    cfg, _, blob = c0
    with_ws = B.Etx(B.make_desc(cfg, precision=0), blob)          # existing path: scratch in the registered workspace
    no_ws = B.Etx(B.make_desc(cfg, precision=0), blob)            # new path: never gets a workspace
    dev = with_ws.device
    # 9001 and 2500 hits: 5 and 2 scan tiles of 2048 (a ragged last tile each); the second call uses fewer block sums
    for n_hits, n_edges, seed, s_min in ((9001, 40000, 1, 0.3), (2500, 9000, 2, 0.0)):
        batch, src, dst, scores = random_case(n_hits, n_edges, seed)
        db = B.DeviceBatch(batch, dev)
        g = device_graph(B, dev, n_hits, src, dst)
        sc = torch.from_numpy(scores).to(dev)
        with_ws.ensure_workspace(db.n_events, n_hits, g.c.edge_capacity)
        want = with_ws.etx_build_triplets(db, g, sc, s_min)
        total = sum(len(want[k]) for k in KINDS)
        assert total > 1000
        ptr = torch.full((3, n_hits + 1), -7, dtype=torch.int32, device=dev)
        rows = torch.full((2, total), -7, dtype=torch.int32, device=dev)
        before = no_ws.launch_count()
        n = no_ws.etx_build_triplets_static(db, g, sc, s_min, ptr, rows)
        torch.cuda.synchronize()
        assert no_ws._ws is None and no_ws.launch_count() > before
        assert n == [len(want[k]) for k in KINDS]
        np.testing.assert_array_equal(ptr.cpu().numpy(), want["ptr"].cpu().numpy())
        o = 0
        for k in KINDS:
            np.testing.assert_array_equal(rows[:, o:o + len(want[k])].t().cpu().numpy(), want[k].cpu().numpy())
            o += len(want[k])
        # too small a row buffer: the counts come back with ETX_ERR_CAPACITY, as in the existing path
        with pytest.raises(B.EtxError) as ei:
            no_ws.etx_build_triplets_static(db, g, sc, s_min, ptr, rows[:, :total - 1].contiguous())
        assert ei.value.status == B.ETX_ERR_CAPACITY


def test_static_scratch_rejects_more_hits_than_its_array_serves(B, c0):
    cfg, _, blob = c0
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    n_hits = (1 << 22) + 1                                        # ETX_STATIC_TRIPLET_MAX_HITS + 1
    batch = {"event_ptr": np.array([0, n_hits], np.int32), "plane": np.zeros(n_hits, np.uint8)}
    for k in ("r", "phi", "z", "x", "y"):
        batch[k] = np.zeros(n_hits, np.float32)
    db = B.DeviceBatch(batch, etx.device)
    g = device_graph(B, etx.device, n_hits, np.zeros(0, np.int32), np.zeros(0, np.int32))
    ptr = torch.zeros(3, n_hits + 1, dtype=torch.int32, device=etx.device)
    rows = torch.zeros(2, 1, dtype=torch.int32, device=etx.device)
    before = etx.launch_count()
    with pytest.raises(B.EtxError) as ei:
        etx.etx_build_triplets_static(db, g, torch.zeros(1, device=etx.device), 0.5, ptr, rows)
    assert ei.value.status == B.ETX_ERR_CAPACITY and "4194304" in str(ei.value)
    assert etx.launch_count() == before                           # nothing was launched
