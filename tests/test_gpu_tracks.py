"""Next row: score cut + WCC track building on the GPU vs the oracle.
Integer work: labels must be bit-equal when both sides cut on the same fp32 scores."""
import numpy as np
import pytest
import torch

from conftest import oracle_path
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def gpu_labels(B, etx, batch, src, dst, scores, s_min):
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    E = len(src)
    g = B.DeviceGraph(db.n_hits, max(E, 1), dev)
    rp = np.zeros(db.n_hits + 1, np.int32)
    np.cumsum(np.bincount(src, minlength=db.n_hits), out=rp[1:])
    g.row_ptr.copy_(torch.from_numpy(rp))
    g.src[:E].copy_(torch.from_numpy(np.ascontiguousarray(src, np.int32)))
    g.dst[:E].copy_(torch.from_numpy(np.ascontiguousarray(dst, np.int32)))
    g.c.n_edges = E
    sc = torch.from_numpy(np.ascontiguousarray(scores, np.float32)).to(dev) if E else torch.zeros(1, device=dev)
    lab = etx.etx_build_tracks(db, g, sc, s_min)
    torch.cuda.synchronize()
    return lab[:db.n_hits].cpu().numpy()


def test_tracks_match_oracle_c1(B, c1, c1_oracle):
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    src, dst, s = c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"]
    n = len(batch["r"])
    for s_min in (0.0, float(np.median(s)), float(np.quantile(s, 0.9)), 2.0):
        got = gpu_labels(B, etx, batch, src, dst, s, s_min)
        np.testing.assert_array_equal(got, orc.wcc(n, src, dst, s, s_min))
    assert etx.launch_count() > 0


def test_tracks_multi_event_and_determinism(B):
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, range(40, 72))
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    n = len(batch["r"])
    s_min = float(np.quantile(ora["scores"], 0.6))
    a = gpu_labels(B, etx, batch, ora["src"], ora["dst"], ora["scores"], s_min)
    b = gpu_labels(B, etx, batch, ora["src"], ora["dst"], ora["scores"], s_min)
    np.testing.assert_array_equal(a, b)
    np.testing.assert_array_equal(a, orc.wcc(n, ora["src"], ora["dst"], ora["scores"], s_min))
    ev = np.repeat(np.arange(32), np.diff(batch["event_ptr"]))
    assert np.array_equal(ev[a], ev)                                # a track never leaves its event


def test_tracks_zigzag_needs_more_than_two_sweeps(B, c0):
    cfg, batch, blob = c0
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    one = {k: batch[k][:5].copy() for k in ("plane", "r", "phi", "z", "x", "y", "track")}
    one["plane"] = np.array([0, 0, 0, 1, 1], np.uint8)
    one["event_ptr"] = np.array([0, 5], np.int32)
    src = np.array([0, 1, 1, 2], np.int32)
    dst = np.array([3, 3, 4, 4], np.int32)
    got = gpu_labels(B, etx, one, src, dst, np.ones(4, np.float32), 0.5)
    np.testing.assert_array_equal(got, [0, 0, 0, 0, 0])             # exact WCC (P:2719's two sweeps leave hit 2 = 1)
    got = gpu_labels(B, etx, one, src, dst, np.array([1, 1, 0.2, 1], np.float32), 0.5)
    np.testing.assert_array_equal(got, [0, 0, 2, 0, 2])             # cutting edge 1->4 splits the component


def test_tracks_end_to_end_consistency(B, c1):
    """GPU scores -> GPU tracks: a valid partition of the GPU's own purified graph, equal to the oracle's
    track building applied to the same GPU scores."""
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg), blob)
    out = B.run_path(etx, batch, synth.r2_max(cfg), cfg.max_plane_gap)
    s_min = 0.5
    got = gpu_labels(B, etx, batch, out["src"], out["dst"], out["scores"], s_min)
    np.testing.assert_array_equal(got, orc.wcc(len(batch["r"]), out["src"], out["dst"], out["scores"], s_min))
    keep = out["scores"] >= np.float32(s_min)
    assert np.all(got[out["src"][keep]] == got[out["dst"][keep]]) and np.all(got[got] == got)


def test_tracks_long_zigzag_converges_beyond_64_rounds(B, c0):
    """Adversarial component: a zig-zag a0->b0<-a1->b1<-a2 ... between two planes.  One forward + one
    backward sweep move the minimum label two hops, so 150 alternations need ~150 rounds: a bounded loop (64 rounds
    in round 1) returned wrong labels with ETX_OK.  The exact WCC (oracle: union-find) is one component."""
    cfg, batch, blob = c0
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    n = 150
    one = {k: np.resize(batch[k], 2 * n).copy() for k in ("r", "phi", "z", "x", "y", "track")}
    one["plane"] = np.repeat(np.array([0, 1], np.uint8), n)
    one["event_ptr"] = np.array([0, 2 * n], np.int32)
    src = np.concatenate([[0], np.repeat(np.arange(1, n), 2)]).astype(np.int32)          # a_i -> b_{i-1}, b_i
    dst = np.concatenate([[n], (n + np.stack([np.arange(0, n - 1), np.arange(1, n)], 1)).ravel()]).astype(np.int32)
    s = np.ones(len(src), np.float32)
    want = orc.wcc(2 * n, src, dst, s, 0.5)
    assert np.all(want == 0)
    np.testing.assert_array_equal(gpu_labels(B, etx, one, src, dst, s, 0.5), want)
    # the same chain cut in the middle: two components, second labelled by its smallest hit
    s[len(s) // 2] = 0.0
    np.testing.assert_array_equal(gpu_labels(B, etx, one, src, dst, s, 0.5), orc.wcc(2 * n, src, dst, s, 0.5))
