"""Next row (rest): triplet classifiers and track building from triplets on the GPU vs the oracle.
Scores within the precision's tolerance; the track building is integer work -- every array bit-equal when both sides
start from the same fp32 edge / triplet scores."""
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


def device_graph(B, etx, batch, src, dst):
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    E, N = len(src), db.n_hits
    g = B.DeviceGraph(N, max(E, 1), dev)
    rp = np.zeros(N + 1, np.int32); np.cumsum(np.bincount(src, minlength=N), out=rp[1:])
    ip = np.zeros(N + 1, np.int32); np.cumsum(np.bincount(dst, minlength=N), out=ip[1:])
    g.row_ptr.copy_(torch.from_numpy(rp)); g.in_ptr.copy_(torch.from_numpy(ip))
    if E:
        g.src[:E].copy_(torch.from_numpy(np.ascontiguousarray(src, np.int32)))
        g.dst[:E].copy_(torch.from_numpy(np.ascontiguousarray(dst, np.int32)))
        g.in_perm[:E].copy_(torch.from_numpy(np.lexsort((np.arange(E), dst)).astype(np.int32)))
    g.c.n_edges = E
    etx.ensure_workspace(db.n_events, N, max(E, 1))
    return db, g


def gpu_tracks(B, etx, batch, src, dst, scores, s_min, ts, t_min):
    """Triplets on the GPU from the given fp32 scores, then tracks from the given triplet scores (dict per kind)."""
    db, g = device_graph(B, etx, batch, src, dst)
    sc = torch.from_numpy(np.ascontiguousarray(scores, np.float32)).to(etx.device) if len(src) else torch.zeros(1, device=etx.device)
    trip = etx.etx_build_triplets(db, g, sc, s_min)
    tsc = torch.from_numpy(np.concatenate([ts[k] for k in ("articulation", "left_elbow", "right_elbow")] + [np.zeros(1, np.float32)])).to(etx.device)
    out = etx.etx_build_tracks_from_triplets(db, g, sc, s_min, trip, tsc, t_min)
    torch.cuda.synchronize()
    tp, th = out["track_ptr"].cpu().numpy(), out["track_hits"].cpu().numpy()
    return {"edge_set": out["edge_set"].cpu().numpy(), "joins": out["joins"].cpu().numpy().reshape(-1, 2),
            "tracks": [tuple(th[tp[i]:tp[i + 1]].tolist()) for i in range(len(tp) - 1)], "n_plain": out["n_plain"]}


def check(got, want):
    np.testing.assert_array_equal(got["edge_set"], want["edge_set"])
    np.testing.assert_array_equal(got["joins"], want["joins"])
    assert got["tracks"] == want["tracks"]
    assert got["n_plain"] == len(want["tracks"]) - len(want["joins"])


def test_hand_built_pair_and_triangle(B, c0):
    cfg, batch, blob = c0
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    one = {k: batch[k][:6].copy() for k in ("r", "phi", "z", "x", "y", "track")}
    one["plane"] = np.array([0, 1, 2, 2, 3, 3], np.uint8)
    one["event_ptr"] = np.array([0, 6], np.int32)
    src, dst = np.array([0, 1, 1, 2, 3], np.int32), np.array([1, 2, 3, 4, 5], np.int32)
    s = np.ones(5, np.float32)
    trip = orc.triplets(6, src, dst, s, 0.5)
    ts = {k: np.ones(len(trip[k]), np.float32) for k in trip}
    ts["left_elbow"][:] = 0.1
    got = gpu_tracks(B, etx, one, src, dst, s, 0.5, ts, 0.5)
    assert got["tracks"] == [(0, 1, 2, 4), (0, 1, 3, 5)]               # the e+e- pair sharing its two initial hits
    check(got, orc.tracks_from_triplets(6, src, dst, s, 0.5, trip, ts, 0.5))
    ts["left_elbow"][:] = 1.0
    check(gpu_tracks(B, etx, one, src, dst, s, 0.5, ts, 0.5), orc.tracks_from_triplets(6, src, dst, s, 0.5, trip, ts, 0.5))
    tri = {k: batch[k][:3].copy() for k in ("r", "phi", "z", "x", "y", "track")}
    tri["plane"] = np.array([0, 1, 2], np.uint8)
    tri["event_ptr"] = np.array([0, 3], np.int32)
    src, dst, s = np.array([0, 0, 1], np.int32), np.array([1, 2, 2], np.int32), np.ones(3, np.float32)
    trip = orc.triplets(3, src, dst, s, 0.5)
    for elb, art in ((1.0, 1.0), (0.0, 1.0), (0.0, 0.0)):
        ts = {"articulation": np.full(1, art, np.float32), "left_elbow": np.full(1, elb, np.float32), "right_elbow": np.full(1, elb, np.float32)}
        check(gpu_tracks(B, etx, tri, src, dst, s, 0.5, ts, 0.5), orc.tracks_from_triplets(3, src, dst, s, 0.5, trip, ts, 0.5))


@pytest.mark.parametrize("edge_cut,tmin,seed", [(0.5, 0.5, 0), (0.3, 0.5, 1), (0.5, 0.2, 2), (0.0, 0.8, 3), (0.5, 0.0, 4), (2.0, 0.5, 5)])
def test_tracks_c1_random_scores(B, c1, c1_oracle, edge_cut, tmin, seed):
    """C1's graph with random edge / triplet scores: many elbows, shared articulations and cycles."""
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    src, dst = c1_oracle["src"], c1_oracle["dst"]
    rng = np.random.default_rng(seed)
    s = rng.random(len(src)).astype(np.float32)
    trip = orc.triplets(len(batch["r"]), src, dst, s, edge_cut)
    ts = {k: rng.random(len(trip[k])).astype(np.float32) for k in trip}
    check(gpu_tracks(B, etx, batch, src, dst, s, edge_cut, ts, tmin),
          orc.tracks_from_triplets(len(batch["r"]), src, dst, s, edge_cut, trip, ts, tmin))


def test_tracks_multi_event_never_cross_events_and_deterministic(B):
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, range(200, 205))
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    n = len(batch["r"])
    rng = np.random.default_rng(11)
    s = rng.random(len(ora["src"])).astype(np.float32)
    trip = orc.triplets(n, ora["src"], ora["dst"], s, 0.45)
    ts = {k: rng.random(len(trip[k])).astype(np.float32) for k in trip}
    a = gpu_tracks(B, etx, batch, ora["src"], ora["dst"], s, 0.45, ts, 0.4)
    b = gpu_tracks(B, etx, batch, ora["src"], ora["dst"], s, 0.45, ts, 0.4)
    check(a, b)
    check(a, orc.tracks_from_triplets(n, ora["src"], ora["dst"], s, 0.45, trip, ts, 0.4))
    ev = np.repeat(np.arange(5), np.diff(batch["event_ptr"]))
    assert all(len(set(ev[list(t)].tolist())) == 1 for t in a["tracks"])


@pytest.mark.parametrize("prec,tol", [(0, 1e-4), (3, 1e-4), (1, 1e-4), (2, 2e-2)])
def test_triplet_scores_and_end_to_end(B, c1, c1_oracle, prec, tol):
    """GPU edge encodings -> GPU triplets -> GPU triplet scores vs the oracle's classifiers on the oracle's encodings of
    the same graph; then tracks from the GPU's own scores equal the oracle's procedure applied to those same scores."""
    cfg, batch, blob = c1
    etx = B.Etx(B.make_desc(cfg, precision=prec), blob)
    tw = synth.generate_triplet_weights(cfg)
    lay = synth.triplet_layout(cfg)
    etx.etx_set_triplet_classifiers(tw)
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    N = db.n_hits
    cap = len(c1_oracle["src"]) + 8
    etx.ensure_workspace(1, N, cap)
    g = B.DeviceGraph(N, cap, dev)
    E = etx.etx_build_graph(db, torch.from_numpy(c1_oracle["emb"]).to(dev), synth.r2_max(cfg), cfg.max_plane_gap, g)
    assert E == len(c1_oracle["src"])
    enc = torch.empty(cap, cfg.gnn_hidden, device=dev)
    sc = torch.empty(cap, device=dev)
    etx.etx_gnn_forward(db, g, enc)
    etx.etx_edge_scores(g, enc, sc)
    s_min = float(np.median(c1_oracle["scores"]))
    # cut on the ORACLE's scores so both sides list the same triplets
    sc_o = torch.from_numpy(c1_oracle["scores"]).to(dev)
    trip = etx.etx_build_triplets(db, g, sc_o, s_min)
    want_rows = orc.triplets(N, c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"], s_min)
    for k in want_rows:
        np.testing.assert_array_equal(trip[k].cpu().numpy(), want_rows[k])
    ts = etx.etx_triplet_scores(g, enc, trip)
    torch.cuda.synchronize()
    want = orc.triplet_scores(c1_oracle["e"], want_rows, cfg.gnn_hidden, cfg.gnn_mlp_hidden_layers + 1, tw,
                              lay["trip_art"][1], lay["trip_elb"][1])
    worst = 0.0
    for k in want:
        assert len(want[k]) > 100
        worst = max(worst, float(np.abs(ts[k].cpu().numpy().astype(np.float64) - want[k]).max()))
    print(f"precision {prec}: {sum(len(v) for v in want.values())} triplets, worst |triplet score - oracle| = {worst:.3g}")
    assert worst <= tol
    # tracks from the GPU's own triplet scores (cut at their median): the oracle's procedure on the same numbers
    got_ts = {k: ts[k].cpu().numpy() for k in want}
    t_min = float(np.median(np.concatenate(list(got_ts.values()))))
    out = etx.etx_build_tracks_from_triplets(db, g, sc_o, s_min, trip, ts["all"], t_min)
    torch.cuda.synchronize()
    ref = orc.tracks_from_triplets(N, c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"], s_min, want_rows, got_ts, t_min)
    tp, th = out["track_ptr"].cpu().numpy(), out["track_hits"].cpu().numpy()
    np.testing.assert_array_equal(out["edge_set"].cpu().numpy(), ref["edge_set"])
    np.testing.assert_array_equal(out["joins"].cpu().numpy().reshape(-1, 2), ref["joins"])
    assert [tuple(th[tp[i]:tp[i + 1]].tolist()) for i in range(len(tp) - 1)] == ref["tracks"]


def test_triplet_api_errors(B, c0):
    cfg, batch, blob = c0
    etx = B.Etx(B.make_desc(cfg, precision=0), blob)
    with pytest.raises(B.EtxError) as ei:
        etx.etx_set_triplet_classifiers(np.zeros(5, np.float32))
    assert ei.value.status == B.ETX_ERR_INVALID
    db, g = device_graph(B, etx, batch, np.zeros(0, np.int32), np.zeros(0, np.int32))
    trip = etx.etx_build_triplets(db, g, torch.zeros(1, device=etx.device), 0.5)
    with pytest.raises(B.EtxError) as ei:                           # no classifiers set
        etx.etx_triplet_scores(g, torch.zeros(4, cfg.gnn_hidden, device=etx.device), trip)
    assert ei.value.status == B.ETX_ERR_INVALID
    out = etx.etx_build_tracks_from_triplets(db, g, torch.zeros(1, device=etx.device), 0.5, trip, torch.zeros(1, device=etx.device), 0.5)
    assert len(out["track_ptr"]) == 1 and len(out["joins"]) == 0    # empty graph: no tracks
