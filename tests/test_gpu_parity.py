"""CUDA path (through the C ABI) vs the CPU oracle, element by element, on the same seeded inputs.

Bars (BASELINE.json north_star; tolerances derived in DESIGN.md "Tolerances"):
  * graph edges: bit-exact arrays when both paths start from the ORACLE's fp32 embeddings;
  * embeddings / encodings: fp32 summation-order noise only;
  * edge scores: |delta| <= 1e-4 absolute (fp32 path), 2e-2 (bf16 MLPs, on the oracle's graph).
"""
import dataclasses

import numpy as np
import pytest
import torch

from conftest import layout_dict, oracle_path
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth

pytestmark = pytest.mark.gpu

TOL_SCORE_FP32 = 1e-4
TOL_SCORE_BF16 = 2e-2


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def make_etx(B, cfg, blob, precision=0):
    return B.Etx(B.make_desc(cfg, precision=precision), blob)


def gpu_from_oracle_graph(B, etx, batch, ora, r2, gap):
    """GNN + scores on the graph the GPU builds from the ORACLE's embeddings (must equal the oracle's)."""
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    cap = max(len(ora["src"]) + 7, 16)
    etx.ensure_workspace(db.n_events, db.n_hits, cap)
    g = B.DeviceGraph(db.n_hits, cap, dev)
    emb = torch.from_numpy(ora["emb"]).to(dev)
    E = etx.etx_build_graph(db, emb, r2, gap, g)
    H = int(etx.desc.gnn_hidden)
    e = torch.empty(max(E, 1), H, device=dev)
    h = torch.empty(max(db.n_hits, 1), H, device=dev)
    s = torch.empty(max(E, 1), device=dev)
    etx.etx_gnn_forward(db, g, e, h)
    etx.etx_edge_scores(g, e, s)
    torch.cuda.synchronize()
    return {"src": g.src[:E].cpu().numpy(), "dst": g.dst[:E].cpu().numpy(), "row_ptr": g.row_ptr.cpu().numpy(),
            "in_ptr": g.in_ptr.cpu().numpy(), "in_perm": g.in_perm[:E].cpu().numpy(),
            "h": h[:db.n_hits].cpu().numpy(), "e": e[:E].cpu().numpy(), "scores": s[:E].cpu().numpy()}


def check_graph_arrays(out, ora, n_hits):
    np.testing.assert_array_equal(out["src"], ora["src"])           # bit-exact, same order
    np.testing.assert_array_equal(out["dst"], ora["dst"])
    E = len(ora["src"])
    rp = np.zeros(n_hits + 1, np.int64); np.cumsum(np.bincount(ora["src"], minlength=n_hits), out=rp[1:])
    ip = np.zeros(n_hits + 1, np.int64); np.cumsum(np.bincount(ora["dst"], minlength=n_hits), out=ip[1:])
    np.testing.assert_array_equal(out["row_ptr"], rp)
    np.testing.assert_array_equal(out["in_ptr"], ip)
    # by-destination lists: a permutation, grouped by destination, ascending edge id inside a group
    want = np.lexsort((np.arange(E), ora["dst"]))
    np.testing.assert_array_equal(out["in_perm"], want)


def rel_close(a, b, tol):
    scale = max(1.0, float(np.abs(b).max()))
    return float(np.abs(a.astype(np.float64) - b).max()) <= tol * scale


@pytest.mark.parametrize("name", ["c0", "c1"])
def test_single_event_configs(B, name, request):
    cfg, batch, blob = request.getfixturevalue(name)
    ora = request.getfixturevalue(name + "_oracle")
    etx = make_etx(B, cfg, blob)
    r2, gap = synth.r2_max(cfg), cfg.max_plane_gap
    # a1: embedding
    full = B.run_path(etx, batch, r2, gap)
    assert np.abs(full["emb"] - ora["emb"]).max() <= 2e-6
    # a2: graph from the oracle's embeddings, bit-exact; a3-a7 on it
    out = gpu_from_oracle_graph(B, etx, batch, ora, r2, gap)
    check_graph_arrays(out, ora, len(batch["r"]))
    assert rel_close(out["h"], ora["h"], 2e-5)
    assert rel_close(out["e"], ora["e"], 2e-5)
    err = np.abs(out["scores"].astype(np.float64) - ora["scores"])
    assert err.max() <= TOL_SCORE_FP32, err.max()
    # end to end (GPU embeddings -> GPU graph): edges may differ only inside the 1e-5 band around r
    _, _, border = orc.build_graph(batch["event_ptr"], batch["plane"], ora["emb"], r2, gap, band=1e-5, want_border=True)
    band = set(map(tuple, border.tolist()))
    got = set(zip(full["src"].tolist(), full["dst"].tolist()))
    want = set(zip(ora["src"].tolist(), ora["dst"].tolist()))
    assert (got ^ want) <= band, sorted(got ^ want)[:10]
    if got == want:
        assert np.abs(full["scores"].astype(np.float64) - ora["scores"]).max() <= TOL_SCORE_FP32


def test_multi_event_batch_and_ragged_tiles(B):
    # 5 events of the throughput config: E and N are not multiples of the 128-row tile
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, [3, 11, 200, 512, 999])
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = make_etx(B, cfg, blob)
    out = gpu_from_oracle_graph(B, etx, batch, ora, synth.r2_max(cfg), cfg.max_plane_gap)
    check_graph_arrays(out, ora, len(batch["r"]))
    assert len(ora["src"]) % 128 != 0 and len(batch["r"]) % 128 != 0
    assert np.abs(out["scores"].astype(np.float64) - ora["scores"]).max() <= TOL_SCORE_FP32


def test_stress_config_events(B):
    cfg = synth.CONFIGS["c4"]
    batch = synth.generate_events(cfg, [0, 1])
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = make_etx(B, cfg, blob)
    out = gpu_from_oracle_graph(B, etx, batch, ora, synth.r2_max(cfg), cfg.max_plane_gap)
    check_graph_arrays(out, ora, len(batch["r"]))
    assert abs(len(ora["src"]) / len(batch["r"]) - 10.0) < 1.0
    assert np.abs(out["scores"].astype(np.float64) - ora["scores"]).max() <= TOL_SCORE_FP32


def test_thesis_settings_gap2_dim3(B):
    # the thesis' own search setting: planes p+1, p+2 and a 3-dimensional embedding
    cfg = dataclasses.replace(synth.CONFIGS["c0"], emb_widths=(3, 64, 64, 3), max_plane_gap=2)
    batch = synth.generate_events(cfg, [0, 1, 2])
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob, r2=2.5e-3, gap=2)
    assert len(ora["src"]) > 100
    etx = make_etx(B, cfg, blob)
    out = gpu_from_oracle_graph(B, etx, batch, ora, 2.5e-3, 2)
    check_graph_arrays(out, ora, len(batch["r"]))
    assert np.abs(out["scores"].astype(np.float64) - ora["scores"]).max() <= TOL_SCORE_FP32


def test_radius_extremes_and_empty_inputs(B, c0, c0_oracle):
    cfg, batch, blob = c0
    etx = make_etx(B, cfg, blob)
    n = len(batch["r"])
    # r = 0: no edges at all; the GNN and the head must accept E = 0
    out = B.run_path(etx, batch, 0.0, cfg.max_plane_gap)
    assert len(out["src"]) == 0 and np.all(out["row_ptr"] == 0) and np.all(out["in_ptr"] == 0)
    lo = layout_dict(cfg)
    h = orc.mlp(c0_oracle["f_node"], lo["node_enc"][0], blob, lo["node_enc"][1])
    for k in range(cfg.n_iter):                                   # isolated hits: m = 0
        x = np.concatenate([h, np.zeros((n, 2 * cfg.gnn_hidden), np.float32)], 1)
        h = h + orc.mlp(x, lo[f"node_net_{k}"][0], blob, lo[f"node_net_{k}"][1])
    assert rel_close(out["h"], h, 2e-5)
    # r = inf: every allowed plane pair (closed form count)
    cnt = np.bincount(batch["plane"], minlength=26)
    want = sum(int(cnt[p]) * int(cnt[p + 1:p + 1 + cfg.max_plane_gap].sum()) for p in range(26))
    out = B.run_path(etx, batch, float("inf"), cfg.max_plane_gap, edge_capacity=want)
    assert len(out["src"]) == want
    s, d = orc.build_graph(batch["event_ptr"], batch["plane"], out["emb"], np.inf, cfg.max_plane_gap)
    np.testing.assert_array_equal(out["src"], s)
    np.testing.assert_array_equal(out["dst"], d)
    # empty batch, and a batch whose events are empty or hold one hit
    empty = {k: v[:0] for k, v in batch.items() if k != "event_ptr"}
    empty["event_ptr"] = np.zeros(1, np.int32)
    out = B.run_path(etx, empty, 1.0, 3)
    assert len(out["src"]) == 0 and len(out["scores"]) == 0
    one = synth.select_events(batch, [0])
    keep = np.array([0, n - 1])
    tiny = {k: one[k][keep] for k in ("plane", "r", "phi", "z", "x", "y", "track")}
    tiny["event_ptr"] = np.array([0, 0, 1, 1, 2], np.int32)       # events: empty, 1 hit, empty, 1 hit
    out = B.run_path(etx, tiny, float("inf"), 3)
    assert len(out["src"]) == 0 and out["h"].shape == (2, cfg.gnn_hidden)


def test_tc_refuses_misaligned_output(B, c1):
    """The tensor-core path writes through TMA tensor maps: an output that is not 16-byte aligned is refused loudly."""
    cfg, batch, blob = c1
    tc = make_etx(B, cfg, blob, precision=3)
    db = B.DeviceBatch(batch, tc.device)
    tc.ensure_workspace(db.n_events, db.n_hits, 100000)
    g = B.DeviceGraph(db.n_hits, 100000, tc.device)
    E = tc.etx_build_graph(db, tc.etx_embed(db), synth.r2_max(cfg), cfg.max_plane_gap, g)
    buf = torch.empty(E * cfg.gnn_hidden + 1, device=tc.device)
    with pytest.raises(B.EtxError) as ei:
        tc.etx_gnn_forward(db, g, buf[1:].view(E, cfg.gnn_hidden))
    assert ei.value.status == B.ETX_ERR_INVALID
    ok = torch.empty(E, cfg.gnn_hidden, device=tc.device)
    tc.etx_gnn_forward(db, g, ok)                                 # the context is usable afterwards
    torch.cuda.synchronize()
    assert torch.isfinite(ok).all()


def test_error_paths(B, c0):
    cfg, batch, blob = c0
    etx = make_etx(B, cfg, blob)
    with pytest.raises(B.EtxError) as ei:                         # capacity: nothing written, E reported
        B.run_path(etx, batch, float("inf"), 3, edge_capacity=10)
    assert ei.value.status == B.ETX_ERR_CAPACITY
    bad = dict(batch)
    bad["plane"] = batch["plane"][::-1].copy()
    with pytest.raises(B.EtxError) as ei:
        B.run_path(etx, bad, 1e-3, 3)
    assert ei.value.status == B.ETX_ERR_UNSORTED
    bad["plane"] = np.full_like(batch["plane"], 26)
    with pytest.raises(B.EtxError) as ei:
        B.run_path(etx, bad, 1e-3, 3)
    assert ei.value.status == B.ETX_ERR_INVALID
    db = B.DeviceBatch(batch, etx.device)
    g = B.DeviceGraph(db.n_hits, 100000, etx.device)
    emb = etx.etx_embed(db)
    with pytest.raises(B.EtxError) as ei:                         # k_max: 0 = no cap, > 0 = cap (next row)
        etx.etx_build_graph(db, emb, 1e-3, 3, g, k_max=-1)
    assert ei.value.status == B.ETX_ERR_INVALID
    fresh = make_etx(B, cfg, blob)
    with pytest.raises(B.EtxError) as ei:                         # no workspace handed over
        fresh.etx_build_graph(db, emb, 1e-3, 3, g)
    assert ei.value.status == B.ETX_ERR_NOMEM


def test_host_buffer_entry_point_equals_device_path(B, c1, c1_oracle):
    cfg, batch, blob = c1
    etx = make_etx(B, cfg, blob)
    r2, gap = synth.r2_max(cfg), cfg.max_plane_gap
    ref = B.run_path(etx, batch, r2, gap)
    cap = len(ref["src"]) + 100
    host = B.pinned_host_batch(batch)
    etx.ensure_workspace(1, len(batch["r"]), cap, with_host_path=True)
    src = torch.empty(cap, dtype=torch.int32).pin_memory()
    dst = torch.empty(cap, dtype=torch.int32).pin_memory()
    sc = torch.empty(cap, dtype=torch.float32).pin_memory()
    E = etx.etx_infer_host(host, r2, gap, cap, src, dst, sc)
    assert E == len(ref["src"])
    np.testing.assert_array_equal(src[:E].numpy(), ref["src"])
    np.testing.assert_array_equal(dst[:E].numpy(), ref["dst"])
    np.testing.assert_array_equal(sc[:E].numpy(), ref["scores"])   # same kernels, same order: bitwise
    assert etx.launch_count() > 0


@pytest.mark.parametrize("prec", [0, 3])
def test_host_path_splits_a_batch_larger_than_the_workspace(B, prec):
    """PAPER.md:2638 (GNN batches bounded by memory) / VERDICT r1: a batch that does not fit the workspace is run as
    consecutive event ranges and returns exactly what one pass returns -- events are independent."""
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, range(300, 348))
    blob = synth.generate_weights(cfg)
    etx = make_etx(B, cfg, blob, precision=prec)
    r2, gap = synth.r2_max(cfg), cfg.max_plane_gap
    n_ev, N = len(batch["event_ptr"]) - 1, len(batch["r"])
    cap = int(N * (cfg.target_degree * 1.25 + 2))
    host = B.pinned_host_batch(batch)

    def run(ws_bytes):
        etx.set_workspace(ws_bytes)
        src = torch.full((cap,), -1, dtype=torch.int32).pin_memory()
        dst = torch.full((cap,), -1, dtype=torch.int32).pin_memory()
        sc = torch.full((cap,), -1.0, dtype=torch.float32).pin_memory()
        l0 = etx.launch_count()
        E = etx.etx_infer_host(host, r2, gap, cap, src, dst, sc)
        return E, src[:E].numpy().copy(), dst[:E].numpy().copy(), sc[:E].numpy().copy(), etx.launch_count() - l0

    full = etx.workspace_bytes(n_ev, N, cap, with_host_path=True)
    E, src, dst, sc, l_one = run(full)
    assert abs(E / N - cfg.target_degree) < 1.0
    for frac in (0.45, 0.2, 0.07):                               # ~3, ~6 and ~16 ranges (ragged: events differ in size)
        E2, src2, dst2, sc2, l_many = run(int(full * frac))
        assert E2 == E and l_many > l_one                        # really ran in several passes
        np.testing.assert_array_equal(src2, src)
        np.testing.assert_array_equal(dst2, dst)
        np.testing.assert_array_equal(sc2, sc)                   # same kernels, row-local arithmetic: bitwise
    one = etx.workspace_bytes(1, int(np.diff(batch["event_ptr"]).max()), 64, with_host_path=True)
    with pytest.raises(B.EtxError) as ei:                        # not even one event fits
        run(one // 4)
    assert ei.value.status == B.ETX_ERR_NOMEM
    with pytest.raises(B.EtxError) as ei:                        # the caller's total capacity still binds
        etx.set_workspace(int(full * 0.2))
        etx.etx_infer_host(host, r2, gap, E // 2, None, None, torch.empty(E).pin_memory())
    assert ei.value.status == B.ETX_ERR_CAPACITY


def test_two_devices_in_one_process(B, c1):
    """the >48 KB shared-memory opt-in is a per-device function attribute; a context on a second device
    must configure its own kernels.  Needs two GPUs (skipped on the one-GPU box)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    cfg, batch, blob = c1
    outs = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            etx = B.Etx(B.make_desc(cfg), blob, device=dev)
            outs.append(B.run_path(etx, batch, synth.r2_max(cfg), cfg.max_plane_gap))
    np.testing.assert_array_equal(outs[0]["scores"], outs[1]["scores"])


def test_graph_build_hardening(B, c0):
    """a huge plane gap must not overflow p + gap; a misaligned 4-d embedding is refused, not faulted."""
    cfg, batch, blob = c0
    etx = make_etx(B, cfg, blob)
    a = B.run_path(etx, batch, synth.r2_max(cfg), 25)
    b = B.run_path(etx, batch, synth.r2_max(cfg), 2**31 - 1)
    np.testing.assert_array_equal(a["src"], b["src"])
    np.testing.assert_array_equal(a["dst"], b["dst"])
    db = B.DeviceBatch(batch, etx.device)
    g = B.DeviceGraph(db.n_hits, 100000, etx.device)
    etx.ensure_workspace(db.n_events, db.n_hits, 100000)
    buf = torch.zeros(db.n_hits * 4 + 1, device=etx.device)
    with pytest.raises(B.EtxError) as ei:
        etx.etx_build_graph(db, buf[1:], 1e-3, 3, g)
    assert ei.value.status == B.ETX_ERR_INVALID


def test_deterministic_repeat(B, c1):
    cfg, batch, blob = c1
    etx = make_etx(B, cfg, blob)
    a = B.run_path(etx, batch, synth.r2_max(cfg), cfg.max_plane_gap)
    b = B.run_path(etx, batch, synth.r2_max(cfg), cfg.max_plane_gap)
    for k in ("src", "dst", "in_perm", "scores", "e"):
        np.testing.assert_array_equal(a[k], b[k])                  # no atomics anywhere on the path


# ------------------------------------------------------------------------------------------------
# tensor-core precisions (tcgen05): ETX_PREC_TF32X3 (fp32-equivalent) and ETX_PREC_BF16
# ------------------------------------------------------------------------------------------------
PREC = {"tf32x3": 1, "bf16": 2, "bf16x3": 3}
REL_ENC = {"tf32x3": 2e-5, "bf16": 3e-2, "bf16x3": 5e-5}          # relative to max |value| of the tensor
TOL_SCORE = {"tf32x3": TOL_SCORE_FP32, "bf16": TOL_SCORE_BF16, "bf16x3": TOL_SCORE_FP32}


@pytest.mark.parametrize("prec", ["tf32x3", "bf16", "bf16x3"])
def test_tc_edge_encoder_alone(B, c1, c1_oracle, prec):
    """n_iter = 0: gnn_forward = node encoder (tcgen05, first layer from the 3 features in the gather warps) +
    per-hit projections + edge encoder (tcgen05, addend path, plain store) — the smallest check of descriptors,
    swizzle and the TMEM operand path."""
    cfg, batch, blob = c1
    cfg0 = dataclasses.replace(cfg, n_iter=0)
    blob0 = synth.generate_weights(cfg0)
    ora = oracle_path(cfg0, batch, blob0, graph=(c1_oracle["src"], c1_oracle["dst"]))
    ora["emb"] = c1_oracle["emb"]
    etx = make_etx(B, cfg0, blob0, precision=PREC[prec])
    out = gpu_from_oracle_graph(B, etx, batch, ora, synth.r2_max(cfg), cfg.max_plane_gap)
    np.testing.assert_array_equal(out["src"], ora["src"])
    assert rel_close(out["h"], ora["h"], REL_ENC[prec]), np.abs(out["h"] - ora["h"]).max()
    assert rel_close(out["e"], ora["e"], REL_ENC[prec]), np.abs(out["e"] - ora["e"]).max()
    assert np.abs(out["scores"].astype(np.float64) - ora["scores"]).max() <= TOL_SCORE[prec]


@pytest.mark.parametrize("prec", ["tf32x3", "bf16", "bf16x3"])
def test_tc_permutation_weights_reveal_layout(B, c1, c1_oracle, prec):
    """Edge-encoder weights = signed permutation-like sparse matrices: any swapped k / n index in the
    swizzled weight image or the TMEM operand layout moves values to the wrong column."""
    cfg, batch, blob = c1
    cfg0 = dataclasses.replace(cfg, n_iter=0)
    blob0 = synth.generate_weights(cfg0).copy()
    spec = [s for s in synth.model_layout(cfg0) if s.name == "edge_enc"][0]
    rng = np.random.default_rng(11)
    for (wo, bo, fi, fo) in spec.layer_offsets():
        W = np.zeros((fo, fi), np.float32)
        cols = rng.permutation(fi)[:fo]
        W[np.arange(fo), cols] = rng.choice([-1.0, 1.0, 0.5, 2.0], size=fo)
        blob0[wo:wo + fi * fo] = W.ravel()
        blob0[bo:bo + fo] = rng.uniform(0.0, 0.25, fo).astype(np.float32)
    ora = oracle_path(cfg0, batch, blob0, graph=(c1_oracle["src"], c1_oracle["dst"]))
    ora["emb"] = c1_oracle["emb"]
    etx = make_etx(B, cfg0, blob0, precision=PREC[prec])
    out = gpu_from_oracle_graph(B, etx, batch, ora, synth.r2_max(cfg), cfg.max_plane_gap)
    assert np.abs(ora["e"]).max() > 0.05
    assert rel_close(out["e"], ora["e"], REL_ENC[prec]), np.abs(out["e"] - ora["e"]).max()


@pytest.mark.parametrize("prec", ["tf32x3", "bf16", "bf16x3"])
def test_tc_single_event_full_path(B, c1, c1_oracle, prec):
    cfg, batch, blob = c1
    etx = make_etx(B, cfg, blob, precision=PREC[prec])
    out = gpu_from_oracle_graph(B, etx, batch, c1_oracle, synth.r2_max(cfg), cfg.max_plane_gap)
    check_graph_arrays(out, c1_oracle, len(batch["r"]))
    err = np.abs(out["scores"].astype(np.float64) - c1_oracle["scores"])
    assert err.max() <= TOL_SCORE[prec], err.max()
    if prec != "bf16":
        assert rel_close(out["e"], c1_oracle["e"], 1e-4)
        assert rel_close(out["h"], c1_oracle["h"], 1e-4)


@pytest.mark.parametrize("prec,name", [("tf32x3", "c2"), ("bf16", "c3"), ("tf32x3", "c4"), ("bf16x3", "c2"), ("bf16x3", "c4")])
def test_tc_multi_event_batches(B, prec, name):
    cfg = synth.CONFIGS[name]
    ids = [3, 11, 200, 512, 999] if name != "c4" else [0, 1]
    batch = synth.generate_events(cfg, ids)
    blob = synth.generate_weights(cfg)
    ora = oracle_path(cfg, batch, blob)
    etx = make_etx(B, cfg, blob, precision=PREC[prec])
    out = gpu_from_oracle_graph(B, etx, batch, ora, synth.r2_max(cfg), cfg.max_plane_gap)
    check_graph_arrays(out, ora, len(batch["r"]))
    err = np.abs(out["scores"].astype(np.float64) - ora["scores"])
    assert err.max() <= TOL_SCORE[prec], err.max()


def test_tc_rejects_unsupported_width(B, c0):
    cfg, batch, blob = c0
    with pytest.raises(B.EtxError) as ei:
        make_etx(B, cfg, blob, precision=1)                          # H = 64: tensor-core path needs H = 128
    assert ei.value.status == B.ETX_ERR_INVALID


@pytest.mark.parametrize("widths", [(3, 128, 128, 3), (3, 128, 128, 128, 8), (3, 128, 128, 128, 128, 1), (3, 128, 128, 128, 4)])
@pytest.mark.parametrize("prec", [synth.PREC_TF32X3, synth.PREC_BF16])
def test_tc_embedding_shapes_and_ragged_tail(B, widths, prec):
    """a0+a1 on the tensor cores (3xTF32 hidden layers, narrow linear output in the epilogue)
    for 1..3 hidden MMA layers and 1..8 output units, on batches whose hit count is not a multiple of the 128-row
    tile, in every GNN precision mode (the embedding is 3xTF32 in all of them): |emb - oracle| <= 2e-6 (section 6),
    rows past n_hits untouched, and an empty batch is a no-op."""
    cfg = dataclasses.replace(synth.CONFIGS["c2"], emb_widths=widths, precision=prec)
    blob = synth.generate_weights(cfg)
    spec = synth.model_layout(cfg)[0]
    etx = B.Etx(B.make_desc(cfg, precision=prec), blob)
    d = widths[-1]
    for events in ([7], [3, 11, 200, 512, 999], []):
        batch = synth.generate_events(cfg, events)
        n = len(batch["r"])
        db = B.DeviceBatch(batch, etx.device)
        out = torch.full((n + 5, d), 7.0, device=etx.device)
        etx.etx_embed(db, emb=out)
        torch.cuda.synchronize()
        assert torch.all(out[n:] == 7.0)
        if n == 0:
            continue
        assert n % 128 != 0
        fe, _ = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
        ora = orc.mlp(fe, spec.dims, blob, spec.offset)
        assert np.abs(out[:n].cpu().numpy().astype(np.float64) - ora).max() <= 2e-6


def test_bf16_embedding_report_entry_point(B, c1, c1_oracle):
    """etx_embed_bf16 (report-only, reading Q16): hidden-layer operands rounded to bf16, fp32 accumulation.  Checked against
    the same arithmetic written with torch CPU ops (bf16 round-to-nearest-even operands, float64 accumulation) and against
    the fp32 oracle embedding: close to both, and genuinely different from the fp32 one."""
    cfg, batch, blob = c1
    etx = make_etx(B, cfg, blob, precision=synth.PREC_BF16X3)
    db = B.DeviceBatch(batch, etx.device)
    etx.ensure_workspace(db.n_events, db.n_hits, 64 * db.n_hits)
    got = etx.etx_embed_bf16(db).cpu().numpy().astype(np.float64)
    lay = {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}
    dims, off = lay["emb"]
    f = np.stack([(batch[k].astype(np.float32) - np.float32(synth.NORM_CENTER[i])) / np.float32(synth.NORM_SCALE[i])
                  for i, k in enumerate(("r", "phi", "z"))], axis=1)
    x = torch.from_numpy(f).double()
    o = off
    n_l = len(dims) - 1
    for l in range(n_l):
        fi, fo = dims[l], dims[l + 1]
        W = torch.from_numpy(blob[o:o + fi * fo].reshape(fo, fi).copy()); o += fi * fo
        b = torch.from_numpy(blob[o:o + fo].copy()).double(); o += fo
        if 0 < l < n_l - 1:                            # tensor-core layers: bf16 operands
            x = x.float().bfloat16().double() @ W.bfloat16().double().T + b
        else:
            x = x @ W.double().T + b
        if l < n_l - 1:
            x = torch.relu(x).float().double()         # every layer output is stored in fp32
    want = x.numpy()
    assert np.abs(got - want).max() <= 2e-3
    ref = c1_oracle["emb"].astype(np.float64)
    d = np.abs(got - ref).max()
    assert 1e-5 < d <= 3e-2
    # a context without tensor-core images of the embedding refuses
    cfg0, batch0, blob0 = synth.CONFIGS["c0"], synth.generate_events(synth.CONFIGS["c0"]), synth.generate_weights(synth.CONFIGS["c0"])
    etx0 = make_etx(B, cfg0, blob0)
    with pytest.raises(B.EtxError):
        etx0.etx_embed_bf16(B.DeviceBatch(batch0, etx0.device))
