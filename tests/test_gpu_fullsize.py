"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the whole
1000-event batch goes through the four C-ABI calls once; sampled events are then recomputed one by
one by the CPU oracle and compared, and size-independent properties are checked on the whole batch."""
import numpy as np
import pytest
import torch

from conftest import oracle_path
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth

pytestmark = pytest.mark.gpu

TOL = {synth.PREC_FP32: 1e-4, synth.PREC_TF32X3: 1e-4, synth.PREC_BF16: 2e-2, synth.PREC_BF16X3: 1e-4}


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_07423_b200 import binding, build
    build.build()
    return binding


def run_full(B, cfg, batch, blob, precision=None, emb_from=None):
    etx = B.Etx(B.make_desc(cfg, precision=precision), blob)  # default: the config's bench precision
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    N = db.n_hits
    cap = int(N * (cfg.target_degree * 1.25 + 2))             # bench.py's capacity rule
    etx.ensure_workspace(db.n_events, N, cap)
    g = B.DeviceGraph(N, cap, dev)
    emb = etx.etx_embed(db) if emb_from is None else torch.from_numpy(emb_from).to(dev)    # (a given embedding: same graph)
    E = etx.etx_build_graph(db, emb, synth.r2_max(cfg), cfg.max_plane_gap, g)
    enc = torch.empty(cap, cfg.gnn_hidden, device=dev)
    sc = torch.empty(cap, device=dev)
    etx.etx_gnn_forward(db, g, enc)
    etx.etx_edge_scores(g, enc, sc)
    torch.cuda.synchronize()
    out = {"E": E, "src": g.src[:E].cpu().numpy(), "dst": g.dst[:E].cpu().numpy(),
           "row_ptr": g.row_ptr.cpu().numpy(), "in_ptr": g.in_ptr.cpu().numpy(),
           "in_perm": g.in_perm[:E].cpu().numpy(), "scores": sc[:E].cpu().numpy(), "emb": emb.cpu().numpy()}
    del enc, sc, g, emb, db, etx
    torch.cuda.empty_cache()
    return out


def check_properties(cfg, batch, out):
    N, E = len(batch["r"]), out["E"]
    src, dst = out["src"].astype(np.int64), out["dst"].astype(np.int64)
    assert out["row_ptr"][0] == 0 and out["row_ptr"][-1] == E and np.all(np.diff(out["row_ptr"]) >= 0)
    assert out["in_ptr"][0] == 0 and out["in_ptr"][-1] == E and np.all(np.diff(out["in_ptr"]) >= 0)
    np.testing.assert_array_equal(np.bincount(src, minlength=N), np.diff(out["row_ptr"]))     # degree sums = E
    np.testing.assert_array_equal(np.bincount(dst, minlength=N), np.diff(out["in_ptr"]))
    key = src * N + dst
    assert np.all(np.diff(key) > 0)                                 # ordered (src, dst): no duplicates
    pl = batch["plane"].astype(np.int64)
    dp = pl[dst] - pl[src]
    assert dp.min() >= 1 and dp.max() <= cfg.max_plane_gap          # allowed plane pairs only
    ev = np.repeat(np.arange(len(batch["event_ptr"]) - 1), np.diff(batch["event_ptr"]))
    assert np.array_equal(ev[src], ev[dst])                         # never across events
    perm = out["in_perm"].astype(np.int64)
    assert np.array_equal(np.sort(perm), np.arange(E))              # a permutation of the edge ids
    assert np.all(np.diff(dst[perm]) >= 0)                          # grouped by destination
    same = np.diff(dst[perm]) == 0
    assert np.all(np.diff(perm)[same] > 0)                          # ascending edge id inside a group
    s = out["scores"]
    assert np.all(np.isfinite(s)) and s.min() >= 0.0 and s.max() <= 1.0
    assert s.std() >= 0.04 and np.mean((s > 0.02) & (s < 0.98)) > 0.5    # neither collapsed nor saturated (Q14; floor 0.05 on the calibration events)
    return ev


def survey_subset(batch, every, n_ext):
    """SURVEY 8(d)'s deterministic event subset: every `every`-th event, the n_ext largest and the n_ext smallest by hit count."""
    n = np.diff(batch["event_ptr"].astype(np.int64))
    order = np.argsort(n, kind="stable")
    return sorted(set(range(0, len(n), every)) | set(order[:n_ext].tolist()) | set(order[len(n) - n_ext:].tolist()))


# (config, every k-th event, extremes by hit count, precision).  The configs' own precisions get the survey's subset
# (every 50th + 16 largest + 16 smallest: 50 events); the other modes a thinner one, the host oracle does ~4 events/s.
@pytest.mark.parametrize("name,every,n_ext,precision", [
    ("c2", 50, 16, None), ("c3", 50, 16, None), ("c4", 50, 16, None),
    ("c2", 250, 4, synth.PREC_TF32X3), ("c2", 500, 2, synth.PREC_FP32)])
def test_full_batch_sampled_events(B, name, every, n_ext, precision):
    cfg = synth.CONFIGS[name]
    if precision is not None:
        import dataclasses
        cfg = dataclasses.replace(cfg, precision=precision)
    batch = synth.generate_events(cfg)
    blob = synth.generate_weights(cfg)
    sample = survey_subset(batch, every, n_ext)
    out = run_full(B, cfg, batch, blob, precision)
    ev = check_properties(cfg, batch, out)
    assert abs(out["E"] / len(batch["r"]) - cfg.target_degree) < 0.08 * cfg.target_degree
    ep = batch["event_ptr"].astype(np.int64)
    oras, emb2, n_border = {}, out["emb"].copy(), 0
    for e in sample:
        sub = synth.select_events(batch, [e])
        ora = oras[e] = oracle_path(cfg, sub, blob)
        sel = ev[out["src"]] == e
        gs, gd = out["src"][sel] - ep[e], out["dst"][sel] - ep[e]
        np.testing.assert_allclose(out["emb"][ep[e]:ep[e + 1]], ora["emb"], rtol=0, atol=2e-6)
        _, _, border = orc.build_graph(sub["event_ptr"], sub["plane"], ora["emb"], synth.r2_max(cfg),
                                       cfg.max_plane_gap, band=1e-5, want_border=True)
        got, want = set(zip(gs.tolist(), gd.tolist())), set(zip(ora["src"].tolist(), ora["dst"].tolist()))
        assert (got ^ want) <= set(map(tuple, border.tolist()))     # end to end: differences only inside the 1e-5 band
        n_border += len(got ^ want)
        emb2[ep[e]:ep[e + 1]] = ora["emb"]
    # Scores: the same full batch again with the sampled events' embeddings replaced by the oracle's, so that their
    # graphs must equal the oracle's bit for bit (BJ's graph gate) and EVERY sampled event's scores are compared
    # (an event whose end-to-end graph differs by a border pair has legitimately different messages).
    out2 = run_full(B, cfg, batch, blob, precision, emb_from=emb2)
    worst = 0.0
    for e in sample:
        ora = oras[e]
        sel = ev[out2["src"]] == e
        np.testing.assert_array_equal(out2["src"][sel] - ep[e], ora["src"])
        np.testing.assert_array_equal(out2["dst"][sel] - ep[e], ora["dst"])
        err = float(np.abs(out2["scores"][sel].astype(np.float64) - ora["scores"]).max())
        worst = max(worst, err)
        assert err <= TOL[cfg.precision], (name, e, err)
    print(f"{name} precision={cfg.precision}: {len(sample)} events (hits {int(np.diff(ep)[sample].min())}..{int(np.diff(ep)[sample].max())}), "
          f"N={len(batch['r'])} E={out['E']} worst sampled |score - oracle| = {worst:.3g} "
          f"({n_border} border-pair differences end to end in the sampled events)")


# Does BASELINE.json's gate hold on EVERY edge of the full batch at the oracle-calibrated gain?  Measured, round 2
# (profiles/r02_parity.md): yes for the fp32-equivalent modes at C2 (max 5.0e-5 / 1.9e-5 of 9.6 M edges); yes for the
# bf16 mode at C3's scale since its per-hit MLPs and classifier run the split (max 1.47e-2 against 2e-2; with every MLP
# in single-pass bf16 it was 2.5e-2: NOT met); NO
# for the split modes at C4's scale (max 4.5e-4 against 1e-4), which is why C4 runs the exact FFMA mode.  The table is
# asserted BOTH ways: a mode listed as failing must really exceed the gate (so this text cannot go stale), and stay
# inside the looser bound given here.
EVERY_EDGE = {("c2", synth.PREC_BF16X3): (True, 1e-4), ("c2", synth.PREC_TF32X3): (True, 1e-4),
              ("c2", synth.PREC_BF16): (True, 2e-2), ("c4", synth.PREC_BF16X3): (False, 1e-3)}


@pytest.mark.parametrize("name,precisions", [("c2", [synth.PREC_BF16X3, synth.PREC_TF32X3, synth.PREC_BF16]),
                                             ("c4", [synth.PREC_BF16X3])])
def test_full_batch_every_edge(B, name, precisions):
    """The score tolerance on EVERY edge of the full batch.  The oracle cannot score 10^7 edges in a test, so
    the chain is: exact-fp32 FFMA mode vs oracle on sampled events (test above, <= 3e-6), then every
    tensor-core mode vs the FFMA mode on all edges with the gate reduced by that 3e-6.  Both runs start from the
    FFMA mode's embedding, so that they score the same graph (the tensor-core modes' own 3xTF32 embedding moves a
    handful of pairs inside the 1e-5 band across the radius; that is checked in the sampled test)."""
    import dataclasses
    cfg0 = synth.CONFIGS[name]
    batch = synth.generate_events(cfg0)
    blob = synth.generate_weights(cfg0)
    ref = run_full(B, dataclasses.replace(cfg0, precision=synth.PREC_FP32), batch, blob, synth.PREC_FP32)
    for prec in precisions:
        out = run_full(B, dataclasses.replace(cfg0, precision=prec), batch, blob, prec, emb_from=ref["emb"])
        assert out["E"] == ref["E"] and np.array_equal(out["dst"], ref["dst"])      # same graph (same embedding)
        own = run_full(B, dataclasses.replace(cfg0, precision=prec), batch, blob, prec)
        assert abs(own["E"] - ref["E"]) <= 1e-4 * ref["E"]                         # its own embedding: a few border pairs
        assert np.abs(own["emb"] - ref["emb"]).max() <= 4e-6
        d = np.abs(out["scores"].astype(np.float64) - ref["scores"].astype(np.float64))
        holds, bound = EVERY_EDGE[(name, prec)]
        print(f"{name} precision={prec}: all {out['E']} edges, max |score - FFMA| = {d.max():.3g}, "
              f"p99.99 = {np.quantile(d, 0.9999):.3g}, median = {np.median(d):.3g}; gate {TOL[prec]:g} on every edge: "
              f"{'holds' if d.max() <= TOL[prec] - 3e-6 else 'NOT met'} (recorded: {'holds' if holds else 'not met'}), "
              f"{int((d > TOL[prec]).sum())} edges above it")
        assert (d.max() <= TOL[prec] - 3e-6) == holds, (name, prec, float(d.max()))
        assert d.max() <= bound and np.quantile(d, 0.999) <= TOL[prec], (name, prec, float(d.max()))


def test_full_batch_next_rows_tracks_and_triplets(B):
    """The next rows at bench.py's size and launch configuration (c2, 1000 events, default precision): closed-form
    triplet counts and CSR offsets from the kept degrees on ALL hits, and tracks / triplets of sampled events
    against the oracle run on that event alone (integer work: bit-equal)."""
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg)
    blob = synth.generate_weights(cfg)
    etx = B.Etx(B.make_desc(cfg), blob)
    dev = etx.device
    db = B.DeviceBatch(batch, dev)
    N = db.n_hits
    cap = int(N * (cfg.target_degree * 1.25 + 2))
    etx.ensure_workspace(db.n_events, N, cap)
    g = B.DeviceGraph(N, cap, dev)
    E = etx.etx_build_graph(db, etx.etx_embed(db), synth.r2_max(cfg), cfg.max_plane_gap, g)
    enc = torch.empty(cap, cfg.gnn_hidden, device=dev)
    sc = torch.empty(cap, device=dev)
    etx.etx_gnn_forward(db, g, enc)
    etx.etx_edge_scores(g, enc, sc)
    s_min = 0.5
    lab = etx.etx_build_tracks(db, g, sc, s_min)[:N].cpu().numpy()
    tr = etx.etx_build_triplets(db, g, sc, s_min)
    torch.cuda.synchronize()
    src, dst, s = g.src[:E].cpu().numpy().astype(np.int64), g.dst[:E].cpu().numpy().astype(np.int64), sc[:E].cpu().numpy()
    keep = s >= np.float32(s_min)
    kout, kin = np.bincount(src[keep], minlength=N), np.bincount(dst[keep], minlength=N)
    ptr = tr["ptr"].cpu().numpy()
    rows = {k: tr[k].cpu().numpy() for k in ("articulation", "left_elbow", "right_elbow")}
    for k, per_hit in enumerate((kin * kout, kout * (kout - 1) // 2, kin * (kin - 1) // 2)):
        off = np.zeros(N + 1, np.int64); np.cumsum(per_hit, out=off[1:])
        np.testing.assert_array_equal(ptr[k], off)
    assert [len(rows[k]) for k in rows] == [int(ptr[k][-1]) for k in range(3)]
    a, l, r = rows["articulation"], rows["left_elbow"], rows["right_elbow"]
    assert np.all(keep[a]) and np.all(keep[l]) and np.all(keep[r])
    assert np.array_equal(dst[a[:, 0]], src[a[:, 1]]) and np.array_equal(src[l[:, 0]], src[l[:, 1]])
    assert np.array_equal(dst[r[:, 0]], dst[r[:, 1]]) and np.all(l[:, 0] < l[:, 1]) and np.all(r[:, 0] < r[:, 1])
    ep = batch["event_ptr"].astype(np.int64)
    rp = g.row_ptr.cpu().numpy().astype(np.int64)
    ev = np.repeat(np.arange(len(ep) - 1), np.diff(ep))
    assert np.array_equal(ev[lab], ev) and np.all(lab <= np.arange(N))          # tracks stay inside their event
    for e in (0, 421, 999):
        h0, h1, e0, e1 = ep[e], ep[e + 1], rp[ep[e]], rp[ep[e + 1]]
        ls, ld, lsc = (src[e0:e1] - h0).astype(np.int32), (dst[e0:e1] - h0).astype(np.int32), s[e0:e1]
        np.testing.assert_array_equal(lab[h0:h1] - h0, orc.wcc(int(h1 - h0), ls, ld, lsc, s_min))
        want = orc.triplets(int(h1 - h0), ls, ld, lsc, s_min)
        for k, name in enumerate(rows):
            got = rows[name][ptr[k][h0]:ptr[k][h1]] - e0                         # the event's rows, local edge ids
            np.testing.assert_array_equal(got, want[name])
