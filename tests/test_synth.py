"""Input generator: geometry, counts, determinism, event independence, weight-blob bookkeeping."""
import numpy as np

from paper_2508_07423_b200 import synth


def test_geometry_and_sorting(c0):
    cfg, b, _ = c0
    n = len(b["r"])
    assert b["event_ptr"][0] == 0 and b["event_ptr"][-1] == n
    assert b["plane"].max() < synth.N_PLANES
    assert np.all(np.diff(b["plane"].astype(int)) >= 0)            # plane-sorted inside the event
    np.testing.assert_allclose(b["z"], -275.0 + 40.0 * b["plane"], atol=0)
    true = b["track"] >= 0
    # true hits lie in the annulus up to 6 sigma of smearing; noise hits exactly inside it
    assert b["r"][true].min() > synth.R_MIN - 0.1 and b["r"][true].max() < synth.R_MAX + 0.1
    assert b["r"][~true].min() >= synth.R_MIN - 1e-4 and b["r"][~true].max() <= synth.R_MAX + 1e-4
    np.testing.assert_allclose(np.hypot(b["x"].astype(np.float64), b["y"]), b["r"], rtol=1e-6)
    np.testing.assert_allclose(np.arctan2(b["y"].astype(np.float64), b["x"]), b["phi"], atol=1e-6)
    assert (~true).sum() == int(np.floor(cfg.noise_frac * true.sum() + 0.5))


def test_tracks_are_straight_lines_from_origin(c0):
    _, b, _ = c0
    for t in np.unique(b["track"][b["track"] >= 0])[:10]:
        sel = b["track"] == t
        if sel.sum() < 3:
            continue
        z, x, y = b["z"][sel].astype(np.float64), b["x"][sel].astype(np.float64), b["y"][sel].astype(np.float64)
        for v in (x, y):
            res = v - np.polyval(np.polyfit(z, v, 1), z)
            assert np.abs(res).max() < 6 * synth.HIT_SMEAR
        assert len(np.unique(z)) == len(z)                        # at most one hit per plane


def test_deterministic_and_event_independent():
    cfg = synth.CONFIGS["c2"]
    a = synth.generate_events(cfg, range(8))
    b = synth.generate_events(cfg, range(8), chunk=3)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    alone = synth.generate_events(cfg, [5, 2])
    sub = synth.select_events(a, [5, 2])
    for k in alone:
        assert np.array_equal(alone[k], sub[k]), k


def test_poisson_track_counts():
    cfg = synth.CONFIGS["c2"]
    nt = synth._n_tracks(cfg, np.arange(1000))
    assert abs(nt.mean() - 150) < 3 * np.sqrt(150 / 1000) + 0.5
    assert abs(nt.var() - 150) < 25
    # workload statistics reported next to every throughput number (SURVEY §8 caveat on counts)
    b = synth.generate_events(cfg, range(16))
    per_ev = np.diff(b["event_ptr"])
    assert 1200 < per_ev.mean() < 2200


def test_weight_layout_and_paper_parameter_counts():
    cfg = synth.CONFIGS["c1"]
    specs = synth.model_layout(cfg)
    off = 0
    for s in specs:
        assert s.offset == off
        off += s.n_floats
    assert off == synth.n_weight_floats(cfg)
    assert [s.name for s in specs][:3] == ["emb", "node_enc", "edge_enc"] and specs[-1].name == "cls"
    # the thesis' printed parameter counts pin the bookkeeping (tests/golden/paper_parameter_counts.txt)
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_parameter_counts.txt")
    seen = 0
    for line in open(path):
        if line.startswith("#") or "|" not in line:
            continue
        name, widths, count, tol, _cite = [t.strip() for t in line.split("|", 4)]
        n = synth.MlpSpec(name, tuple(int(w) for w in widths.split(",")), 0).n_floats
        if name.endswith("with_layernorm"):
            n += 3 * (8 + 8)
        assert abs(n - int(count)) <= int(tol), (name, n)
        seen += 1
    assert seen == 3


def test_xavier_bounds_and_gain():
    cfg = synth.CONFIGS["c0"]
    blob = synth.generate_weights(cfg)
    assert np.array_equal(blob, synth.generate_weights(cfg))
    for s in synth.model_layout(cfg):
        layers = s.layer_offsets()
        for li, (wo, bo, fi, fo) in enumerate(layers):
            g = s.gain if li == len(layers) - 1 else 1.0
            w, b = blob[wo:wo + fi * fo], blob[bo:bo + fo]
            bound = np.sqrt(6.0 / (fi + fo)) * g
            assert np.abs(w).max() <= bound * (1 + 1e-6)
            if fi * fo >= 4096:
                assert np.abs(w).max() > 0.97 * bound and abs(w.mean()) < 0.05 * bound
            assert np.abs(b).max() <= 0.05 * g * (1 + 1e-6)
