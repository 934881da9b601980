"""Pins for the oracle's radius search (Eq. 8.1; Alg. 1 / P:2674)."""
import numpy as np
import torch

from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def brute_force(event_ptr, plane, emb, r2, gap):
    """All N^2 ordered pairs with the predicate (same event, 1 <= dplane <= G, d^2 < r^2);
    d^2 in fp32, left to right, every numpy op individually rounded (no FMA)."""
    n = len(plane)
    ev = np.repeat(np.arange(len(event_ptr) - 1), np.diff(event_ptr))
    e = emb.astype(np.float32)
    d2 = np.zeros((n, n), np.float32)
    for c in range(e.shape[1]):
        diff = (e[:, None, c] - e[None, :, c]).astype(np.float32)
        sq = (diff * diff).astype(np.float32)
        d2 = sq if c == 0 else (d2 + sq).astype(np.float32)
    dp = plane[None, :].astype(int) - plane[:, None].astype(int)
    ok = (ev[:, None] == ev[None, :]) & (dp >= 1) & (dp <= gap) & (d2 < np.float32(r2))
    i, j = np.nonzero(ok)                                     # row-major = (src asc, dst asc)
    return i.astype(np.int32), j.astype(np.int32)


def test_windowed_search_equals_brute_force_c0(c0, c0_oracle):
    cfg, b, _ = c0
    i, j = brute_force(b["event_ptr"], b["plane"], c0_oracle["emb"], synth.r2_max(cfg), cfg.max_plane_gap)
    np.testing.assert_array_equal(c0_oracle["src"], i)
    np.testing.assert_array_equal(c0_oracle["dst"], j)
    assert abs(len(i) / len(b["r"]) - cfg.target_degree) < 0.05


def test_brute_force_multi_event_and_gap2():
    cfg = synth.CONFIGS["c0"]
    b = synth.generate_events(cfg, [0, 1, 2])
    rng = np.random.default_rng(3)
    emb = rng.normal(size=(len(b["r"]), 3)).astype(np.float32)   # d = 3 (the thesis' final embedding dim)
    for gap, r2 in ((2, 0.9), (3, 0.3), (1, 2.0)):
        s, d = orc.build_graph(b["event_ptr"], b["plane"], emb, r2, gap)
        i, j = brute_force(b["event_ptr"], b["plane"], emb, r2, gap)
        np.testing.assert_array_equal(s, i)
        np.testing.assert_array_equal(d, j)
        assert len(s) > 0


def test_distance_against_torch_cdist(c0, c0_oracle):
    _, b, _ = c0
    emb = c0_oracle["emb"]
    d2 = orc.candidate_d2(b["event_ptr"], b["plane"], emb, 3)
    t = torch.cdist(torch.from_numpy(emb).double(), torch.from_numpy(emb).double()) ** 2
    pl = b["plane"].astype(int)
    dp = pl[None, :] - pl[:, None]
    ref = t.numpy()[(dp >= 1) & (dp <= 3)]
    np.testing.assert_allclose(np.sort(d2), np.sort(ref), rtol=1e-9, atol=1e-12)


def test_closed_forms():
    cfg = synth.CONFIGS["c0"]
    b = synth.generate_events(cfg, [0, 1])
    n = len(b["r"])
    emb = np.random.default_rng(0).normal(size=(n, 4)).astype(np.float32)
    for gap in (1, 2, 3):
        # r -> infinity: E = sum over events and planes of n_p (n_{p+1} + ... + n_{p+G})
        want = 0
        for e in range(2):
            cnt = np.bincount(b["plane"][b["event_ptr"][e]:b["event_ptr"][e + 1]], minlength=26)
            want += sum(cnt[p] * cnt[p + 1:p + 1 + gap].sum() for p in range(26))
        s, d = orc.build_graph(b["event_ptr"], b["plane"], emb, np.inf, gap)
        assert len(s) == want
    s, _ = orc.build_graph(b["event_ptr"], b["plane"], emb, 0.0, 3)
    assert len(s) == 0                                         # strict "<": nothing is closer than 0


def test_lattice_and_strict_inequality():
    # one event, 3 planes x 5 hits on a 1-D lattice (embedding = (x, 0)), spacing 1
    plane = np.repeat(np.arange(3), 5).astype(np.uint8)
    emb = np.zeros((15, 2), np.float32)
    emb[:, 0] = np.tile(np.arange(5), 3)
    ptr = np.array([0, 15], np.int32)
    # r^2 = 1 exactly: |dx| = 1 is NOT an edge (d^2 < r^2 strict) -> only dx = 0 pairs
    s, d = orc.build_graph(ptr, plane, emb, 1.0, 2)
    assert len(s) == 5 * 3 and np.all(emb[s, 0] == emb[d, 0])
    # r^2 just above 1: dx in {-1, 0, 1} -> per plane pair 5 + 2*4 = 13; three pairs (0-1, 1-2, 0-2)
    s, d = orc.build_graph(ptr, plane, emb, np.nextafter(np.float32(1), np.float32(2)), 2)
    assert len(s) == 13 * 3
    s, d = orc.build_graph(ptr, plane, emb, 1.5, 1)            # gap 1: pairs 0-1, 1-2 only
    assert len(s) == 13 * 2 and np.all(plane[d] - plane[s] == 1)


def test_invariants_c1(c1, c1_oracle):
    cfg, b, _ = c1
    s, d = c1_oracle["src"], c1_oracle["dst"]
    pl = b["plane"].astype(int)
    assert np.all((pl[d] - pl[s] >= 1) & (pl[d] - pl[s] <= cfg.max_plane_gap))   # allowed plane pairs only
    assert np.all(s != d)                                       # no self loops
    key = s.astype(np.int64) * len(pl) + d
    assert np.all(np.diff(key) > 0)                             # (src, dst) strictly ascending: no duplicates
    n = len(pl)
    assert np.bincount(s, minlength=n).sum() == np.bincount(d, minlength=n).sum() == len(s)
    assert abs(len(s) / n - cfg.target_degree) < 0.01


def test_monotone_in_radius_and_batch_is_concatenation():
    cfg = synth.CONFIGS["c0"]
    b = synth.generate_events(cfg, [0, 1, 2])
    emb = np.random.default_rng(5).normal(size=(len(b["r"]), 4)).astype(np.float32) * 0.5
    prev = set()
    for r2 in (0.05, 0.2, 0.8):
        s, d = orc.build_graph(b["event_ptr"], b["plane"], emb, r2, 3)
        cur = set(zip(s.tolist(), d.tolist()))
        assert prev <= cur and len(cur) > len(prev)
        prev = cur
    s, d = orc.build_graph(b["event_ptr"], b["plane"], emb, 0.2, 3)
    parts_s, parts_d = [], []
    for e in range(3):
        lo, hi = b["event_ptr"][e], b["event_ptr"][e + 1]
        ss, dd = orc.build_graph(np.array([0, hi - lo], np.int32), b["plane"][lo:hi], emb[lo:hi], 0.2, 3)
        parts_s.append(ss + lo)
        parts_d.append(dd + lo)
    np.testing.assert_array_equal(s, np.concatenate(parts_s))
    np.testing.assert_array_equal(d, np.concatenate(parts_d))


def test_borderline_band():
    plane = np.array([0, 1, 1, 1], np.uint8)
    emb = np.array([[0, 0], [1.0, 0], [1.000004, 0], [1.1, 0]], np.float32)
    s, d, bp = orc.build_graph(np.array([0, 4], np.int32), plane, emb, 1.0, 1, band=1e-5, want_border=True)
    assert set(map(tuple, bp.tolist())) == {(0, 1), (0, 2)}     # |d - r| <= 1e-5 listed; 1.1 is not
    assert len(s) == 0
