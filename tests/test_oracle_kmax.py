"""Pins for the oracle's k_max-capped radius search (next row NEXT-2: Algorithm 1)."""
import numpy as np

from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def _d2_fp32(e):
    """All-pairs d^2 in fp32, left to right, every numpy op individually rounded (the oracle's predicate)."""
    d2 = None
    for c in range(e.shape[1]):
        diff = (e[:, None, c] - e[None, :, c]).astype(np.float32)
        sq = (diff * diff).astype(np.float32)
        d2 = sq if d2 is None else (d2 + sq).astype(np.float32)
    return d2


def brute_force_kmax(event_ptr, plane, emb, r2, gap, k_max):
    """Algorithm 1 per source over ALL hits: list (j, d_j) of the allowed candidates inside the radius, sort by
    d ascending (numpy stable argsort: equal d keeps ascending j), first k, reported in ascending j."""
    n = len(plane)
    ev = np.repeat(np.arange(len(event_ptr) - 1), np.diff(event_ptr))
    d2 = _d2_fp32(emb.astype(np.float32))
    pl = plane.astype(int)
    src, dst = [], []
    for i in range(n):
        dp = pl - pl[i]
        cand = np.nonzero((ev == ev[i]) & (dp >= 1) & (dp <= gap) & (d2[i] < np.float32(r2)))[0]
        if k_max > 0 and len(cand) > k_max:
            cand = np.sort(cand[np.argsort(d2[i, cand], kind="stable")[:k_max]])
        src += [i] * len(cand)
        dst += list(cand)
    return np.array(src, np.int32), np.array(dst, np.int32)


def streaming_replace_farthest(event_ptr, plane, emb, r2, gap, k_max):
    """The thesis' own loop: candidates in ascending index; inside the radius -> appended to the list; if
    the list is full, the farthest entry is replaced when the new hit is (strictly) closer."""
    d2 = _d2_fp32(emb.astype(np.float32))
    pl = plane.astype(int)
    ev = np.repeat(np.arange(len(event_ptr) - 1), np.diff(event_ptr))
    out = []
    for i in range(len(plane)):
        lst = []
        for j in range(i + 1, len(plane)):
            if ev[j] != ev[i] or not (1 <= pl[j] - pl[i] <= gap) or not (d2[i, j] < np.float32(r2)):
                continue
            if len(lst) < k_max:
                lst.append(j)
            else:
                far = max(lst, key=lambda q: (d2[i, q], q))
                if d2[i, j] < d2[i, far]:
                    lst[lst.index(far)] = j
        out.append(sorted(lst))
    return out


def _events(n_ev=2, seed=5, dim=3):
    cfg = synth.CONFIGS["c0"]
    b = synth.generate_events(cfg, list(range(n_ev)))
    emb = np.random.default_rng(seed).normal(size=(len(b["r"]), dim)).astype(np.float32)
    return b, emb


def test_kmax_equals_algorithm1_brute_force():
    b, emb = _events()
    for gap, r2, k in ((2, 0.9, 3), (3, 1.5, 5), (1, 4.0, 2), (3, 1.5, 1)):
        s, d = orc.build_graph_kmax(b["event_ptr"], b["plane"], emb, r2, gap, k)
        i, j = brute_force_kmax(b["event_ptr"], b["plane"], emb, r2, gap, k)
        np.testing.assert_array_equal(s, i)
        np.testing.assert_array_equal(d, j)
        deg = np.bincount(s, minlength=len(b["r"]))
        assert deg.max() == k                       # the cap binds in these settings


def test_kmax_equals_thesis_streaming_loop():
    b, emb = _events(n_ev=1, seed=9)
    s, d = orc.build_graph_kmax(b["event_ptr"], b["plane"], emb, 2.0, 2, 4)
    lists = streaming_replace_farthest(b["event_ptr"], b["plane"], emb, 2.0, 2, 4)
    got = [sorted(d[s == i].tolist()) for i in range(len(b["r"]))]
    assert got == lists
    assert max(len(x) for x in got) == 4


def test_cap_not_binding_is_the_plain_radius_graph(c0, c0_oracle):
    cfg, b, _ = c0
    for k in (0, 10 ** 6, int(np.bincount(c0_oracle["src"]).max())):
        s, d = orc.build_graph_kmax(b["event_ptr"], b["plane"], c0_oracle["emb"], synth.r2_max(cfg), cfg.max_plane_gap, k)
        np.testing.assert_array_equal(s, c0_oracle["src"])
        np.testing.assert_array_equal(d, c0_oracle["dst"])


def test_k1_is_the_nearest_neighbour_and_ties_keep_the_lower_index():
    # 1-D lattice embedding, 3 planes: hit positions chosen so the nearest neighbour is known in closed form
    event_ptr = np.array([0, 7], np.int32)
    plane = np.array([0, 0, 1, 1, 1, 2, 2], np.uint8)
    emb = np.array([[0.0], [10.0], [1.0], [-1.0], [10.5], [0.25], [9.0]], np.float32)
    s, d = orc.build_graph_kmax(event_ptr, plane, emb, 100.0, 2, 1)
    # hit 0 (x=0): candidates 2 (d=1), 3 (d=1, tie -> lower index 2 wins), 4, 5 (d=0.25 -> nearest), 6
    # hit 1 (x=10): nearest is 4 (0.5);  hit 2 (x=1): plane-2 hits 5 (0.75), 6 (8) -> 5;  hit 3 (x=-1) -> 5;  hit 4 (10.5) -> 6
    assert list(zip(s.tolist(), d.tolist())) == [(0, 5), (1, 4), (2, 5), (3, 5), (4, 6)]
    s, d = orc.build_graph_kmax(event_ptr, plane, emb, 100.0, 1, 1)      # gap 1: hit 0 sees only plane 1 -> tie 2 vs 3
    assert (0, 2) in set(zip(s.tolist(), d.tolist())) and (0, 3) not in set(zip(s.tolist(), d.tolist()))


def test_invariants_subset_degree_monotone():
    b, emb = _events(n_ev=3, seed=11, dim=4)
    r2, gap = 1.2, 3
    full = set(zip(*[a.tolist() for a in orc.build_graph(b["event_ptr"], b["plane"], emb, r2, gap)]))
    prev = set()
    for k in (1, 2, 4, 8, 64):
        s, d = orc.build_graph_kmax(b["event_ptr"], b["plane"], emb, r2, gap, k)
        cur = set(zip(s.tolist(), d.tolist()))
        assert len(cur) == len(s)                                   # no duplicates
        assert cur <= full and prev <= cur                          # subset of the radius graph, monotone in k
        assert np.bincount(s, minlength=1).max() <= k
        order = np.lexsort((d, s))
        np.testing.assert_array_equal(order, np.arange(len(s)))     # (src asc, dst asc)
        prev = cur
    assert prev == full
