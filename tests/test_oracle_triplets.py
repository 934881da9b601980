"""Pins for the oracle's triplet building (NEXT-4, Fig. 8.13): brute force over all pairs of kept
edges straight from the three definitions, closed-form counts from the degrees, a hand-built graph, invariants."""
import numpy as np

from oracle import etx_oracle as orc

KINDS = ("articulation", "left_elbow", "right_elbow")


def brute_force(src, dst, keep):
    """All pairs of kept edges, classified by the definitions of P:2355-2357 (no adjacency lists)."""
    ids = np.flatnonzero(keep)
    art, left, right = set(), set(), set()
    for a in ids:
        for b in ids:
            if a == b:
                continue
            if dst[a] == src[b]:
                art.add((int(a), int(b)))            # A -> C, C -> B
            if a < b and src[a] == src[b]:
                left.add((int(a), int(b)))           # C -> A, C -> B
            if a < b and dst[a] == dst[b]:
                right.add((int(a), int(b)))          # A -> C, B -> C
    return {"articulation": art, "left_elbow": left, "right_elbow": right}


def as_set(a):
    return set(map(tuple, a.tolist()))


def test_brute_force_on_the_tiny_event(c0_oracle):
    src, dst, s = c0_oracle["src"], c0_oracle["dst"], c0_oracle["scores"]
    n = c0_oracle["h"].shape[0]
    for s_min in (0.0, float(np.median(s)), float(np.quantile(s, 0.8))):
        keep = s >= np.float32(s_min)
        t = orc.triplets(n, src, dst, s, s_min)
        bf = brute_force(src, dst, keep)
        for k in KINDS:
            assert len(t[k]) == len(as_set(t[k])), "duplicates"
            assert as_set(t[k]) == bf[k], k
        assert len(t["articulation"]) > 0 and len(t["left_elbow"]) > 0 and len(t["right_elbow"]) > 0


def test_counts_closed_form_and_order(c1_oracle):
    src, dst, s = c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"]
    n = c1_oracle["h"].shape[0]
    prev = None
    for s_min in (0.0, 0.3, 0.5, 0.9, 2.0):
        keep = s >= np.float32(s_min)
        t = orc.triplets(n, src, dst, s, s_min)
        kout = np.bincount(src[keep], minlength=n).astype(np.int64)
        kin = np.bincount(dst[keep], minlength=n).astype(np.int64)
        assert len(t["articulation"]) == int((kin * kout).sum())
        assert len(t["left_elbow"]) == int((kout * (kout - 1) // 2).sum())
        assert len(t["right_elbow"]) == int((kin * (kin - 1) // 2).sum())
        # the definitions, row by row, and the listing order (shared hit, first edge, second edge)
        a, l, r = t["articulation"], t["left_elbow"], t["right_elbow"]
        assert np.all(keep[a]) and np.all(keep[l]) and np.all(keep[r])
        assert np.array_equal(dst[a[:, 0]], src[a[:, 1]])
        assert np.array_equal(src[l[:, 0]], src[l[:, 1]]) and np.all(l[:, 0] < l[:, 1])
        assert np.array_equal(dst[r[:, 0]], dst[r[:, 1]]) and np.all(r[:, 0] < r[:, 1])
        for arr, shared in ((a, dst[a[:, 0]]), (l, src[l[:, 0]]), (r, dst[r[:, 0]])):
            key = np.stack([shared, arr[:, 0], arr[:, 1]], 1)
            assert np.array_equal(key, key[np.lexsort((key[:, 2], key[:, 1], key[:, 0]))])
        cnt = tuple(len(t[k]) for k in KINDS)
        if prev is not None:
            assert all(c <= p for c, p in zip(cnt, prev))           # a higher cut keeps fewer triplets
        prev = cnt
    assert prev == (0, 0, 0)                                        # nothing kept


def test_hand_built_graph():
    # hits 0,1 (left plane) -> 2,3 (middle) -> 4 (right).  Edge ids: 0: 0->2, 1: 0->3, 2: 1->2, 3: 2->4, 4: 3->4,
    # 5: 1->3 with a score below the cut.
    src = np.array([0, 0, 1, 2, 3, 1], np.int32)
    dst = np.array([2, 3, 2, 4, 4, 3], np.int32)
    sc = np.array([0.9, 0.8, 0.7, 0.9, 0.6, 0.1], np.float32)
    t = orc.triplets(5, src, dst, sc, 0.5)
    # shared hit 2: in {0, 2}, out {3}; shared hit 3: in {1}, out {4}
    np.testing.assert_array_equal(t["articulation"], [[0, 3], [2, 3], [1, 4]])
    np.testing.assert_array_equal(t["left_elbow"], [[0, 1]])                       # hit 0: out {0, 1}
    np.testing.assert_array_equal(t["right_elbow"], [[0, 2], [3, 4]])              # hit 2: in {0, 2}; hit 4: in {3, 4}
    t = orc.triplets(5, src, dst, sc, 0.1)                                         # inclusive cut: edge 5 is kept
    np.testing.assert_array_equal(t["articulation"], [[0, 3], [2, 3], [1, 4], [5, 4]])
    np.testing.assert_array_equal(t["left_elbow"], [[0, 1], [2, 5]])
    np.testing.assert_array_equal(t["right_elbow"], [[0, 2], [1, 5], [3, 4]])
    e = orc.triplets(5, src[:0], dst[:0], sc[:0], 0.5)
    assert all(e[k].shape == (0, 2) for k in KINDS)
