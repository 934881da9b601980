"""Pins for the oracle's score cut + weakly-connected-components track building
(edges below the minimum score are removed; WCC)."""
import numpy as np
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

from oracle import etx_oracle as orc


def scipy_labels(n, src, dst, keep):
    a = coo_matrix((np.ones(keep.sum()), (src[keep], dst[keep])), shape=(n, n))
    _, comp = connected_components(a, directed=True, connection="weak")
    first = np.full(comp.max() + 1, n, np.int64)
    np.minimum.at(first, comp, np.arange(n))
    return first[comp].astype(np.int32)                     # smallest index of each component


def test_against_scipy_on_c1(c1_oracle):
    src, dst, s = c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"]
    n = c1_oracle["h"].shape[0]
    for s_min in (0.0, float(np.median(s)), float(np.quantile(s, 0.9)), 2.0):
        lab = orc.wcc(n, src, dst, s, s_min)
        np.testing.assert_array_equal(lab, scipy_labels(n, src, dst, s >= np.float32(s_min)))
    assert np.array_equal(orc.wcc(n, src, dst, s, 2.0), np.arange(n))      # nothing kept: every hit alone
    lab0 = orc.wcc(n, src, dst, s, 0.0)
    assert len(np.unique(lab0)) < len(np.unique(orc.wcc(n, src, dst, s, float(np.median(s)))))   # cutting splits


def test_hand_built_graphs():
    # two straight tracks 0-2-4 and 1-3-5, plus a low-score fake edge 2->5 joining them
    src = np.array([0, 2, 1, 3, 2], np.int32)
    dst = np.array([2, 4, 3, 5, 5], np.int32)
    sc = np.array([0.9, 0.8, 0.95, 0.7, 0.2], np.float32)
    np.testing.assert_array_equal(orc.wcc(6, src, dst, sc, 0.5), [0, 1, 0, 1, 0, 1])
    np.testing.assert_array_equal(orc.wcc(6, src, dst, sc, 0.1), [0, 0, 0, 0, 0, 0])   # fake edge kept: merged
    np.testing.assert_array_equal(orc.wcc(6, src, dst, sc, 0.2), [0, 0, 0, 0, 0, 0])   # >= is inclusive
    np.testing.assert_array_equal(orc.wcc(6, src, dst, sc, np.nextafter(np.float32(0.2), np.float32(1))), [0, 1, 0, 1, 0, 1])
    # zig-zag a0->b1, c0->b1, c0->d1, e0->d1 (hits 0,1,2 on the left plane; 3,4 on the right): one
    # forward + one backward plane sweep leaves hit 2 with label 1; the exact WCC is all 0
    src = np.array([0, 1, 1, 2], np.int32)
    dst = np.array([3, 3, 4, 4], np.int32)
    np.testing.assert_array_equal(orc.wcc(5, src, dst, np.ones(4, np.float32), 0.5), [0, 0, 0, 0, 0])
    # weakly connected: direction does not matter
    np.testing.assert_array_equal(orc.wcc(3, np.array([2, 2], np.int32), np.array([0, 1], np.int32),
                                          np.ones(2, np.float32), 0.5), [0, 0, 0])


def test_partition_invariants(c1_oracle):
    src, dst, s = c1_oracle["src"], c1_oracle["dst"], c1_oracle["scores"]
    n = c1_oracle["h"].shape[0]
    s_min = float(np.median(s))
    lab = orc.wcc(n, src, dst, s, s_min)
    assert np.all(lab <= np.arange(n)) and np.all(lab[lab] == lab)           # representative = smallest member
    keep = s >= np.float32(s_min)
    assert np.all(lab[src[keep]] == lab[dst[keep]])                          # kept edges never cross components
    # minimality: every component is connected by kept edges (a spanning check via scipy above), and
    # removing edges can only refine the partition
    finer = orc.wcc(n, src, dst, s, float(np.quantile(s, 0.95)))
    assert np.all(lab[finer] == lab)                                          # each fine component inside a coarse one
