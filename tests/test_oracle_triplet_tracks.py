"""Pins of the oracle's triplet classifiers and track building from triplets:
hand-built graphs (the e+e- pair sharing its two initial hits; a plane-skipping triangle), a re-computation with
scipy's connected_components on the EDGE graph, special cases that reduce to the hit-level WCC (``orc.wcc``), and
invariants.  No GPU."""
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components

from conftest import layout_dict
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def all_kept(trip, value=1.0):
    return {k: np.full(len(trip[k]), value, np.float32) for k in ("articulation", "left_elbow", "right_elbow")}


def test_pair_sharing_two_initial_hits_gives_two_tracks():
    # hits: S1=0 S2=1 (shared), positron 2, 4; electron 3, 5.  Edges in (src, dst) order:
    src = np.array([0, 1, 1, 2, 3], np.int32)          # e0: S1->S2   e1: S2->P3   e2: S2->E3   e3: P3->P4   e4: E3->E4
    dst = np.array([1, 2, 3, 4, 5], np.int32)
    s = np.ones(5, np.float32)
    trip = orc.triplets(6, src, dst, s, 0.5)
    assert trip["articulation"].tolist() == [[0, 1], [0, 2], [1, 3], [2, 4]] and trip["left_elbow"].tolist() == [[1, 2]]
    ts = all_kept(trip)
    ts["left_elbow"][:] = 0.1                          # the two branches are different particles: the elbow is rejected
    out = orc.tracks_from_triplets(6, src, dst, s, 0.5, trip, ts, 0.5)
    assert out["edge_set"].tolist() == [0, 1, 2, 1, 2]
    assert out["joins"].tolist() == [[0, 1], [0, 2]]   # two articulations share the edge S1->S2
    assert out["tracks"] == [(0, 1, 2, 4), (0, 1, 3, 5)]
    # plain WCC on hits would have merged everything into one track
    assert len(set(orc.wcc(6, src, dst, s, 0.5).tolist())) == 1
    # accepting the elbow glues the two branches' first edges: the shared set grows, still two tracks
    out = orc.tracks_from_triplets(6, src, dst, s, 0.5, trip, all_kept(trip), 0.5)
    assert out["tracks"] == [(0, 1, 2, 3, 4), (0, 1, 2, 3, 5)]


def test_plane_skipping_triangle_elbows_remove_the_duplicate():
    src = np.array([0, 0, 1], np.int32)                # e0: A1->A2  e1: A1->A3 (skips a plane)  e2: A2->A3
    dst = np.array([1, 2, 2], np.int32)
    s = np.ones(3, np.float32)
    trip = orc.triplets(3, src, dst, s, 0.5)
    assert trip["articulation"].tolist() == [[0, 2]] and trip["left_elbow"].tolist() == [[0, 1]] and trip["right_elbow"].tolist() == [[1, 2]]
    assert orc.tracks_from_triplets(3, src, dst, s, 0.5, trip, all_kept(trip), 0.5)["tracks"] == [(0, 1, 2)]
    ts = all_kept(trip)
    ts["left_elbow"][:] = 0.0
    ts["right_elbow"][:] = 0.0
    assert orc.tracks_from_triplets(3, src, dst, s, 0.5, trip, ts, 0.5)["tracks"] == [(0, 1, 2), (0, 2)]
    ts["articulation"][:] = 0.0                        # no connection at all: every kept edge is its own 2-hit track
    assert orc.tracks_from_triplets(3, src, dst, s, 0.5, trip, ts, 0.5)["tracks"] == [(0, 1), (0, 2), (1, 2)]
    s[1] = 0.2                                         # the skipping edge cut by the EDGE score: it is no node of the edge graph
    trip = orc.triplets(3, src, dst, s, 0.5)
    out = orc.tracks_from_triplets(3, src, dst, s, 0.5, trip, all_kept(trip), 0.5)
    assert out["edge_set"].tolist() == [0, -1, 0] and out["tracks"] == [(0, 1, 2)]


def scipy_recomputation(n_hits, src, dst, scores, score_min, trip, ts, tmin):
    """The same four steps with library routines: connected_components on the edge graph, numpy unique for the
    duplicate removal and the sharing test."""
    E = len(src)
    keep = scores >= np.float32(score_min)
    elb = np.concatenate([trip[k][ts[k] >= np.float32(tmin)] for k in ("left_elbow", "right_elbow")]).reshape(-1, 2)
    _, sup = connected_components(sp.coo_matrix((np.ones(len(elb)), (elb[:, 0], elb[:, 1])), shape=(E, E)), directed=False)
    art = trip["articulation"][ts["articulation"] >= np.float32(tmin)].reshape(-1, 2)
    pairs = np.unique(np.stack([sup[art[:, 0]], sup[art[:, 1]]], 1).reshape(-1, 2), axis=0)
    pairs = pairs[pairs[:, 0] != pairs[:, 1]]
    n_succ = np.bincount(pairs[:, 0], minlength=E)
    n_pred = np.bincount(pairs[:, 1], minlength=E)
    shared = (n_succ[pairs[:, 0]] > 1) | (n_pred[pairs[:, 1]] > 1)
    un = pairs[~shared]
    # components of super-edges under the unshared pairs, expressed on the original edges
    rows = np.concatenate([elb[:, 0], art[:0, 0]]); cols = np.concatenate([elb[:, 1], art[:0, 1]])
    rep = np.zeros(E, np.int64)                         # a representative edge of every super-edge label
    rep[sup[::-1]] = np.arange(E)[::-1]
    rows = np.concatenate([rows, rep[un[:, 0]]]); cols = np.concatenate([cols, rep[un[:, 1]]])
    _, comp = connected_components(sp.coo_matrix((np.ones(len(rows)), (rows, cols)), shape=(E, E)), directed=False)
    name = np.full(comp.max() + 1, E, np.int64)
    np.minimum.at(name, comp[keep], np.arange(E)[keep])  # smallest kept edge id of the component
    edge_set = np.where(keep, name[comp], -1)
    joins = np.unique(np.stack([name[comp[rep[pairs[shared][:, 0]]]], name[comp[rep[pairs[shared][:, 1]]]]], 1).reshape(-1, 2), axis=0)
    hits = {}
    for e in np.flatnonzero(keep):
        hits.setdefault(int(edge_set[e]), set()).update((int(src[e]), int(dst[e])))
    touched = set(joins.ravel().tolist())
    tracks = [tuple(sorted(hits[c])) for c in sorted(hits) if c not in touched]
    tracks += [tuple(sorted(hits[a] | hits[b])) for a, b in joins.tolist()]
    return edge_set, joins, tracks


@pytest.mark.parametrize("seed,edge_cut,tmin", [(0, 0.5, 0.5), (1, 0.3, 0.5), (2, 0.5, 0.2), (3, 0.0, 0.8), (4, 0.5, 0.0)])
def test_against_scipy_on_the_c0_graph_with_random_triplet_scores(c0_oracle, seed, edge_cut, tmin):
    src, dst = c0_oracle["src"], c0_oracle["dst"]
    rng = np.random.default_rng(seed)
    s = rng.random(len(src)).astype(np.float32)        # random edge scores: many shared articulations, elbows, cycles
    trip = orc.triplets(239, src, dst, s, edge_cut)
    ts = {k: rng.random(len(trip[k])).astype(np.float32) for k in trip}
    out = orc.tracks_from_triplets(239, src, dst, s, edge_cut, trip, ts, tmin)
    es, joins, tracks = scipy_recomputation(239, src, dst, s, edge_cut, trip, ts, tmin)
    np.testing.assert_array_equal(out["edge_set"], es)
    np.testing.assert_array_equal(out["joins"], joins.reshape(-1, 2))
    assert out["tracks"] == tracks
    # invariants: both hits of every kept edge sit together in some track; a track never leaves the kept hit graph's component
    keep = s >= np.float32(edge_cut)
    lab = orc.wcc(239, src, dst, s, edge_cut)
    member = {}
    for t, tr in enumerate(out["tracks"]):
        assert len(set(lab[list(tr)].tolist())) == 1 and list(tr) == sorted(set(tr)) and len(tr) >= 2
        for h in tr:
            member.setdefault(h, set()).add(t)
    for e in np.flatnonzero(keep):
        assert member[int(src[e])] & member[int(dst[e])]
    n_sets = len(set(out["edge_set"][keep].tolist()))
    assert len(out["tracks"]) == n_sets - len(set(out["joins"].ravel().tolist())) + len(out["joins"])


def test_without_sharing_it_reduces_to_the_hit_level_wcc():
    """Disjoint simple paths (every hit has at most one kept edge in and one out), all triplets kept: no elbows, no shared
    articulation, so the tracks are exactly the hit-level WCC components with at least two hits (NEXT-1, ``orc.wcc``)."""
    rng = np.random.default_rng(7)
    n_tracks, length = 40, 9
    hits = np.arange(n_tracks * length).reshape(length, n_tracks)          # plane-major like the generator
    src = hits[:-1].ravel().astype(np.int32)
    dst = hits[1:].ravel().astype(np.int32)
    order = np.lexsort((dst, src))
    src, dst = src[order], dst[order]
    s = rng.random(len(src)).astype(np.float32)                            # the edge cut breaks the paths at random places
    trip = orc.triplets(hits.size, src, dst, s, 0.4)
    assert len(trip["left_elbow"]) == 0 and len(trip["right_elbow"]) == 0
    out = orc.tracks_from_triplets(hits.size, src, dst, s, 0.4, trip, all_kept(trip), 0.5)
    lab = orc.wcc(hits.size, src, dst, s, 0.4)
    want = sorted(tuple(np.flatnonzero(lab == l).tolist()) for l in np.unique(lab) if np.sum(lab == l) >= 2)
    assert sorted(out["tracks"]) == want and len(out["joins"]) == 0


def test_triplet_scores_are_the_classifier_on_concatenated_edge_encodings(c0, c0_oracle):
    import torch
    cfg, batch, blob = c0
    H, nl = cfg.gnn_hidden, cfg.gnn_mlp_hidden_layers + 1
    tw = synth.generate_triplet_weights(cfg)
    off = synth.triplet_layout(cfg)
    e = c0_oracle["e"]
    trip = orc.triplets(len(batch["r"]), c0_oracle["src"], c0_oracle["dst"], c0_oracle["scores"], 0.49)
    ts = orc.triplet_scores(e, trip, H, nl, tw, off["trip_art"][1], off["trip_elb"][1])
    assert all(len(ts[k]) == len(trip[k]) for k in trip) and sum(len(v) for v in ts.values()) > 500
    # library routine: torch float64 linear layers on the same weight blob
    for kind, name in (("articulation", "trip_art"), ("left_elbow", "trip_elb"), ("right_elbow", "trip_elb")):
        dims, o = off[name]
        x = torch.from_numpy(np.concatenate([e[trip[kind][:, 0]], e[trip[kind][:, 1]]], 1)).double()
        for l in range(len(dims) - 1):
            W = torch.from_numpy(tw[o:o + dims[l] * dims[l + 1]].reshape(dims[l + 1], dims[l])).double()
            b = torch.from_numpy(tw[o + dims[l] * dims[l + 1]:o + dims[l] * dims[l + 1] + dims[l + 1]]).double()
            x = torch.nn.functional.linear(x, W, b)
            if l < len(dims) - 2:
                x = torch.relu(x.float().double())                         # stored activations are fp32
            o += dims[l] * dims[l + 1] + dims[l + 1]
        np.testing.assert_allclose(ts[kind], torch.sigmoid(x[:, 0]).numpy(), rtol=0, atol=2e-6)
    # the order of the two edges matters (concatenation, not a sum), and zero weights give exactly 0.5
    sw = {k: v[:, ::-1].copy() for k, v in trip.items()}
    assert np.abs(orc.triplet_scores(e, sw, H, nl, tw, off["trip_art"][1], off["trip_elb"][1])["articulation"] - ts["articulation"]).max() > 1e-4
    z = orc.triplet_scores(e, trip, H, nl, np.zeros_like(tw), off["trip_art"][1], off["trip_elb"][1])
    assert all(np.all(v == 0.5) for v in z.values())
    assert ts["articulation"].std() > 1e-3
