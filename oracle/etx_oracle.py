"""TEST INFRASTRUCTURE — Python (ctypes) face of the CPU oracle ``etx_oracle.cpp``.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference`` legs
may import this.  It imports nothing from the CUDA package; inputs are plain numpy arrays.
Every function cites the passage of the thesis (P:line of PAPER.md) its C++ body follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "etx_oracle.cpp")
_LIB = os.path.join(_DIR, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (the radius predicate must not be FMA-contracted) -fopenmp."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-fPIC",
                               "-shared", "-o", _LIB, _SRC])
    return _LIB


def _p(a: Optional[np.ndarray], t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_build_graph.restype = C.c_int64
        _lib.orc_candidate_d2.restype = C.c_int64
        _lib.orc_build_graph_kmax.restype = C.c_int64
    return _lib


def n_threads() -> int:
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def features(batch: Dict[str, np.ndarray], center: Sequence[float], scale: Sequence[float]):
    """a0: returns f_emb [N,3] (r,phi,z) and f_node [N,3] (x,y,z)."""
    n = len(batch["r"])
    fe = np.empty((n, 3), np.float32)
    fn = np.empty((n, 3), np.float32)
    c, s = _f32(center), _f32(scale)
    arrs = [_f32(batch[k]) for k in ("r", "phi", "z", "x", "y")]
    lib().orc_features(C.c_int64(n), *[_p(a, C.c_float) for a in arrs], _p(c, C.c_float),
                       _p(s, C.c_float), _p(fe, C.c_float), _p(fn, C.c_float))
    return fe, fn


def mlp(x: np.ndarray, dims: Sequence[int], blob: np.ndarray, offset: int) -> np.ndarray:
    """Eqs. 4.24-4.27: ReLU hidden layers, linear output, weights at blob[offset:]."""
    x = _f32(x)
    n = x.shape[0]
    d = np.asarray(dims, dtype=np.int32)
    assert x.shape[1] == d[0]
    out = np.empty((n, int(d[-1])), np.float32)
    w = blob[offset:]
    lib().orc_mlp(C.c_int64(n), C.c_int32(len(d) - 1), _p(d, C.c_int32), _p(w, C.c_float),
                  _p(x, C.c_float), _p(out, C.c_float))
    return out


def quantize(x: np.ndarray, alpha: float):
    """Eqs. 4.31-4.33: S = alpha / 127, codes = clip(round(x / S), -127, 127).  Returns (codes, S)."""
    x = _f32(x).ravel()
    codes = np.empty(x.size, np.int8)
    S = C.c_float(0.0)
    lib().orc_quantize(C.c_int64(x.size), _p(x, C.c_float), C.c_float(alpha), _p(codes, C.c_int8), C.byref(S))
    return codes, float(S.value)


def mlp_int8(x: np.ndarray, dims: Sequence[int], blob: np.ndarray, offset: int, act_alpha: Sequence[float]) -> np.ndarray:
    """Next row: the MLP chain with INT8 weights and activations (static PTQ, symmetric per-tensor
    scales); act_alpha[l] = calibrated range of layer l's input."""
    x = _f32(x)
    d = np.ascontiguousarray(dims, np.int32)
    al = _f32(np.asarray(act_alpha, np.float32))
    assert len(al) == len(d) - 1
    n = x.shape[0]
    out = np.empty((n, int(d[-1])), np.float32)
    w = blob[offset:]
    lib().orc_mlp_int8(C.c_int64(n), C.c_int32(len(d) - 1), _p(d, C.c_int32), _p(w, C.c_float),
                       _p(x, C.c_float), _p(al, C.c_float), _p(out, C.c_float))
    return out


def quantize_fp8(x: np.ndarray, alpha: float):
    """Next row (NEXT-3, FP8; DESIGN reading Q26): S = alpha / 448, value = e4m3(clip(x * fl(1/S), -448, 448)), round to
    nearest even.  Returns (e4m3 values as float32 -- multiply by S to de-quantise --, S)."""
    x = _f32(x).ravel()
    vals = np.empty(x.size, np.float32)
    S = C.c_float(0.0)
    lib().orc_quantize_fp8(C.c_int64(x.size), _p(x, C.c_float), C.c_float(alpha), _p(vals, C.c_float), C.byref(S))
    return vals, float(S.value)


def mlp_fp8(x: np.ndarray, dims: Sequence[int], blob: np.ndarray, offset: int, act_alpha: Sequence[float]) -> np.ndarray:
    """The MLP chain with e4m3 weights and activations (static per-tensor scales, exact sums, fp32 de-quantisation and
    biases); act_alpha[l] = calibrated range of layer l's input (the ranges of the INT8 row: a max observer)."""
    x = _f32(x)
    d = np.ascontiguousarray(dims, np.int32)
    al = _f32(np.asarray(act_alpha, np.float32))
    assert len(al) == len(d) - 1
    n = x.shape[0]
    out = np.empty((n, int(d[-1])), np.float32)
    w = blob[offset:]
    lib().orc_mlp_fp8(C.c_int64(n), C.c_int32(len(d) - 1), _p(d, C.c_int32), _p(w, C.c_float),
                      _p(x, C.c_float), _p(al, C.c_float), _p(out, C.c_float))
    return out


def int8_calibration(x: np.ndarray, dims: Sequence[int], blob: np.ndarray, offset: int) -> np.ndarray:
    """Static PTQ calibration with a max observer: range of every layer's INPUT over the sample x,
    taken from the fp32 oracle MLP."""
    x = _f32(x)
    alphas = [float(np.abs(x).max())]
    for l in range(1, len(dims) - 1):
        z = mlp(x, list(dims[:l + 1]), blob, offset)          # linear output of layer l
        alphas.append(float(np.maximum(z, 0.0).max()))        # its ReLU is the next layer's input
    return np.asarray(alphas, np.float32)


def build_graph(event_ptr, plane, emb, r2_max: float, gap: int, n_planes: int = 26,
                band: float = 0.0, want_border: bool = False):
    """a2 (Eq. 8.1): edges (src, dst) in (src asc, dst asc) order.
    With want_border also the (i, j) pairs with |d - r| <= band, d evaluated in double (Q17)."""
    event_ptr = np.ascontiguousarray(event_ptr, np.int32)
    plane = np.ascontiguousarray(plane, np.uint8)
    emb = _f32(emb)
    n_ev = len(event_ptr) - 1
    d = emb.shape[1]
    nb = C.c_int64(0)
    cap = 1 << 16
    while True:
        src = np.empty(cap, np.int32)
        dst = np.empty(cap, np.int32)
        bp = np.empty((cap, 2), np.int32) if want_border else None
        E = lib().orc_build_graph(C.c_int32(n_ev), _p(event_ptr, C.c_int32), _p(plane, C.c_uint8),
                                  C.c_int32(n_planes), _p(emb, C.c_float), C.c_int32(d),
                                  C.c_float(r2_max), C.c_int32(gap), _p(src, C.c_int32),
                                  _p(dst, C.c_int32), C.c_int64(cap), C.c_double(band),
                                  _p(bp, C.c_int32), C.c_int64(cap), C.byref(nb))
        if E <= cap and nb.value <= cap:
            break
        cap = max(int(E), int(nb.value)) + 16
    if want_border:
        return src[:E].copy(), dst[:E].copy(), bp[:nb.value].copy()
    return src[:E].copy(), dst[:E].copy()


def build_graph_kmax(event_ptr, plane, emb, r2_max: float, gap: int, k_max: int, n_planes: int = 26):
    """Next row (Algorithm 1): the radius graph with at most k_max out-edges per hit, the
    k_max nearest by (d^2 fp32, then j); edges in (src asc, dst asc) order.  k_max <= 0: no cap."""
    event_ptr = np.ascontiguousarray(event_ptr, np.int32)
    plane = np.ascontiguousarray(plane, np.uint8)
    emb = _f32(emb)
    n_ev = len(event_ptr) - 1
    cap = 1 << 16
    while True:
        src = np.empty(cap, np.int32)
        dst = np.empty(cap, np.int32)
        E = lib().orc_build_graph_kmax(C.c_int32(n_ev), _p(event_ptr, C.c_int32), _p(plane, C.c_uint8),
                                       C.c_int32(n_planes), _p(emb, C.c_float), C.c_int32(emb.shape[1]),
                                       C.c_float(r2_max), C.c_int32(gap), C.c_int32(k_max),
                                       _p(src, C.c_int32), _p(dst, C.c_int32), C.c_int64(cap))
        if E <= cap:
            break
        cap = int(E) + 16
    return src[:E].copy(), dst[:E].copy()


def candidate_d2(event_ptr, plane, emb, gap: int, n_planes: int = 26) -> np.ndarray:
    """All candidate pairs' d^2 in double (for the Q4 radius calibration)."""
    event_ptr = np.ascontiguousarray(event_ptr, np.int32)
    plane = np.ascontiguousarray(plane, np.uint8)
    emb = _f32(emb)
    args = (C.c_int32(len(event_ptr) - 1), _p(event_ptr, C.c_int32), _p(plane, C.c_uint8),
            C.c_int32(n_planes), _p(emb, C.c_float), C.c_int32(emb.shape[1]), C.c_int32(gap))
    n = lib().orc_candidate_d2(*args, None, C.c_int64(0))
    out = np.empty(n, np.float64)
    lib().orc_candidate_d2(*args, _p(out, C.c_double), C.c_int64(n))
    return out


def scatter(n_nodes: int, src, dst, e) -> np.ndarray:
    """a4, Eq. 8.5: m [n_nodes, 2H] = [sum of outgoing, sum of incoming]."""
    e = _f32(e)
    src = np.ascontiguousarray(src, np.int32)
    dst = np.ascontiguousarray(dst, np.int32)
    H = e.shape[1]
    m = np.empty((n_nodes, 2 * H), np.float32)
    lib().orc_scatter(C.c_int64(n_nodes), C.c_int64(len(src)), _p(src, C.c_int32), _p(dst, C.c_int32),
                      _p(e, C.c_float), C.c_int32(H), _p(m, C.c_float))
    return m


def gnn_forward(f_node, src, dst, H: int, n_layers: int, n_iter: int, blob: np.ndarray,
                off_node_enc: int, off_edge_enc: int, off_node_net: Sequence[int],
                off_edge_net: Sequence[int]) -> Tuple[np.ndarray, np.ndarray]:
    """a3-a6: returns h^n [N,H], e^n [E,H]."""
    f_node = _f32(f_node)
    src = np.ascontiguousarray(src, np.int32)
    dst = np.ascontiguousarray(dst, np.int32)
    n, E = f_node.shape[0], len(src)
    h = np.empty((n, H), np.float32)
    e = np.empty((E, H), np.float32)
    base = blob.ctypes.data
    PP = C.POINTER(C.c_float)
    nn = (PP * max(n_iter, 1))(*[C.cast(base + 4 * o, PP) for o in off_node_net])
    en = (PP * max(n_iter, 1))(*[C.cast(base + 4 * o, PP) for o in off_edge_net])
    lib().orc_gnn_forward(C.c_int64(n), C.c_int64(E), _p(src, C.c_int32), _p(dst, C.c_int32),
                          _p(f_node, C.c_float), C.c_int32(H), C.c_int32(n_layers), C.c_int32(n_iter),
                          C.cast(base + 4 * off_node_enc, PP), C.cast(base + 4 * off_edge_enc, PP),
                          nn, en, _p(h, C.c_float), _p(e, C.c_float))
    return h, e


def edge_scores(e, H: int, n_layers: int, blob: np.ndarray, off_cls: int, want_logits=False):
    """a7 (sigma P:1309): scores [E] fp32."""
    e = _f32(e)
    E = e.shape[0]
    s = np.empty(E, np.float32)
    lg = np.empty(E, np.float32)
    lib().orc_edge_scores(C.c_int64(E), _p(e, C.c_float), C.c_int32(H), C.c_int32(n_layers),
                          _p(blob[off_cls:], C.c_float), _p(s, C.c_float), _p(lg, C.c_float))
    return (s, lg) if want_logits else s


def scatter_f32(n_nodes: int, src, dst, e) -> np.ndarray:
    """NEXT-3 (GNN part): Eq. 8.5 in plain fp32, sequential adds in ascending edge id (see orc_scatter_f32)."""
    e = _f32(e)
    src = np.ascontiguousarray(src, np.int32)
    dst = np.ascontiguousarray(dst, np.int32)
    H = e.shape[1]
    m = np.empty((n_nodes, 2 * H), np.float32)
    lib().orc_scatter_f32(C.c_int64(n_nodes), C.c_int64(len(src)), _p(src, C.c_int32), _p(dst, C.c_int32),
                          _p(e, C.c_float), C.c_int32(H), _p(m, C.c_float))
    return m


GNN_MLPS = ("node_enc", "edge_enc", "node_net", "edge_net", "cls")


def gnn_mlp_names(n_iter: int) -> List[str]:
    """The GNN's MLPs in the order their calibrated ranges are stored / handed to the library."""
    return ["node_enc", "edge_enc"] + [f"{n}_{k}" for k in range(n_iter) for n in ("node_net", "edge_net")] + ["cls"]


def _relu(x):
    return np.where(x > 0, x, np.float32(0.0)).astype(np.float32)


def gnn_forward_steps(f_node, src, dst, n_iter: int, mlp_fn, scatter_fn):
    """a3-a7 written out step by step in the thesis' order on top of an MLP
    evaluator ``mlp_fn(name, x) -> y`` and an aggregator ``scatter_fn(n_nodes, src, dst, e) -> m``; the concatenation
    orders are those of the hot path (Q10: [h, m_out, m_in], [h_src, h_dst, e], [h_src, h_dst]); residual adds are
    single fp32 additions.  Returns h^n, e^n and the classifier's logits."""
    f_node = _f32(f_node)
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    n = f_node.shape[0]
    h = mlp_fn("node_enc", f_node)
    e = mlp_fn("edge_enc", np.concatenate([h[src], h[dst]], axis=1))
    for k in range(n_iter):
        m = scatter_fn(n, src, dst, e)
        h = (h + mlp_fn(f"node_net_{k}", np.concatenate([h, m], axis=1))).astype(np.float32)
        e = (e + mlp_fn(f"edge_net_{k}", np.concatenate([h[src], h[dst], e], axis=1))).astype(np.float32)
    return h, e, mlp_fn("cls", e)[:, 0]


def gnn_int8_calibration(f_node, src, dst, n_iter: int, blob: np.ndarray, layout) -> Dict[str, List[float]]:
    """Static PTQ calibration of the GNN's MLPs with a max observer: the fp32 model (this module's
    plain MLP and double-accumulating scatter) runs on the sample and the range of every layer's INPUT is recorded."""
    blob = _f32(blob)
    ranges: Dict[str, List[float]] = {}

    def fp32_mlp(name, x):
        dims, off = layout[name]
        ranges[name] = [float(a) for a in int8_calibration(x, dims, blob, off)]
        return mlp(x, dims, blob, off)

    gnn_forward_steps(f_node, src, dst, n_iter, fp32_mlp, scatter)
    return ranges


def gnn_forward_int8(f_node, src, dst, n_iter: int, blob: np.ndarray, layout, act_alpha: Dict[str, Sequence[float]]):
    """NEXT-3 (GNN part; "quantization of the GNN holds the most potential"; scheme of Eqs. 4.31-4.33): every MLP
    of the GNN evaluated by ``mlp_int8`` (INT8 codes for every layer's input and weight, exact integer sums, fp32
    de-quantisation and biases), state h, e and the aggregate m in fp32, fp32 scatter (``scatter_f32``), fp32 residual
    adds.  One exception (DESIGN Q24): the node encoder's FIRST layer -- 3 raw geometry features in -- stays the fp32
    layer of the hot path (double accumulation), its ReLU output is the first quantised tensor.  act_alpha[name][l] is
    the calibrated range of layer l's input (entry 0 of node_enc is unused).  Returns h^n, e^n, logits, scores."""
    blob = _f32(blob)

    def q_mlp(name, x):
        dims, off = layout[name]
        al = list(act_alpha[name])
        if name == "node_enc":
            x = _relu(mlp(x, dims[:2], blob, off))
            off += dims[0] * dims[1] + dims[1]
            dims, al = dims[1:], al[1:]
        return mlp_int8(x, dims, blob, off, al)

    h, e, logit = gnn_forward_steps(f_node, src, dst, n_iter, q_mlp, scatter_f32)
    s = (1.0 / (1.0 + np.exp(-logit.astype(np.float64)))).astype(np.float32)
    return h, e, logit, s


def gnn_forward_fp8(f_node, src, dst, n_iter: int, blob: np.ndarray, layout, act_alpha: Dict[str, Sequence[float]]):
    """NEXT-3 (GNN part) in FP8 e4m3: ``gnn_forward_int8`` with ``mlp_fp8`` in place of ``mlp_int8`` -- e4m3 values for every
    layer's input and weight, fp32 state, fp32 sequential scatter, fp32 residual adds, the node encoder's first layer in
    fp32; the same calibrated ranges.  Returns h^n, e^n, logits, scores."""
    blob = _f32(blob)

    def q_mlp(name, x):
        dims, off = layout[name]
        al = list(act_alpha[name])
        if name == "node_enc":
            x = _relu(mlp(x, dims[:2], blob, off))
            off += dims[0] * dims[1] + dims[1]
            dims, al = dims[1:], al[1:]
        return mlp_fp8(x, dims, blob, off, al)

    h, e, logit = gnn_forward_steps(f_node, src, dst, n_iter, q_mlp, scatter_f32)
    s = (1.0 / (1.0 + np.exp(-logit.astype(np.float64)))).astype(np.float32)
    return h, e, logit, s


def wcc(n_hits: int, src, dst, scores, score_min: float) -> np.ndarray:
    """NEXT-1: labels [n_hits] = smallest hit index of the weakly connected
    component of the purified graph (edges with score >= score_min)."""
    src = np.ascontiguousarray(src, np.int32)
    dst = np.ascontiguousarray(dst, np.int32)
    scores = _f32(scores)
    labels = np.empty(n_hits, np.int32)
    lib().orc_wcc(C.c_int64(n_hits), C.c_int64(len(src)), _p(src, C.c_int32), _p(dst, C.c_int32),
                  _p(scores, C.c_float), C.c_float(score_min), _p(labels, C.c_int32))
    return labels


def triplets(n_hits: int, src, dst, scores, score_min: float) -> Dict[str, np.ndarray]:
    """NEXT-4 (triplet building, Fig. 8.13): the edge connections of the purified hit graph (edges
    with score >= score_min, the same cut as ``wcc``).  A triplet is two kept edges sharing a hit C:

    * articulation: A -> C and C -> B (the common hit in the middle)        -> rows (edge A->C, edge C->B)
    * left elbow:   C -> A and C -> B (the common hit on the left)          -> rows (e1, e2), e1 < e2
    * right elbow:  A -> C and B -> C (the common hit on the right)         -> rows (e1, e2), e1 < e2

    Plain definition, pure Python loops: for every hit C in ascending order, its kept incoming edges I(C) and
    kept outgoing edges O(C) in ascending edge id; articulations = I(C) x O(C) (first index slowest), elbows =
    the unordered pairs of O(C) / of I(C) in lexicographic order.  Returns int32 arrays [n, 2] of EDGE IDS under
    "articulation", "left_elbow", "right_elbow".  The thesis fixes no order (several listings are correct);
    this one is the order the GPU path is required to reproduce, so the comparison is an array comparison."""
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    keep = _f32(scores) >= np.float32(score_min)
    ins: List[List[int]] = [[] for _ in range(n_hits)]
    outs: List[List[int]] = [[] for _ in range(n_hits)]
    for e in range(len(src)):                       # ascending edge id
        if keep[e]:
            outs[src[e]].append(e)
            ins[dst[e]].append(e)
    art, left, right = [], [], []
    for c in range(n_hits):
        for a in ins[c]:
            for b in outs[c]:
                art.append((a, b))
        for i, a in enumerate(outs[c]):
            for b in outs[c][i + 1:]:
                left.append((a, b))
        for i, a in enumerate(ins[c]):
            for b in ins[c][i + 1:]:
                right.append((a, b))
    as_arr = lambda t: np.asarray(t, np.int32).reshape(-1, 2)
    return {"articulation": as_arr(art), "left_elbow": as_arr(left), "right_elbow": as_arr(right)}


def triplet_scores(e, trip: Dict[str, np.ndarray], H: int, n_layers: int, blob: np.ndarray, off_art: int,
                   off_elb: int) -> Dict[str, np.ndarray]:
    """NEXT-4 (triplet classifiers, "edge encodings are sufficient for both the edge classifier and triplet
    classifier"; Fig. 8.12 caption P:2330 "[.,.] represents concatenation"; "separate triplet classifiers for
    articulations and elbows ... each an MLP ending with a layer with 1 unit, and a sigmoid").  Reading (DESIGN Q23):
    s = sigmoid(MLP_k([e_first, e_second])) on the rows ``triplets`` lists, MLP_art for articulations
    (first = A->C, second = C->B), MLP_elb for BOTH elbow kinds (first < second edge id); each MLP is 2H -> H .. H -> 1
    with the GNN's layer count, ReLU hidden layers, weights at blob[off_*].  Double accumulation (orc_mlp), sigmoid in
    double, stored fp32 -- the same arithmetic convention as ``edge_scores``."""
    e = _f32(e)
    dims = [2 * H] + [H] * (n_layers - 1) + [1]
    out = {}
    for name, off in (("articulation", off_art), ("left_elbow", off_elb), ("right_elbow", off_elb)):
        rows = np.asarray(trip[name], np.int64).reshape(-1, 2)
        if len(rows) == 0:
            out[name] = np.zeros(0, np.float32)
            continue
        x = np.concatenate([e[rows[:, 0]], e[rows[:, 1]]], axis=1)
        logit = mlp(x, dims, blob, off)[:, 0].astype(np.float64)
        out[name] = (1.0 / (1.0 + np.exp(-logit))).astype(np.float32)
    return out


def tracks_from_triplets(n_hits: int, src, dst, scores, score_min: float, trip: Dict[str, np.ndarray],
                         trip_scores: Dict[str, np.ndarray], trip_min: float) -> Dict[str, object]:
    """NEXT-4 (track building from triplets, the four steps of P:2363, section 8.3.5).  Plain Python, step by step.

    Nodes of the EDGE graph are the kept edges (score >= score_min); its connections are the kept triplets
    (triplet score >= trip_min, inclusive like the edge cut).  Reading of the four steps (DESIGN Q23):

    1. "the left elbows and right elbows are connected ... Duplicate edges resulting from elbow connections are removed":
       the two edges of every kept elbow are merged into one super-edge (union-find); every kept articulation (a, b)
       becomes the pair (S(a), S(b)) of super-edges, pairs with S(a) == S(b) vanish and equal pairs count once.
    2. "a WCC algorithm is applied to the edge graph, excluding these shared articulations": an articulation pair (u, v)
       is SHARED iff u has two or more distinct successors or v has two or more distinct predecessors among the pairs
       ("two articulations sharing an edge").  Connected sets = components of the super-edges under the unshared pairs.
    3. "a new track is formed for each remaining articulation, effectively duplicating the shared set of connected
       edges": every distinct pair (set of u, set of v) of a shared articulation gives the track  set(u) U set(v);  a
       connected set touched by no shared articulation is a track by itself.
    4. "edges are replaced by their corresponding hits": a track is the ascending list of the hits of its edges.

    Labels: a connected set is named by its smallest edge id.  Returns
      "edge_set"  int32 [E]   the set of every edge (-1 for an edge cut by score_min),
      "joins"     int32 [J,2] the distinct (set of u, set of v) pairs of the shared articulations, ascending,
      "tracks"    list of ascending hit tuples, ordered: untouched sets by label, then the joins in order."""
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    E = len(src)
    keep = _f32(scores) >= np.float32(score_min)
    parent = list(range(E))

    def find(parent, x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x

    def union(parent, a, b):
        ra, rb = find(parent, a), find(parent, b)
        if ra != rb:
            parent[max(ra, rb)] = min(ra, rb)              # the root is the smallest edge id

    tmin = np.float32(trip_min)
    for kind in ("left_elbow", "right_elbow"):             # step 1: connect the elbows
        for (a, b), s in zip(np.asarray(trip[kind], np.int64).reshape(-1, 2), _f32(trip_scores[kind])):
            if s >= tmin:
                union(parent, int(a), int(b))
    pairs = set()
    for (a, b), s in zip(np.asarray(trip["articulation"], np.int64).reshape(-1, 2), _f32(trip_scores["articulation"])):
        if s >= tmin:
            u, v = find(parent, int(a)), find(parent, int(b))
            if u != v:
                pairs.add((u, v))                          # duplicates removed
    succ: Dict[int, set] = {}
    pred: Dict[int, set] = {}
    for u, v in pairs:
        succ.setdefault(u, set()).add(v)
        pred.setdefault(v, set()).add(u)
    shared = {(u, v) for (u, v) in pairs if len(succ[u]) > 1 or len(pred[v]) > 1}
    comp = list(parent)                                    # step 2: WCC without the shared articulations
    for u, v in sorted(pairs - shared):
        union(comp, u, v)
    edge_set = np.full(E, -1, np.int32)
    for e in range(E):
        if keep[e]:
            edge_set[e] = find(comp, e)
    joins = sorted({(int(edge_set[u]), int(edge_set[v])) for (u, v) in shared})      # step 3
    touched = {c for j in joins for c in j}
    hits_of: Dict[int, set] = {}
    for e in range(E):                                     # step 4: edges -> hits
        if keep[e]:
            hits_of.setdefault(int(edge_set[e]), set()).update((int(src[e]), int(dst[e])))
    tracks = [tuple(sorted(hits_of[c])) for c in sorted(hits_of) if c not in touched]
    tracks += [tuple(sorted(hits_of[a] | hits_of[b])) for (a, b) in joins]
    return {"edge_set": edge_set, "joins": np.asarray(joins, np.int32).reshape(-1, 2), "tracks": tracks}


def run_path(batch: Dict[str, np.ndarray], blob: np.ndarray, layout: Dict[str, Tuple[Tuple[int, ...], int]],
             H: int, n_iter: int, r2_max: float, gap: int, center, scale, n_planes: int = 26,
             graph: Optional[Tuple[np.ndarray, np.ndarray]] = None) -> Dict[str, np.ndarray]:
    """Whole hot path hits -> edge scores, steps a0..a7 in the thesis' order.

    ``layout`` maps MLP name -> (dims, float offset in blob): "emb", "node_enc", "edge_enc",
    "node_net_k", "edge_net_k", "cls".  ``graph`` overrides the built graph (for Q16-style tests)."""
    blob = _f32(blob)
    fe, fn = features(batch, center, scale)
    emb = mlp(fe, *_lo(layout, "emb", blob))
    if graph is None:
        src, dst = build_graph(batch["event_ptr"], batch["plane"], emb, r2_max, gap, n_planes)
    else:
        src, dst = graph
    n_layers = len(layout["node_enc"][0]) - 1
    h, e = gnn_forward(fn, src, dst, H, n_layers, n_iter, blob, layout["node_enc"][1],
                       layout["edge_enc"][1], [layout[f"node_net_{k}"][1] for k in range(n_iter)],
                       [layout[f"edge_net_{k}"][1] for k in range(n_iter)])
    s, lg = edge_scores(e, H, n_layers, blob, layout["cls"][1], want_logits=True)
    return {"f_emb": fe, "f_node": fn, "emb": emb, "src": src, "dst": dst, "h": h, "e": e,
            "scores": s, "logits": lg}


def _lo(layout, name, blob):
    dims, off = layout[name]
    return dims, blob, off
