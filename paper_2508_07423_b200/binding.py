"""ctypes binding of libetx (include/etx.h): same names, argument marshalling only.

PyTorch supplies device memory (tensors) and the stream; every step of the path runs in the library's
kernels.  There is no fallback: if ``libetx.so`` is missing or fails to load, importing the symbols
raises, and every failed call raises ``EtxError`` with the library's message.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np
import torch

from . import synth

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libetx.so")
ETX_MAX_MLP_LAYERS = 8
ETX_OK, ETX_ERR_INVALID, ETX_ERR_CAPACITY, ETX_ERR_CUDA, ETX_ERR_UNSORTED, ETX_ERR_NOMEM = 0, -1, -2, -3, -4, -5

EXPORTS = ["etx_weight_count", "etx_create", "etx_destroy", "etx_last_error", "etx_workspace_bytes",
           "etx_set_workspace", "etx_embed", "etx_embed_bf16", "etx_embed_int8", "etx_build_graph", "etx_gnn_forward", "etx_edge_scores",
           "etx_infer_host", "etx_launch_count", "etx_profile_enable", "etx_profile_read", "etx_build_tracks",
           "etx_build_triplets", "etx_build_triplets_static", "etx_triplet_weight_count", "etx_set_triplet_classifiers", "etx_triplet_scores",
           "etx_triplet_tracks_workspace_bytes", "etx_build_tracks_from_triplets", "etx_set_int8_ranges",
           "etx_measure_alu_peak"]
KERNEL_CLASSES = ["embed", "graph", "node_enc", "edge_enc", "scatter", "node_net", "edge_net", "cls", "tracks", "edge_proj"]


class EtxError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libetx status {status}: {msg}")
        self.status = status


def etx_measure_alu_peak(device: int, kind: int) -> float:
    """Arithmetic operations per second of the ALU microbenchmark (etx.h): kind 0 scalar add+mul, 1 packed pairs, 2 FFMA."""
    out = C.c_double(0.0)
    st = load_library().etx_measure_alu_peak(int(device), int(kind), C.byref(out))
    if st != 0:
        raise EtxError(st, "etx_measure_alu_peak failed")
    return float(out.value)


class ModelDesc(C.Structure):
    _fields_ = [("emb_n_layers", C.c_int32), ("emb_dims", C.c_int32 * (ETX_MAX_MLP_LAYERS + 1)),
                ("gnn_hidden", C.c_int32), ("gnn_n_layers", C.c_int32), ("n_iter", C.c_int32),
                ("precision", C.c_int32), ("n_planes", C.c_int32),
                ("norm_center", C.c_float * 5), ("norm_scale", C.c_float * 5)]


class Batch(C.Structure):
    _fields_ = [("n_events", C.c_int32), ("n_hits", C.c_int32), ("d_event_ptr", C.c_void_p),
                ("d_plane", C.c_void_p), ("d_r", C.c_void_p), ("d_phi", C.c_void_p), ("d_z", C.c_void_p),
                ("d_x", C.c_void_p), ("d_y", C.c_void_p)]


class BatchHost(C.Structure):
    _fields_ = [("n_events", C.c_int32), ("n_hits", C.c_int32), ("h_event_ptr", C.c_void_p),
                ("h_plane", C.c_void_p), ("h_r", C.c_void_p), ("h_phi", C.c_void_p), ("h_z", C.c_void_p),
                ("h_x", C.c_void_p), ("h_y", C.c_void_p)]


class Graph(C.Structure):
    _fields_ = [("edge_capacity", C.c_int64), ("n_edges", C.c_int64), ("d_row_ptr", C.c_void_p),
                ("d_src", C.c_void_p), ("d_dst", C.c_void_p), ("d_in_ptr", C.c_void_p),
                ("d_in_perm", C.c_void_p)]


class Triplets(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("n", C.c_int64 * 3), ("d_ptr", C.c_void_p), ("d_first", C.c_void_p),
                ("d_second", C.c_void_p)]


class Tracks(C.Structure):
    _fields_ = [("join_capacity", C.c_int64), ("track_capacity", C.c_int64), ("hit_capacity", C.c_int64),
                ("n_joins", C.c_int64), ("n_plain", C.c_int64), ("n_tracks", C.c_int64), ("n_track_hits", C.c_int64),
                ("d_edge_set", C.c_void_p), ("d_joins", C.c_void_p), ("d_track_ptr", C.c_void_p),
                ("d_track_hits", C.c_void_p)]


_lib = None


def load_library():
    """Load libetx.so (in-tree).  Raises if it is missing — the product has no other path."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise FileNotFoundError(f"{_LIB_PATH} not built: run `python -m paper_2508_07423_b200.build` "
                                    "(there is no CPU or PyTorch fallback)")
        lib = C.CDLL(_LIB_PATH)
        lib.etx_weight_count.restype = C.c_size_t
        lib.etx_weight_count.argtypes = [C.POINTER(ModelDesc)]
        lib.etx_create.restype = C.c_int
        lib.etx_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(ModelDesc), C.c_void_p, C.c_size_t, C.c_int]
        lib.etx_destroy.restype = C.c_int
        lib.etx_destroy.argtypes = [C.c_void_p]
        lib.etx_last_error.restype = C.c_char_p
        lib.etx_last_error.argtypes = [C.c_void_p]
        lib.etx_workspace_bytes.restype = C.c_size_t
        lib.etx_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int]
        lib.etx_set_workspace.restype = C.c_int
        lib.etx_set_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        lib.etx_embed.restype = C.c_int
        lib.etx_embed.argtypes = [C.c_void_p, C.POINTER(Batch), C.c_void_p, C.c_void_p]
        lib.etx_embed_bf16.restype = C.c_int
        lib.etx_embed_bf16.argtypes = [C.c_void_p, C.POINTER(Batch), C.c_void_p, C.c_void_p]
        lib.etx_embed_int8.restype = C.c_int
        lib.etx_embed_int8.argtypes = [C.c_void_p, C.POINTER(Batch), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        lib.etx_build_graph.restype = C.c_int
        lib.etx_build_graph.argtypes = [C.c_void_p, C.POINTER(Batch), C.c_void_p, C.c_float, C.c_int32,
                                        C.c_int32, C.POINTER(Graph), C.c_void_p]
        lib.etx_gnn_forward.restype = C.c_int
        lib.etx_gnn_forward.argtypes = [C.c_void_p, C.POINTER(Batch), C.POINTER(Graph), C.c_void_p,
                                        C.c_void_p, C.c_void_p]
        lib.etx_edge_scores.restype = C.c_int
        lib.etx_edge_scores.argtypes = [C.c_void_p, C.POINTER(Graph), C.c_void_p, C.c_void_p, C.c_void_p]
        lib.etx_infer_host.restype = C.c_int
        lib.etx_infer_host.argtypes = [C.c_void_p, C.POINTER(BatchHost), C.c_float, C.c_int32, C.c_int64,
                                       C.POINTER(C.c_int64), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.etx_launch_count.restype = C.c_int64
        lib.etx_launch_count.argtypes = [C.c_void_p]
        lib.etx_measure_alu_peak.restype = C.c_int
        lib.etx_measure_alu_peak.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double)]
        lib.etx_build_tracks.restype = C.c_int
        lib.etx_build_tracks.argtypes = [C.c_void_p, C.POINTER(Batch), C.POINTER(Graph), C.c_void_p, C.c_float,
                                         C.c_void_p, C.c_void_p]
        lib.etx_build_triplets.restype = C.c_int
        lib.etx_build_triplets.argtypes = [C.c_void_p, C.POINTER(Batch), C.POINTER(Graph), C.c_void_p, C.c_float,
                                           C.POINTER(Triplets), C.c_void_p]
        lib.etx_build_triplets_static.restype = C.c_int
        lib.etx_build_triplets_static.argtypes = lib.etx_build_triplets.argtypes
        lib.etx_triplet_weight_count.restype = C.c_size_t
        lib.etx_triplet_weight_count.argtypes = [C.POINTER(ModelDesc)]
        lib.etx_set_triplet_classifiers.restype = C.c_int
        lib.etx_set_triplet_classifiers.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        lib.etx_triplet_scores.restype = C.c_int
        lib.etx_triplet_scores.argtypes = [C.c_void_p, C.POINTER(Graph), C.c_void_p, C.POINTER(Triplets), C.c_void_p, C.c_void_p]
        lib.etx_triplet_tracks_workspace_bytes.restype = C.c_size_t
        lib.etx_triplet_tracks_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int64]
        lib.etx_build_tracks_from_triplets.restype = C.c_int
        lib.etx_build_tracks_from_triplets.argtypes = [C.c_void_p, C.POINTER(Batch), C.POINTER(Graph), C.c_void_p, C.c_float,
                                                       C.POINTER(Triplets), C.c_void_p, C.c_float, C.POINTER(Tracks), C.c_void_p]
        lib.etx_set_int8_ranges.restype = C.c_int
        lib.etx_set_int8_ranges.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        lib.etx_profile_enable.restype = C.c_int
        lib.etx_profile_enable.argtypes = [C.c_void_p, C.c_int]
        lib.etx_profile_read.restype = C.c_int
        lib.etx_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        _lib = lib
    return _lib


def make_desc(cfg: synth.Config, precision: Optional[int] = None) -> ModelDesc:
    d = ModelDesc()
    d.emb_n_layers = len(cfg.emb_widths) - 1
    for i, w in enumerate(cfg.emb_widths):
        d.emb_dims[i] = w
    d.gnn_hidden = cfg.gnn_hidden
    d.gnn_n_layers = cfg.gnn_mlp_hidden_layers + 1
    d.n_iter = cfg.n_iter
    d.precision = cfg.precision if precision is None else precision
    d.n_planes = synth.N_PLANES
    for i in range(5):
        d.norm_center[i] = synth.NORM_CENTER[i]
        d.norm_scale[i] = synth.NORM_SCALE[i]
    return d


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


class DeviceBatch:
    """Device-resident CSR batch (torch tensors) + the etx_batch struct that points at them."""

    def __init__(self, batch: Dict[str, np.ndarray], device: torch.device):
        self.n_events = len(batch["event_ptr"]) - 1
        self.n_hits = len(batch["r"])
        self.t = {k: torch.from_numpy(np.ascontiguousarray(batch[k])).to(device)
                  for k in ("event_ptr", "plane", "r", "phi", "z", "x", "y")}
        self.c = Batch(self.n_events, self.n_hits, *[_ptr(self.t[k]) for k in
                                                     ("event_ptr", "plane", "r", "phi", "z", "x", "y")])


class DeviceGraph:
    def __init__(self, n_hits: int, capacity: int, device: torch.device):
        i32 = dict(dtype=torch.int32, device=device)
        self.row_ptr = torch.empty(n_hits + 1, **i32)
        self.in_ptr = torch.empty(n_hits + 1, **i32)
        self.src = torch.empty(max(capacity, 1), **i32)
        self.dst = torch.empty(max(capacity, 1), **i32)
        self.in_perm = torch.empty(max(capacity, 1), **i32)
        self.c = Graph(capacity, 0, _ptr(self.row_ptr), _ptr(self.src), _ptr(self.dst), _ptr(self.in_ptr),
                       _ptr(self.in_perm))

    @property
    def n_edges(self) -> int:
        return int(self.c.n_edges)


class Etx:
    """One libetx context.  Methods mirror the C entry points one to one."""

    def __init__(self, desc: ModelDesc, weights: np.ndarray, device: int = 0):
        self.lib = load_library()
        self.desc = desc
        self.device = torch.device("cuda", device)
        w = np.ascontiguousarray(weights, dtype=np.float32)
        self.handle = C.c_void_p()
        st = self.lib.etx_create(C.byref(self.handle), C.byref(desc), w.ctypes.data_as(C.c_void_p), w.size, device)
        if st != ETX_OK:
            raise EtxError(st, self.lib.etx_last_error(None).decode())
        self._ws = None
        self._ws_bytes = 0

    def close(self):
        if getattr(self, "handle", None):
            self.lib.etx_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != ETX_OK:
            raise EtxError(st, self.lib.etx_last_error(self.handle).decode())

    @property
    def emb_dim(self) -> int:
        return int(self.desc.emb_dims[self.desc.emb_n_layers])

    @staticmethod
    def _stream() -> C.c_void_p:
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    # ---- workspace
    def workspace_bytes(self, n_events: int, n_hits: int, edge_capacity: int, with_host_path: bool = False) -> int:
        return int(self.lib.etx_workspace_bytes(self.handle, n_events, n_hits, edge_capacity, int(with_host_path)))

    def ensure_workspace(self, n_events: int, n_hits: int, edge_capacity: int, with_host_path: bool = False):
        need = self.workspace_bytes(n_events, n_hits, edge_capacity, with_host_path)
        if self._ws is None or self._ws_bytes < need:      # compare with what was REGISTERED, not the padded tensor
            self._ws = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
            self._check(self.lib.etx_set_workspace(self.handle, C.c_void_p(self._ws.data_ptr() + off), need))
            self._ws_bytes = need

    def set_workspace(self, nbytes: int):
        """Register a workspace of exactly ``nbytes`` (etx_set_workspace); etx_infer_host splits a batch that does
        not fit it into event ranges (include/etx.h)."""
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self._ws.data_ptr()) % 256
        self._check(self.lib.etx_set_workspace(self.handle, C.c_void_p(self._ws.data_ptr() + off), nbytes))
        self._ws_bytes = nbytes

    def launch_count(self) -> int:
        return int(self.lib.etx_launch_count(self.handle))

    def profile_enable(self, on: bool = True):
        self._check(self.lib.etx_profile_enable(self.handle, int(on)))

    def profile_read(self):
        """{class: (ms, launches)} accumulated since the last read."""
        n = len(KERNEL_CLASSES)
        ms = (C.c_double * n)()
        ln = (C.c_int64 * n)()
        self._check(self.lib.etx_profile_read(self.handle, ms, ln))
        return {k: (float(ms[i]), int(ln[i])) for i, k in enumerate(KERNEL_CLASSES)}

    # ---- the four path calls
    def etx_embed(self, batch: DeviceBatch, emb: Optional[torch.Tensor] = None) -> torch.Tensor:
        if emb is None:
            emb = torch.empty(batch.n_hits, self.emb_dim, dtype=torch.float32, device=self.device)
        self._check(self.lib.etx_embed(self.handle, C.byref(batch.c), _ptr(emb), self._stream()))
        return emb

    def etx_embed_bf16(self, batch: DeviceBatch, emb: Optional[torch.Tensor] = None) -> torch.Tensor:
        if emb is None:
            emb = torch.empty(batch.n_hits, self.emb_dim, dtype=torch.float32, device=self.device)
        self._check(self.lib.etx_embed_bf16(self.handle, C.byref(batch.c), _ptr(emb), self._stream()))
        return emb

    def etx_embed_int8(self, batch: DeviceBatch, act_alpha, emb: Optional[torch.Tensor] = None) -> torch.Tensor:
        if emb is None:
            emb = torch.empty(batch.n_hits, self.emb_dim, dtype=torch.float32, device=self.device)
        al = np.ascontiguousarray(act_alpha, dtype=np.float32)
        self._check(self.lib.etx_embed_int8(self.handle, C.byref(batch.c), al.ctypes.data_as(C.c_void_p), len(al),
                                            _ptr(emb), self._stream()))
        return emb

    def etx_build_graph(self, batch: DeviceBatch, emb: torch.Tensor, r2_max: float, max_plane_gap: int,
                        graph: DeviceGraph, k_max: int = 0) -> int:
        self._check(self.lib.etx_build_graph(self.handle, C.byref(batch.c), _ptr(emb), r2_max, max_plane_gap,
                                             k_max, C.byref(graph.c), self._stream()))
        return graph.n_edges

    def etx_gnn_forward(self, batch: DeviceBatch, graph: DeviceGraph, edge_enc: torch.Tensor,
                        hit_enc: Optional[torch.Tensor] = None) -> torch.Tensor:
        self._check(self.lib.etx_gnn_forward(self.handle, C.byref(batch.c), C.byref(graph.c), _ptr(edge_enc),
                                             _ptr(hit_enc), self._stream()))
        return edge_enc

    def etx_edge_scores(self, graph: DeviceGraph, edge_enc: torch.Tensor, scores: torch.Tensor) -> torch.Tensor:
        self._check(self.lib.etx_edge_scores(self.handle, C.byref(graph.c), _ptr(edge_enc), _ptr(scores),
                                             self._stream()))
        return scores

    def etx_build_tracks(self, batch: DeviceBatch, graph: DeviceGraph, scores: torch.Tensor, score_min: float,
                         labels: Optional[torch.Tensor] = None) -> torch.Tensor:
        if labels is None:
            labels = torch.empty(max(batch.n_hits, 1), dtype=torch.int32, device=self.device)
        self._check(self.lib.etx_build_tracks(self.handle, C.byref(batch.c), C.byref(graph.c), _ptr(scores),
                                              score_min, _ptr(labels), self._stream()))
        return labels

    def etx_build_triplets(self, batch: DeviceBatch, graph: DeviceGraph, scores: torch.Tensor, score_min: float,
                           capacity: Optional[int] = None) -> Dict[str, torch.Tensor]:
        """Rows of edge ids per kind ("articulation", "left_elbow", "right_elbow": int32 [n, 2] views of one
        buffer) and "ptr" [3, n_hits + 1].  capacity=None sizes the row buffer from a first counting call."""
        ptr = torch.empty(3, batch.n_hits + 1, dtype=torch.int32, device=self.device)
        t = Triplets()
        t.d_ptr = ptr.data_ptr()

        def call(cap):
            rows = torch.empty(2, max(cap, 1), dtype=torch.int32, device=self.device)
            t.capacity, t.d_first, t.d_second = cap, rows[0].data_ptr(), rows[1].data_ptr()
            st = self.lib.etx_build_triplets(self.handle, C.byref(batch.c), C.byref(graph.c), _ptr(scores), score_min,
                                             C.byref(t), self._stream())
            return st, rows

        st, rows = call(0 if capacity is None else capacity)
        if st == ETX_ERR_CAPACITY and capacity is None and min(t.n) >= 0:
            st, rows = call(sum(t.n))
        self._check(st)
        n = [int(x) for x in t.n]
        o = [0, n[0], n[0] + n[1], n[0] + n[1] + n[2]]
        out = {"ptr": ptr, "c": t, "rows": rows}          # "c": the etx_triplets struct (points into "ptr" / "rows")
        for k, name in enumerate(("articulation", "left_elbow", "right_elbow")):
            out[name] = torch.stack([rows[0, o[k]:o[k + 1]], rows[1, o[k]:o[k + 1]]], dim=1)
        return out

    def etx_build_triplets_static(self, batch: DeviceBatch, graph: DeviceGraph, scores: torch.Tensor, score_min: float,
                                  ptr: torch.Tensor, rows: torch.Tensor):
        """etx_build_triplets without any allocation (include/etx.h): the caller passes the outputs -- ptr int32
        [3, n_hits + 1] and rows int32 [2, capacity], both contiguous on the device -- and gets the three counts back.
        rows[0, :sum(n)] / rows[1, :sum(n)] are the first / second edge ids, sections in the order of etx_build_triplets."""
        assert ptr.dtype == torch.int32 and ptr.is_contiguous() and ptr.numel() == 3 * (batch.n_hits + 1)
        assert rows.dtype == torch.int32 and rows.is_contiguous() and rows.dim() == 2 and rows.shape[0] == 2
        t = Triplets()
        t.d_ptr = ptr.data_ptr()
        t.capacity, t.d_first, t.d_second = rows.shape[1], rows[0].data_ptr(), rows[1].data_ptr()
        self._check(self.lib.etx_build_triplets_static(self.handle, C.byref(batch.c), C.byref(graph.c), _ptr(scores),
                                                       score_min, C.byref(t), self._stream()))
        return [int(x) for x in t.n]

    # ---- next row: INT8 GNN (context created with precision ETX_PREC_INT8 = 4)
    def etx_set_int8_ranges(self, alpha: Dict[str, list]):
        """alpha: MLP name -> per-layer input ranges (synth.int8_gnn_alpha); flattened in the library's MLP order."""
        n_iter = int(self.desc.n_iter)
        names = ["node_enc", "edge_enc"] + [f"{n}_{k}" for k in range(n_iter) for n in ("node_net", "edge_net")] + ["cls"]
        flat = np.ascontiguousarray(np.concatenate([np.asarray(alpha[n], np.float32) for n in names]))
        self._check(self.lib.etx_set_int8_ranges(self.handle, flat.ctypes.data_as(C.c_void_p), flat.size))

    # ---- next row: triplet classifiers and track building from triplets
    def etx_set_triplet_classifiers(self, weights: np.ndarray):
        w = np.ascontiguousarray(weights, dtype=np.float32)
        self._check(self.lib.etx_set_triplet_classifiers(self.handle, w.ctypes.data_as(C.c_void_p), w.size))

    def etx_triplet_scores(self, graph: DeviceGraph, edge_enc: torch.Tensor, trip: Dict[str, torch.Tensor]) -> Dict[str, torch.Tensor]:
        """Scores per kind (views of one buffer under "all", row for row with the triplet rows)."""
        n = [int(x) for x in trip["c"].n]
        s = torch.empty(max(sum(n), 1), dtype=torch.float32, device=self.device)
        self._check(self.lib.etx_triplet_scores(self.handle, C.byref(graph.c), _ptr(edge_enc), C.byref(trip["c"]), _ptr(s),
                                                self._stream()))
        o = [0, n[0], n[0] + n[1], sum(n)]
        out = {"all": s}
        for k, name in enumerate(("articulation", "left_elbow", "right_elbow")):
            out[name] = s[o[k]:o[k + 1]]
        return out

    def etx_build_tracks_from_triplets(self, batch: DeviceBatch, graph: DeviceGraph, scores: torch.Tensor, score_min: float,
                                       trip: Dict[str, torch.Tensor], trip_scores: torch.Tensor, trip_min: float) -> Dict[str, torch.Tensor]:
        """edge_set [E], joins [J, 2], track_ptr [T + 1], track_hits; sized from a first counting call.  Uses (and
        clobbers) the context workspace."""
        E = graph.n_edges
        need = int(self.lib.etx_triplet_tracks_workspace_bytes(self.handle, batch.n_hits, E, int(trip["c"].n[0])))
        if self._ws is None or self._ws_bytes < need:
            self.set_workspace(need)
        i32 = dict(dtype=torch.int32, device=self.device)
        edge_set = torch.empty(max(E, 1), **i32)
        tk = Tracks()
        tk.d_edge_set = edge_set.data_ptr()

        def call(nj, nt, nh):
            joins = torch.empty(max(nj, 1), 2, **i32)
            tptr = torch.empty(nt + 1, **i32)
            thits = torch.empty(max(nh, 1), **i32)
            tk.join_capacity, tk.track_capacity, tk.hit_capacity = nj, nt, nh
            tk.d_joins, tk.d_track_ptr, tk.d_track_hits = joins.data_ptr(), tptr.data_ptr(), thits.data_ptr()
            st = self.lib.etx_build_tracks_from_triplets(self.handle, C.byref(batch.c), C.byref(graph.c), _ptr(scores), score_min,
                                                         C.byref(trip["c"]), _ptr(trip_scores), trip_min, C.byref(tk), self._stream())
            return st, joins, tptr, thits

        st, joins, tptr, thits = call(0, 0, 0)
        if st == ETX_ERR_CAPACITY:
            st, joins, tptr, thits = call(int(tk.n_joins), int(tk.n_tracks), int(tk.n_track_hits))
        self._check(st)
        return {"edge_set": edge_set[:E], "joins": joins[:int(tk.n_joins)], "track_ptr": tptr[:int(tk.n_tracks) + 1],
                "track_hits": thits[:int(tk.n_track_hits)], "n_plain": int(tk.n_plain)}

    # ---- whole path with host buffers (pinned torch tensors or numpy arrays)
    def etx_infer_host(self, host: Dict[str, torch.Tensor], r2_max: float, max_plane_gap: int,
                       edge_capacity: int, out_src: Optional[torch.Tensor], out_dst: Optional[torch.Tensor],
                       out_scores: torch.Tensor) -> int:
        hb = BatchHost(len(host["event_ptr"]) - 1, len(host["r"]),
                       *[C.c_void_p(host[k].data_ptr()) for k in ("event_ptr", "plane", "r", "phi", "z", "x", "y")])
        n = C.c_int64(0)
        st = self.lib.etx_infer_host(self.handle, C.byref(hb), r2_max, max_plane_gap, edge_capacity, C.byref(n),
                                     None if out_src is None else C.c_void_p(out_src.data_ptr()),
                                     None if out_dst is None else C.c_void_p(out_dst.data_ptr()),
                                     C.c_void_p(out_scores.data_ptr()), self._stream())
        self._check(st)
        return int(n.value)


def pinned_host_batch(batch: Dict[str, np.ndarray]) -> Dict[str, torch.Tensor]:
    return {k: torch.from_numpy(np.ascontiguousarray(batch[k])).pin_memory()
            for k in ("event_ptr", "plane", "r", "phi", "z", "x", "y")}


def run_path(etx: Etx, batch: Dict[str, np.ndarray], r2_max: float, max_plane_gap: int,
             edge_capacity: Optional[int] = None, graph_override=None, embed: str = "etx_embed") -> Dict[str, np.ndarray]:
    """Convenience for tests: the four calls in order on device-resident inputs, results to numpy.  `embed` names the
    embedding call (etx_embed, or the report-only etx_embed_bf16)."""
    dev = etx.device
    db = DeviceBatch(batch, dev)
    cap = edge_capacity if edge_capacity is not None else max(64 * db.n_hits, 1024)
    etx.ensure_workspace(db.n_events, db.n_hits, cap)
    emb = getattr(etx, embed)(db)
    g = DeviceGraph(db.n_hits, cap, dev)
    E = etx.etx_build_graph(db, emb, r2_max, max_plane_gap, g)
    H = int(etx.desc.gnn_hidden)
    e = torch.empty(max(E, 1), H, dtype=torch.float32, device=dev)
    h = torch.empty(max(db.n_hits, 1), H, dtype=torch.float32, device=dev)
    s = torch.empty(max(E, 1), dtype=torch.float32, device=dev)
    etx.etx_gnn_forward(db, g, e, h)
    etx.etx_edge_scores(g, e, s)
    torch.cuda.synchronize()
    return {"emb": emb.cpu().numpy(), "src": g.src[:E].cpu().numpy(), "dst": g.dst[:E].cpu().numpy(),
            "row_ptr": g.row_ptr.cpu().numpy(), "in_ptr": g.in_ptr.cpu().numpy(),
            "in_perm": g.in_perm[:E].cpu().numpy(), "h": h[:db.n_hits].cpu().numpy(), "e": e[:E].cpu().numpy(),
            "scores": s[:E].cpu().numpy()}
