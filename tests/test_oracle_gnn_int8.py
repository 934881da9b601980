"""Pins of the quantised-GNN oracle (GNN part; Eqs. 4.31-4.33).  No GPU."""
import numpy as np
import pytest

from conftest import layout_dict
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def test_step_by_step_forward_equals_the_compiled_hot_path_oracle(c0, c0_oracle):
    """The Python step-by-step forward (the skeleton the quantised forward shares) with the fp32 MLP and the
    double-accumulating scatter IS the hot path: bitwise equal to orc_gnn_forward / orc_edge_scores."""
    cfg, batch, blob = c0
    lay = layout_dict(cfg)
    h, e, logit = orc.gnn_forward_steps(c0_oracle["f_node"], c0_oracle["src"], c0_oracle["dst"], cfg.n_iter,
                                        lambda n, x: orc.mlp(x, lay[n][0], blob, lay[n][1]), orc.scatter)
    np.testing.assert_array_equal(h, c0_oracle["h"])
    np.testing.assert_array_equal(e, c0_oracle["e"])
    np.testing.assert_array_equal(logit, c0_oracle["logits"])


def test_fp32_scatter_is_the_sequential_sum(c0_oracle):
    src, dst, e = c0_oracle["src"], c0_oracle["dst"], c0_oracle["e"]
    n, H = 239, e.shape[1]
    m = orc.scatter_f32(n, src, dst, e)
    want = np.zeros((n, 2 * H), np.float32)
    np.add.at(want[:, :H], src, e)                      # numpy: unbuffered, in index order, fp32
    np.add.at(want[:, H:], dst, e)
    np.testing.assert_array_equal(m, want)
    np.testing.assert_allclose(m, orc.scatter(n, src, dst, e), rtol=0, atol=1e-5)     # the double-accumulated one
    # a sum whose fp32 order matters: 1e8 + 1 + 1 + ... loses the ones one by one, a double sum would not
    ee = np.array([[1e8], [1.0], [1.0], [-1e8]], np.float32)
    m = orc.scatter_f32(2, np.zeros(4, np.int32), np.ones(4, np.int32), ee)
    assert m[0, 0] == 0.0 and m[1, 1] == 0.0 and orc.scatter(2, np.zeros(4, np.int32), np.ones(4, np.int32), ee)[0, 0] == 2.0


def test_integer_valued_network_is_computed_exactly():
    """Weights in {-1, 0, 1} (S_w = 1/127, codes +-127) and ranges alpha = 127 (S_a = 1, codes = values): every
    quantisation is exact while activations are integers <= 127, so the quantised GNN must equal plain int64 arithmetic."""
    rng = np.random.default_rng(5)
    H, L, n_iter, n, E = 4, 3, 2, 6, 7
    names = orc.gnn_mlp_names(n_iter)
    dims = {"node_enc": (3, H, H, H), "edge_enc": (2 * H, H, H, H), "cls": (H, H, H, 1)}
    for k in range(n_iter):
        dims[f"node_net_{k}"] = dims[f"edge_net_{k}"] = (3 * H, H, H, H)
    blob, lay, off = [], {}, 0
    for nm in names:
        lay[nm] = (dims[nm], off)
        for l in range(L):
            fi, fo = dims[nm][l], dims[nm][l + 1]
            W = rng.integers(-1, 2, size=(fo, fi)).astype(np.float32)
            W[0, 0] = 1.0                               # max |W| = 1 exactly
            W *= (rng.random((fo, fi)) < 0.25)          # sparse: keeps the activations on the grid
            W[0, 0] = 1.0
            b = rng.integers(-1, 2, size=fo).astype(np.float32)
            blob += [W.ravel(), b]
            off += fi * fo + fo
    blob = np.concatenate(blob).astype(np.float32)
    f = rng.integers(-2, 3, size=(n, 3)).astype(np.float32)
    src = np.sort(rng.integers(0, n // 2, E)).astype(np.int32)
    dst = rng.integers(n // 2, n, E).astype(np.int32)
    al = {nm: [127.0] * L for nm in names}
    h, e, logit, s = orc.gnn_forward_int8(f, src, dst, n_iter, blob, lay, al)

    def int_mlp(nm, x):
        d, o = lay[nm]
        a = x.astype(np.int64)
        for l in range(L):
            W = blob[o:o + d[l] * d[l + 1]].reshape(d[l + 1], d[l]).astype(np.int64)
            b = blob[o + d[l] * d[l + 1]:o + d[l] * d[l + 1] + d[l + 1]].astype(np.int64)
            assert np.abs(a).max() <= 127, "test construction: every layer INPUT must sit on the INT8 grid"
            a = a @ W.T + b
            if l < L - 1:
                a = np.maximum(a, 0)
            o += d[l] * d[l + 1] + d[l + 1]
        return a

    def int_scatter(nn, s_, d_, ee):
        m = np.zeros((nn, 2 * H), np.int64)
        np.add.at(m[:, :H], s_, ee)
        np.add.at(m[:, H:], d_, ee)
        return m

    hi = int_mlp("node_enc", f)
    ei = int_mlp("edge_enc", np.concatenate([hi[src], hi[dst]], 1))
    for k in range(n_iter):
        mi = int_scatter(n, src, dst, ei)
        hi = hi + int_mlp(f"node_net_{k}", np.concatenate([hi, mi], 1))
        ei = ei + int_mlp(f"edge_net_{k}", np.concatenate([hi[src], hi[dst], ei], 1))
    li = int_mlp("cls", ei)[:, 0]
    np.testing.assert_array_equal(h, hi.astype(np.float32))
    np.testing.assert_array_equal(e, ei.astype(np.float32))
    np.testing.assert_array_equal(logit, li.astype(np.float32))
    np.testing.assert_allclose(s, 1.0 / (1.0 + np.exp(-li.astype(np.float64))), rtol=0, atol=1e-7)
    assert np.abs(e).max() > 1                                   # not a degenerate all-zero network


def test_calibrated_is_close_to_fp32_and_wrong_ranges_are_worse(c0, c0_oracle):
    cfg, batch, blob = c0
    lay = layout_dict(cfg)
    fn, src, dst = c0_oracle["f_node"], c0_oracle["src"], c0_oracle["dst"]
    al = orc.gnn_int8_calibration(fn, src, dst, cfg.n_iter, blob, lay)
    assert sorted(al) == sorted(orc.gnn_mlp_names(cfg.n_iter)) and all(len(v) == 3 and min(v) > 0 for v in al.values())
    h, e, logit, s = orc.gnn_forward_int8(fn, src, dst, cfg.n_iter, blob, lay, al)
    err = np.abs(s.astype(np.float64) - c0_oracle["scores"]).max()
    wide = {k: [20.0 * a for a in v] for k, v in al.items()}
    err_wide = np.abs(orc.gnn_forward_int8(fn, src, dst, cfg.n_iter, blob, lay, wide)[3].astype(np.float64) - c0_oracle["scores"]).max()
    narrow = {k: [0.05 * a for a in v] for k, v in al.items()}
    err_narrow = np.abs(orc.gnn_forward_int8(fn, src, dst, cfg.n_iter, blob, lay, narrow)[3].astype(np.float64) - c0_oracle["scores"]).max()
    print(f"int8 GNN on c0: max |score - fp32 oracle| calibrated {err:.3g}, ranges x20 {err_wide:.3g}, ranges x0.05 {err_narrow:.3g}")
    assert err < 0.05 and err_wide > 2 * err and err_narrow > 2 * err
    # the node encoder's first layer is the hot path's fp32 layer: with every OTHER weight zero the state is exactly its ReLU
    z = blob.copy()
    d, o = lay["node_enc"]
    z[o + d[0] * d[1] + d[1]:] = 0.0
    h0 = orc.gnn_forward_int8(fn, src, dst, 0, z, lay, al)[0]
    assert np.all(h0 == 0.0)                                     # layers 2.. are zero -> h0 = their (zero) output
