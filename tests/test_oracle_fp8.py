"""Pins of the oracle's FP8 (e4m3) quantiser and MLP (next row NEXT-3; the symmetric per-tensor scheme of Eqs. 4.31-4.33
P:1469-1481 on the e4m3 grid, DESIGN reading Q26).  No GPU."""
import numpy as np
import pytest
import torch

from conftest import layout_dict
from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def test_e4m3_grid_facts():
    # the format itself: largest finite value 448 = 1.75 * 2^8, smallest normal 2^-6, subnormal spacing 2^-9, 3 mantissa bits
    x = np.array([448.0, 449.0, 1e6, -1e6, 2.0 ** -6, 2.0 ** -9, 2.0 ** -10, 0.75 * 2.0 ** -9, 0.0, -0.0], np.float32)
    v, S = orc.quantize_fp8(x, 448.0)                       # alpha = 448 -> S = 1: the values are the e4m3 roundings of x
    assert S == 1.0
    assert v.tolist() == [448.0, 448.0, 448.0, -448.0, 2.0 ** -6, 2.0 ** -9, 0.0, 2.0 ** -9, 0.0, 0.0]
    # ties go to the even mantissa: 1.0625 lies between 1.0 (000) and 1.125 (001); 1.1875 between 1.125 (001) and 1.25 (010)
    v, _ = orc.quantize_fp8(np.array([1.0625, 1.1875, -1.0625, 240.0, 232.0], np.float32), 448.0)
    assert v.tolist() == [1.0, 1.25, -1.0, 240.0, 224.0]    # 232 = midpoint of 224 (1.110) and 240 (1.111) -> 224
    # exactly 2 x 8 x 15 + 7 (subnormals) + zero = 127 distinct non-negative values up to 448
    grid, _ = orc.quantize_fp8(np.linspace(0.0, 448.0, 2_000_001, dtype=np.float32), 448.0)
    assert len(np.unique(grid)) == 127


def test_rounding_equals_the_library_cast():
    # torch's float8_e4m3fn cast rounds to nearest even; it does not saturate, so the comparison clips first
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.normal(size=200_000) * 10.0 ** rng.uniform(-4, 3, 200_000),
                        np.linspace(-460.0, 460.0, 100_001), np.arange(-2048, 2049) * 2.0 ** -11]).astype(np.float32)
    v, _ = orc.quantize_fp8(x, 448.0)
    ref = torch.from_numpy(np.clip(x, -448.0, 448.0)).to(torch.float8_e4m3fn).float().numpy()
    np.testing.assert_array_equal(v, ref)


def test_scale_maps_the_range_to_448_and_error_bound():
    rng = np.random.default_rng(1)
    alpha = 3.7
    x = rng.uniform(-alpha, alpha, 20000).astype(np.float32)
    v, S = orc.quantize_fp8(x, alpha)
    assert S == np.float32(np.float32(alpha) / np.float32(448.0))
    top, _ = orc.quantize_fp8(np.array([alpha, -alpha, 10 * alpha], np.float32), alpha)
    assert top.tolist() == [448.0, -448.0, 448.0]           # alpha -> the largest value (as P:1487 maps it to 127); clipping beyond
    # relative error <= 2^-4 for normal values (3 mantissa bits), absolute error <= S 2^-10 in the subnormal range
    err = np.abs(x.astype(np.float64) - S * v.astype(np.float64))
    assert np.all(err <= np.maximum(np.abs(x) * 2.0 ** -4, S * 2.0 ** -10) * (1 + 1e-5))
    order = np.argsort(x)
    assert np.all(np.diff(v[order]) >= 0)                   # monotone


def test_exact_on_grid_values_equals_float64_linear_layer():
    # inputs and weights that ARE e4m3 values times power-of-two scales: quantisation is the identity, every product and sum exact
    rng = np.random.default_rng(4)
    fi, fo, n = 16, 8, 50
    grid, _ = orc.quantize_fp8(np.linspace(-448.0, 448.0, 4001, dtype=np.float32), 448.0)
    grid = np.unique(grid)
    xq = rng.choice(grid, size=(n, fi)); xq[0, 0] = 448.0
    Wq = rng.choice(grid, size=(fo, fi)); Wq[0, 0] = 448.0
    x = (xq * 2.0 ** -7).astype(np.float32)
    W = (Wq * 2.0 ** -11).astype(np.float32)
    b = (rng.integers(-8, 9, size=fo) * 2.0 ** -4).astype(np.float32)
    blob = np.concatenate([W.ravel(), b])
    out = orc.mlp_fp8(x, (fi, fo), blob, 0, [448.0 * 2.0 ** -7])
    ref = torch.nn.functional.linear(torch.from_numpy(x).double(), torch.from_numpy(W).double(), torch.from_numpy(b).double())
    # exact sum, one rounding to fp32, exact power-of-two de-quantisation, + b: compare with the float64 layer rounded once
    np.testing.assert_allclose(out.astype(np.float64), ref.numpy(), rtol=2.0 ** -23, atol=0)


def test_two_layers_by_hand():
    # 2 -> 2 -> 1; alpha chosen so that S is a power of two and every value can be followed by hand
    W1 = np.array([[448.0, -224.0], [112.0, 448.0]], np.float32) * np.float32(2.0 ** -9)    # S_w1 = 2^-9, values on the grid
    b1 = np.array([0.25, -0.5], np.float32)
    W2 = np.array([[448.0, 208.0]], np.float32) * np.float32(2.0 ** -8)                     # S_w2 = 2^-8
    b2 = np.array([0.125], np.float32)
    blob = np.concatenate([W1.ravel(), b1, W2.ravel(), b2])
    a1, a2 = 448.0 * 2.0 ** -8, 448.0 * 2.0 ** -7                                           # S_a1 = 2^-8, S_a2 = 2^-7
    x = np.array([[1.0, 0.5], [0.26, -1.0]], np.float32)
    # row 0: x/S_a1 = (256, 128) on the grid.  layer 1: (448*256 - 224*128, 112*256 + 448*128) * 2^-17 + b = (0.65625 + 0.25, 0.65625 - 0.5)
    #        -> ReLU -> (0.90625, 0.15625); /S_a2 = (116, 20): 116 lies between 112 (1.110 * 2^6) and 120 -> tie -> 112 (even); 20 is on the grid
    #        layer 2: (448*112 + 208*20) * 2^-15 + 0.125 = 54336 / 32768 + 0.125 = 1.783203125
    # row 1: 0.26/S_a1 = 66.56 -> grid spacing 8 in [64, 128) -> 64;  -1.0/S_a1 = -256
    #        layer 1: (448*64 + 224*256, 112*64 - 448*256) * 2^-17 + b = (0.65625 + 0.25, -0.8203125 - 0.5) -> ReLU -> (0.90625, 0)
    #        layer 2: 448*112 * 2^-15 + 0.125 = 1.65625
    out = orc.mlp_fp8(x, (2, 2, 1), blob, 0, [a1, a2])
    assert out[:, 0].tolist() == [1.783203125, 1.65625]


def test_calibrated_ranges_track_fp32_and_wrong_ranges_do_not(c0, c0_oracle):
    cfg, batch, blob = c0
    lay = layout_dict(cfg)
    alpha = synth.int8_gnn_alpha(cfg)
    src, dst = c0_oracle["src"], c0_oracle["dst"]
    h, e, logit, s = orc.gnn_forward_fp8(c0_oracle["f_node"], src, dst, cfg.n_iter, blob, lay, alpha)
    ref = c0_oracle["scores"].astype(np.float64)
    d_cal = np.abs(s.astype(np.float64) - ref)
    assert h.shape == c0_oracle["h"].shape and e.shape == c0_oracle["e"].shape
    assert 0 < d_cal.max() < 0.25 and np.median(d_cal) < 0.05        # 3 mantissa bits per operand: close, not equal
    # FP8 keeps relative precision across magnitudes where INT8 keeps absolute precision: different results
    _, _, _, s8 = orc.gnn_forward_int8(c0_oracle["f_node"], src, dst, cfg.n_iter, blob, lay, alpha)
    assert np.abs(s.astype(np.float64) - s8.astype(np.float64)).max() > 1e-4
    # ranges 64x too narrow saturate most activations at 448 S: clearly worse
    narrow = {k: [a / 64.0 for a in v] for k, v in alpha.items()}
    _, _, _, s_bad = orc.gnn_forward_fp8(c0_oracle["f_node"], src, dst, cfg.n_iter, blob, lay, narrow)
    assert np.median(np.abs(s_bad.astype(np.float64) - ref)) > 2 * np.median(d_cal)
