"""Pins for the oracle's INT8 embedding MLP (next row NEXT-3, embedding part: Eqs. 4.31-4.33 P:1469-1481,
static PTQ P:1487-1499, INT8 embedding P:2723-2742)."""
import numpy as np
import torch

from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def test_scale_and_codes_of_the_thesis_example():
    # "For the values shown ... the scale will have to be S = 10.8/127": alpha maps to the highest INT8 value
    x = np.array([10.8, -10.8, 0.0, 5.4, 100.0, -100.0, 10.8 / 127 * 3.0, 10.8 / 127 * 2.5, 10.8 / 127 * 3.5], np.float32)
    codes, S = orc.quantize(x, 10.8)
    assert S == np.float32(np.float32(10.8) / np.float32(127.0))
    # Eq. 4.33: alpha -> +-127, values outside the interval are clipped, in-grid values keep their integer
    assert codes[:3].tolist() == [127, -127, 0]
    assert codes[3] in (63, 64)                                  # 63.5 up to the rounding of 5.4f / S
    assert codes[4:6].tolist() == [127, -127]
    assert codes[6] == 3
    assert codes[7] in (2, 3) and codes[8] in (3, 4)             # half-way cases: nearest integer either way


def test_quantisation_error_bound_and_monotonicity():
    rng = np.random.default_rng(0)
    alpha = 3.0
    x = rng.uniform(-alpha, alpha, 5000).astype(np.float32)
    codes, S = orc.quantize(x, alpha)
    assert np.abs(x - S * codes.astype(np.float64)).max() <= 0.5 * S * (1 + 1e-5)     # Eq. 4.31: x = S x_q within S/2
    order = np.argsort(x)
    assert np.all(np.diff(codes[order].astype(int)) >= 0)                             # monotone
    assert codes.min() >= -127 and codes.max() <= 127


def _grid_net(rng, dims):
    """Weights, biases and inputs that sit exactly on their INT8 grids (max |.| = 127 steps): quantisation is then
    the identity and the INT8 MLP must equal the exact MLP."""
    blob, alphas = [], []
    for fi, fo in zip(dims[:-1], dims[1:]):
        Wq = rng.integers(-127, 128, size=(fo, fi))
        Wq[0, 0] = 127                                           # pins max|W| -> S_w = step exactly
        blob += [(Wq * 2.0 ** -9).astype(np.float32).ravel(), (rng.integers(-8, 9, size=fo) * 2.0 ** -4).astype(np.float32)]
    return np.concatenate(blob)


def test_exact_on_grid_values_equals_float64_linear_layer():
    # one layer: x = S_a * integers, W = S_w * integers with power-of-two steps -> every product and sum is exact
    rng = np.random.default_rng(4)
    fi, fo, n = 16, 8, 50
    step_a, step_w = 2.0 ** -6, 2.0 ** -9
    xq = rng.integers(-127, 128, size=(n, fi)); xq[0, 0] = 127
    x = (xq * step_a).astype(np.float32)
    blob = _grid_net(rng, (fi, fo))
    W = blob[:fi * fo].reshape(fo, fi); b = blob[fi * fo:]
    out = orc.mlp_int8(x, (fi, fo), blob, 0, [127 * step_a])
    ref = torch.nn.functional.linear(torch.from_numpy(x).double(), torch.from_numpy(W).double(), torch.from_numpy(b).double())
    np.testing.assert_array_equal(out.astype(np.float64), ref.numpy())              # exact: all values are dyadic


def test_two_layers_relu_and_requantisation_by_hand():
    # 2 -> 2 -> 1, numbers chosen so every code can be checked by hand
    #   layer 1: W = [[1.27, 0], [0, -1.27]] (S_w = 0.01, codes +-127), b = [0, 0.5]; input alpha 2.54 (S_a = 0.02)
    #   x = [1.0, 0.3] -> codes [50, 15] -> sums [6350, -1905] * 2e-4 = [1.27, -0.381] + b = [1.27, 0.119]; ReLU keeps both
    #   layer 2: W = [[0.635, -1.27]] (S_w = 0.01, codes [64 (63.5 -> even 64), -127]), b = [0.1]; input alpha 1.27 (S_a = 0.01)
    #   a = [1.27, 0.119] -> codes [127, 12] -> sum 127*64 - 12*127 = 6604 * 1e-4 = 0.6604 + 0.1 = 0.7604
    blob = np.array([1.27, 0.0, 0.0, -1.27, 0.0, 0.5, 0.635, -1.27, 0.1], np.float32)
    out = orc.mlp_int8(np.array([[1.0, 0.3]], np.float32), (2, 2, 1), blob, 0, [2.54, 1.27])
    assert abs(float(out[0, 0]) - 0.7604) < 2e-6
    # the second input drives the hidden unit negative -> ReLU -> code 0:  x = [0, 2.0]: unit 2 = -1.27*2.0+0.5 < 0
    out = orc.mlp_int8(np.array([[0.0, 2.0]], np.float32), (2, 2, 1), blob, 0, [2.54, 1.27])
    assert abs(float(out[0, 0]) - 0.1) < 2e-6                                         # both hidden values 0 -> bias only


def test_int8_embedding_tracks_the_fp32_embedding(c1):
    # the calibrated INT8 embedding is an APPROXIMATION of the fp32 one (the thesis: 5-10 % more edges): its
    # error must be of the order of the quantisation steps, not more
    cfg, b, blob = c1
    spec = synth.model_layout(cfg)[0]
    fe, _ = orc.features(b, synth.NORM_CENTER, synth.NORM_SCALE)
    alphas = orc.int8_calibration(fe, spec.dims, blob, spec.offset)
    assert len(alphas) == len(spec.dims) - 1 and np.all(alphas > 0)
    e32 = orc.mlp(fe, spec.dims, blob, spec.offset)
    e8 = orc.mlp_int8(fe, spec.dims, blob, spec.offset, alphas)
    rel = np.abs(e8 - e32).max() / np.abs(e32).max()
    assert 1e-4 < rel < 0.15, rel
    # uncalibrated (a range 20x too wide wastes the code space): clearly worse
    e8_bad = orc.mlp_int8(fe, spec.dims, blob, spec.offset, alphas * 20)
    assert np.abs(e8_bad - e32).max() > 3 * np.abs(e8 - e32).max()
