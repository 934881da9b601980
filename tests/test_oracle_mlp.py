"""Pins for the oracle's MLP and features (Eqs. 4.24-4.27)."""
import numpy as np
import torch
import torch.nn.functional as F

from oracle import etx_oracle as orc
from paper_2508_07423_b200 import synth


def _blob(layers):
    """layers: [(W[out,in], b[out])] -> flat blob in the [W, b] per layer format."""
    return np.concatenate([np.concatenate([W.ravel(), b.ravel()]) for W, b in layers]).astype(np.float32)


def test_identity_weights_give_relu():
    # special case W = I, b = 0: hidden layer returns ReLU(x), output layer returns its input
    x = np.linspace(-2, 2, 40, dtype=np.float32).reshape(5, 8)
    eye, z = np.eye(8, dtype=np.float32), np.zeros(8, np.float32)
    out = orc.mlp(x, (8, 8, 8), _blob([(eye, z), (eye, z)]), 0)
    np.testing.assert_array_equal(out, np.maximum(x, 0))
    out1 = orc.mlp(x, (8, 8), _blob([(eye, z)]), 0)          # single (output) layer: linear, no ReLU
    np.testing.assert_array_equal(out1, x)


def test_zero_weights_give_bias_and_last_layer_is_linear():
    x = np.random.default_rng(0).normal(size=(7, 5)).astype(np.float32)
    b1 = np.array([0.5, -0.25, 1.0], np.float32)
    b2 = np.array([-3.0, 2.0], np.float32)
    out = orc.mlp(x, (5, 3, 2), _blob([(np.zeros((3, 5)), b1), (np.zeros((2, 3)), b2)]), 0)
    np.testing.assert_array_equal(out, np.tile(b2, (7, 1)))   # negative output survives: no ReLU at the end
    W2 = np.array([[1, 1, 1], [1, -1, 2]], np.float32)
    out = orc.mlp(x, (5, 3, 2), _blob([(np.zeros((3, 5)), b1), (W2, b2)]), 0)
    hid = np.maximum(b1, 0)                                    # -0.25 is clipped by the hidden ReLU
    np.testing.assert_allclose(out, np.tile(W2 @ hid + b2, (7, 1)), rtol=1e-7)


def test_transposed_operand_would_fail():
    # a non-square, asymmetric layer: W[out][in] row-major; hand-computed
    W = np.array([[1, 2, 3], [4, 5, 6]], np.float32)           # out=2, in=3
    x = np.array([[1, 0, -1]], np.float32)
    out = orc.mlp(x, (3, 2), _blob([(W, np.array([10, 20], np.float32))]), 0)
    np.testing.assert_array_equal(out, [[1 - 3 + 10, 4 - 6 + 20]])


def test_against_torch_float64_linear(c1):
    cfg, batch, blob = c1
    rng = np.random.default_rng(1)
    for spec in synth.model_layout(cfg)[:4] + synth.model_layout(cfg)[-1:]:
        x = rng.normal(size=(33, spec.dims[0])).astype(np.float32)
        got = orc.mlp(x, spec.dims, blob, spec.offset)
        a = torch.from_numpy(x).double()
        layers = spec.layer_offsets()
        for li, (wo, bo, fi, fo) in enumerate(layers):
            W = torch.from_numpy(blob[wo:wo + fi * fo].reshape(fo, fi)).double()
            b = torch.from_numpy(blob[bo:bo + fo]).double()
            a = F.linear(a, W, b).float().double()            # stored activations are fp32
            if li < len(layers) - 1:
                a = torch.relu(a)
        ref = a.numpy()
        np.testing.assert_allclose(got, ref, rtol=2e-6, atol=2e-7), spec.name


def test_features_normalisation(c0):
    _, b, _ = c0
    fe, fn = orc.features(b, synth.NORM_CENTER, synth.NORM_SCALE)
    np.testing.assert_allclose(fe[:, 0], b["r"] / 42.0, rtol=1e-6)
    np.testing.assert_allclose(fe[:, 1], b["phi"] / np.pi, rtol=1e-6)
    np.testing.assert_allclose(fe[:, 2], (b["z"] - 225.0) / 500.0, rtol=1e-6, atol=1e-7)
    np.testing.assert_allclose(fn[:, 0], b["x"] / 42.0, rtol=1e-6)
    np.testing.assert_allclose(fn[:, 1], b["y"] / 42.0, rtol=1e-6)
    np.testing.assert_array_equal(fn[:, 2], fe[:, 2])
    assert np.abs(fe).max() <= 1.06 and np.abs(fn).max() <= 1.06
