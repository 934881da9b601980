"""Shared fixtures.  `-m "not gpu"` tests: generator, oracle pins, host logic, C-ABI symbol check.
`-m gpu` tests: CUDA path vs oracle through the C ABI (need a B200)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


from paper_2508_07423_b200 import synth  # noqa: E402


def layout_dict(cfg):
    return {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}


def oracle_path(cfg, batch, blob, graph=None, r2=None, gap=None):
    from oracle import etx_oracle as orc
    return orc.run_path(batch, blob, layout_dict(cfg), cfg.gnn_hidden, cfg.n_iter,
                        synth.r2_max(cfg) if r2 is None else r2,
                        cfg.max_plane_gap if gap is None else gap,
                        synth.NORM_CENTER, synth.NORM_SCALE, graph=graph)


@pytest.fixture(scope="session")
def c0():
    cfg = synth.CONFIGS["c0"]
    batch = synth.generate_events(cfg)
    blob = synth.generate_weights(cfg)
    return cfg, batch, blob


@pytest.fixture(scope="session")
def c0_oracle(c0):
    cfg, batch, blob = c0
    return oracle_path(cfg, batch, blob)


@pytest.fixture(scope="session")
def c1():
    cfg = synth.CONFIGS["c1"]
    return cfg, synth.generate_events(cfg), synth.generate_weights(cfg)


@pytest.fixture(scope="session")
def c1_oracle(c1):
    cfg, batch, blob = c1
    return oracle_path(cfg, batch, blob)
