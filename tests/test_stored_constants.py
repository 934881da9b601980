"""The stored per-config constants (radius r^2, INT8 activation ranges, weight gain g) are what the committed
ORACLE-ONLY calibration scripts produce: each script is re-run here and compared with
paper_2508_07423_b200/config_constants.json, so a stale or hand-edited constant fails (DESIGN Q21).
Nothing in this file touches the CUDA library."""
import numpy as np
import pytest

from oracle import calibrate_gain, calibrate_int8, calibrate_int8_gnn, calibrate_radius
from paper_2508_07423_b200 import synth

NAMES = ("c0", "c1", "c2", "c4")


@pytest.fixture(scope="module")
def stored():
    return synth.load_constants()


@pytest.mark.parametrize("name", NAMES)
def test_radius_is_regenerated_by_the_oracle_script(stored, name):
    got = calibrate_radius.calibrate(name)
    for k, v in got.items():
        assert stored[name][k] == v, (name, k)
    assert abs(got["calib_mean_out_degree"] - got["target_degree"]) < 0.01


@pytest.mark.parametrize("name", NAMES)
def test_int8_ranges_are_regenerated_by_the_oracle_script(stored, name):
    np.testing.assert_array_equal(np.float32(calibrate_int8.calibrate(name)), np.float32(stored[name]["int8_act_alpha"]))


@pytest.mark.parametrize("name", NAMES)
def test_gain_is_regenerated_by_the_oracle_script(stored, name):
    got = calibrate_gain.calibrate(name)
    assert got["gain"] == stored[name]["gain"] == synth.CONFIGS[name].gain
    assert got["gain_stats"] == stored[name]["gain_stats"]
    st = got["gain_stats"]
    # the criterion itself, re-stated: unsaturated, bounded, not collapsed
    assert st["frac_unsaturated"] >= 0.5 and st["max_abs_h"] < 1e3 and st["max_abs_e"] < 1e3 and st["score_std"] >= 0.05
    # ... and every smaller grid value was rejected (the rule takes the smallest accepted one)
    assert all(not calibrate_gain.accept(t) for t in got["gain_tried"][:-1])
    assert [t["gain"] for t in got["gain_tried"]] == calibrate_gain.GRID[:len(got["gain_tried"])]


@pytest.mark.parametrize("name", NAMES)
def test_int8_gnn_ranges_are_regenerated_by_the_oracle_script(stored, name):
    got = calibrate_int8_gnn.calibrate(name)
    assert sorted(got) == sorted(stored[name]["int8_gnn_alpha"])
    for k, v in got.items():
        np.testing.assert_array_equal(np.float32(v), np.float32(stored[name]["int8_gnn_alpha"][k]))


def test_c3_shares_c2_constants():
    assert synth.CONFIGS["c3"].gain == synth.CONFIGS["c2"].gain and synth.r2_max(synth.CONFIGS["c3"]) == synth.r2_max(synth.CONFIGS["c2"])
