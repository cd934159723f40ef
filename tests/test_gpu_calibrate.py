"""-m gpu parity: echo_calibrate (CUDA, through the C ABI) against the oracle -- bit-exact: AUC is one fp64 division
of exact integers on both sides, tau is an observed fp32 value, counts and the sweet-spot mask are integers."""
import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from gpu_util import dev, get_ctx

pytestmark = pytest.mark.gpu


def _check(ctx, depth, conf, acc, delta):
    got = ctx.calibrate(dev(depth), dev(conf), dev(acc), delta)
    want = orc.calibrate(depth, conf, acc, delta)
    np.testing.assert_array_equal(got["n_pos"].cpu().numpy(), want["n_pos"])
    np.testing.assert_array_equal(got["n_neg"].cpu().numpy(), want["n_neg"])
    np.testing.assert_array_equal(got["auc"].cpu().numpy(), want["auc"])
    np.testing.assert_array_equal(got["tau"].cpu().numpy(), want["tau"])
    assert int(got["depth_mask"].item()) & 0xFFFFFFFF == want["depth_mask"]
    return want


@pytest.mark.parametrize("M,ties", [(0, False), (1, False), (37, True), (1000, True), (5000, False), (180000, False)])
def test_calibrate_synthetic_traces(M, ties):
    rng = np.random.default_rng(M + 1)
    depth, conf, acc = W.draw_calibration_traces(rng, M, ties=ties)
    ctx = get_ctx()
    want = _check(ctx, depth, conf, acc, 0.65)
    assert ctx.device_status() == 0
    if M >= 5000:
        assert want["depth_mask"] & 0b100001 == 0b100001     # depths 0 and 5 are built to be sweet spots


def test_calibrate_edge_cases():
    ctx = get_ctx()
    # a depth with one class only, perfectly separated depth, all-equal confidences, values 0 and 1
    depth = np.asarray([0, 0, 0, 1, 1, 1, 1, 2, 2, 2, 2, 3, 3, 31], np.uint8)
    conf = np.asarray([.2, .4, .9, .1, .2, .7, .8, .5, .5, .5, .5, 0.0, 1.0, 0.3], np.float32)
    acc = np.asarray([1, 1, 1, 0, 0, 1, 1, 0, 1, 0, 1, 0, 1, 0], np.uint8)
    want = _check(ctx, depth, conf, acc, 0.4)
    assert want["auc"][1] == 1.0 and want["tau"][1] == np.float32(0.2) and want["auc"][2] == 0.5
    assert ctx.device_status() == 0
    # the full shared-memory capacity at one depth, and one sample more (status bit, excess dropped)
    from paper_2604_09603_b200 import echo
    rng = np.random.default_rng(3)
    n = echo.CALIB_MAX_PER_DEPTH
    conf = rng.random(n).astype(np.float32)
    acc = (rng.random(n) < conf).astype(np.uint8)
    _check(ctx, np.full(n, 4, np.uint8), conf, acc, 0.6)
    assert ctx.device_status() == 0
    ctx.calibrate(dev(np.full(n + 1, 4, np.uint8)), dev(np.append(conf, np.float32(0.5))), dev(np.append(acc, 1).astype(np.uint8)), 0.6)
    assert ctx.device_status() == echo.DEV_CALIB_OVERFLOW
    # precondition violations are flagged and skipped, never trap
    bad = np.asarray([0.5, np.nan, -0.1, 1.5, 0.25], np.float32)
    got = ctx.calibrate(dev(np.asarray([0, 0, 0, 0, 40], np.uint8)), dev(bad), dev(np.ones(5, np.uint8)), 0.6)
    assert ctx.device_status() == echo.DEV_BAD_TRACE
    assert int(got["n_pos"][0].item()) == 1
