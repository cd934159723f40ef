"""Pins of the calibration oracle (NEXT-3): closed forms, brute force over pairs, and scikit-learn's
roc_auc_score / roc_curve (an independent library routine for the same textbook statistics)."""
import numpy as np
import pytest

from oracle import echo_oracle as orc


def _traces(rng, M, sep):
    depth = rng.integers(0, 8, M).astype(np.uint8)
    acc = rng.random(M) < 0.4
    conf = np.clip(rng.beta(2, 2, M) + sep[depth] * (acc - 0.5), 1e-6, 1.0).astype(np.float32)
    conf = (np.round(conf * 64) / 64).astype(np.float32) if M < 600 else conf     # small cases: plenty of ties
    return depth, conf, acc.astype(np.uint8)


def test_closed_forms():
    # perfectly separated: AUC 1, tau = the largest rejected confidence; swapped: AUC 0; identical: AUC 0.5
    depth = np.zeros(6, np.uint8)
    conf = np.asarray([0.1, 0.2, 0.3, 0.6, 0.7, 0.8], np.float32)
    acc = np.asarray([0, 0, 0, 1, 1, 1], np.uint8)
    c = orc.calibrate(depth, conf, acc, 0.7)
    assert c["auc"][0] == 1.0 and c["tau"][0] == np.float32(0.3) and c["depth_mask"] == 1
    c = orc.calibrate(depth, conf, 1 - acc, 0.7)
    assert c["auc"][0] == 0.0 and c["depth_mask"] == 0
    c = orc.calibrate(np.zeros(4, np.uint8), np.asarray([0.5] * 4, np.float32), np.asarray([0, 1, 0, 1], np.uint8), 0.4)
    assert c["auc"][0] == 0.5 and c["depth_mask"] == 1 and c["n_pos"][0] == 2 and c["n_neg"][0] == 2
    # one class missing: undefined separability -> 0.5, never a sweet spot, even with delta below 0.5
    c = orc.calibrate(np.ones(3, np.uint8), np.asarray([0.2, 0.4, 0.9], np.float32), np.ones(3, np.uint8), 0.1)
    assert c["auc"][1] == 0.5 and c["depth_mask"] == 0 and c["tau"][1] == 0.0
    # hand example with a tie: pos {0.5, 0.9}, neg {0.5, 0.1}: pairs > : (0.5,0.1) (0.9,0.5) (0.9,0.1) = 3, ties 1
    c = orc.calibrate(np.zeros(4, np.uint8), np.asarray([0.5, 0.9, 0.5, 0.1], np.float32),
                      np.asarray([1, 1, 0, 0], np.uint8), 0.5)
    assert c["auc"][0] == (3 + 0.5) / 4
    # J(0.1) = 2/2 - 1/2 = 0.5, J(0.5) = 1/2 - 0 = 0.5, J(0.9) = 0: tie -> the smaller threshold
    assert c["tau"][0] == np.float32(0.1)


@pytest.mark.parametrize("seed", range(4))
def test_bruteforce_pairs_and_thresholds(seed):
    rng = np.random.default_rng(seed)
    depth, conf, acc = _traces(rng, 400, np.linspace(0.6, 0.0, 8))
    c = orc.calibrate(depth, conf, acc, 0.6)
    for d in range(8):
        pos = conf[(depth == d) & (acc == 1)].astype(np.float64)
        neg = conf[(depth == d) & (acc == 0)].astype(np.float64)
        gt = sum(1 for p in pos for n in neg if p > n)
        eq = sum(1 for p in pos for n in neg if p == n)
        assert c["auc"][d] == (gt + 0.5 * eq) / (len(pos) * len(neg))
        best = max(((np.mean(pos > v) - np.mean(neg > v)), -v) for v in np.unique(np.concatenate([pos, neg])))
        j_tau = np.mean(pos > c["tau"][d]) - np.mean(neg > c["tau"][d])
        assert abs(j_tau - best[0]) < 1e-12
        assert (c["depth_mask"] >> d) & 1 == int(c["auc"][d] > 0.6)


def test_against_scikit_learn():
    sk = pytest.importorskip("sklearn.metrics")
    rng = np.random.default_rng(7)
    depth, conf, acc = _traces(rng, 20000, np.asarray([0.7, 0.1, 0.1, 0.3, 0.1, 0.6, 0.05, 0.0]))
    c = orc.calibrate(depth, conf, acc, 0.65)
    for d in range(8):
        m = depth == d
        assert abs(c["auc"][d] - sk.roc_auc_score(acc[m], conf[m].astype(np.float64))) < 1e-12
        fpr, tpr, thr = sk.roc_curve(acc[m], conf[m].astype(np.float64), drop_intermediate=False)
        # roc_curve predicts positive for score >= thr; our gate is c > tau: J over its curve has the same maximum
        j_tau = np.mean(conf[m & (acc == 1)] > c["tau"][d]) - np.mean(conf[m & (acc == 0)] > c["tau"][d])
        assert abs(j_tau - np.max(tpr - fpr)) < 1e-12
    assert c["depth_mask"] == sum(1 << d for d in range(8) if c["auc"][d] > 0.65)
    assert (c["depth_mask"] & 0b100001) == 0b100001   # the two depths built to be sweet spots
