"""-m "not gpu": the host-side arithmetic of bench.py's measurement contract: the algorithmic
bytes / FLOPs of SURVEY 8(d) on the seeded workloads, the clock-sampler parsing, the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from helpers import oracle_gate_select  # noqa: E402
from oracle import echo_oracle as orc  # noqa: E402
from paper_2604_09603_b200 import workloads as W  # noqa: E402

# bytes_alg / FLOPs_alg of the drawn instances (seed 60480 + config).  cfg2's byte count is the one VERDICT r1
# recomputed by hand from SURVEY 8(d)'s formula (1 365 385 216 B); SURVEY's table gives the expected values from mean
# prefix lengths (189 MB, 1 418 MB, 1 627 MB static, 1 378 MB).
PINS = {(1, False): (194228224, 22043230208, 189e6), (2, False): (1365385216, 162863874048, 1418e6),
        (2, True): (1574445056, 619870912512, 1627e6), (3, False): (1397528576, 174253735936, 1378e6)}


@pytest.mark.parametrize("cfg,static", sorted(PINS))
def test_algorithmic_bytes_formula_and_pins(cfg, static):
    wl = W.make_config(cfg, static=static, gated=not static)
    sel = oracle_gate_select(orc, wl)
    got_b, got_f = bench.algorithmic_bytes(wl, sel)
    # SURVEY 8(d) spelled out request by request and node by node
    b = f = 0
    off = sel["sel_offsets"]
    for i in range(wl.R):
        K, P = int(off[i + 1] - off[i]), int(wl.prefix_len[i])
        if K > 0:
            b += 2 * wl.Hkv * 128 * 2 * (P + K)                  # K and V, every visible token once per KV head
        b += 2 * K * wl.Hq * 128 * 2 + 4 * K * wl.Hq             # Q read + O write (bf16), LSE (fp32)
        for l in range(K):
            f += 4 * 128 * wl.Hq * (P + int(sel["sel_depth"][off[i] + l]) + 1)   # QK^T and PV on visible keys only
    assert (got_b, got_f) == (b, f)
    pin_b, pin_f, survey_b = PINS[(cfg, static)]
    assert (got_b, got_f) == (pin_b, pin_f)
    assert abs(got_b - survey_b) / survey_b < 0.05               # the drawn instance against the table's expectation


def test_roofline_picks_the_bounding_roof():
    """elastic configs are HBM-bound by FLOP per byte, the static-60 run is tensor-bound (SURVEY 8(d) 'Which roof')"""
    ridge = bench.tensor_peak(False)[0] * 1e12 / (bench.peaks()[0] * 1e9)
    ai = {k: v[1] / v[0] for k, v in PINS.items()}
    assert ai[(2, False)] < ridge and ai[(1, False)] < ridge and ai[(3, False)] < ridge
    assert ai[(2, True)] > ridge
    assert 100 < ai[(2, False)] < 130 and 380 < ai[(2, True)] < 410          # AI ~ K_i G: SURVEY's 114-126 / 396


def test_roofline_object_arithmetic():
    """Case.roofline on the pinned cfg2 / static-60 work: achieved = algorithmic bytes (FLOPs) / time, fractions
    against the measured and the nominal roof (no GPU needed: the object only holds the two counts)"""
    c = bench.Case.__new__(bench.Case)
    c.bytes_alg, c.flops_alg = PINS[(2, False)][:2]
    r = c.roofline(0.25)
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["bytes_per_launch"] == 1365385216
    assert r["achieved"] == pytest.approx(1365385216 / 0.25e-3 / 1e9)
    assert r["frac"] == pytest.approx(r["achieved"] / bench.peaks()[0])
    assert r["frac_nominal"] == pytest.approx(r["achieved"] / 8000.0) and r["peak_nominal"] == 8000.0
    c.bytes_alg, c.flops_alg = PINS[(2, True)][:2]
    r = c.roofline(0.64, sustained=True)
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s"
    assert r["achieved"] == pytest.approx(619870912512 / 0.64e-3 / 1e12)
    assert r["frac"] == pytest.approx(r["achieved"] / bench.tensor_peak(True)[0])
    assert r["frac_nominal"] == pytest.approx(r["achieved"] / 2250.0)


def test_clock_sampler_summary_parses_nvidia_smi_rows():
    s = bench.ClockSampler(0)
    rows = [["1965", "1965", "310.5", "Not Active", "Not Active", "Not Active", "Not Active"],
            ["1500", "1965", "990.1", "Not Active", "Not Active", "Not Active", "Active"],
            ["1470", "1965", "1001.0", "Not Active", "Not Active", "Not Active", "Active"]]
    out = s.summary(rows, [1480.0, 1500.0, 1490.0])
    assert out["sm_mhz"] == 1490.0 and out["sm_max_mhz"] == 1965 and out["nvml_sm_mhz"] == 1500
    assert out["power_w_max"] == 1001.0 and out["reasons"] == ["sw_power_cap"] and out["nvml_samples"] == 3
    empty = s.summary([], [])
    assert empty["sm_mhz"] is None and empty["reasons"] == [] and empty["nvml_samples"] == 0


def test_reference_arm_prints_the_contract_line():
    """bench.py --impl reference: the oracle timed on the host, one JSON line with the arm's keys"""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--ref-nodes", "1", "--config", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "verified draft tokens/s" and line["unit"] == "tokens/s"
    assert line["higher_is_better"] is True and line["value"] > 0 and line["steps"] == 1 and line["gpu_launches"] == 0
    assert line["config"]["workload"].startswith("cfg1")
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["value"] == line["value"] and "packed nodes" in cb["sample"]
    assert cb["cores"] == len(os.sched_getaffinity(0)) and f"on {cb['cores']} threads" in cb["sample"]   # the cores it used
    assert line["e2e"] == {"value": line["value"], "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
