"""Host-side checks of bench.py (no GPU): the JSON contract of the reference arm, the roofline arithmetic on a recorded
profile, the traffic look-up, and the whole-job aggregation -- a typo here would cost the round its BENCH record."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402
import gmco_cases as gc  # noqa: E402


class _G:
    GMCO_PREC_TF32X3, GMCO_PREC_SIMT_FP32 = 0, 1


PROF = {"eval_launches": 230, "eval_plans": 230 * 906, "eval_ms": 230 * 0.0645, "dose_ms": 230 * 0.0350, "grad_ms": 230 * 0.0295,
        "step_ms": 230 * 0.016, "dose_kernel": 2, "dose_kernel_name": "k_dose_tc_pair<4,6>"}
PEAKS = dict(hbm_gbs=6455.3, bf16_burst=1721.3, bf16_sustained=1428.5, source="measured")


def test_roofline_arithmetic_per_kernel():
    c = gc.make_case("C3")
    tf32 = {"tf32_tflops": 950.0, "tf32_tflops_sustained": 800.0, "how": "test"}
    r = bench.roofline(c, 0, _G, PROF, PEAKS, tf32, {"sm_mhz": 1965.0})
    flops = 2.0 * 12000 * 252 * 906
    assert r["kernel"] == "k_dose_tc_pair<4,6>" and r["bound"] == "tensor" and r["unit"] == "TFLOP/s"
    assert r["achieved"] == pytest.approx(3 * flops / 35e-6 / 1e12) and r["peak"] == 950.0
    assert r["frac"] == pytest.approx(r["achieved"] / 950.0) and r["achieved_fp32_equivalent"] == pytest.approx(r["achieved"] / 3)
    pk = r["per_kernel"]
    assert pk["grad"]["achieved"] == pytest.approx(3 * flops / 29.5e-6 / 1e12) and pk["grad"]["kernel"] == "k_grad_tc<16>"
    step_bytes = (4 * 10 * 252 + 10 * 252) * 4.0 * 906
    assert pk["step"]["bound"] == "hbm" and pk["step"]["achieved"] == pytest.approx(step_bytes / 16e-6 / 1e9)
    assert pk["step"]["frac"] == pytest.approx(pk["step"]["achieved"] / 6455.3)
    alts = r["peak_alternatives"]
    assert alts["issue_limit_4096_flop_per_clk_per_sm_at_sampled_clock"] == pytest.approx(4096 * 148 * 1.965e9 / 1e12)
    assert alts["nominal_ratio_of_measured_bf16_burst"] == pytest.approx(1721.3 * 1.1 / 2.25)
    assert alts["measured_tf32_sustained"] == 800.0
    assert r["traffic"] == 26060000 + 3100000 and pk["grad"]["traffic"] == 74339328 + 4086272
    assert r["traffic_source"] == "profiles/ncu_traffic.csv"
    json.dumps(r)
    # no live peak: falls back to the nominal ratio and says so
    r2 = bench.roofline(c, 0, _G, PROF, PEAKS, None, {"sm_mhz": None})
    assert r2["peak"] == pytest.approx(1721.3 * 1.1 / 2.25) and "no live tf32" in r2["peak_source"]
    assert bench.roofline(c, 0, _G, None, PEAKS, None, None) is None
    r3 = bench.roofline(c, 1, _G, PROF, PEAKS, None, None)
    assert r3["bound"] == "alu" and r3["frac"] > 0


def test_traffic_lookup_and_job_value():
    assert bench.ncu_traffic("C3", "k_step") == 42398720 + 41472
    assert bench.ncu_traffic("C4", "k_step") is None and bench.ncu_traffic("C3", "nope") is None
    assert bench.job_value(1000, 4, 5, 100.0) == pytest.approx(4 * 1000 * 5 / 0.1)
    assert bench.max_over_ranks_ms(3.5, 1, "cpu") == 3.5
    assert bench.load_peaks()["hbm_gbs"] > 1000


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` on a tiny sample: one JSON line with the keys the driver reads."""
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--config", "C1", "--steps", "1",
                          "--warmup", "0", "--ref-sample", "2"], capture_output=True, text=True, check=True, cwd=str(ROOT)).stdout
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "plans_per_s" and line["unit"] == "plans/s"
    assert line["value"] > 0 and line["higher_is_better"] is True and line["dtype"] == "f64"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "plans/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["config"]["workload"].startswith("C1")
