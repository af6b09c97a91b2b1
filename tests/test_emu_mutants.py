"""Does the CPU emulation of the kernels (tests/emu, tests/test_emu_kernels.py) notice a wrong kernel?  Each MUTANT is the
product's source with ONE planted error -- a barrier wait left out, a phase that never flips, a shared-memory size
that is too small, a wrong index, a missing dealloc (tests/emu/build_emu.py MUTANTS).  Every one of them must be
DETECTED: by a hazard the emulated hardware reports (slot refilled under its reader, operand read before it landed,
accumulator touched before its commit, access outside the shared-memory window, TMEM not freed), by the library's own
containment (device error word -> GMCO_E_CUDA, never a hang), or by parity with the oracle.  A clean run of the
unmodified source in tests/test_emu_kernels.py means something only because these fail.

One of these mutants found a real defect in round 2's fault containment: with a planted phase error some lanes of the
gradient kernel's issuing warp saw the abort flag and left while others went on to `elect.sync` and waited for the full
warp for ever -- the bounded waits now vote, so that a warp gives up as a whole (kernels_tc.cu mbar_wait_addr)."""
import json
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

import platform

import pytest

pytestmark = pytest.mark.skipif(platform.machine() != "x86_64", reason="tests/emu switches fibers with x86-64 assembly")

ROOT = Path(__file__).resolve().parents[1]
STREAMED = dict(n_plans=128, n_cath=24, n_pos=16, sm_count=2, counts=[500, 100, 120, 120])   # 5-entry ring, 24 entries per chunk
C1 = dict(sm_count=4)

# mutant -> (scenario arguments, how it must show)
CASES = {
    "producer_skips_empty_wait": (dict(scenario="evaluate", **STREAMED), "hazard_or_error"),
    "issuer_skips_full_wait": (dict(scenario="evaluate", **STREAMED), "hazard"),
    "grad_issuer_skips_conv_wait": (dict(scenario="evaluate", **STREAMED), "hazard"),
    "epilogue_skips_acc_full_wait": (dict(scenario="evaluate", **STREAMED), "hazard_or_error"),
    "issuer_skips_acc_empty_wait": (dict(scenario="evaluate", **STREAMED), "hazard"),
    "accumulator_handed_back_too_early": (dict(scenario="evaluate", **STREAMED), "hazard"),
    "tmem_never_freed": (dict(scenario="evaluate", **STREAMED), "hazard"),
    "wrong_chunk_loaded": (dict(scenario="evaluate", **STREAMED), "parity"),
    "wrong_k_step_descriptor": (dict(scenario="evaluate", **STREAMED), "parity"),
    "host_smem_too_small": (dict(scenario="fault", drop="drop_tma", nth=-1, no_recovery=1, **STREAMED), "contained"),
    "host_smem_too_small_unchecked": (dict(scenario="fault", drop="drop_tma", nth=-1, no_recovery=1, **STREAMED), "hazard"),
    "producer_phase_never_flips": (dict(scenario="fault", drop="drop_tma", nth=-1, no_recovery=1, **STREAMED), "contained"),
    "gpair_converter_skips_full_wait": (dict(scenario="evaluate", sm_count=4, n_plans=256, n_cath=18, n_pos=14, dose_kernel=2, max_delay=3000, mma_delay=20, counts=[500, 100, 120, 120]), "any"),
    "gpair_peer_loads_wrong_half": (dict(scenario="evaluate", sm_count=4, n_plans=256, n_cath=18, n_pos=14, dose_kernel=2, counts=[500, 100, 120, 120]), "parity"),
    # k_step overwrites a staged history slot while its bulk copy may still be on its way: a late copy puts the old pair back
    "step_skips_history_wait": (dict(scenario="optimize", iters=12, seed=1, max_delay=20000, **C1), "parity"),
}


@pytest.fixture(scope="module")
def results():
    sys.path.insert(0, str(ROOT / "tests" / "emu"))
    import build_emu
    build_emu.build()
    import oracle
    oracle.build()

    def run(item):
        name, (args, _) = item
        lib = build_emu.build_mutant(name)
        p = subprocess.run([sys.executable, str(ROOT / "tests" / "emu" / "driver.py"), json.dumps(dict(args, lib=str(lib)))],
                           capture_output=True, text=True, timeout=900)
        line = [l for l in p.stdout.splitlines() if l.startswith("EMU_RESULT ")]
        if not line:
            return name, dict(crashed=True, returncode=p.returncode, stderr=p.stderr[-2000:])
        return name, json.loads(line[-1][len("EMU_RESULT "):])

    with ThreadPoolExecutor(max_workers=8) as ex:
        return dict(ex.map(run, CASES.items()))


@pytest.mark.parametrize("name", list(CASES))
def test_planted_error_is_detected(results, name):
    r, how = results[name], CASES[name][1]
    assert not r.get("crashed"), f"{name}: the driver died instead of reporting: {r.get('stderr')}"
    hazard = r["violations"] > 0
    error = r.get("code") == -3
    bad_numbers = any(v > 1e-4 for v in (r.get("errors") or {}).values()) or (r.get("rel_F_max") or 0.0) > 1e-3
    if how == "hazard":
        assert hazard, (name, r)
    elif how == "hazard_or_error":
        assert hazard or error, (name, r)
    elif how == "any":
        assert hazard or error or bad_numbers, (name, r)
    elif how == "parity":
        assert bad_numbers and not hazard and not error, (name, r)       # nothing but the numbers shows an index error
    elif how == "contained":
        # the library's own containment: an error code through the normal teardown -- no hang, TMEM freed, nothing in flight
        assert error and r["hangs"] == 0, (name, r)
        assert "barrier wait did not complete" in r["error"] or "carve-up does not fit" in r["error"], r["error"]


def test_hazard_messages_name_what_happened(results):
    assert "before its consumer's commit" in results["issuer_skips_full_wait"]["violation"] or "in flight" in results["issuer_skips_full_wait"]["violation"]
    assert "accumulator touched before its commit arrived" in results["issuer_skips_acc_empty_wait"]["violation"]
    assert "without tcgen05.dealloc" in results["tmem_never_freed"]["violation"]
    # barriers and ring then overlap / run past the launched window: whichever consequence comes first under the schedule
    v = results["host_smem_too_small_unchecked"]["violation"]
    assert any(t in v for t in ("outside the CTA's window", "still in flight", "was overwritten", "no initialised mbarrier", "hangs")), v
