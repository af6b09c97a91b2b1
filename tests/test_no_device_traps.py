"""The library must not be able to raise an SM exception or hang a GPU by itself: no `__trap()` /
`trap;` / `brkpt;` in the sources, every barrier wait bounded, and in the built SASS no trap instruction other than the
one ptxas itself emits inside its expansion of tcgen05.alloc / dealloc / relinquish_alloc_permit (an unreachable-by-design
error stub: one `BPT.TRAP` per `UTCATOMSWS`, whatever the kernel's source says)."""
import re
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
CSRC = ROOT / "paper_1904_01567_b200" / "csrc"


def _sources():
    return [p for p in CSRC.rglob("*") if p.suffix in (".cu", ".cuh", ".h")]


def test_sources_hold_no_trap_and_no_unbounded_spin():
    for p in _sources():
        code = re.sub(r"//[^\n]*", "", p.read_text())            # comments may talk about traps
        assert "__trap" not in code and not re.search(r"\btrap\s*;", code) and "brkpt" not in code, p
        assert "getenv" not in code and "fprintf" not in code and "printf(" not in code.replace("snprintf(", ""), p
    # all inline assembly lives in gmco_ptx.cuh (the seam the CPU-side kernel emulation of tests/emu replaces)
    for p in _sources():
        if p.name != "gmco_ptx.cuh":
            assert not re.search(r"\basm\b", re.sub(r"//[^\n]*", "", p.read_text())), p
    ptx = re.sub(r"//[^\n]*", "", (CSRC / "gmco_ptx.cuh").read_text())
    assert len(re.findall(r"try_wait\.parity", ptx)) == 2               # the two raw (unbounded-by-themselves) polls
    # every mbarrier wait of the tensor kernels goes through the bounded helpers: the raw polls are called from
    # mbar_wait_slow / mbar_wait_addr / mbar_wait_cluster / mbar_wait1_addr / mbar_wait1_cluster only (6 calls, each
    # followed by the bounded slow path), and from k_step's bounded history wait (1 call)
    tc = re.sub(r"//[^\n]*", "", (CSRC / "kernels_tc.cu").read_text())
    assert "kWaitLimitNs" in tc and "mbar_wait_slow" in tc and "drain_if_aborted" in tc
    assert len(re.findall(r"mbar_try_wait(?:_cluster)?_addr\(", tc)) == 6
    assert len(re.findall(r"return mbar_wait_slow\(", tc)) == 2 and len(re.findall(r"ok = mbar_wait_slow\(", tc)) == 2
    lb = re.sub(r"//[^\n]*", "", (CSRC / "kernels_lbfgs.cu").read_text())
    assert len(re.findall(r"mbar_try_wait(?:_cluster)?_addr\(", lb)) == 1
    assert "4000000000ull" in lb and "DEVERR_W_HISTORY" in lb            # k_step's history wait is bounded too
    for p in _sources():
        if p.name not in ("gmco_ptx.cuh", "kernels_tc.cu", "kernels_lbfgs.cu"):
            assert "mbar_try_wait" not in p.read_text(), p


def test_sass_holds_no_trap_besides_the_tcgen05_alloc_stubs():
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not Path(cuobjdump).exists():
        pytest.skip("cuobjdump not available")
    from paper_1904_01567_b200 import build
    lib = build.build()
    sass = subprocess.run([cuobjdump, "-sass", str(lib)], capture_output=True, text=True, check=True).stdout
    per_kernel, name = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            per_kernel[name] = [0, 0]
        elif name and re.search(r"\bBPT\b|\bTRAP\b", line):
            per_kernel[name][0] += 1
        elif name and "UTCATOMSWS" in line:
            per_kernel[name][1] += 1
    assert per_kernel, "no kernels found in the library"
    for k, (traps, allocs) in per_kernel.items():
        assert traps == allocs, f"{k}: {traps} trap instructions for {allocs} tcgen05 alloc-family instructions"
    assert sum(t for t, _ in per_kernel.values()) == 21            # 7 tensor kernels x (alloc, relinquish, dealloc)
    assert "UTCHMMA" in sass and "UTMALDG" in sass and "LDTM" in sass   # and it still is tcgen05 / TMA / TMEM code
