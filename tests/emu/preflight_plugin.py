"""Pre-flight of the `-m gpu` tests on the CPU emulation.  TEST INFRASTRUCTURE, opt-in only:

    PYTHONPATH=tests/emu python -m pytest -p preflight_plugin -m gpu tests/test_gpu_parity.py -k "c1 or ragged" -n 8

Loaded with `-p` (and only then), this plugin points the product's ctypes binding at tests/emu/_build/libgmco_emu.so --
the kernels' own source executed on the CPU -- and lets the test modules' `g` fixtures believe that a
CUDA device is present, so that the BODIES of the GPU tests (shapes, calls, tolerances, edge cases) run unchanged
before a GPU is available.  Without `-p preflight_plugin` nothing here is imported: `pytest -m gpu` runs the
real library on a real B200 and fails loudly without one.  Tests that hand torch CUDA tensors to the library cannot run
here and fail with torch's own error; deselect them with -k.  At the end of the session the plugin fails the run if the
emulated hardware recorded a violation (access outside the shared-memory window / TMEM / device allocations, barrier
misuse, hazards, work left in flight).
"""
import ctypes as C
import os
import sys
from pathlib import Path

import pytest

HERE = Path(__file__).resolve().parent
ROOT = HERE.parents[1]
_E = None


def pytest_configure(config):
    global _E
    for p in (str(ROOT), str(HERE)):
        if p not in sys.path:
            sys.path.insert(0, p)
    import build_emu
    lib = build_emu.build()
    import paper_1904_01567_b200.binding as b
    from paper_1904_01567_b200 import build as product_build
    b.lib_path = lambda: lib
    b._lib = None
    b._stream = lambda stream: None
    product_build.build = lambda *a, **k: lib          # the fixtures call build(): nothing to compile for the emulation
    import torch
    torch.cuda.is_available = lambda: True              # only inside this opt-in session
    _E = C.CDLL(str(lib))
    _E.emu_violation_message.restype = C.c_char_p
    _E.emu_set.argtypes = [C.c_char_p, C.c_long]
    _E.emu_set(b"sm_count", int(os.environ.get("GMCO_EMU_SMS", "148")))
    config._gmco_emu = _E


def pytest_report_header(config):
    return "gmco pre-flight: the gpu tests run on the CPU EMULATION of the kernels (tests/emu), not on a GPU"


@pytest.hookimpl(trylast=True)
def pytest_runtest_teardown(item):
    # a violation is attributed to the test during which it was recorded
    if _E is not None and _E.emu_violations():
        msg = (_E.emu_violation_message() or b"").decode()
        _E.emu_clear()
        pytest.fail(f"emulated hardware recorded a violation: {msg}", pytrace=False)
