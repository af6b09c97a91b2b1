"""The C-ABI library loads and exports every symbol include/gmco.h declares (no GPU needed)."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def built_lib():
    from paper_1904_01567_b200 import build
    return build.build()


def _declared_functions():
    text = (ROOT / "include" / "gmco.h").read_text()
    return sorted(set(re.findall(r"GMCO_API\s+[\w\s\*]+?\b(gmco_\w+)\s*\(", text)))


def test_header_declares_the_three_calls_of_the_north_star():
    names = _declared_functions()
    for required in ("gmco_create", "gmco_optimize", "gmco_result", "gmco_evaluate", "gmco_destroy",
                     "gmco_last_error", "gmco_version", "gmco_default_options", "gmco_get_stats", "gmco_sa_run", "gmco_select_plan",
                     "gmco_pareto_front", "gmco_dose_rate_matrix", "gmco_tc_schedule", "gmco_set_profiling"):
        assert required in names


def test_library_exports_every_declared_symbol(built_lib):
    L = ctypes.CDLL(str(built_lib))
    for name in _declared_functions():
        assert hasattr(L, name), name


def test_version_and_default_options(built_lib):
    import paper_1904_01567_b200 as g
    assert g.gmco_version() == 140
    o = g.binding.make_options()
    assert (o.m, o.max_trials, o.precision) == (10, 20, g.GMCO_PREC_TF32X3)
    assert o.c1 == pytest.approx(1e-4) and o.eps == 0.0
    assert o.compaction == 1 and o.dose_kernel == 0 and o.wide_accum == 0 and o.line_search == 0


def test_struct_layouts_match_the_header(built_lib):
    import paper_1904_01567_b200.binding as b
    assert ctypes.sizeof(b._Structure) == 28 and ctypes.sizeof(b.Options) == 40 and ctypes.sizeof(b.Stats) == 56
    assert ctypes.sizeof(b.TcInfo) == 31 * 4
    assert ctypes.sizeof(b.Criterion) == 20


def test_argument_errors_are_reported_without_a_gpu(built_lib):
    """Validation happens before any CUDA call: these paths are safe on a CPU-only box."""
    import gmco_cases as gc
    import paper_1904_01567_b200 as g
    c = gc.make_case("C1", counts=(64, 16, 16, 16), n_plans=2)
    bad = [gc.Structure(s.name, s.n_points, s.d_lo, s.d_hi, s.w_lo, s.w_hi, s.dvh_kind, s.dvh_level) for s in c.structures]
    bad[0].n_points += 1
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(c.D, bad, c.rx)
    assert e.value.code == -1 and "add up" in str(e.value)
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(c.D, c.structures, -1.0)
    assert e.value.code == -1
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(compaction=2))
    assert e.value.code == -1 and "options" in str(e.value)
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(dose_kernel=3))
    assert e.value.code == -1 and "options" in str(e.value)
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(np.zeros((8, 500), np.float32), [gc.Structure("s", 8, 1, 2, 1, 1, 0, 0)], 15.0)
    assert e.value.code == -2


def test_no_cpu_fallback_exists(built_lib):
    """Without a GPU the product path must fail loudly, never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import gmco_cases as gc
    import paper_1904_01567_b200 as g
    c = gc.make_case("C1", counts=(64, 16, 16, 16), n_plans=2)
    with pytest.raises(g.GmcoError) as e:
        g.gmco_create(c.D, c.structures, c.rx)
    assert e.value.code in (-2, -3)


def test_product_never_imports_the_oracle():
    for p in (ROOT / "paper_1904_01567_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            txt = p.read_text().replace("shares nothing with oracle/", "")
            assert not re.search(r"(import|from|include|dlopen|CDLL).*oracle", txt), p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".c"):
            txt = p.read_text()
            assert "import paper_1904_01567_b200" not in txt and "from paper_1904_01567_b200" not in txt
            assert "gmco.h" not in txt


def test_ctypes_field_offsets_match_the_header_as_gcc_lays_it_out(tmp_path):
    """Every field of the binding's ctypes mirrors sits where a C compiler puts it in include/gmco.h (a drifted binding
    would read the wrong statistic or set the wrong option without any error)."""
    import shutil
    import subprocess
    import paper_1904_01567_b200.binding as b
    if not shutil.which("gcc"):
        pytest.skip("gcc not available")
    pairs = [("gmco_structure", b._Structure), ("gmco_options", b.Options), ("gmco_stats", b.Stats),
             ("gmco_criterion", b.Criterion), ("gmco_tc_info", b.TcInfo)]
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "gmco.h"', 'int main(void) {']
    for cname, ct in pairs:
        lines.append(f'  printf("{cname} %zu\\n", sizeof({cname}));')
        for fname, _ in ct._fields_:
            lines.append(f'  printf("{cname}.{fname} %zu\\n", offsetof({cname}, {fname}));')
    lines += ['  return 0;', '}']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", str(ROOT / "include"), "-o", str(exe), str(src)], check=True)
    out = dict(ln.split() for ln in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for cname, ct in pairs:
        assert int(out[cname]) == ctypes.sizeof(ct), cname
        for fname, _ in ct._fields_:
            assert int(out[f"{cname}.{fname}"]) == getattr(ct, fname).offset, f"{cname}.{fname}"


def test_binding_argument_counts_match_the_prototypes(built_lib):
    """The number of arguments the binding marshals for each entry point equals the header's prototype."""
    import paper_1904_01567_b200.binding as b
    text = (ROOT / "include" / "gmco.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    protos = dict(re.findall(r"GMCO_API\s+[\w\s\*]+?\b(gmco_\w+)\s*\(([^;]*?)\)\s*;", text, flags=re.S))
    L = b.lib()
    checked = 0
    for name, args in protos.items():
        n = 0 if args.strip() in ("", "void") else len([a for a in args.split(",") if a.strip()])
        fn = getattr(L, name)
        if fn.argtypes is not None:
            assert len(fn.argtypes) == n, (name, len(fn.argtypes), n)
            checked += 1
    assert checked >= 12
