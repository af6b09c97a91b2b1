"""libgmco's HOST logic driven on a machine without a GPU ("what can be proven without a GPU").

The product's object files are linked a second time against tests/fake_cuda/fake_cudart.c instead of libcudart.  That
stand-in executes no kernel: it validates and records every launch (kernel, grid, block, dynamic shared memory, inside a
graph capture or not), hands out zero-filled host memory as "device" memory, range-checks every copy, memset and tensor
map against the allocation it touches, and checks the arguments of cuTensorMapEncodeTiled.  What this proves: the C ABI
runs through create / evaluate / optimize / result / destroy and the pool calls without a crash or an API error for
every route (tensor single-CTA, CTA pair, streamed T_lo, SIMT, profiling mode), every copy stays inside its
allocation, every launch configuration is legal and is the one gmco_tc_schedule announces, nothing leaks.
What it cannot prove: anything a kernel computes.  The driver script runs in a subprocess so that the real library
loaded by the other tests is untouched."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
FAKE = ROOT / "tests" / "fake_cuda"
OUT = FAKE / "_build"


@pytest.fixture(scope="module")
def host_lib():
    from paper_1904_01567_b200 import build
    build.build()
    OUT.mkdir(exist_ok=True)
    fake = OUT / "libfakecudart.so"
    subprocess.run(["gcc", "-O1", "-Wall", "-shared", "-fPIC", "-o", str(fake), str(FAKE / "fake_cudart.c")], check=True)
    objs = sorted(str(p) for p in (ROOT / "paper_1904_01567_b200" / "build").glob("*.cu.o"))
    assert len(objs) == len(build.SOURCES)
    lib = OUT / "libgmco_host.so"
    subprocess.run([build._nvcc(), "-shared", "-o", str(lib), *objs, "-cudart", "none", f"-L{OUT}", "-lfakecudart",
                    "-Xlinker", f"-rpath={OUT}", "-Wno-deprecated-gpu-targets"], check=True)
    return lib


DRIVER = r'''
import ctypes as C, json, sys
import numpy as np
sys.path.insert(0, sys.argv[2])
import gmco_cases as gc
import paper_1904_01567_b200.binding as b
from pathlib import Path
b.lib_path = lambda: Path(sys.argv[1])          # the host-logic build, not the product library
b._lib = None
import paper_1904_01567_b200 as g
F = C.CDLL(str(Path(sys.argv[1]).parent / "libfakecudart.so"))
F.fake_violation_message.restype = C.c_char_p

def launches():
    out = []
    name = C.create_string_buffer(200); dims = (C.c_uint * 6)(); smem = C.c_ulonglong(); cap = C.c_int()
    for i in range(F.fake_launch_count()):
        F.fake_launch(i, name, 200, dims, C.byref(smem), C.byref(cap))
        out.append(dict(name=name.value.decode(), grid=list(dims[:3]), block=list(dims[3:]), smem=int(smem.value), captured=int(cap.value)))
    return out

def kernel(l, frag):
    return [x for x in l if frag in x["name"]]

report = {}

def scenario(tag, case, opts, profile=False, iters=7):
    F.fake_reset_launches()
    K = case.n_plans
    h = g.gmco_create(case.D, case.structures, case.rx, opts)
    T = np.repeat(case.T0[None], K, axis=0)
    ev = g.gmco_evaluate(h, T, case.weights, want_dose=True, want_grad=True, host=True)
    n_eval = F.fake_launch_count()
    if profile:
        g.gmco_set_profiling(h, True)
    g.gmco_optimize(h, case.T0, case.weights, iters)
    out = g.gmco_result(h, host=True)
    st = g.gmco_get_stats(h)
    again = g.gmco_result(h, host=True)                     # a second read of the same result is allowed
    g.gmco_optimize(h, T, case.weights[: max(K // 2, 1)], 3)  # other K on the same handle: workspaces re-made
    g.gmco_result(h, host=True)
    g.gmco_optimize(h, case.T0, case.weights[:0], 3)         # empty batch
    g.gmco_result(h, host=True)
    g.gmco_destroy(h)
    l = launches()
    report[tag] = dict(stats=st, n_launches=len(l), n_eval_launches=n_eval, graph_launches=F.fake_graph_launches(),
                       kernels=sorted({x["name"] for x in l}), launches=l[:40],
                       shapes=dict(dose=list(ev["dose"].shape), T=list(out["T"].shape), again=list(again["T"].shape)),
                       live=F.fake_live_allocations(), violations=F.fake_violations(),
                       message=(F.fake_violation_message() or b"").decode())

c1 = gc.make_case("C1")
scenario("c1_tf32", c1, b.make_options(m=c1.m))
scenario("c1_simt", c1, b.make_options(m=c1.m, precision=1))
scenario("c1_profile", c1, b.make_options(m=c1.m), profile=True)
scenario("c1_simt_profile", c1, b.make_options(m=c1.m, precision=1), profile=True)
pair = gc.make_case("C1", n_plans=256)
scenario("pair_ring", pair, b.make_options(m=pair.m))
scenario("pair_forced_single", pair, b.make_options(m=pair.m, dose_kernel=1))
scenario("pair_both_contractions", pair, b.make_options(m=pair.m, dose_kernel=2))
wide = gc.make_case("C1", n_cath=24, n_pos=16, counts=(700, 130, 250, 190), n_plans=130, seed_points=9)
scenario("wide_streamed", wide, b.make_options(m=wide.m, eps=1e-3, compaction=0))
scenario("wide_split_main", wide, b.make_options(m=wide.m, wide_accum=1))
scenario("poly_ls_tf32", c1, b.make_options(m=c1.m, line_search=1))
scenario("poly_ls_simt_profile", c1, b.make_options(m=c1.m, line_search=1, precision=1), profile=True)
scenario("poly_ls_wide", wide, b.make_options(m=wide.m, line_search=1))
c3 = gc.make_case("C3")
scenario("c3_pair_static", c3, b.make_options(m=c3.m), iters=200)
widest = gc.make_case("C1", n_cath=35, n_pos=11, counts=(300, 64, 100, 100), n_plans=5, seed_points=5)   # 385 dwell positions: SIMT route
scenario("a385_falls_to_simt", widest, b.make_options(m=5))

# the pool calls and gSA with host arrays
F.fake_reset_launches()
h = g.gmco_create(c1.D, c1.structures, c1.rx)
jdx, z, u = gc.sa_draws(c1.n_dwell, c1.n_plans, 300, seed=5)
sa = g.gmco_sa_run(h, c1.T0, c1.weights, jdx, z, u, float(c1.T0[0]), host=True)
sa32 = g.gmco_sa_run(h, c1.T0, c1.weights, jdx[0], z[0], u[0], float(c1.T0[0]), precision=1, host=True)
dvh = np.random.default_rng(0).uniform(0, 100, (c1.n_plans, 4)).astype(np.float32)
sel = g.gmco_select_plan(h, dvh, [(0, 1, 90.0, 95.0, 0), (1, -1, 118.0, 118.0, 1), (2, -1, 10.0, 10.0, 2), (3, -1, 10.0, 10.0, 2)])
par = g.gmco_pareto_front(h, dvh)
g.gmco_destroy(h)
geo = c1.geometry if hasattr(c1, "geometry") else None
pts = np.random.default_rng(1).uniform(-20, 20, (100, 3)).astype(np.float32); dw = np.random.default_rng(2).uniform(-10, 10, (7, 3)).astype(np.float32)
Dm = g.gmco_dose_rate_matrix(pts, dw, [1.0, -0.01], 0.125, 0.1, host=True)
report["pool"] = dict(kernels=sorted({x["name"] for x in launches()}), sa_shape=list(sa["T"].shape), sa32=list(sa32["T"].shape),
                      selected=sel["selected"], n_nd=par["n_nondominated"], D=list(Dm.shape), live=F.fake_live_allocations(),
                      violations=F.fake_violations(), message=(F.fake_violation_message() or b"").decode())

# errors surface as codes, not crashes
errs = {}
h = g.gmco_create(c1.D, c1.structures, c1.rx)
try:
    g.gmco_result(h, host=True)
except g.GmcoError as e:
    errs["result_before_optimize"] = e.code
bad = np.repeat(c1.T0[None], c1.n_plans, 0).copy(); bad[1, 2] = np.nan
try:
    g.gmco_optimize(h, bad, c1.weights, 3)
except g.GmcoError as e:
    errs["nan_T0"] = e.code
g.gmco_destroy(h)
# a kernel that reported a protocol error through the device error word: GMCO_E_CUDA with kernel and wait site, then a state error
F.fake_plant_error_word(1, 1, (3 << 8) | 6, 5 | (2 << 16), 77)
h = g.gmco_create(c1.D, c1.structures, c1.rx)
g.gmco_optimize(h, c1.T0, c1.weights, 3)
try:
    g.gmco_result(h, host=True)
except g.GmcoError as e:
    errs["error_word_result"] = [e.code, str(e)]
try:
    g.gmco_result(h, host=True)
except g.GmcoError as e:
    errs["error_word_result_again"] = e.code
try:
    g.gmco_evaluate(h, np.repeat(c1.T0[None], c1.n_plans, 0), c1.weights, host=True)
except g.GmcoError as e:
    errs["error_word_evaluate"] = e.code
F.fake_plant_error_word(0, 0, 0, 0, 0)
g.gmco_optimize(h, c1.T0, c1.weights, 3)                 # the handle is usable again once the word is clear
g.gmco_result(h, host=True)
g.gmco_destroy(h)
report["errors"] = errs
report["final_live"] = F.fake_live_allocations()
report["tensor_maps"] = F.fake_tensor_maps()
print("REPORT" + json.dumps(report))
'''


@pytest.fixture(scope="module")
def report(host_lib):
    r = subprocess.run([sys.executable, "-c", DRIVER, str(host_lib), str(ROOT)], capture_output=True, text=True, cwd=str(ROOT))
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("REPORT")][-1]
    return json.loads(line[len("REPORT"):])


def _one(rep, frag, captured=None):
    sel = [x for x in rep["launches"] if frag in x["name"] and (captured is None or x["captured"] == captured)]
    assert sel, f"no launch of {frag}: {rep['kernels']}"
    return sel[0]


def test_no_copy_leaves_its_allocation_and_nothing_leaks(report):
    for tag, rep in report.items():
        if isinstance(rep, dict) and "violations" in rep:
            assert rep["violations"] == 0, f"{tag}: {rep['message']}"
            assert rep["live"] == 0, f"{tag}: {rep['live']} device allocations alive after gmco_destroy"
    assert report["final_live"] == 0 and report["tensor_maps"] > 0
    errs = dict(report["errors"])
    code, msg = errs.pop("error_word_result")
    assert code == -3 and "k_dose_tc_pair" in msg and "accumulator free" in msg and "block (5, 2)" in msg and "detail 77" in msg
    assert errs == {"result_before_optimize": -5, "nan_T0": -1, "error_word_result_again": -5, "error_word_evaluate": -3}


def test_shapes_and_statistics_of_every_route(report):
    import gmco_cases as gc
    c1 = gc.make_case("C1")
    for tag in ("c1_tf32", "c1_simt", "c1_profile", "c1_simt_profile"):
        rep = report[tag]
        assert rep["shapes"] == dict(dose=[c1.n_points, 8], T=[8, c1.n_dwell], again=[8, c1.n_dwell])
        assert rep["stats"]["plans_iters"] + rep["stats"]["plans_converged"] + rep["stats"]["plans_stalled"] == 8
        assert rep["stats"]["device_bytes"] > 0 and rep["stats"]["kernel_launches"] >= 3
    assert report["c1_tf32"]["stats"]["dose_kernel"] == 0 and report["c1_simt"]["stats"]["dose_kernel"] == -1
    assert report["pair_ring"]["stats"]["dose_kernel"] == 3 and report["pair_forced_single"]["stats"]["dose_kernel"] == 0
    assert report["wide_streamed"]["stats"]["dose_kernel"] == 1 and report["c3_pair_static"]["stats"]["dose_kernel"] == 2
    assert report["a385_falls_to_simt"]["stats"]["dose_kernel"] == -1
    # the device loop is ONE graph launch per gmco_optimize with K > 0 (two per scenario); profiling mode drives the rounds from the host
    assert report["c1_tf32"]["graph_launches"] == 2 and report["c1_profile"]["graph_launches"] == 0
    assert report["c1_profile"]["stats"]["eval_launches"] == 0        # nothing ran: no round had a running plan
    assert report["pool"]["sa_shape"] == [8, c1.n_dwell] and report["pool"]["D"] == [100, 7]
    assert any("k_sa" in k for k in report["pool"]["kernels"]) and any("k_pareto" in k for k in report["pool"]["kernels"])


def test_polynomial_line_search_option_adds_its_two_kernels_to_every_round(report):
    import gmco_cases as gc
    c1 = gc.make_case("C1")
    n_alloc = 256 * ((sum(64 * ((s.n_points + 63) // 64) for s in c1.structures) + 255) // 256)
    rep = report["poly_ls_tf32"]
    cols, pick = _one(rep, "k_ls_cols", captured=1), _one(rep, "k_ls_pick", captured=1)
    assert cols["grid"] == [n_alloc // 64, 128 // 16, 1] and cols["block"] == [256, 1, 1]
    assert pick["grid"] == [128, 1, 1] and pick["block"] == [256, 1, 1]
    assert _one(report["poly_ls_simt_profile"], "k_ls_pick", captured=0) and _one(report["poly_ls_wide"], "k_ls_cols", captured=1)
    for tag in ("c1_tf32", "c1_simt", "c3_pair_static", "wide_streamed"):          # off by default: not a single launch
        assert not [k for k in report[tag]["kernels"] if "k_ls_" in k], tag


def test_every_launch_is_the_one_the_schedule_announces(report):
    import gmco_cases as gc
    import paper_1904_01567_b200 as g
    wide = gc.make_case("C1", n_cath=24, n_pos=16, counts=(700, 130, 250, 190), n_plans=130, seed_points=9)
    cases = {"c1_tf32": (gc.make_case("C1"), 0, 0), "pair_ring": (gc.make_case("C1", n_plans=256), 0, 0),
             "pair_forced_single": (gc.make_case("C1", n_plans=256), 1, 0),
             "wide_streamed": (wide, 0, 0), "wide_split_main": (wide, 0, 1),
             "c3_pair_static": (gc.make_case("C3"), 0, 0), "pair_both_contractions": (gc.make_case("C1", n_plans=256), 2, 0)}
    names = {0: "k_dose_tcILb1ELb0", 1: "k_dose_tcILb0ELb0", 2: "k_dose_tc_pairILi4ELi6", 3: "k_dose_tc_pairILi0ELi0"}
    for tag, (c, dk, wa) in cases.items():
        q = g.gmco_tc_schedule(c.n_dwell, [s.n_points for s in c.structures], c.n_plans, 148, dk, wa)
        rep = report[tag]
        names[1] = "k_dose_tcILb0ELb1" if wa else "k_dose_tcILb0ELb0"
        dose = _one(rep, names[q["dose_kernel"]])
        grid = [q["n_tiles"], q["segs"], 1] if q["dose_kernel"] >= 2 else [q["segs"], q["n_tiles"], 1]
        assert dose["grid"] == grid and dose["block"] == [320, 1, 1] and dose["smem"] == q["dose_smem_bytes"], tag
        if q["grad_pair"]:                 # gmco_options.dose_kernel = 2: CTA pairs for the gradient contraction as well
            grad = _one(rep, "k_grad_tc_pair")
            assert grad["grid"] == [q["n_tiles"], q["segs"], 1], tag     # (the scenario's later 128-plan call has one tile: k_grad_tc)
            first_grad = [x for x in rep["launches"] if "k_grad_tc" in x["name"]][0]
            assert "k_grad_tc_pair" in first_grad["name"], tag
        else:
            grad = _one(rep, "k_grad_tcILi16")
            assert grad["grid"] == [q["segs"], q["n_tiles"], 1], tag
        assert grad["block"] == [192, 1, 1] and grad["smem"] == q["grad_smem_bytes"], tag
        # the same kernels inside the captured loop body
        assert _one(rep, names[q["dose_kernel"]], captured=1)["smem"] == q["dose_smem_bytes"]
        assert _one(rep, "k_step", captured=1) and _one(rep, "k_loop_cond", captured=1)
        assert not [k for k in rep["kernels"] if "k_simt_grad" in k]          # the tensor route never falls back
    simt = report["c1_simt"]
    assert _one(simt, "k_simt_grad") and not [k for k in simt["kernels"] if "k_dose_tc" in k or "k_grad_tc" in k]
    assert not [k for k in report["a385_falls_to_simt"]["kernels"] if "k_dose_tc" in k]
