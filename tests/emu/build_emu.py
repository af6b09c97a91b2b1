"""Build tests/emu/_build/libgmco_emu.so: libgmco's SOURCE compiled for the host (TEST INFRASTRUCTURE ONLY).

Every csrc/*.cu file is rewritten by three textual rules and compiled with g++ against emu_core.h / emu_ptx.h /
emu_runtime.cc (a fiber-per-thread model of CUDA's SIMT execution with software models of mbarriers, TMA and tcgen05):

  1. `#include "gmco_ptx.cuh"`  ->  `#include "emu_ptx.h"`  (the PTX layer is the one seam, see csrc/gmco_ptx.cuh)
  2. `K<<<grid, block, smem, stream>>>(args)`  ->  `emu::Launch(grid, block, smem, stream)[.cluster(n)].run("K", K, args)`
     (n from the kernel's __cluster_dims__)
  3. `extern __shared__ [__align__(n)] T name[];`  ->  `T* name = (T*)emu::dyn_smem_ptr();`

Nothing else of the product source is touched, so what runs is the kernels' own control flow, index arithmetic,
descriptor construction and barrier protocol.  The product never builds, links or loads any of this.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
ROOT = HERE.parents[1]
CSRC = ROOT / "paper_1904_01567_b200" / "csrc"
OUT = HERE / "_build"
LIB = OUT / "libgmco_emu.so"
CUDA_INC = Path(os.environ.get("CUDA_HOME", "/usr/local/cuda")) / "include"

LAUNCH = re.compile(r"([A-Za-z_]\w*(?:<[^<>;()]*>)?)\s*<<<(.*?)>>>\s*\(", re.S)
EXT_SHARED = re.compile(r"extern\s+__shared__\s+(?:__align__\(\s*\d+\s*\)\s+)?([A-Za-z_][\w ]*?)\s+(\w+)\s*\[\s*\]\s*;")
CLUSTER = re.compile(r"__cluster_dims__\(\s*(\d+)\s*,\s*1\s*,\s*1\s*\)[^;{]*?\b(k_\w+)\s*\(", re.S)


def transform(text: str) -> str:
    clusters = {name: int(n) for n, name in CLUSTER.findall(text)}
    text = text.replace('#include "gmco_ptx.cuh"', '#include "emu_ptx.h"')

    def launch(m: re.Match) -> str:
        kernel, cfg = m.group(1), m.group(2)
        base = kernel.split("<")[0]
        cl = f".cluster({clusters[base]})" if base in clusters else ""
        return f'emu::Launch({cfg}){cl}.run("{kernel}", {kernel}, '

    text, n_launch = LAUNCH.subn(launch, text)
    # a launch without arguments would leave `run("K", K, )`
    text = re.sub(r'(\.run\("[^"]*", [^,()]+(?:<[^<>;()]*>)?), \)', r"\1)", text)
    text = EXT_SHARED.sub(lambda m: f"{m.group(1)}* {m.group(2)} = ({m.group(1)}*)emu::dyn_smem_ptr();", text)
    text = re.sub(r"\b__noinline__\b", "__attribute__((noinline))", text)     # (libstdc++ uses the bare word as an attribute name)
    assert "<<<" not in text and "extern __shared__" not in text, "a launch or a dynamic shared array was not rewritten"
    return '#include "emu_core.h"\n' + text


def build(force: bool = False, sanitize: bool = False) -> Path:
    """Builds are serialised by a lock file: pytest-xdist workers and concurrent sessions may all ask for the library."""
    import fcntl
    OUT.mkdir(parents=True, exist_ok=True)
    with open(OUT / ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        return _build(force, sanitize)


def _build(force: bool, sanitize: bool) -> Path:
    lib = OUT / ("libgmco_emu_asan.so" if sanitize else "libgmco_emu.so")
    srcs = sorted(CSRC.glob("*.cu"))
    deps = srcs + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + [ROOT / "include" / "gmco.h"] + \
        [HERE / n for n in ("emu_core.h", "emu_ptx.h", "emu_runtime.cc", "build_emu.py")]
    if not force and lib.exists() and all(d.stat().st_mtime <= lib.stat().st_mtime for d in deps):
        return lib
    gen = OUT / "gen"
    gen.mkdir(parents=True, exist_ok=True)
    flags = ["-std=c++17", "-O2", "-g", "-fPIC", "-mfma", "-mavx2", "-fvisibility=hidden", "-w",
             "-I", str(HERE), "-I", str(CSRC), "-I", str(ROOT / "include"), "-I", str(CUDA_INC), "-DGMCO_EMULATED=1"]
    if sanitize:
        flags += ["-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-O1"]
    tag = "asan" if sanitize else "plain"
    procs, objs = [], []
    for src in srcs:
        cc = gen / (src.stem + ".cc")
        cc.write_text(transform(src.read_text()))
        obj = gen / f"{src.stem}.{tag}.o"
        objs.append(str(obj))
        procs.append((src.name, subprocess.Popen(["g++", *flags, "-c", str(cc), "-o", str(obj)],
                                                 stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    obj = gen / f"emu_runtime.{tag}.o"
    objs.append(str(obj))
    procs.append(("emu_runtime.cc", subprocess.Popen(["g++", *flags, "-c", str(HERE / "emu_runtime.cc"), "-o", str(obj)],
                                                     stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for name, p in procs:
        out, _ = p.communicate()
        if p.returncode:
            sys.stderr.write(f"---- {name}\n{out[-6000:]}\n")
            failed = True
    if failed:
        raise RuntimeError("emulation build failed")
    tmp = lib.with_suffix(f".{os.getpid()}.tmp")
    link = ["g++", "-shared", "-o", str(tmp), *objs]
    if sanitize:
        link += ["-fsanitize=address,undefined"]
    subprocess.run(link, check=True)
    os.replace(tmp, lib)                                   # processes that have the old library open keep it
    return lib


# ---- mutants: the emulation must notice planted protocol and indexing errors (tests/test_emu_mutants.py) ----------------
# name -> (file, text to find, replacement, occurrences expected)
MUTANTS = {
    # producer refills a ring slot without waiting for the commit of the MMAs that read it
    "producer_skips_empty_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait1_addr(w, smem_u32(empty + st), ph ^ 1, DEVERR_W_EMPTY));", "", 3),
    # MMAs issued before the TMA bytes of their operands have landed
    "issuer_skips_full_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait1_addr(w, full0 + 8 * st, ph, DEVERR_W_FULL));", "", 2),
    # gradient MMAs issued before the converter warps have split the R tile (and before it has landed)
    "grad_issuer_skips_conv_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait1_addr(w, conv0 + 8 * st, ph, DEVERR_W_CONV));", "", 1),
    # epilogue reads the accumulator without waiting for the chunk's last commit
    "epilogue_skips_acc_full_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait(w, acc_full + b, use & 1, DEVERR_W_ACC_FULL));", "", 2),
    # issuer overwrites the accumulator without waiting for the epilogue to hand it back
    "issuer_skips_acc_empty_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait1_addr(w, smem_u32(acc_empty + b), (use & 1) ^ 1, DEVERR_W_ACC_EMPTY));", "", 1),
    # the epilogue hands the accumulator back before it has read it
    "accumulator_handed_back_too_early": ("kernels_tc.cu", "        tmem_ld32(t_main, v[0]);\n        tmem_ld32(t_main + 32, v[1]);\n        if (a.sep_corr) {",
                                          "        mbar_arrive(acc_empty + b);\n        tmem_ld32(t_main, v[0]);\n        tmem_ld32(t_main + 32, v[1]);\n        if (a.sep_corr) {", 1),
    # the host launches 4 KB less dynamic shared memory than the kernel's carve-up needs (caught by the kernel's self-check)
    "host_smem_too_small": ("tc_layout.h", "t.dose_smem = fixed + t.dose_stages * probe.stage_bytes;", "t.dose_smem = fixed + t.dose_stages * probe.stage_bytes - 4096;", 1),
    # ... and the same with the self-check gone: the emulated hardware's window check is what is left
    "host_smem_too_small_unchecked": ("*", None, None, 0),
    # producer's ring phase never flips: the second trip round the ring waits for ever -> bounded wait -> error word
    "producer_phase_never_flips": ("kernels_tc.cu", "if (++st == a.n_stage) { st = 0; ph ^= 1; }", "if (++st == a.n_stage) { st = 0; }", 5),
    # TMEM is never given back
    "tmem_never_freed": ("kernels_tc.cu", "tc_fence_after(); tmem_dealloc(tmem, 512); }", "tc_fence_after(); }", 2),
    # the D slab of the wrong chunk is loaded (index error: wrong numbers, nothing else)
    "wrong_chunk_loaded": ("kernels_tc.cu", "tma_load_3d(lo ? &tmD_lo : &tmD_hi, dst, full + st, 0, c * kPC, g, polD);", "tma_load_3d(lo ? &tmD_lo : &tmD_hi, dst, full + st, 0, (c + (c & 1)) * kPC, g, polD);", 1),
    # a K-step of the main product uses the wrong 32 B of the swizzled row
    "wrong_k_step_descriptor": ("kernels_tc.cu", "mma_ts2(acc, thi + 8 * j, bd + 2 * j, dhi, idesc, 1);", "mma_ts2(acc, thi + 8 * j, bd + 2 * (j ^ 1), dhi, idesc, 1);", 1),
    # pair gradient kernel: the converters split the R tile without waiting for it (and the D halves) to land
    "gpair_converter_skips_full_wait": ("kernels_tc.cu", "GMCO_WAIT(mbar_wait(w, full + st, ph, DEVERR_W_FULL));   // this CTA's R tile AND its D halves have landed", "", 1),
    # pair gradient kernel: the peer CTA loads the leader's half of the dwell groups (index error)
    "gpair_peer_loads_wrong_half": ("kernels_tc.cu", "tma_load_3d(&tmD_hi, dst + 2 * kRBytes, full + st, 0, s * PS, rank * Gh, polD);", "tma_load_3d(&tmD_hi, dst + 2 * kRBytes, full + st, 0, s * PS, 0, polD);", 1),
    # k_step pushes the history pair without waiting for the staged copies it overwrites
    "step_skips_history_wait": ("kernels_lbfgs.cu", "      hist_wait();                                           // the staged copy of slot hh is about to be replaced\n", "", 1),
}


def build_mutant(name: str) -> Path:
    """libgmco_emu with one planted error.  Only the mutated translation units are recompiled."""
    import fcntl
    plain = build()
    with open(OUT / f".lock_{name}", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        return _build_mutant(name, plain)


def _build_mutant(name: str, plain: Path) -> Path:
    lib = OUT / f"libgmco_emu_mut_{name}.so"
    if lib.exists() and lib.stat().st_mtime >= plain.stat().st_mtime and lib.stat().st_mtime >= Path(__file__).stat().st_mtime:
        return lib
    gen = OUT / "gen" / f"mut_{name}"
    gen.mkdir(parents=True, exist_ok=True)
    edits = []
    if name == "host_smem_too_small_unchecked":
        edits = [MUTANTS["host_smem_too_small"][:4],
                 ("kernels_tc.cu", "const bool smem_ok = pad + (uint32_t)smem_end <= dynamic_smem_size(), tmem_ok", "const bool smem_ok = true, tmem_ok", 1)]
    else:
        edits = [MUTANTS[name]]
    texts = {}
    for fname, old, new, count in edits:
        text = texts.get(fname) or (CSRC / fname).read_text()
        assert text.count(old) == count, f"mutant {name}: expected {count} occurrences of the target in {fname}, found {text.count(old)}"
        texts[fname] = text.replace(old, new)
    # a mutated header reaches every translation unit that includes it: put it first on the include path
    flags = ["-std=c++17", "-O2", "-g", "-fPIC", "-mfma", "-mavx2", "-fvisibility=hidden", "-w",
             "-I", str(gen), "-I", str(HERE), "-I", str(CSRC), "-I", str(ROOT / "include"), "-I", str(CUDA_INC), "-DGMCO_EMULATED=1"]
    headers = [f for f in texts if not f.endswith(".cu")]
    for f in headers:
        (gen / f).write_text(texts[f])
    redo = [s for s in sorted(CSRC.glob("*.cu")) if s.name in texts or (headers and any(f'"{h}"' in s.read_text() for h in headers))]
    objs, procs = [], []
    for src in sorted(CSRC.glob("*.cu")):
        if src in redo:
            cc = gen / (src.stem + ".cc")
            text = texts.get(src.name) or src.read_text()
            if headers:                                   # quote-includes look beside the including file first: the copy is in gen
                pass
            cc.write_text(transform(text))
            obj = gen / f"{src.stem}.o"
            procs.append(subprocess.Popen(["g++", *flags, "-c", str(cc), "-o", str(obj)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
            objs.append(str(obj))
        else:
            objs.append(str(OUT / "gen" / f"{src.stem}.plain.o"))
    objs.append(str(OUT / "gen" / "emu_runtime.plain.o"))
    for p in procs:
        out, _ = p.communicate()
        if p.returncode:
            raise RuntimeError(f"mutant {name} does not compile:\n{out[-3000:]}")
    subprocess.run(["g++", "-shared", "-o", str(lib), *objs], check=True)
    return lib


if __name__ == "__main__":
    if len(sys.argv) > 2 and sys.argv[1] == "--mutant":
        print(build_mutant(sys.argv[2]))
    else:
        print(build(force="--force" in sys.argv, sanitize="--asan" in sys.argv))
