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
    link = ["g++", "-shared", "-o", str(lib), *objs]
    if sanitize:
        link += ["-fsanitize=address,undefined"]
    subprocess.run(link, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize="--asan" in sys.argv))
