"""In-tree build of the C-ABI CUDA library (liblofar_moon.so) for sm_100a.

`python -m paper_1612_06592_b200.build [--force] [--verbose]` or `build()` from Python.
nvcc cross-compiles without a GPU; the .so sits next to this file so that it travels with the tree.

Ablation builds (the measurements DESIGN.md section 8 quotes): `--define NAME [--define NAME ...] --out PATH` compiles a
variant with -DNAME into PATH (objects under build/<names>/); run it with LOFAR_MOON_LIB=PATH, which the binding
honours. Switches: LOFAR_FIR_PACKED (synthesis FIR with packed FFMA2 instead of scalar FFMA), LOFAR_FFT_SCALAR (the
transform's complex adds / butterflies as scalar pairs instead of FADD2 / FFMA2), LOFAR_ST_PLAIN (series stores with
the default cache policy instead of st.global.cs), LOFAR_ABLATE_STORES
(inverse PPF without its series stores), LOFAR_ABLATE_FIR (no FIR arithmetic), LOFAR_ABLATE_FFT (no transform
arithmetic). Ablated variants compute wrong results by design; they exist to attribute time. Extra nvcc flags for an
experiment go in the environment variable LOFAR_NVCC_FLAGS (e.g. "-Xptxas --allow-expensive-optimizations=true": measured, no
effect).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblofar_moon.so")
SOURCES = ["api.cu", "beamform.cu", "beamform_tc.cu", "ippf.cu", "trigger.cu", "lsmr.cu", "dedisp.cu", "noalloc.cu"]
HEADERS = ["plan.h", "fft_math.cuh", "fft_warp.cuh", os.path.join(ROOT, "include", "lofar_moon.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-fvisibility=hidden", "-DLOFAR_MOON_BUILD",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), out: str | None = None) -> str:
    if not defines and out is None and not force and not _stale():
        return LIB
    objdir = os.path.join(HERE, "build", *(["_".join(defines)] if defines else []))
    os.makedirs(objdir, exist_ok=True)
    lib = out or LIB
    procs = []
    objs = []
    for s in SOURCES:
        o = os.path.join(objdir, s.replace(".cu", ".o"))
        objs.append(o)
        cmd = [NVCC, *FLAGS, *os.environ.get("LOFAR_NVCC_FLAGS", "").split(), *[f"-D{d}" for d in defines], "-c",
               os.path.join(CSRC, s), "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for s, p in procs:
        log, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {s} (exit {p.returncode})\n{log}\n")
        failed = failed or p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, "-shared", "-o", tmp, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    argv = sys.argv[1:]
    defs = [argv[i + 1] for i, a in enumerate(argv) if a == "--define"]
    outs = [argv[i + 1] for i, a in enumerate(argv) if a == "--out"]
    print(build(force="--force" in argv, verbose="--verbose" in argv, defines=tuple(defs), out=outs[0] if outs else None))
