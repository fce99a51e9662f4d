"""Build libfredec_b200.so (the C-ABI library of include/fredec.h) and libfredec_bench.so (the FP64 roofline
probes of include/fredec_bench.h, for bench.py) in-tree with nvcc for sm_100a.  `python -m paper_1309_0100_b200.build [--force]`.  nvcc cross-compiles without a GPU.

Measurement builds: `python -m paper_1309_0100_b200.build --variant NAME -DMACRO[=V] ...` compiles the
same sources with extra macros (the FREDEC_EXP_* switches documented where they appear in csrc/) into
libfredec_b200.NAME.so beside the product library; `FREDEC_LIB=<path>` makes the binding load it.  Such a
library is for A/B timings only (profiles/r2_experiments.md): some switches give wrong results."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "libfredec_b200.so")
SOURCES = ["fredec_api.cu", "prep_kernel.cu", "scan_mma_kernel.cu", "topk_kernel.cu", "topk_noalloc.cu", "stat_kernel.cu", "trig_kernel.cu", "subset_kernel.cu", "refine_kernel.cu"]
# the FP64 roofline probes of include/fredec_bench.h: a library of their own, loaded by bench.py only
BENCH_LIB = os.path.join(PKG, "libfredec_bench.so")
BENCH_SOURCES = ["bench_api.cu", "peak_kernel.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _newest_header() -> float:
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]
    hs += [os.path.join(ROOT, "include", h) for h in os.listdir(os.path.join(ROOT, "include")) if h.endswith(".h")]
    hs.append(os.path.abspath(__file__))
    return max(os.path.getmtime(h) for h in hs)


def build(force: bool = False, verbose: bool = False, variant: str = "", defines=()) -> str:
    obj_dir = OBJ if not variant else os.path.join(OBJ, "variant_" + variant)
    lib_path = LIB if not variant else os.path.join(PKG, f"libfredec_b200.{variant}.so")
    os.makedirs(obj_dir, exist_ok=True)
    nvcc = _nvcc()
    hdr = _newest_header()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(obj_dir, src.replace(".cu", ".o"))
        if force or variant or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr):
            jobs.append([nvcc, *NVCC_FLAGS, *defines, *(["-Xptxas", "-v"] if verbose else []), "-c", s, "-o", o])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            for out in ex.map(run, jobs):
                if verbose and out:
                    print(out, file=sys.stderr)
    objs = [os.path.join(obj_dir, s.replace(".cu", ".o")) for s in SOURCES]
    if jobs or not os.path.exists(lib_path):
        run([nvcc, "-shared", "-o", lib_path, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    if not variant:
        bench_objs, stale = [], False
        for src in BENCH_SOURCES:
            s = os.path.join(CSRC, src)
            o = os.path.join(obj_dir, src.replace(".cu", ".o"))
            bench_objs.append(o)
            if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr):
                run([nvcc, *NVCC_FLAGS, "-c", s, "-o", o])
                stale = True
        if stale or not os.path.exists(BENCH_LIB):
            run([nvcc, "-shared", "-o", BENCH_LIB, *bench_objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    return lib_path


if __name__ == "__main__":
    _variant = sys.argv[sys.argv.index("--variant") + 1] if "--variant" in sys.argv else ""
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, variant=_variant,
                defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
