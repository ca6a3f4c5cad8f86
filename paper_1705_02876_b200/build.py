"""Build libkf_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1705_02876_b200.build [--force]

The shared library is the product's C ABI (include/kf_b200.h).  It is git-ignored but travels to
the GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libkf_b200.so")
SOURCES = ["kf_api.cu", "kf_fit.cu", "kf_smooth.cu", "kf_host.cu", "kf_bin.cu", "kf_score.cu", "kf_comb.cu", "kf_peak.cu"]
HEADERS = ["kf_math.cuh", "kf_pair.cuh", "kf_rts.cuh", "kf_tma.cuh", "kf_internal.h", "kf_score_common.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "kf_b200.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines: list[str] | None = None, out: str | None = None) -> str:
    """One nvcc process per translation unit (they run side by side), then one link step.
    defines / out: build a tuning variant (-DNAME=VALUE ...) into another file (kernel experiments; the binding
    loads it when KF_B200_LIB points there)."""
    if out is None and not defines and not force and not needs_build():
        return LIB
    lib = out or LIB
    objdir = os.path.join(HERE, "build") if out is None else out + ".obj"
    os.makedirs(objdir, exist_ok=True)
    flags = NVCC_FLAGS[:-2] + (["-Xptxas", "-v"] if verbose else []) + ["-D" + d for d in (defines or [])]   # (-cudart static belongs to the link step)
    procs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        procs.append((src, obj, subprocess.Popen([_nvcc()] + flags + ["-c", "-o", obj, os.path.join(CSRC, src)])))
    failed = [src for src, _, p in procs if p.wait() != 0]
    if failed:
        raise subprocess.CalledProcessError(1, "nvcc -c " + " ".join(failed))
    subprocess.check_call([_nvcc()] + NVCC_FLAGS + ["-shared", "-o", lib] + [obj for _, obj, _ in procs])
    return lib


if __name__ == "__main__":
    defs = [a[2:] for a in sys.argv[1:] if a.startswith("-D")]
    outs = [a[6:] for a in sys.argv[1:] if a.startswith("--out=")]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=defs, out=outs[0] if outs else None))
