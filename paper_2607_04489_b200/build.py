"""Builds libeiger.so in-tree with nvcc for sm_100a (no torch involved).

    python -m paper_2607_04489_b200.build [--force] [--verbose] [--define NAME=VALUE ...] [--out FILE]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libeiger.so")
SOURCES = ["api.cu", "profile.cu", "aggregate.cu", "hashagg.cu", "hashagg_i32.cu", "hashagg_i64.cu", "hashagg_pre.cu", "partition.cu", "sortagg.cu", "dictenc.cu", "splitagg.cu", "probe.cu", "noalloc.cu"]
HEADERS = ["dev.cuh", "rows.cuh", "ring.cuh", "scatter.cuh", "hashagg.cuh", "internal.h", os.path.join("..", "..", "include", "eiger.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-Xptxas", "-warn-spills"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, defines: tuple = (), out: str | None = None) -> str:
    """defines / out: an experiment build (e.g. defines=("EIGER_STREAM_L2_HINT=0",)) into another file; always rebuilt."""
    if out or defines:
        return _build(verbose, tuple(defines), out or LIB, os.path.join(HERE, "build", "x_" + "_".join(d.replace("=", "") for d in defines)))
    if not force and not _stale():
        return LIB
    return _build(verbose, (), LIB, os.path.join(HERE, "build"))


def _build(verbose: bool, defines: tuple, lib: str, objdir: str) -> str:
    nvcc = _nvcc()
    os.makedirs(objdir, exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *[f"-D{d}" for d in defines], *(["-Xptxas", "-v"] if verbose else []), "-c",
               os.path.join(CSRC, src), "-o", obj]
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    for src, obj, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
        if verbose or "warning" in out.lower():
            sys.stderr.write(out)
        objs.append(obj)
    subprocess.check_call([nvcc, "-shared", "-o", lib, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    return lib


if __name__ == "__main__":
    # --define NAME=VALUE (repeatable) and --out FILE: an experiment build next to the ordinary one
    defs = tuple(sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define")
    outs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--out"]
    print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv, defines=defs, out=outs[0] if outs else None))
