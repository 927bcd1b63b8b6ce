"""Builds libetx.so (the C-ABI library of include/etx.h) in-tree with nvcc for sm_100a.

    python -m paper_2407_12119_b200._build [--force] [-v]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libetx.so")
SOURCES = ["etx_api.cu", "k_graph.cu", "k_mlp_simt.cu", "k_mlp_umma.cu", "k_mlp_ws.cu", "k_edge_tma.cu", "k_embed_ws.cu", "k_edge_i8.cu",
           "k_tracks_static.cu", "k_triplet_tracks.cu"]
HEADERS = [os.path.join(CSRC, "etx_internal.h"), os.path.join(CSRC, "umma_common.cuh"), os.path.join(HERE, "..", "include", "etx.h")]
# no fast-math, no FTZ, no implicit contraction: every fp32 op is the one written (R4)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--extended-lambda",
              "-Xcompiler", "-fPIC", "-ftz=false", "-prec-div=true", "-prec-sqrt=true", "-fmad=false"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return "nvcc"


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    objs = [os.path.join(objdir, s.replace(".cu", ".o")) for s in SOURCES]
    todo = [(s, o) for s, o in zip(srcs, objs) if force or _stale(o, [s] + HEADERS)]

    def compile_one(so):
        s, o = so
        cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("ETX_NVCC_EXTRA", "").split(), "-c", s, "-o", o] + (["-Xptxas", "-v"] if verbose else [])
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    if todo:
        with cf.ThreadPoolExecutor(max_workers=len(todo)) as ex:
            for log in ex.map(compile_one, todo):
                if verbose and log:
                    print(log)
    if todo or force or _stale(LIB, objs):
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", tmp, *objs]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
