"""Builds paper_2311_18482_b200/liblegs.so (all CUDA kernels + the C-ABI of include/legs.h) for sm_100a with nvcc.

In-tree and explicit: `python -m paper_2311_18482_b200.build` (or __graft_entry__.build()). nvcc cross-compiles
without a GPU. Per-file flags: the projection kernel (preprocess.cu) is compiled without FMA contraction and with IEEE
division and square root (rule P-0: its integer outputs must be bit-exact); everything else with default fast
FP32 contraction (project_backward.cu keeps IEEE division and square root)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "liblegs.so")
OBJ = os.path.join(HERE, "build")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-lineinfo", "-std=c++17", "-I", INCLUDE, "-I", CSRC, "-Xcompiler", "-fPIC"]
STRICT_FP = ["--fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false"]
SOURCES = {
    "api.cu": [],
    "preprocess.cu": STRICT_FP,
    "binning.cu": [],
    "forward.cu": [],
    "backward.cu": [],
    "project_backward.cu": ["-prec-div=true", "-prec-sqrt=true"],
    "decode.cu": [],
    "loss.cu": [],
    "loss3.cu": [],
    "peaks.cu": [],
    "quantize.cu": [],
    "smooth.cu": [],
    "optim.cu": ["-prec-div=true", "-prec-sqrt=true"],
    "lerf.cu": [],
    "relevancy_map.cu": [],
    "tile_order.cu": [],
}


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    extra_env = os.environ.get("LEGS_NVCC_FLAGS", "").split()   # measurement builds, e.g. -DLEGS_DECODE_TIMING
    os.makedirs(OBJ, exist_ok=True)
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    headers.append(os.path.join(INCLUDE, "legs.h"))
    objs, procs = [], []
    for src, extra in SOURCES.items():
        path = os.path.join(CSRC, src)
        if not os.path.exists(path):
            continue
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        objs.append(obj)
        if force or _newer(obj, [path] + headers):
            cmd = [nvcc] + ARCH + COMMON + extra + extra_env + (["-Xptxas", "-v"] if verbose else []) + ["-c", path, "-o", obj]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {src}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if force or procs or _newer(LIB, objs):
        subprocess.run([nvcc] + ARCH + ["-shared", "-o", LIB] + objs + ["-lcuda"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
