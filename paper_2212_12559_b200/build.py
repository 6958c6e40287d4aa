"""Build step for libcoarseop.so (hand-written sm_100a CUDA behind a C ABI).

`python -m paper_2212_12559_b200.build` or `build_library()`; nvcc cross-compiles without a GPU.
The library is several translation units compiled in parallel (one per kernel family and colour-spin
size Nc, see csrc/internal.h) and linked into one .so, built in-tree (git-ignored) so that it travels
with the repo snapshot to the GPU box.
"""
from __future__ import annotations

import concurrent.futures
import glob
import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
OBJ_DIR = os.path.join(PKG_DIR, "build", "obj")
LIB_PATH = os.path.join(PKG_DIR, "libcoarseop.so")
HEADER = os.path.join(os.path.dirname(PKG_DIR), "include", "coarse_op.h")

NVCC_FLAGS = [
    "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo",
    "-Xcompiler", "-fPIC",
]

NC_SET = (32, 48, 64, 96, 128, 192)        # COARSE_FOR_EACH_NC in csrc/internal.h


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libcoarseop cannot be built (there is no CPU fallback)")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  glob.glob(os.path.join(CSRC, "*.h")) + [HEADER])


def units():
    """(object name, source file, extra defines) of every translation unit."""
    out = [("coarse_op", "coarse_op.cu", []), ("link_map", "link_map.cu", []), ("static_scratch", "static_scratch.cu", [])]
    for fam in ("launch_stream", "launch_stream_mr", "launch_block", "launch_tensor"):
        for nc in NC_SET:
            out.append((f"{fam}_nc{nc}", f"{fam}.cu", [f"-DCOARSE_NC={nc}"]))
    return out


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(s) > t for s in sources())


def _compile(nvcc, name, src, defines, verbose):
    obj = os.path.join(OBJ_DIR, name + ".o")
    extra = os.environ.get("COARSE_EXTRA_NVCC_FLAGS", "").split()      # experiments: -D switches of the kernels
    cmd = [nvcc] + NVCC_FLAGS + defines + extra + (["-Xptxas", "-v"] if verbose else []) + \
          ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    return obj, cmd, res


def build_library(force: bool = False, verbose: bool = False, jobs: int = 0) -> str:
    """Compile csrc/*.cu into libcoarseop.so if it is missing or out of date."""
    if not force and not is_stale():
        return LIB_PATH
    nvcc = _nvcc()
    os.makedirs(OBJ_DIR, exist_ok=True)
    jobs = jobs or max(1, min(len(units()), os.cpu_count() or 1))
    objs = []
    # the biggest units first so that the pool drains evenly
    order = sorted(units(), key=lambda u: (0 if u[1] == "launch_stream.cu" else 1, -int(u[2][0].split("=")[1]) if u[2] else 0))
    with concurrent.futures.ThreadPoolExecutor(max_workers=jobs) as pool:
        futs = [pool.submit(_compile, nvcc, n, s, d, verbose) for n, s, d in order]
        for f in futs:
            obj, cmd, res = f.result()
            if verbose:
                sys.stderr.write(res.stderr)
            if res.returncode != 0:
                raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
            objs.append(obj)
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB_PATH] + sorted(objs)
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
