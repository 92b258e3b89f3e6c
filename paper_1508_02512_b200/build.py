"""In-tree build of libqmcfeyn.so (C-ABI library: host decomposer + sm_100a CUDA kernels).

    python -m paper_1508_02512_b200.build [--force]

nvcc cross-compiles for sm_100a without a GPU.  One object per translation unit, compiled in parallel,
then linked with a static CUDA runtime so that the library loads on a box without a driver-side toolkit.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libqmcfeyn.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

SOURCES = ["qmc_prepare.cpp", "qmc_flops.cpp", "qmc_image4.cpp", "qmc_image3.cpp", "qmc_cbc.cpp", "qmc_api.cu", "qmc_dispatch.cu"] + [f"qmc_inst_d{d}.cu" for d in range(1, 7)] + [f"qmc4_inst_d{d}.cu" for d in range(1, 7)] + [f"qmc5_inst_d{d}.cu" for d in range(1, 7)]
HEADERS = ["qmc_tables.h", "qmc_launch.h", "qmc_kernels.cuh", "qmc_inst.cuh", "qmc_fold.cuh", "qmc_kernels4.cuh", "qmc_inst4.cuh", "qmc_kernels5.cuh", "qmc_inst5.cuh", "qmc_bpe.h", os.path.join("..", "..", "include", "qmc_feynman.h")]


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _compile(src: str, force: bool) -> str:
    s = os.path.join(CSRC, src)
    o = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    if not force and os.path.exists(o) and os.path.getmtime(o) > max(os.path.getmtime(s), _newest_header()):
        return o
    cmd = [NVCC] + ARCH + FLAGS + ["-c", s, "-o", o]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(o + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {src}:\n{r.stderr[-4000:]}")
    return o


def build(force: bool = False, jobs: int | None = None) -> str:
    os.makedirs(OBJ, exist_ok=True)
    jobs = jobs or min(len(SOURCES), os.cpu_count() or 4)
    with cf.ThreadPoolExecutor(max_workers=jobs) as ex:
        objs = list(ex.map(lambda s: _compile(s, force), SOURCES))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        cmd = [NVCC] + ARCH + ["-shared", "-cudart", "static", "-o", LIB] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stderr[-4000:]}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
