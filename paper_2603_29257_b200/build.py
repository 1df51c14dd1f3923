"""Build librisp.so (all CUDA sources, sm_100a) in-tree with nvcc.  `python -m paper_2603_29257_b200.build [--force]`."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "librisp.so")
SOURCES = ["gemm.cu", "gemm_tma.cu", "gemm_tc.cu", "gemm_tc_static.cu", "eri_kernels.cu", "linalg.cu", "elementwise.cu", "setup.cu", "matvec.cu", "solve.cu", "solve_tddft.cu", "host_eig.cu", "yardstick.cu", "properties.cu", "api.cu"]
NVCC_FLAGS = ["-std=c++17", "--extended-lambda", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def _newest_source() -> float:
    t = max(os.path.getmtime(os.path.join(HERE, "..", "include", f)) for f in ("risp.h", "risp_debug.h"))
    for f in os.listdir(CSRC):
        t = max(t, os.path.getmtime(os.path.join(CSRC, f)))
    return t


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    hdr_time = max(os.path.getmtime(os.path.join(CSRC, f)) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh")))
    hdr_time = max(hdr_time, os.path.getmtime(os.path.join(HERE, "..", "include", "risp.h")))

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        s = os.path.join(CSRC, src)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) > max(os.path.getmtime(s), hdr_time):
            return obj
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    if not force and os.path.exists(SO) and os.path.getmtime(SO) > _newest_source():
        return SO
    with ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    r = subprocess.run([nvcc, "-shared", "-o", SO] + objs + ["-lcudart", "-lpthread"], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
