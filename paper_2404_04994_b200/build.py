"""Build the CUDA library in-tree: paper_2404_04994_b200/libqarray_b200.so (sm_100a only).

    python -m paper_2404_04994_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  --fmad=false: no implicit contraction, every fused multiply-add in the kernels is an
explicit fma() (reading R1 needs bit-identical N_c on both sides).  -lineinfo so ncu's source page maps to the .cu files.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libqarray_b200.so")
OBJ = os.path.join(HERE, "build")
SOURCES = ["qa_api.cu", "qa_kernels_generic.cu", "qa_kernels_walk.cu", "qa_kernels_minplus.cu", "qa_kernels_fused.cu", "qa_kernels_fused_open.cu", "qa_kernels_thermal.cu", "qa_kernels_closed.cu", "qa_kernels_sensor.cu", "qa_kernels_thermal_sp.cu", "qa_kernels_minplus32.cu", "qa_kernels_fused_mid.cu", "qa_static_workspace.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "--fmad=false",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fvisibility=hidden", "-Xptxas", "-v"]


def _deps():
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    files.append(os.path.join(os.path.dirname(HERE), "include", "qarray_b200.h"))
    return files


def _stale():
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    return any(os.path.getmtime(f) > t for f in _deps())


def _compile(src):
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    cmd = ["nvcc", *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(obj + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return OUT
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(_compile, SOURCES))
    cmd = ["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", OUT, *objs, "-Xlinker",
           "--exclude-libs,ALL"]
    if verbose:
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
