"""Builds paper_2404_14401_b200/libgpe.so with nvcc for sm_100a (in-tree, no JIT cache).

One translation unit per (dtype, N) for the FFT passes plus gpe_api.cu; compiled in parallel
and linked into one shared library with a C ABI (include/gpe.h).  Cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libgpe.so")
SIZES = (64, 128, 256, 512, 1024, 2048)
SIZES3 = (64, 128, 256, 512, 1024)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _sources():
    out = []
    for f in sorted(os.listdir(CSRC)):
        out.append(os.path.join(CSRC, f))
    out.append(os.path.join(os.path.dirname(HERE), "include", "gpe.h"))
    out.append(os.path.abspath(__file__))
    return out


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(s) <= t for s in _sources())


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False, ptxas_v: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = (["-Xptxas", "-v"] if ptxas_v else []) + os.environ.get("GPE_NVCC_FLAGS", "").split()
    jobs = []
    objs = []
    for tag, typ in (("f", "float"), ("d", "double")):
        for n in SIZES:
            o = os.path.join(OBJ, f"inst_{tag}_{n}.o")
            objs.append(o)
            jobs.append([nvcc, *NVCC_FLAGS, *extra, f"-DGPE_T={typ}", f"-DGPE_N={n}", f"-DGPE_TAG={tag}",
                         "-c", os.path.join(CSRC, "gpe_inst.cu"), "-o", o])
    for tag, typ in (("f", "float"), ("d", "double")):   # the 3-D passes (gpe3_kernels.cuh)
        for n in SIZES3:
            o = os.path.join(OBJ, f"inst3_{tag}_{n}.o")
            objs.append(o)
            jobs.append([nvcc, *NVCC_FLAGS, *extra, f"-DGPE_T={typ}", f"-DGPE_N={n}", f"-DGPE_TAG={tag}",
                         "-c", os.path.join(CSRC, "gpe3_inst.cu"), "-o", o])
    o = os.path.join(OBJ, "api3.o")
    objs.append(o)
    jobs.append([nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, "gpe3_api.cu"), "-o", o])
    o = os.path.join(OBJ, "api.o")
    objs.append(o)
    jobs.append([nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, "gpe_api.cu"), "-o", o])
    o = os.path.join(OBJ, "noalloc.o")
    objs.append(o)
    jobs.append([nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, "gpe_noalloc.cu"), "-o", o])
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        logs = list(ex.map(_run, jobs))
    if verbose or ptxas_v:
        for j, l in zip(jobs, logs):
            if l.strip():
                print(" ".join(j[-3:]), "\n", l, file=sys.stderr)
    _run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp", *objs])
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, ptxas_v="--ptxas-v" in sys.argv))
