"""Build libpic_b200.so in-tree with nvcc for sm_100a (cross-compiles without a
GPU).  ``python -m paper_2303_12873_b200.build`` or ``build_library()``."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpic_b200.so")
SOURCES = ["pic_api.cu", "yee.cu", "particles_global.cu", "particles_tile.cu", "sort.cu", "bricks.cu", "noalloc.cu"]
# measurement probes (the only code that calls cudaMalloc): a library of their own, include/pic_probes.h
PROBE_SOURCES = ["peaks.cu"]
PROBE_LIB = os.path.join(HERE, "libpic_probes.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps_mtime() -> float:
    t = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for fn in os.listdir(root):
            if fn.endswith((".h", ".cuh")):
                t = max(t, os.path.getmtime(os.path.join(root, fn)))
    return t


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ and link libpic_b200.so (the product) and libpic_probes.so (measurement probes).
    Returns the path of the former."""
    os.makedirs(OBJ, exist_ok=True)
    hdr_t = _deps_mtime()
    nvcc = _nvcc()
    jobs = []
    for src in SOURCES + PROBE_SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_t):
            jobs.append((s, o))

    def compile_one(job):
        s, o = job
        r = subprocess.run([nvcc, *NVCC_FLAGS, "-c", s, "-o", o], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s\n%s" % (s, r.stdout, r.stderr))
        with open(o + ".ptxas.txt", "w") as fh:      # registers / spills / shared memory per kernel
            fh.write(r.stderr)
        if verbose:
            sys.stderr.write(r.stderr)
        return o

    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        list(ex.map(compile_one, jobs))
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if jobs or force or not os.path.exists(LIB):
        tmp = LIB + ".tmp%d" % os.getpid()
        r = subprocess.run([nvcc, "-shared", "-o", tmp, *objs, "-lcudart"], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
        os.replace(tmp, LIB)
    pobjs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in PROBE_SOURCES]
    if jobs or force or not os.path.exists(PROBE_LIB):
        tmp = PROBE_LIB + ".tmp%d" % os.getpid()
        r = subprocess.run([nvcc, "-shared", "-o", tmp, *pobjs, "-lcudart"], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
        os.replace(tmp, PROBE_LIB)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
