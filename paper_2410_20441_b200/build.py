"""Build libdr.so (hand-written sm_100a CUDA kernels + C ABI) in-tree with nvcc.

    python -m paper_2410_20441_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdr.so")
SOURCES = ["dr_api.cu", "dr_static.cu"]      # dr_static.cu: dr_avg_stress_static, its own translation unit
HEADERS = ["dr_layout.cuh", "dr_kernels_aux.cuh", "dr_kernels_split.cuh", "dr_kernels_fused.cuh", "dr_kernels_tma.cuh", "dr_kernels_tb2.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def source_hash():
    """sha256 (first 16 hex digits) of the CUDA kernel sources (csrc/*.cuh): identifies the kernels a profile under
    profiles/ was taken with (bench.py emits roofline.traffic only for a matching hash).  The host file dr_api.cu and the
    public header are left out on purpose: they launch the kernels but do not change what a launch moves."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted(HEADERS):
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "dr.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libdr.so")
    with open(os.path.join(HERE, "libdr.ptxas.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    if "--hash" in sys.argv:
        print(source_hash())
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
