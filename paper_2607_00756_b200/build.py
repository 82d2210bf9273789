"""Build libbip.so in-tree with nvcc for sm_100a (no GPU needed: nvcc cross-compiles).

    python -m paper_2607_00756_b200.build [--force] [--verbose] [--tuning]

--tuning compiles with -DBIP_TUNING: only then does the library read the BIP_TUNE_* launch-shape environment variables
(experiments); the shipped build ignores them.

The CUDA runtime is linked statically and nothing links libcuda, so the library loads on a box with
no GPU driver (the CPU test box); cuFFT is the toolkit's shared library, found through an rpath.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libbip.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC = os.path.join(CUDA_HOME, "bin", "nvcc")

SOURCES = ["bip_api.cu", "bip_multislice.cu", "bip_fft.cu", "bip_focal.cu", "bip_recon.cu", "bip_gemm_simt.cu", "bip_gemm_tc.cu", "bip_gemm_sliced.cu", "bip_noalloc.cu", "bip_geometry.cpp"]
COMMON = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          "-Xcompiler", "-fPIC,-fvisibility=hidden,-ffp-contract=off,-Wall,-Wno-unknown-pragmas", "-I", os.path.join(HERE, "..", "include")]


def _stamp(tuning: bool = False) -> str:
    h = hashlib.sha256(b"tuning" if tuning else b"")
    for name in sorted(os.listdir(CSRC)) + ["../../include/bip.h", "../build.py"]:
        with open(os.path.join(CSRC, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False, tuning: bool = False) -> str:
    os.makedirs(BUILD, exist_ok=True)
    stamp_file = os.path.join(BUILD, "stamp")
    stamp = _stamp(tuning)
    if not force and os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return LIB
    if not os.path.exists(NVCC):
        raise RuntimeError(f"nvcc not found at {NVCC}; cannot build libbip.so")

    def compile_one(src: str) -> str:
        obj = os.path.join(BUILD, os.path.splitext(src)[0] + ".o")
        cmd = [NVCC, *COMMON, *(["-DBIP_TUNING"] if tuning else []), "-x", "cu" if src.endswith(".cu") else "c++", "-c",
               os.path.join(CSRC, src), "-o", obj]
        if verbose and src.endswith(".cu"):
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    link = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs,
            "-L", os.path.join(CUDA_HOME, "lib64"), "-lcufft", "-cudart", "static",
            "-Xlinker", "--exclude-libs=ALL", "-Xlinker", "-rpath=" + os.path.join(CUDA_HOME, "lib64"),
            "-lpthread", "-ldl", "-lrt"]
    r = subprocess.run(link, capture_output=True, text=True)
    if verbose or r.returncode:
        sys.stderr.write(" ".join(link) + "\n" + r.stdout + r.stderr)
    if r.returncode:
        raise RuntimeError("link of libbip.so failed")
    with open(stamp_file, "w") as f:
        f.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, tuning="--tuning" in sys.argv))
