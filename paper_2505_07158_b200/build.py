"""Builds libvcrypt.so in-tree: nvcc for the sm_100a kernels, g++ for the host subsystem.

Every floating-point translation unit is compiled with -ffp-contract=off (and never -ffast-math): the
chaotic-map arithmetic must be the IEEE binary64 operation sequence written in the source, on every ISA
(DESIGN.md "Bit-exact floating point").  Run as `python -m paper_2505_07158_b200.build [--force]`.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libvcrypt.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
CXX_FLAGS = ["-O3", "-std=c++17", "-fPIC", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
             "-fvisibility=hidden", f"-I{CUDA_HOME}/include"]
# (source, extra flags); derive.cu holds the chaotic-map arithmetic: no FMA contraction
CU_SOURCES = [("kernels.cu", []), ("cipher.cu", []), ("derive.cu", ["-fmad=false"]), ("sha256.cu", []), ("stats.cu", [])]
# (source, extra flags)
CXX_SOURCES = [
    ("vcrypt.cpp", []),
    ("host_sha256.cpp", []),
    ("host_derive.cpp", []),
    ("host_lhcs_scalar.cpp", []),
    ("host_lhcs_avx2.cpp", ["-mavx2", "-mclflushopt"]),
    ("host_lhcs_avx512.cpp", ["-mavx512f", "-mavx512dq", "-mprefer-vector-width=512", "-mclflushopt"]),
]
HEADERS = ["host.hpp", "kernels.cuh", "ptx.cuh", "smem_attr.hpp", "thread_pool.hpp", "host_lhcs_lanes.inc", os.path.join("..", "..", "include", "vcrypt.h")]


def _nvcc() -> str:
    cand = os.path.join(CUDA_HOME, "bin", "nvcc")
    return cand if os.path.exists(cand) else (shutil.which("nvcc") or "nvcc")


def _stale(out: str, deps: list[str]) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def _run(cmd: list[str], log: list[str]):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        sys.stderr.write(log[-1])
        raise RuntimeError("build step failed: " + " ".join(cmd[:3]))


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile (if stale) and return the path of libvcrypt.so."""
    os.makedirs(OBJ, exist_ok=True)
    hdrs = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    log: list[str] = []
    objs = []
    for name, extra in CU_SOURCES:
        cu, cu_o = os.path.join(CSRC, name), os.path.join(OBJ, name.replace(".cu", ".o"))
        if force or _stale(cu_o, [cu] + hdrs):
            _run([_nvcc(), *NVCC_FLAGS, *extra, "-c", cu, "-o", cu_o], log)
        objs.append(cu_o)
    for src, extra in CXX_SOURCES:
        s, o = os.path.join(CSRC, src), os.path.join(OBJ, src.replace(".cpp", ".o"))
        if force or _stale(o, [s] + hdrs):
            _run(["g++", *CXX_FLAGS, *extra, "-c", s, "-o", o], log)
        objs.append(o)
    if force or _stale(LIB, objs):
        tmp = LIB + ".tmp.%d" % os.getpid()
        _run(["g++", "-shared", "-o", tmp, *objs, f"-L{CUDA_HOME}/lib64", "-lcudart_static", "-ldl", "-lrt",
              "-lpthread"], log)
        os.replace(tmp, LIB)
    if verbose:
        sys.stdout.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
