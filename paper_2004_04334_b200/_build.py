"""In-tree build of libpixreco.so (nvcc, sm_100a only).  No JIT cache: the .so sits next to the
package so that it travels to the GPU box with the repo snapshot."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libpixreco.so")
SOURCES = ["pixreco_api.cu", "pool.cpp"]
DEPS = SOURCES + ["kernels.cuh", "common.cuh", "k_unpack.cuh", "k_cluster.cuh", "k_finalize.cuh", "k_chain.cuh", "k_bucket.cuh", "chain_api.cuh", "static_api.cuh", "pool.hpp"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, d) for d in DEPS] + [os.path.join(INCLUDE, "pixreco.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-I", INCLUDE, "-o", tmp,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


# The multi-threaded C++ client of the C ABI (include/pixreco_driver.h): host-only, links against libpixreco.so.
DRIVER_LIB = os.path.join(_HERE, "libpixreco_driver.so")
DRIVER_SRC = os.path.join(CSRC, "stream_driver.cpp")


def build_driver(force: bool = False) -> str:
    build()
    deps = [DRIVER_SRC, os.path.join(INCLUDE, "pixreco_driver.h"), os.path.join(INCLUDE, "pixreco.h")]
    if force or not os.path.exists(DRIVER_LIB) or any(os.path.getmtime(d) > os.path.getmtime(DRIVER_LIB) for d in deps):
        tmp = DRIVER_LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-I", INCLUDE, "-o", tmp, DRIVER_SRC,
                               "-L", _HERE, "-l:libpixreco.so", "-Wl,-rpath,$ORIGIN"])
        os.replace(tmp, DRIVER_LIB)
    return DRIVER_LIB
