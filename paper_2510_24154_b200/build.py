"""Build libaepid.so (the C-ABI of include/aepid.h) in-tree with nvcc for sm_100a.

    python -m paper_2510_24154_b200.build [--force]

nvcc cross-compiles without a GPU.  The CUDA runtime is linked statically, so the library's
only run-time dependency is the driver (libcuda).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libaepid.so")
SOURCES = ["transport.cu", "postpass.cu", "analysis.cu", "api.cu"]
HEADERS = [os.path.join(CSRC, "params.h"), os.path.join(os.path.dirname(HERE), "include", "aepid.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]
# The transport kernel is bound by instruction fetch: approximate division / square root keep its SASS small.
EXTRA_FLAGS = {"transport.cu": ["-prec-div=false", "-prec-sqrt=false", "-ftz=true"]}


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    objs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = ([nvcc()] + NVCC_FLAGS + EXTRA_FLAGS.get(s, []) + (["-Xptxas", "-v"] if verbose else [])
               + ["-c", os.path.join(CSRC, s), "-o", o])
        subprocess.check_call(cmd)
        objs.append(o)
    subprocess.check_call([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"])
    return LIB


LIB_CHECKED = os.path.join(HERE, "libaepid_checked.so")


def build_checked(force=False):
    """The same library with the transport kernel compiled -DAEPID_CHECKED (index and queue-protocol checks inside the kernel,
    csrc/transport.cu); used by tests/test_gpu_checked_build.py through the AEPID_LIBRARY environment variable."""
    build(force=force)
    src = os.path.join(CSRC, "transport.cu")
    if not force and os.path.exists(LIB_CHECKED) and all(os.path.getmtime(d) <= os.path.getmtime(LIB_CHECKED) for d in [src, LIB] + HEADERS):
        return LIB_CHECKED
    o = os.path.join(CSRC, "transport_checked.o")
    subprocess.check_call([nvcc()] + NVCC_FLAGS + EXTRA_FLAGS["transport.cu"] + ["-DAEPID_CHECKED", "-c", src, "-o", o])
    objs = [o] + [os.path.join(CSRC, s.replace(".cu", ".o")) for s in SOURCES if s != "transport.cu"]
    subprocess.check_call([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB_CHECKED] + objs + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"])
    return LIB_CHECKED


def build_variant(name, flags, force=False):
    """libaepid_<name>.so: the library with transport.cu compiled with extra flags (e.g. the analysis build -DAEPID_PHASE_CLOCK of
    phase_clocks.py); the other objects are shared with the product build."""
    build()
    lib = os.path.join(HERE, "libaepid_%s.so" % name)
    src = os.path.join(CSRC, "transport.cu")
    if not force and os.path.exists(lib) and all(os.path.getmtime(d) <= os.path.getmtime(lib) for d in [src, LIB] + HEADERS):
        return lib
    o = os.path.join(CSRC, "transport_%s.o" % name)
    subprocess.check_call([nvcc()] + NVCC_FLAGS + EXTRA_FLAGS["transport.cu"] + list(flags) + ["-c", src, "-o", o])
    objs = [o] + [os.path.join(CSRC, s.replace(".cu", ".o")) for s in SOURCES if s != "transport.cu"]
    subprocess.check_call([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib] + objs + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"])
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
