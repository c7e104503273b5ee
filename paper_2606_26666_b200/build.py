"""In-tree build of libpkv.so (nvcc, sm_100a only).

``python -m paper_2606_26666_b200.build`` or ``build()`` compiles ``csrc/*.cu|*.cpp`` into
``paper_2606_26666_b200/libpkv.so``.  nvcc cross-compiles without a GPU; the CUDA runtime is
linked statically and the driver entry points the library needs (cuTensorMapEncodeTiled,
cuMemsetD32Async) are resolved at run time through cudaGetDriverEntryPoint, so the library
loads on a box without a driver (the CPU-only tests check its exports there).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
BUILD_DIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpkv.so")

TMA_PARTS = 16     # pkv_decode_tma.cu is compiled once per group of instantiations (-DPKV_TMA_PART=k), in parallel
SOURCES = (["pkv_host.cpp", "pkv_aux.cu", "pkv_decode_simt.cu", "pkv_api.cu", "pkv_calibrate.cu", "pkv_static.cu"]
           + [("pkv_decode_tma.cu", k) for k in range(TMA_PARTS)])
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC,-fvisibility=hidden", "-I", INCLUDE, "-I", CSRC]


def _nvcc() -> str:
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found: libpkv.so cannot be built")
    return nvcc


def _deps_mtime() -> float:
    paths = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "pkv.h")]
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """Compile if libpkv.so is missing or older than any source.  Returns the library path.
    trace=True builds libpkv_trace.so instead: the same sources with -DPKV_TRACE (phase stamps in
    the kernels and the pkv_debug_set_trace hook; never loaded by the package)."""
    lib = LIB if not trace else os.path.join(HERE, "libpkv_trace.so")
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= _deps_mtime():
        return lib
    nvcc = _nvcc()
    bdir = BUILD_DIR if not trace else BUILD_DIR + "_trace"
    os.makedirs(bdir, exist_ok=True)
    objs = []

    def compile_one(item):
        src, part = item if isinstance(item, tuple) else (item, None)
        obj = os.path.join(bdir, os.path.splitext(src)[0] + ("" if part is None else "_part%d" % part) + ".o")
        cmd = ([nvcc] + ARCH + COMMON + (["-DPKV_TRACE"] if trace else []) + (["-Xptxas", "-v"] if verbose else [])
               + ([] if part is None else ["-DPKV_TMA_PART=%d" % part]) + ["-c", os.path.join(CSRC, src), "-o", obj])
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + ARCH + ["-shared", "-o", tmp] + objs + ["-cudart", "static"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
