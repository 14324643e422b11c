"""Build libising_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension).

    python -m paper_1006_3865_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libising_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-ldl"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))
    deps += [os.path.join(HERE, "..", "include", n) for n in ("ising.h", "heisenberg.h")]
    return any(os.path.getmtime(d) > t for d in deps)


JIT_SOURCES = {   # generated file -> device headers in inclusion order
    "jit_source.inc": ["philox.cuh", "planes_common.cuh", "tile_planes_device.cuh", "grid_planes_device.cuh", "flow_planes_device.cuh"],
    "jit_source3d.inc": ["philox.cuh", "planes_common.cuh", "tile3d_planes_device.cuh", "grid3d_device.cuh"],
}


def write_jit_source() -> None:
    """csrc/jit_source*.inc = the device headers of the multi-spin kernels as one C++ raw string literal each: the
    sources planes_jit.cu hands to NVRTC at run time (local #include lines and #pragma once dropped)."""
    for inc, headers in JIT_SOURCES.items():
        parts = []
        for name in headers:
            for line in open(os.path.join(CSRC, name)):
                t = line.strip()
                if t.startswith('#include "') or t == "#pragma once":
                    continue
                parts.append(line)
        text = 'R"ISINGJIT(\n' + "".join(parts) + ')ISINGJIT"\n'
        path = os.path.join(CSRC, inc)
        if not os.path.exists(path) or open(path).read() != text:
            with open(path, "w") as f:
                f.write(text)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ (one nvcc process per file, in parallel) and link them into one shared library;
    returns its path."""
    write_jit_source()
    if not force and not _stale():
        return LIB
    if not os.path.exists(NVCC):
        raise RuntimeError(f"nvcc not found at {NVCC}: cannot build libising_b200.so")
    import shutil
    import tempfile
    from concurrent.futures import ThreadPoolExecutor
    compile_flags = [f for f in FLAGS if f not in ("-shared", "-ldl")]
    tmpdir = tempfile.mkdtemp(prefix="ising_b200_build_")
    try:
        def compile_one(src):
            obj = os.path.join(tmpdir, os.path.basename(src) + ".o")
            subprocess.check_call([NVCC, *compile_flags, *(["-Xptxas", "-v"] if verbose else []), "-c", src, "-o", obj])
            return obj
        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
            objs = list(pool.map(compile_one, sources()))
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC, *FLAGS, "-o", tmp, *objs])
        os.replace(tmp, LIB)
    finally:
        shutil.rmtree(tmpdir, ignore_errors=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
