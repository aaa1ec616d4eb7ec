"""Build libcuhpx.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2510_01785_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcuhpx.so")
SOURCES = ["plan.cu", "legendre.cu", "legendre_tc.cu", "ring_fft.cu", "reorder.cu", "ring_weights.cu", "noalloc.cu"]
HEADERS = [os.path.join(CSRC, "cuhpx_internal.h"), os.path.join(CSRC, "block_fft.cuh"),
           os.path.join(CSRC, "legendre_common.cuh"), os.path.join(CSRC, "tc_common.cuh"),
           os.path.join(HERE, "..", "include", "cuhpx.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def _compile_one(args):
    nvcc, src, obj = args
    cmd = [nvcc] + NVCC_FLAGS + ["-c", "-o", obj, src]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return res.returncode, res.stdout + res.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every csrc/*.cu to an object file (in parallel, only the stale ones) and link libcuhpx.so."""
    if not (force or needs_build()):
        return LIB
    from concurrent.futures import ThreadPoolExecutor

    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    hdr_t = max(os.path.getmtime(h) for h in HEADERS)
    jobs, objs = [], []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(objdir, s.replace(".cu", ".o"))
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_t):
            jobs.append((nvcc, src, obj))
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        for rc, out in ex.map(_compile_one, jobs):
            if verbose or rc != 0:
                sys.stderr.write(out)
            if rc != 0:
                raise RuntimeError("nvcc failed building libcuhpx.so")
    res = subprocess.run([nvcc, "-shared", "-o", LIB] + objs, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libcuhpx.so")
    return LIB


PROBES = {"tcgen05_probe": "tcgen05_probe.cu", "dfma_probe": "dfma_probe.cu"}


def build_probe() -> list:
    """Compile the micro-benchmarks (measurement tools outside libcuhpx.so): csrc/tcgen05_probe.cu
    (profiles/r2_tcgen05_probe.md) and csrc/dfma_probe.cu (profiles/r2_dfma_probe.md)."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    built = []
    for exe, src in PROBES.items():
        out = os.path.join(HERE, exe)
        cmd = [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", out, os.path.join(CSRC, src)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError(f"nvcc failed building {exe}")
        built.append(out)
    return built


if __name__ == "__main__":
    if "--probe" in sys.argv:
        print("\n".join(build_probe()))
    else:
        build(force="--force" in sys.argv, verbose=True)
        print(LIB)
