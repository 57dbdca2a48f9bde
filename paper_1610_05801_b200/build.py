"""Builds liblongtrack.so and liblongtrack_probe.so for sm_100a with nvcc (in-tree, next to this file).

    python -m paper_1610_05801_b200.build [--force]

The library links the CUDA runtime statically, so it loads (and its host-only entry points
work) on a machine without a GPU or a CUDA installation; device calls then return LT_E_CUDA.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblongtrack.so")
SOURCES = [os.path.join(CSRC, "longtrack.cu"), os.path.join(CSRC, "longtrack_next.cu"),
           os.path.join(CSRC, "longtrack_ramp.cu"), os.path.join(CSRC, "longtrack_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "kernels.cuh"), os.path.join(CSRC, "kernels_next.cuh"), os.path.join(CSRC, "kernels_ramp.cuh"),
                  os.path.join(CSRC, "tracker.hpp"), os.path.join(CSRC, "sinpi_coeffs.h"),
                  os.path.join(ROOT, "include", "longtrack.h")]

# measurement tooling (FP64-pipe probes), its own library: liblongtrack.so exports the tracking calls only
PROBE_LIB = os.path.join(HERE, "liblongtrack_probe.so")
PROBE_SOURCES = [os.path.join(CSRC, "longtrack_probe.cu")]
PROBE_DEPS = PROBE_SOURCES + [os.path.join(CSRC, "kernels.cuh"), os.path.join(CSRC, "kernels_probe.cuh"),
                              os.path.join(CSRC, "sinpi_coeffs.h"), os.path.join(ROOT, "include", "longtrack.h"),
                              os.path.join(ROOT, "include", "longtrack_probe.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "2"]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: liblongtrack.so cannot be built")
    return exe


def _build_one(lib: str, sources: list, deps: list, force: bool, verbose: bool) -> str:
    newest = max(os.path.getmtime(p) for p in deps)
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
        return lib
    # nvcc/ld write their output in place: link to a private name and rename it onto the library, so
    # that another process (the non-zero ranks of a torchrun launch, wait_until_built below) can never
    # dlopen a half-written file -- os.replace is atomic within one directory
    tmp = "%s.tmp.%d" % (lib, os.getpid())
    cmd = [nvcc(), *NVCC_FLAGS, "-o", tmp, *sources]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    try:
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, lib)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    """liblongtrack.so (the product) and liblongtrack_probe.so (bench.py's FP64-pipe probes)."""
    _build_one(PROBE_LIB, PROBE_SOURCES, PROBE_DEPS, force, verbose)
    return _build_one(LIB, SOURCES, DEPS, force, verbose)       # last: wait_until_built watches this one


def wait_until_built(timeout_s: float = 900.0) -> str:
    """For the ranks of a torchrun launch that do NOT build: block until rank 0's build is there."""
    import time
    t0 = time.time()
    newest = max(os.path.getmtime(p) for p in DEPS)
    newest_probe = max(os.path.getmtime(p) for p in PROBE_DEPS)
    while not (os.path.exists(LIB) and os.path.getmtime(LIB) >= newest and
               os.path.exists(PROBE_LIB) and os.path.getmtime(PROBE_LIB) >= newest_probe):
        if time.time() - t0 > timeout_s:
            raise RuntimeError("liblongtrack.so was not built within %.0f s" % timeout_s)
        time.sleep(0.5)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
