"""Build the C-ABI CUDA libraries in-tree with nvcc for sm_100a.

    python -m paper_1612_09491_b200._build [--force] [-v]

  libpsd.so        include/psd.h        the deposit path (csrc/psd_abi.cu + *.cuh)
  libpsd_peaks.so  include/psd_peaks.h  roofline-denominator micro-benchmarks (csrc/psd_peaks.cu)

nvcc cross-compiles without a GPU.  The .so files are git-ignored but travel to the GPU box.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpsd.so")
PEAKS_LIB = os.path.join(_HERE, "libpsd_peaks.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
              "-I", os.path.join(ROOT, "include")]


def _headers():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))]


# target -> (sources, dependencies)
TARGETS = {
    LIB: ([os.path.join(CSRC, "psd_abi.cu")],
          lambda: _headers() + [os.path.join(ROOT, "include", "psd.h")]),
    PEAKS_LIB: ([os.path.join(CSRC, "psd_peaks.cu")],
                lambda: [os.path.join(ROOT, "include", "psd_peaks.h")]),
}


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpsd cannot be built (there is no CPU fallback)")


def is_stale(target: str = LIB) -> bool:
    if not os.path.exists(target):
        return True
    srcs, deps = TARGETS[target]
    t = os.path.getmtime(target)
    return any(os.path.getmtime(f) > t for f in srcs + deps() + [__file__])


def build(force: bool = False, verbose: bool = False, target: str = LIB) -> str:
    if not force and not is_stale(target):
        return target
    srcs, _ = TARGETS[target]
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + srcs + ["-o", target + ".tmp"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    os.replace(target + ".tmp", target)
    return target


def build_all(force: bool = False, verbose: bool = False):
    return [build(force, verbose, t) for t in TARGETS]


if __name__ == "__main__":
    print("\n".join(build_all(force="--force" in sys.argv, verbose="-v" in sys.argv)))
