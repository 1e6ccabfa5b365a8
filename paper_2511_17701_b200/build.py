"""Build step of the CUDA library: nvcc -> libgrpic_f32.so / libgrpic_f64.so, in-tree, sm_100a only.

    python -m paper_2511_17701_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so files are git-ignored but travel with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
_SOURCES = ["grpic.cu", "grpic_kernels.cuh", "grpic_device.cuh", "grpic_tiled.cuh", "grpic_lanes.cuh", "grpic_fields.cuh", "grpic_probe.cuh"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "--cudart", "static"]


def lib_path(precision: str) -> str:
    assert precision in ("f32", "f64")
    return os.path.join(_HERE, f"libgrpic_{precision}.so")


def _stale(out: str) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    deps = [os.path.join(_CSRC, s) for s in _SOURCES] + [os.path.join(_INC, "grpic.h"), os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> dict:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = "nvcc"
    out = {}
    procs = []
    for prec, defs in (("f32", []), ("f64", ["-DGRPIC_F64"])):
        so = lib_path(prec)
        out[prec] = so
        if force or _stale(so):
            extra = os.environ.get("GRPIC_NVCC_EXTRA", "").split()      # e.g. "-DGRPIC_TILED_MINB=2" for tuning runs
            cmd = [nvcc] + NVCC_FLAGS + defs + extra + (["-Xptxas", "-v"] if verbose else []) + \
                  [os.path.join(_CSRC, "grpic.cu"), "-o", so]
            procs.append((prec, cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for prec, cmd, p in procs:
        log, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed for {prec}:\n{' '.join(cmd)}\n{log}")
        if verbose:
            print(log)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
