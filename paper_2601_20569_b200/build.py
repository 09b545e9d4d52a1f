"""Build the native pieces in-tree: libtpctrack.so (CUDA, sm_100a) and libtpcgen.so (host).

nvcc cross-compiles sm_100a without a GPU.  The kernel translation unit is compiled twice:
deterministic (-DTPC_DET=1 --fmad=false) and fast (-DTPC_DET=0 --fmad=true).
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB_PATH = os.path.join(CSRC, "libtpctrack.so")

_NVCC_BASE = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I" + INCLUDE, "-I" + CSRC]


def _newer(target: str, sources) -> bool:
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(s) for s in sources)


def build_tpctrack(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, f) for f in ("tpc_kernels.cu", "tpc_api.cu", "tpc_internal.h")]
    srcs.append(os.path.join(INCLUDE, "tpc_track.h"))
    if not force and _newer(LIB_PATH, srcs):
        return LIB_PATH
    extra = ["-Xptxas", "-v"] if verbose else []
    det_o, fast_o, api_o = (os.path.join(CSRC, f"tpc_{n}.o") for n in ("kernels_det", "kernels_fast", "api"))
    cmds = [
        _NVCC_BASE + extra + ["-DTPC_DET=1", "--fmad=false", "-c", srcs[0], "-o", det_o],
        # fast build: FMA contraction, approximate division / square root (MUFU based), denormals
        # flushed: rounding-level differences only, which is all fast mode may differ by
        _NVCC_BASE + extra + ["-DTPC_DET=0", "--fmad=true", "--use_fast_math", "-c", srcs[0], "-o", fast_o],
        _NVCC_BASE + ["-c", srcs[1], "-o", api_o],
        ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB_PATH, det_o, fast_o, api_o],
    ]
    procs = [subprocess.Popen(c) for c in cmds[:3]]
    for p, c in zip(procs, cmds[:3]):
        if p.wait() != 0:
            raise RuntimeError("build failed: " + " ".join(c))
    subprocess.run(cmds[3], check=True)
    return LIB_PATH


def build_all(force: bool = False) -> None:
    from . import datagen
    build_tpctrack(force)
    datagen.build(force)


if __name__ == "__main__":
    build_all(force=True)
    print(LIB_PATH)
