"""Build libcomem_decode.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2605_30842_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  cudart is linked statically and the one
driver symbol needed (cuTensorMapEncodeTiled) is fetched at run time through
cudaGetDriverEntryPoint, so the library LOADS on a box without libcuda — it
just cannot compute there.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcomem_decode.so")
SOURCES = ["api.cu", "decode_split.cu", "combine.cu", "kv_append.cu", "kstep_pipeline.cu", "kstep_step.cu", "decode_fp8_tc.cu", "prefill_attn.cu", "read_ceiling.cu"]
HEADERS = ["ptx.cuh", "schedule.cuh", "decode_params.cuh", "merge.cuh", "tcgen05.cuh", "prefill_params.cuh", os.path.join("..", "..", "include", "comem_decode_attn.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
