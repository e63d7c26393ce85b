"""Build the sm_100a CUDA library in-tree: paper_2505_04155_b200/libamp_pcg.so.

nvcc cross-compiles without a GPU, so this runs on the CPU build box; the .so then travels
with the repository snapshot to the B200 box (it is git-ignored, not gpurun-ignored).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libamp_pcg.so")
SOURCES = ["amp_pcg.cu", "xr_static.cu"]
HEADERS = ["common.cuh", "phases.cuh", "spmv.cuh", "spmv_pipe.cuh", "kernels.cuh", "persistent.cuh", "shard.cuh", "shard_host.cuh", "vec_pipe.cuh", "vec_fused.cuh", "async_copy.cuh"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "--expt-extended-lambda",
    "-Xcompiler", "-fPIC", "-shared",
]


def needs_build(lib: str = None) -> bool:
    lib = lib or LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "amp_pcg.h")]
    return any(os.path.getmtime(d) > t for d in deps)


LIB_COUNT = os.path.join(HERE, "libamp_pcg_count.so")


def build_counting(force: bool = False) -> str:
    """The counting build (-DAMP_COUNT_FP16): every FP16 store of z and p is classified (subnormal / flushed to
    zero / overflowed) into amp_stats_t.fp16_*.  Slower (atomics); used by the tests and the omega study only."""
    return build(force=force, extra_flags=("-DAMP_COUNT_FP16",), out=LIB_COUNT)


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str = LIB) -> str:
    if not force and not needs_build(out):
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, *extra_flags]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", out]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building " + os.path.basename(out))
    return out


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
    if "--counting" in sys.argv:
        print(build_counting(force=True))
