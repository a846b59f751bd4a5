"""Build libhadpsgd.so (sm_100a only) in-tree with nvcc.   python -m paper_1907_05701_b200.build"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhadpsgd.so")
SOURCES = ["hadpsgd.cu", "step_f32.cu", "step_bf16.cu", "step_f32_emit.cu", "step_bf16_emit.cu", "consensus.cu", "consensus_noalloc.cu", "peer_flush.cu",
           "allocator.cpp", "scheduler.cpp", "schedule.cpp"]
DEPS = SOURCES + ["internal.h", "step_kernel.cuh", "step_dispatch.cuh", os.path.join("..", "..", "include", "hadpsgd.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--ftz=false", "--prec-div=true", "--prec-sqrt=true",   # IEEE: no flush-to-zero (R17)
              "-Xcompiler", "-fPIC,-Wall", "-shared", "-cudart", "static",
              "--threads", "4"]           # the four step_*.cu instantiation units compile in parallel


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("HADPSGD_NVCC_EXTRA", "").split()     # development: extra -D switches
    cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
           *[os.path.join(CSRC, s) for s in SOURCES]]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
