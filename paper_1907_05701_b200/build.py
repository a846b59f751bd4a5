"""Build libhadpsgd.so (sm_100a only) in-tree with nvcc.   python -m paper_1907_05701_b200.build

Every source is compiled to an object of its own under build/ (git-ignored), in parallel, and only
when it is older than the source or any header; then the objects are linked.  The flags are fixed
here: nothing is read from the environment except NVCC (the compiler's path)."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libhadpsgd.so")
SOURCES = ["hadpsgd.cu", "step_f32.cu", "step_bf16.cu", "step_f32_emit.cu", "step_bf16_emit.cu", "consensus.cu",
           "consensus_noalloc.cu", "peer_flush.cu", "allocator.cpp", "scheduler.cpp", "schedule.cpp"]
HEADERS = ["internal.h", "step_kernel.cuh", "step_dispatch.cuh", os.path.join("..", "..", "include", "hadpsgd.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--ftz=false", "--prec-div=true", "--prec-sqrt=true",   # IEEE: no flush-to-zero (R17)
              "-Xcompiler", "-fPIC,-Wall"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    newest_header = max(os.path.getmtime(os.path.join(CSRC, d)) for d in HEADERS + [os.path.join("..", "build.py")])
    objs, stale = [], []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), newest_header):
            stale.append((src, obj))

    def compile_one(pair):
        src, obj = pair
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", src, "-o", obj + ".tmp"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(obj + ".tmp", obj)

    if stale:
        with ThreadPoolExecutor(max_workers=min(len(stale), os.cpu_count() or 4)) as pool:
            list(pool.map(compile_one, stale))
    if stale or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.run([nvcc, *LINK_FLAGS, "-o", LIB + ".tmp", *objs], check=True, cwd=HERE)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
