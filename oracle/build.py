"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product).

    python -m oracle.build

g++ -O2 -ffp-contract=off -fno-fast-math: one rounding per fp32 operation, which is
what DESIGN.md section 3 defines and the deterministic CUDA mode must reproduce.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hadpsgd_oracle.cpp")
HDR = os.path.join(HERE, "hadpsgd_oracle.h")
LIB = os.path.join(HERE, "libhadpsgd_oracle.so")

FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c++17", "-fPIC", "-shared",
         "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
