"""Build the CPU oracle (test infrastructure) into oracle/libvr_oracle.so.

    python -m oracle.build

gcc only; no CUDA, no code shared with paper_1001_2049_b200/.  The flags keep
the IEEE-754 binary32 op sequence exactly as written in vr_oracle.c:
-ffp-contract=off (GCC's GNU-mode default would fuse a*b+c when -mfma is on),
-fno-fast-math; -mfma only makes fmaf() a single instruction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "vr_oracle.c")
LIB = os.path.join(HERE, "libvr_oracle.so")

FLAGS = ["-std=c99", "-O2", "-fPIC", "-shared", "-fopenmp", "-mfma",
         "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "vr_oracle.h"), os.path.abspath(__file__)]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["gcc"] + FLAGS + ["-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
