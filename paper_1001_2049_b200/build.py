"""Build libvr.so (the C-ABI library of include/vr.h) in-tree for sm_100a.

    python -m paper_1001_2049_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  -fmad=false: the numerical contract
 allows only the explicit __fmaf_rn fusions.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvr.so")
SOURCES = ["vr_api.cu", "vr_kernels.cu", "vr_pipe.cu", "vr_beam.cu"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-Wall",
              "-shared", "-cudart", "static"]


def _deps():
    out = [os.path.abspath(__file__), os.path.join(HERE, "..", "include", "vr.h")]
    for f in os.listdir(CSRC):
        out.append(os.path.join(CSRC, f))
    return out


def build(force=False, verbose=False):
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps())):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    # one object per translation unit, compiled side by side, then one link
    compile_flags = [f for f in NVCC_FLAGS if f != "-shared"]
    objs, procs = [], []
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        os.makedirs(os.path.dirname(obj), exist_ok=True)
        objs.append(obj)
        cmd = [nvcc] + compile_flags + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
        procs.append(subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    failed = False
    for pr in procs:
        out, err = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out + err)
        failed = failed or pr.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libvr.so")
    r = subprocess.run([nvcc, "-shared", "-cudart", "static", "-o", LIB] + objs, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed linking libvr.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
