"""TEST INFRASTRUCTURE: builds tests/hostemu/libvr_hostemu.so -- the product's own sources
(paper_1001_2049_b200/csrc/*.cu) compiled by g++ against the host emulation of the CUDA subset they use
(cuda_runtime.h in this directory).  Same C ABI as libvr.so; "device memory" is host memory.

    python tests/hostemu/build.py [--force]

Only tests load it (tests/emu_backend.py); the package never does.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_1001_2049_b200", "csrc")
LIB = os.path.join(HERE, "libvr_hostemu.so")
SOURCES = ["vr_api.cu", "vr_kernels.cu", "vr_pipe.cu", "vr_beam.cu"]
# -D__CUDA_ARCH__: the sources take their DEVICE branches (intrinsics), which the emulation defines one by one;
# -ffp-contract=off / no fast-math: nothing is fused or reassociated behind the contract's back
FLAGS = ["-std=c++17", "-O2", "-g", "-fPIC", "-fopenmp", "-mfma", "-ffp-contract=off", "-fno-fast-math", "-frounding-math",
         "-D__CUDA_ARCH__=1000", "-DVR_HOSTEMU=1", "-Wall", "-Wno-unknown-pragmas", "-Wno-unused-function",
         "-Wno-unused-variable", "-I", HERE]


def _deps():
    out = [os.path.abspath(__file__), os.path.join(ROOT, "include", "vr.h")]
    out += [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out += [os.path.join(HERE, f) for f in os.listdir(HERE) if f.endswith((".h", ".cpp"))]
    return out


def build(force=False, asan=False):
    """asan=True: a second library, libvr_hostemu_asan.so, built with AddressSanitizer -- every "device" buffer is then a
    red-zoned host allocation and a kernel that reads or writes one element past it aborts the process with a report
    (the host stand-in for compute-sanitizer memcheck; the process must run with libasan preloaded, see
    tests/test_emu_asan.py)."""
    lib = LIB.replace(".so", "_asan.so") if asan else LIB
    flags = FLAGS + (["-fsanitize=address", "-fno-omit-frame-pointer"] if asan else [])
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in _deps()):
        return lib
    cxx = os.environ.get("VR_EMU_CXX", "g++")
    bdir = os.path.join(HERE, "build_asan" if asan else "build")
    os.makedirs(bdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(bdir, src.replace(".cu", ".o"))
        objs.append(obj)
        procs.append(subprocess.Popen([cxx] + flags + ["-x", "c++", "-c", os.path.join(CSRC, src), "-o", obj],
                                      stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    obj = os.path.join(bdir, "emu_runtime.o")
    objs.append(obj)
    procs.append(subprocess.Popen([cxx] + flags + ["-c", os.path.join(HERE, "emu_runtime.cpp"), "-o", obj],
                                  stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    failed = False
    for pr in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0:
            sys.stderr.write(out)
            failed = True
    if failed:
        raise RuntimeError("g++ failed building libvr_hostemu.so")
    r = subprocess.run([cxx, "-shared", "-fopenmp"] + (["-fsanitize=address"] if asan else []) + ["-o", lib] + objs,
                       capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("g++ failed linking " + os.path.basename(lib))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, asan="--asan" in sys.argv))
