"""Build paper_1303_5057_b200/libgray.so (the C-ABI library of include/gray.h) for sm_100a.

    python -m paper_1303_5057_b200.build [--force] [--verbose]

Plain nvcc, in-tree output (the .so travels with the repository snapshot to the GPU box).
GRAY_NVCC_EXTRA (environment) appends flags, e.g. "-DGRAY_BLOCK=64 -DGRAY_F2_MIN_BLOCKS=8" or "-DGRAY_COMP_MASK=0x6e":
the tuning macros of csrc/gray_integrate.cu and csrc/gray_math.cuh (DESIGN.md lists what they measured).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgray.so")
SOURCES = ["gray_api.cu", "gray_init.cu", "gray_integrate.cu", "gray_shadow.cu", "gray_host.cu"]
HEADERS = [os.path.join(CSRC, "gray_internal.h"), os.path.join(CSRC, "gray_math.cuh"), os.path.join(CSRC, "gray_vec.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "gray.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(p) for p in srcs + HEADERS + [os.path.abspath(__file__)])
        if os.path.getmtime(LIB) >= newest:
            return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s) + ".o")
        cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("GRAY_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        if p.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [_nvcc(), "-shared", "-Wno-deprecated-gpu-targets", "-o", LIB] + objs
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
