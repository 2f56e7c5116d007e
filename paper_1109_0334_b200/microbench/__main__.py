"""Build and run the stand-alone microbenchmarks (afm_probes.cu).

    python -m paper_1109_0334_b200.microbench [all|latency|rk4chain|dispatch]

A separate program: not part of libafm_b200.so, not on the product path.  Needs a
B200 to run; nvcc cross-compiles it anywhere.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
ROOT = os.path.dirname(PKG)
SRC = os.path.join(HERE, "afm_probes.cu")
EXE = os.path.join(HERE, "afm_probes.bin")


def build(force=False):
    deps = [SRC, os.path.join(PKG, "csrc", "afm_device.cuh"),
            os.path.join(PKG, "csrc", "afm_device_common.cuh")]
    if force or not os.path.exists(EXE) or any(os.path.getmtime(d) > os.path.getmtime(EXE)
                                               for d in deps):
        subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3",
                               "-lineinfo", "-std=c++17", "--fmad=true", "-I",
                               os.path.join(ROOT, "include"), "-I", os.path.join(PKG, "csrc"),
                               SRC, "-o", EXE])
    return EXE


if __name__ == "__main__":
    args = [a for a in sys.argv[1:] if a != "--build-only"]
    exe = build()
    if "--build-only" not in sys.argv:
        sys.exit(subprocess.call([exe] + args))
