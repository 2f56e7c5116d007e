"""Build libafm_b200.so (the C-ABI library of include/afm.h) in-tree.

    python -m paper_1109_0334_b200.build [--force] [--verbose] [--ptxas-v]
                                         [--bounds-check]

nvcc cross-compiles for sm_100a only (no GPU needed to build).  The output
sits next to this file so that it travels with the source tree; it is
git-ignored.
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["afm_kernels.cu", "afm_kernels_f32.cu", "afm_microbench.cu", "afm_beam.cu", "afm_sort.cu", "afm_api.cu"]
HEADERS = ["afm_internal.h", "afm_device_common.cuh", "afm_device.cuh", "afm_device_f32.cuh"]
OUT = os.path.join(HERE, "libafm_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "--cudart", "static",
    "-shared",
]


def source_sha():
    """Hash of the library source (csrc/* and include/afm.h, in sorted file order).
    bench.py reports ncu-derived figures from profiles/ only while this equals the
    hash recorded in the summary they come from."""
    h = hashlib.sha256()
    files = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))
    files.append(os.path.join(ROOT, "include", "afm.h"))
    for f in files:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale():
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps += [os.path.join(ROOT, "include", "afm.h"), os.path.abspath(__file__)]
    return any(os.path.exists(d) and os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, extra_flags=()):
    """Compile if stale; returns the path of the shared library."""
    if force or _stale():
        cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags)
        cmd += ["-I", os.path.join(ROOT, "include"), "-I", CSRC]
        cmd += [os.path.join(CSRC, s) for s in SOURCES]
        cmd += ["-o", OUT]
        if verbose:
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    extra = ["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else []
    if "--bounds-check" in sys.argv:    # checked build for debugging, see AFM_CHECK
        extra.append("-DAFM_BOUNDS_CHECK")
    print("built", build(force="--force" in sys.argv,
                         verbose="--verbose" in sys.argv or bool(extra),
                         extra_flags=extra))
