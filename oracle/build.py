"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product).

    python oracle/build.py

writes oracle/libafm_oracle.so (single-threaded; the timed baseline) and
oracle/libafm_oracle_omp.so (OpenMP over particles; parity checks only).
-ffp-contract=off keeps every operation a separately rounded IEEE operation.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "afm_oracle.c"), os.path.join(HERE, "afm_oracle_beam.c")]
FLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fPIC",
         "-shared", "-Wall", "-Wextra"]


def _stale(out):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t
               for f in ("afm_oracle.c", "afm_oracle.h", "afm_oracle_beam.c",
                         "afm_oracle_beam.h", "build.py"))


def build(force=False, verbose=False):
    outs = []
    for name, extra in (("libafm_oracle.so", []),
                        ("libafm_oracle_omp.so", ["-fopenmp", "-DORC_OPENMP"])):
        out = os.path.join(HERE, name)
        if force or _stale(out):
            cmd = ["gcc"] + FLAGS + extra + SRCS + ["-o", out, "-lm"]
            if verbose:
                print(" ".join(cmd))
            subprocess.check_call(cmd)
        outs.append(out)
    return outs


if __name__ == "__main__":
    for o in build(force="--force" in sys.argv, verbose=True):
        print("built", o)
