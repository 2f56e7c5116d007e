"""Microbenchmarks behind the roofline of DESIGN.md section 6.

    python -m paper_1109_0334_b200.probe

Prints the measured register-only FMA peaks (afm_fma_peak) and the dispatch
probe (afm_dispatch_probe): what one FP64 warp-instruction costs an SM
sub-partition depending on its operands, on neighbouring integer work and on
the lane mask.  Needs a B200; there is no CPU fallback.
"""
from . import afm

MODES = ("x=fma(x,a,b), a,b reused", "x=fma(x,y,z), 3 register operands",
         "fma(x,y,z) + 2 integer instr", "fma(x,y,z) + 4 integer instr",
         "fma(x,y,z), 16 of 32 lanes active")


def main():
    print("register-only FMA peak: FP64 %.2f TFLOP/s, FP32 %.2f TFLOP/s"
          % (afm.afm_fma_peak(afm.F64, 0.3), afm.afm_fma_peak(afm.F32, 0.3)))
    print("ns per DFMA warp-instruction per SM sub-partition")
    print("%-36s %8s %8s %8s %8s" % ("warps per sub-partition:", 1, 2, 4, 8))
    for m, name in enumerate(MODES):
        row = [afm.afm_dispatch_probe(m, w) for w in (1, 2, 4, 8)]
        print("%-36s %8.3f %8.3f %8.3f %8.3f" % ((name,) + tuple(row)))


if __name__ == "__main__":
    main()
