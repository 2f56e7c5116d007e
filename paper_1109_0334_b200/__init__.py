"""paper_1109_0334_b200 -- B200-native hot path of the dAFM tip-sample force
inversion of arxiv/paper_1109_0334: batched RK4 forward solve + squared-misfit
reduction + PSO update, as hand-written sm_100a CUDA kernels behind a C ABI
(include/afm.h).  `afm` is the thin ctypes binding; `workloads` the seeded
synthetic inputs.  There is no CPU fallback: `afm` raises if the CUDA library
is missing."""

__all__ = ["afm", "workloads"]
