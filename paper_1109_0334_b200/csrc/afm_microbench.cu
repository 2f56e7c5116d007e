// afm_microbench.cu -- register-only FMA throughput probe (SURVEY.md 8(d):
// "measure both FMA peaks with a register-only DFMA/FFMA microbenchmark").
// Not on the hot path; it gives bench.py the measured denominator that sits
// beside the lane-model peak in the roofline object.
#include "afm_internal.h"

namespace afm {

// 8 independent dependent-FMA chains per thread: enough ILP to cover the
// 4-cycle (FP32) / ~8-cycle (FP64) pipe latency at any occupancy.
template <typename T>
__global__ void fma_peak_kernel(T a, T b, int iters, T* __restrict__ sink) {
  T x0 = (T)threadIdx.x, x1 = x0 + (T)1, x2 = x0 + (T)2, x3 = x0 + (T)3;
  T x4 = x0 + (T)4, x5 = x0 + (T)5, x6 = x0 + (T)6, x7 = x0 + (T)7;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b);
      x1 = fma(x1, a, b);
      x2 = fma(x2, a, b);
      x3 = fma(x3, a, b);
      x4 = fma(x4, a, b);
      x5 = fma(x5, a, b);
      x6 = fma(x6, a, b);
      x7 = fma(x7, a, b);
    }
  }
  const T s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == (T)123456789) sink[0] = s;  // never true: keeps the chains alive
}

// Returns the number of launches; *ms receives the duration of the timed one.
int launch_fma_peak(int precision, int iters, int blocks, int threads,
                    void* sink, float* ms, cudaStream_t st) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return -2;
  if (cudaEventCreate(&e1) != cudaSuccess) return -2;
  int n = 0;
  for (int rep = 0; rep < 2; ++rep) {  // first launch warms up
    cudaEventRecord(e0, st);
    if (precision == AFM_F32)
      fma_peak_kernel<float><<<blocks, threads, 0, st>>>(0.999f, 0.001f, iters,
                                                       (float*)sink);
    else
      fma_peak_kernel<double><<<blocks, threads, 0, st>>>(0.999, 0.001, iters,
                                                        (double*)sink);
    cudaEventRecord(e1, st);
    ++n;
  }
  cudaEventSynchronize(e1);
  cudaEventElapsedTime(ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return n;
}

}  // namespace afm
