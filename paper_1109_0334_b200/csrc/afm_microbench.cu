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

// Dispatch probe: what an FP64 instruction costs next to other work.
//   mode 0: x = fma(x, a, b)      one changing register operand, a and b reused
//   mode 1: x = fma(x, y, z)      three distinct 64-bit register operands
//   mode 2: mode 1 + 2 integer ALU instructions per DFMA (independent of it)
//   mode 3: mode 1 + 4 integer ALU instructions per DFMA
//   mode 4: mode 1 with only 16 of 32 lanes active
template <int MODE>
__global__ void dispatch_probe_kernel(const double* __restrict__ in, int iters,
                                      double* __restrict__ sink) {
  if (MODE == 4 && (threadIdx.x & 16)) return;
  double x[8], y[8], z[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    x[i] = in[(threadIdx.x + i) & 63];
    y[i] = in[(threadIdx.x + 8 + i) & 63];
    z[i] = in[(threadIdx.x + 16 + i) & 63];
  }
  const double a = in[0], b = in[1];
  int c0 = threadIdx.x, c1 = threadIdx.x * 3;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (MODE == 0) x[i] = fma(x[i], a, b);
        if (MODE == 1 || MODE == 4) x[i] = fma(x[i], y[i], z[i]);
        if (MODE == 2) {
          x[i] = fma(x[i], y[i], z[i]);
          c0 = (c0 ^ c1) + i;
        }
        if (MODE == 3) {
          x[i] = fma(x[i], y[i], z[i]);
          c0 = (c0 ^ c1) + i;
          c1 = (c1 & c0) ^ u;
        }
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  if (s == 1234.5 || c0 == 0x7fffffff) sink[0] = s + c1;
}

// ns per DFMA warp-instruction per SM sub-partition (64 DFMA per loop trip).
int launch_dispatch_probe(int mode, int warps_per_subpartition, int n_sm,
                          const double* in, double* sink, double* ns_per_dfma,
                          cudaStream_t st) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return -2;
  if (cudaEventCreate(&e1) != cudaSuccess) return -2;
  const int threads = 128 * warps_per_subpartition, iters = 20000;
  float ms = 0.f;
  for (int rep = 0; rep < 2; ++rep) {
    const int it = rep ? iters : 200;
    cudaEventRecord(e0, st);
    switch (mode) {
      case 0: dispatch_probe_kernel<0><<<n_sm, threads, 0, st>>>(in, it, sink); break;
      case 1: dispatch_probe_kernel<1><<<n_sm, threads, 0, st>>>(in, it, sink); break;
      case 2: dispatch_probe_kernel<2><<<n_sm, threads, 0, st>>>(in, it, sink); break;
      case 3: dispatch_probe_kernel<3><<<n_sm, threads, 0, st>>>(in, it, sink); break;
      default: dispatch_probe_kernel<4><<<n_sm, threads, 0, st>>>(in, it, sink); break;
    }
    cudaEventRecord(e1, st);
  }
  cudaEventSynchronize(e1);
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *ns_per_dfma = (double)ms * 1e6 / ((double)iters * 64.0 * warps_per_subpartition);
  return 2;
}

}  // namespace afm
