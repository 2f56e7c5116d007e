// afm_probes.cu -- stand-alone microbenchmarks behind DESIGN.md section 6 ("what
// bounds the kernels").  NOT part of libafm_b200.so and not on the product path:
// a separate program (python -m paper_1109_0334_b200.microbench builds and runs it)
// that includes the library's own device arithmetic (csrc/afm_device.cuh) so that
// the chains it times are the ones the integrate kernel executes.
//
//   latency   dependent-issue latency of DFMA, DADD, DMUL, MUFU.RCP64H (+ the one
//             DFMA that consumes it) and of a warp vote + branch, in SM cycles
//   rk4chain  cycles per RK4 step of ONE warp per SM sub-partition running the
//             exact arithmetic of the FP64 kernel's free-flight step (latency form
//             and throughput form, with and without the speculation vote): the
//             latency floor of the sequential time loop (configs[2], [3])
//   dispatch  cost of a DFMA warp-instruction per SM sub-partition depending on
//             its operands, neighbouring integer work and the lane mask, at 1..8
//             resident warps
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "afm_device.cuh"

using namespace afm;

#define CK(x)                                                                    \
  do {                                                                           \
    cudaError_t e_ = (x);                                                        \
    if (e_ != cudaSuccess) {                                                     \
      fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));                   \
      exit(2);                                                                   \
    }                                                                            \
  } while (0)

// ---- dependent-issue latencies ------------------------------------------------
// One warp; a chain of N dependent operations between two clock64() reads.
template <int OP>
__global__ void latency_kernel(double a, double b, int iters, long long* cyc,
                               double* sink) {
  double x = a + threadIdx.x * 1e-9;
  int vote_acc = 0;
  const long long t0 = clock64();
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 32; ++u) {
      if (OP == 0) x = fma(x, a, b);                 // DFMA
      if (OP == 1) x = x + b;                        // DADD
      if (OP == 2) x = x * a;                        // DMUL
      if (OP == 3) x = fma(-b, rcp_seed(x), a);      // MUFU.RCP64H + 1 DFMA
      if (OP == 4) {                                 // DFMA + vote + branch
        x = fma(x, a, b);
        if (!__all_sync(0xffffffffu, __double2hiint(x) > 0)) vote_acc += u;
      }
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cyc[0] = t1 - t0;
  if (x == 12345.678 || vote_acc == 77) sink[0] = x;
}

// ---- the RK4 step's own chain ---------------------------------------------------
// One warp per CTA, `ctas` CTAs (one per SM sub-partition when ctas = 4 x SMs):
// the exact free-flight arithmetic of integrate_misfit_f64, state in registers, the
// stream row held constant (no shared-memory traffic).  VOTE = the kernel's own
// rk4_step (speculation vote + branch); otherwise the bare arithmetic.
// VOTE 0: the bare arithmetic (free_step, no vote); 1: the kernel's rk4_step (one
// vote and branch per step); 4: four speculative steps per vote, as the latency
// form of the kernel could take them (measured and rejected in the kernel itself:
// every contact entry costs a failed block).
template <bool LAT, int VOTE>
__global__ void rk4chain_kernel(Particle64 P0, double s, double d0, double w0,
                                long long a0_bits, DivergeTest T, int steps,
                                long long* cyc, double* sink) {
  Particle64 P[1] = {P0};
  double d[1] = {d0 + threadIdx.x * 1e-12}, w[1] = {w0};
  bool bad[1] = {false};
  int mode = 0, fails = 0;
  const long long t0 = clock64();
  if (VOTE == 4) {
#pragma unroll 1
    for (int i = 0; i < steps; i += 4) {
      double dd = d[0], ww = w[0];
      bool ok = true;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        double dn, wn;
        ok &= free_step<LAT>(P[0], s, s, s, a0_bits, T, dd, ww, dn, wn);
        dd = dn;
        ww = wn;
      }
      if (__all_sync(0xffffffffu, ok)) {
        d[0] = dd;
        w[0] = ww;
      } else {
        ++fails;
      }
    }
  } else {
#pragma unroll 2
    for (int i = 0; i < steps; ++i) {
      if (VOTE == 1) {
        rk4_step<AFM_LAW_DMT, 1, LAT>(P, s, s, s, a0_bits, d, w, mode, bad, T);
      } else {
        double dn, wn;
        if (!free_step<LAT>(P[0], s, s, s, a0_bits, T, d[0], w[0], dn, wn)) ++fails;
        d[0] = dn;
        w[0] = wn;
      }
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
  if (d[0] == 1234.5 || bad[0] || fails == 12345) sink[0] = d[0] + w[0] + mode;
}

// ---- dispatch probe ----------------------------------------------------------------
//   mode 0: x = fma(x, a, b)      one changing register operand, a and b reused
//   mode 1: x = fma(x, y, z)      three distinct 64-bit register operands
//   mode 2: mode 1 + 2 integer ALU instructions per DFMA (independent of it)
//   mode 3: mode 1 + 4 integer ALU instructions per DFMA
//   mode 4: mode 1 with only 16 of 32 lanes active
template <int MODE>
__global__ void dispatch_kernel(const double* __restrict__ in, int iters,
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

template <int MODE>
static double dispatch_ns(int n_sm, int warps, const double* in, double* sink) {
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  const int iters = 20000;
  dispatch_kernel<MODE><<<n_sm, 128 * warps>>>(in, 200, sink);
  CK(cudaEventRecord(e0));
  dispatch_kernel<MODE><<<n_sm, 128 * warps>>>(in, iters, sink);
  CK(cudaEventRecord(e1));
  CK(cudaEventSynchronize(e1));
  float ms = 0.f;
  CK(cudaEventElapsedTime(&ms, e0, e1));
  return (double)ms * 1e6 / ((double)iters * 64.0 * warps);
}

int main(int argc, char** argv) {
  const char* what = argc > 1 ? argv[1] : "all";
  int dev = 0, n_sm = 0, khz = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  long long* cyc;
  double* sink;
  double* in;
  CK(cudaMalloc(&cyc, 8 * 4096));
  CK(cudaMalloc(&sink, 64));
  CK(cudaMalloc(&in, 64 * 8));
  double h[64];
  for (int i = 0; i < 64; ++i) h[i] = 0.999 + 1e-6 * i;
  CK(cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice));
  printf("device: %d SMs, max SM clock %.0f MHz\n", n_sm, khz / 1e3);

  if (!strcmp(what, "all") || !strcmp(what, "latency")) {
    printf("\n## dependent-issue latency, one warp, SM cycles per operation\n");
    const char* names[5] = {"DFMA", "DADD", "DMUL", "MUFU.RCP64H + DFMA", "DFMA + vote + branch"};
    for (int op = 0; op < 5; ++op) {
      const int iters = 2000;
      long long c = 0;
      for (int rep = 0; rep < 2; ++rep) {
        switch (op) {
          case 0: latency_kernel<0><<<1, 32>>>(0.999, 0.001, iters, cyc, sink); break;
          case 1: latency_kernel<1><<<1, 32>>>(0.999, 0.001, iters, cyc, sink); break;
          case 2: latency_kernel<2><<<1, 32>>>(0.999999, 0.001, iters, cyc, sink); break;
          case 3: latency_kernel<3><<<1, 32>>>(1.5, 0.7, iters, cyc, sink); break;
          default: latency_kernel<4><<<1, 32>>>(0.999, 0.001, iters, cyc, sink); break;
        }
        CK(cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost));
      }
      printf("%-24s %8.2f\n", names[op], (double)c / (iters * 32.0));
    }
  }

  if (!strcmp(what, "all") || !strcmp(what, "rk4chain")) {
    // configs[2]'s cantilever and ground truth in the kernel's per-step variables
    const double PI = 3.14159265358979323846;
    const double k = 2.0, f0 = 7e4, Q = 100.0, zc = 8e-9, R = 1e-8, a0 = 0.3e-9, H = 1e-19;
    const double w0 = 2 * PI * f0, m = k / (w0 * w0), hh = 1.0 / (f0 * 256.0);
    Particle64 P;
    memset(&P, 0, sizeof(P));
    P.nalpha = -hh * w0 / Q;
    P.nbeta = -hh * hh * (k / m);
    P.a0 = a0;
    P.c0 = -H * hh * hh * R / (6.0 * m);
    DivergeTest T;
    T.key_max = 0x7fe0000000000000LL;
    T.key_min = -0x7fe0000000000000LL;
    double safe = 1e-6;
    memcpy(&T.safe_hi, (char*)&safe + 4, 4);
    long long a0_bits;
    memcpy(&a0_bits, &a0, 8);
    // a state that stays in free flight: d = z_c (tip at rest height), tiny velocity,
    // drive term chosen to balance the spring so that d hardly moves
    const double d0 = zc, s = -P.nbeta * zc - P.c0 / (zc * zc);
    printf("\n## RK4 step chain, free flight, register-only, SM cycles per step\n");
    printf("%-44s %10s %10s\n", "", "1 warp/SM", "1 warp/sub-partition");
    const char* names[6] = {"throughput form, arithmetic only",
                            "throughput form, rk4_step (vote per step)",
                            "throughput form, vote per 4 steps",
                            "latency form, arithmetic only",
                            "latency form, rk4_step (vote per step)",
                            "latency form, vote per 4 steps"};
    for (int v = 0; v < 6; ++v) {
      double res[2];
      for (int g = 0; g < 2; ++g) {
        const int ctas = g ? 4 * n_sm : n_sm;
        const int steps = 20000;
        for (int rep = 0; rep < 2; ++rep) {
          switch (v) {
            case 0: rk4chain_kernel<false, 0><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
            case 1: rk4chain_kernel<false, 1><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
            case 2: rk4chain_kernel<false, 4><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
            case 3: rk4chain_kernel<true, 0><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
            case 4: rk4chain_kernel<true, 1><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
            default: rk4chain_kernel<true, 4><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink); break;
          }
          CK(cudaDeviceSynchronize());
        }
        static long long hc[4096];
        CK(cudaMemcpy(hc, cyc, 8 * ctas, cudaMemcpyDeviceToHost));
        double mx = 0;
        for (int i = 0; i < ctas; ++i) mx = hc[i] > mx ? (double)hc[i] : mx;
        res[g] = mx / steps;
      }
      printf("%-44s %10.1f %10.1f\n", names[v], res[0], res[1]);
    }
  }

  if (!strcmp(what, "all") || !strcmp(what, "rk4chain")) {
    // the same warp with its tip resting inside the sample (d = a0 / 2, the contact
    // force balanced by the stream term): every step runs in the general form
    const double PI = 3.14159265358979323846;
    const double k = 2.0, f0 = 7e4, Q = 100.0, R = 1e-8, a0 = 0.3e-9, H = 1e-19, Es = 1e9;
    const double w0 = 2 * PI * f0, m = k / (w0 * w0), hh = 1.0 / (f0 * 256.0);
    Particle64 P;
    memset(&P, 0, sizeof(P));
    P.nalpha = -hh * w0 / Q;
    P.nbeta = -hh * hh * (k / m);
    P.a0 = a0;
    P.c0 = -H * hh * hh * R / (6.0 * m);
    P.c1 = (4.0 / 3.0) * Es * sqrt(R) * hh * hh / m;
    P.c2 = P.c0 / (a0 * a0);
    DivergeTest T;
    T.key_max = 0x7fe0000000000000LL;
    T.key_min = -0x7fe0000000000000LL;
    double safe = 1e-6;
    memcpy(&T.safe_hi, (char*)&safe + 4, 4);
    long long a0_bits;
    memcpy(&a0_bits, &a0, 8);
    const double d0 = 0.5 * a0, del = a0 - d0;
    const double s = -P.nbeta * d0 - (P.c2 + P.c1 * del * sqrt(del));
    printf("\n## RK4 step chain, tip in contact (general form), register-only, SM cycles per step\n");
    printf("%-44s %10s %10s\n", "", "1 warp/SM", "1 warp/sub-partition");
    const char* names[2] = {"throughput form, rk4_step", "latency form, rk4_step"};
    for (int v = 0; v < 2; ++v) {
      double res[2];
      for (int g = 0; g < 2; ++g) {
        const int ctas = g ? 4 * n_sm : n_sm;
        const int steps = 20000;
        for (int rep = 0; rep < 2; ++rep) {
          if (v == 0) rk4chain_kernel<false, 1><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink);
          else rk4chain_kernel<true, 1><<<ctas, 32>>>(P, s, d0, 0.0, a0_bits, T, steps, cyc, sink);
          CK(cudaDeviceSynchronize());
        }
        static long long hc[4096];
        CK(cudaMemcpy(hc, cyc, 8 * ctas, cudaMemcpyDeviceToHost));
        double mx = 0;
        for (int i = 0; i < ctas; ++i) mx = hc[i] > mx ? (double)hc[i] : mx;
        res[g] = mx / steps;
      }
      printf("%-44s %10.1f %10.1f\n", names[v], res[0], res[1]);
    }
  }

  if (!strcmp(what, "all") || !strcmp(what, "dispatch")) {
    printf("\n## ns per DFMA warp-instruction per SM sub-partition\n");
    printf("%-36s %8d %8d %8d %8d\n", "warps per sub-partition:", 1, 2, 4, 8);
    const char* names[5] = {"x=fma(x,a,b), a,b reused", "x=fma(x,y,z), 3 register operands",
                            "fma(x,y,z) + 2 integer instr", "fma(x,y,z) + 4 integer instr",
                            "fma(x,y,z), 16 of 32 lanes active"};
    for (int mo = 0; mo < 5; ++mo) {
      printf("%-36s", names[mo]);
      for (int wps = 1; wps <= 8; wps *= 2) {
        double ns = 0;
        switch (mo) {
          case 0: ns = dispatch_ns<0>(n_sm, wps, in, sink); break;
          case 1: ns = dispatch_ns<1>(n_sm, wps, in, sink); break;
          case 2: ns = dispatch_ns<2>(n_sm, wps, in, sink); break;
          case 3: ns = dispatch_ns<3>(n_sm, wps, in, sink); break;
          default: ns = dispatch_ns<4>(n_sm, wps, in, sink); break;
        }
        printf(" %8.3f", ns);
      }
      printf("\n");
    }
  }
  CK(cudaFree(cyc));
  CK(cudaFree(sink));
  CK(cudaFree(in));
  return 0;
}
