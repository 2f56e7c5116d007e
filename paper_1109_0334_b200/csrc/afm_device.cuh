// afm_device.cuh -- device-side arithmetic of the forward solve (FP64):
// short reciprocal / square-root sequences on the MUFU seeds, the three
// tip-sample force laws in per-step variables, one classical RK4 step, and the
// PTX wrappers for the TMA-staged (cp.async.bulk + mbarrier) time-tile ring.
//
// Variables (see afm_internal.h): d = z + z_c [m], w = h z' [m per step],
//     w' = g(s, d, w) = s - alpha w - beta d + f(d, w),
// s = Dp(t) read from the time-tile stream, f = (h^2/m) F_ts.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "afm.h"

namespace afm {

// ---- mbarrier / bulk-copy PTX (sm_90+; SASS: SYNCS.*, UBLKCP) ---------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(count)
               : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar,
                                                      uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(
                   smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
// 1-D bulk async copy global -> shared, completion counted on an mbarrier.
// dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src,
                                         uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "AFM_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra AFM_DONE;\n"
      "bra AFM_WAIT;\n"
      "AFM_DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// ---- short FP64 reciprocal / sqrt ------------------------------------------
// rcp.approx.ftz.f64 / rsqrt.approx.ftz.f64 are the MUFU.RCP64H / RSQ64H
// seeds (about 20 good bits, low word zero).  With residual e = 1 - q r0 the
// exact value is r0 / (1 - e) = r0 (1 + e + e^2 + e^3 + ...); keeping terms
// through e^3 leaves a relative error of e^4 < 2^-70, below FP64 rounding.
__device__ __forceinline__ double rcp_seed(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double rsqrt_seed(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double rcp_fast(double q) {
  double r0 = rcp_seed(q);
  double e = fma(-q, r0, 1.0);
  double p = fma(e, e, e);   // e + e^2
  p = fma(p, e, e);          // e + e^2 + e^3
  return fma(r0, p, r0);
}
// sqrt(x), x > 0 normal: g0 = x y0, e = 1 - x y0^2,
// sqrt(x) = g0 (1 - e)^(-1/2) = g0 (1 + e/2 + 3 e^2/8 + 5 e^3/16 + ...).
__device__ __forceinline__ double sqrt_fast(double x) {
  double y0 = rsqrt_seed(x);
  double g0 = x * y0;
  double e = fma(-g0, y0, 1.0);
  double p = fma(0.3125, e, 0.375);
  p = fma(p, e, 0.5);
  p = p * e;
  return fma(g0, p, g0);
}

// ---- per-particle constants in registers ------------------------------------
struct Particle64 {
  double nalpha;  // -alpha
  double nbeta;   // -beta
  double a0;
  // law coefficients (scaled):
  //   DMT:    c0 = -kappa, c1 = eps, c2 = -kappa/a0^2, c3 = -nu
  //   LJ_EXP: c0 = crep,   c1 = -catt, c2 = -fad,      c3 = -1/lambda
  double c0, c1, c2, c3;
};

// g(s, d, w): the acceleration term in per-step variables.
template <int LAW>
__device__ __forceinline__ double accel(const Particle64& P, double s, double d,
                                        double w) {
  double base = fma(P.nbeta, d, fma(P.nalpha, w, s));
  if (LAW == AFM_LAW_NONE) {
    return base;
  } else if (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) {
    // at d == a0 both branches give -kappa/a0^2 (the law is continuous), so
    // the contact branch only ever sees a0 - d > 0.
    if (d >= P.a0) {
      double r = rcp_fast(d * d);
      return fma(P.c0, r, base);
    } else {
      double del = P.a0 - d;
      double sq = sqrt_fast(del);
      double f = fma(P.c1 * del, sq, P.c2);
      if (LAW == AFM_LAW_DMT_VISC) f = fma(P.c3 * sq, w, f);
      return base + f;
    }
  } else {  // AFM_LAW_LJ_EXP
    double r = rcp_fast(d * d);
    double r2 = r * r;
    double r4 = r2 * r2;
    double f = fma(P.c0, r4, P.c1 * r);
    double ex = exp(d * P.c3);
    f = fma(P.c2, ex, f);
    return base + f;
  }
}

// One classical RK4 step (tableau c = (0, 1/2, 1/2, 1),
// b = (1/6, 1/3, 1/3, 1/6)) of unit length in per-step variables.  With
// k_jd = stage velocity and k_j = stage acceleration:
//   k_1d = w, k_2d = w + k1/2, k_3d = w + k2/2, k_4d = w + k3
//   d' = d + (k_1d + 2 k_2d + 2 k_3d + k_4d)/6 = d + w + (k1 + k2 + k3)/6
//   w' = w + (k1 + 2 k2 + 2 k3 + k4)/6
// s0, sh, s1: Dp at t_n, t_n + h/2, t_n + h.
template <int LAW>
__device__ __forceinline__ void rk4_step(const Particle64& P, double s0,
                                         double sh, double s1, double& d,
                                         double& w) {
  const double sixth = 1.0 / 6.0;
  double dw = d + w;
  double k1 = accel<LAW>(P, s0, d, w);
  double w2 = fma(0.5, k1, w);
  double k2 = accel<LAW>(P, sh, fma(0.5, w, d), w2);
  double w3 = fma(0.5, k2, w);
  double k3 = accel<LAW>(P, sh, fma(0.5, w2, d), w3);
  double k4 = accel<LAW>(P, s1, d + w3, w + k3);
  double t23 = k2 + k3;
  double s3 = k1 + t23;
  d = fma(s3, sixth, dw);
  w = fma((s3 + t23) + k4, sixth, w);
}

// Monotone integer key of a double (total order equal to the numeric order
// for non-NaN; +NaN above +Inf, -NaN below -Inf), for the divergence test on
// the ALU pipe instead of two FP64 compares.
__device__ __forceinline__ long long order_key(double x) {
  long long b = __double_as_longlong(x);
  return b ^ ((b >> 63) & 0x7fffffffffffffffLL);
}

// Scaled law coefficients from physical parameters theta.
__device__ __forceinline__ void load_particle(Particle64& P, int law,
                                              const double* th, double alpha,
                                              double beta, double a0,
                                              double inv_a0sq, double c_vdw,
                                              double c_hertz, double c_visc,
                                              double c_force) {
  P.nalpha = -alpha;
  P.nbeta = -beta;
  P.a0 = a0;
  P.c0 = P.c1 = P.c2 = P.c3 = 0.0;
  if (law == AFM_LAW_DMT || law == AFM_LAW_DMT_VISC) {
    double kappa = th[0] * c_vdw;
    P.c0 = -kappa;
    P.c1 = th[1] * c_hertz;
    P.c2 = -kappa * inv_a0sq;
    if (law == AFM_LAW_DMT_VISC) P.c3 = -(th[2] * c_visc);
  } else if (law == AFM_LAW_LJ_EXP) {
    P.c0 = th[0] * c_force;
    P.c1 = -(th[1] * c_force);
    P.c2 = -(th[2] * c_force);
    P.c3 = -1.0 / th[3];
  }
}

}  // namespace afm
