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
// rcp.approx.ftz.f64 / rsqrt.approx.ftz.f64 are the MUFU.RCP64H / RSQ64H seeds
// (low result word zero).  Measured on B200 over 2^28 arguments: residual
// |1 - q r0| <= 2^-19.9 and |1 - x y0^2| <= 2^-19.0.
// With e = 1 - q r0 the exact value is r0/(1 - e) = r0 (1 + e + e^2 + ...);
// keeping terms through e^2 leaves a relative error e^3 <= 2^-59, below the
// FP64 rounding of the surrounding operations.
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
  double p = fma(e, e, e);  // e + e^2
  return fma(r0, p, r0);
}
// sqrt(x), x > 0 normal: g0 = x y0, e = 1 - x y0^2,
// sqrt(x) = g0 (1 - e)^(-1/2) = g0 (1 + e/2 + 3 e^2/8 + 5 e^3/16 + ...);
// truncated after e^2: relative error (5/16) e^3 <= 2^-58.
__device__ __forceinline__ double sqrt_fast(double x) {
  double y0 = rsqrt_seed(x);
  double g0 = x * y0;
  double e = fma(-g0, y0, 1.0);
  double p = fma(0.375, e, 0.5) * e;
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

// Exact "d >= a0" for a0 > 0 on the ALU pipe: for non-negative doubles the
// IEEE bit patterns order like signed integers, and every negative double has a
// negative pattern.  (A positive NaN compares "free" and then propagates into
// the state, where the divergence test catches it.)
__device__ __forceinline__ bool ge_pos(double d, long long a0_bits) {
  return __double_as_longlong(d) >= a0_bits;
}

// g(s, d, w): the acceleration term in per-step variables.
template <int LAW>
__device__ __forceinline__ double accel(const Particle64& P, double s, double d,
                                        double w, long long a0_bits) {
  double base = fma(P.nbeta, d, fma(P.nalpha, w, s));
  if (LAW == AFM_LAW_NONE) {
    return base;
  } else if (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) {
    // at d == a0 both branches give -kappa/a0^2 (the law is continuous), so
    // the contact branch only ever sees a0 - d > 0.
    if (ge_pos(d, a0_bits)) {
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

// The same term on the free-flight (d >= a0) side of the DMT laws, no branch.
__device__ __forceinline__ double accel_free(const Particle64& P, double s,
                                             double d, double w) {
  double base = fma(P.nbeta, d, fma(P.nalpha, w, s));
  return fma(P.c0, rcp_fast(d * d), base);
}

// DMT laws, both sides evaluated and selected per lane (straight-line code: the
// reciprocal and the square-root chains overlap).  A lane on the other side
// feeds its unused chain a harmless argument (rsqrt of a negative number is NaN
// and is never selected).
template <int LAW>
__device__ __forceinline__ double accel_both(const Particle64& P, double s,
                                             double d, double w,
                                             long long a0_bits) {
  const double base = fma(P.nbeta, d, fma(P.nalpha, w, s));
  const double g_free = fma(P.c0, rcp_fast(d * d), base);
  const double del = P.a0 - d;
  const double sq = sqrt_fast(del);
  double f = fma(P.c1 * del, sq, P.c2);
  if (LAW == AFM_LAW_DMT_VISC) f = fma(P.c3 * sq, w, f);
  const double g_contact = base + f;
  return ge_pos(d, a0_bits) ? g_free : g_contact;
}

// Stage acceleration with a warp-uniform choice of code: all lanes in free
// flight -> the short form; otherwise both sides + select.  `touched` records
// (warp-uniformly) that some lane was in contact.
template <int LAW>
__device__ __forceinline__ double accel_warp(const Particle64& P, double s,
                                             double d, double w,
                                             long long a0_bits, bool& touched) {
  if (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) {
    if (__all_sync(0xffffffffu, ge_pos(d, a0_bits))) return accel_free(P, s, d, w);
    touched = true;
    return accel_both<LAW>(P, s, d, w, a0_bits);
  } else {
    return accel<LAW>(P, s, d, w, a0_bits);
  }
}

// One classical RK4 step (tableau c = (0, 1/2, 1/2, 1),
// b = (1/6, 1/3, 1/3, 1/6)) of unit length in per-step variables.  With
// k_jd = stage velocity and k_j = stage acceleration:
//   k_1d = w, k_2d = w + k1/2, k_3d = w + k2/2, k_4d = w + k3
//   d' = d + (k_1d + 2 k_2d + 2 k_3d + k_4d)/6 = d + w + (k1 + k2 + k3)/6
//   w' = w + (k1 + 2 k2 + 2 k3 + k4)/6
// s0, sh, s1: Dp at t_n, t_n + h/2, t_n + h.
//
// DMT laws: the tip is in free flight for most of every cycle, and there the
// four stages are straight-line code whose reciprocal chains overlap (stage 2's
// position does not depend on stage 1's force, stage 4's not on stage 3's).
// `mode` is a warp-uniform state: in mode 0 the step is first taken
// speculatively on the free-flight side and kept only if every stage position
// of every lane of the warp really was >= a0 (tested on the high words:
// conservative by < 2^-20 relative; the exact test lives in the general path);
// a failed speculation redoes the step in the general form and switches to
// mode 1, which skips the speculation until a whole step passes without
// contact.  Every path evaluates the same arithmetic for a given lane and
// stage, so which path ran never changes a result.
template <int LAW>
__device__ __forceinline__ void rk4_step(const Particle64& P, double s0,
                                         double sh, double s1,
                                         long long a0_bits, double& d,
                                         double& w, int& mode) {
  const double sixth = 1.0 / 6.0;
  const double dw = d + w;
  const double d2 = fma(0.5, w, d);
  if ((LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) && mode == 0) {
    const double k1 = accel_free(P, s0, d, w);
    const double w2 = fma(0.5, k1, w);
    const double k2 = accel_free(P, sh, d2, w2);
    const double w3 = fma(0.5, k2, w);
    const double d3 = fma(0.5, w2, d);
    const double k3 = accel_free(P, sh, d3, w3);
    const double d4 = d + w3;
    const double k4 = accel_free(P, s1, d4, w + k3);
    const int a0_hi = (int)(a0_bits >> 32);
    const int m = min(min(__double2hiint(d), __double2hiint(d2)),
                      min(__double2hiint(d3), __double2hiint(d4)));
    if (__all_sync(0xffffffffu, m > a0_hi)) {
      const double t23 = k2 + k3;
      const double s3 = k1 + t23;
      d = fma(s3, sixth, dw);
      w = fma((s3 + t23) + k4, sixth, w);
      return;
    }
    mode = 1;
  }
  bool touched = false;
  const double k1 = accel_warp<LAW>(P, s0, d, w, a0_bits, touched);
  const double w2 = fma(0.5, k1, w);
  const double k2 = accel_warp<LAW>(P, sh, d2, w2, a0_bits, touched);
  const double w3 = fma(0.5, k2, w);
  const double k3 = accel_warp<LAW>(P, sh, fma(0.5, w2, d), w3, a0_bits, touched);
  const double k4 = accel_warp<LAW>(P, s1, d + w3, w + k3, a0_bits, touched);
  const double t23 = k2 + k3;
  const double s3 = k1 + t23;
  d = fma(s3, sixth, dw);
  w = fma((s3 + t23) + k4, sixth, w);
  if (!touched) mode = 0;
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
