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
#include <math_constants.h>
#include <stdint.h>

#include "afm.h"
#include "afm_device_common.cuh"

namespace afm {

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
// c/q + b with the correction folded into the sum: c r0 (1 + p) + b =
// (c r0) p + (c r0 + b).  The two products with r0 run beside the e -> p chain,
// so the result is one dependent FMA after p instead of two (the stage-to-stage
// recurrence of the RK4 step is latency-bound at low occupancy).
__device__ __forceinline__ double vdw_plus(double c, double q, double b) {
  const double r0 = rcp_seed(q);
  const double e = fma(-q, r0, 1.0);
  const double cr0 = c * r0;
  const double cb = fma(c, r0, b);
  const double p = fma(e, e, e);
  return fma(cr0, p, cb);
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

// exp(x) with few instructions and a short dependent chain (the LJ+exp law runs in
// the latency regime: a swarm of 8 192 particles is 256 warps on 592 sub-partitions,
// and a lone warp issues one FP64 instruction every 2.5 cycles).  x = n ln2 + f with
// n = rint(x log2 e), |f| <= 0.3466; exp(f) by a polynomial of degree 11 -- the
// Chebyshev fit on [-ln2/2, ln2/2] (mpmath.chebyfit at 60 digits, coefficients
// rounded to FP64: relative error <= 1.7e-17; the Taylor polynomial needs degree 13
// for that) -- evaluated by Estrin's scheme: four FMA levels; 2^n goes into the
// exponent field.  n is clamped on the ALU pipe (two FP64 compares and four selects
// on the result cost 15 % of a configs[3] batch): at n = 1024 the exponent field is
// all ones (non-finite: a diverging trajectory, R12), at n = -1022 the result is
// below 2^-1021 (the true value is smaller still; the adhesion term vanishes against
// any tolerance either way).
__device__ __forceinline__ double exp_fast(double x) {
  const double magic = 6755399441055744.0;  // 1.5 * 2^52: rint by add/sub
  const double nm = fma(x, 1.4426950408889634, magic);
  const double n = nm - magic;
  double f = fma(n, -6.93147180369123816490e-01, x);  // ln2 high part
  f = fma(n, -1.90821492927058770002e-10, f);         // ln2 low part
  const double f2 = f * f;
  const double a0 = f + 1.0;
  const double a1 = fma(f, 0.1666666666666668, 0.5000000000000019);
  const double a2 = fma(f, 0.008333333333319601, 0.0416666666664881);
  const double a3 = fma(f, 0.00019841269890047113, 0.0013888888952314775);
  const double a4 = fma(f, 2.755724091857897e-06, 2.4801485482328494e-05);
  const double a5 = fma(f, 2.5110037605963777e-08, 2.763263963904103e-07);
  const double f4 = f2 * f2;
  const double b0 = fma(a1, f2, a0);
  const double b1 = fma(a3, f2, a2);
  const double b2 = fma(a5, f2, a4);
  const double f8 = f4 * f4;
  const double g0 = fma(b1, f4, b0);
  const double pv = fma(b2, f8, g0);
  // 2^n into the exponent: n is the low word of nm (two's complement)
  const int nc = max(min(__double2loint(nm), 1024), -1022);
  return __hiloint2double(__double2hiint(pv) + (nc << 20), __double2loint(pv));
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

// g(s, d, w) = s - alpha w - beta d + f(d, w): the acceleration term in
// per-step variables.  The stage velocity w is the last operand to arrive, so
// everything else is folded first and w enters through one final FMA.

// Free-flight (d >= a0) side of the DMT laws, and the whole of law NONE when
// c0 = 0 is skipped by the caller.
// WFOLD (latency form only): the stage velocity is already known when the
// reciprocal chain starts (stages 1 and 3: w, and w3 which comes from the short
// k2 path), so -alpha w joins the constant term and the stage ends with the one
// FMA after the correction polynomial; in stages 2 and 4 w is the last operand to
// arrive and enters through a final FMA.
template <bool LAT, bool WFOLD = false>
__device__ __forceinline__ double accel_free(const Particle64& P, double s,
                                             double d, double w) {
  const double b0 = fma(P.nbeta, d, s);
  if (LAT && WFOLD) return vdw_plus(P.c0, d * d, fma(P.nalpha, w, b0));
  if (LAT) return fma(P.nalpha, w, vdw_plus(P.c0, d * d, b0));
  return fma(P.nalpha, w, fma(P.c0, rcp_fast(d * d), b0));
}

// DMT laws, both sides evaluated and selected per lane (straight-line code: the
// reciprocal and the square-root chains are independent and overlap).  A lane
// on the other side feeds its unused chain a harmless argument (rsqrt of a
// negative number is NaN and is never selected).  The free-flight value is
// computed exactly as in accel_free<LAT>, so within one form a lane's result
// does not depend on which path ran.
// (Measured and rejected: one shared rsqrt chain on a per-lane selected argument
// with selected tail coefficients -- 14 instead of 19 FP64 instructions per
// stage, but ten more 32-bit selects; 19.8 ms against 19.1 ms on configs[1].)
template <int LAW, bool LAT, bool WFOLD = false>
__device__ __forceinline__ double accel_both(const Particle64& P, double s,
                                             double d, double w,
                                             long long a0_bits) {
  const double b0 = fma(P.nbeta, d, s);
  const double g_free =
      (LAT && WFOLD) ? vdw_plus(P.c0, d * d, fma(P.nalpha, w, b0))
      : LAT          ? fma(P.nalpha, w, vdw_plus(P.c0, d * d, b0))
                     : fma(P.nalpha, w, fma(P.c0, rcp_fast(d * d), b0));
  const double del = P.a0 - d;
  if (WFOLD && (LAT || LAW != AFM_LAW_DMT_VISC)) {
    // stages 1 and 3 (their velocity is known before the square-root chain ends):
    // the correction of the square root is folded into the sum,
    //   c1 del sqrt(del) [+ c3 sqrt(del) w] = M (1 + p),  M = (c1 del [+ c3 w]) g0,
    // so the stage ends one FMA after p instead of three operations (the general
    // form is what the slowest warp of a batch runs, and a lone warp in the latency
    // regime: configs[1] 12.21 -> 12.03 ms, configs[2] 693 -> 671 ms, configs[0]
    // 6.05 -> 5.90 ms).  One more instruction for the plain DMT law, three more
    // with the viscous term: there the throughput form keeps the short count
    // (configs[4] 54.7 ms against 55.4).
    const double y0 = rsqrt_seed(del);
    const double g0 = del * y0;
    const double e = fma(-g0, y0, 1.0);
    const double p = fma(0.375, e, 0.5) * e;
    const double cm = (LAW == AFM_LAW_DMT_VISC) ? fma(P.c3, w, P.c1 * del) : P.c1 * del;
    const double M = cm * g0;
    const double R = fma(P.nalpha, w, P.c2 + b0);
    const double g_c = fma(M, p, M + R);
    return ge_pos(d, a0_bits) ? g_free : g_c;
  }
  const double sq = sqrt_fast(del);
  const double part = fma(P.c1 * del, sq, P.c2 + b0);
  // viscous term -nu sqrt(delta) w joins the -alpha w term: one coefficient
  const double cw = (LAW == AFM_LAW_DMT_VISC) ? fma(P.c3, sq, P.nalpha) : P.nalpha;
  const double g_contact = fma(cw, w, part);
  return ge_pos(d, a0_bits) ? g_free : g_contact;
}

// Laws without a contact switch.
template <int LAW>
__device__ __forceinline__ double accel_smooth(const Particle64& P, double s,
                                               double d, double w) {
  const double b0 = fma(P.nbeta, d, s);
  if (LAW == AFM_LAW_LJ_EXP) {
    const double r = rcp_fast(d * d);
    const double r2 = r * r;
    const double r4 = r2 * r2;
    // the exponential is the last operand to arrive (its chain is the longer one),
    // so everything else is summed before it (configs[3] FP64 batch 22.1 -> 21.2 ms)
    const double g = fma(P.nalpha, w, fma(P.c0, r4, fma(P.c1, r, b0)));
    return fma(P.c2, exp_fast(d * P.c3), g);
  }
  if (LAW == AFM_LAW_HOOKE || LAW == AFM_LAW_KELVIN_VOIGT) {
    // the paper's sample models (Eq. 11, 12): a spring (and a damper) that act
    // while the tip is pressed in, d < P.a0 (= z_c - h for Hooke, 0 for
    // Kelvin-Voigt).  Coefficients selected per lane, then two FMAs.
    const bool in = d < P.a0;
    const double ks = in ? P.c1 : 0.0;
    const double cw = (LAW == AFM_LAW_KELVIN_VOIGT && in) ? P.c3 : P.nalpha;
    return fma(cw, w, fma(ks, P.a0 - d, b0));
  }
  return fma(P.nalpha, w, b0);  // AFM_LAW_NONE
}

template <int LAW>
struct IsDmt {
  static constexpr bool value = (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC);
};

// Monotone integer key of a double (total order equal to the numeric order
// for non-NaN; +NaN above +Inf, -NaN below -Inf), for the divergence test on
// the ALU pipe instead of two FP64 compares.
__device__ __forceinline__ long long order_key(double x) {
  long long b = __double_as_longlong(x);
  return b ^ ((b >> 63) & 0x7fffffffffffffffLL);
}

// Divergence rule R12 on d = z + z_c, every step: |z| > 100 A0 or non-finite.
// Cheap sound filter first (ALU pipe, high word only): |d| below the double
// whose high word is `safe_hi` implies |z| <= 100 A0; only a suspect value
// takes the exact two-sided test.
struct DivergeTest {
  long long key_min, key_max;  // order_key(z_c -+ 100 A0)
  int safe_hi;                 // high word of max(0, 100 A0 - |z_c|)
};
__device__ __forceinline__ bool diverged_step(double d, const DivergeTest& T) {
  const int hi = __double2hiint(d) & 0x7fffffff;
  if (__builtin_expect(hi >= T.safe_hi, 0)) {
    const long long key = order_key(d);
    return (key > T.key_max) | (key < T.key_min);
  }
  return false;
}

// Stage-3 position and the RK4 combination.  d3 = d2 + k1/4 (= d + w2/2 without
// waiting for w2: one dependent operation fewer, same instruction count) in both
// forms (configs[1]: 12.89 -> 12.68 ms in the throughput form).  The combination in
// the throughput form is the textbook association with the fewest operations; in
// the latency form the same sums are associated so that the loop-carried chain
// d_n -> k1 -> d3 -> k3 -> d_{n+1} is as short as it can be:
// d_{n+1} = [d + w + (k1 + k2)/6] + k3/6 (one FMA after k3); two more additions,
// two fewer dependent operations per step (8.1 cycles each).  (In the
// throughput form that association, the folded van der Waals term and the folded
// -alpha w each cost more than they save: 12.99, 13.69 and 13.27 ms.)
__device__ __forceinline__ double stage3_gap(double d2, double k1) {
  return fma(0.25, k1, d2);
}
template <bool LAT>
__device__ __forceinline__ void rk4_combine(double dw, double w, double k1, double k2,
                                            double k3, double k4, double& dn,
                                            double& wn) {
  const double sixth = 1.0 / 6.0;
  if (LAT) {
    const double a12 = k1 + k2;
    dn = fma(k3, sixth, fma(a12, sixth, dw));
    // w' one FMA after k4 and two after k3 (k1 + 2 k2 is ready before k3): the next
    // step's first stage takes w' into its constant term, and w' used to arrive
    // after that stage's reciprocal (configs[2] 671 -> 641 ms, configs[0] 5.9 -> 5.7)
    wn = fma(k4, sixth, fma(fma(2.0, k3, fma(2.0, k2, k1)), sixth, w));
  } else {
    const double t23 = k2 + k3;
    const double s3 = k1 + t23;
    dn = fma(s3, sixth, dw);
    wn = fma((s3 + t23) + k4, sixth, w);
  }
}

// One speculative free-flight step of one particle, without the vote: new state
// in (dn, wn); returns whether this lane's four stage gaps stayed above a0 and the
// new gap is a positive number below the divergence filter -- the conditions
// under which the step may be kept (see rk4_step).
template <bool LAT>
__device__ __forceinline__ bool free_step(const Particle64& P, double s0, double sh,
                                          double s1, long long a0_bits,
                                          const DivergeTest& T, double d, double w,
                                          double& dn, double& wn) {
  const double dw = d + w;
  const double d2 = fma(0.5, w, d);
  const double k1 = accel_free<LAT, true>(P, s0, d, w);
  const double w2 = fma(0.5, k1, w);
  const double k2 = accel_free<LAT, false>(P, sh, d2, w2);
  const double w3 = fma(0.5, k2, w);
  const double d3 = stage3_gap(d2, k1);
  const double k3 = accel_free<LAT, true>(P, sh, d3, w3);
  const double d4 = d + w3;
  const double k4 = accel_free<LAT, false>(P, s1, d4, w + k3);
  const int m = min(min(__double2hiint(d), __double2hiint(d2)),
                    min(__double2hiint(d3), __double2hiint(d4)));
  rk4_combine<LAT>(dw, w, k1, k2, k3, k4, dn, wn);
  // unsigned compare: a negative or NaN high word is huge
  return (m > (int)(a0_bits >> 32)) &
         ((unsigned)__double2hiint(dn) < (unsigned)T.safe_hi);
}

// One classical RK4 step (tableau c = (0, 1/2, 1/2, 1),
// b = (1/6, 1/3, 1/3, 1/6)) of unit length in per-step variables, for the PPT
// particles of one thread.  With k_jd = stage velocity, k_j = stage acceleration:
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
// of every particle of the warp really was >= a0 (tested on the high words:
// conservative by < 2^-20 relative; the exact test lives in the general path);
// a failed speculation redoes the step in the general form and switches to
// mode 1, which skips the speculation until a whole step passes without
// contact.  The general form evaluates both sides of the law in every stage
// and selects per lane.  A given particle and stage sees the same arithmetic
// whichever path ran, so the path never changes a result.
template <int LAW, int PPT, bool LAT>
__device__ __forceinline__ void rk4_step(const Particle64 (&P)[PPT], double s0,
                                         double sh, double s1,
                                         long long a0_bits, double (&d)[PPT],
                                         double (&w)[PPT], int& mode,
                                         bool (&bad)[PPT],
                                         const DivergeTest& T) {
  double dw[PPT], d2[PPT];
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    dw[q] = d[q] + w[q];
    d2[q] = fma(0.5, w[q], d[q]);
  }
  if (!IsDmt<LAW>::value) {
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
      const double k1 = accel_smooth<LAW>(P[q], s0, d[q], w[q]);
      const double w2 = fma(0.5, k1, w[q]);
      const double k2 = accel_smooth<LAW>(P[q], sh, d2[q], w2);
      const double w3 = fma(0.5, k2, w[q]);
      const double k3 =
          accel_smooth<LAW>(P[q], sh, stage3_gap(d2[q], k1), w3);
      const double k4 = accel_smooth<LAW>(P[q], s1, fma(0.5, k2, dw[q]), w[q] + k3);  // = d + w3
      rk4_combine<LAT>(dw[q], w[q], k1, k2, k3, k4, d[q], w[q]);
      bad[q] |= diverged_step(d[q], T);
    }
    return;
  }
  if (mode == 0) {
    double dn[PPT], wn[PPT];
    bool ok = true;
#pragma unroll
    for (int q = 0; q < PPT; ++q)
      ok &= free_step<LAT>(P[q], s0, sh, s1, a0_bits, T, d[q], w[q], dn[q], wn[q]);
    // kept only if no stage touched the sample and the new gap is a positive
    // number below the divergence filter -- so a kept step needs no divergence test
    if (__all_sync(0xffffffffu, ok)) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) {
        d[q] = dn[q];
        w[q] = wn[q];
      }
      return;
    }
    mode = 1;
  }
  // general form: every stage evaluates both sides of the law and selects per
  // lane -- straight-line code, no vote between the stages, so the four
  // reciprocal and four square-root chains overlap like in the fast form
  int m = 0x7fffffff;
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    const double k1 = accel_both<LAW, LAT, true>(P[q], s0, d[q], w[q], a0_bits);
    const double w2 = fma(0.5, k1, w[q]);
    const double k2 = accel_both<LAW, LAT, false>(P[q], sh, d2[q], w2, a0_bits);
    const double w3 = fma(0.5, k2, w[q]);
    const double d3 = stage3_gap(d2[q], k1);
    const double k3 = accel_both<LAW, LAT, true>(P[q], sh, d3, w3, a0_bits);
    const double d4 = d[q] + w3;
    const double k4 = accel_both<LAW, LAT, false>(P[q], s1, d4, w[q] + k3, a0_bits);
    m = min(m, min(min(__double2hiint(d[q]), __double2hiint(d2[q])),
                   min(__double2hiint(d3), __double2hiint(d4))));
    rk4_combine<LAT>(dw[q], w[q], k1, k2, k3, k4, d[q], w[q]);
    bad[q] |= diverged_step(d[q], T);
  }
  // back to speculation once a whole step stayed clear of the sample
  if (__all_sync(0xffffffffu, m > (int)(a0_bits >> 32))) mode = 0;
}

// Scaled law coefficients from physical parameters theta.
__device__ __forceinline__ void load_particle(Particle64& P, int law,
                                              const double* th, double alpha,
                                              double beta, double a0,
                                              double inv_a0sq, double c_vdw,
                                              double c_hertz, double c_visc,
                                              double c_force, double zc,
                                              double c_damp) {
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
  } else if (law == AFM_LAW_HOOKE) {
    P.c1 = th[0] * c_force;          // (h^2/m) k_s
    P.a0 = zc - th[1];               // pressed in while z + h < 0, i.e. d < z_c - h
  } else if (law == AFM_LAW_KELVIN_VOIGT) {
    P.c1 = th[0] * c_force;
    P.a0 = 0.0;
    P.c3 = -alpha - th[1] * c_damp;  // -(alpha + (h/m) zeta_s)
  }
}

}  // namespace afm
