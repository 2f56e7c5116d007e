// afm_device_f32.cuh -- device-side arithmetic of the FP32 forward solve
// (reading R14 and section 6 "integrate_misfit_f32").
//
// Kernel units: length 1 nm, one RK4 step = unit time.  State per particle:
// gap d = z + z_c [nm] and per-step displacement w = h z' [nm per step], each
// carried as an unevaluated sum of two floats (hi + lo).  Stage accelerations
// are evaluated in plain FP32 on the hi parts and are pre-scaled by 1/6 on the
// host (alpha6 = alpha/6, beta6 = beta/6, stream s6 = Dp/6, law coefficients
// /6), so that the classical RK4 combination
//     w' = w + (k1 + 2 k2 + 2 k3 + k4)/6,   d' = d + w + (k1 + k2 + k3)/6
// needs no multiplication by the inexact constant 1/6:
//     g_j = k_j/6:  w2 = w + 3 g1, w3 = w + 3 g2, w4 = w + 6 g3,
//     w' = w + (g1 + 2 g2 + 2 g3 + g4),  d' = d + w + (g1 + g2 + g3).
//
// Why the lo parts: with Q = 100..400 the resonant cantilever integrates
// every systematic 1e-8-relative error of the linear terms over ~Q cycles.  A
// rounded beta6 (or a rounded stream value shared by all particles) shows up as
// a 1e-4..1e-3 relative misfit error.  The first-order residuals of everything
// that is rounded once and used every step are therefore added back into the
// lo parts once per step:
//     cc = -beta6_lo d_mid - alpha6_lo w_mid - beta6 d_lo
// (d_mid, w_mid: stage-2 values = the weighted mean stage argument to first
// order) enters w' with weight 6 and d' with weight 3, and the stream carries
// e_w = exact (s0 + 4 sh + s1)/6 minus the float sum actually used.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "afm.h"

namespace afm {

// ---- MUFU approximations (1 ulp class; SASS MUFU.RCP / MUFU.SQRT / MUFU.EX2) -
__device__ __forceinline__ float rcp32(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float sqrt32(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float ex2_32(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// Error-free sum (Knuth): s + e = a + b exactly, no ordering assumption.
// Written with explicit round-to-nearest intrinsics so that the compiler can
// neither contract nor re-associate it.
__device__ __forceinline__ void two_sum32(float a, float b, float& s, float& e) {
  s = __fadd_rn(a, b);
  const float bb = __fsub_rn(s, a);
  e = __fadd_rn(__fsub_rn(a, __fsub_rn(s, bb)), __fsub_rn(b, bb));
}

// Uniform (per-launch) model coefficients, all pre-scaled by 1/6.
struct Model32 {
  float nalpha, nbeta;        // -alpha/6, -beta/6 (rounded)
  float nalpha_lo, nbeta_lo;  // -(alpha/6 - fl(alpha/6)), same for beta
  float a0;                   // nm
  float d_safe;               // |d| < d_safe => not diverged (R12)
  float d_max, d_min;         // z_c +- 100 A0, nm
};

// Per-particle law coefficients (scaled by beta/6 and the unit factors):
//   DMT:    c0 = -kappa, c1 = eps, c2 = -kappa/a0^2, c3 = -nu
//   LJ_EXP: c0 = crep,   c1 = -catt, c2 = -fad,      c3 = -log2(e)/lambda
//   HOOKE / KELVIN_VOIGT: c1 = spring, c3 = -(alpha/6 + damper), thr = contact
//           threshold on d (z_c - h, or 0)
struct Particle32 {
  float c0, c1, c2, c3;
  float thr;
};

__device__ __forceinline__ float accel_free32(const Model32& M,
                                              const Particle32& P, float s,
                                              float d, float w) {
  const float part = fmaf(P.c0, rcp32(d * d), fmaf(M.nbeta, d, s));
  return fmaf(M.nalpha, w, part);
}

template <int LAW>
__device__ __forceinline__ float accel_both32(const Model32& M,
                                              const Particle32& P, float s,
                                              float d, float w) {
  const float b0 = fmaf(M.nbeta, d, s);
  const float g_free = fmaf(M.nalpha, w, fmaf(P.c0, rcp32(d * d), b0));
  const float del = M.a0 - d;
  const float sq = sqrt32(fmaxf(del, 0.0f));
  const float part = fmaf(P.c1 * del, sq, P.c2 + b0);
  const float cw = (LAW == AFM_LAW_DMT_VISC) ? fmaf(P.c3, sq, M.nalpha) : M.nalpha;
  const float g_contact = fmaf(cw, w, part);
  return (d >= M.a0) ? g_free : g_contact;
}

template <int LAW>
__device__ __forceinline__ float accel_smooth32(const Model32& M,
                                                const Particle32& P, float s,
                                                float d, float w) {
  const float b0 = fmaf(M.nbeta, d, s);
  if (LAW == AFM_LAW_LJ_EXP) {
    const float r = rcp32(d * d);
    const float r2 = r * r;
    const float r4 = r2 * r2;
    float f = fmaf(P.c0, r4, fmaf(P.c1, r, b0));
    f = fmaf(P.c2, ex2_32(d * P.c3), f);
    return fmaf(M.nalpha, w, f);
  }
  if (LAW == AFM_LAW_HOOKE || LAW == AFM_LAW_KELVIN_VOIGT) {
    const bool in = d < P.thr;
    const float ks = in ? P.c1 : 0.0f;
    const float cw = (LAW == AFM_LAW_KELVIN_VOIGT && in) ? P.c3 : M.nalpha;
    return fmaf(cw, w, fmaf(ks, P.thr - d, b0));
  }
  return fmaf(M.nalpha, w, b0);  // AFM_LAW_NONE
}

// Compensated state of one particle.
struct State32 {
  float dh, dl, wh, wl;
};

// Fold the four scaled stage accelerations into the compensated state.
//   d2, w2: stage-2 arguments (for the lo-part correction), ew: stream residual
__device__ __forceinline__ void commit32(const Model32& M, State32& S, float g1,
                                         float g2, float g3, float g4, float d2,
                                         float w2, float ew) {
  const float t23 = g2 + g3;
  const float s3 = g1 + t23;
  const float X = (s3 + t23) + g4;
  const float cc = fmaf(M.nbeta, S.dl, fmaf(M.nbeta_lo, d2, M.nalpha_lo * w2));
  // d' = d + w + s3 (+ 3 cc).  The large part w_hi is added by a fast two-sum:
  // exact while |d_hi| >= |w_hi|; when the gap is smaller than one step's
  // travel (deep contact) its error is <= ulp(w_hi) ~ 1e-8 nm, once.
  const float sd = __fadd_rn(S.dh, S.wh);
  const float e = __fsub_rn(S.wh, __fsub_rn(sd, S.dh));
  // everything but g3 is summed before g3 arrives, so that d' is two additions
  // after g3 (the loop-carried chain; configs[3] FP32 batch 6.36 -> 5.77 ms, and
  // 7.25 -> 6.36 ms from the stage-3 gap taken as d2 + 1.5 g1)
  const float lo = __fadd_rn(
      __fadd_rn(__fadd_rn(__fadd_rn(S.dl, fmaf(3.0f, cc, S.wl)), e), __fadd_rn(g1, g2)), g3);
  const float dn = __fadd_rn(sd, lo);
  S.dl = __fsub_rn(lo, __fsub_rn(dn, sd));
  S.dh = dn;
  // w' = w + X (+ 6 cc + ew): |X| << |w_hi| except where w crosses zero, and
  // there the error is <= ulp(X) -- the rounding X carries anyway
  const float t = __fadd_rn(__fadd_rn(S.wl, fmaf(6.0f, cc, ew)), X);
  const float wn = __fadd_rn(S.wh, t);
  S.wl = __fsub_rn(t, __fsub_rn(wn, S.wh));
  S.wh = wn;
}

template <int LAW>
struct IsDmt32 {
  static constexpr bool value = (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC);
};

// One classical RK4 step for the PPT particles of a thread.  Same warp-uniform
// two-mode scheme as the FP64 kernel (afm_device.cuh): mode 0 takes the step
// speculatively with the free-flight law and keeps it only if every stage gap
// of every lane was >= a0 and the new gap is inside the divergence filter.
template <int LAW, int PPT>
__device__ __forceinline__ void rk4_step32(const Model32& M,
                                           const Particle32 (&P)[PPT], float s0,
                                           float sh, float s1, float ew,
                                           State32 (&S)[PPT], int& mode,
                                           bool (&bad)[PPT]) {
  if (!IsDmt32<LAW>::value) {
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
      const float d = S[q].dh, w = S[q].wh;
      const float g1 = accel_smooth32<LAW>(M, P[q], s0, d, w);
      const float w2 = fmaf(3.0f, g1, w);
      const float d2 = fmaf(0.5f, w, d);
      const float g2 = accel_smooth32<LAW>(M, P[q], sh, d2, w2);
      const float w3 = fmaf(3.0f, g2, w);
      const float g3 = accel_smooth32<LAW>(M, P[q], sh, fmaf(1.5f, g1, d2), w3);
      const float g4 = accel_smooth32<LAW>(M, P[q], s1, d + w3, fmaf(6.0f, g3, w));
      commit32(M, S[q], g1, g2, g3, g4, d2, w2, ew);
      // NaN fails the comparison and is flagged
      bad[q] |= !(fabsf(S[q].dh) < M.d_safe) &&
                !(S[q].dh <= M.d_max && S[q].dh >= M.d_min);
    }
    return;
  }
  if (mode == 0) {
    State32 Sn[PPT];
    bool ok = true;
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
      const float d = S[q].dh, w = S[q].wh;
      const float g1 = accel_free32(M, P[q], s0, d, w);
      const float w2 = fmaf(3.0f, g1, w);
      const float d2 = fmaf(0.5f, w, d);
      const float g2 = accel_free32(M, P[q], sh, d2, w2);
      const float w3 = fmaf(3.0f, g2, w);
      const float d3 = fmaf(1.5f, g1, d2);  // = d + w2/2 without waiting for w2
      const float g3 = accel_free32(M, P[q], sh, d3, w3);
      const float d4 = d + w3;
      const float g4 = accel_free32(M, P[q], s1, d4, fmaf(6.0f, g3, w));
      Sn[q] = S[q];
      commit32(M, Sn[q], g1, g2, g3, g4, d2, w2, ew);
      const float m = fminf(fminf(d, d2), fminf(d3, d4));
      ok = ok && (m >= M.a0) && (fabsf(Sn[q].dh) < M.d_safe);
    }
    if (__all_sync(0xffffffffu, ok)) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) S[q] = Sn[q];
      return;
    }
    mode = 1;
  }
  bool clear = true;
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    const float d = S[q].dh, w = S[q].wh;
    const float g1 = accel_both32<LAW>(M, P[q], s0, d, w);
    const float w2 = fmaf(3.0f, g1, w);
    const float d2 = fmaf(0.5f, w, d);
    const float g2 = accel_both32<LAW>(M, P[q], sh, d2, w2);
    const float w3 = fmaf(3.0f, g2, w);
    const float d3 = fmaf(1.5f, g1, d2);  // = d + w2/2 without waiting for w2
    const float g3 = accel_both32<LAW>(M, P[q], sh, d3, w3);
    const float d4 = d + w3;
    const float g4 = accel_both32<LAW>(M, P[q], s1, d4, fmaf(6.0f, g3, w));
    commit32(M, S[q], g1, g2, g3, g4, d2, w2, ew);
    const float m = fminf(fminf(d, d2), fminf(d3, d4));
    clear = clear && (m >= M.a0);
    bad[q] |= !(fabsf(S[q].dh) < M.d_safe) &&
              !(S[q].dh <= M.d_max && S[q].dh >= M.d_min);
  }
  if (__all_sync(0xffffffffu, clear)) mode = 0;
}

}  // namespace afm
