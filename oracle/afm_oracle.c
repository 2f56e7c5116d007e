/*
 * afm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See afm_oracle.h.
 *
 * Written from PAPER.md (arxiv/paper_1109_0334) and BASELINE.json:north_star;
 * every function cites the passage it follows.  No blocking, fusion or
 * reordering beyond what the cited definition states.  Compile with
 *   gcc -O2 -ffp-contract=off -fno-fast-math
 */
#include "afm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------
 * Constants of the m = 1 case of Eq. 2 written as the
 * point-mass equation of BASELINE.json:north_star:
 *     m z'' + (m w0/Q) z' + k z = F0 cos(w t) + F_ts(z + z_c; theta).
 * F0 is chosen so that the free (F_ts = 0) steady-state amplitude is A0:
 *     A = (F0/k) / sqrt((1-r^2)^2 + (r/Q)^2),  r = w/w0
 * (SURVEY.md 8(c) step 1).  dt = one drive period / S.
 * ---------------------------------------------------------------------- */
void orc_constants(const orc_model* M, orc_consts* C) {
  C->w0 = 2.0 * M_PI * M->f0;
  C->w = 2.0 * M_PI * M->f_drive;
  C->m = M->k / (C->w0 * C->w0);
  C->c = C->m * C->w0 / M->Q;
  C->r = C->w / C->w0;
  {
    double a = 1.0 - C->r * C->r;
    double b = C->r / M->Q;
    C->F0 = M->k * M->A0 * sqrt(a * a + b * b);
  }
  C->dt = 2.0 * M_PI / (C->w * (double)M->S);
  C->N = (int64_t)M->S * (int64_t)M->n_cycles;
  C->W = (int64_t)M->S * (int64_t)(M->n_cycles - M->n_skip);
}

/* ------------------------------------------------------------------------
 * Tip-sample force laws, BASELINE.json configs[0], [2], [3]
 * ("Hertzian contact and Van der Waals forces").
 *   DMT:      d >  a0:  -H R / (6 d^2)
 *             d <= a0:  -H R / (6 a0^2) + (4/3) E* sqrt(R) (a0-d)^{3/2}
 *   DMT+visc: additionally, for d <= a0:  - eta sqrt(R (a0-d)) d'
 *   LJ+exp:   C_rep/d^8 - C_att/d^2 - F_ad exp(-d/lambda)
 * The paper's own two sample models (R19/R20),
 * active only while the tip is pressed into the sample (gap < 0):
 *   Hooke (Eq. 11):  f = -k_s (u - h), theta = (k_s, h); the
 *     cantilever-sample separation h is an unknown and replaces z_c: the gap
 *     is z + h = d - z_c + h, and F = -k_s (z + h) for z + h < 0, else 0.
 *   Kelvin-Voigt (Eq. 12):  f = -k_s (u - h) - zeta_s u',
 *     theta = (k_s, zeta_s), separation known (= z_c):
 *     F = -k_s d - zeta_s v for d < 0, else 0.
 * (a0-d)^{3/2} is evaluated as delta*sqrt(delta); 1/d^8 as 1/((d^2)^2)^2.
 * ---------------------------------------------------------------------- */
double orc_force(const orc_model* M, const double* theta, double d, double v) {
  switch (M->law) {
    case ORC_LAW_NONE:
      return 0.0;
    case ORC_LAW_DMT:
    case ORC_LAW_DMT_VISC: {
      double H = theta[0];
      double Es = theta[1];
      double F;
      if (d > M->a0) {
        F = -H * M->R / (6.0 * d * d);
      } else {
        double delta = M->a0 - d;
        F = -H * M->R / (6.0 * M->a0 * M->a0) +
            (4.0 / 3.0) * Es * sqrt(M->R) * delta * sqrt(delta);
        if (M->law == ORC_LAW_DMT_VISC) {
          double eta = theta[2];
          F = F - eta * sqrt(M->R * delta) * v;
        }
      }
      return F;
    }
    case ORC_LAW_LJ_EXP: {
      double C_rep = theta[0];
      double C_att = theta[1];
      double F_ad = theta[2];
      double lambda = theta[3];
      double d2 = d * d;
      double d4 = d2 * d2;
      double d8 = d4 * d4;
      return C_rep / d8 - C_att / d2 - F_ad * exp(-d / lambda);
    }
    case ORC_LAW_HOOKE: {
      double k_s = theta[0];
      double h = theta[1];
      double gap = d - M->z_c + h;
      if (gap < 0.0) return -k_s * gap;
      return 0.0;
    }
    case ORC_LAW_KELVIN_VOIGT: {
      double k_s = theta[0];
      double zeta = theta[1];
      if (d < 0.0) return -k_s * d - zeta * v;
      return 0.0;
    }
    default:
      return NAN;
  }
}

/* ------------------------------------------------------------------------
 * First-order form of the ODE:  z' = v,
 *   v' = [F0 cos(w t) - c v - k z + F_ts(z + z_c, v)] / m.
 * ---------------------------------------------------------------------- */
static void rhs_c(const orc_model* M, const orc_consts* C, const double* theta,
                  double t, double z, double v, double* dz, double* dv) {
  double F_ts = orc_force(M, theta, z + M->z_c, v);
  *dz = v;
  *dv = (C->F0 * cos(C->w * t) - C->c * v - M->k * z + F_ts) / C->m;
}

void orc_rhs(const orc_model* M, const double* theta, double t, double z,
             double v, double* dz, double* dv) {
  orc_consts C;
  orc_constants(M, &C);
  rhs_c(M, &C, theta, t, z, v, dz, dv);
}

/* ------------------------------------------------------------------------
 * "explicit 4th order Runge-Kutta": the classical tableau
 *   c = (0, 1/2, 1/2, 1),  b = (1/6, 1/3, 1/3, 1/6).
 * ---------------------------------------------------------------------- */
static void rk4_step_c(const orc_model* M, const orc_consts* C,
                       const double* theta, double t, double dt, double* z,
                       double* v) {
  double k1z, k1v, k2z, k2v, k3z, k3v, k4z, k4v;
  double z0 = *z, v0 = *v;
  rhs_c(M, C, theta, t, z0, v0, &k1z, &k1v);
  rhs_c(M, C, theta, t + 0.5 * dt, z0 + 0.5 * dt * k1z, v0 + 0.5 * dt * k1v,
        &k2z, &k2v);
  rhs_c(M, C, theta, t + 0.5 * dt, z0 + 0.5 * dt * k2z, v0 + 0.5 * dt * k2v,
        &k3z, &k3v);
  rhs_c(M, C, theta, t + dt, z0 + dt * k3z, v0 + dt * k3v, &k4z, &k4v);
  *z = z0 + dt / 6.0 * (k1z + 2.0 * k2z + 2.0 * k3z + k4z);
  *v = v0 + dt / 6.0 * (k1v + 2.0 * k2v + 2.0 * k3v + k4v);
}

void orc_rk4_step(const orc_model* M, const double* theta, double t, double dt,
                  double* z, double* v) {
  orc_consts C;
  orc_constants(M, &C);
  rk4_step_c(M, &C, theta, t, dt, z, v);
}

/* Divergence rule (reading R12; the paper is silent): a state that
 * is non-finite or has |z| > 100 A0 marks the whole trajectory diverged. */
static int diverged(const orc_model* M, double z, double v) {
  if (!isfinite(z) || !isfinite(v)) return 1;
  if (fabs(z) > 100.0 * M->A0) return 1;
  return 0;
}

/* N fixed steps; t_n = n*dt is never accumulated. */
int orc_integrate(const orc_model* M, const double* theta, double z0,
                  double v0, double* zs, double* vs) {
  orc_consts C;
  double z = z0, v = v0;
  int64_t n;
  orc_constants(M, &C);
  if (zs) zs[0] = z;
  if (vs) vs[0] = v;
  for (n = 0; n < C.N; ++n) {
    double t = (double)n * C.dt;
    rk4_step_c(M, &C, theta, t, C.dt, &z, &v);
    if (diverged(M, z, v)) {
      int64_t j;
      for (j = n + 1; j <= C.N; ++j) {
        if (zs) zs[j] = NAN;
        if (vs) vs[j] = NAN;
      }
      return 1;
    }
    if (zs) zs[n + 1] = z;
    if (vs) vs[n + 1] = v;
  }
  return 0;
}

/* The 'experimental' deflection before noise: the last W
 * post-step positions z_{N-W+1} .. z_N. */
int orc_window(const orc_model* M, const double* theta, double z0, double v0,
               double* window) {
  orc_consts C;
  double* zs;
  int bad;
  int64_t j;
  orc_constants(M, &C);
  zs = (double*)malloc((size_t)(C.N + 1) * sizeof(double));
  bad = orc_integrate(M, theta, z0, v0, zs, NULL);
  for (j = 0; j < C.W; ++j) window[j] = zs[C.N - C.W + 1 + j];
  free(zs);
  return bad;
}

/* ------------------------------------------------------------------------
 * Cost functional, Eq. 5:  J^2_L2 = int [U - u]^2 dt, reduced
 * as the plain sum of squares over the window (no sqrt, no dt; DESIGN.md
 * reading R5):  J = sum_{n=N-W+1}^{N} (z_n - U_{n-(N-W)-1})^2.
 * ---------------------------------------------------------------------- */
double orc_misfit(const orc_model* M, const double* theta, double z0,
                  double v0, const double* trace) {
  orc_consts C;
  double z = z0, v = v0, J = 0.0;
  int64_t n;
  orc_constants(M, &C);
  for (n = 0; n < C.N; ++n) {
    double t = (double)n * C.dt;
    rk4_step_c(M, &C, theta, t, C.dt, &z, &v);
    if (diverged(M, z, v)) return INFINITY;
    if (n + 1 >= C.N - C.W + 1) {
      double res = z - trace[(n + 1) - (C.N - C.W) - 1];
      J = J + res * res;
    }
  }
  return J;
}

void orc_forward_batch(const orc_model* M, const double* params, int64_t P,
                       const double* trace, int32_t n_traces,
                       const double* z0v0, double z0_default,
                       double v0_default, double* misfit) {
  orc_consts C;
  int64_t p, per;
  orc_constants(M, &C);
  per = P / (int64_t)n_traces;
#ifdef ORC_OPENMP /* parity-only build; never the timed baseline */
#pragma omp parallel for schedule(dynamic, 4)
#endif
  for (p = 0; p < P; ++p) {
    const double* theta = params + p * (int64_t)M->n_theta;
    const double* U = trace + (p / per) * C.W;
    double z0 = z0v0 ? z0v0[2 * p] : z0_default;
    double v0 = z0v0 ? z0v0[2 * p + 1] : v0_default;
    misfit[p] = orc_misfit(M, theta, z0, v0, U);
  }
}

/* ------------------------------------------------------------------------
 * Philox4x32-10, Salmon et al., "Parallel random numbers: as easy as 1, 2,
 * 3", SC'11 (the counter-based generator north_star names).
 * ---------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                       uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  int round;
  for (round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += W0;
    k1 += W1;
  }
  out[0] = c0;
  out[1] = c1;
  out[2] = c2;
  out[3] = c3;
}

/* DESIGN.md reading R11: key = (seed lo, seed hi); counter = (gp lo,
 * it, blk + 16*purpose, gp hi) where blk indexes a pair of dimensions; the four
 * output words are (a[2 blk], b[2 blk], a[2 blk + 1], b[2 blk + 1]);
 * u = (word >> 8) * 2^-24, exact in FP32 and FP64. */
void orc_pso_uniforms(uint64_t seed, uint64_t gp, uint32_t it,
                      uint32_t purpose, int32_t D, double* a, double* b) {
  uint32_t key[2];
  int32_t blk;
  key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
  key[1] = (uint32_t)(seed >> 32);
  for (blk = 0; 2 * blk < D; ++blk) {
    uint32_t ctr[4], o[4];
    ctr[0] = (uint32_t)(gp & 0xFFFFFFFFu);
    ctr[1] = it;
    ctr[2] = (uint32_t)blk + 16u * purpose;
    ctr[3] = (uint32_t)(gp >> 32);
    orc_philox4x32_10(ctr, key, o);
    a[2 * blk] = (double)(o[0] >> 8) * (1.0 / 16777216.0);
    b[2 * blk] = (double)(o[1] >> 8) * (1.0 / 16777216.0);
    if (2 * blk + 1 < D) {
      a[2 * blk + 1] = (double)(o[2] >> 8) * (1.0 / 16777216.0);
      b[2 * blk + 1] = (double)(o[3] >> 8) * (1.0 / 16777216.0);
    }
  }
}

void orc_theta_of_x(const orc_box* B, int32_t D, const double* x,
                    double* theta) {
  int32_t j;
  for (j = 0; j < D; ++j) theta[j] = B->log10[j] ? pow(10.0, x[j]) : x[j];
}

/* ------------------------------------------------------------------------
 * Particle swarm optimisation.  "particle locations and
 * velocities are chosen using a uniform distribution in the search space";
 * velocity update Eq. 8:
 *     v_i = w v_{i-1} + c1 r1 (b_l - x_{i-1}) + c2 r2 (b_g - x_{i-1}),
 * b_l the particle's own ("local") best, b_g the global best.  The details
 * Eq. 8 leaves open are DESIGN.md readings R10/R11:
 *   x0 = lo + a (hi - lo);  v0 = ((lo + b (hi - lo)) - x0) / 2;
 *   r1, r2 drawn per particle, per dimension, per iteration;
 *   x_i = x_{i-1} + v_i, then clamp to [lo, hi] zeroing that velocity;
 *   personal best on strict <, global best = lowest index among minima;
 *   synchronous: every particle of iteration i sees the global best found
 *   up to and including batch i;
 *   n_iters forward batches; the result is the global best after the last.
 * Each trace (pixel) owns an independent swarm of n_particles.
 *
 * Cost cutoff (R24; "generations to convergence", 236
 * "convergence cutoff", 264 "cutoff convergence threshold of J_L2"): with
 * j_target > 0 the run ends after the first batch at which every trace's
 * global-best J is <= j_target; that batch is not followed by a move.  The
 * return value is the number of batches run.
 *
 * Asynchronous swarm (R25; the paper is silent): with
 * 0 < async_chunk = B < n_particles the particles of every swarm are taken in
 * chunks [c, c + B) in index order.  A chunk is evaluated, its personal bests
 * and the swarm's best are updated from it, and it moves at once (Eq. 8 with
 * the best known at that moment; same random numbers as the synchronous
 * swarm), so later chunks of the same batch see what earlier chunks found.
 * The chunks of the last batch (n_iters reached) do not move; the cutoff is
 * still tested once per batch, after its last chunk.  B >= n_particles or 0 is
 * the synchronous swarm: the whole swarm is one chunk and moves after the
 * cutoff test.
 * ---------------------------------------------------------------------- */

/* Eq. 8 + position update + bound rule for particles [p0, p1) of every swarm. */
static void pso_move_range(int32_t D, const orc_box* B, const orc_swarm* Sw,
                           uint64_t seed, int32_t it, int32_t n_traces,
                           int64_t p0, int64_t p1, double* x, double* vel,
                           const double* pbest, const double* pbestJ,
                           const double* gbest) {
  const int64_t P = Sw->n_particles;
  int32_t s, j;
  int64_t p;
  for (s = 0; s < n_traces; ++s) {
    for (p = p0; p < p1; ++p) {
      const int64_t gp = (int64_t)s * P + p;
      double r1[4], r2[4];
      const double* social = gbest + s * D;
      orc_pso_uniforms(seed, (uint64_t)gp, (uint32_t)it, 1u, D, r1, r2);
      if (Sw->topology == 1) {
        /* ring of three inside the swarm of trace s */
        int64_t cand[3], best, c;
        cand[0] = (p + P - 1) % P;
        cand[1] = p;
        cand[2] = (p + 1) % P;
        best = cand[0];
        for (c = 1; c < 3; ++c) {
          double Jc = pbestJ[(int64_t)s * P + cand[c]];
          double Jb = pbestJ[(int64_t)s * P + best];
          if (Jc < Jb || (Jc == Jb && cand[c] < best)) best = cand[c];
        }
        social = pbest + ((int64_t)s * P + best) * D;
      }
      for (j = 0; j < D; ++j) {
        double xi = x[gp * D + j];
        double vi = Sw->w * vel[gp * D + j] +
                    Sw->c1 * r1[j] * (pbest[gp * D + j] - xi) +
                    Sw->c2 * r2[j] * (social[j] - xi);
        xi = xi + vi;
        if (xi < B->lo[j]) {
          xi = B->lo[j];
          vi = 0.0;
        }
        if (xi > B->hi[j]) {
          xi = B->hi[j];
          vi = 0.0;
        }
        x[gp * D + j] = xi;
        vel[gp * D + j] = vi;
      }
    }
  }
}

int32_t orc_pso_core(orc_eval_fn eval, const void* ctx, int64_t W, int32_t D,
                     const orc_box* B, const orc_swarm* Sw, uint64_t seed,
                     const double* trace, int32_t n_traces, double* theta_star,
                     double* J_star, double* dump, double* gbest_hist) {
  const int64_t P = Sw->n_particles;
  const int64_t PT = P * (int64_t)n_traces;
  const int64_t rec = 3 * D + 2;
  const int64_t chunk =
      (Sw->async_chunk > 0 && Sw->async_chunk < P) ? Sw->async_chunk : P;
  const int asynchronous = chunk < P;
  double* x = (double*)malloc((size_t)(PT * D) * sizeof(double));
  double* vel = (double*)malloc((size_t)(PT * D) * sizeof(double));
  double* pbest = (double*)malloc((size_t)(PT * D) * sizeof(double));
  double* pbestJ = (double*)malloc((size_t)PT * sizeof(double));
  double* J = (double*)malloc((size_t)PT * sizeof(double));
  double* gbest = (double*)malloc((size_t)(n_traces * D) * sizeof(double));
  double* gbestJ = (double*)malloc((size_t)n_traces * sizeof(double));
  int64_t gp, i, c0;
  int32_t it, j, s, done = 0;

  if (dump)
    for (i = 0; i < (int64_t)Sw->n_iters * PT * rec; ++i) dump[i] = NAN;
  if (gbest_hist)
    for (i = 0; i < (int64_t)Sw->n_iters * n_traces * (D + 1); ++i)
      gbest_hist[i] = NAN;

  /* initialisation: uniform positions and velocities in the search space */
  for (gp = 0; gp < PT; ++gp) {
    double a[4], b[4];
    orc_pso_uniforms(seed, (uint64_t)gp, 0u, 0u, D, a, b);
    for (j = 0; j < D; ++j) {
      double x0 = B->lo[j] + a[j] * (B->hi[j] - B->lo[j]);
      double y0 = B->lo[j] + b[j] * (B->hi[j] - B->lo[j]);
      x[gp * D + j] = x0;
      vel[gp * D + j] = 0.5 * (y0 - x0);
      pbest[gp * D + j] = x0;
    }
    pbestJ[gp] = INFINITY;
  }
  for (s = 0; s < n_traces; ++s) {
    gbestJ[s] = INFINITY;
    for (j = 0; j < D; ++j) gbest[s * D + j] = x[(int64_t)s * P * D + j];
  }

  for (it = 0; it < Sw->n_iters; ++it) {
    const int last = (it == Sw->n_iters - 1);
    int reached;
    for (c0 = 0; c0 < P; c0 += chunk) {
      const int64_t c1 = (c0 + chunk < P) ? c0 + chunk : P;
      const int64_t cn = c1 - c0;
      /* forward batch on the particles of this chunk */
#ifdef ORC_OPENMP /* parity-only build; never the timed baseline */
#pragma omp parallel for schedule(dynamic, 4)
#endif
      for (i = 0; i < cn * n_traces; ++i) {
        const int64_t q = (i / cn) * P + c0 + (i % cn);
        double theta[4];
        orc_theta_of_x(B, D, x + q * D, theta);
        J[q] = eval(ctx, theta, trace + (q / P) * W);
      }
      for (s = 0; s < n_traces; ++s) {
        int64_t p;
        /* personal best (strict <; NaN and +Inf never win) */
        for (p = c0; p < c1; ++p) {
          gp = (int64_t)s * P + p;
          if (J[gp] < pbestJ[gp]) {
            pbestJ[gp] = J[gp];
            for (j = 0; j < D; ++j) pbest[gp * D + j] = x[gp * D + j];
          }
        }
        /* global best per swarm: lowest index among equal minima */
        for (p = c0; p < c1; ++p) {
          gp = (int64_t)s * P + p;
          if (pbestJ[gp] < gbestJ[s]) {
            gbestJ[s] = pbestJ[gp];
            for (j = 0; j < D; ++j) gbest[s * D + j] = pbest[gp * D + j];
          }
        }
        if (dump) {
          for (p = c0; p < c1; ++p) {
            double* r;
            gp = (int64_t)s * P + p;
            r = dump + ((int64_t)it * PT + gp) * rec;
            for (j = 0; j < D; ++j) {
              r[j] = x[gp * D + j];
              r[D + j] = vel[gp * D + j];
              r[2 * D + j] = pbest[gp * D + j];
            }
            r[3 * D] = J[gp];
            r[3 * D + 1] = pbestJ[gp];
          }
        }
      }
      /* asynchronous swarm: the chunk moves before the next one is evaluated */
      if (asynchronous && !last)
        pso_move_range(D, B, Sw, seed, it, n_traces, c0, c1, x, vel, pbest,
                       pbestJ, gbest);
    }
    if (gbest_hist) {
      for (s = 0; s < n_traces; ++s) {
        double* r = gbest_hist + ((int64_t)it * n_traces + s) * (D + 1);
        for (j = 0; j < D; ++j) r[j] = gbest[s * D + j];
        r[D] = gbestJ[s];
      }
    }
    done = it + 1;
    if (last) break;
    /* cost cutoff: every trace's best is at or below the target */
    reached = (Sw->j_target > 0.0);
    for (s = 0; s < n_traces; ++s)
      if (!(gbestJ[s] <= Sw->j_target)) reached = 0;
    if (reached) break;
    /* synchronous swarm: move after the whole batch (Eq. 8, x <- x + v, bounds) */
    if (!asynchronous)
      pso_move_range(D, B, Sw, seed, it, n_traces, 0, P, x, vel, pbest, pbestJ,
                     gbest);
  }

  for (s = 0; s < n_traces; ++s) {
    orc_theta_of_x(B, D, gbest + s * D, theta_star + s * D);
    J_star[s] = gbestJ[s];
  }
  free(x);
  free(vel);
  free(pbest);
  free(pbestJ);
  free(J);
  free(gbest);
  free(gbestJ);
  return done;
}

/* The point-mass forward solve as the PSO's cost function. */
typedef struct {
  const orc_model* M;
  double z0, v0;
} pm_ctx;

static double pm_eval(const void* ctx, const double* theta, const double* U) {
  const pm_ctx* c = (const pm_ctx*)ctx;
  return orc_misfit(c->M, theta, c->z0, c->v0, U);
}

int32_t orc_pso_invert(const orc_model* M, const orc_box* B,
                       const orc_swarm* Sw, uint64_t seed, const double* trace,
                       int32_t n_traces, double z0, double v0,
                       double* theta_star, double* J_star, double* dump,
                       double* gbest_hist) {
  orc_consts C;
  pm_ctx ctx;
  orc_constants(M, &C);
  ctx.M = M;
  ctx.z0 = z0;
  ctx.v0 = v0;
  return orc_pso_core(pm_eval, &ctx, C.W, M->n_theta, B, Sw, seed, trace,
                      n_traces, theta_star, J_star, dump, gbest_hist);
}
