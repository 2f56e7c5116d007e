/* afm_oracle_beam.c -- see afm_oracle_beam.h.  Plain C99, FP64, built with
 * -ffp-contract=off; every formula in the order the paper states it. */
#include "afm_oracle_beam.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* Roots of cos(x) cosh(x) + 1 = 0 by Newton's method
 * (PAPER.md:130), on the equivalent g(x) = cos(x) + 1/cosh(x), which cannot
 * overflow; start at (i + 1/2) pi, i = 0, 1, ... */
static double beam_root(int32_t i) {
  double x = ((double)i + 0.5) * M_PI;
  int it;
  for (it = 0; it < 50; ++it) {
    double ch = cosh(x);
    double g = cos(x) + 1.0 / ch;
    double dg = -sin(x) - sinh(x) / (ch * ch);
    double step = g / dg;
    x = x - step;
    if (fabs(step) < 1e-15 * x) break;
  }
  return x;
}

/* G of Eq. 7.  As printed, numerator and denominator both carry
 * "- exp(-2 beta L) + 1"; expanding G = (sinh + sin)/(cosh + cos) times
 * 2 exp(-beta L) gives "+ exp(-2 beta L)" in the denominator (R22);
 * the printed form is kept behind literal_eq7 for the pin that rejects it. */
static double beam_G(const orc_beam* B, double bL) {
  double e1 = exp(-bL);
  double e2 = exp(-2.0 * bL);
  double num = 2.0 * e1 * sin(bL) - e2 + 1.0;
  double den = B->literal_eq7 ? (2.0 * e1 * cos(bL) - e2 + 1.0)
                              : (2.0 * e1 * cos(bL) + e2 + 1.0);
  return num / den;
}

/* Eq. 6: the overflow-free exponential form of the clamped-free
 * mode shape. */
static double beam_phi(const orc_beam* B, double bL, double x) {
  double b = bL / B->L;
  double G = beam_G(B, bL);
  return (2.0 * sin(b * x) - 2.0 * G * cos(b * x) + (G - 1.0) * exp(b * x) +
          (G + 1.0) * exp(-b * x)) /
         2.0;
}

/* Composite Simpson rule on n (odd) points over [0, L] of Phi^p, p = 1 or 2. */
static double beam_simpson(const orc_beam* B, double bL, int p) {
  int32_t n = B->n_points, j;
  double h = B->L / (double)(n - 1);
  double sum = 0.0;
  for (j = 0; j < n; ++j) {
    double f = beam_phi(B, bL, (double)j * h);
    double wgt = (j == 0 || j == n - 1) ? 1.0 : ((j % 2) ? 4.0 : 2.0);
    if (p == 2) f = f * f;
    sum = sum + wgt * f;
  }
  return sum * h / 3.0;
}

void orc_beam_setup(const orc_beam* B, orc_beam_modes* Mo) {
  int32_t i;
  double w = 2.0 * M_PI * B->f_drive;
  memset(Mo, 0, sizeof(*Mo));
  Mo->w = w;
  Mo->dt = 2.0 * M_PI / (w * (double)B->S);
  Mo->N = (int64_t)B->S * B->n_cycles;
  Mo->W = (int64_t)B->S * (B->n_cycles - B->n_skip);
  for (i = 0; i < B->n_modes; ++i) {
    double bL = beam_root(i);
    Mo->bL[i] = bL;
    Mo->omega[i] = bL * bL * sqrt(B->E * B->I / (B->mu * B->L * B->L * B->L * B->L));
    Mo->phiL[i] = beam_phi(B, bL, B->L);
    Mo->norm[i] = beam_simpson(B, bL, 2);
    Mo->intphi[i] = beam_simpson(B, bL, 1);
    Mo->gain[i] = B->A_base * w * w * Mo->intphi[i] / Mo->norm[i];
    Mo->fgain[i] = Mo->phiL[i] / (B->mu * Mo->norm[i]);
  }
}

double orc_beam_shape(const orc_beam* B, const orc_beam_modes* Mo, int32_t i,
                      double x) {
  return beam_phi(B, Mo->bL[i], x);
}

/* Right-hand side of the 2m first-order system y = (eta_0.., eta'_0..). */
static void beam_rhs(const orc_beam* B, const orc_beam_modes* Mo,
                     const double* theta, double t, const double* y,
                     double* dy) {
  int32_t m = B->n_modes, i;
  double u = 0.0, v = 0.0, F;
  orc_model fm;
  for (i = 0; i < m; ++i) {
    u = u + Mo->phiL[i] * y[i];
    v = v + Mo->phiL[i] * y[m + i];
  }
  memset(&fm, 0, sizeof(fm));
  fm.z_c = B->z_c;
  fm.R = B->R;
  fm.a0 = B->a0;
  fm.law = B->law;
  fm.n_theta = B->n_theta;
  F = orc_force(&fm, theta, u + B->z_c, v);
  for (i = 0; i < m; ++i) {
    dy[i] = y[m + i];
    dy[m + i] = Mo->gain[i] * cos(Mo->w * t) - Mo->omega[i] / B->Q * y[m + i] -
                Mo->omega[i] * Mo->omega[i] * y[i] + Mo->fgain[i] * F;
  }
}

/* One classical RK4 step (tableau c = (0, 1/2, 1/2, 1), b = (1/6, 1/3, 1/3, 1/6)). */
static void beam_rk4(const orc_beam* B, const orc_beam_modes* Mo,
                     const double* theta, double t, double dt, double* y) {
  double k1[2 * ORC_MAX_MODES], k2[2 * ORC_MAX_MODES], k3[2 * ORC_MAX_MODES];
  double k4[2 * ORC_MAX_MODES], s[2 * ORC_MAX_MODES] = {0.0};
  int32_t n = 2 * B->n_modes, j;
  beam_rhs(B, Mo, theta, t, y, k1);
  for (j = 0; j < n; ++j) s[j] = y[j] + 0.5 * dt * k1[j];
  beam_rhs(B, Mo, theta, t + 0.5 * dt, s, k2);
  for (j = 0; j < n; ++j) s[j] = y[j] + 0.5 * dt * k2[j];
  beam_rhs(B, Mo, theta, t + 0.5 * dt, s, k3);
  for (j = 0; j < n; ++j) s[j] = y[j] + dt * k3[j];
  beam_rhs(B, Mo, theta, t + dt, s, k4);
  for (j = 0; j < n; ++j)
    y[j] = y[j] + dt / 6.0 * (k1[j] + 2.0 * k2[j] + 2.0 * k3[j] + k4[j]);
}

static void beam_tip(const orc_beam* B, const orc_beam_modes* Mo, const double* y,
                     double* u, double* v) {
  int32_t m = B->n_modes, i;
  double uu = 0.0, vv = 0.0;
  for (i = 0; i < m; ++i) {
    uu = uu + Mo->phiL[i] * y[i];
    vv = vv + Mo->phiL[i] * y[m + i];
  }
  *u = uu;
  *v = vv;
}

static int beam_diverged(const orc_beam* B, const double* y, double u) {
  int32_t j;
  for (j = 0; j < 2 * B->n_modes; ++j)
    if (!isfinite(y[j])) return 1;
  if (!isfinite(u) || fabs(u) > 100.0 * B->A_ref) return 1;
  return 0;
}

int orc_beam_integrate(const orc_beam* B, const double* theta, const double* eta0,
                       double* tip_u, double* tip_v, double* eta) {
  orc_beam_modes Mo;
  double y[2 * ORC_MAX_MODES];
  int32_t n2 = 2 * B->n_modes, j;
  int64_t n;
  double u, v;
  orc_beam_setup(B, &Mo);
  for (j = 0; j < n2; ++j) y[j] = eta0 ? eta0[j] : 0.0;
  beam_tip(B, &Mo, y, &u, &v);
  if (tip_u) tip_u[0] = u;
  if (tip_v) tip_v[0] = v;
  if (eta) memcpy(eta, y, (size_t)n2 * sizeof(double));
  for (n = 0; n < Mo.N; ++n) {
    beam_rk4(B, &Mo, theta, (double)n * Mo.dt, Mo.dt, y);
    beam_tip(B, &Mo, y, &u, &v);
    if (beam_diverged(B, y, u)) {
      int64_t q;
      for (q = n + 1; q <= Mo.N; ++q) {
        if (tip_u) tip_u[q] = NAN;
        if (tip_v) tip_v[q] = NAN;
      }
      return 1;
    }
    if (tip_u) tip_u[n + 1] = u;
    if (tip_v) tip_v[n + 1] = v;
    if (eta) memcpy(eta + (n + 1) * n2, y, (size_t)n2 * sizeof(double));
  }
  return 0;
}

int orc_beam_window(const orc_beam* B, const double* theta, double* window) {
  orc_beam_modes Mo;
  double* us;
  int bad;
  int64_t j;
  orc_beam_setup(B, &Mo);
  us = (double*)malloc((size_t)(Mo.N + 1) * sizeof(double));
  bad = orc_beam_integrate(B, theta, NULL, us, NULL, NULL);
  for (j = 0; j < Mo.W; ++j) window[j] = us[Mo.N - Mo.W + 1 + j];
  free(us);
  return bad;
}

/* Eq. 5 as a plain sum of squares over the window, on the tip deflection. */
double orc_beam_misfit(const orc_beam* B, const double* theta,
                       const double* trace) {
  orc_beam_modes Mo;
  double y[2 * ORC_MAX_MODES];
  double J = 0.0, u, v;
  int32_t j;
  int64_t n;
  orc_beam_setup(B, &Mo);
  for (j = 0; j < 2 * B->n_modes; ++j) y[j] = 0.0;
  for (n = 0; n < Mo.N; ++n) {
    beam_rk4(B, &Mo, theta, (double)n * Mo.dt, Mo.dt, y);
    beam_tip(B, &Mo, y, &u, &v);
    if (beam_diverged(B, y, u)) return INFINITY;
    if (n + 1 >= Mo.N - Mo.W + 1) {
      double res = u - trace[(n + 1) - (Mo.N - Mo.W) - 1];
      J = J + res * res;
    }
  }
  return J;
}

void orc_beam_forward_batch(const orc_beam* B, const double* params, int64_t P,
                            const double* trace, int32_t n_traces,
                            double* misfit) {
  orc_beam_modes Mo;
  int64_t p, per = P / (int64_t)n_traces;
  orc_beam_setup(B, &Mo);
#ifdef ORC_OPENMP /* parity-only build; never the timed baseline */
#pragma omp parallel for schedule(dynamic, 2)
#endif
  for (p = 0; p < P; ++p)
    misfit[p] = orc_beam_misfit(B, params + p * (int64_t)B->n_theta,
                                trace + (p / per) * Mo.W);
}

static double beam_eval(const void* ctx, const double* theta, const double* U) {
  return orc_beam_misfit((const orc_beam*)ctx, theta, U);
}

int32_t orc_beam_pso_invert(const orc_beam* B, const orc_box* Bx,
                            const orc_swarm* Sw, uint64_t seed,
                            const double* trace, int32_t n_traces,
                            double* theta_star, double* J_star, double* dump,
                            double* gbest_hist) {
  orc_beam_modes Mo;
  orc_beam_setup(B, &Mo);
  return orc_pso_core(beam_eval, B, Mo.W, B->n_theta, Bx, Sw, seed, trace,
                      n_traces, theta_star, J_star, dump, gbest_hist);
}
