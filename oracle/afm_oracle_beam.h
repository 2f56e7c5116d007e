/* afm_oracle_beam.h -- CPU oracle for the paper's OWN forward model, the
 * multi-mode Euler-Bernoulli cantilever (PAPER.md:59-66
 * Eq. 1-2, Eq. 6-7, Appendix A/B).  TEST INFRASTRUCTURE, like
 * afm_oracle.h: only tests/, __graft_entry__.smoke() and bench.py's CPU legs
 * may use it; it shares no code with the CUDA path.
 *
 * Model (all SI, FP64, single-threaded, formulas in the paper's order):
 *   u(x,t) = sum_i Phi_i(x) eta_i(t)                               (B.1)
 *   eta_i'' + (w_i/Q) eta_i' + w_i^2 eta_i
 *       = [ f_tip(t) Phi_i(L) - mu y_ex''(t) <1, Phi_i> ] / (mu <Phi_i, Phi_i>)
 *   i.e. Eq. 2 with 2 zeta = 1/Q (R2), the tip-sample force a point
 *   load at x = L, and the base motion y_ex(t) = A_base cos(w t);
 *   f_tip = F_ts(u(L,t) + z_c, u'(L,t); theta) with the force laws of
 *   afm_oracle.h (gap measured from the RELATIVE deflection u, as Eq. 3/11 do);
 *   beta_i: roots of cos(bL) cosh(bL) + 1 = 0 by Newton, w_i = (b_i L)^2
 *   sqrt(E I / (mu L^4)); Phi_i by Eq. 6-7; <.,.> by Simpson's rule on
 *   n_points points (Appendix A "501");
 *   classical RK4 on the 2m-vector (eta, eta'), from rest.
 *   Misfit: sum over the window of (u(L,t_n) - U_n)^2.
 *   Divergence: a non-finite state or |u(L)| > 100 A_ref gives +Inf (R12).
 */
#ifndef AFM_ORACLE_BEAM_H
#define AFM_ORACLE_BEAM_H

#include <stdint.h>

#include "afm_oracle.h"

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_MODES 8

typedef struct {
  double L, E, I, mu;   /* length m, Young's modulus Pa, area moment m^4, kg/m */
  double Q;             /* modal quality factor (2 zeta = 1/Q)                */
  double f_drive;       /* Hz                                                 */
  double A_base;        /* base displacement amplitude, m                     */
  double A_ref;         /* reference tip amplitude for the divergence rule, m */
  double z_c, R, a0;    /* as in orc_model                                    */
  int32_t law, n_theta; /* ORC_LAW_*, D                                       */
  int32_t n_modes;      /* 1..8                                               */
  int32_t n_points;     /* Simpson points (odd), 501 in the paper             */
  int32_t S, n_cycles, n_skip;
  int32_t literal_eq7;  /* 1: Eq. 7 as printed (for the pin that rejects it)  */
} orc_beam;

typedef struct {
  double bL[ORC_MAX_MODES];     /* beta_i L                                   */
  double omega[ORC_MAX_MODES];  /* rad/s                                      */
  double phiL[ORC_MAX_MODES];   /* Phi_i(L)                                   */
  double norm[ORC_MAX_MODES];   /* <Phi_i, Phi_i>                             */
  double intphi[ORC_MAX_MODES]; /* <1, Phi_i>                                 */
  double gain[ORC_MAX_MODES];   /* A_base w^2 <1,Phi_i>/<Phi_i,Phi_i>         */
  double fgain[ORC_MAX_MODES];  /* Phi_i(L) / (mu <Phi_i,Phi_i>)              */
  double w, dt;
  int64_t N, W;
} orc_beam_modes;

void   orc_beam_setup(const orc_beam* B, orc_beam_modes* Mo);
/* Phi_i(x), i = 0..n_modes-1 (Eq. 6-7). */
double orc_beam_shape(const orc_beam* B, const orc_beam_modes* Mo, int32_t i,
                      double x);
/* N steps from rest (or from eta0 [2m] = eta_0.., eta'_0.. if non-NULL).
 * tip_u, tip_v [N+1] and eta [N+1][2m] may be NULL.  Returns 1 if diverged. */
int    orc_beam_integrate(const orc_beam* B, const double* theta,
                          const double* eta0, double* tip_u, double* tip_v,
                          double* eta);
int    orc_beam_window(const orc_beam* B, const double* theta, double* window);
double orc_beam_misfit(const orc_beam* B, const double* theta,
                       const double* trace);
void   orc_beam_forward_batch(const orc_beam* B, const double* params,
                              int64_t P, const double* trace, int32_t n_traces,
                              double* misfit);
/* The PSO of afm_oracle.h around the beam forward batch (same streams, same
 * cutoff and chunk rules); returns the number of batches run. */
int32_t orc_beam_pso_invert(const orc_beam* B, const orc_box* Bx,
                            const orc_swarm* Sw, uint64_t seed,
                            const double* trace, int32_t n_traces,
                            double* theta_star, double* J_star, double* dump,
                            double* gbest_hist);

#ifdef __cplusplus
}
#endif
#endif
