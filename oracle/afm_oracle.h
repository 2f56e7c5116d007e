/*
 * afm_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded FP64 CPU statement of the dAFM force-inversion
 * hot path of arxiv/paper_1109_0334 (Busch, Zou, Ganapathysubramanian):
 * forward problem FP, cost functional Eq. 5,
 * unconstrained optimisation, explicit 4th-order Runge-Kutta
 * (PAPER.md:139), PSO velocity update Eq. 8, on the
 * single-mode (m = 1 case of Eq. 2) point-mass cantilever that
 * BASELINE.json:north_star names.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header,
 * table or constant generator with the CUDA path under
 * paper_1109_0334_b200/csrc/ and include/; the struct layouts below are the
 * oracle's own.
 *
 * Everything is SI and double.  Built with -ffp-contract=off so every
 * operation is a separately rounded IEEE-754 operation in source order.
 *
 * Parity pins (tests/test_oracle_*.py):
 *   RK4 tableau, linear closed forms, step-halving order, force-law hand
 *   values, energy balance, misfit identities, Philox known answers, PSO
 *   invariants and a hand-computed PSO step, scipy DOP853 on the nonlinear
 *   problem; the cost cutoff and the asynchronous swarm on a hand-made cost
 *   callback whose stopping batch and result are written down by hand
 *   (tests/test_oracle_pso_rules.py).
 *   The bound rule (clamp + zero velocity), the velocity-then-position order
 *   and the strict-improvement / lowest-index tie-break are readings (R10) the
 *   paper does not fix; what this file does with them is pinned: the inertia-only
 *   swarm (c1 = c2 = 0) against its closed form, a geometric series with an
 *   absorbing bound, and exact ties on a scripted cost with the winners written
 *   down by hand (tests/test_oracle_pso_rules.py).
 * PARITY UNPINNED (design choices with nothing outside this file to check
 * against): the initial-velocity rule
 * v0 = (U(lo,hi) - x0)/2 beyond its range, the Philox counter layout, the
 * divergence rule (R12), the ring of three (R23) and the chunked reading of
 * "asynchronous" (R25); the last two have hand-written expectations on scripted
 * costs only.
 */
#ifndef AFM_ORACLE_H
#define AFM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Tip-sample force laws (BASELINE.json configs[0], [2], [3]; the paper names
 * them only as extensions). */
enum {
  ORC_LAW_NONE = 0,    /* F_ts = 0 (linear oscillator; used by the pins)      */
  ORC_LAW_DMT = 1,     /* theta = (H, E*)                                     */
  ORC_LAW_DMT_VISC = 2,/* theta = (H, E*, eta)                                */
  ORC_LAW_LJ_EXP = 3,  /* theta = (C_rep, C_att, F_ad, lambda)                */
  ORC_LAW_HOOKE = 4,   /* theta = (k_s, h): paper Eq. 11                      */
  ORC_LAW_KELVIN_VOIGT = 5 /* theta = (k_s, zeta_s): paper Eq. 12              */
};

/* Cantilever, drive and time grid.  All SI. */
typedef struct {
  double k;        /* spring constant, N/m                                   */
  double f0;       /* natural frequency, Hz                                  */
  double Q;        /* quality factor                                         */
  double f_drive;  /* drive frequency, Hz                                    */
  double A0;       /* free steady-state amplitude, m (defines F0)            */
  double z_c;      /* rest height of the tip above the sample, m             */
  double R;        /* tip radius, m (DMT laws)                               */
  double a0;       /* intermolecular distance, m (DMT laws)                  */
  int32_t law;     /* ORC_LAW_*                                              */
  int32_t n_theta; /* number of force parameters D                           */
  int32_t S;       /* RK4 steps per drive cycle                              */
  int32_t n_cycles;/* total drive cycles integrated                          */
  int32_t n_skip;  /* cycles skipped before the misfit window                */
  int32_t pad_;
} orc_model;

/* Derived constants (returned for the pins to inspect). */
typedef struct {
  double w0, w, m, c, r, F0, dt;
  int64_t N;  /* total steps  S * n_cycles            */
  int64_t W;  /* window steps S * (n_cycles - n_skip) */
} orc_consts;

/* PSO search box in PSO coordinates x; theta_j = 10^x_j where log10[j] != 0,
 * else theta_j = x_j. */
typedef struct {
  double lo[4];
  double hi[4];
  int32_t log10[4];
} orc_box;

typedef struct {
  int32_t n_particles; /* per trace                                          */
  int32_t n_iters;     /* number of forward batches (iteration 0 = x0)       */
  double w, c1, c2;    /* Eq. 8 weights                                      */
  double j_target;     /* cost cutoff ("convergence cutoff",
                          264 "cutoff convergence threshold of J_L2 = 0.0005";
                          DESIGN.md R24): > 0: the run ends after the first
                          batch at which EVERY trace's global-best J is
                          <= j_target, and no move follows that batch;
                          <= 0: off, all n_iters batches are run            */
  int32_t topology;    /* 0: global best (the paper's "g_b");
                          1: ring of three (R23): the social attractor
                          of particle p is the best personal best among
                          p-1, p, p+1 (indices wrap inside the swarm; lowest
                          index among equal minima)                          */
  int32_t async_chunk; /* 0 (or >= n_particles): synchronous swarm, the paper's
                          generation-by-generation PSO.  B in 1..n_particles-1:
                          asynchronous swarm (R25):
                          every swarm is processed in chunks of B particles in
                          index order; a chunk is evaluated, its personal bests
                          and the swarm's best are updated, and the chunk moves
                          at once with the best known at that moment, so later
                          chunks of the same batch already see it           */
} orc_swarm;

void   orc_constants(const orc_model* M, orc_consts* C);

/* F_ts(d, ddot; theta) in newtons; d = z + z_c is the tip-sample gap. */
double orc_force(const orc_model* M, const double* theta, double d, double v);

/* Right-hand side of the first-order system (z' = v, v' = a). */
void   orc_rhs(const orc_model* M, const double* theta, double t, double z,
               double v, double* dz, double* dv);

/* One classical RK4 step of size dt from (t, z, v). */
void   orc_rk4_step(const orc_model* M, const double* theta, double t,
                    double dt, double* z, double* v);

/* Integrate N steps from (z0, v0).  If zs/vs are non-NULL they receive the
 * N+1 states (index 0 = initial state, index n = state after step n).
 * Returns 0, or 1 if the trajectory diverged (non-finite, or |z| > 100 A0);
 * on divergence the remaining outputs are filled with NaN. */
int    orc_integrate(const orc_model* M, const double* theta, double z0,
                     double v0, double* zs, double* vs);

/* Clean (noise-free) window of a trajectory: the last W post-step positions. */
int    orc_window(const orc_model* M, const double* theta, double z0,
                  double v0, double* window /* [W] */);

/* Misfit J = sum_{n=N-W+1..N} (z_n - U_{n-(N-W)-1})^2 (Eq. 5 as a plain sum
 * of squares, metres^2).  +Inf if the trajectory diverged. */
double orc_misfit(const orc_model* M, const double* theta, double z0,
                  double v0, const double* trace /* [W] */);

/* Batch of forward problems.  params [P][D]; z0v0 [P][2] or NULL (then
 * z0_default, v0_default); n_traces >= 1 splits the P particles into
 * n_traces equal contiguous segments, segment s using trace[s][W]. */
void   orc_forward_batch(const orc_model* M, const double* params, int64_t P,
                         const double* trace, int32_t n_traces,
                         const double* z0v0, double z0_default,
                         double v0_default, double* misfit /* [P] */);

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11). */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                         uint32_t out[4]);

/* Uniforms used by the PSO: for global particle index gp, iteration it and
 * purpose (0 = initialisation, 1 = velocity update), fills a[d], b[d] for
 * d < D with u = (word >> 8) * 2^-24 in [0, 1). */
void   orc_pso_uniforms(uint64_t seed, uint64_t gp, uint32_t it,
                        uint32_t purpose, int32_t D, double* a, double* b);

/* Map PSO coordinates to physical parameters. */
void   orc_theta_of_x(const orc_box* B, int32_t D, const double* x,
                      double* theta);

/* PSO around the forward batch (synchronous global best unless Sw says
 * otherwise).
 * dump (or NULL): [n_iters][n_traces*P][3D+2] = x, v, pbest, J, pbestJ,
 * recorded after the personal-best update of each iteration and before the
 * move.  gbest_hist (or NULL): [n_iters][n_traces][D+1] = gbest x, gbestJ.
 * Rows of batches that the cost cutoff left unrun are NaN.
 * Outputs theta_star [n_traces][D], J_star [n_traces].
 * Returns the number of forward batches run (n_iters unless j_target cut the
 * run short): the paper's "generations to convergence". */
int32_t orc_pso_invert(const orc_model* M, const orc_box* B,
                      const orc_swarm* Sw, uint64_t seed, const double* trace,
                      int32_t n_traces, double z0, double v0,
                      double* theta_star, double* J_star, double* dump,
                      double* gbest_hist);

/* The PSO loop itself, around any cost function eval(ctx, theta, U_s) (the
 * point-mass misfit above, or the beam misfit of afm_oracle_beam.h). */
typedef double (*orc_eval_fn)(const void* ctx, const double* theta,
                              const double* trace_s);
int32_t orc_pso_core(orc_eval_fn eval, const void* ctx, int64_t W, int32_t D,
                    const orc_box* B, const orc_swarm* Sw, uint64_t seed,
                    const double* trace, int32_t n_traces, double* theta_star,
                    double* J_star, double* dump, double* gbest_hist);

#ifdef __cplusplus
}
#endif
#endif
