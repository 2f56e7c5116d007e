/*
 * afm.h -- C ABI of the B200-native dAFM force-inversion hot path
 * (arxiv/paper_1109_0334, Busch, Zou, Ganapathysubramanian).
 *
 * The library computes, entirely in hand-written sm_100a CUDA kernels:
 *   - the batched forward problem FP: for every candidate
 *     force-parameter vector theta, integrate
 *         m z'' + (m w0/Q) z' + k z = F0 cos(w t) + F_ts(z + z_c, z'; theta)
 *     (the m = 1 case of the modal equation, Eq. 2, as the
 *     point mass BASELINE.json:north_star names) with the explicit classical
 *     4th-order Runge-Kutta scheme at a fixed step of 1/S of a
 *     drive period;
 *   - the cost functional of Eq. 5 as the plain sum of squares
 *         J = sum_{n=N-W+1..N} (z_n - U_{n-(N-W)-1})^2        [m^2]
 *     over the last W post-step states (readings R5, R7);
 *   - the particle-swarm optimisation of PAPER.md:209-214 (velocity update
 *     Eq. 8, personal best, global best) that solves the inverse problem IP
 *      as an unconstrained minimisation of J over theta.
 *
 * Conventions
 *   - Every entry point returns AFM_OK (0) or a negative afm_status; the text
 *     of the last error on the calling thread is afm_last_error().  Nothing
 *     throws, nothing is allocated on behalf of the caller, every buffer is
 *     caller-owned.  The library keeps one lazily created device workspace
 *     per process (time-tile stream, swarm state); afm_shutdown() frees it.
 *   - There is NO CPU fallback: without a CUDA device of compute capability
 *     10.x the compute calls return AFM_EUNSUPPORTED / AFM_ECUDA.
 *   - "device" pointers are CUDA device pointers valid on the current device;
 *     "host" pointers are ordinary host memory.  All arrays are dense,
 *     row-major, FP64, SI units at the ABI, whatever cfg->precision says: the
 *     FP32 kernel converts internally.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default
 *     stream).  PyTorch is only ever the allocator and the stream provider.
 */
#ifndef AFM_H
#define AFM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  AFM_OK = 0,
  AFM_EINVAL = -1,       /* NULL pointer, bad size, law/D mismatch, ...        */
  AFM_ECUDA = -2,        /* a CUDA runtime call failed; see afm_last_error()   */
  AFM_EUNSUPPORTED = -3  /* no sm_100-class device, or an unsupported option   */
} afm_status;

/* Tip-sample force laws F_ts(d, d'; theta), d = z + z_c the tip-sample gap
 * (BASELINE.json configs[0], [2], [3]; "Hertzian contact and Van der Waals
 * forces").
 *   AFM_LAW_NONE      F_ts = 0                                   D = 0..4
 *   AFM_LAW_DMT       theta = (H, E*)                            D = 2
 *       d >  a0:  -H R / (6 d^2)
 *       d <= a0:  -H R / (6 a0^2) + (4/3) E* sqrt(R) (a0 - d)^{3/2}
 *   AFM_LAW_DMT_VISC  theta = (H, E*, eta)                       D = 3
 *       DMT, plus  -eta sqrt(R (a0 - d)) d'  for d <= a0
 *   AFM_LAW_LJ_EXP    theta = (C_rep, C_att, F_ad, lambda)       D = 4
 *       C_rep / d^8 - C_att / d^2 - F_ad exp(-d / lambda)
 * The paper's own sample models, active while the tip is pressed in:
 *   AFM_LAW_HOOKE     theta = (k_s, h)   Eq. 11, PAPER.md:260    D = 2
 *       gap = z + h (h, the cantilever-sample separation, is an unknown and
 *       takes the place of z_c):  -k_s gap  for gap < 0, else 0
 *   AFM_LAW_KELVIN_VOIGT  theta = (k_s, zeta_s)  Eq. 12, PAPER.md:270   D = 2
 *       separation known (z_c):  -k_s d - zeta_s d'  for d < 0, else 0
 */
typedef enum {
  AFM_LAW_NONE = 0,
  AFM_LAW_DMT = 1,
  AFM_LAW_DMT_VISC = 2,
  AFM_LAW_LJ_EXP = 3,
  AFM_LAW_HOOKE = 4,
  AFM_LAW_KELVIN_VOIGT = 5
} afm_law;

typedef enum { AFM_F64 = 0, AFM_F32 = 1 } afm_precision;

/* Cantilever, drive, time grid.  Host, read-only, plain POD.
 * F0 is fixed by A0: F0 = k A0 sqrt((1-r^2)^2 + (r/Q)^2), r = f_drive/f0, so
 * that the free (F_ts = 0) steady-state amplitude is exactly A0.
 * dt = 1 / (f_drive * steps_per_cycle); t_n = n dt; N = steps_per_cycle *
 * n_cycles steps are taken; the misfit window is the last
 * W = steps_per_cycle * (n_cycles - n_skip_cycles) post-step states.
 * A trajectory whose state becomes non-finite or leaves |z| <= 100 A0 at any
 * step is "diverged" and its misfit is +Inf (reading R12). */
typedef struct {
  double k;        /* spring constant, N/m                                  */
  double f0;       /* natural frequency, Hz                                 */
  double Q;        /* quality factor                                        */
  double f_drive;  /* drive frequency, Hz                                   */
  double A0;       /* free steady-state amplitude, m                        */
  double z_c;      /* rest height of the tip above the sample, m            */
  double R;        /* tip radius, m (DMT laws)                              */
  double a0;       /* intermolecular distance, m (DMT laws)                 */
  double z0, v0;   /* initial state used when z0v0 == NULL (m, m/s)         */
  int32_t law;             /* afm_law                                       */
  int32_t n_params;        /* D, must match the law (NONE: any 0..4)        */
  int32_t steps_per_cycle; /* S >= 1                                        */
  int32_t n_cycles;        /* >= 1                                          */
  int32_t n_skip_cycles;   /* 0 <= n_skip_cycles < n_cycles                 */
  int32_t n_traces;        /* >= 1: the particles are n_traces equal,
                              contiguous segments; segment s is compared
                              with trace[s][0..W)                           */
  int32_t precision;       /* afm_precision of the integrate kernel         */
  int32_t reserved_;       /* must be 0                                     */
} afm_cfg;

/* Search box in PSO coordinates x; theta_j = 10^x_j where log10_scale[j] != 0,
 * else theta_j = x_j.  Entries j >= D are ignored. */
typedef struct {
  double lo[4];
  double hi[4];
  int32_t log10_scale[4];
} afm_bounds;

/* Swarm: n_particles PER TRACE; n_iters forward batches (iteration 0
 * evaluates the initial positions; the result is the global best after the
 * last batch).  w, c1, c2 are the weights of Eq. 8.
 * j_target > 0 enables the paper's cutoff rule (
 * DESIGN.md R24): the run ends after the first batch at which every trace's
 * global best J is <= j_target, that batch is not followed by a move, and
 * n_iters_done reports the batches run; <= 0 disables it. */
typedef struct {
  int32_t n_particles;
  int32_t n_iters;
  double w, c1, c2;
  double j_target;
  int32_t topology;   /* 0: global best (the paper's g_b);
                         1: ring of three (R23): the social attractor
                         of particle p is the best personal best among p-1, p,
                         p+1, wrapping inside the swarm, lowest index among
                         equal minima.  theta*, J* are the swarm's best either
                         way. */
  int32_t async_chunk; /* 0 (or >= n_particles): the synchronous, generation by
                         generation swarm of the paper.  B in 1..n_particles-1:
                         asynchronous swarm (R25): every swarm is
                         processed in chunks of B particles in index order; a
                         chunk is evaluated, the bests are updated from it and
                         it moves at once with the best known at that moment
                         (same random streams).  afm_pso_invert[_host] only. */
} afm_swarm_cfg;

/* ---- forward problem + cost (Eq. 5) -------------
 * misfit[p] = J(theta_p) for p in [0, n_particles).
 *   params   device  [n_particles][D]   physical SI parameters
 *   trace    device  [n_traces][W]      measured deflection U, metres
 *   z0v0     device  [n_particles][2]   per-particle (z0, v0), or NULL ->
 *                                       (cfg->z0, cfg->v0) for all
 *   misfit   device  [n_particles]      out, m^2; +Inf if diverged
 * n_particles must be a positive multiple of cfg->n_traces.
 * Asynchronous on cuda_stream: returns after enqueueing. */
int afm_forward_batch(const double* params, int64_t n_particles,
                      const double* trace, const afm_cfg* cfg,
                      const double* z0v0, double* misfit, void* cuda_stream);

/* Same computation with HOST buffers: copies params/trace/z0v0 to the device,
 * runs the batch, copies misfit back and synchronises the stream before
 * returning (the end-to-end path bench.py times).  All pointers host. */
int afm_forward_batch_host(const double* params, int64_t n_particles,
                           const double* trace, const afm_cfg* cfg,
                           const double* z0v0, double* misfit,
                           void* cuda_stream);

/* ---- forward problem + cost for callers that must not allocate ------------
 * Same computation and same arguments as afm_forward_batch (device pointers,
 * asynchronous on cuda_stream), for callers that cannot let this library call
 * cudaMalloc / cudaFree on their behalf.  The ordinary calls keep a device
 * workspace that is created on first use and re-created (free + malloc)
 * whenever a larger batch arrives.  Two kinds of caller cannot live with that:
 *   - the acquisition loop of a running microscope, the paper's "near
 *     real-time" setting: cudaMalloc and cudaFree take
 *     driver-wide locks, may wait for all work on the device and have no upper
 *     bound on their duration, so one of them in the middle of a scan line
 *     breaks the loop's timing;
 *   - a process whose device memory is already owned by someone else's pool
 *     (a framework's caching allocator, a vendor acquisition stack): an
 *     allocation made behind the pool's back can fail although the pool has
 *     room, or take memory the pool counts on.
 * This entry point calls no cudaMalloc, cudaFree, event/stream creation or
 * allocating library routine.  Its only scratch, the time-tile stream (one
 * 32-byte row per trace and RK4 step: the drive at the three RK4 abscissae and
 * the shifted trace sample), lives in an array of AFM_NOALLOC_MAX_ROWS rows
 * (4 MiB) that is compiled into the library's device image: every GPU on which
 * this library's kernels are loaded holds those 4 MiB until the process exits,
 * whether or not this call is ever used.
 *   Limit: cfg->n_traces * cfg->steps_per_cycle * cfg->n_cycles must not
 *     exceed AFM_NOALLOC_MAX_ROWS, else AFM_EINVAL with the numbers in
 *     afm_last_error() (configs[0]..[3] of BASELINE.json fit with one trace;
 *     configs[4]'s 256 traces do not: use afm_forward_batch there).
 *   First call on a device: looks up the device address of the built-in array
 *     (a runtime query that also loads the library's kernels onto that device)
 *     and remembers it for the life of the process.  Make that first call once
 *     per device at start-up, with that device current and outside any stream
 *     capture; later calls only enqueue two kernels.
 *   Sharing: there is ONE array per device, used by every call and never
 *     cleared; it holds what the previous call left there.  That is harmless
 *     in sequence, because each call writes every row it is going to read
 *     before it reads it, but two calls that overlap on the GPU (different
 *     streams, or different host threads, without an ordering between them)
 *     overwrite each other's rows and both return garbage.  Keep all calls on
 *     one stream, or order them with events of your own.
 *   Scheduling: runs the plain one-launch integrate kernel.  The warp packing
 *     and the segment queue of afm_forward_batch need scratch that grows with
 *     the batch and are not used here, so large batches run at the speed of
 *     afm_set_option("queue", 1) + ("pack", 1); the misfits are the same. */
#define AFM_NOALLOC_MAX_ROWS 131072
int afm_forward_batch_noalloc(const double* params, int64_t n_particles,
                              const double* trace, const afm_cfg* cfg,
                              const double* z0v0, double* misfit,
                              void* cuda_stream);

/* ---- inverse problem by PSO (Eq. 8) -------------
 * One independent swarm per trace.  Philox4x32-10 random numbers, key =
 * seed, counter = (particle, iteration, purpose) (reading R11), so
 * a run is a pure function of its arguments.
 *   bounds, swarm, cfg  host
 *   trace       device [n_traces][W]
 *   theta_star  host   [n_traces][D]   out: physical parameters of the best
 *   J_star      host   [n_traces]      out: its misfit
 *   swarm_dump  device [n_iters][n_traces*n_particles][3D+2] or NULL:
 *               per iteration and particle (x[D], v[D], pbest[D], J, pbestJ)
 *               after the personal-best update and before the move
 *   gbest_hist  device [n_iters][n_traces][D+1] or NULL: (gbest x[D], gbestJ)
 *   n_iters_done host  int32 or NULL: batches actually run (j_target)
 * Synchronous: returns when the host outputs are valid. */
int afm_pso_invert(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                   uint64_t seed, const double* trace, const afm_cfg* cfg,
                   double* theta_star, double* J_star, double* swarm_dump,
                   double* gbest_hist, int32_t* n_iters_done,
                   void* cuda_stream);

/* Same inversion with the trace in HOST memory (copied inside the call). */
int afm_pso_invert_host(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                        uint64_t seed, const double* trace, const afm_cfg* cfg,
                        double* theta_star, double* J_star,
                        int32_t* n_iters_done, void* cuda_stream);

/* One PSO move applied to caller-held swarm state (the a5-a7 steps of
 * SURVEY.md 8(a) on their own, for tests and for callers that supply their
 * own misfits): personal-best update from J, global best per trace, then
 * Eq. 8 + position update + bound rule.  All device, FP64:
 *   x, v, pbest [PT][D]; J, pbestJ [PT]; gbest [n_traces][D];
 *   gbestJ [n_traces]; PT = n_traces * swarm->n_particles.
 * do_move == 0 stops after the best updates.  Asynchronous. */
int afm_pso_step(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                 int32_t n_dims, int32_t n_traces, uint64_t seed,
                 int32_t iteration, int32_t do_move, const double* J,
                 double* x, double* v, double* pbest, double* pbestJ,
                 double* gbest, double* gbestJ, void* cuda_stream);

/* afm_pso_step with the swarm state and the misfits in HOST memory: copies
 * J, x, v, pbest, pbestJ, gbest, gbestJ to the device, steps, copies the six
 * state arrays back and synchronises the stream (with afm_forward_batch_host the
 * end-to-end step that bench.py times).  All pointers host. */
int afm_pso_step_host(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                      int32_t n_dims, int32_t n_traces, uint64_t seed,
                      int32_t iteration, int32_t do_move, const double* J,
                      double* x, double* v, double* pbest, double* pbestJ,
                      double* gbest, double* gbestJ, void* cuda_stream);

/* Initial swarm (uniform positions and velocities in the box):
 * fills x, v, pbest [PT][D] and sets pbestJ [PT], gbestJ [n_traces] to +Inf,
 * gbest [n_traces][D] to the first particle of each trace.  Asynchronous. */
int afm_pso_init(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                 int32_t n_dims, int32_t n_traces, uint64_t seed, double* x,
                 double* v, double* pbest, double* pbestJ, double* gbest,
                 double* gbestJ, void* cuda_stream);

/* ---- Sharded swarm ------------------------------------------
 * One process per GPU holds a contiguous slice of a larger swarm: local
 * particle i of this process is global particle first_particle + i (global
 * indices run trace-major: trace * particles_per_trace + i, as in
 * afm_pso_invert).  Philox counters and the lowest-index tie-break use the
 * global index, so a sharded run replays the unsharded one bit for bit.  The
 * only data exchanged per iteration is the candidate row of every rank
 * (per trace D + 2 doubles, or 3 D + 4 with the ring topology, whose rows also
 * carry the personal bests of the shard's first and last particle: the ring
 * neighbours of the adjacent shards), which the CALLER all-gathers
 * (torch.distributed / NCCL) between afm_pso_shard_eval and afm_pso_shard_move;
 * sharding whole traces needs no exchange (n_ranks = 1, gathered = own
 * cand_out).  swarm->n_particles is the LOCAL particle count per local trace.
 * The asynchronous swarm (async_chunk) is not available here. */

/* afm_pso_init for a shard.  Note: gbest is set to the first LOCAL particle;
 * when one trace is sharded over ranks, copy rank 0's gbest to the others. */
int afm_pso_shard_init(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       int32_t n_dims, int32_t n_traces, uint64_t seed,
                       int64_t first_particle, double* x, double* v,
                       double* pbest, double* pbestJ, double* gbest,
                       double* gbestJ, void* cuda_stream);

/* Rows a1-a5 + the local part of a6 for this shard: theta = map(x), forward
 * solve + misfit, personal bests, and the shard's best candidate per trace.
 * All device, FP64:  trace [cfg->n_traces][W]; x, pbest [PT][D]; J, pbestJ
 * [PT]; cand_out [cfg->n_traces][R], R = D + 2 = { pbestJ, global index, pbest
 * x[D] }, or with swarm->topology == 1 R = 3 D + 4 = that + { pbestJ, pbest
 * x[D] } of the first and of the last local particle of the trace.
 * Asynchronous. */
int afm_pso_shard_eval(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       const double* trace, const afm_cfg* cfg,
                       int64_t first_particle, const double* x, double* J,
                       double* pbest, double* pbestJ, double* cand_out,
                       void* cuda_stream);

/* Rest of a6 + a7: global best per trace from the gathered candidates
 * (device [n_ranks][n_traces][R]; lowest global index among equal minima,
 * replaced only on a strict improvement), then Eq. 8 + move + bound rule when
 * do_move != 0.  rank: which of the n_ranks row blocks is this process's own;
 * swarm_particles: particles per trace of the WHOLE swarm (= swarm->n_particles
 * when whole traces are sharded).  With the ring topology and a swarm split
 * over ranks (one trace, consecutive slices in rank order) the neighbours of
 * the shard's edge particles are read from the rows of rank - 1 and rank + 1
 * (wrapping), and pbestJ [PT] (device) is required; otherwise pbestJ may be
 * NULL.  theta_star [n_traces][D], J_star [n_traces]: device or NULL.
 * Asynchronous. */
int afm_pso_shard_move(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       int32_t n_dims, int32_t n_traces, uint64_t seed,
                       int32_t iteration, int32_t do_move,
                       int64_t first_particle, const double* gathered,
                       int32_t n_ranks, int32_t rank, int64_t swarm_particles,
                       double* x, double* v, const double* pbest,
                       const double* pbestJ, double* gbest, double* gbestJ,
                       double* theta_star, double* J_star, void* cuda_stream);

/* ---- Multi-mode Euler-Bernoulli cantilever (the paper's own forward model) ----
 * PAPER.md:59-66 (Eq. 1-2), 128-139 (Eq. 6-7, Newton + Simpson initialisation,
 * RK4), Appendix A/B; R21/R22.
 *   u(x,t) = sum_i Phi_i(x) eta_i(t),  i < n_modes <= 8
 *   eta_i'' + (w_i/Q) eta_i' + w_i^2 eta_i =
 *       [ F_ts(u(L)+z_c, u'(L); theta) Phi_i(L) + mu A_base w^2 cos(w t) <1,Phi_i> ]
 *       / (mu <Phi_i,Phi_i>)
 * from rest, classical RK4 with steps_per_cycle steps per drive period; the
 * misfit is sum over the window of (u(L,t_n) - U_n)^2; +Inf if a state is
 * non-finite or |u(L)| > 100 A_ref.  FP64 only.  Host struct, plain POD. */
typedef struct {
  double L, E, I, mu;      /* length m, Young's modulus Pa, area moment m^4, kg/m */
  double Q;                /* modal quality factor (2 zeta = 1/Q)                */
  double f_drive;          /* Hz                                                 */
  double A_base;           /* base displacement amplitude y_ex = A_base cos(wt)  */
  double A_ref;            /* reference tip amplitude of the divergence rule, m  */
  double z_c, R, a0;       /* as in afm_cfg                                      */
  int32_t law, n_params;   /* afm_law and its D                                  */
  int32_t n_modes;         /* 1, 2, 4 or 8                                       */
  int32_t n_points;        /* Simpson points for the inner products (odd, >= 3)  */
  int32_t steps_per_cycle, n_cycles, n_skip_cycles;
  int32_t n_traces;
} afm_beam_cfg;

/* Modal data computed by the library's initialisation kernel (tests): all host,
 * [n_modes] each, any may be NULL.  omega rad/s; phi_L = Phi_i(L);
 * participation = Phi_i(L) <1,Phi_i>/<Phi_i,Phi_i>;
 * compliance = Phi_i(L)^2 / (mu <Phi_i,Phi_i>)  [1/kg].  Synchronous. */
int afm_beam_modes(const afm_beam_cfg* cfg, double* beta_L, double* omega,
                   double* phi_L, double* participation, double* compliance,
                   void* cuda_stream);

/* Forward batch of the beam model.  params device [P][D]: physical theta, or
 * PSO coordinates when bounds != NULL (theta_j = 10^x_j where
 * bounds->log10_scale[j]); trace device [n_traces][W]; misfit device [P].
 * Asynchronous apart from one 512-byte read-back of the modal constants. */
int afm_beam_forward_batch(const double* params, int64_t n_particles,
                           const double* trace, const afm_beam_cfg* cfg,
                           const afm_bounds* bounds, double* misfit,
                           void* cuda_stream);

/* afm_pso_invert around the beam forward batch: same swarm rules (cutoff, ring),
 * same Philox streams, same outputs; the asynchronous swarm is not available. */
int afm_beam_pso_invert(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                        uint64_t seed, const double* trace,
                        const afm_beam_cfg* cfg, double* theta_star,
                        double* J_star, double* swarm_dump, double* gbest_hist,
                        int32_t* n_iters_done, void* cuda_stream);

/* Tip deflection and velocity of ONE particle, device [N+1] each (or NULL),
 * index 0 = rest.  theta host [D].  Asynchronous. */
int afm_beam_trajectory(const double* theta, const afm_beam_cfg* cfg,
                        double* tip_u, double* tip_v, void* cuda_stream);

/* Philox4x32-10 on the device for n counters (tests: known answers).
 *   ctr device [n][4] uint32, key host [2], out device [n][4].  Async. */
int afm_philox4x32_10(const uint32_t* ctr, int64_t n, const uint32_t* key,
                      uint32_t* out, void* cuda_stream);

/* Trajectory of ONE particle through the same device step routine the batch
 * kernel uses (tests and diagnostics only): zs, vs device [N+1] or NULL;
 * index 0 is the initial state.  theta host [D].  Asynchronous. */
int afm_trajectory(const double* theta, const afm_cfg* cfg, double z0,
                   double v0, double* zs, double* vs, void* cuda_stream);

/* Register-only FMA throughput of the device (the measured
 * denominator reported beside the lane-model peak).  Runs a kernel of
 * independent dependent-FMA chains for about `seconds` (0 < seconds <= 10) in
 * the given afm_precision and writes the sustained rate, counting 2 flops per
 * FMA, to *tflops (host).  Synchronous.  Not part of the hot path. */
int afm_fma_peak(int32_t precision, double seconds, double* tflops,
                 void* cuda_stream);

/* Measurement aid: after afm_set_option("kernel_events", 1)
 * every launch of an integrate-and-misfit kernel (the dominant kernel of every
 * compute call) is bracketed by a pair of CUDA events recorded on the stream it
 * is launched on.  afm_kernel_times waits for the recorded launches and writes
 * the durations of the most recent min(max_n, 64, launches recorded) of them,
 * oldest first, in milliseconds, to ms (host); *n_out = how many.  Switching
 * the option on or off resets the record. */
int afm_kernel_times(double* ms, int32_t max_n, int32_t* n_out);

/* Health of the segment-queue kernels (option "queue").  A queue worker that
 * waits about 20 s for a task gives up, which only a corrupted queue can cause;
 * the chains it would have run keep whatever their output slots held before.
 * The synchronous calls check for this themselves and return AFM_ECUDA.  The
 * asynchronous device-pointer calls (afm_forward_batch, afm_beam_forward_batch,
 * afm_pso_shard_eval) cannot: call this after them, before trusting their
 * outputs.  Waits for cuda_stream, then returns AFM_OK, or AFM_ECUDA if a worker
 * has given up since the last check (the flag is cleared by the check). */
int afm_queue_status(void* cuda_stream);

/* Name of the integrate kernel that the most recent compute call on the calling
 * thread launched: "integrate_misfit_f64", "integrate_misfit_f64_q" (segment
 * queue), "integrate_misfit_f32", "integrate_misfit_f32_q", "beam_integrate_f64",
 * "beam_integrate_f64_q", or "" before the first one.  The event pairs of
 * afm_kernel_times bracket exactly that kernel (the queue's reset kernel is
 * launched before the start event).  Static storage; never NULL. */
const char* afm_last_integrate_kernel(void);

/* Kernel launches enqueued by this library on the calling thread since the
 * last reset (bench.py's gpu_launches). */
int64_t afm_launch_count(void);
void afm_reset_launch_count(void);

/* Tuning knobs (optional).  name: "block" (threads per CTA of the integrate
 * kernel: 32, 64 or 128; 0 = auto), "tile" (steps per time tile; 0 = auto),
 * "ppt" (particles per thread of the FP32 kernel: 1 or 2; 0 = auto = 1; the FP64
 * kernels always take one), "form" (FP64 kernel form:
 * 1 = throughput, fewest FP64 instructions; 2 = latency, shortest dependent
 * chains; 0 = auto by warps per SM sub-partition), "lanes" (latency form of the
 * DMT laws: particles per warp, a power of two up to 32; 0 = auto, as many as
 * spread the batch over all SM sub-partitions), "pack" (order the particles
 * of a DMT-law batch by trace, initial phase and stiffness so that the lanes of a
 * warp touch the sample together: 1 = never, 2 = always, 0 = auto in the
 * throughput regime; results do not depend on it), "queue" (segment-queue
 * scheduling of the throughput forms and of the beam kernel: the time loop of
 * every warp of particles is cut into segments that persistent workers take from
 * a priority queue keyed by the segment index, fewer workers than warps of
 * particles, so that the warps that are ahead wait for the ones that are behind;
 * 1 = never, 2 = always,
 * 0 = auto: batches of at least 1.5 warps per SM sub-partition; results do not
 * depend on it), "segs" (segments per trajectory, 0 = auto, about 1 000 steps
 * each), "workers" (queue workers per SM sub-partition, 1..8, 0 = auto),
 * "boost" (0 = auto, 1 = off, k >= 2: a worker that takes a segment which more
 * than 1/k of the warps of particles have already finished makes one other
 * worker of its sub-partition pause for that segment; auto = 2), "boost2"
 * (0 = auto: a segment two behind makes two other workers pause, 1 = off).
 * Returns AFM_EINVAL for an unknown name or value. */
int afm_set_option(const char* name, int64_t value);

const char* afm_last_error(void);
const char* afm_version(void);
void afm_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* AFM_H */
