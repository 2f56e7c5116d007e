// afm_internal.h -- shared between the kernel translation unit and the C-ABI
// host code of libafm_b200.so.  Not part of the public interface (include/afm.h)
// and shared with nothing outside csrc/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "afm.h"

namespace afm {

// Scaled constants of the point-mass ODE (north_star; m = 1 case of Eq. 2,
// PAPER.md:64) in "per-step" variables: state (d, w) with d = z + z_c the gap
// and w = h z' the displacement per step, so one RK4 step has unit length and
//     w' = Dp(t) - alpha w - beta d + f(d, w),
//     Dp(t) = (h^2 F0/m) cos(w_drive t) + beta z_c,   f = (h^2/m) F_ts.
// Everything here is computed on the host in FP64 from afm_cfg.
struct ModelConsts {
  double h;          // dt = 2 pi / (w_drive S)
  double w_drive;    // 2 pi f_drive
  double alpha;      // h w0 / Q
  double beta;       // (h w0)^2
  double drive_amp;  // h^2 F0 / m
  double beta_zc;    // beta z_c
  double zc, a0;
  double inv_a0sq;   // 1 / a0^2
  double c_vdw;      // h^2 R / (6 m):        kappa = H c_vdw
  double c_hertz;    // h^2 (4/3) sqrt(R)/m:  eps   = E* c_hertz
  double c_visc;     // h sqrt(R) / m:        nu    = eta c_visc
  double c_force;    // h^2 / m
  double c_damp;     // h / m:  (h/m) zeta_s adds to alpha (Kelvin-Voigt)
  double d_max;      // z_c + 100 A0   (divergence rule R12 on d)
  double d_min;      // z_c - 100 A0   (negative)
  double d_safe;     // max(0, 100 A0 - |z_c|): |d| < d_safe => not diverged
  double z0, v0;     // default initial state, SI
  int32_t law, D;
  int32_t N;         // total steps
  int32_t n0;        // first step whose post-state is in the misfit window
  int32_t W;         // window length
  int32_t T;         // steps per time tile
  int32_t n_tiles;
  int32_t pad_;
};

// FP32 kernel constants (R14; afm_device_f32.cuh).  Kernel units:
// length 1 nm, one RK4 step = unit time; every acceleration coefficient is
// pre-scaled by 1/6 (b6 = beta/6, a6 = alpha/6).  Computed on the host in FP64.
struct ModelConstsF32 {
  double len;        // metres per kernel length unit (1e-9)
  double h;          // step, seconds
  double w_drive;
  double a6, b6;     // alpha/6, beta/6 in FP64 (split hi/lo by the kernel)
  double drive6;     // b6 * (F0/k) / len: drive amplitude of the scaled stream
  double b6_zc;      // b6 * z_c / len
  double zc, a0;     // nm
  double c_vdw;      // c0 = -theta0 c_vdw, c2 = c0 / a0^2        (DMT)
  double c_hertz;    // c1 = theta1 c_hertz
  double c_visc;     // c3 = -theta2 c_visc
  double c_rep, c_att, c_fad;  // LJ+exp: c0 = theta0 c_rep, c1 = -theta1 c_att, c2 = -theta2 c_fad
  double c_lam;      // c3 = -c_lam / theta3  (log2(e) len)
  double c_ks;       // Hooke / Kelvin-Voigt: c1 = theta0 c_ks   (b6 / k)
  double c_zeta;     // Kelvin-Voigt: c3 = -(a6 + theta1 c_zeta)  (b6 / (h k))
  double d_max, d_min, d_safe;  // nm
  double z0, v0;     // default initial state, SI
  int32_t law, D, N, n0, W, T, n_tiles, pad_;
};

// Per-mode constants of the beam kernel in per-step, tip-weighted variables
// (afm_beam.cu): a_i = Phi_i(L) eta_i, b_i = h Phi_i(L) eta_i',
//   b_i' = Gamma_i cos(w t) - alpha_i b_i - beta_i a_i + kappa_i fhat,
// fhat = (h^2/m_1) F_ts, m_1 = first-mode effective mass, kappa_0 = 1.
struct BeamModeConsts {
  double Gamma[8], alpha[8], beta[8], kappa[8];
  // raw modal data for afm_beam_modes
  double bL[8], omega[8], phiL[8], part[8], compl_[8];
  double m1;  // mu <Phi_0,Phi_0> / Phi_0(L)^2
};

struct BeamConsts {
  double h, w_drive;
  double zc, a0, inv_a0sq;
  double c_vdw, c_hertz, c_visc, c_force, c_damp;  // as ModelConsts, with m = m_1
  double u_max;      // 100 A_ref
  int32_t law, D, M, N, n0, W, T, n_tiles;
};

struct BoxDev {
  double lo[4], hi[4];
  int32_t lg[4];
};

struct SwarmDev {
  double w, c1, c2;
  int32_t topology;  // 0 global best, 1 ring of three
  int32_t pad_;
};

// One block-level (pbestJ, particle index) candidate of the global-best search.
struct Cand {
  double J;
  long long idx;
};

// ---- launchers (afm_kernels.cu) -------------------------------------------
// Every launcher returns the number of kernels it enqueued (>= 1) or a
// negative value after setting a CUDA error (checked by the caller with
// cudaGetLastError()).

struct IntegrateIO {
  const double* params;   // MODE 0: theta [PT][D]; MODE 1: x [PT][D]
  const double* z0v0;     // [PT][2] or nullptr
  const double* stream;   // [n_traces][N][4] time-tile stream (FP32 kernel: float4 rows)
  double* J;              // [PT]
  // MODE 1 (PSO) only:
  double* pbest;          // [PT][D]
  double* pbestJ;         // [PT]
  Cand* cand;             // [n_traces][blocks_per_trace]
  BoxDev box;
  int64_t per;            // particles per trace
  int32_t n_traces;
  int32_t mode;           // 0 forward, 1 PSO
  int32_t lanes;          // latency form: particles per warp (power of two, 1..32)
  int32_t pad_;
};

// Segment queue of integrate_misfit_f64_q (afm_kernels.cu): tasks are
// (chain, segment) = (warp of 32 particles, run of tiles_per_seg time tiles).
struct SegQueue {
  int* slots;            // [n_segs][n_chains]  chain, or -1 = not yet published
  unsigned* ctrl;        // [0] lowest level not handed out in full, [2] time-out flag
  unsigned* head;        // [n_segs] tasks handed out per level
  unsigned* tail;        // [n_segs] tasks published (slots reserved) per level
  unsigned* park;        // [n_park] parking place per SM sub-partition (segq_pop)
  int32_t n_park;        // 4 * SMs, or 0: no boost of the chains that are behind
  int32_t boost_two;     // 1: a task two levels behind gets a second parking place
  int32_t boost_div;     // a task is behind when more than n_chains / boost_div chains
                         // have finished its level
  double* ckpt;          // [n_chains][4][32] doubles: d, w, J, diverged flag of a chain at
                         // rest (FP32 kernel: [n_chains][8][32] floats, same size; beam
                         // kernel: [n_chains][2 M + 2][32] doubles)
  long long timeout_cycles;
  int32_t n_chains;
  int32_t n_segs;
  int32_t n_tasks;       // n_chains * n_segs
  int32_t tiles_per_seg;
};

int blocks_per_trace(int64_t per, int block);
int launch_segq_init(const SegQueue& q, cudaStream_t st);
int launch_integrate_f64_q(const ModelConsts& mc, const IntegrateIO& io,
                           const SegQueue& q, int workers, cudaStream_t st);
int launch_integrate_f32_q(const ModelConstsF32& mf, const IntegrateIO& io,
                           const SegQueue& q, int workers, cudaStream_t st);

int launch_build_stream(const ModelConsts& mc, const double* trace, int n_traces,
                        double* stream, cudaStream_t st);
int launch_build_stream_f32(const ModelConstsF32& mf, const double* trace,
                            int n_traces, float* stream, cudaStream_t st);
int launch_integrate_f64(const ModelConsts& mc, const IntegrateIO& io, int block,
                         int variant, cudaStream_t st);
int launch_integrate_f32(const ModelConstsF32& mf, const IntegrateIO& io,
                         int block, int ppt, cudaStream_t st);
int launch_trajectory(const ModelConsts& mc, const double* theta_dev,
                      const double* stream, double z0, double v0, double* zs,
                      double* vs, cudaStream_t st);

int launch_pso_init(const BoxDev& box, int D, int64_t per, int n_traces,
                    uint64_t seed, int64_t first, double* x, double* v,
                    double* pbest, double* pbestJ, double* gbest, double* gbestJ,
                    cudaStream_t st);
// Ring of three in a sharded swarm: where the neighbours outside the shard live.
// total = 0: the shard holds whole swarms (plain wrap inside the local swarm).
struct RingEdges {
  int64_t total;        // particles of the whole swarm over all shards, or 0
  int64_t off;          // in-swarm index of local particle 0
  const double* left;   // { pbestJ, pbest x[D] } of the particle before the shard,
  const double* right;  //   after the shard; trace 0's row, `stride` doubles per trace
  int64_t stride;
};

int launch_pso_best(int D, int64_t per, int64_t off, int64_t cnt, int n_traces,
                    double* J, const double* Jc, const double* x, double* pbest,
                    double* pbestJ, Cand* cand, int block, cudaStream_t st);
int launch_chunk_gather(const BoxDev& box, int D, int64_t per, int64_t off,
                        int64_t cnt, int n_traces, const double* x, double* theta_c,
                        cudaStream_t st);
int launch_pso_gbest(const BoxDev& box, int D, int n_traces, int n_cand,
                     const Cand* cand, const double* pbest, double* gbest,
                     double* gbestJ, double* hist_row, double* theta_star,
                     double* J_star, cudaStream_t st);
int launch_pso_move(const BoxDev& box, const SwarmDev& sw, int D, int64_t per,
                    int64_t off, int64_t cnt, int n_traces, uint64_t seed,
                    int64_t first, uint32_t it, int do_move, const RingEdges& re,
                    const double* J, double* x, double* v, const double* pbest,
                    const double* pbestJ, const double* gbest, double* dump_row,
                    cudaStream_t st);
int launch_pso_shard_cand(int D, int n_traces, int n_cand, int64_t first,
                          int64_t per, int ring, const Cand* cand,
                          const double* pbest, const double* pbestJ,
                          double* cand_out, cudaStream_t st);
int launch_pso_shard_gbest(const BoxDev& box, int D, int n_traces, int n_ranks,
                           int width, const double* gathered, double* gbest,
                           double* gbestJ, double* theta_star, double* J_star,
                           cudaStream_t st);
int launch_fma_peak(int precision, int iters, int blocks, int threads,
                    void* sink, float* ms, cudaStream_t st);
int launch_beam_setup(const afm_beam_cfg& cfg, double h, BeamModeConsts* dev_out,
                      cudaStream_t st);
int launch_beam_integrate(const BeamConsts& bc, const BeamModeConsts& mo,
                          const IntegrateIO& io, int block, cudaStream_t st);
int launch_beam_integrate_q(const BeamConsts& bc, const BeamModeConsts& mo,
                            const IntegrateIO& io, const SegQueue& q, int workers,
                            cudaStream_t st);
int launch_beam_trajectory(const BeamConsts& bc, const BeamModeConsts& mo,
                           const double* theta_dev, const double* stream,
                           double* tip_u, double* tip_v, cudaStream_t st);
// Warp packing (afm_sort.cu): order[] = particle indices sorted by (trace, initial
// phase bin, stiffness-like parameter), so that the lanes of a warp touch the
// sample at about the same time.  ws/ws_bytes: scratch for the radix sort.  The
// integrate kernels are left untouched: inputs are gathered into packed copies
// and the misfits scattered back.
size_t sort_workspace_bytes(int64_t PT);
int launch_pack_order(const double* params, const double* z0v0, int D, int64_t per,
                      int64_t PT, double w_drive, double z0_default,
                      double v0_default, void* ws, size_t ws_bytes,
                      uint32_t* order, cudaStream_t st);
int launch_pack_gather(const uint32_t* order, const double* params,
                       const double* z0v0, int D, int64_t PT, double* params_s,
                       double* z0v0_s, const BoxDev* map, cudaStream_t st);
int launch_pack_scatter(const uint32_t* order, const double* J_s, int64_t PT,
                        double* J, cudaStream_t st);
int launch_philox(const uint32_t* ctr, int64_t n, uint32_t k0, uint32_t k1,
                  uint32_t* out, cudaStream_t st);

}  // namespace afm
