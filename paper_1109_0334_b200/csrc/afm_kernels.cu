// afm_kernels.cu -- sm_100a kernels of the dAFM force-inversion hot path.
//
//   build_stream_kernel     time-tile stream: drive at the three RK4 abscissae
//                           of every step + the measured trace, 32 B per step
//   integrate_misfit_f64    a1-a5 of SURVEY.md 8(a): parameter map, RK4 forward
//                           solve with register-resident state, squared misfit,
//                           personal best + block argmin candidate (PSO mode)
//   pso_init/best/gbest/move  a5-a7: Philox-driven swarm (Eq. 8)
//
// One thread integrates one particle; the particles of a CTA share one trace,
// which (with the drive) is streamed global -> shared by 1-D bulk async copies
// (cp.async.bulk, SASS UBLKCP) into a two-stage mbarrier ring.
#include <math_constants.h>

#include "afm_device.cuh"
#include "afm_internal.h"

namespace afm {

constexpr int kPadRows = kPadBytes / 32;  // pad rows after each stage of the tile ring

// ============================================================================
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): the counter-based
// generator north_star names.  DESIGN.md reading R11 fixes key and counter.
// ============================================================================
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1,
                                              uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1,
                                              uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    c0 = n0;
    c1 = lo1;
    c2 = n2;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0;
  out[1] = c1;
  out[2] = c2;
  out[3] = c3;
}

// 24-bit uniform in [0, 1), exact in FP32 and FP64.
__device__ __forceinline__ double u24(uint32_t word) {
  return (double)(word >> 8) * (1.0 / 16777216.0);
}

// a[j], b[j] for j < D: counter = (particle lo, iteration, pair + 16*purpose,
// particle hi); the four words of pair q are (a[2q], b[2q], a[2q+1], b[2q+1]).
__device__ __forceinline__ void pso_uniforms(uint64_t seed, uint64_t gp,
                                             uint32_t it, uint32_t purpose,
                                             int D, double a[4], double b[4]) {
  const uint32_t k0 = (uint32_t)(seed & 0xffffffffu);
  const uint32_t k1 = (uint32_t)(seed >> 32);
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    if (2 * q < D) {
      uint32_t o[4];
      philox4x32_10((uint32_t)(gp & 0xffffffffu), it,
                    (uint32_t)q + 16u * purpose, (uint32_t)(gp >> 32), k0, k1,
                    o);
      a[2 * q] = u24(o[0]);
      b[2 * q] = u24(o[1]);
      a[2 * q + 1] = u24(o[2]);
      b[2 * q + 1] = u24(o[3]);
    }
  }
}

__global__ void philox_kernel(const uint32_t* __restrict__ ctr, int64_t n,
                              uint32_t k0, uint32_t k1,
                              uint32_t* __restrict__ out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t o[4];
  philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0,
                k1, o);
  out[4 * i] = o[0];
  out[4 * i + 1] = o[1];
  out[4 * i + 2] = o[2];
  out[4 * i + 3] = o[3];
}

// ============================================================================
// Time-tile stream.  Row n of trace s: { Dp(t_n), Dp(t_n + h/2), Dp(t_n + h),
// U_s[n - n0] + z_c (0 before the window) },  t_n = n h (never accumulated),
// Dp(t) = drive_amp cos(w t) + beta z_c.
// ============================================================================
__global__ void build_stream_kernel(ModelConsts mc,
                                    const double* __restrict__ trace,
                                    int n_traces, double* __restrict__ stream) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t total = (int64_t)n_traces * mc.N;
  if (i >= total) return;
  int s = (int)(i / mc.N);
  int n = (int)(i - (int64_t)s * mc.N);
  double t = __dmul_rn((double)n, mc.h);
  double th = __dadd_rn(t, __dmul_rn(0.5, mc.h));
  double t1 = __dadd_rn(t, mc.h);
  double4 row;
  row.x = fma(mc.drive_amp, cos(__dmul_rn(mc.w_drive, t)), mc.beta_zc);
  row.y = fma(mc.drive_amp, cos(__dmul_rn(mc.w_drive, th)), mc.beta_zc);
  row.z = fma(mc.drive_amp, cos(__dmul_rn(mc.w_drive, t1)), mc.beta_zc);
  row.w = (n >= mc.n0) ? trace[(int64_t)s * mc.W + (n - mc.n0)] + mc.zc : 0.0;
  reinterpret_cast<double4*>(stream)[i] = row;
}

// ============================================================================
// integrate-and-misfit, FP64
// ============================================================================
// T steps of one time tile, [i0, i1), with (WIN) or without the misfit sum.
template <int LAW, int PPT, bool LAT, bool WIN>
__device__ __forceinline__ void run_steps(const double4* sp, int i0, int i1,
                                          const Particle64 (&P)[PPT],
                                          long long a0_bits,
                                          const DivergeTest& T,
                                          double (&d)[PPT], double (&w)[PPT],
                                          double (&J)[PPT], bool (&bad)[PPT],
                                          int& mode) {
  if (i0 >= i1) return;
  AFM_CHECK(i0 >= 0);
  double4 r = sp[i0];
#pragma unroll 2
  for (int i = i0; i < i1; ++i) {
    // next row fetched one step ahead; the fetch past the last row of a tile
    // reads the stage's own pad row (zeroed once, never a bulk-copy target)
    const double4 rn = sp[i + 1];
    rk4_step<LAW, PPT, LAT>(P, r.x, r.y, r.z, a0_bits, d, w, mode, bad, T);
    if (WIN) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) {
        const double res = d[q] - r.w;
        J[q] = fma(res, res, J[q]);
      }
    }
    r = rn;
  }
}

// PPT particles per thread: particle q of a thread is local index
// base + q * blockDim.x + tid (coalesced).  PPT = 2 interleaves two independent
// dependency chains per thread for the throughput-bound batches.
template <int LAW, int MODE, int PPT, bool LAT>
__global__ void integrate_misfit_f64(ModelConsts mc, IntegrateIO io,
                                     int blocks_per_tr) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // two stages of T rows, each followed by one pad row for the one-step-ahead fetch
  double4* tile0 = reinterpret_cast<double4*>(smem_raw);
  double4* tile1 = tile0 + (mc.T + kPadRows);
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (mc.T + kPadRows));
  __shared__ Cand red[32];

  const int tid = threadIdx.x;
  const int s = blockIdx.x / blocks_per_tr;  // trace (segment) of this CTA
  // Latency form: only io.lanes lanes of the (single) warp carry particles, the
  // others shadow them.  With one warp or less per SM sub-partition nothing is
  // gained by filling warps, and a warp of few particles leaves the free-flight
  // form only when ITS particles touch the sample, not when any of 32 does.
  const int64_t base =
      LAT ? (int64_t)(blockIdx.x - s * blocks_per_tr) * io.lanes + (tid & (io.lanes - 1))
          : (int64_t)(blockIdx.x - s * blocks_per_tr) * blockDim.x * PPT + tid;
  bool active[PPT];
  int64_t gp[PPT];
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    const int64_t li = base + (int64_t)q * blockDim.x;
    active[q] = (li < io.per) && (!LAT || tid < io.lanes);
    // an inactive slot of a ragged last CTA integrates a copy of the segment's
    // last particle (keeps every vote and barrier uniform) and writes nothing
    gp[q] = (int64_t)s * io.per + (active[q] ? li : io.per - 1);
    AFM_CHECK(s < io.n_traces && gp[q] >= 0 && gp[q] < io.per * io.n_traces);
  }

  const double* stream = io.stream + (int64_t)s * mc.N * 4;

  if (tid == 0) {
    tile0[mc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    tile1[mc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int st = 0; st < 2; ++st) {
      if (st < mc.n_tiles) {
        int n_begin = st * mc.T;
        uint32_t bytes = (uint32_t)min(mc.T, mc.N - n_begin) * 32u;
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + (int64_t)n_begin * 4, bytes,
                 &bars[st]);
      }
    }
  }

  // ---- a1: parameter map ---------------------------------------------------
  double xloc[PPT][4];
  Particle64 P[PPT];
  double d[PPT], w[PPT], J[PPT];
  bool bad[PPT];
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    double th[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      xloc[q][j] = 0.0;
      if (j < mc.D) {
        const double xv = io.params[gp[q] * mc.D + j];
        xloc[q][j] = xv;
        th[j] = (MODE == 1 && io.box.lg[j]) ? pow(10.0, xv) : xv;
      }
    }
    load_particle(P[q], LAW, th, mc.alpha, mc.beta, mc.a0, mc.inv_a0sq,
                  mc.c_vdw, mc.c_hertz, mc.c_visc, mc.c_force, mc.zc, mc.c_damp);
    double z0 = mc.z0, v0 = mc.v0;
    if (io.z0v0 != nullptr) {
      z0 = io.z0v0[2 * gp[q]];
      v0 = io.z0v0[2 * gp[q] + 1];
    }
    d[q] = z0 + mc.zc;
    w[q] = v0 * mc.h;
    J[q] = 0.0;
    bad[q] = false;
  }
  const long long a0_bits = __double_as_longlong(mc.a0);
  DivergeTest T;
  T.key_max = order_key(mc.d_max);
  T.key_min = order_key(mc.d_min);
  T.safe_hi = __double2hiint(mc.d_safe);
  int mode = 0;  // warp-uniform: 0 = speculate free flight, 1 = general

  // ---- a2-a4: RK4 over the time tiles -------------------------------------
  for (int tile = 0; tile < mc.n_tiles; ++tile) {
    const int st = tile & 1;
    const double4* sp = st ? tile1 : tile0;
    mbar_wait(&bars[st], (uint32_t)((tile >> 1) & 1));
    const int n_begin = tile * mc.T;
    const int n_steps = min(mc.T, mc.N - n_begin);
    AFM_CHECK(n_steps >= 1 && n_steps <= mc.T && n_begin + n_steps <= mc.N);
    // steps [0, k0) of this tile precede the misfit window
    const int k0 = max(0, min(n_steps, mc.n0 - n_begin));
    run_steps<LAW, PPT, LAT, false>(sp, 0, k0, P, a0_bits, T, d, w, J, bad, mode);
    run_steps<LAW, PPT, LAT, true>(sp, k0, n_steps, P, a0_bits, T, d, w, J, bad, mode);
    __syncthreads();  // every thread is done reading stage st
    if (tid == 0 && tile + 2 < mc.n_tiles) {
      const int nb = (tile + 2) * mc.T;
      const uint32_t bytes = (uint32_t)min(mc.T, mc.N - nb) * 32u;
      fence_proxy_async();
      mbar_arrive_expect_tx(&bars[st], bytes);
      bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
    }
  }

  double pb = CUDART_INF;
  long long idx = 0x7fffffffffffffffLL;
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    // the velocity of the last state must be finite too (R12)
    const long long kw = __double_as_longlong(w[q]) & 0x7fffffffffffffffLL;
    bad[q] |= (kw >= 0x7ff0000000000000LL);
    if (bad[q] || !(J[q] == J[q])) J[q] = CUDART_INF;
    if (active[q]) io.J[gp[q]] = J[q];

    // ---- a5 + first level of a6 (PSO mode) ---------------------------------
    if (MODE == 1 && active[q]) {
      double pq = io.pbestJ[gp[q]];
      if (J[q] < pq) {  // strict: NaN/+Inf never win
        pq = J[q];
        io.pbestJ[gp[q]] = J[q];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (j < mc.D) io.pbest[gp[q] * mc.D + j] = xloc[q][j];
      }
      if (cand_less(pq, gp[q], pb, idx)) {
        pb = pq;
        idx = gp[q];
      }
    }
  }
  if (MODE == 1) {
    block_argmin(pb, idx, red);
    if (tid == 0) {
      io.cand[blockIdx.x].J = pb;
      io.cand[blockIdx.x].idx = idx;
    }
  }
}

// ============================================================================
// integrate-and-misfit, FP64, segment queue (throughput form, one warp per CTA).
//
// With every warp of particles bound to one SM sub-partition for its whole
// trajectory a batch is unbalanced twice over: 2 048 warps on 592 sub-partitions
// leave 3 on some and 4 on others, and warps differ up to 2x in cost (general-form
// steps; a warp with one particle stuck to the sample runs every step in the
// general form), so the slowest warp sets the time.  Here the time loop of a warp
// of particles (a "chain") is cut into segments of q.tiles_per_seg time tiles; a
// grid of persistent one-warp CTAs (workers, a whole number per sub-partition,
// FEWER than chains) takes (chain, segment) tasks from a priority queue in global
// memory keyed by the segment index (segq_pop / segq_push in
// afm_device_common.cuh).  A worker that finishes a segment stores the chain's
// state (d, w, J, diverged flag: 32 B per particle), publishes the chain's next
// segment and takes the oldest task of the lowest segment index on offer: the
// chains that are ahead wait, the ones that are behind are picked up at once, and
// the few that still cannot keep up get their sub-partition to themselves (the
// boost in segq_pop).  The arithmetic of a particle is that of
// integrate_misfit_f64<LAW, MODE, 1, false>, step for step: results are
// bit-identical.
// ============================================================================
__global__ void segq_init_kernel(SegQueue q) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < q.n_tasks) q.slots[i] = (i < q.n_chains) ? i : -1;  // level 0: every chain
  if (i < q.n_segs) {
    q.head[i] = 0u;
    q.tail[i] = (i == 0) ? (unsigned)q.n_chains : 0u;
  }
  if (i < q.n_park) q.park[i] = 0u;
  if (i == 0) q.ctrl[0] = 0u;
}

template <int LAW, int MODE>
__global__ void __launch_bounds__(32)
integrate_misfit_f64_q(ModelConsts mc, IntegrateIO io, int blocks_per_tr, SegQueue q) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double4* tile0 = reinterpret_cast<double4*>(smem_raw);
  double4* tile1 = tile0 + (mc.T + kPadRows);
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (mc.T + kPadRows));
  __shared__ Cand red[32];
  __shared__ SegqWorker qworker;  // lane 0's queue state (one warp per CTA)

  const int tid = threadIdx.x;
  if (tid == 0) {
    qworker.offered = 0u;
    tile0[mc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    tile1[mc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t n_wait0 = 0u, n_wait1 = 0u;  // completed phases of the two stages
  const long long a0_bits = __double_as_longlong(mc.a0);
  DivergeTest T;
  T.key_max = order_key(mc.d_max);
  T.key_min = order_key(mc.d_min);
  T.safe_hi = __double2hiint(mc.d_safe);

  for (;;) {
    int task = 0;
    if (tid == 0) task = segq_pop(q, &qworker);
    task = __shfl_sync(0xffffffffu, task, 0);
    if (task < 0) break;
    const int chain = task & 0xfffff;
    const int seg = task >> 20;
    const int s = chain / blocks_per_tr;  // trace of this chain
    const int64_t li = (int64_t)(chain - s * blocks_per_tr) * 32 + tid;
    const bool active = li < io.per;
    const int64_t gp = (int64_t)s * io.per + (active ? li : io.per - 1);
    AFM_CHECK(s < io.n_traces && gp >= 0 && gp < io.per * io.n_traces);
    const double* stream = io.stream + (int64_t)s * mc.N * 4;
    const int tile_begin = seg * q.tiles_per_seg;
    const int tile_end = min(tile_begin + q.tiles_per_seg, mc.n_tiles);

    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const int tile = tile_begin + k;
        if (tile < tile_end) {
          const int st = tile & 1;
          const int nb = tile * mc.T;
          const uint32_t bytes = (uint32_t)min(mc.T, mc.N - nb) * 32u;
          fence_proxy_async();
          mbar_arrive_expect_tx(&bars[st], bytes);
          bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
        }
      }
    }

    // a1: parameter map (every segment: the chain may have come from another SM)
    double xloc[4];
    Particle64 P[1];
    double d[1], w[1], J[1];
    bool bad[1];
    {
      double th[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        xloc[j] = 0.0;
        if (j < mc.D) {
          const double xv = io.params[gp * mc.D + j];
          xloc[j] = xv;
          th[j] = (MODE == 1 && io.box.lg[j]) ? pow(10.0, xv) : xv;
        }
      }
      load_particle(P[0], LAW, th, mc.alpha, mc.beta, mc.a0, mc.inv_a0sq, mc.c_vdw,
                    mc.c_hertz, mc.c_visc, mc.c_force, mc.zc, mc.c_damp);
    }
    double* ck = q.ckpt + (int64_t)chain * 128 + tid;
    if (seg == 0) {
      double z0 = mc.z0, v0 = mc.v0;
      if (io.z0v0 != nullptr) {
        z0 = io.z0v0[2 * gp];
        v0 = io.z0v0[2 * gp + 1];
      }
      d[0] = z0 + mc.zc;
      w[0] = v0 * mc.h;
      J[0] = 0.0;
      bad[0] = false;
    } else {
      d[0] = __ldcg(ck);
      w[0] = __ldcg(ck + 32);
      J[0] = __ldcg(ck + 64);
      bad[0] = __ldcg(ck + 96) != 0.0;
    }
    int mode = 0;

    for (int tile = tile_begin; tile < tile_end; ++tile) {
      const int st = tile & 1;
      const double4* sp = st ? tile1 : tile0;
      mbar_wait(&bars[st], (st ? n_wait1 : n_wait0) & 1u);
      if (st) ++n_wait1; else ++n_wait0;
      const int n_begin = tile * mc.T;
      const int n_steps = min(mc.T, mc.N - n_begin);
      AFM_CHECK(n_steps >= 1 && n_steps <= mc.T && n_begin + n_steps <= mc.N);
      AFM_CHECK(tile >= 0 && tile < mc.n_tiles && tile_end <= mc.n_tiles);
      const int k0 = max(0, min(n_steps, mc.n0 - n_begin));
      run_steps<LAW, 1, false, false>(sp, 0, k0, P, a0_bits, T, d, w, J, bad, mode);
      run_steps<LAW, 1, false, true>(sp, k0, n_steps, P, a0_bits, T, d, w, J, bad, mode);
      __syncthreads();
      if (tid == 0 && tile + 2 < tile_end) {
        const int nb = (tile + 2) * mc.T;
        const uint32_t bytes = (uint32_t)min(mc.T, mc.N - nb) * 32u;
        fence_proxy_async();
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
      }
    }

    if (tile_end < mc.n_tiles) {
      // hand the chain on: state first, then the task (release / acquire)
      __stcg(ck, d[0]);
      __stcg(ck + 32, w[0]);
      __stcg(ck + 64, J[0]);
      __stcg(ck + 96, bad[0] ? 1.0 : 0.0);
      __threadfence();
      __syncwarp();
      if (tid == 0) segq_push(q, chain, seg + 1);
      continue;
    }

    // last segment: the epilogue of integrate_misfit_f64
    const long long kw = __double_as_longlong(w[0]) & 0x7fffffffffffffffLL;
    bad[0] |= (kw >= 0x7ff0000000000000LL);
    if (bad[0] || !(J[0] == J[0])) J[0] = CUDART_INF;
    if (active) io.J[gp] = J[0];
    if (MODE == 1) {
      double pb = CUDART_INF;
      long long idx = 0x7fffffffffffffffLL;
      if (active) {
        double pq = io.pbestJ[gp];
        if (J[0] < pq) {
          pq = J[0];
          io.pbestJ[gp] = J[0];
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (j < mc.D) io.pbest[gp * mc.D + j] = xloc[j];
        }
        pb = pq;
        idx = gp;
      }
      block_argmin(pb, idx, red);
      if (tid == 0) {
        io.cand[chain].J = pb;
        io.cand[chain].idx = idx;
      }
    }
  }
}

// Trajectory of one particle through the same rk4_step (tests/diagnostics).
template <int LAW>
__global__ void trajectory_kernel(ModelConsts mc, const double* __restrict__ th,
                                  const double* __restrict__ stream, double z0,
                                  double v0, double* __restrict__ zs,
                                  double* __restrict__ vs) {
  // one warp, every lane integrates the same particle (rk4_step votes across
  // the full warp); lane 0 writes
  const bool writer = (threadIdx.x == 0);
  double t4[4] = {0.0, 0.0, 0.0, 0.0};
  for (int j = 0; j < mc.D && j < 4; ++j) t4[j] = th[j];
  Particle64 P[1];
  load_particle(P[0], LAW, t4, mc.alpha, mc.beta, mc.a0, mc.inv_a0sq, mc.c_vdw,
                mc.c_hertz, mc.c_visc, mc.c_force, mc.zc, mc.c_damp);
  double d[1] = {z0 + mc.zc}, w[1] = {v0 * mc.h};
  const long long a0_bits = __double_as_longlong(mc.a0);
  const double inv_h = 1.0 / mc.h;
  int mode = 0;
  bool bad[1] = {false};
  DivergeTest T;
  T.key_max = order_key(mc.d_max);
  T.key_min = order_key(mc.d_min);
  T.safe_hi = __double2hiint(mc.d_safe);
  if (zs && writer) zs[0] = z0;
  if (vs && writer) vs[0] = v0;
  const double4* rows = reinterpret_cast<const double4*>(stream);
  for (int n = 0; n < mc.N; ++n) {
    const double4 r = rows[n];
    rk4_step<LAW, 1, true>(P, r.x, r.y, r.z, a0_bits, d, w, mode, bad, T);
    if (zs && writer) zs[n + 1] = d[0] - mc.zc;
    if (vs && writer) vs[n + 1] = w[0] * inv_h;
  }
}

// ============================================================================
// PSO kernels (readings R10/R11).  All FP64; every product
// and sum is written with explicit round-to-nearest intrinsics so that no FMA
// contraction changes the value: the swarm state replays bit for bit.
// ============================================================================
__global__ void pso_init_kernel(BoxDev box, int D, int64_t per, int n_traces,
                                uint64_t seed, int64_t first,
                                double* __restrict__ x,
                                double* __restrict__ v,
                                double* __restrict__ pbest,
                                double* __restrict__ pbestJ,
                                double* __restrict__ gbest,
                                double* __restrict__ gbestJ) {
  const int64_t gp = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t PT = per * n_traces;
  if (gp >= PT) return;
  double a[4], b[4];
  pso_uniforms(seed, (uint64_t)(first + gp), 0u, 0u, D, a, b);
  const bool head = (gp % per) == 0;
  const int64_t s = gp / per;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (j < D) {
      const double span = __dsub_rn(box.hi[j], box.lo[j]);
      const double x0 = __dadd_rn(box.lo[j], __dmul_rn(a[j], span));
      const double y0 = __dadd_rn(box.lo[j], __dmul_rn(b[j], span));
      x[gp * D + j] = x0;
      v[gp * D + j] = __dmul_rn(0.5, __dsub_rn(y0, x0));
      pbest[gp * D + j] = x0;
      if (head) gbest[s * D + j] = x0;
    }
  }
  pbestJ[gp] = CUDART_INF;
  if (head) gbestJ[s] = CUDART_INF;
}

// Personal best from caller-supplied J + block candidates (the stand-alone
// form of the epilogue fused into integrate_misfit_f64<., 1>), for the particles
// [off, off + cnt) of every swarm.  Jc != nullptr: the misfits arrive compact,
// [n_traces][cnt] (asynchronous swarm: a chunk was integrated on its own), and
// are also stored at the particles' own places in J.
__global__ void pso_best_kernel(int D, int64_t per, int64_t off, int64_t cnt,
                                int blocks_per_tr, double* __restrict__ J,
                                const double* __restrict__ Jc,
                                const double* __restrict__ x,
                                double* __restrict__ pbest,
                                double* __restrict__ pbestJ,
                                Cand* __restrict__ cand) {
  __shared__ Cand red[32];
  const int s = blockIdx.x / blocks_per_tr;
  const int64_t li =
      (int64_t)(blockIdx.x - s * blocks_per_tr) * blockDim.x + threadIdx.x;
  const bool active = li < cnt;
  const int64_t gp = (int64_t)s * per + off + li;
  AFM_CHECK(!active || (off + li < per));
  double pb = CUDART_INF;
  long long idx = 0x7fffffffffffffffLL;
  if (active) {
    double Jp;
    if (Jc != nullptr) {
      Jp = Jc[(int64_t)s * cnt + li];
      J[gp] = Jp;
    } else {
      Jp = J[gp];
    }
    pb = pbestJ[gp];
    if (Jp < pb) {
      pb = Jp;
      pbestJ[gp] = Jp;
      for (int j = 0; j < D; ++j) pbest[gp * D + j] = x[gp * D + j];
    }
    idx = gp;
  }
  block_argmin(pb, idx, red);
  if (threadIdx.x == 0) {
    cand[blockIdx.x].J = pb;
    cand[blockIdx.x].idx = idx;
  }
}

// theta = map(x) of the particles [off, off + cnt) of every swarm, compact
// [n_traces][cnt][D]: the forward batch of one chunk of an asynchronous swarm.
__global__ void chunk_gather_kernel(BoxDev box, int D, int64_t per, int64_t off,
                                    int64_t cnt, int n_traces,
                                    const double* __restrict__ x,
                                    double* __restrict__ theta_c) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cnt * n_traces) return;
  const int64_t s = i / cnt;
  const int64_t gp = s * per + off + (i - s * cnt);
  for (int j = 0; j < D; ++j) {
    const double xv = x[gp * D + j];
    theta_c[i * D + j] = box.lg[j] ? pow(10.0, xv) : xv;
  }
}

// Global best of one trace per CTA: lowest index among the minima of pbestJ,
// taken only on a strict improvement over the stored gbestJ.
__global__ void pso_gbest_kernel(BoxDev box, int D, int n_cand,
                                 const Cand* __restrict__ cand,
                                 const double* __restrict__ pbest,
                                 double* __restrict__ gbest,
                                 double* __restrict__ gbestJ,
                                 double* __restrict__ hist_row,
                                 double* __restrict__ theta_star,
                                 double* __restrict__ J_star) {
  __shared__ Cand red[32];
  const int s = blockIdx.x;
  double Jm = CUDART_INF;
  long long im = 0x7fffffffffffffffLL;
  for (int c = threadIdx.x; c < n_cand; c += blockDim.x) {
    const Cand cd = cand[(int64_t)s * n_cand + c];
    if (cand_less(cd.J, cd.idx, Jm, im)) {
      Jm = cd.J;
      im = cd.idx;
    }
  }
  block_argmin(Jm, im, red);
  if (threadIdx.x == 0) {
    double gJ = gbestJ[s];
    if (Jm < gJ) {
      gJ = Jm;
      gbestJ[s] = Jm;
      for (int j = 0; j < D; ++j) gbest[s * D + j] = pbest[im * D + j];
    }
    for (int j = 0; j < D; ++j) {
      const double g = gbest[s * D + j];
      if (hist_row) hist_row[s * (D + 1) + j] = g;
      if (theta_star) theta_star[s * D + j] = box.lg[j] ? pow(10.0, g) : g;
    }
    if (hist_row) hist_row[s * (D + 1) + D] = gJ;
    if (J_star) J_star[s] = gJ;
  }
}

// Sharded swarm: this process's best candidate of every local
// trace, in a form that can be exchanged: row s = { pbestJ, global particle
// index (exact in a double below 2^53), pbest x[D] }.  With the ring topology the
// row also carries the personal bests of the shard's first and last particle,
// { pbestJ, pbest x[D] } each, which are the ring neighbours of the adjacent
// shards: 3 D + 4 doubles.
__global__ void pso_shard_cand_kernel(int D, int n_cand, int64_t first, int64_t per,
                                      int ring, const Cand* __restrict__ cand,
                                      const double* __restrict__ pbest,
                                      const double* __restrict__ pbestJ,
                                      double* __restrict__ cand_out) {
  __shared__ Cand red[32];
  const int s = blockIdx.x;
  double Jm = CUDART_INF;
  long long im = 0x7fffffffffffffffLL;
  for (int c = threadIdx.x; c < n_cand; c += blockDim.x) {
    const Cand cd = cand[(int64_t)s * n_cand + c];
    if (cand_less(cd.J, cd.idx, Jm, im)) {
      Jm = cd.J;
      im = cd.idx;
    }
  }
  block_argmin(Jm, im, red);
  if (threadIdx.x == 0) {
    const int width = ring ? 3 * D + 4 : D + 2;
    double* r = cand_out + (int64_t)s * width;
    r[0] = Jm;
    r[1] = (double)(first + im);
    for (int j = 0; j < D; ++j) r[2 + j] = pbest[im * D + j];
    if (ring) {
      const int64_t p0 = (int64_t)s * per, p1 = p0 + per - 1;
      double* e = r + D + 2;
      e[0] = pbestJ[p0];
      for (int j = 0; j < D; ++j) e[1 + j] = pbest[p0 * D + j];
      e += D + 1;
      e[0] = pbestJ[p1];
      for (int j = 0; j < D; ++j) e[1 + j] = pbest[p1 * D + j];
    }
  }
}

// Global best of every local trace from the candidates of all ranks
// (gathered [n_ranks][n_traces][D+2]): lowest global index among the minima,
// taken only on a strict improvement -- the rule of pso_gbest_kernel.
__global__ void pso_shard_gbest_kernel(BoxDev box, int D, int n_traces,
                                       int n_ranks, int width,
                                       const double* __restrict__ gathered,
                                       double* __restrict__ gbest,
                                       double* __restrict__ gbestJ,
                                       double* __restrict__ theta_star,
                                       double* __restrict__ J_star) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_traces) return;
  double Jm = CUDART_INF;
  long long im = 0x7fffffffffffffffLL;
  int rm = -1;
  for (int r = 0; r < n_ranks; ++r) {
    const double* row = gathered + ((int64_t)r * n_traces + s) * width;
    const long long idx = (long long)row[1];
    if (cand_less(row[0], idx, Jm, im)) {
      Jm = row[0];
      im = idx;
      rm = r;
    }
  }
  double gJ = gbestJ[s];
  if (rm >= 0 && Jm < gJ) {
    gJ = Jm;
    gbestJ[s] = Jm;
    const double* row = gathered + ((int64_t)rm * n_traces + s) * width;
    for (int j = 0; j < D; ++j) gbest[s * D + j] = row[2 + j];
  }
  for (int j = 0; j < D; ++j) {
    const double g = gbest[s * D + j];
    if (theta_star) theta_star[s * D + j] = box.lg[j] ? pow(10.0, g) : g;
  }
  if (J_star) J_star[s] = gJ;
}

// Optional dump, then Eq. 8, x <- x + v, clamp + zero velocity, for
// the particles [off, off + cnt) of every (local) swarm.
// Ring of three (R23): the social attractor is the best personal best among the
// in-swarm indices g - 1, g, g + 1 (mod the swarm size rg.total), g = rg.off +
// local index; a neighbour outside this shard is the last particle of the shard
// before (row rg.left) or the first particle of the shard after (row rg.right),
// { pbestJ, pbest x[D] } per trace, rg.stride doubles apart.
struct RingShard {
  int64_t total;        // particles of the whole swarm (all shards)
  int64_t off;          // in-swarm index of this shard's local particle 0
  const double* left;   // neighbour rows of trace 0, or nullptr (whole swarm here)
  const double* right;
  int64_t stride;
};

__global__ void pso_move_kernel(BoxDev box, SwarmDev sw, int D, int64_t per,
                                int64_t off, int64_t cnt, int n_traces,
                                uint64_t seed, int64_t first, uint32_t it,
                                int do_move, RingShard rg,
                                const double* __restrict__ J,
                                double* __restrict__ x, double* __restrict__ v,
                                const double* __restrict__ pbest,
                                const double* __restrict__ pbestJ,
                                const double* __restrict__ gbest,
                                double* __restrict__ dump_row) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cnt * n_traces) return;
  const int64_t s = i / cnt;
  const int64_t p = off + (i - s * cnt);  // local index inside the (local) swarm
  const int64_t gp = s * per + p;
  AFM_CHECK(p < per && s < n_traces);
  double xi[4], vi[4], pb[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (j < D) {
      xi[j] = x[gp * D + j];
      vi[j] = v[gp * D + j];
      pb[j] = pbest[gp * D + j];
    }
  }
  if (dump_row) {
    double* r = dump_row + gp * (3 * D + 2);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (j < D) {
        r[j] = xi[j];
        r[D + j] = vi[j];
        r[2 * D + j] = pb[j];
      }
    }
    r[3 * D] = J[gp];
    r[3 * D + 1] = pbestJ[gp];
  }
  if (!do_move) return;
  double r1[4], r2[4];
  pso_uniforms(seed, (uint64_t)(first + gp), it, 1u, D, r1, r2);
  const double* social = gbest + s * D;
  if (sw.topology == 1) {
    const int64_t g = rg.off + p;
    const int64_t gl = (g + rg.total - 1) % rg.total, gr = (g + 1) % rg.total;
    // personal best (J, position) of in-swarm index c
    auto best_of = [&](int64_t c, double& Jc) -> const double* {
      const int64_t lc = c - rg.off;
      if (lc >= 0 && lc < per) {
        Jc = pbestJ[s * per + lc];
        return pbest + (s * per + lc) * D;
      }
      AFM_CHECK(rg.left != nullptr && rg.right != nullptr);
      const double* row = (c == gl ? rg.left : rg.right) + s * rg.stride;
      Jc = row[0];
      return row + 1;
    };
    double Jb, J1, J2;
    const double* xb = best_of(gl, Jb);
    int64_t best = gl;
    const double* x1 = best_of(g, J1);
    if (J1 < Jb || (J1 == Jb && g < best)) {
      best = g;
      Jb = J1;
      xb = x1;
    }
    const double* x2 = best_of(gr, J2);
    if (J2 < Jb || (J2 == Jb && gr < best)) xb = x2;
    social = xb;
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (j < D) {
      const double gb = social[j];
      const double t0 = __dmul_rn(sw.w, vi[j]);
      const double t1 =
          __dmul_rn(__dmul_rn(sw.c1, r1[j]), __dsub_rn(pb[j], xi[j]));
      const double t2 =
          __dmul_rn(__dmul_rn(sw.c2, r2[j]), __dsub_rn(gb, xi[j]));
      double vn = __dadd_rn(__dadd_rn(t0, t1), t2);
      double xn = __dadd_rn(xi[j], vn);
      if (xn < box.lo[j]) {
        xn = box.lo[j];
        vn = 0.0;
      }
      if (xn > box.hi[j]) {
        xn = box.hi[j];
        vn = 0.0;
      }
      x[gp * D + j] = xn;
      v[gp * D + j] = vn;
    }
  }
}

// ============================================================================
// launchers
// ============================================================================
int blocks_per_trace(int64_t per, int block) {
  return (int)((per + block - 1) / block);
}

int launch_build_stream(const ModelConsts& mc, const double* trace, int n_traces,
                        double* stream, cudaStream_t st) {
  int64_t total = (int64_t)n_traces * mc.N;
  int threads = 256;
  int64_t blocks = (total + threads - 1) / threads;
  build_stream_kernel<<<(unsigned)blocks, threads, 0, st>>>(mc, trace, n_traces,
                                                           stream);
  return 1;
}

template <int LAW, int MODE, int PPT, bool LAT>
static int launch_integrate_t(const ModelConsts& mc, const IntegrateIO& io,
                              int block, cudaStream_t st) {
  const int bpt = LAT ? blocks_per_trace(io.per, io.lanes)
                      : blocks_per_trace(io.per, block * PPT);
  if (LAT) block = 32;  // one warp per CTA
  const unsigned grid = (unsigned)(bpt * io.n_traces);
  const size_t smem = (size_t)(mc.T + kPadRows) * 32 * 2 + 64;  // two stages + pad rows + barriers
  auto kern = integrate_misfit_f64<LAW, MODE, PPT, LAT>;
  if (smem > 48 * 1024)
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem);
  kern<<<grid, block, smem, st>>>(mc, io, bpt);
  return 1;
}

// variant: 0 = throughput form, 1 = latency form (short dependent chains).
// (Two particles per thread, PPT = 2, was measured and rejected for FP64 -- 28 %
// slower on configs[1], DESIGN.md 6 -- and is no longer instantiated.)
int launch_integrate_f64(const ModelConsts& mc, const IntegrateIO& io, int block,
                         int variant, cudaStream_t st) {
#define AFM_DISPATCH(LAWV)                                                      \
  case LAWV:                                                                    \
    if (variant == 1)                                                           \
      return io.mode ? launch_integrate_t<LAWV, 1, 1, true>(mc, io, block, st)  \
                     : launch_integrate_t<LAWV, 0, 1, true>(mc, io, block, st); \
    return io.mode ? launch_integrate_t<LAWV, 1, 1, false>(mc, io, block, st)   \
                   : launch_integrate_t<LAWV, 0, 1, false>(mc, io, block, st);
  switch (mc.law) {
    AFM_DISPATCH(AFM_LAW_NONE)
    AFM_DISPATCH(AFM_LAW_DMT)
    AFM_DISPATCH(AFM_LAW_DMT_VISC)
    AFM_DISPATCH(AFM_LAW_LJ_EXP)
    AFM_DISPATCH(AFM_LAW_HOOKE)
    AFM_DISPATCH(AFM_LAW_KELVIN_VOIGT)
    default:
      return -1;
  }
#undef AFM_DISPATCH
}

int launch_segq_init(const SegQueue& q, cudaStream_t st) {
  const int n_init = q.n_tasks > q.n_park ? q.n_tasks : q.n_park;
  segq_init_kernel<<<(unsigned)((n_init + 255) / 256), 256, 0, st>>>(q);
  return 1;
}

template <int LAW, int MODE>
static int launch_integrate_q_t(const ModelConsts& mc, const IntegrateIO& io,
                                const SegQueue& q, int workers, cudaStream_t st) {
  const int bpt = blocks_per_trace(io.per, 32);
  const size_t smem = (size_t)(mc.T + kPadRows) * 32 * 2 + 64;
  auto kern = integrate_misfit_f64_q<LAW, MODE>;
  if (smem > 48 * 1024)
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  kern<<<(unsigned)workers, 32, smem, st>>>(mc, io, bpt, q);
  return 1;
}

// Segment-queue form of the throughput kernel (one warp per CTA, `workers`
// persistent CTAs); q.n_chains must be blocks_per_trace(io.per, 32) * n_traces.
// The caller resets the queue first (launch_segq_init on the same stream).
int launch_integrate_f64_q(const ModelConsts& mc, const IntegrateIO& io,
                           const SegQueue& q, int workers, cudaStream_t st) {
#define AFM_DISPATCH_Q(LAWV)                                                   \
  case LAWV:                                                                   \
    return io.mode ? launch_integrate_q_t<LAWV, 1>(mc, io, q, workers, st)     \
                   : launch_integrate_q_t<LAWV, 0>(mc, io, q, workers, st);
  switch (mc.law) {
    AFM_DISPATCH_Q(AFM_LAW_NONE)
    AFM_DISPATCH_Q(AFM_LAW_DMT)
    AFM_DISPATCH_Q(AFM_LAW_DMT_VISC)
    AFM_DISPATCH_Q(AFM_LAW_LJ_EXP)
    AFM_DISPATCH_Q(AFM_LAW_HOOKE)
    AFM_DISPATCH_Q(AFM_LAW_KELVIN_VOIGT)
    default:
      return -1;
  }
#undef AFM_DISPATCH_Q
}

int launch_trajectory(const ModelConsts& mc, const double* theta_dev,
                      const double* stream, double z0, double v0, double* zs,
                      double* vs, cudaStream_t st) {
  switch (mc.law) {
    case AFM_LAW_NONE:
      trajectory_kernel<AFM_LAW_NONE>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    case AFM_LAW_DMT:
      trajectory_kernel<AFM_LAW_DMT>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    case AFM_LAW_DMT_VISC:
      trajectory_kernel<AFM_LAW_DMT_VISC>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    case AFM_LAW_LJ_EXP:
      trajectory_kernel<AFM_LAW_LJ_EXP>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    case AFM_LAW_HOOKE:
      trajectory_kernel<AFM_LAW_HOOKE>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    case AFM_LAW_KELVIN_VOIGT:
      trajectory_kernel<AFM_LAW_KELVIN_VOIGT>
          <<<1, 32, 0, st>>>(mc, theta_dev, stream, z0, v0, zs, vs);
      break;
    default:
      return -1;
  }
  return 1;
}

int launch_pso_init(const BoxDev& box, int D, int64_t per, int n_traces,
                    uint64_t seed, int64_t first, double* x, double* v,
                    double* pbest,
                    double* pbestJ, double* gbest, double* gbestJ,
                    cudaStream_t st) {
  const int64_t PT = per * n_traces;
  const int threads = 128;
  pso_init_kernel<<<(unsigned)((PT + threads - 1) / threads), threads, 0, st>>>(
      box, D, per, n_traces, seed, first, x, v, pbest, pbestJ, gbest, gbestJ);
  return 1;
}

int launch_pso_best(int D, int64_t per, int64_t off, int64_t cnt, int n_traces,
                    double* J, const double* Jc, const double* x, double* pbest,
                    double* pbestJ, Cand* cand, int block, cudaStream_t st) {
  const int bpt = blocks_per_trace(cnt, block);
  pso_best_kernel<<<(unsigned)(bpt * n_traces), block, 0, st>>>(
      D, per, off, cnt, bpt, J, Jc, x, pbest, pbestJ, cand);
  return 1;
}

int launch_chunk_gather(const BoxDev& box, int D, int64_t per, int64_t off,
                        int64_t cnt, int n_traces, const double* x, double* theta_c,
                        cudaStream_t st) {
  const int threads = 128;
  const int64_t n = cnt * n_traces;
  chunk_gather_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(
      box, D, per, off, cnt, n_traces, x, theta_c);
  return 1;
}

int launch_pso_gbest(const BoxDev& box, int D, int n_traces, int n_cand,
                     const Cand* cand, const double* pbest, double* gbest,
                     double* gbestJ, double* hist_row, double* theta_star,
                     double* J_star, cudaStream_t st) {
  int threads = n_cand <= 32 ? 32 : (n_cand <= 64 ? 64 : 128);
  pso_gbest_kernel<<<(unsigned)n_traces, threads, 0, st>>>(
      box, D, n_cand, cand, pbest, gbest, gbestJ, hist_row, theta_star, J_star);
  return 1;
}

int launch_pso_move(const BoxDev& box, const SwarmDev& sw, int D, int64_t per,
                    int64_t off, int64_t cnt, int n_traces, uint64_t seed,
                    int64_t first, uint32_t it, int do_move, const RingEdges& re,
                    const double* J, double* x, double* v, const double* pbest,
                    const double* pbestJ, const double* gbest, double* dump_row,
                    cudaStream_t st) {
  const int64_t n = cnt * n_traces;
  const int threads = 128;
  RingShard rg;
  rg.total = re.total > 0 ? re.total : per;
  rg.off = re.total > 0 ? re.off : 0;
  rg.left = re.left;
  rg.right = re.right;
  rg.stride = re.stride;
  pso_move_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(
      box, sw, D, per, off, cnt, n_traces, seed, first, it, do_move, rg, J, x, v,
      pbest, pbestJ, gbest, dump_row);
  return 1;
}

int launch_pso_shard_cand(int D, int n_traces, int n_cand, int64_t first,
                          int64_t per, int ring, const Cand* cand,
                          const double* pbest, const double* pbestJ,
                          double* cand_out, cudaStream_t st) {
  int threads = n_cand <= 32 ? 32 : (n_cand <= 64 ? 64 : 128);
  pso_shard_cand_kernel<<<(unsigned)n_traces, threads, 0, st>>>(
      D, n_cand, first, per, ring, cand, pbest, pbestJ, cand_out);
  return 1;
}

int launch_pso_shard_gbest(const BoxDev& box, int D, int n_traces, int n_ranks,
                           int width, const double* gathered, double* gbest,
                           double* gbestJ, double* theta_star, double* J_star,
                           cudaStream_t st) {
  const int threads = 64;
  pso_shard_gbest_kernel<<<(unsigned)((n_traces + threads - 1) / threads),
                           threads, 0, st>>>(box, D, n_traces, n_ranks, width,
                                             gathered, gbest, gbestJ, theta_star,
                                             J_star);
  return 1;
}

int launch_philox(const uint32_t* ctr, int64_t n, uint32_t k0, uint32_t k1,
                  uint32_t* out, cudaStream_t st) {
  const int threads = 128;
  philox_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(
      ctr, n, k0, k1, out);
  return 1;
}

}  // namespace afm
