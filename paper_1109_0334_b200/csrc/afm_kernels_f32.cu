// afm_kernels_f32.cu -- FP32 variant of the integrate-and-misfit kernel
// (north_star "an FP64 and an FP32 variant"; R14, section 6).
//
//   build_stream_f32_kernel   time-tile stream in kernel units, 16 B per step:
//                             { s6(t_n + h/2), s6(t_n + h), U_n + z_c, e_w }
//   integrate_misfit_f32      a1-a5 of SURVEY.md 8(a) with FP32 stage arithmetic
//                             and a two-float compensated state
//
// Inputs and outputs at the kernel boundary stay FP64/SI (params, z0v0, misfit,
// PSO state); only the time loop runs in FP32.
#include <math_constants.h>

#include "afm_device_common.cuh"
#include "afm_device_f32.cuh"
#include "afm_internal.h"

namespace afm {

constexpr int kPadRows = kPadBytes / 16;  // pad rows after each stage of the tile ring

// s6(t) = (beta/6) (F0/k) cos(w t) + (beta/6) z_c  [nm per step^2 / 6], FP64.
__device__ __forceinline__ double s6_of(const ModelConstsF32& mf, double t) {
  return fma(mf.drive6, cos(__dmul_rn(mf.w_drive, t)), mf.b6_zc);
}

// Row n of trace s.  The abscissae are t_n = n h, t_n + h/2 and t_{n+1} =
// (n + 1) h, so that s1 of row n is bit-identical to s0 of row n + 1 (the
// kernel carries it over instead of storing it twice).  e_w is the rounding
// residual of the stream values this step uses: exact (s0 + 4 sh + s1) minus
// the sum of the three floats, added back into the lo part of w.
__global__ void build_stream_f32_kernel(ModelConstsF32 mf,
                                        const double* __restrict__ trace,
                                        int n_traces,
                                        float4* __restrict__ stream) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = (int64_t)n_traces * mf.N;
  if (i >= total) return;
  const int s = (int)(i / mf.N);
  const int n = (int)(i - (int64_t)s * mf.N);
  const double t0 = __dmul_rn((double)n, mf.h);
  const double th = __dadd_rn(t0, __dmul_rn(0.5, mf.h));
  const double t1 = __dmul_rn((double)(n + 1), mf.h);
  const double S0 = s6_of(mf, t0), SH = s6_of(mf, th), S1 = s6_of(mf, t1);
  const float s0f = (float)S0, shf = (float)SH, s1f = (float)S1;
  const double used = (double)s0f + 4.0 * (double)shf + (double)s1f;
  float4 row;
  row.x = shf;
  row.y = s1f;
  row.z = (n >= mf.n0)
              ? (float)(trace[(int64_t)s * mf.W + (n - mf.n0)] / mf.len + mf.zc)
              : 0.0f;
  row.w = (float)((S0 + 4.0 * SH + S1) - used);
  stream[i] = row;
}

// Steps [i0, i1) of one time tile, with (WIN) or without the misfit sum.
template <int LAW, int PPT, bool WIN>
__device__ __forceinline__ void run_steps32(const float4* sp, int i0, int i1,
                                            const Model32& M,
                                            const Particle32 (&P)[PPT],
                                            State32 (&S)[PPT], float (&Jt)[PPT],
                                            bool (&bad)[PPT], int& mode,
                                            float& s_prev) {
  if (i0 >= i1) return;
  AFM_CHECK(i0 >= 0);
  float4 r = sp[i0];
#pragma unroll 2
  for (int i = i0; i < i1; ++i) {
    const float4 rn = sp[i + 1];  // one step ahead; past the tile: the pad row
    rk4_step32<LAW, PPT>(M, P, s_prev, r.x, r.y, r.w, S, mode, bad);
    if (WIN) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) {
        const float res = __fadd_rn(__fsub_rn(S[q].dh, r.z), S[q].dl);
        Jt[q] = fmaf(res, res, Jt[q]);
      }
    }
    s_prev = r.y;
    r = rn;
  }
}

template <int LAW, int MODE, int PPT>
__global__ void integrate_misfit_f32(ModelConstsF32 mf, IntegrateIO io,
                                     int blocks_per_tr) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* tile0 = reinterpret_cast<float4*>(smem_raw);
  float4* tile1 = tile0 + (mf.T + kPadRows);  // one pad row per stage for the row fetched ahead
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (mf.T + kPadRows));
  __shared__ Cand red[32];

  const int tid = threadIdx.x;
  const int s = blockIdx.x / blocks_per_tr;
  const int64_t base =
      (int64_t)(blockIdx.x - s * blocks_per_tr) * blockDim.x * PPT + tid;
  bool active[PPT];
  int64_t gp[PPT];
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    const int64_t li = base + (int64_t)q * blockDim.x;
    active[q] = li < io.per;
    gp[q] = (int64_t)s * io.per + (active[q] ? li : io.per - 1);
    AFM_CHECK(s < io.n_traces && gp[q] >= 0 && gp[q] < io.per * io.n_traces);
  }

  const float4* stream =
      reinterpret_cast<const float4*>(io.stream) + (int64_t)s * mf.N;

  if (tid == 0) {
    tile0[mf.T] = make_float4(0.f, 0.f, 0.f, 0.f);
    tile1[mf.T] = make_float4(0.f, 0.f, 0.f, 0.f);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int st = 0; st < 2; ++st) {
      if (st < mf.n_tiles) {
        const int n_begin = st * mf.T;
        const uint32_t bytes = (uint32_t)min(mf.T, mf.N - n_begin) * 16u;
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + n_begin, bytes, &bars[st]);
      }
    }
  }

  // ---- a1: parameter map (FP64, then rounded once) --------------------------
  Model32 M;
  {
    const float a6f = (float)mf.a6, b6f = (float)mf.b6;
    M.nalpha = -a6f;
    M.nbeta = -b6f;
    M.nalpha_lo = -(float)(mf.a6 - (double)a6f);
    M.nbeta_lo = -(float)(mf.b6 - (double)b6f);
    M.a0 = (float)mf.a0;
    M.d_safe = (float)mf.d_safe;
    M.d_max = (float)mf.d_max;
    M.d_min = (float)mf.d_min;
  }
  double xloc[PPT][4];
  Particle32 P[PPT];
  State32 S[PPT];
  float Jt[PPT], Jh[PPT], Jl[PPT];
  bool bad[PPT];
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    double th[4] = {0.0, 0.0, 0.0, 1.0};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      xloc[q][j] = 0.0;
      if (j < mf.D) {
        const double xv = io.params[gp[q] * mf.D + j];
        xloc[q][j] = xv;
        th[j] = (MODE == 1 && io.box.lg[j]) ? pow(10.0, xv) : xv;
      }
    }
    P[q].c0 = P[q].c1 = P[q].c2 = P[q].c3 = P[q].thr = 0.0f;
    if (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) {
      const double kappa = th[0] * mf.c_vdw;
      P[q].c0 = (float)(-kappa);
      P[q].c1 = (float)(th[1] * mf.c_hertz);
      P[q].c2 = (float)(-kappa / (mf.a0 * mf.a0));
      if (LAW == AFM_LAW_DMT_VISC) P[q].c3 = (float)(-(th[2] * mf.c_visc));
    } else if (LAW == AFM_LAW_LJ_EXP) {
      P[q].c0 = (float)(th[0] * mf.c_rep);
      P[q].c1 = (float)(-(th[1] * mf.c_att));
      P[q].c2 = (float)(-(th[2] * mf.c_fad));
      P[q].c3 = (float)(-mf.c_lam / th[3]);
    } else if (LAW == AFM_LAW_HOOKE) {
      P[q].c1 = (float)(th[0] * mf.c_ks);
      P[q].thr = (float)(mf.zc - th[1] / mf.len);
    } else if (LAW == AFM_LAW_KELVIN_VOIGT) {
      P[q].c1 = (float)(th[0] * mf.c_ks);
      P[q].c3 = (float)(-mf.a6 - th[1] * mf.c_zeta);
    }
    double z0 = mf.z0, v0 = mf.v0;
    if (io.z0v0 != nullptr) {
      z0 = io.z0v0[2 * gp[q]];
      v0 = io.z0v0[2 * gp[q] + 1];
    }
    const double d0 = z0 / mf.len + mf.zc;
    const double w0 = v0 * mf.h / mf.len;
    S[q].dh = (float)d0;
    S[q].dl = (float)(d0 - (double)S[q].dh);
    S[q].wh = (float)w0;
    S[q].wl = (float)(w0 - (double)S[q].wh);
    Jt[q] = Jh[q] = Jl[q] = 0.0f;
    bad[q] = false;
  }
  int mode = 0;
  float s_prev = (float)(mf.drive6 + mf.b6_zc);  // s6(0): cos(0) = 1

  // ---- a2-a4: RK4 over the time tiles ---------------------------------------
  for (int tile = 0; tile < mf.n_tiles; ++tile) {
    const int st = tile & 1;
    const float4* sp = st ? tile1 : tile0;
    mbar_wait(&bars[st], (uint32_t)((tile >> 1) & 1));
    const int n_begin = tile * mf.T;
    const int n_steps = min(mf.T, mf.N - n_begin);
    AFM_CHECK(n_steps >= 1 && n_steps <= mf.T && n_begin + n_steps <= mf.N);
    const int k0 = max(0, min(n_steps, mf.n0 - n_begin));
    run_steps32<LAW, PPT, false>(sp, 0, k0, M, P, S, Jt, bad, mode, s_prev);
    run_steps32<LAW, PPT, true>(sp, k0, n_steps, M, P, S, Jt, bad, mode, s_prev);
    // fold the tile's partial sum into the two-float total
#pragma unroll
    for (int q = 0; q < PPT; ++q) {
      float e;
      two_sum32(Jh[q], Jt[q], Jh[q], e);
      Jl[q] = __fadd_rn(Jl[q], e);
      Jt[q] = 0.0f;
    }
    __syncthreads();
    if (tid == 0 && tile + 2 < mf.n_tiles) {
      const int nb = (tile + 2) * mf.T;
      const uint32_t bytes = (uint32_t)min(mf.T, mf.N - nb) * 16u;
      fence_proxy_async();
      mbar_arrive_expect_tx(&bars[st], bytes);
      bulk_g2s(st ? tile1 : tile0, stream + nb, bytes, &bars[st]);
    }
  }

  double pb = CUDART_INF;
  long long idx = 0x7fffffffffffffffLL;
  const double to_si = mf.len * mf.len;
#pragma unroll
  for (int q = 0; q < PPT; ++q) {
    double J = ((double)Jh[q] + (double)Jl[q]) * to_si;
    bad[q] |= !(fabsf(S[q].wh) <= 3.0e38f);  // last velocity finite too (R12)
    if (bad[q] || !(J == J)) J = CUDART_INF;
    if (active[q]) io.J[gp[q]] = J;
    if (MODE == 1 && active[q]) {
      double pq = io.pbestJ[gp[q]];
      if (J < pq) {
        pq = J;
        io.pbestJ[gp[q]] = J;
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (j < mf.D) io.pbest[gp[q] * mf.D + j] = xloc[q][j];
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
// Segment-queue form (see integrate_misfit_f64_q in afm_kernels.cu): persistent
// one-warp workers take (chain, segment) tasks; between segments a chain rests as
// { d hi, d lo, w hi, w lo, J hi, J lo, diverged } (the per-tile partial sum is
// folded at every tile end, and the carried stream value s_prev is re-read from
// the row before the segment).  Same arithmetic per particle as
// integrate_misfit_f32<LAW, MODE, 1>: bit-identical results.
// ============================================================================
template <int LAW, int MODE>
__global__ void __launch_bounds__(32)
integrate_misfit_f32_q(ModelConstsF32 mf, IntegrateIO io, int blocks_per_tr, SegQueue q) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* tile0 = reinterpret_cast<float4*>(smem_raw);
  float4* tile1 = tile0 + (mf.T + kPadRows);  // one pad row per stage for the row fetched ahead
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (mf.T + kPadRows));
  __shared__ Cand red[32];
  __shared__ SegqWorker qworker;  // lane 0's queue state (one warp per CTA)

  const int tid = threadIdx.x;
  if (tid == 0) {
    qworker.offered = 0u;
    tile0[mf.T] = make_float4(0.f, 0.f, 0.f, 0.f);
    tile1[mf.T] = make_float4(0.f, 0.f, 0.f, 0.f);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t n_wait0 = 0u, n_wait1 = 0u;

  Model32 M;
  {
    const float a6f = (float)mf.a6, b6f = (float)mf.b6;
    M.nalpha = -a6f;
    M.nbeta = -b6f;
    M.nalpha_lo = -(float)(mf.a6 - (double)a6f);
    M.nbeta_lo = -(float)(mf.b6 - (double)b6f);
    M.a0 = (float)mf.a0;
    M.d_safe = (float)mf.d_safe;
    M.d_max = (float)mf.d_max;
    M.d_min = (float)mf.d_min;
  }

  for (;;) {
    int task = 0;
    if (tid == 0) task = segq_pop(q, &qworker);
    task = __shfl_sync(0xffffffffu, task, 0);
    if (task < 0) break;
    const int chain = task & 0xfffff;
    const int seg = task >> 20;
    const int s = chain / blocks_per_tr;
    const int64_t li = (int64_t)(chain - s * blocks_per_tr) * 32 + tid;
    const bool active = li < io.per;
    const int64_t gp = (int64_t)s * io.per + (active ? li : io.per - 1);
    const float4* stream = reinterpret_cast<const float4*>(io.stream) + (int64_t)s * mf.N;
    const int tile_begin = seg * q.tiles_per_seg;
    const int tile_end = min(tile_begin + q.tiles_per_seg, mf.n_tiles);

    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const int tile = tile_begin + k;
        if (tile < tile_end) {
          const int st = tile & 1;
          const int nb = tile * mf.T;
          const uint32_t bytes = (uint32_t)min(mf.T, mf.N - nb) * 16u;
          fence_proxy_async();
          mbar_arrive_expect_tx(&bars[st], bytes);
          bulk_g2s(st ? tile1 : tile0, stream + nb, bytes, &bars[st]);
        }
      }
    }

    double xloc[4];
    Particle32 P[1];
    State32 S[1];
    float Jt[1], Jh, Jl, s_prev;
    bool bad[1];
    {
      double th[4] = {0.0, 0.0, 0.0, 1.0};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        xloc[j] = 0.0;
        if (j < mf.D) {
          const double xv = io.params[gp * mf.D + j];
          xloc[j] = xv;
          th[j] = (MODE == 1 && io.box.lg[j]) ? pow(10.0, xv) : xv;
        }
      }
      P[0].c0 = P[0].c1 = P[0].c2 = P[0].c3 = P[0].thr = 0.0f;
      if (LAW == AFM_LAW_DMT || LAW == AFM_LAW_DMT_VISC) {
        const double kappa = th[0] * mf.c_vdw;
        P[0].c0 = (float)(-kappa);
        P[0].c1 = (float)(th[1] * mf.c_hertz);
        P[0].c2 = (float)(-kappa / (mf.a0 * mf.a0));
        if (LAW == AFM_LAW_DMT_VISC) P[0].c3 = (float)(-(th[2] * mf.c_visc));
      } else if (LAW == AFM_LAW_LJ_EXP) {
        P[0].c0 = (float)(th[0] * mf.c_rep);
        P[0].c1 = (float)(-(th[1] * mf.c_att));
        P[0].c2 = (float)(-(th[2] * mf.c_fad));
        P[0].c3 = (float)(-mf.c_lam / th[3]);
      } else if (LAW == AFM_LAW_HOOKE) {
        P[0].c1 = (float)(th[0] * mf.c_ks);
        P[0].thr = (float)(mf.zc - th[1] / mf.len);
      } else if (LAW == AFM_LAW_KELVIN_VOIGT) {
        P[0].c1 = (float)(th[0] * mf.c_ks);
        P[0].c3 = (float)(-mf.a6 - th[1] * mf.c_zeta);
      }
    }
    float* ck = reinterpret_cast<float*>(q.ckpt) + (int64_t)chain * 256 + tid;
    if (seg == 0) {
      double z0 = mf.z0, v0 = mf.v0;
      if (io.z0v0 != nullptr) {
        z0 = io.z0v0[2 * gp];
        v0 = io.z0v0[2 * gp + 1];
      }
      const double d0 = z0 / mf.len + mf.zc;
      const double w0 = v0 * mf.h / mf.len;
      S[0].dh = (float)d0;
      S[0].dl = (float)(d0 - (double)S[0].dh);
      S[0].wh = (float)w0;
      S[0].wl = (float)(w0 - (double)S[0].wh);
      Jh = Jl = 0.0f;
      bad[0] = false;
      s_prev = (float)(mf.drive6 + mf.b6_zc);  // s6(0): cos(0) = 1
    } else {
      S[0].dh = __ldcg(ck);
      S[0].dl = __ldcg(ck + 32);
      S[0].wh = __ldcg(ck + 64);
      S[0].wl = __ldcg(ck + 96);
      Jh = __ldcg(ck + 128);
      Jl = __ldcg(ck + 160);
      bad[0] = __ldcg(ck + 192) != 0.0f;
      AFM_CHECK(tile_begin >= 1);
      s_prev = stream[tile_begin * mf.T - 1].y;  // s1 of the step before this segment
    }
    Jt[0] = 0.0f;
    int mode = 0;

    for (int tile = tile_begin; tile < tile_end; ++tile) {
      const int st = tile & 1;
      const float4* sp = st ? tile1 : tile0;
      mbar_wait(&bars[st], (st ? n_wait1 : n_wait0) & 1u);
      if (st) ++n_wait1; else ++n_wait0;
      const int n_begin = tile * mf.T;
      const int n_steps = min(mf.T, mf.N - n_begin);
      AFM_CHECK(n_steps >= 1 && n_steps <= mf.T && n_begin + n_steps <= mf.N);
      AFM_CHECK(tile >= 0 && tile < mf.n_tiles && tile_end <= mf.n_tiles);
      const int k0 = max(0, min(n_steps, mf.n0 - n_begin));
      run_steps32<LAW, 1, false>(sp, 0, k0, M, P, S, Jt, bad, mode, s_prev);
      run_steps32<LAW, 1, true>(sp, k0, n_steps, M, P, S, Jt, bad, mode, s_prev);
      {
        float e;
        two_sum32(Jh, Jt[0], Jh, e);
        Jl = __fadd_rn(Jl, e);
        Jt[0] = 0.0f;
      }
      __syncthreads();
      if (tid == 0 && tile + 2 < tile_end) {
        const int nb = (tile + 2) * mf.T;
        const uint32_t bytes = (uint32_t)min(mf.T, mf.N - nb) * 16u;
        fence_proxy_async();
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + nb, bytes, &bars[st]);
      }
    }

    if (tile_end < mf.n_tiles) {
      __stcg(ck, S[0].dh);
      __stcg(ck + 32, S[0].dl);
      __stcg(ck + 64, S[0].wh);
      __stcg(ck + 96, S[0].wl);
      __stcg(ck + 128, Jh);
      __stcg(ck + 160, Jl);
      __stcg(ck + 192, bad[0] ? 1.0f : 0.0f);
      __threadfence();
      __syncwarp();
      if (tid == 0) segq_push(q, chain, seg + 1);
      continue;
    }

    const double to_si = mf.len * mf.len;
    double J = ((double)Jh + (double)Jl) * to_si;
    bad[0] |= !(fabsf(S[0].wh) <= 3.0e38f);  // last velocity finite too (R12)
    if (bad[0] || !(J == J)) J = CUDART_INF;
    if (active) io.J[gp] = J;
    if (MODE == 1) {
      double pb = CUDART_INF;
      long long idx = 0x7fffffffffffffffLL;
      if (active) {
        double pq = io.pbestJ[gp];
        if (J < pq) {
          pq = J;
          io.pbestJ[gp] = J;
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (j < mf.D) io.pbest[gp * mf.D + j] = xloc[j];
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

// ---- launchers ------------------------------------------------------------------
int launch_build_stream_f32(const ModelConstsF32& mf, const double* trace,
                            int n_traces, float* stream, cudaStream_t st) {
  const int64_t total = (int64_t)n_traces * mf.N;
  const int threads = 256;
  const int64_t blocks = (total + threads - 1) / threads;
  build_stream_f32_kernel<<<(unsigned)blocks, threads, 0, st>>>(
      mf, trace, n_traces, reinterpret_cast<float4*>(stream));
  return 1;
}

template <int LAW, int MODE, int PPT>
static int launch_integrate32_t(const ModelConstsF32& mf, const IntegrateIO& io,
                                int block, cudaStream_t st) {
  const int bpt = blocks_per_trace(io.per, block * PPT);
  const unsigned grid = (unsigned)(bpt * io.n_traces);
  const size_t smem = (size_t)(mf.T + kPadRows) * 16 * 2 + 64;
  auto kern = integrate_misfit_f32<LAW, MODE, PPT>;
  if (smem > 48 * 1024)
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem);
  kern<<<grid, block, smem, st>>>(mf, io, bpt);
  return 1;
}

int launch_integrate_f32(const ModelConstsF32& mf, const IntegrateIO& io,
                         int block, int ppt, cudaStream_t st) {
#define AFM_DISPATCH32(LAWV)                                                    \
  case LAWV:                                                                    \
    if (ppt == 2)                                                               \
      return io.mode ? launch_integrate32_t<LAWV, 1, 2>(mf, io, block, st)      \
                     : launch_integrate32_t<LAWV, 0, 2>(mf, io, block, st);     \
    return io.mode ? launch_integrate32_t<LAWV, 1, 1>(mf, io, block, st)        \
                   : launch_integrate32_t<LAWV, 0, 1>(mf, io, block, st);
  switch (mf.law) {
    AFM_DISPATCH32(AFM_LAW_NONE)
    AFM_DISPATCH32(AFM_LAW_DMT)
    AFM_DISPATCH32(AFM_LAW_DMT_VISC)
    AFM_DISPATCH32(AFM_LAW_LJ_EXP)
    AFM_DISPATCH32(AFM_LAW_HOOKE)
    AFM_DISPATCH32(AFM_LAW_KELVIN_VOIGT)
    default:
      return -1;
  }
#undef AFM_DISPATCH32
}

template <int LAW, int MODE>
static int launch_integrate32_q_t(const ModelConstsF32& mf, const IntegrateIO& io,
                                  const SegQueue& q, int workers, cudaStream_t st) {
  const int bpt = blocks_per_trace(io.per, 32);
  const size_t smem = (size_t)(mf.T + kPadRows) * 16 * 2 + 64;
  auto kern = integrate_misfit_f32_q<LAW, MODE>;
  if (smem > 48 * 1024)
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  kern<<<(unsigned)workers, 32, smem, st>>>(mf, io, bpt, q);  // queue reset by the caller
  return 1;
}

int launch_integrate_f32_q(const ModelConstsF32& mf, const IntegrateIO& io,
                           const SegQueue& q, int workers, cudaStream_t st) {
#define AFM_DISPATCH32_Q(LAWV)                                                 \
  case LAWV:                                                                   \
    return io.mode ? launch_integrate32_q_t<LAWV, 1>(mf, io, q, workers, st)   \
                   : launch_integrate32_q_t<LAWV, 0>(mf, io, q, workers, st);
  switch (mf.law) {
    AFM_DISPATCH32_Q(AFM_LAW_NONE)
    AFM_DISPATCH32_Q(AFM_LAW_DMT)
    AFM_DISPATCH32_Q(AFM_LAW_DMT_VISC)
    AFM_DISPATCH32_Q(AFM_LAW_LJ_EXP)
    AFM_DISPATCH32_Q(AFM_LAW_HOOKE)
    AFM_DISPATCH32_Q(AFM_LAW_KELVIN_VOIGT)
    default:
      return -1;
  }
#undef AFM_DISPATCH32_Q
}

}  // namespace afm
