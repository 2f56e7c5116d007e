// afm_beam.cu -- the paper's own forward model on sm_100a: the multi-mode
// Euler-Bernoulli cantilever (Eq. 1-2; 128-139 Eq. 6-7, Newton +
// Simpson initialisation, RK4; Appendix A/B).
//
//   beam_setup_kernel     initialisation: roots of
//                         cos(bL)cosh(bL) + 1 = 0 by Newton, mode shapes by
//                         Eq. 6-7, <Phi,Phi> and <1,Phi> by Simpson's rule
//   beam_integrate_f64    one thread per particle, all 2M modal states in
//                         registers, the same TMA-staged time-tile ring and PSO
//                         epilogue as integrate_misfit_f64
//
// Variables (per-step, tip-weighted): a_i = Phi_i(L) eta_i [m], b_i = h Phi_i(L)
// eta_i' [m per step], so the tip deflection is u = sum a_i, the tip travel per
// step w = sum b_i, and
//     b_i' = Gamma_i cos(w t) - alpha_i b_i - beta_i a_i + kappa_i fhat(u+z_c, w)
// with fhat = (h^2/m_1) F_ts, m_1 the first mode's effective mass (kappa_0 = 1):
// the tip-force arithmetic is that of the point-mass kernel.
#include <math_constants.h>

#include "afm_device.cuh"
#include "afm_internal.h"

namespace afm {

constexpr int kPadRows = kPadBytes / 32;  // pad rows after each stage of the tile ring

// ---- initialisation -------------------------------------------------------------
// Eq. 7 with "+ exp(-2 beta L)" in the denominator (R22).
__device__ __forceinline__ double beam_G(double bL) {
  const double e1 = exp(-bL), e2 = exp(-2.0 * bL);
  return (2.0 * e1 * sin(bL) - e2 + 1.0) / (2.0 * e1 * cos(bL) + e2 + 1.0);
}
// Eq. 6.
__device__ __forceinline__ double beam_phi(double b, double G, double x) {
  return 0.5 * (2.0 * sin(b * x) - 2.0 * G * cos(b * x) + (G - 1.0) * exp(b * x) +
                (G + 1.0) * exp(-b * x));
}

// One thread per mode (the paper does this serially at start-up; it is 8 x 501
// evaluations).  Thread 0 then scales the tip compliances by the first mode's.
__global__ void beam_setup_kernel(afm_beam_cfg cfg, double h,
                                  BeamModeConsts* __restrict__ out) {
  __shared__ double compl_sh[8];
  const int i = threadIdx.x;
  const double w = 2.0 * CUDART_PI * cfg.f_drive;
  if (i < cfg.n_modes) {
    double x = ((double)i + 0.5) * CUDART_PI;  // Newton on cos x + 1/cosh x
    for (int it = 0; it < 50; ++it) {
      const double ch = cosh(x);
      const double g = cos(x) + 1.0 / ch;
      const double dg = -sin(x) - sinh(x) / (ch * ch);
      const double step = g / dg;
      x -= step;
      if (fabs(step) < 1e-15 * x) break;
    }
    const double bL = x, b = bL / cfg.L, G = beam_G(bL);
    const int n = cfg.n_points;
    const double hx = cfg.L / (double)(n - 1);
    double s1 = 0.0, s2 = 0.0;
    for (int j = 0; j < n; ++j) {  // composite Simpson
      const double f = beam_phi(b, G, (double)j * hx);
      const double wgt = (j == 0 || j == n - 1) ? 1.0 : ((j & 1) ? 4.0 : 2.0);
      s1 += wgt * f;
      s2 += wgt * f * f;
    }
    const double intphi = s1 * hx / 3.0, norm = s2 * hx / 3.0;
    const double phiL = beam_phi(b, G, cfg.L);
    const double omega =
        bL * bL * sqrt(cfg.E * cfg.I / (cfg.mu * cfg.L * cfg.L * cfg.L * cfg.L));
    const double gain = cfg.A_base * w * w * intphi / norm;
    const double compl_ = phiL * phiL / (cfg.mu * norm);
    out->bL[i] = bL;
    out->omega[i] = omega;
    out->phiL[i] = phiL;
    out->part[i] = phiL * intphi / norm;
    out->compl_[i] = compl_;
    out->Gamma[i] = h * h * phiL * gain;
    out->alpha[i] = h * omega / cfg.Q;
    out->beta[i] = (h * omega) * (h * omega);
    compl_sh[i] = compl_;
  }
  __syncthreads();
  if (i < cfg.n_modes) out->kappa[i] = compl_sh[i] / compl_sh[0];
  if (i == 0) out->m1 = 1.0 / compl_sh[0];
}

// ---- tip force in per-step variables ----------------------------------------------
// fhat(d, w) = (h^2/m_1) F_ts; P holds the point-mass kernel's scaled
// coefficients (load_particle with m = m_1).  The law is a run-time switch:
// the force is one evaluation per stage against 8 modes of linear algebra.
__device__ __forceinline__ double tip_force(const Particle64& P, int law,
                                            long long a0_bits, double d,
                                            double w) {
  switch (law) {
    case AFM_LAW_DMT:
    case AFM_LAW_DMT_VISC: {
      if (ge_pos(d, a0_bits)) return P.c0 * rcp_fast(d * d);
      const double del = P.a0 - d;
      const double sq = sqrt_fast(del);
      double f = fma(P.c1 * del, sq, P.c2);
      if (law == AFM_LAW_DMT_VISC) f = fma(P.c3 * sq, w, f);
      return f;
    }
    case AFM_LAW_LJ_EXP: {
      const double r = rcp_fast(d * d);
      const double r2 = r * r;
      return fma(P.c2, exp_fast(d * P.c3), fma(P.c0, r2 * r2, P.c1 * r));
    }
    case AFM_LAW_HOOKE:
    case AFM_LAW_KELVIN_VOIGT: {
      if (!(d < P.a0)) return 0.0;
      double f = P.c1 * (P.a0 - d);
      // P.c3 = -(alpha + nu): only the damper's part -nu w acts here
      if (law == AFM_LAW_KELVIN_VOIGT) f = fma(P.c3 - P.nalpha, w, f);
      return f;
    }
    default:
      return 0.0;
  }
}

// Stage acceleration of every mode: acc_i = Gamma_i c - alpha_i b_i - beta_i a_i
// + kappa_i fhat(sum a + z_c, sum b).
template <int M>
__device__ __forceinline__ void beam_accel(const BeamModeConsts& mo,
                                           const Particle64& P, int law,
                                           long long a0_bits, double zc, double c,
                                           const double (&a)[M],
                                           const double (&b)[M],
                                           double (&acc)[M]) {
  double u = a[0], w = b[0];
#pragma unroll
  for (int i = 1; i < M; ++i) {
    u += a[i];
    w += b[i];
  }
  const double f = tip_force(P, law, a0_bits, u + zc, w);
#pragma unroll
  for (int i = 0; i < M; ++i)
    acc[i] = fma(mo.Gamma[i], c,
                 fma(mo.kappa[i], f, fma(-mo.alpha[i], b[i], -mo.beta[i] * a[i])));
}

// One classical RK4 step of unit length on (a, b); c0, ch, c1 = cos(w t) at the
// three abscissae.  Running sums keep the register count at ~6M doubles.
template <int M>
__device__ __forceinline__ void beam_rk4(const BeamModeConsts& mo,
                                         const Particle64& P, int law,
                                         long long a0_bits, double zc, double c0,
                                         double ch, double c1, double (&a)[M],
                                         double (&b)[M]) {
  const double sixth = 1.0 / 6.0;
  double k[M], as[M], bs[M], sa[M], sb[M];
  beam_accel<M>(mo, P, law, a0_bits, zc, c0, a, b, k);  // k1
#pragma unroll
  for (int i = 0; i < M; ++i) {
    as[i] = fma(0.5, b[i], a[i]);
    bs[i] = fma(0.5, k[i], b[i]);
    sa[i] = k[i];  // k1 + k2 + k3 for a'
    sb[i] = k[i];  // k1 + 2 k2 + 2 k3 + k4 for b'
  }
  beam_accel<M>(mo, P, law, a0_bits, zc, ch, as, bs, k);  // k2
#pragma unroll
  for (int i = 0; i < M; ++i) {
    as[i] = fma(0.5, bs[i], a[i]);  // a + (b + k1/2)/2
    bs[i] = fma(0.5, k[i], b[i]);
    sa[i] += k[i];
    sb[i] = fma(2.0, k[i], sb[i]);
  }
  beam_accel<M>(mo, P, law, a0_bits, zc, ch, as, bs, k);  // k3
#pragma unroll
  for (int i = 0; i < M; ++i) {
    as[i] = a[i] + bs[i];  // a + (b + k2/2)
    bs[i] = b[i] + k[i];
    sa[i] += k[i];
    sb[i] = fma(2.0, k[i], sb[i]);
  }
  beam_accel<M>(mo, P, law, a0_bits, zc, c1, as, bs, k);  // k4
#pragma unroll
  for (int i = 0; i < M; ++i) {
    a[i] = fma(sa[i], sixth, a[i] + b[i]);
    b[i] = fma(sb[i] + k[i], sixth, b[i]);
  }
}

template <int M>
__device__ __forceinline__ double beam_tip(const double (&a)[M]) {
  double u = a[0];
#pragma unroll
  for (int i = 1; i < M; ++i) u += a[i];
  return u;
}

// ---- integrate-and-misfit, beam --------------------------------------------------
// Stream rows (build_stream_kernel with unit amplitude and no offset):
// { cos(w t_n), cos(w (t_n + h/2)), cos(w (t_n + h)), U_n }.
template <int M, int MODE>
__global__ void beam_integrate_f64(BeamConsts bc, BeamModeConsts mo, IntegrateIO io,
                                   int blocks_per_tr) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double4* tile0 = reinterpret_cast<double4*>(smem_raw);
  double4* tile1 = tile0 + (bc.T + kPadRows);  // one pad row per stage for the row fetched ahead
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (bc.T + kPadRows));
  __shared__ Cand red[32];

  const int tid = threadIdx.x;
  const int s = blockIdx.x / blocks_per_tr;
  const int64_t li = (int64_t)(blockIdx.x - s * blocks_per_tr) * blockDim.x + tid;
  const bool active = li < io.per;
  const int64_t gp = (int64_t)s * io.per + (active ? li : io.per - 1);
  const double* stream = io.stream + (int64_t)s * bc.N * 4;

  if (tid == 0) {
    tile0[bc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    tile1[bc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int st = 0; st < 2; ++st) {
      if (st < bc.n_tiles) {
        const int n_begin = st * bc.T;
        const uint32_t bytes = (uint32_t)min(bc.T, bc.N - n_begin) * 32u;
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + (int64_t)n_begin * 4, bytes, &bars[st]);
      }
    }
  }

  // a1: parameter map
  double xloc[4], th[4] = {0.0, 0.0, 0.0, 1.0};
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    xloc[j] = 0.0;
    if (j < bc.D) {
      const double xv = io.params[gp * bc.D + j];
      xloc[j] = xv;
      th[j] = (io.mode != 0 && io.box.lg[j]) ? pow(10.0, xv) : xv;
    }
  }
  Particle64 P;
  load_particle(P, bc.law, th, 0.0, 0.0, bc.a0, bc.inv_a0sq, bc.c_vdw, bc.c_hertz,
                bc.c_visc, bc.c_force, bc.zc, bc.c_damp);
  const long long a0_bits = __double_as_longlong(bc.a0);
  double a[M], b[M];
#pragma unroll
  for (int i = 0; i < M; ++i) a[i] = b[i] = 0.0;  // from rest
  double J = 0.0;
  bool bad = false;

  for (int tile = 0; tile < bc.n_tiles; ++tile) {
    const int st = tile & 1;
    const double4* sp = st ? tile1 : tile0;
    mbar_wait(&bars[st], (uint32_t)((tile >> 1) & 1));
    const int n_begin = tile * bc.T;
    const int n_steps = min(bc.T, bc.N - n_begin);
    AFM_CHECK(n_steps >= 1 && n_steps <= bc.T && n_begin + n_steps <= bc.N);
    double4 r = sp[0];
    for (int i = 0; i < n_steps; ++i) {
      const double4 rn = sp[i + 1];
      beam_rk4<M>(mo, P, bc.law, a0_bits, bc.zc, r.x, r.y, r.z, a, b);
      const double u = beam_tip<M>(a);
      bad |= !(fabs(u) <= bc.u_max);  // NaN fails the comparison
      if (n_begin + i >= bc.n0) {
        const double res = u - r.w;
        J = fma(res, res, J);
      }
      r = rn;
    }
    __syncthreads();
    if (tid == 0 && tile + 2 < bc.n_tiles) {
      const int nb = (tile + 2) * bc.T;
      const uint32_t bytes = (uint32_t)min(bc.T, bc.N - nb) * 32u;
      fence_proxy_async();
      mbar_arrive_expect_tx(&bars[st], bytes);
      bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
    }
  }
#pragma unroll
  for (int i = 0; i < M; ++i) bad |= !(fabs(a[i]) < CUDART_INF && fabs(b[i]) < CUDART_INF);
  if (bad || !(J == J)) J = CUDART_INF;
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
          if (j < bc.D) io.pbest[gp * bc.D + j] = xloc[j];
      }
      pb = pq;
      idx = gp;
    }
    block_argmin(pb, idx, red);
    if (tid == 0) {
      io.cand[blockIdx.x].J = pb;
      io.cand[blockIdx.x].idx = idx;
    }
  }
}

// Segment-queue form (see integrate_misfit_f64_q in afm_kernels.cu): persistent
// one-warp workers take (chain, segment) tasks from the priority queue; between
// segments a chain rests as { a[M], b[M], J, diverged } per particle.  Same
// arithmetic per particle as beam_integrate_f64: bit-identical results.  65 536
// particles are 3.46 warps per SM sub-partition, which one CTA per warp spreads as
// 3 on some sub-partitions and 4 on others for the whole solve.
template <int M, int MODE>
__global__ void __launch_bounds__(32)
beam_integrate_f64_q(BeamConsts bc, BeamModeConsts mo, IntegrateIO io, int blocks_per_tr,
                     SegQueue q) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double4* tile0 = reinterpret_cast<double4*>(smem_raw);
  double4* tile1 = tile0 + (bc.T + kPadRows);
  uint64_t* bars = reinterpret_cast<uint64_t*>(tile1 + (bc.T + kPadRows));
  __shared__ Cand red[32];
  __shared__ SegqWorker qworker;  // lane 0's queue state (one warp per CTA)

  const int tid = threadIdx.x;
  if (tid == 0) {
    qworker.offered = 0u;
    tile0[bc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    tile1[bc.T] = make_double4(0.0, 0.0, 0.0, 0.0);
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t n_wait0 = 0u, n_wait1 = 0u;  // completed phases of the two stages
  const long long a0_bits = __double_as_longlong(bc.a0);

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
    AFM_CHECK(s < io.n_traces && gp >= 0 && gp < io.per * io.n_traces);
    const double* stream = io.stream + (int64_t)s * bc.N * 4;
    const int tile_begin = seg * q.tiles_per_seg;
    const int tile_end = min(tile_begin + q.tiles_per_seg, bc.n_tiles);

    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const int tile = tile_begin + k;
        if (tile < tile_end) {
          const int st = tile & 1;
          const int nb = tile * bc.T;
          const uint32_t bytes = (uint32_t)min(bc.T, bc.N - nb) * 32u;
          fence_proxy_async();
          mbar_arrive_expect_tx(&bars[st], bytes);
          bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
        }
      }
    }

    // a1: parameter map (every segment: the chain may have come from another SM)
    double xloc[4], th[4] = {0.0, 0.0, 0.0, 1.0};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      xloc[j] = 0.0;
      if (j < bc.D) {
        const double xv = io.params[gp * bc.D + j];
        xloc[j] = xv;
        th[j] = (io.mode != 0 && io.box.lg[j]) ? pow(10.0, xv) : xv;
      }
    }
    Particle64 P;
    load_particle(P, bc.law, th, 0.0, 0.0, bc.a0, bc.inv_a0sq, bc.c_vdw, bc.c_hertz,
                  bc.c_visc, bc.c_force, bc.zc, bc.c_damp);
    double a[M], b[M];
    double J = 0.0;
    bool bad = false;
    double* ck = q.ckpt + (int64_t)chain * (32 * (2 * M + 2)) + tid;
    if (seg == 0) {
#pragma unroll
      for (int i = 0; i < M; ++i) a[i] = b[i] = 0.0;  // from rest
    } else {
#pragma unroll
      for (int i = 0; i < M; ++i) {
        a[i] = __ldcg(ck + 32 * i);
        b[i] = __ldcg(ck + 32 * (M + i));
      }
      J = __ldcg(ck + 32 * (2 * M));
      bad = __ldcg(ck + 32 * (2 * M + 1)) != 0.0;
    }

    for (int tile = tile_begin; tile < tile_end; ++tile) {
      const int st = tile & 1;
      const double4* sp = st ? tile1 : tile0;
      mbar_wait(&bars[st], (st ? n_wait1 : n_wait0) & 1u);
      if (st) ++n_wait1; else ++n_wait0;
      const int n_begin = tile * bc.T;
      const int n_steps = min(bc.T, bc.N - n_begin);
      AFM_CHECK(n_steps >= 1 && n_steps <= bc.T && n_begin + n_steps <= bc.N);
      double4 r = sp[0];
      for (int i = 0; i < n_steps; ++i) {
        const double4 rn = sp[i + 1];
        beam_rk4<M>(mo, P, bc.law, a0_bits, bc.zc, r.x, r.y, r.z, a, b);
        const double u = beam_tip<M>(a);
        bad |= !(fabs(u) <= bc.u_max);  // NaN fails the comparison
        if (n_begin + i >= bc.n0) {
          const double res = u - r.w;
          J = fma(res, res, J);
        }
        r = rn;
      }
      __syncthreads();
      if (tid == 0 && tile + 2 < tile_end) {
        const int nb = (tile + 2) * bc.T;
        const uint32_t bytes = (uint32_t)min(bc.T, bc.N - nb) * 32u;
        fence_proxy_async();
        mbar_arrive_expect_tx(&bars[st], bytes);
        bulk_g2s(st ? tile1 : tile0, stream + (int64_t)nb * 4, bytes, &bars[st]);
      }
    }

    if (tile_end < bc.n_tiles) {
      // hand the chain on: state first, then the task (release / acquire)
#pragma unroll
      for (int i = 0; i < M; ++i) {
        __stcg(ck + 32 * i, a[i]);
        __stcg(ck + 32 * (M + i), b[i]);
      }
      __stcg(ck + 32 * (2 * M), J);
      __stcg(ck + 32 * (2 * M + 1), bad ? 1.0 : 0.0);
      __threadfence();
      __syncwarp();
      if (tid == 0) segq_push(q, chain, seg + 1);
      continue;
    }

    // last segment: the epilogue of beam_integrate_f64
#pragma unroll
    for (int i = 0; i < M; ++i) bad |= !(fabs(a[i]) < CUDART_INF && fabs(b[i]) < CUDART_INF);
    if (bad || !(J == J)) J = CUDART_INF;
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
            if (j < bc.D) io.pbest[gp * bc.D + j] = xloc[j];
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

// One particle through the same step routine (tests, trace synthesis).
template <int M>
__global__ void beam_trajectory_kernel(BeamConsts bc, BeamModeConsts mo,
                                       const double* __restrict__ theta,
                                       const double* __restrict__ stream,
                                       double* __restrict__ tip_u,
                                       double* __restrict__ tip_v) {
  const bool writer = (threadIdx.x == 0);
  double th[4] = {0.0, 0.0, 0.0, 1.0};
  for (int j = 0; j < bc.D && j < 4; ++j) th[j] = theta[j];
  Particle64 P;
  load_particle(P, bc.law, th, 0.0, 0.0, bc.a0, bc.inv_a0sq, bc.c_vdw, bc.c_hertz,
                bc.c_visc, bc.c_force, bc.zc, bc.c_damp);
  const long long a0_bits = __double_as_longlong(bc.a0);
  double a[M], b[M];
#pragma unroll
  for (int i = 0; i < M; ++i) a[i] = b[i] = 0.0;
  const double inv_h = 1.0 / bc.h;
  if (writer && tip_u) tip_u[0] = 0.0;
  if (writer && tip_v) tip_v[0] = 0.0;
  const double4* rows = reinterpret_cast<const double4*>(stream);
  for (int n = 0; n < bc.N; ++n) {
    const double4 r = rows[n];
    beam_rk4<M>(mo, P, bc.law, a0_bits, bc.zc, r.x, r.y, r.z, a, b);
    if (writer && tip_u) tip_u[n + 1] = beam_tip<M>(a);
    if (writer && tip_v) tip_v[n + 1] = beam_tip<M>(b) * inv_h;
  }
}

// ---- launchers --------------------------------------------------------------------
int launch_beam_setup(const afm_beam_cfg& cfg, double h, BeamModeConsts* dev_out,
                      cudaStream_t st) {
  beam_setup_kernel<<<1, 32, 0, st>>>(cfg, h, dev_out);
  return 1;
}

template <int M>
static int launch_beam_t(const BeamConsts& bc, const BeamModeConsts& mo,
                         const IntegrateIO& io, int block, cudaStream_t st) {
  const int bpt = blocks_per_trace(io.per, block);
  const unsigned grid = (unsigned)(bpt * io.n_traces);
  const size_t smem = (size_t)(bc.T + kPadRows) * 32 * 2 + 64;
  if (smem > 48 * 1024) {  // afm_set_option("tile") above 767 steps
    cudaFuncSetAttribute(beam_integrate_f64<M, 1>,
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(beam_integrate_f64<M, 0>,
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  if (io.mode == 1)
    beam_integrate_f64<M, 1><<<grid, block, smem, st>>>(bc, mo, io, bpt);
  else
    beam_integrate_f64<M, 0><<<grid, block, smem, st>>>(bc, mo, io, bpt);
  return 1;
}

int launch_beam_integrate(const BeamConsts& bc, const BeamModeConsts& mo,
                          const IntegrateIO& io, int block, cudaStream_t st) {
  switch (bc.M) {
    case 1: return launch_beam_t<1>(bc, mo, io, block, st);
    case 2: return launch_beam_t<2>(bc, mo, io, block, st);
    case 4: return launch_beam_t<4>(bc, mo, io, block, st);
    case 8: return launch_beam_t<8>(bc, mo, io, block, st);
    default: return -1;
  }
}

template <int M>
static int launch_beam_q_t(const BeamConsts& bc, const BeamModeConsts& mo,
                           const IntegrateIO& io, const SegQueue& q, int workers,
                           cudaStream_t st) {
  const int bpt = blocks_per_trace(io.per, 32);
  const size_t smem = (size_t)(bc.T + kPadRows) * 32 * 2 + 64;
  if (smem > 48 * 1024) {
    cudaFuncSetAttribute(beam_integrate_f64_q<M, 1>,
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(beam_integrate_f64_q<M, 0>,
                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  launch_segq_init(q, st);
  if (io.mode == 1)
    beam_integrate_f64_q<M, 1><<<(unsigned)workers, 32, smem, st>>>(bc, mo, io, bpt, q);
  else
    beam_integrate_f64_q<M, 0><<<(unsigned)workers, 32, smem, st>>>(bc, mo, io, bpt, q);
  return 2;
}

int launch_beam_integrate_q(const BeamConsts& bc, const BeamModeConsts& mo,
                            const IntegrateIO& io, const SegQueue& q, int workers,
                            cudaStream_t st) {
  switch (bc.M) {
    case 1: return launch_beam_q_t<1>(bc, mo, io, q, workers, st);
    case 2: return launch_beam_q_t<2>(bc, mo, io, q, workers, st);
    case 4: return launch_beam_q_t<4>(bc, mo, io, q, workers, st);
    case 8: return launch_beam_q_t<8>(bc, mo, io, q, workers, st);
    default: return -1;
  }
}

int launch_beam_trajectory(const BeamConsts& bc, const BeamModeConsts& mo,
                           const double* theta_dev, const double* stream,
                           double* tip_u, double* tip_v, cudaStream_t st) {
  switch (bc.M) {
    case 1: beam_trajectory_kernel<1><<<1, 32, 0, st>>>(bc, mo, theta_dev, stream, tip_u, tip_v); break;
    case 2: beam_trajectory_kernel<2><<<1, 32, 0, st>>>(bc, mo, theta_dev, stream, tip_u, tip_v); break;
    case 4: beam_trajectory_kernel<4><<<1, 32, 0, st>>>(bc, mo, theta_dev, stream, tip_u, tip_v); break;
    case 8: beam_trajectory_kernel<8><<<1, 32, 0, st>>>(bc, mo, theta_dev, stream, tip_u, tip_v); break;
    default: return -1;
  }
  return 1;
}

}  // namespace afm
