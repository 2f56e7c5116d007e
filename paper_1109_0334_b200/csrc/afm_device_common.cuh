// afm_device_common.cuh -- pieces shared by the FP64 and FP32 integrate kernels:
// the PTX wrappers of the TMA-staged (cp.async.bulk + mbarrier) time-tile ring
// and the block argmin of the global-best search.
#pragma once

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "afm_internal.h"

// Bounds checks of our own (compute-sanitizer is not available on the B200 pool):
// python -m paper_1109_0334_b200.build --force --bounds-check compiles every index
// computation below into a checked one that prints and traps; the GPU test suite
// is then run once against that build (profiles/r2_bounds_check.md).
#ifdef AFM_BOUNDS_CHECK
#include <stdio.h>
#define AFM_CHECK(cond)                                                          \
  do {                                                                           \
    if (!(cond)) {                                                               \
      printf("AFM_CHECK failed: %s (%s:%d) block %d thread %d\n", #cond, __FILE__, \
             __LINE__, (int)blockIdx.x, (int)threadIdx.x);                       \
      __trap();                                                                  \
    }                                                                            \
  } while (0)
#else
#define AFM_CHECK(cond) \
  do {                  \
  } while (0)
#endif

namespace afm {

// Each stage of a time-tile ring is followed by pad rows: the kernels fetch the
// next row one step ahead, so the row after a stage's last one is read (and
// discarded); it must be neither a bulk-copy target nor a barrier word.  128
// bytes keep the second stage aligned like the first; only the first pad row is
// ever read (it is zeroed once).
constexpr int kPadBytes = 128;

// ---- mbarrier / bulk-copy PTX (sm_90+; SASS: SYNCS.*, UBLKCP) ---------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(count)
               : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar,
                                                      uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(
                   smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
// 1-D bulk async copy global -> shared, completion counted on an mbarrier.
// dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src,
                                         uint32_t bytes, uint64_t* bar) {
  AFM_CHECK(bytes > 0 && (bytes & 15u) == 0 && (smem_u32(dst) & 15u) == 0 &&
            ((uintptr_t)src & 15u) == 0);
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "AFM_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra AFM_DONE;\n"
      "bra AFM_WAIT;\n"
      "AFM_DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// ---- segment queue of the *_q integrate kernels (see afm_kernels.cu) ----------
__device__ __forceinline__ int ld_relaxed_s32(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_s32(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Next task of this worker: -1 when every task has been handed out, -2 after a
// time-out (cannot happen unless the queue is corrupted; keeps a bug from
// hanging the device).  Called by one lane.
__device__ __forceinline__ int segq_pop(const SegQueue& q) {
  const unsigned t = atomicAdd(&q.ctrl[0], 1u);
  if (t >= (unsigned)q.n_tasks) return -1;
  AFM_CHECK(q.n_tasks == q.n_chains * q.n_segs);
  const long long t_start = clock64();
  int v;
  unsigned ns = 250;  // poll with back-off: a waiting worker shares its issue port
  while ((v = ld_relaxed_s32(&q.slots[t])) < 0) {
    __nanosleep(ns);
    if (ns < 4000) ns *= 2;
    if (clock64() - t_start > q.timeout_cycles) {
      atomicExch(&q.ctrl[2], 1u);
      return -2;
    }
  }
  __threadfence();  // acquire: the chain's checkpoint was written before the slot
  AFM_CHECK((v & 0xfffff) < q.n_chains && (v >> 20) < q.n_segs);
  return v;
}


// Publish segment `seg` of `chain` at the tail of the queue.  The caller has
// stored the chain's checkpoint, fenced and synchronised its warp.  One lane.
__device__ __forceinline__ void segq_push(const SegQueue& q, int chain, int seg) {
  const unsigned slot = atomicAdd(&q.ctrl[1], 1u);
  AFM_CHECK(slot < (unsigned)q.n_tasks && chain < q.n_chains && seg < q.n_segs);
  st_release_s32(&q.slots[slot], (seg << 20) | chain);
}

__device__ __forceinline__ bool cand_less(double Ja, long long ia, double Jb,
                                          long long ib) {
  return (Ja < Jb) || (Ja == Jb && ia < ib);
}

// Block argmin of (J, idx), lowest idx among equal J; result valid in thread 0.
__device__ __forceinline__ void block_argmin(double& J, long long& idx,
                                             Cand* red /* [32] shared */) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nwarps = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    double Jo = __shfl_down_sync(0xffffffffu, J, off);
    long long io = __shfl_down_sync(0xffffffffu, idx, off);
    if (cand_less(Jo, io, J, idx)) {
      J = Jo;
      idx = io;
    }
  }
  if (nwarps == 1) return;
  if (lane == 0) {
    red[warp].J = J;
    red[warp].idx = idx;
  }
  __syncthreads();
  if (warp == 0) {
    J = (lane < nwarps) ? red[lane].J : CUDART_INF;
    idx = (lane < nwarps) ? red[lane].idx : 0x7fffffffffffffffLL;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
      double Jo = __shfl_down_sync(0xffffffffu, J, off);
      long long io = __shfl_down_sync(0xffffffffu, idx, off);
      if (cand_less(Jo, io, J, idx)) {
        J = Jo;
        idx = io;
      }
    }
  }
}

}  // namespace afm
