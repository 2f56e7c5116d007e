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
// A priority queue keyed by the segment index ("level"): level l holds one slot
// per chain, filled in the order the chains finish segment l - 1 and consumed in
// that order; a worker always takes the oldest published task of the LOWEST level
// that has one, so a chain that has fallen behind (more general-form steps, a
// higher cost per segment) is picked up the moment it is published while the
// chains that are ahead wait.  With fewer workers than chains the chains thus
// advance within about one segment of one another and finish together.
__device__ __forceinline__ int ld_relaxed_s32(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_s32(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Next task of this worker, (segment << 20) | chain: -1 when every task has been
// handed out, -2 after a time-out (cannot happen unless the queue is corrupted;
// keeps a bug from hanging the device).  Called by one lane.
__device__ __forceinline__ int segq_take(const SegQueue& q) {
  AFM_CHECK(q.n_tasks == q.n_chains * q.n_segs);
  const unsigned nc = (unsigned)q.n_chains;
  long long t_start = 0;
  unsigned ns = 250;  // poll with back-off: a waiting worker shares its issue port
  for (;;) {
    int l = (int)ld_relaxed_u32(&q.ctrl[0]);  // lowest level not yet handed out in full
    if (l >= q.n_segs) return -1;
    bool lowest = true;
    for (; l < q.n_segs; ++l) {
      const unsigned h = ld_relaxed_u32(&q.head[l]);
      if (h >= nc) {  // level handed out in full
        if (lowest) atomicMax(&q.ctrl[0], (unsigned)(l + 1));
        continue;
      }
      lowest = false;
      const unsigned t = ld_relaxed_u32(&q.tail[l]);
      if (t == 0u) break;    // nothing was ever published here, so nothing above either
      if (h >= t) continue;  // nothing ready at this level right now
      const unsigned ticket = atomicAdd(&q.head[l], 1u);
      if (ticket >= nc) continue;  // lost the race for the level's last tasks
      // the ticket's slot is published already unless other workers raced for the
      // same tasks; then it is the next chain to finish segment l - 1
      const int* slot = &q.slots[(size_t)l * nc + ticket];
      int v;
      while ((v = ld_relaxed_s32(slot)) < 0) {
        if (t_start == 0) t_start = clock64();
        __nanosleep(ns);
        if (ns < 4000) ns *= 2;
        if (clock64() - t_start > q.timeout_cycles) {
          atomicExch(&q.ctrl[2], 1u);
          return -2;
        }
      }
      __threadfence();  // acquire: the chain's checkpoint was written before the slot
      AFM_CHECK(v < q.n_chains);
      return (l << 20) | v;
    }
    if (t_start == 0) t_start = clock64();
    __nanosleep(ns);
    if (ns < 4000) ns *= 2;
    if (clock64() - t_start > q.timeout_cycles) {
      atomicExch(&q.ctrl[2], 1u);
      return -2;
    }
  }
}

// SM sub-partition of the calling warp: warp slots w, w + 4, w + 8, ... of an SM share
// a scheduler and its FP64 pipe (measured: two DFMA-bound warps slow each other down
// exactly when their %warpid agree modulo 4).
__device__ __forceinline__ unsigned smsp_id() {
  unsigned smid, wid;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
  asm volatile("mov.u32 %0, %%warpid;" : "=r"(wid));
  return smid * 4u + (wid & 3u);
}

// segq_take plus the boost of the chains on the critical path.  Chains advance
// within about a segment of one another, except the few whose cost per step is
// far above the rest (a warp with a particle stuck to the sample runs every step
// in the general form): always picked up at once, always running, they still
// fall behind and set the time of the batch.  A worker that takes a task of a
// level most chains have already finished offers a parking place on its
// sub-partition -- two places if most chains have finished the level after it as
// well: another worker there, when it next comes for a task, takes a place and
// sleeps until the marked segment is over, and the chain that is behind runs
// beside one warp fewer (a third faster at three warps per sub-partition) or
// alone.  q.park[smsp]: bits 0-7 = places on offer, bits 8-15 = epoch, advanced
// when a marked segment ends (which wakes the sleepers).  Called by one lane.
struct SegqWorker {
  unsigned offered;  // places this worker has put on offer for its current segment
};
__device__ __forceinline__ int segq_pop(const SegQueue& q, SegqWorker* wk) {
  unsigned& offered = wk->offered;
  const unsigned sp = smsp_id();
  if (sp >= (unsigned)q.n_park) return segq_take(q);
  unsigned* pk = &q.park[sp];
  if (offered != 0u) {
    // the marked segment is over: withdraw what is left of the offer, wake the rest
    offered = 0u;
    unsigned w = ld_relaxed_u32(pk), seen;
    do {
      seen = w;
      w = atomicCAS(pk, seen, ((seen & 0xff00u) + 0x100u) & 0xff00u);
    } while (w != seen);
  } else {
    unsigned w = ld_relaxed_u32(pk);
    while ((w & 0xffu) != 0u) {
      const unsigned seen = w;
      w = atomicCAS(pk, seen, seen - 1u);
      if (w != seen) continue;
      const unsigned epoch = seen & 0xff00u;
      unsigned waited = 0;
      while ((ld_relaxed_u32(pk) & 0xff00u) == epoch &&
             (int)ld_relaxed_u32(&q.ctrl[0]) < q.n_segs && ++waited < 200000u)
        __nanosleep(2000);
      break;
    }
  }
  const int task = segq_take(q);
  if (task >= 0) {
    const int l = task >> 20;
    const unsigned nc = (unsigned)q.n_chains, div = (unsigned)q.boost_div;
    unsigned want = 0u;
    if (l + 1 < q.n_segs && div * ld_relaxed_u32(&q.tail[l + 1]) > nc) {
      want = 1u;
      if (q.boost_two && l + 2 < q.n_segs && div * ld_relaxed_u32(&q.tail[l + 2]) > nc)
        want = 2u;
    }
    if (want != 0u) {
      atomicAdd(pk, want);
      offered = want;
    }
  }
  return task;
}

// Publish segment `seg` of `chain` at its level.  The caller has stored the
// chain's checkpoint, fenced and synchronised its warp.  One lane.
__device__ __forceinline__ void segq_push(const SegQueue& q, int chain, int seg) {
  AFM_CHECK(chain < q.n_chains && seg >= 1 && seg < q.n_segs);
  const unsigned slot = atomicAdd(&q.tail[seg], 1u);
  AFM_CHECK(slot < (unsigned)q.n_chains);
  st_release_s32(&q.slots[(size_t)seg * q.n_chains + slot], chain);
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
