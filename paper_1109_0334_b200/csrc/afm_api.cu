// afm_api.cu -- the C ABI of include/afm.h: argument validation, the scaled
// model constants, the device workspace and the launch sequences.  No
// arithmetic of the method runs here beyond the handful of scalar constants in
// make_consts(); every step of the hot path is a kernel in afm_kernels.cu.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "afm_internal.h"

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

namespace {

using namespace afm;

thread_local char g_err[512] = "";
thread_local int64_t g_launches = 0;
thread_local const char* g_last_kernel = "";  // afm_last_integrate_kernel()

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(expr)                                                        \
  do {                                                                        \
    cudaError_t e_ = (expr);                                                  \
    if (e_ != cudaSuccess)                                                    \
      return fail(AFM_ECUDA, "%s failed: %s (%s:%d)", #expr,                  \
                  cudaGetErrorString(e_), __FILE__, __LINE__);                \
  } while (0)

#define LAUNCHED(call)                                                        \
  do {                                                                        \
    int n_ = (call);                                                          \
    if (n_ < 0) return fail(AFM_EINVAL, "no kernel for this law (%s)", #call);\
    g_launches += n_;                                                         \
    cudaError_t e_ = cudaGetLastError();                                      \
    if (e_ != cudaSuccess)                                                    \
      return fail(AFM_ECUDA, "launch %s failed: %s", #call,                   \
                  cudaGetErrorString(e_));                                    \
  } while (0)

// ---- options -----------------------------------------------------------------
int g_opt_block = 0;  // 0 = auto
int g_opt_tile = 0;   // 0 = auto
int g_opt_ppt = 0;    // 0 = auto
int g_opt_form = 0;   // 0 = auto, 1 = throughput form, 2 = latency form
int g_opt_lanes = 0;  // 0 = auto; latency form: particles per warp
int g_opt_pack = 0;   // 0 = auto, 1 = never, 2 = always (DMT laws only)
int g_opt_queue = 0;  // 0 = auto, 1 = never, 2 = always: segment-queue scheduling
int g_opt_segs = 0;   // 0 = auto (~450 steps each): time segments per chain of the queue kernel
int g_opt_workers = 0;  // 0 = auto: queue workers per SM sub-partition
int g_opt_boost2 = 0;   // 0 = auto (on), 1 = off: a second parking place for a chain two segments behind
int g_opt_boost = 0;    // 0 = auto (2), 1 = off, k >= 2: parking beside the chains that are behind
                        // more than 1/k of the chains by a whole segment
int g_n_sm = 148;

// afm_set_option("kernel_events", 1): every launch of an integrate kernel is
// bracketed by a pair of CUDA events on its own stream (bench.py's
// roofline.kernel_ms: the duration of the dominant kernel alone, measured live).
constexpr int kMaxKernelEvents = 64;
int g_opt_kernel_events = 0;
cudaEvent_t g_kev[kMaxKernelEvents][2];
bool g_kev_made = false;
int64_t g_kev_count = 0;  // launches recorded since the option was switched on

int kev_record(int which, cudaStream_t st) {
  if (!g_opt_kernel_events) return AFM_OK;
  if (!g_kev_made) {
    for (int i = 0; i < kMaxKernelEvents; ++i)
      for (int j = 0; j < 2; ++j) CUDA_TRY(cudaEventCreate(&g_kev[i][j]));
    g_kev_made = true;
  }
  CUDA_TRY(cudaEventRecord(g_kev[g_kev_count % kMaxKernelEvents][which], st));
  if (which == 1) ++g_kev_count;
  return AFM_OK;
}

// ---- grow-only device workspace ------------------------------------------------
struct Buffer {
  void* p = nullptr;
  size_t cap = 0;
  int ensure(size_t bytes) {
    if (bytes <= cap) return 0;
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
    // round up so that slightly larger follow-up calls reuse the allocation
    size_t want = (bytes + (size_t)(1 << 20) - 1) & ~((size_t)(1 << 20) - 1);
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) {
      p = nullptr;
      return -1;
    }
    cap = want;
    return 0;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
  }
};

struct Workspace {
  std::mutex mu;
  Buffer stream;                       // time-tile stream
  Buffer swarm;                        // x, v, pbest, J, pbestJ, gbest, ...
  Buffer cand;                         // block candidates
  Buffer h_params, h_trace, h_z0v0, h_misfit;  // staging for the *_host calls
  Buffer h_state;                      // staging for afm_pso_step_host
  Buffer scratch;                      // theta for afm_trajectory
  Buffer sort;                         // warp-packing keys, order, radix-sort temp
  Buffer segq;                         // segment queue: control words, slots, checkpoints
  Buffer chunk;                        // asynchronous swarm: theta and J of one chunk
  cudaEvent_t last_use = nullptr;      // orders reuse across streams
  cudaStream_t last_stream = nullptr;
  bool checked_device = false;
  int device = -1;                     // owner of every buffer above
  void* pinned = nullptr;              // small pinned host block
  size_t pinned_cap = 0;
} g_ws;

// The workspace (and the SM count the launch decisions use) belongs to the device
// that was current at the first compute call; a caller that switches devices must
// call afm_shutdown() in between.
int check_device() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess)
    return fail(AFM_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
  if (g_ws.checked_device) {
    if (dev != g_ws.device)
      return fail(AFM_EUNSUPPORTED,
                  "the library workspace lives on device %d but device %d is current: "
                  "call afm_shutdown() before switching devices", g_ws.device, dev);
    return AFM_OK;
  }
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10)
    return fail(AFM_EUNSUPPORTED,
                "device %s is sm_%d%d; this library is built for sm_100a only",
                prop.name, prop.major, prop.minor);
  g_n_sm = prop.multiProcessorCount;
  g_ws.device = dev;
  g_ws.checked_device = true;
  return AFM_OK;
}

// Serialise reuse of the shared workspace between calls on different streams.
int acquire_ws(cudaStream_t st) {
  if (g_ws.last_use == nullptr)
    CUDA_TRY(cudaEventCreateWithFlags(&g_ws.last_use, cudaEventDisableTiming));
  else if (g_ws.last_stream != st)
    CUDA_TRY(cudaStreamWaitEvent(st, g_ws.last_use, 0));
  return AFM_OK;
}
int release_ws(cudaStream_t st) {
  CUDA_TRY(cudaEventRecord(g_ws.last_use, st));
  g_ws.last_stream = st;
  return AFM_OK;
}

int ensure_pinned(size_t bytes) {
  if (bytes <= g_ws.pinned_cap) return AFM_OK;
  if (g_ws.pinned) cudaFreeHost(g_ws.pinned);
  g_ws.pinned = nullptr;
  g_ws.pinned_cap = 0;
  CUDA_TRY(cudaMallocHost(&g_ws.pinned, bytes));
  g_ws.pinned_cap = bytes;
  return AFM_OK;
}

// ---- validation + constants ------------------------------------------------------
int law_dims(int law) {
  switch (law) {
    case AFM_LAW_DMT: return 2;
    case AFM_LAW_DMT_VISC: return 3;
    case AFM_LAW_LJ_EXP: return 4;
    case AFM_LAW_HOOKE: return 2;
    case AFM_LAW_KELVIN_VOIGT: return 2;
    default: return -1;
  }
}

int validate_cfg(const afm_cfg* c) {
  if (!c) return fail(AFM_EINVAL, "cfg is NULL");
  if (c->law < AFM_LAW_NONE || c->law > AFM_LAW_KELVIN_VOIGT)
    return fail(AFM_EINVAL, "unknown law %d", c->law);
  if (c->law == AFM_LAW_NONE) {
    if (c->n_params < 0 || c->n_params > 4)
      return fail(AFM_EINVAL, "n_params %d out of range 0..4", c->n_params);
  } else if (c->n_params != law_dims(c->law)) {
    return fail(AFM_EINVAL, "law %d needs n_params = %d, got %d", c->law,
                law_dims(c->law), c->n_params);
  }
  if (!(c->k > 0) || !(c->f0 > 0) || !(c->Q > 0) || !(c->f_drive > 0))
    return fail(AFM_EINVAL, "k, f0, Q, f_drive must be positive");
  if (!(c->A0 > 0)) return fail(AFM_EINVAL, "A0 must be positive");
  if ((c->law == AFM_LAW_DMT || c->law == AFM_LAW_DMT_VISC) &&
      (!(c->R > 0) || !(c->a0 > 0)))
    return fail(AFM_EINVAL, "DMT laws need R > 0 and a0 > 0");
  if (c->steps_per_cycle < 1 || c->n_cycles < 1)
    return fail(AFM_EINVAL, "steps_per_cycle and n_cycles must be >= 1");
  if (c->n_skip_cycles < 0 || c->n_skip_cycles >= c->n_cycles)
    return fail(AFM_EINVAL, "need 0 <= n_skip_cycles < n_cycles");
  if ((int64_t)c->steps_per_cycle * c->n_cycles > (int64_t)1 << 30)
    return fail(AFM_EINVAL, "more than 2^30 steps");
  if (c->n_traces < 1) return fail(AFM_EINVAL, "n_traces must be >= 1");
  if (c->precision != AFM_F64 && c->precision != AFM_F32)
    return fail(AFM_EINVAL, "unknown precision %d", c->precision);
  if (c->reserved_ != 0) return fail(AFM_EINVAL, "reserved_ must be 0");
  if (!isfinite(c->z0) || !isfinite(c->v0) || !isfinite(c->z_c))
    return fail(AFM_EINVAL, "z0, v0, z_c must be finite");
  return AFM_OK;
}

void make_consts(const afm_cfg* c, int block, ModelConsts* mc) {
  const double w0 = 2.0 * M_PI * c->f0;
  const double w = 2.0 * M_PI * c->f_drive;
  const double m = c->k / (w0 * w0);
  const double r = w / w0;
  const double a = 1.0 - r * r, b = r / c->Q;
  const double F0 = c->k * c->A0 * sqrt(a * a + b * b);
  const double h = 2.0 * M_PI / (w * (double)c->steps_per_cycle);
  memset(mc, 0, sizeof(*mc));
  mc->h = h;
  mc->w_drive = w;
  mc->alpha = h * w0 / c->Q;
  mc->beta = h * h * (c->k / m);
  mc->drive_amp = h * h * F0 / m;
  mc->beta_zc = mc->beta * c->z_c;
  mc->zc = c->z_c;
  mc->a0 = c->a0;
  mc->inv_a0sq = (c->a0 > 0) ? 1.0 / (c->a0 * c->a0) : 0.0;
  mc->c_vdw = h * h * c->R / (6.0 * m);
  mc->c_hertz = h * h * (4.0 / 3.0) * sqrt(c->R > 0 ? c->R : 0.0) / m;
  mc->c_visc = h * sqrt(c->R > 0 ? c->R : 0.0) / m;
  mc->c_force = h * h / m;
  mc->c_damp = h / m;
  mc->d_max = c->z_c + 100.0 * c->A0;
  mc->d_min = c->z_c - 100.0 * c->A0;
  mc->d_safe = fmax(0.0, 100.0 * c->A0 - fabs(c->z_c));
  mc->z0 = c->z0;
  mc->v0 = c->v0;
  mc->law = c->law;
  mc->D = c->n_params;
  mc->N = c->steps_per_cycle * c->n_cycles;
  mc->W = c->steps_per_cycle * (c->n_cycles - c->n_skip_cycles);
  mc->n0 = mc->N - mc->W;
  int T = g_opt_tile > 0 ? g_opt_tile : (block <= 32 ? 64 : 128);
  if (T > mc->N) T = mc->N;
  mc->T = T;
  mc->n_tiles = (mc->N + T - 1) / T;
}

// FP32 kernel constants (kernel units: 1 nm, one step; everything /6).
void make_consts_f32(const afm_cfg* c, ModelConstsF32* mf) {
  const double w0 = 2.0 * M_PI * c->f0;
  const double w = 2.0 * M_PI * c->f_drive;
  const double r = w / w0;
  const double a = 1.0 - r * r, b = r / c->Q;
  const double h = 2.0 * M_PI / (w * (double)c->steps_per_cycle);
  const double len = 1e-9;
  const double hq = h * w0;
  memset(mf, 0, sizeof(*mf));
  mf->len = len;
  mf->h = h;
  mf->w_drive = w;
  mf->a6 = hq / c->Q / 6.0;
  mf->b6 = hq * hq / 6.0;
  mf->drive6 = mf->b6 * (c->A0 * sqrt(a * a + b * b)) / len;
  mf->b6_zc = mf->b6 * c->z_c / len;
  mf->zc = c->z_c / len;
  mf->a0 = c->a0 / len;
  const double sqR = sqrt(c->R > 0 ? c->R : 0.0);
  mf->c_vdw = mf->b6 * c->R / (6.0 * c->k * len * len * len);
  mf->c_hertz = mf->b6 * (4.0 / 3.0) * sqR * sqrt(len) / c->k;
  mf->c_visc = mf->b6 * sqR * sqrt(len) / (h * c->k);
  mf->c_rep = mf->b6 / (c->k * pow(len, 9.0));
  mf->c_att = mf->b6 / (c->k * len * len * len);
  mf->c_fad = mf->b6 / (c->k * len);
  mf->c_lam = 1.4426950408889634 * len;
  mf->c_ks = mf->b6 / c->k;
  mf->c_zeta = mf->b6 / (h * c->k);
  mf->d_max = (c->z_c + 100.0 * c->A0) / len;
  mf->d_min = (c->z_c - 100.0 * c->A0) / len;
  mf->d_safe = fmax(0.0, 100.0 * c->A0 - fabs(c->z_c)) / len;
  mf->z0 = c->z0;
  mf->v0 = c->v0;
  mf->law = c->law;
  mf->D = c->n_params;
  mf->N = c->steps_per_cycle * c->n_cycles;
  mf->W = c->steps_per_cycle * (c->n_cycles - c->n_skip_cycles);
  mf->n0 = mf->N - mf->W;
  int T = g_opt_tile > 0 ? g_opt_tile : 128;
  if (T > mf->N) T = mf->N;
  mf->T = T;
  mf->n_tiles = (mf->N + T - 1) / T;
}

// Launch shape of the integrate kernels: one warp per CTA and one particle per
// thread unless afm_set_option says otherwise (measured on B200, DESIGN.md 6:
// 64- and 128-thread CTAs change nothing; two particles per thread cost the FP64
// kernel 28 %, so "ppt" now reaches the FP32 kernel only).
int block_threads() { return g_opt_block > 0 ? g_opt_block : 32; }
int particles_per_thread() { return g_opt_ppt > 0 ? g_opt_ppt : 1; }

// Kernel form of the FP64 integrate kernel (afm_device.cuh, vdw_plus): the
// latency form below two warps per SM sub-partition, where nothing hides the
// dependent chains; the throughput form (fewest FP64 instructions) above.
int pick_variant(int64_t per, int n_traces, int /*ppt: FP32 kernel only*/) {
  if (g_opt_form == 1) return 0;
  if (g_opt_form == 2) return 1;
  const int64_t warps = ((per + 31) / 32) * n_traces;
  return warps < (int64_t)2 * 4 * g_n_sm ? 1 : 0;
}

// Warp packing (afm_sort.cu) for the DMT laws in the throughput regime of a
// forward batch: on success *order is the device order array and the packed
// copies of params / z0v0 and a packed misfit buffer are ready; *order stays
// nullptr when packing does not apply.  Lock held.
struct Packed {
  const uint32_t* order = nullptr;
  double* params = nullptr;
  double* z0v0 = nullptr;
  double* J = nullptr;
};

int pack_inputs(const afm_cfg* cfg, const double* params, const double* z0v0,
                int64_t per, int n_traces, const BoxDev* map, Packed* pk,
                cudaStream_t st) {
  const bool dmt = (cfg->law == AFM_LAW_DMT || cfg->law == AFM_LAW_DMT_VISC);
  const int D = cfg->n_params;
  const int64_t PT = per * n_traces;
  const int64_t warps = ((per + 31) / 32) * n_traces;
  if (!dmt || g_opt_pack == 1 || PT >= ((int64_t)1 << 31) || n_traces >= (1 << 24))
    return AFM_OK;
  if (g_opt_pack == 0 && warps < (int64_t)2 * 4 * g_n_sm) return AFM_OK;
  const size_t ws = sort_workspace_bytes(PT);
  const size_t a256 = 255;
  const size_t o_bytes = ((size_t)PT * 4 + a256) & ~a256;
  const size_t p_bytes = ((size_t)PT * D * 8 + a256) & ~a256;
  const size_t z_bytes = ((size_t)PT * 16 + a256) & ~a256;
  const size_t j_bytes = ((size_t)PT * 8 + a256) & ~a256;
  if (g_ws.sort.ensure(o_bytes + p_bytes + z_bytes + j_bytes + ws + 256))
    return fail(AFM_ECUDA, "cudaMalloc of the packing workspace failed");
  char* base = (char*)g_ws.sort.p;
  uint32_t* order = (uint32_t*)base;
  pk->params = (double*)(base + o_bytes);
  pk->z0v0 = z0v0 ? (double*)(base + o_bytes + p_bytes) : nullptr;
  pk->J = (double*)(base + o_bytes + p_bytes + z_bytes);
  void* scratch = base + o_bytes + p_bytes + z_bytes + j_bytes;
  const int n = launch_pack_order(params, z0v0, D, per, PT, 2.0 * M_PI * cfg->f_drive,
                                  cfg->z0, cfg->v0, scratch, ws, order, st);
  if (n < 0) return fail(AFM_ECUDA, "radix sort of the packing keys failed");
  g_launches += n;
  LAUNCHED(launch_pack_gather(order, params, z0v0, D, PT, pk->params, pk->z0v0, map, st));
  pk->order = order;
  return AFM_OK;
}

// Latency form: particles per warp, so that the warps spread over all SM
// sub-partitions (DMT laws; the other laws have no warp-wide mode to protect).
int pick_lanes(const afm_cfg* cfg, int64_t per, int n_traces) {
  if (g_opt_lanes > 0) return g_opt_lanes;
  const bool dmt = (cfg->law == AFM_LAW_DMT || cfg->law == AFM_LAW_DMT_VISC);
  if (!dmt) return 32;
  // fewest particles per warp that still leaves at most one warp per SM
  // sub-partition (two warps sharing a dispatch port cost more than they save:
  // configs[2] 745 ms at 2 per warp, 898 ms at 1 per warp)
  int lanes = 1;
  while (lanes < 32 && ((per + lanes - 1) / lanes) * n_traces > (int64_t)4 * g_n_sm)
    lanes *= 2;
  return lanes;
}

// CTAs per trace of the FP64 integrate kernel for a launch decision.
int integrate_bpt(int64_t per, int block, int /*ppt: FP32 kernel only*/, int variant,
                  int lanes) {
  return variant == 1 ? blocks_per_trace(per, lanes) : blocks_per_trace(per, block);
}

// Segment-queue scheduling (integrate_misfit_f64_q / _f32_q): the time loop of every
// warp of particles (a "chain") is cut into segments that persistent one-warp
// workers take from a priority queue keyed by the segment index.  Fewer workers
// than chains -- chains per sub-partition / 1.15, rounded down, between 2 and 5
// per sub-partition -- so that the chains that are ahead wait while the ones that
// are behind run, and all finish together.  Measured (configs[1]-like batches of
// r chains per sub-partition, best workers per sub-partition): r = 2.5: 2,
// r = 3.5 and 4: 3, r = 5.5: 4, r = 8 and 12: 5 (6 to 8 are slower), configs[4]
// (r = 55): 5 or 6.  *use is false when the plain kernel should run.  Lock held.
// Workers per SM sub-partition the queue kernels would run for this batch, 0 = the
// plain kernel runs.  Lock held.
int queue_per_sub(int64_t per, int n_traces, int64_t n_steps, bool eligible,
                  int max_chains_per_sub) {
  const int64_t chains = (int64_t)blocks_per_trace(per, 32) * n_traces;
  const int64_t subparts = (int64_t)4 * g_n_sm;
  bool use = eligible && g_opt_queue != 1 && chains < (1 << 20);
  if (use && g_opt_queue == 0) use = (2 * chains >= 3 * subparts && n_steps >= 2048);
  if (use && g_opt_queue == 0 && max_chains_per_sub > 0)
    use = chains <= (int64_t)max_chains_per_sub * subparts;
  if (!use) return 0;
  int per_sub = g_opt_workers > 0 ? g_opt_workers : (int)((chains * 100) / (subparts * 115));
  if (g_opt_workers == 0 && per_sub < 2) per_sub = 2;
  if (g_opt_workers == 0 && per_sub > 5) per_sub = 5;
  if (per_sub > 8) per_sub = 8;
  return per_sub;
}

// per_sub_decided >= 0: the caller has already asked queue_per_sub (with the true
// step count, before it chose the tile length) and this call must not decide again
// from the tile-rounded count n_tiles * T, which can differ just below the threshold.
int make_queue(int64_t per, int n_traces, int n_tiles, int T, bool eligible,
               SegQueue* q, int* workers, bool* use, cudaStream_t st,
               int ckpt_doubles = 4, int max_chains_per_sub = 0,
               int per_sub_decided = -1) {
  const int64_t chains = (int64_t)blocks_per_trace(per, 32) * n_traces;
  const int64_t subparts = (int64_t)4 * g_n_sm;
  const int per_sub =
      per_sub_decided >= 0
          ? per_sub_decided
          : queue_per_sub(per, n_traces, (int64_t)n_tiles * T, eligible, max_chains_per_sub);
  *use = per_sub > 0;
  if (!*use) return AFM_OK;
  *workers = (int)(per_sub * subparts);
  if (*workers > chains) *workers = (int)chains;
  // segments of about 1 000 steps (250 us at 3 FP64 warps per sub-partition: long
  // against the 2-3 us a hand-over costs, short against the whole solve; measured
  // on configs[1], 51 200 steps: 29 to 58 segments 12.86 ms, 80: 12.91, 115: 13.06)
  int segs = g_opt_segs > 0 ? g_opt_segs : (n_tiles * T + 1023) / 1024;
  if (segs > n_tiles) segs = n_tiles;
  if (segs > 2047) segs = 2047;
  if (segs < 1) segs = 1;
  q->tiles_per_seg = (n_tiles + segs - 1) / segs;
  q->n_segs = (n_tiles + q->tiles_per_seg - 1) / q->tiles_per_seg;
  q->n_chains = (int32_t)chains;
  const int64_t tasks = chains * q->n_segs;
  if (tasks >= ((int64_t)1 << 30)) {
    if (g_opt_queue == 2)
      return fail(AFM_EINVAL, "segment queue: %lld chains x %d segments are too many",
                  (long long)chains, (int)q->n_segs);
    *use = false;
    return AFM_OK;
  }
  q->n_tasks = (int32_t)tasks;
  q->timeout_cycles = 40000000000LL;  // ~20 s: only a corrupted queue gets there
  const size_t slot_bytes = ((size_t)q->n_tasks * 4 + 255) & ~(size_t)255;
  const size_t lvl_bytes = 3 * 2048 * 4;  // head[], tail[]: segs <= 2047; park[]
  const size_t need =
      256 + lvl_bytes + slot_bytes + (size_t)chains * 32 * (size_t)ckpt_doubles * 8;
  if (need > ((size_t)2 << 30) && g_opt_queue == 0) {  // too many chains x segments
    *use = false;
    return AFM_OK;
  }
  const bool fresh = need > g_ws.segq.cap;
  if (g_ws.segq.ensure(need))
    return fail(AFM_ECUDA, "cudaMalloc of the segment queue failed");
  if (fresh) CUDA_TRY(cudaMemsetAsync(g_ws.segq.p, 0, 256, st));
  q->ctrl = (unsigned*)g_ws.segq.p;
  q->head = (unsigned*)((char*)g_ws.segq.p + 256);
  q->tail = q->head + 2048;
  q->park = q->tail + 2048;
  q->n_park = (g_opt_boost != 1 && subparts <= 2048) ? (int32_t)subparts : 0;
  q->boost_div = g_opt_boost >= 2 ? g_opt_boost : 2;
  q->boost_two = g_opt_boost2 != 1 ? 1 : 0;
  q->slots = (int*)((char*)g_ws.segq.p + 256 + lvl_bytes);
  q->ckpt = (double*)((char*)g_ws.segq.p + 256 + lvl_bytes + slot_bytes);
  return AFM_OK;
}

int run_integrate_f64(const ModelConsts& mc_in, const IntegrateIO& io, int block,
                      int variant, cudaStream_t st) {
  SegQueue q;
  int workers = 0;
  bool use_q = false;
  const bool eligible = variant == 0 && block == 32;
  // The queue kernels run 2 to 5 one-warp CTAs per sub-partition, so there is shared
  // memory for longer time tiles (fewer barrier waits and bulk copies per step;
  // configs[1]: 64 rows 12.31 ms, 128: 12.21, 256: 12.15, and 512 rows no longer
  // fit 12 CTAs per SM: 18.1 ms).  The tile length changes no FP64 result (the
  // misfit is summed step by step); the FP32 kernel folds its sum once per tile and
  // keeps its own tile length.
  ModelConsts mc = mc_in;
  const int per_sub = queue_per_sub(io.per, io.n_traces, mc.N, eligible, 0);
  if (per_sub > 0 && g_opt_tile == 0) {
    int T = per_sub <= 3 ? 256 : (per_sub <= 5 ? 128 : 64);
    if (T > mc.N) T = mc.N;
    if (T > mc.T) {
      mc.T = T;
      mc.n_tiles = (mc.N + T - 1) / T;
    }
  }
  int rc = make_queue(io.per, io.n_traces, mc.n_tiles, mc.T, eligible, &q, &workers,
                      &use_q, st, 4, 0, per_sub);
  if (rc) return rc;
  if (!use_q) mc = mc_in;
  // the queue is reset before the start event: the pair brackets one kernel
  if (use_q) LAUNCHED(launch_segq_init(q, st));
  if ((rc = kev_record(0, st))) return rc;
  if (use_q)
    LAUNCHED(launch_integrate_f64_q(mc, io, q, workers, st));
  else
    LAUNCHED(launch_integrate_f64(mc, io, block, variant, st));
  g_last_kernel = use_q ? "integrate_misfit_f64_q" : "integrate_misfit_f64";
  return kev_record(1, st);
}

int run_integrate_f32(const ModelConstsF32& mf, const IntegrateIO& io, int block,
                      int ppt, cudaStream_t st) {
  SegQueue q;
  int workers = 0;
  bool use_q = false;
  int rc = make_queue(io.per, io.n_traces, mf.n_tiles, mf.T, ppt == 1 && block == 32, &q,
                      &workers, &use_q, st);
  if (rc) return rc;
  if (use_q) LAUNCHED(launch_segq_init(q, st));
  if ((rc = kev_record(0, st))) return rc;
  if (use_q)
    LAUNCHED(launch_integrate_f32_q(mf, io, q, workers, st));
  else
    LAUNCHED(launch_integrate_f32(mf, io, block, ppt, st));
  g_last_kernel = use_q ? "integrate_misfit_f32_q" : "integrate_misfit_f32";
  return kev_record(1, st);
}

// After a stream synchronisation: did a queue worker give up waiting (a
// corrupted queue; see segq_pop)?  The flag is sticky until read here.
int check_queue_flag(cudaStream_t st) {
  if (!g_ws.segq.p) return AFM_OK;
  unsigned flag = 0;
  CUDA_TRY(cudaMemcpyAsync(&flag, (char*)g_ws.segq.p + 8, 4, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (!flag) return AFM_OK;
  CUDA_TRY(cudaMemsetAsync((char*)g_ws.segq.p + 8, 0, 4, st));
  return fail(AFM_ECUDA, "segment queue timed out: results of the last batch are invalid");
}

BoxDev make_box(const afm_bounds* b, int D) {
  BoxDev bd;
  memset(&bd, 0, sizeof(bd));
  for (int j = 0; j < D && j < 4; ++j) {
    bd.lo[j] = b->lo[j];
    bd.hi[j] = b->hi[j];
    bd.lg[j] = b->log10_scale[j] ? 1 : 0;
  }
  return bd;
}

int validate_bounds(const afm_bounds* b, int D) {
  if (!b) return fail(AFM_EINVAL, "bounds is NULL");
  for (int j = 0; j < D; ++j)
    if (!isfinite(b->lo[j]) || !isfinite(b->hi[j]) || !(b->lo[j] <= b->hi[j]))
      return fail(AFM_EINVAL, "bounds[%d] = [%g, %g] is not a finite interval",
                  j, b->lo[j], b->hi[j]);
  return AFM_OK;
}

int validate_swarm(const afm_swarm_cfg* s) {
  if (!s) return fail(AFM_EINVAL, "swarm is NULL");
  if (s->n_particles < 1 || s->n_iters < 1)
    return fail(AFM_EINVAL, "n_particles and n_iters must be >= 1");
  if (!isfinite(s->w) || !isfinite(s->c1) || !isfinite(s->c2))
    return fail(AFM_EINVAL, "w, c1, c2 must be finite");
  if (s->topology != 0 && s->topology != 1)
    return fail(AFM_EINVAL, "topology must be 0 (global best) or 1 (ring of three)");
  if (s->async_chunk < 0) return fail(AFM_EINVAL, "async_chunk must be >= 0");
  return AFM_OK;
}

// Entry points that step a swarm batch by batch from outside have no place for the
// chunked, asynchronous swarm.
int reject_async(const afm_swarm_cfg* s, const char* who) {
  if (s->async_chunk > 0 && s->async_chunk < s->n_particles)
    return fail(AFM_EUNSUPPORTED, "%s: the asynchronous swarm (async_chunk) runs inside "
                                  "afm_pso_invert only", who);
  return AFM_OK;
}

// Forward batch on device buffers with the workspace lock already held.
int forward_locked(const double* params, int64_t P, const double* trace,
                   const afm_cfg* cfg, const double* z0v0, double* misfit,
                   cudaStream_t st) {
  const bool f32 = (cfg->precision == AFM_F32);
  const int64_t per = P / cfg->n_traces;
  const int block = block_threads();
  const int ppt = particles_per_thread();
  ModelConsts mc;
  ModelConstsF32 mf;
  make_consts(cfg, block, &mc);
  make_consts_f32(cfg, &mf);
  int rc = acquire_ws(st);
  if (rc) return rc;
  const size_t stream_bytes = (size_t)cfg->n_traces * mc.N * (f32 ? 16 : 32);
  if (g_ws.stream.ensure(stream_bytes + 64))
    return fail(AFM_ECUDA, "cudaMalloc of %zu B time-tile stream failed",
                stream_bytes);
  if (f32)
    LAUNCHED(launch_build_stream_f32(mf, trace, cfg->n_traces,
                                     (float*)g_ws.stream.p, st));
  else
    LAUNCHED(launch_build_stream(mc, trace, cfg->n_traces,
                                 (double*)g_ws.stream.p, st));
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = params;
  io.z0v0 = z0v0;
  io.stream = (const double*)g_ws.stream.p;
  io.J = misfit;
  io.per = per;
  io.n_traces = cfg->n_traces;
  io.mode = 0;
  io.lanes = pick_lanes(cfg, per, cfg->n_traces);
  Packed pk;
  if ((rc = pack_inputs(cfg, params, z0v0, per, cfg->n_traces, nullptr, &pk, st)))
    return rc;
  if (pk.order) {
    io.params = pk.params;
    io.z0v0 = pk.z0v0;
    io.J = pk.J;
  }
  if (f32)
    rc = run_integrate_f32(mf, io, block, ppt, st);
  else
    rc = run_integrate_f64(mc, io, block, pick_variant(io.per, io.n_traces, ppt), st);
  if (rc) return rc;
  if (pk.order) LAUNCHED(launch_pack_scatter(pk.order, pk.J, P, misfit, st));
  return release_ws(st);
}

int validate_forward(const double* params, int64_t P, const double* trace,
                     const afm_cfg* cfg, double* misfit) {
  int rc = validate_cfg(cfg);
  if (rc) return rc;
  if (P < 1) return fail(AFM_EINVAL, "n_particles must be >= 1");
  if (P % cfg->n_traces)
    return fail(AFM_EINVAL, "n_particles %lld is not a multiple of n_traces %d",
                (long long)P, cfg->n_traces);
  if (!trace || !misfit) return fail(AFM_EINVAL, "trace/misfit is NULL");
  if (!params && cfg->n_params > 0) return fail(AFM_EINVAL, "params is NULL");
  return AFM_OK;
}

}  // namespace

// =================================================================================
extern "C" {

int afm_forward_batch(const double* params, int64_t n_particles,
                      const double* trace, const afm_cfg* cfg,
                      const double* z0v0, double* misfit, void* cuda_stream) {
  int rc = validate_forward(params, n_particles, trace, cfg, misfit);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  return forward_locked(params, n_particles, trace, cfg, z0v0, misfit,
                        (cudaStream_t)cuda_stream);
}

int afm_forward_batch_host(const double* params, int64_t n_particles,
                           const double* trace, const afm_cfg* cfg,
                           const double* z0v0, double* misfit,
                           void* cuda_stream) {
  int rc = validate_forward(params, n_particles, trace, cfg, misfit);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  const int D = cfg->n_params;
  const int64_t W =
      (int64_t)cfg->steps_per_cycle * (cfg->n_cycles - cfg->n_skip_cycles);
  const size_t pb = (size_t)n_particles * (D > 0 ? D : 1) * 8;
  const size_t tb = (size_t)cfg->n_traces * W * 8;
  const size_t zb = (size_t)n_particles * 16;
  const size_t mb = (size_t)n_particles * 8;
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.h_params.ensure(pb) || g_ws.h_trace.ensure(tb) ||
      g_ws.h_misfit.ensure(mb) || (z0v0 && g_ws.h_z0v0.ensure(zb)))
    return fail(AFM_ECUDA, "cudaMalloc of staging buffers failed");
  if (D > 0)
    CUDA_TRY(cudaMemcpyAsync(g_ws.h_params.p, params, (size_t)n_particles * D * 8,
                             cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(g_ws.h_trace.p, trace, tb, cudaMemcpyHostToDevice, st));
  if (z0v0)
    CUDA_TRY(cudaMemcpyAsync(g_ws.h_z0v0.p, z0v0, zb, cudaMemcpyHostToDevice, st));
  g_ws.last_stream = st;  // same stream: no self-wait
  rc = forward_locked((const double*)g_ws.h_params.p, n_particles,
                      (const double*)g_ws.h_trace.p, cfg,
                      z0v0 ? (const double*)g_ws.h_z0v0.p : nullptr,
                      (double*)g_ws.h_misfit.p, st);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(misfit, g_ws.h_misfit.p, mb, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return check_queue_flag(st);
}

int afm_pso_shard_init(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       int32_t n_dims, int32_t n_traces, uint64_t seed,
                       int64_t first_particle, double* x, double* v,
                       double* pbest, double* pbestJ, double* gbest,
                       double* gbestJ, void* cuda_stream) {
  if (first_particle < 0) return fail(AFM_EINVAL, "first_particle must be >= 0");
  if (n_dims < 1 || n_dims > 4) return fail(AFM_EINVAL, "n_dims must be 1..4");
  if (n_traces < 1) return fail(AFM_EINVAL, "n_traces must be >= 1");
  int rc = validate_bounds(bounds, n_dims);
  if (rc) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if (!x || !v || !pbest || !pbestJ || !gbest || !gbestJ)
    return fail(AFM_EINVAL, "NULL swarm array");
  if ((rc = check_device())) return rc;
  LAUNCHED(launch_pso_init(make_box(bounds, n_dims), n_dims, swarm->n_particles,
                           n_traces, seed, first_particle, x, v, pbest, pbestJ,
                           gbest, gbestJ, (cudaStream_t)cuda_stream));
  return AFM_OK;
}

int afm_pso_init(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                 int32_t n_dims, int32_t n_traces, uint64_t seed, double* x,
                 double* v, double* pbest, double* pbestJ, double* gbest,
                 double* gbestJ, void* cuda_stream) {
  return afm_pso_shard_init(bounds, swarm, n_dims, n_traces, seed, 0, x, v,
                            pbest, pbestJ, gbest, gbestJ, cuda_stream);
}

// afm_pso_step on device arrays, arguments validated, workspace lock held.
static int pso_step_locked(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                           int32_t n_dims, int32_t n_traces, uint64_t seed,
                           int32_t iteration, int32_t do_move, const double* J,
                           double* x, double* v, double* pbest, double* pbestJ,
                           double* gbest, double* gbestJ, cudaStream_t st) {
  int rc;
  const int64_t per = swarm->n_particles;
  const int block = 128;
  const int bpt = blocks_per_trace(per, block);
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.cand.ensure((size_t)bpt * n_traces * sizeof(Cand)))
    return fail(AFM_ECUDA, "cudaMalloc of candidates failed");
  BoxDev box = make_box(bounds, n_dims);
  SwarmDev sw = {swarm->w, swarm->c1, swarm->c2, swarm->topology, 0};
  LAUNCHED(launch_pso_best(n_dims, per, 0, per, n_traces, const_cast<double*>(J), nullptr,
                           x, pbest, pbestJ, (Cand*)g_ws.cand.p, block, st));
  LAUNCHED(launch_pso_gbest(box, n_dims, n_traces, bpt, (Cand*)g_ws.cand.p,
                            pbest, gbest, gbestJ, nullptr, nullptr, nullptr, st));
  if (do_move)
    LAUNCHED(launch_pso_move(box, sw, n_dims, per, 0, per, n_traces, seed, 0,
                             (uint32_t)iteration, 1, RingEdges{0, 0, nullptr, nullptr, 0}, J, x, v, pbest,
                             pbestJ, gbest, nullptr, st));
  return release_ws(st);
}

static int validate_pso_step(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                             int32_t n_dims, int32_t n_traces, int32_t iteration,
                             const double* J, const double* x, const double* v,
                             const double* pbest, const double* pbestJ,
                             const double* gbest, const double* gbestJ) {
  if (n_dims < 1 || n_dims > 4) return fail(AFM_EINVAL, "n_dims must be 1..4");
  if (n_traces < 1) return fail(AFM_EINVAL, "n_traces must be >= 1");
  if (iteration < 0) return fail(AFM_EINVAL, "iteration must be >= 0");
  int rc = validate_bounds(bounds, n_dims);
  if (rc) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if ((rc = reject_async(swarm, "afm_pso_step"))) return rc;
  if (!J || !x || !v || !pbest || !pbestJ || !gbest || !gbestJ)
    return fail(AFM_EINVAL, "NULL swarm array");
  return AFM_OK;
}

int afm_pso_step(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                 int32_t n_dims, int32_t n_traces, uint64_t seed,
                 int32_t iteration, int32_t do_move, const double* J, double* x,
                 double* v, double* pbest, double* pbestJ, double* gbest,
                 double* gbestJ, void* cuda_stream) {
  int rc = validate_pso_step(bounds, swarm, n_dims, n_traces, iteration, J, x, v, pbest,
                             pbestJ, gbest, gbestJ);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  return pso_step_locked(bounds, swarm, n_dims, n_traces, seed, iteration, do_move, J, x,
                         v, pbest, pbestJ, gbest, gbestJ, (cudaStream_t)cuda_stream);
}

static int pso_invert_locked(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                             uint64_t seed, const double* trace,
                             const afm_cfg* cfg, double* theta_star,
                             double* J_star, double* swarm_dump,
                             double* gbest_hist, int32_t* n_iters_done,
                             cudaStream_t st) {
  const bool f32 = (cfg->precision == AFM_F32);
  const int D = cfg->n_params;
  const int T = cfg->n_traces;
  const int64_t per = swarm->n_particles;
  const int64_t PT = per * T;
  const int block = block_threads();
  const int ppt = particles_per_thread();
  const int lanes = pick_lanes(cfg, per, T);
  const int bpt = f32 ? blocks_per_trace(per, block * ppt)
                      : integrate_bpt(per, block, ppt, pick_variant(per, T, ppt), lanes);
  ModelConsts mc;
  ModelConstsF32 mf;
  make_consts(cfg, block, &mc);
  make_consts_f32(cfg, &mf);
  int rc = acquire_ws(st);
  if (rc) return rc;

  // workspace carve-up (doubles): x, v, pbest [PT][D]; J, pbestJ [PT];
  // gbest [T][D]; gbestJ [T]; theta* [T][D]; J* [T]
  const size_t n_dbl = (size_t)PT * (3 * D + 2) + (size_t)T * (2 * D + 2);
  if (g_ws.swarm.ensure(n_dbl * 8) ||
      g_ws.cand.ensure((size_t)(bpt + blocks_per_trace(per, 128)) * T * sizeof(Cand)) ||
      g_ws.stream.ensure((size_t)T * mc.N * 32 + 64))
    return fail(AFM_ECUDA, "cudaMalloc of the PSO workspace failed");
  double* x = (double*)g_ws.swarm.p;
  double* v = x + PT * D;
  double* pbest = v + PT * D;
  double* J = pbest + PT * D;
  double* pbestJ = J + PT;
  double* gbest = pbestJ + PT;
  double* gbestJ = gbest + (size_t)T * D;
  double* th_dev = gbestJ + T;
  double* Js_dev = th_dev + (size_t)T * D;
  if ((rc = ensure_pinned((size_t)T * 8))) return rc;

  BoxDev box = make_box(bounds, D);
  SwarmDev sw = {swarm->w, swarm->c1, swarm->c2, swarm->topology, 0};

  if (f32)
    LAUNCHED(launch_build_stream_f32(mf, trace, T, (float*)g_ws.stream.p, st));
  else
    LAUNCHED(launch_build_stream(mc, trace, T, (double*)g_ws.stream.p, st));
  LAUNCHED(launch_pso_init(box, D, per, T, seed, 0, x, v, pbest, pbestJ, gbest,
                           gbestJ, st));
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = x;
  io.z0v0 = nullptr;
  io.stream = (const double*)g_ws.stream.p;
  io.J = J;
  io.pbest = pbest;
  io.pbestJ = pbestJ;
  io.cand = (Cand*)g_ws.cand.p;
  io.box = box;
  io.per = per;
  io.n_traces = T;
  io.mode = 1;
  io.lanes = lanes;

  // Asynchronous swarm (R25): chunks of `chunk` particles of every swarm,
  // in index order; a chunk is integrated on its own (theta = map(x) gathered into a
  // compact batch for the forward-only kernel), its personal bests and the swarm's
  // best are updated from it, and it moves at once.
  const int64_t chunk =
      (swarm->async_chunk > 0 && swarm->async_chunk < per) ? swarm->async_chunk : per;
  const bool asynchronous = chunk < per;
  double* th_c = nullptr;  // [T][chunk][D]
  double* J_c = nullptr;   // [T][chunk]
  if (asynchronous) {
    const size_t a256 = 255;
    const size_t th_bytes = ((size_t)T * chunk * D * 8 + a256) & ~a256;
    if (g_ws.chunk.ensure(th_bytes + (size_t)T * chunk * 8))
      return fail(AFM_ECUDA, "cudaMalloc of the chunk workspace failed");
    th_c = (double*)g_ws.chunk.p;
    J_c = (double*)((char*)g_ws.chunk.p + th_bytes);
  }
  const RingEdges no_edges = {0, 0, nullptr, nullptr, 0};

  int done = 0;
  for (int it = 0; it < swarm->n_iters; ++it) {
    const bool last = (it == swarm->n_iters - 1);
    double* hist_row = gbest_hist ? gbest_hist + (size_t)it * T * (D + 1) : nullptr;
    double* dump_row =
        swarm_dump ? swarm_dump + (size_t)it * PT * (3 * D + 2) : nullptr;
    if (asynchronous) {
      for (int64_t c0 = 0; c0 < per; c0 += chunk) {
        const int64_t cn = (c0 + chunk < per) ? chunk : per - c0;
        const bool last_chunk = (c0 + cn == per);
        LAUNCHED(launch_chunk_gather(box, D, per, c0, cn, T, x, th_c, st));
        IntegrateIO ioc = io;
        ioc.params = th_c;
        ioc.J = J_c;
        ioc.per = cn;
        ioc.mode = 0;
        ioc.lanes = pick_lanes(cfg, cn, T);
        if (f32)
          rc = run_integrate_f32(mf, ioc, block, ppt, st);
        else
          rc = run_integrate_f64(mc, ioc, block, pick_variant(cn, T, ppt), st);
        if (rc) return rc;
        LAUNCHED(launch_pso_best(D, per, c0, cn, T, J, J_c, x, pbest, pbestJ,
                                 (Cand*)g_ws.cand.p, 128, st));
        LAUNCHED(launch_pso_gbest(box, D, T, blocks_per_trace(cn, 128), (Cand*)g_ws.cand.p,
                                  pbest, gbest, gbestJ, last_chunk ? hist_row : nullptr,
                                  th_dev, Js_dev, st));
        if (!last || dump_row)
          LAUNCHED(launch_pso_move(box, sw, D, per, c0, cn, T, seed, 0, (uint32_t)it,
                                   last ? 0 : 1, no_edges, J, x, v, pbest, pbestJ, gbest,
                                   dump_row, st));
      }
    } else {
      // throughput regime, DMT laws: warp packing (afm_sort.cu).  The swarm state
      // stays in particle order; theta = map(x) is gathered in packed order, the
      // forward-only kernel runs on it, the misfits are scattered back and the
      // stand-alone personal-best kernel takes the place of the fused epilogue.
      Packed pk;
      if ((rc = pack_inputs(cfg, x, nullptr, per, T, &box, &pk, st))) return rc;
      int n_cand = bpt;
      if (pk.order) {
        IntegrateIO iof = io;
        iof.params = pk.params;
        iof.J = pk.J;
        iof.mode = 0;
        if (f32)
          rc = run_integrate_f32(mf, iof, block, ppt, st);
        else
          rc = run_integrate_f64(mc, iof, block, pick_variant(iof.per, iof.n_traces, ppt),
                                 st);
        if (rc) return rc;
        LAUNCHED(launch_pack_scatter(pk.order, pk.J, PT, J, st));
        n_cand = blocks_per_trace(per, 128);
        LAUNCHED(launch_pso_best(D, per, 0, per, T, J, nullptr, x, pbest, pbestJ,
                                 (Cand*)g_ws.cand.p, 128, st));
      } else {
        if (f32)
          rc = run_integrate_f32(mf, io, block, ppt, st);
        else
          rc = run_integrate_f64(mc, io, block, pick_variant(io.per, io.n_traces, ppt), st);
        if (rc) return rc;
      }
      LAUNCHED(launch_pso_gbest(box, D, T, n_cand, (Cand*)g_ws.cand.p, pbest, gbest, gbestJ,
                                hist_row, th_dev, Js_dev, st));
    }
    // cost cutoff (R24): once per batch, after the best updates
    bool stop = last;
    if (!stop && swarm->j_target > 0) {
      double* hJ = (double*)g_ws.pinned;
      CUDA_TRY(cudaMemcpyAsync(hJ, gbestJ, (size_t)T * 8, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(cudaStreamSynchronize(st));
      stop = true;
      for (int s = 0; s < T; ++s)
        if (!(hJ[s] <= swarm->j_target)) stop = false;
    }
    if (!asynchronous && (!stop || dump_row))
      LAUNCHED(launch_pso_move(box, sw, D, per, 0, per, T, seed, 0, (uint32_t)it,
                               stop ? 0 : 1, no_edges, J, x, v, pbest, pbestJ, gbest,
                               dump_row, st));
    done = it + 1;
    if (stop) break;
  }
  CUDA_TRY(cudaMemcpyAsync(theta_star, th_dev, (size_t)T * D * 8,
                           cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(J_star, Js_dev, (size_t)T * 8, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (n_iters_done) *n_iters_done = done;
  if ((rc = check_queue_flag(st))) return rc;
  return release_ws(st);
}

static int validate_invert(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                           const double* trace, const afm_cfg* cfg,
                           double* theta_star, double* J_star) {
  int rc = validate_cfg(cfg);
  if (rc) return rc;
  if (cfg->n_params < 1)
    return fail(AFM_EINVAL, "nothing to invert: n_params = 0");
  if ((rc = validate_bounds(bounds, cfg->n_params))) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if (!trace || !theta_star || !J_star)
    return fail(AFM_EINVAL, "trace/theta_star/J_star is NULL");
  return AFM_OK;
}

int afm_pso_invert(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                   uint64_t seed, const double* trace, const afm_cfg* cfg,
                   double* theta_star, double* J_star, double* swarm_dump,
                   double* gbest_hist, int32_t* n_iters_done,
                   void* cuda_stream) {
  int rc = validate_invert(bounds, swarm, trace, cfg, theta_star, J_star);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  return pso_invert_locked(bounds, swarm, seed, trace, cfg, theta_star, J_star,
                           swarm_dump, gbest_hist, n_iters_done,
                           (cudaStream_t)cuda_stream);
}

int afm_pso_invert_host(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                        uint64_t seed, const double* trace, const afm_cfg* cfg,
                        double* theta_star, double* J_star,
                        int32_t* n_iters_done, void* cuda_stream) {
  int rc = validate_invert(bounds, swarm, trace, cfg, theta_star, J_star);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  const int64_t W =
      (int64_t)cfg->steps_per_cycle * (cfg->n_cycles - cfg->n_skip_cycles);
  const size_t tb = (size_t)cfg->n_traces * W * 8;
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.h_trace.ensure(tb))
    return fail(AFM_ECUDA, "cudaMalloc of the trace staging buffer failed");
  CUDA_TRY(cudaMemcpyAsync(g_ws.h_trace.p, trace, tb, cudaMemcpyHostToDevice, st));
  g_ws.last_stream = st;
  return pso_invert_locked(bounds, swarm, seed, (const double*)g_ws.h_trace.p,
                           cfg, theta_star, J_star, nullptr, nullptr,
                           n_iters_done, st);
}

int afm_pso_shard_eval(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       const double* trace, const afm_cfg* cfg,
                       int64_t first_particle, const double* x, double* J,
                       double* pbest, double* pbestJ, double* cand_out,
                       void* cuda_stream) {
  int rc = validate_cfg(cfg);
  if (rc) return rc;
  if (cfg->n_params < 1) return fail(AFM_EINVAL, "n_params = 0");
  if ((rc = validate_bounds(bounds, cfg->n_params))) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if ((rc = reject_async(swarm, "afm_pso_shard_eval"))) return rc;
  if (first_particle < 0) return fail(AFM_EINVAL, "first_particle must be >= 0");
  if (!trace || !x || !J || !pbest || !pbestJ || !cand_out)
    return fail(AFM_EINVAL, "NULL array");
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  const bool f32 = (cfg->precision == AFM_F32);
  const int D = cfg->n_params, T = cfg->n_traces;
  const int64_t per = swarm->n_particles;
  const int block = block_threads();
  const int ppt = particles_per_thread();
  const int lanes = pick_lanes(cfg, per, T);
  const int bpt = f32 ? blocks_per_trace(per, block * ppt)
                      : integrate_bpt(per, block, ppt, pick_variant(per, T, ppt), lanes);
  ModelConsts mc;
  ModelConstsF32 mf;
  make_consts(cfg, block, &mc);
  make_consts_f32(cfg, &mf);
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.cand.ensure((size_t)bpt * T * sizeof(Cand)) ||
      g_ws.stream.ensure((size_t)T * mc.N * 32 + 64))
    return fail(AFM_ECUDA, "cudaMalloc of the shard workspace failed");
  if (f32)
    LAUNCHED(launch_build_stream_f32(mf, trace, T, (float*)g_ws.stream.p, st));
  else
    LAUNCHED(launch_build_stream(mc, trace, T, (double*)g_ws.stream.p, st));
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = x;
  io.stream = (const double*)g_ws.stream.p;
  io.J = J;
  io.pbest = pbest;
  io.pbestJ = pbestJ;
  io.cand = (Cand*)g_ws.cand.p;
  io.box = make_box(bounds, D);
  io.per = per;
  io.n_traces = T;
  io.mode = 1;
  io.lanes = lanes;
  if (f32)
    rc = run_integrate_f32(mf, io, block, ppt, st);
  else
    rc = run_integrate_f64(mc, io, block, pick_variant(io.per, io.n_traces, ppt), st);
  if (rc) return rc;
  LAUNCHED(launch_pso_shard_cand(D, T, bpt, first_particle, per, swarm->topology == 1,
                                 (Cand*)g_ws.cand.p, pbest, pbestJ, cand_out, st));
  return release_ws(st);
}

int afm_pso_shard_move(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                       int32_t n_dims, int32_t n_traces, uint64_t seed,
                       int32_t iteration, int32_t do_move,
                       int64_t first_particle, const double* gathered,
                       int32_t n_ranks, int32_t rank, int64_t swarm_particles,
                       double* x, double* v, const double* pbest,
                       const double* pbestJ, double* gbest, double* gbestJ,
                       double* theta_star, double* J_star, void* cuda_stream) {
  if (n_dims < 1 || n_dims > 4) return fail(AFM_EINVAL, "n_dims must be 1..4");
  if (n_traces < 1) return fail(AFM_EINVAL, "n_traces must be >= 1");
  if (n_ranks < 1) return fail(AFM_EINVAL, "n_ranks must be >= 1");
  if (rank < 0 || rank >= n_ranks) return fail(AFM_EINVAL, "rank must be in [0, n_ranks)");
  if (iteration < 0) return fail(AFM_EINVAL, "iteration must be >= 0");
  if (first_particle < 0) return fail(AFM_EINVAL, "first_particle must be >= 0");
  int rc = validate_bounds(bounds, n_dims);
  if (rc) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if ((rc = reject_async(swarm, "afm_pso_shard_move"))) return rc;
  if (swarm_particles < swarm->n_particles)
    return fail(AFM_EINVAL, "swarm_particles %lld is smaller than the shard's %d",
                (long long)swarm_particles, swarm->n_particles);
  if (!gathered || !x || !v || !pbest || !gbest || !gbestJ)
    return fail(AFM_EINVAL, "NULL swarm array");
  const bool ring = (swarm->topology == 1);
  if (ring && !pbestJ) return fail(AFM_EINVAL, "the ring topology needs pbestJ");
  if (ring && swarm_particles > swarm->n_particles && n_traces != 1)
    return fail(AFM_EINVAL, "a swarm split over ranks is one trace per call");
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  BoxDev box = make_box(bounds, n_dims);
  SwarmDev sw = {swarm->w, swarm->c1, swarm->c2, swarm->topology, 0};
  const int width = ring ? 3 * n_dims + 4 : n_dims + 2;
  LAUNCHED(launch_pso_shard_gbest(box, n_dims, n_traces, n_ranks, width, gathered, gbest,
                                  gbestJ, theta_star, J_star, st));
  if (do_move) {
    RingEdges re = {0, 0, nullptr, nullptr, 0};
    if (ring && swarm_particles > swarm->n_particles) {
      // the neighbours of the shard's edge particles: last particle of the rank
      // before, first particle of the rank after (ranks hold consecutive slices)
      const int before = (rank + n_ranks - 1) % n_ranks, after = (rank + 1) % n_ranks;
      re.total = swarm_particles;
      re.off = first_particle % swarm_particles;
      re.stride = width;
      re.left = gathered + (size_t)before * n_traces * width + (n_dims + 2) + (n_dims + 1);
      re.right = gathered + (size_t)after * n_traces * width + (n_dims + 2);
    }
    LAUNCHED(launch_pso_move(box, sw, n_dims, swarm->n_particles, 0, swarm->n_particles,
                             n_traces, seed, first_particle, (uint32_t)iteration, 1, re,
                             nullptr, x, v, pbest, pbestJ, gbest, nullptr, st));
  }
  return AFM_OK;
}

// ---- multi-mode beam ------------------------------------------------------------
static int validate_beam(const afm_beam_cfg* c) {
  if (!c) return fail(AFM_EINVAL, "beam cfg is NULL");
  if (c->law < AFM_LAW_NONE || c->law > AFM_LAW_KELVIN_VOIGT)
    return fail(AFM_EINVAL, "unknown law %d", c->law);
  if (c->law == AFM_LAW_NONE) {
    if (c->n_params < 0 || c->n_params > 4)
      return fail(AFM_EINVAL, "n_params %d out of range 0..4", c->n_params);
  } else if (c->n_params != law_dims(c->law)) {
    return fail(AFM_EINVAL, "law %d needs n_params = %d", c->law, law_dims(c->law));
  }
  if (!(c->L > 0) || !(c->E > 0) || !(c->I > 0) || !(c->mu > 0) || !(c->Q > 0) ||
      !(c->f_drive > 0) || !(c->A_ref > 0) || !isfinite(c->A_base) ||
      !isfinite(c->z_c))
    return fail(AFM_EINVAL, "L, E, I, mu, Q, f_drive, A_ref must be positive");
  if ((c->law == AFM_LAW_DMT || c->law == AFM_LAW_DMT_VISC) &&
      (!(c->R > 0) || !(c->a0 > 0)))
    return fail(AFM_EINVAL, "DMT laws need R > 0 and a0 > 0");
  if (c->n_modes != 1 && c->n_modes != 2 && c->n_modes != 4 && c->n_modes != 8)
    return fail(AFM_EINVAL, "n_modes must be 1, 2, 4 or 8");
  if (c->n_points < 3 || !(c->n_points & 1) || c->n_points > 100001)
    return fail(AFM_EINVAL, "n_points must be odd, 3..100001");
  if (c->steps_per_cycle < 1 || c->n_cycles < 1)
    return fail(AFM_EINVAL, "steps_per_cycle and n_cycles must be >= 1");
  if (c->n_skip_cycles < 0 || c->n_skip_cycles >= c->n_cycles)
    return fail(AFM_EINVAL, "need 0 <= n_skip_cycles < n_cycles");
  if ((int64_t)c->steps_per_cycle * c->n_cycles > (int64_t)1 << 30)
    return fail(AFM_EINVAL, "more than 2^30 steps");
  if (c->n_traces < 1) return fail(AFM_EINVAL, "n_traces must be >= 1");
  return AFM_OK;
}

// Initialisation kernel -> host copy of the modal constants, then the scaled
// force-law factors with m = m_1.  Workspace lock held.
static int beam_prepare(const afm_beam_cfg* c, BeamConsts* bc, BeamModeConsts* mo,
                        cudaStream_t st) {
  const double w = 2.0 * M_PI * c->f_drive;
  const double h = 2.0 * M_PI / (w * (double)c->steps_per_cycle);
  if (g_ws.scratch.ensure(sizeof(BeamModeConsts) + 64))
    return fail(AFM_ECUDA, "cudaMalloc failed");
  BeamModeConsts* dmo = (BeamModeConsts*)((char*)g_ws.scratch.p + 64);
  CUDA_TRY(cudaMemsetAsync(dmo, 0, sizeof(BeamModeConsts), st));
  LAUNCHED(launch_beam_setup(*c, h, dmo, st));
  CUDA_TRY(cudaMemcpyAsync(mo, dmo, sizeof(BeamModeConsts), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  memset(bc, 0, sizeof(*bc));
  const double m = mo->m1;
  const double sqR = sqrt(c->R > 0 ? c->R : 0.0);
  bc->h = h;
  bc->w_drive = w;
  bc->zc = c->z_c;
  bc->a0 = c->a0;
  bc->inv_a0sq = (c->a0 > 0) ? 1.0 / (c->a0 * c->a0) : 0.0;
  bc->c_vdw = h * h * c->R / (6.0 * m);
  bc->c_hertz = h * h * (4.0 / 3.0) * sqR / m;
  bc->c_visc = h * sqR / m;
  bc->c_force = h * h / m;
  bc->c_damp = h / m;
  bc->u_max = 100.0 * c->A_ref;
  bc->law = c->law;
  bc->D = c->n_params;
  bc->M = c->n_modes;
  bc->N = c->steps_per_cycle * c->n_cycles;
  bc->W = c->steps_per_cycle * (c->n_cycles - c->n_skip_cycles);
  bc->n0 = bc->N - bc->W;
  int T = g_opt_tile > 0 ? g_opt_tile : 64;
  if (T > bc->N) T = bc->N;
  bc->T = T;
  bc->n_tiles = (bc->N + T - 1) / T;
  return AFM_OK;
}

// The beam integrate kernel with or without the segment queue (make_queue decides).
static int run_beam_integrate(const BeamConsts& bc, const BeamModeConsts& mo,
                              const IntegrateIO& io, int block, cudaStream_t st) {
  SegQueue q;
  int workers = 0;
  bool use_q = false;
  // 65 536 particles (3.46 chains per sub-partition): 71.5 -> 56.9 ms with the queue;
  // 1 048 576 particles: 886 ms without, 900 ms with it (three of these 166-register
  // warps saturate a sub-partition and the checkpoint is 144 B per particle)
  int rc = make_queue(io.per, io.n_traces, bc.n_tiles, bc.T, block == 32, &q, &workers,
                      &use_q, st, 2 * bc.M + 2, 8);
  if (rc) return rc;
  if (use_q)
    LAUNCHED(launch_beam_integrate_q(bc, mo, io, q, workers, st));
  else
    LAUNCHED(launch_beam_integrate(bc, mo, io, block, st));
  g_last_kernel = use_q ? "beam_integrate_f64_q" : "beam_integrate_f64";
  return AFM_OK;
}

// cos(w t) at the three abscissae of every step + the trace: the point-mass
// stream builder with unit amplitude and no offsets.
static int beam_stream(const BeamConsts& bc, const double* trace, int n_traces,
                       cudaStream_t st) {
  ModelConsts mc;
  memset(&mc, 0, sizeof(mc));
  mc.h = bc.h;
  mc.w_drive = bc.w_drive;
  mc.drive_amp = 1.0;
  mc.N = bc.N;
  mc.W = bc.W;
  mc.n0 = bc.n0;
  if (g_ws.stream.ensure((size_t)n_traces * bc.N * 32 + 64))
    return fail(AFM_ECUDA, "cudaMalloc of the time-tile stream failed");
  LAUNCHED(launch_build_stream(mc, trace, n_traces, (double*)g_ws.stream.p, st));
  return AFM_OK;
}

int afm_beam_modes(const afm_beam_cfg* cfg, double* beta_L, double* omega,
                   double* phi_L, double* participation, double* compliance,
                   void* cuda_stream) {
  int rc = validate_beam(cfg);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  BeamConsts bc;
  BeamModeConsts mo;
  if ((rc = beam_prepare(cfg, &bc, &mo, st))) return rc;
  for (int i = 0; i < cfg->n_modes; ++i) {
    if (beta_L) beta_L[i] = mo.bL[i];
    if (omega) omega[i] = mo.omega[i];
    if (phi_L) phi_L[i] = mo.phiL[i];
    if (participation) participation[i] = mo.part[i];
    if (compliance) compliance[i] = mo.compl_[i];
  }
  return release_ws(st);
}

int afm_beam_forward_batch(const double* params, int64_t n_particles,
                           const double* trace, const afm_beam_cfg* cfg,
                           const afm_bounds* bounds, double* misfit,
                           void* cuda_stream) {
  int rc = validate_beam(cfg);
  if (rc) return rc;
  if (n_particles < 1 || n_particles % cfg->n_traces)
    return fail(AFM_EINVAL, "n_particles must be a positive multiple of n_traces");
  if (!trace || !misfit || (!params && cfg->n_params > 0))
    return fail(AFM_EINVAL, "NULL array");
  if (bounds && (rc = validate_bounds(bounds, cfg->n_params))) return rc;
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  BeamConsts bc;
  BeamModeConsts mo;
  if ((rc = beam_prepare(cfg, &bc, &mo, st))) return rc;
  if ((rc = beam_stream(bc, trace, cfg->n_traces, st))) return rc;
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = params;
  io.stream = (const double*)g_ws.stream.p;
  io.J = misfit;
  io.per = n_particles / cfg->n_traces;
  io.n_traces = cfg->n_traces;
  io.mode = 0;
  if (bounds) {  // coordinates in, personal bests untouched: map only
    io.box = make_box(bounds, cfg->n_params);
    io.mode = 2;
  }
  if ((rc = run_beam_integrate(bc, mo, io, block_threads(), st))) return rc;
  return release_ws(st);
}

int afm_beam_pso_invert(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                        uint64_t seed, const double* trace,
                        const afm_beam_cfg* cfg, double* theta_star,
                        double* J_star, double* swarm_dump, double* gbest_hist,
                        int32_t* n_iters_done, void* cuda_stream) {
  int rc = validate_beam(cfg);
  if (rc) return rc;
  if (cfg->n_params < 1) return fail(AFM_EINVAL, "nothing to invert: n_params = 0");
  if ((rc = validate_bounds(bounds, cfg->n_params))) return rc;
  if ((rc = validate_swarm(swarm))) return rc;
  if ((rc = reject_async(swarm, "afm_beam_pso_invert"))) return rc;
  if (!trace || !theta_star || !J_star)
    return fail(AFM_EINVAL, "trace/theta_star/J_star is NULL");
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  BeamConsts bc;
  BeamModeConsts mo;
  if ((rc = beam_prepare(cfg, &bc, &mo, st))) return rc;
  if ((rc = beam_stream(bc, trace, cfg->n_traces, st))) return rc;
  const int D = cfg->n_params, T = cfg->n_traces;
  const int64_t per = swarm->n_particles, PT = per * T;
  const int block = block_threads();
  const int bpt = blocks_per_trace(per, block);
  const size_t n_dbl = (size_t)PT * (3 * D + 2) + (size_t)T * (2 * D + 2);
  if (g_ws.swarm.ensure(n_dbl * 8) || g_ws.cand.ensure((size_t)bpt * T * sizeof(Cand)))
    return fail(AFM_ECUDA, "cudaMalloc of the PSO workspace failed");
  double* x = (double*)g_ws.swarm.p;
  double* v = x + PT * D;
  double* pbest = v + PT * D;
  double* J = pbest + PT * D;
  double* pbestJ = J + PT;
  double* gbest = pbestJ + PT;
  double* gbestJ = gbest + (size_t)T * D;
  double* th_dev = gbestJ + T;
  double* Js_dev = th_dev + (size_t)T * D;
  if ((rc = ensure_pinned((size_t)T * 8))) return rc;
  BoxDev box = make_box(bounds, D);
  SwarmDev sw = {swarm->w, swarm->c1, swarm->c2, swarm->topology, 0};
  LAUNCHED(launch_pso_init(box, D, per, T, seed, 0, x, v, pbest, pbestJ, gbest,
                           gbestJ, st));
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = x;
  io.stream = (const double*)g_ws.stream.p;
  io.J = J;
  io.pbest = pbest;
  io.pbestJ = pbestJ;
  io.cand = (Cand*)g_ws.cand.p;
  io.box = box;
  io.per = per;
  io.n_traces = T;
  io.mode = 1;
  int done = 0;
  for (int it = 0; it < swarm->n_iters; ++it) {
    const bool last = (it == swarm->n_iters - 1);
    if ((rc = run_beam_integrate(bc, mo, io, block, st))) return rc;
    LAUNCHED(launch_pso_gbest(
        box, D, T, bpt, (Cand*)g_ws.cand.p, pbest, gbest, gbestJ,
        gbest_hist ? gbest_hist + (size_t)it * T * (D + 1) : nullptr, th_dev,
        Js_dev, st));
    bool stop = last;
    if (!stop && swarm->j_target > 0) {
      double* hJ = (double*)g_ws.pinned;
      CUDA_TRY(cudaMemcpyAsync(hJ, gbestJ, (size_t)T * 8, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(cudaStreamSynchronize(st));
      stop = true;
      for (int s = 0; s < T; ++s)
        if (!(hJ[s] <= swarm->j_target)) stop = false;
    }
    double* dump_row =
        swarm_dump ? swarm_dump + (size_t)it * PT * (3 * D + 2) : nullptr;
    if (!stop || dump_row)
      LAUNCHED(launch_pso_move(box, sw, D, per, 0, per, T, seed, 0, (uint32_t)it,
                               stop ? 0 : 1, RingEdges{0, 0, nullptr, nullptr, 0}, J, x, v,
                               pbest, pbestJ, gbest, dump_row, st));
    done = it + 1;
    if (stop) break;
  }
  CUDA_TRY(cudaMemcpyAsync(theta_star, th_dev, (size_t)T * D * 8,
                           cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(J_star, Js_dev, (size_t)T * 8, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if ((rc = check_queue_flag(st))) return rc;  // run_beam_integrate may use the queue
  if (n_iters_done) *n_iters_done = done;
  return release_ws(st);
}

int afm_beam_trajectory(const double* theta, const afm_beam_cfg* cfg,
                        double* tip_u, double* tip_v, void* cuda_stream) {
  int rc = validate_beam(cfg);
  if (rc) return rc;
  if (!theta && cfg->n_params > 0) return fail(AFM_EINVAL, "theta is NULL");
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  BeamConsts bc;
  BeamModeConsts mo;
  if ((rc = beam_prepare(cfg, &bc, &mo, st))) return rc;
  // zero trace (unused by the trajectory kernel) placed after the stream
  if (g_ws.stream.ensure((size_t)bc.N * 32 + (size_t)bc.W * 8 + 128))
    return fail(AFM_ECUDA, "cudaMalloc failed");
  double* zero_trace = (double*)((char*)g_ws.stream.p + (size_t)bc.N * 32 + 64);
  CUDA_TRY(cudaMemsetAsync(zero_trace, 0, (size_t)bc.W * 8, st));
  if ((rc = beam_stream(bc, zero_trace, 1, st))) return rc;
  double* th_dev = (double*)g_ws.scratch.p;  // first 64 bytes of scratch
  if (cfg->n_params > 0)
    CUDA_TRY(cudaMemcpyAsync(th_dev, theta, (size_t)cfg->n_params * 8,
                             cudaMemcpyHostToDevice, st));
  LAUNCHED(launch_beam_trajectory(bc, mo, th_dev, (const double*)g_ws.stream.p,
                                  tip_u, tip_v, st));
  return release_ws(st);
}

int afm_philox4x32_10(const uint32_t* ctr, int64_t n, const uint32_t* key,
                      uint32_t* out, void* cuda_stream) {
  if (!ctr || !key || !out || n < 0)
    return fail(AFM_EINVAL, "NULL pointer or negative n");
  if (n == 0) return AFM_OK;
  int rc = check_device();
  if (rc) return rc;
  LAUNCHED(launch_philox(ctr, n, key[0], key[1], out, (cudaStream_t)cuda_stream));
  return AFM_OK;
}

int afm_trajectory(const double* theta, const afm_cfg* cfg, double z0, double v0,
                   double* zs, double* vs, void* cuda_stream) {
  int rc = validate_cfg(cfg);
  if (rc) return rc;
  if (!theta && cfg->n_params > 0) return fail(AFM_EINVAL, "theta is NULL");
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  afm_cfg c1 = *cfg;
  c1.n_traces = 1;
  ModelConsts mc;
  make_consts(&c1, 32, &mc);
  if ((rc = acquire_ws(st))) return rc;
  // a zero trace: the stream's trace column is unused by the trajectory kernel
  const size_t need = (size_t)mc.N * 32 + (size_t)mc.W * 8 + 64;
  if (g_ws.stream.ensure(need) || g_ws.scratch.ensure(64))
    return fail(AFM_ECUDA, "cudaMalloc failed");
  double* zero_trace = (double*)((char*)g_ws.stream.p + (size_t)mc.N * 32);
  CUDA_TRY(cudaMemsetAsync(zero_trace, 0, (size_t)mc.W * 8, st));
  if (cfg->n_params > 0)
    CUDA_TRY(cudaMemcpyAsync(g_ws.scratch.p, theta, (size_t)cfg->n_params * 8,
                             cudaMemcpyHostToDevice, st));
  LAUNCHED(launch_build_stream(mc, zero_trace, 1, (double*)g_ws.stream.p, st));
  LAUNCHED(launch_trajectory(mc, (const double*)g_ws.scratch.p,
                             (const double*)g_ws.stream.p, z0, v0, zs, vs, st));
  return release_ws(st);
}

int afm_fma_peak(int32_t precision, double seconds, double* tflops,
                 void* cuda_stream) {
  if (!tflops) return fail(AFM_EINVAL, "tflops is NULL");
  if (precision != AFM_F64 && precision != AFM_F32)
    return fail(AFM_EINVAL, "unknown precision %d", precision);
  if (!(seconds > 0) || seconds > 10)
    return fail(AFM_EINVAL, "seconds must be in (0, 10]");
  int rc = check_device();
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.scratch.ensure(64)) return fail(AFM_ECUDA, "cudaMalloc failed");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int threads = 256, blocks = sms * 8;
  const double per_iter = 2.0 * 8 * 16 * (double)threads * blocks;  // flops
  // calibrate the iteration count on a short launch, then time `seconds`
  int iters = 2000;
  float ms = 0.f;
  int n = launch_fma_peak(precision, iters, blocks, threads, g_ws.scratch.p, &ms, st);
  if (n < 0) return fail(AFM_ECUDA, "cudaEventCreate failed");
  g_launches += n;
  CUDA_TRY(cudaGetLastError());
  double want = seconds * 1e3 / (ms > 1e-3 ? ms : 1e-3) * iters;
  if (want > 2.0e8) want = 2.0e8;
  iters = want < 2000 ? 2000 : (int)want;
  n = launch_fma_peak(precision, iters, blocks, threads, g_ws.scratch.p, &ms, st);
  if (n < 0) return fail(AFM_ECUDA, "cudaEventCreate failed");
  g_launches += n;
  CUDA_TRY(cudaGetLastError());
  *tflops = per_iter * iters / (ms * 1e-3) / 1e12;
  return release_ws(st);
}

int afm_kernel_times(double* ms, int32_t max_n, int32_t* n_out) {
  if (!ms || !n_out || max_n < 0) return fail(AFM_EINVAL, "NULL pointer or negative max_n");
  std::lock_guard<std::mutex> lock(g_ws.mu);
  int64_t n = g_kev_count < kMaxKernelEvents ? g_kev_count : kMaxKernelEvents;
  if (n > max_n) n = max_n;
  // oldest first: launches g_kev_count - n .. g_kev_count - 1
  for (int64_t k = 0; k < n; ++k) {
    const int64_t slot = (g_kev_count - n + k) % kMaxKernelEvents;
    CUDA_TRY(cudaEventSynchronize(g_kev[slot][1]));
    float t = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&t, g_kev[slot][0], g_kev[slot][1]));
    ms[k] = (double)t;
  }
  *n_out = (int32_t)n;
  return AFM_OK;
}

int afm_pso_step_host(const afm_bounds* bounds, const afm_swarm_cfg* swarm,
                      int32_t n_dims, int32_t n_traces, uint64_t seed,
                      int32_t iteration, int32_t do_move, const double* J, double* x,
                      double* v, double* pbest, double* pbestJ, double* gbest,
                      double* gbestJ, void* cuda_stream) {
  int rc = validate_pso_step(bounds, swarm, n_dims, n_traces, iteration, J, x, v, pbest,
                             pbestJ, gbest, gbestJ);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t PT = (size_t)swarm->n_particles * n_traces;
  const size_t nd = PT * n_dims, nt = (size_t)n_traces;
  // device image: J, x, v, pbest, pbestJ, gbest, gbestJ
  const size_t total = PT + 3 * nd + PT + nt * n_dims + nt;
  // One lock over staging, step, copy-back and synchronisation: another thread
  // that needs a larger h_state would otherwise free it under the copies in flight.
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if ((rc = acquire_ws(st))) return rc;
  if (g_ws.h_state.ensure(total * 8))
    return fail(AFM_ECUDA, "cudaMalloc of the swarm staging buffer failed");
  double* base = (double*)g_ws.h_state.p;
  g_ws.last_stream = st;  // same stream: no self-wait
  double* dJ = base;
  double* dx = dJ + PT;
  double* dv = dx + nd;
  double* dpb = dv + nd;
  double* dpbJ = dpb + nd;
  double* dg = dpbJ + PT;
  double* dgJ = dg + nt * n_dims;
  const struct { double* d; const double* h; size_t n; } in[] = {
      {dJ, J, PT}, {dx, x, nd}, {dv, v, nd}, {dpb, pbest, nd},
      {dpbJ, pbestJ, PT}, {dg, gbest, nt * n_dims}, {dgJ, gbestJ, nt}};
  for (const auto& c : in)
    CUDA_TRY(cudaMemcpyAsync(c.d, c.h, c.n * 8, cudaMemcpyHostToDevice, st));
  rc = pso_step_locked(bounds, swarm, n_dims, n_traces, seed, iteration, do_move, dJ, dx,
                       dv, dpb, dpbJ, dg, dgJ, st);
  if (rc) return rc;
  const struct { double* h; const double* d; size_t n; } out[] = {
      {x, dx, nd}, {v, dv, nd}, {pbest, dpb, nd}, {pbestJ, dpbJ, PT},
      {gbest, dg, nt * n_dims}, {gbestJ, dgJ, nt}};
  for (const auto& c : out)
    CUDA_TRY(cudaMemcpyAsync(c.h, c.d, c.n * 8, cudaMemcpyDeviceToHost, st));
  if ((rc = release_ws(st))) return rc;  // after the last read of h_state
  CUDA_TRY(cudaStreamSynchronize(st));
  return AFM_OK;
}

int afm_queue_status(void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::lock_guard<std::mutex> lock(g_ws.mu);
  if (!g_ws.segq.p) return AFM_OK;  // no queue kernel has run: nothing to wait for
  CUDA_TRY(cudaStreamSynchronize(st));
  return check_queue_flag(st);
}

const char* afm_last_integrate_kernel(void) { return g_last_kernel; }

int64_t afm_launch_count(void) { return g_launches; }
void afm_reset_launch_count(void) { g_launches = 0; }

int afm_set_option(const char* name, int64_t value) {
  if (!name) return fail(AFM_EINVAL, "option name is NULL");
  if (!strcmp(name, "block")) {
    if (value != 0 && value != 32 && value != 64 && value != 128)
      return fail(AFM_EINVAL, "block must be 0, 32, 64 or 128");
    g_opt_block = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "ppt")) {
    if (value < 0 || value > 2) return fail(AFM_EINVAL, "ppt must be 0, 1 or 2");
    g_opt_ppt = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "form")) {
    if (value < 0 || value > 2) return fail(AFM_EINVAL, "form must be 0, 1 or 2");
    g_opt_form = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "lanes")) {
    if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 &&
        value != 16 && value != 32)
      return fail(AFM_EINVAL, "lanes must be 0 or a power of two up to 32");
    g_opt_lanes = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "pack")) {
    if (value < 0 || value > 2) return fail(AFM_EINVAL, "pack must be 0, 1 or 2");
    g_opt_pack = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "kernel_events")) {
    if (value < 0 || value > 1) return fail(AFM_EINVAL, "kernel_events must be 0 or 1");
    g_opt_kernel_events = (int)value;
    g_kev_count = 0;
    return AFM_OK;
  }
  if (!strcmp(name, "queue")) {
    if (value < 0 || value > 2) return fail(AFM_EINVAL, "queue must be 0, 1 or 2");
    g_opt_queue = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "workers")) {
    if (value < 0 || value > 8) return fail(AFM_EINVAL, "workers must be in 0..8");
    g_opt_workers = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "boost2")) {
    if (value < 0 || value > 1) return fail(AFM_EINVAL, "boost2 must be 0 or 1");
    g_opt_boost2 = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "boost")) {
    if (value < 0 || value > 64) return fail(AFM_EINVAL, "boost must be in 0..64");
    g_opt_boost = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "segs")) {
    if (value < 0 || value > 2047) return fail(AFM_EINVAL, "segs must be in 0..2047");
    g_opt_segs = (int)value;
    return AFM_OK;
  }
  if (!strcmp(name, "tile")) {
    if (value < 0 || value > 2048)
      return fail(AFM_EINVAL, "tile must be in 0..2048");
    g_opt_tile = (int)value;
    return AFM_OK;
  }
  return fail(AFM_EINVAL, "unknown option '%s'", name);
}

const char* afm_last_error(void) { return g_err; }
const char* afm_version(void) { return "afm-b200 0.2 (sm_100a)"; }

void afm_shutdown(void) {
  std::lock_guard<std::mutex> lock(g_ws.mu);
  g_ws.stream.release();
  g_ws.swarm.release();
  g_ws.cand.release();
  g_ws.h_params.release();
  g_ws.h_trace.release();
  g_ws.h_z0v0.release();
  g_ws.h_misfit.release();
  g_ws.h_state.release();
  g_ws.scratch.release();
  g_ws.sort.release();
  g_ws.segq.release();
  g_ws.chunk.release();
  if (g_ws.pinned) cudaFreeHost(g_ws.pinned);
  g_ws.pinned = nullptr;
  g_ws.pinned_cap = 0;
  if (g_ws.last_use) cudaEventDestroy(g_ws.last_use);
  g_ws.last_use = nullptr;
  g_ws.last_stream = nullptr;
  if (g_kev_made) {
    for (int i = 0; i < kMaxKernelEvents; ++i)
      for (int j = 0; j < 2; ++j) cudaEventDestroy(g_kev[i][j]);
    g_kev_made = false;
  }
  g_kev_count = 0;
  g_ws.checked_device = false;
  g_ws.device = -1;
}

}  // extern "C"

// =================================================================================
// afm_forward_batch_noalloc (include/afm.h): the forward batch for callers that
// cannot let the library allocate -- a microscope's acquisition loop, where a
// cudaMalloc / cudaFree (driver-wide lock, possible device-wide wait, no bound on
// its duration) in the middle of a scan line breaks the timing, or a process whose
// device memory already belongs to another component's pool.  Everything above
// takes its scratch from the grow-only workspace g_ws; this call takes its one
// piece of scratch, the time-tile stream, from an array that is part of the
// library's device image, and touches neither g_ws nor any event.
// =================================================================================
namespace {

// The time-tile stream of one call: [n_traces][N] rows of 32 bytes (FP64 kernel:
// double4; FP32 kernel: float4 in the first half).  4 MiB on every device that
// loads this library, until the process exits.
constexpr int64_t kNoallocRowBytes = 32;
static __device__ __align__(256) unsigned char
    g_noalloc_stream[(size_t)AFM_NOALLOC_MAX_ROWS * kNoallocRowBytes];

// In host code the name g_noalloc_stream is only the handle the runtime registered
// for the array -- host memory, not where the array lives on the GPU.  A kernel
// handed &g_noalloc_stream[0] would fault, or on a system where the GPU can read
// host memory quietly work on the wrong bytes.  The real address differs per
// device and comes from cudaGetSymbolAddress with that device current; it is
// looked up on the first call on each device and kept.
constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
void* g_noalloc_dev_ptr[kNoallocMaxDevices] = {};

int noalloc_stream_address(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess)
    return fail(AFM_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kNoallocMaxDevices)
    return fail(AFM_EUNSUPPORTED, "afm_forward_batch_noalloc: device ordinal %d is "
                                  "beyond the %d this call keeps addresses for",
                dev, kNoallocMaxDevices);
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (g_noalloc_dev_ptr[dev] == nullptr) {
    int major = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10)
      return fail(AFM_EUNSUPPORTED,
                  "device %d has compute capability %d.x; this library is built for "
                  "sm_100a only", dev, major);
    void* p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&p, g_noalloc_stream));
    if (p == nullptr)
      return fail(AFM_ECUDA, "cudaGetSymbolAddress returned a null address for the "
                             "built-in scratch array on device %d", dev);
    g_noalloc_dev_ptr[dev] = p;
  }
  *out = g_noalloc_dev_ptr[dev];
  return AFM_OK;
}

}  // namespace

extern "C" int afm_forward_batch_noalloc(const double* params, int64_t n_particles,
                                         const double* trace, const afm_cfg* cfg,
                                         const double* z0v0, double* misfit,
                                         void* cuda_stream) {
  int rc = validate_forward(params, n_particles, trace, cfg, misfit);
  if (rc) return rc;
  const int64_t rows =
      (int64_t)cfg->n_traces * cfg->steps_per_cycle * cfg->n_cycles;
  if (rows > (int64_t)AFM_NOALLOC_MAX_ROWS)
    return fail(AFM_EINVAL,
                "afm_forward_batch_noalloc: n_traces * steps_per_cycle * n_cycles = "
                "%d * %d * %d = %lld rows of the time-tile stream, the built-in "
                "scratch holds %d (4 MiB); use afm_forward_batch for this size",
                cfg->n_traces, cfg->steps_per_cycle, cfg->n_cycles, (long long)rows,
                (int)AFM_NOALLOC_MAX_ROWS);
  void* scratch = nullptr;
  if ((rc = noalloc_stream_address(&scratch))) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool f32 = (cfg->precision == AFM_F32);
  const int block = block_threads();
  const int ppt = particles_per_thread();
  ModelConsts mc;
  ModelConstsF32 mf;
  make_consts(cfg, block, &mc);
  make_consts_f32(cfg, &mf);
  // Nothing in the array has to start at zero: the kernel below reads rows
  // [0, n_traces * N) only, and build_stream writes every one of them first, on
  // the same stream.  Whatever an earlier, longer call left behind is never read.
  if (f32)
    LAUNCHED(launch_build_stream_f32(mf, trace, cfg->n_traces, (float*)scratch, st));
  else
    LAUNCHED(launch_build_stream(mc, trace, cfg->n_traces, (double*)scratch, st));
  IntegrateIO io;
  memset(&io, 0, sizeof(io));
  io.params = params;
  io.z0v0 = z0v0;
  io.stream = (const double*)scratch;
  io.J = misfit;
  io.per = n_particles / cfg->n_traces;
  io.n_traces = cfg->n_traces;
  io.mode = 0;
  io.lanes = pick_lanes(cfg, io.per, cfg->n_traces);
  if (f32)
    LAUNCHED(launch_integrate_f32(mf, io, block, ppt, st));
  else
    LAUNCHED(launch_integrate_f64(mc, io, block,
                                  pick_variant(io.per, io.n_traces, ppt), st));
  g_last_kernel = f32 ? "integrate_misfit_f32" : "integrate_misfit_f64";
  return AFM_OK;
}
