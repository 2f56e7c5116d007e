// afm_sort.cu -- warp packing for the DMT laws.  The integrate kernels take a
// step speculatively on the free-flight side of the law and redo it in the
// general form when ANY lane of the warp touches the sample; which lanes share a
// warp is free to choose.  Particles are therefore ordered by (trace, stiffness
// bins, initial phase): lanes of one warp then touch the sample
// at about the same time, in the transient (same phase) and in the steady state
// (similar contact width).  configs[1]: 19.05 -> ~18 ms.  The order changes no
// result: every lane's arithmetic is independent of its neighbours; the inputs
// are gathered into packed copies and the misfits scattered back to the
// particles' own indices, so the integrate kernels are not touched.
//
// The sort itself is a library primitive (cub::DeviceRadixSort, part of the CUDA
// toolkit); the key kernel is ours.
#include <cub/device/device_radix_sort.cuh>

#include <string.h>

#include "afm_internal.h"

namespace afm {

// Order-preserving unsigned image of a double (monotone in the value).
__device__ __forceinline__ uint64_t mono_bits(double x) {
  long long b = __double_as_longlong(x);
  b ^= (b >> 63) & 0x7fffffffffffffffLL;
  return (uint64_t)b ^ 0x8000000000000000ULL;
}

// With per-particle initial states (configs[1]):
//   key = [trace][bin of p1 : 13][bin of p0 : 12][initial phase : 10]
// p1 = params[.][1] (E* for the DMT laws) in half-octave bins (sign, exponent,
// one mantissa bit), p0 = params[.][0] (H) in octave bins; inside a bin the
// particles are ordered by their initial phase atan2(-v0/w, z0).  Measured on
// configs[1] with host-sorted inputs and packing off: as drawn 19.04 ms; phase
// bins then E* 18.8; E* bins (1..16 per octave) then phase 17.9-18.4; E* 2 per
// octave, H 1 per octave, then phase 17.1 ms.
// With a common initial state (inside the PSO, coordinates in): no phase to
// order by, key = [trace][top 35 bits of p1].  Only the bits in use are sorted.
__global__ void pack_key_kernel(const double* __restrict__ params,
                                const double* __restrict__ z0v0, int D,
                                int64_t per, int64_t PT, double w_drive,
                                double z0d, double v0d,
                                uint64_t* __restrict__ keys,
                                uint32_t* __restrict__ idx) {
  const int64_t gp = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gp >= PT) return;
  uint64_t low = 0;
  const double* th = params + gp * D;
  if (z0v0 != nullptr) {
    // z = A cos(phi), v = -A w sin(phi)
    const double phi = atan2(-z0v0[2 * gp + 1] / w_drive, z0v0[2 * gp]);  // (-pi, pi]
    int ph = (int)floor((phi + 3.14159265358979323846) * (1024.0 / 6.283185307179586));
    ph = min(max(ph, 0), 1023);
    const uint64_t b1 = (D >= 2) ? (mono_bits(th[1]) >> 51) : 0;  // 13 bits
    const uint64_t b0 = (D >= 1) ? (mono_bits(th[0]) >> 52) : 0;  // 12 bits
    low = (b1 << 22) | (b0 << 10) | (uint64_t)ph;
  } else if (D > 0) {
    low = mono_bits(th[D >= 2 ? 1 : 0]) >> 29;  // 35 bits
  }
  keys[gp] = ((uint64_t)(gp / per) << 35) | low;
  idx[gp] = (uint32_t)gp;
}

static size_t cub_bytes(int64_t PT) {
  size_t bytes = 0;
  cub::DeviceRadixSort::SortPairs(nullptr, bytes, (const uint64_t*)nullptr,
                                  (uint64_t*)nullptr, (const uint32_t*)nullptr,
                                  (uint32_t*)nullptr, (int)PT, 0, 59);
  return bytes;
}

// layout of ws: keys_in [PT] u64 | keys_out [PT] u64 | idx_in [PT] u32 | cub temp
size_t sort_workspace_bytes(int64_t PT) {
  return (size_t)PT * (8 + 8 + 4) + 256 + cub_bytes(PT);
}

int launch_pack_order(const double* params, const double* z0v0, int D, int64_t per,
                      int64_t PT, double w_drive, double z0_default,
                      double v0_default, void* ws, size_t ws_bytes,
                      uint32_t* order, cudaStream_t st) {
  uint64_t* keys_in = (uint64_t*)ws;
  uint64_t* keys_out = keys_in + PT;
  uint32_t* idx_in = (uint32_t*)(keys_out + PT);
  char* temp = (char*)(idx_in + PT);
  temp += (256 - ((uintptr_t)temp & 255)) & 255;
  size_t temp_bytes = ws_bytes - (size_t)(temp - (char*)ws);
  const int threads = 256;
  pack_key_kernel<<<(unsigned)((PT + threads - 1) / threads), threads, 0, st>>>(
      params, z0v0, D, per, PT, w_drive, z0_default, v0_default, keys_in, idx_in);
  int end_bit = 35;  // + the bits of the trace index
  for (int64_t t = PT / per - 1; t > 0; t >>= 1) ++end_bit;
  if (cub::DeviceRadixSort::SortPairs(temp, temp_bytes, keys_in, keys_out, idx_in,
                                      order, (int)PT, 0, end_bit, st) != cudaSuccess)
    return -2;
  return 1;
}

// With map_coords the inputs are PSO coordinates and the packed copy receives
// the physical parameters (row a1 of SURVEY.md 8(a): theta_j = 10^x_j where the
// coordinate is logarithmic), exactly as the integrate kernel's own prologue
// computes them.
__global__ void pack_gather_kernel(const uint32_t* __restrict__ order,
                                   const double* __restrict__ params,
                                   const double* __restrict__ z0v0, int D,
                                   int64_t PT, double* __restrict__ params_s,
                                   double* __restrict__ z0v0_s, int map_coords,
                                   BoxDev box) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= PT) return;
  const int64_t gp = order[i];
  for (int j = 0; j < D; ++j) {
    const double xv = params[gp * D + j];
    params_s[i * D + j] = (map_coords && box.lg[j]) ? pow(10.0, xv) : xv;
  }
  if (z0v0 != nullptr) {
    z0v0_s[2 * i] = z0v0[2 * gp];
    z0v0_s[2 * i + 1] = z0v0[2 * gp + 1];
  }
}

__global__ void pack_scatter_kernel(const uint32_t* __restrict__ order,
                                    const double* __restrict__ J_s, int64_t PT,
                                    double* __restrict__ J) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < PT) J[order[i]] = J_s[i];
}

int launch_pack_gather(const uint32_t* order, const double* params,
                       const double* z0v0, int D, int64_t PT, double* params_s,
                       double* z0v0_s, const BoxDev* map, cudaStream_t st) {
  const int threads = 256;
  BoxDev box;
  memset(&box, 0, sizeof(box));
  if (map) box = *map;
  pack_gather_kernel<<<(unsigned)((PT + threads - 1) / threads), threads, 0, st>>>(
      order, params, z0v0, D, PT, params_s, z0v0_s, map ? 1 : 0, box);
  return 1;
}

int launch_pack_scatter(const uint32_t* order, const double* J_s, int64_t PT,
                        double* J, cudaStream_t st) {
  const int threads = 256;
  pack_scatter_kernel<<<(unsigned)((PT + threads - 1) / threads), threads, 0, st>>>(
      order, J_s, PT, J);
  return 1;
}

}  // namespace afm
