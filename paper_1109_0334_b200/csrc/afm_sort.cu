// afm_sort.cu -- warp packing for the DMT laws.  The integrate kernels take a
// step speculatively on the free-flight side of the law and redo it in the
// general form when ANY lane of the warp touches the sample; which lanes share a
// warp is free to choose.  Particles are therefore ordered by (trace, initial
// stiffness bin, initial phase): lanes of one warp then touch the sample
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

// key = [trace : 24][stiffness bin : 14][initial phase : 14].  The stiffness bin
// is the top of the order-preserving bit pattern of params[.][j] (sign, exponent
// and two mantissa bits: four bins per octave), j = 1 when D >= 2 (E* for the DMT
// laws), else 0; inside a bin the particles are ordered by their initial phase
// atan2(-v0/w, z0).  Measured on configs[1] (host-sorted inputs, packing off):
// stiffness bins then phase 18.9 ms, phase bins then stiffness 19.4 ms, as drawn
// 20.1 ms (this build's kernel; profiles/r1c_beam.md lists the sweep).
__global__ void pack_key_kernel(const double* __restrict__ params,
                                const double* __restrict__ z0v0, int D,
                                int64_t per, int64_t PT, double w_drive,
                                double z0d, double v0d,
                                uint64_t* __restrict__ keys,
                                uint32_t* __restrict__ idx) {
  const int64_t gp = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gp >= PT) return;
  const double z0 = z0v0 ? z0v0[2 * gp] : z0d;
  const double v0 = z0v0 ? z0v0[2 * gp + 1] : v0d;
  // z = A cos(phi), v = -A w sin(phi)
  const double phi = atan2(-v0 / w_drive, z0);  // (-pi, pi]
  int ph = (int)floor((phi + 3.14159265358979323846) * (16384.0 / 6.283185307179586));
  ph = min(max(ph, 0), 16383);
  uint64_t stiff = 0;
  if (D > 0) {
    long long b = __double_as_longlong(params[gp * D + (D >= 2 ? 1 : 0)]);
    b ^= (b >> 63) & 0x7fffffffffffffffLL;              // monotone in the value
    stiff = (uint64_t)b ^ 0x8000000000000000ULL;  // unsigned, monotone
  }
  // a common start (z0v0 == nullptr, e.g. inside the PSO): no phase to order by,
  // all 28 bits go to the stiffness parameter
  const uint64_t low = z0v0 ? (((stiff >> 50) << 14) | (uint64_t)ph) : (stiff >> 36);
  keys[gp] = ((uint64_t)(gp / per) << 28) | low;
  idx[gp] = (uint32_t)gp;
}

static size_t cub_bytes(int64_t PT) {
  size_t bytes = 0;
  cub::DeviceRadixSort::SortPairs(nullptr, bytes, (const uint64_t*)nullptr,
                                  (uint64_t*)nullptr, (const uint32_t*)nullptr,
                                  (uint32_t*)nullptr, (int)PT, 0, 52);
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
  if (cub::DeviceRadixSort::SortPairs(temp, temp_bytes, keys_in, keys_out, idx_in,
                                      order, (int)PT, 0, 52, st) != cudaSuccess)
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
