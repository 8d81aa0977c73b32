// gc_frontend.cuh — workload front end: the X-ray initial cloud of PAPER.md:100-102,
// drawn on the GPU so that a photon list becomes carriers without a host round trip.
//   N = floor(E_e / w_e) holes (w_e = 3.77 eV at 140 K); positions ~ 3-D Gaussian of standard
//   deviation sigma around the interaction point (the sigma(E_e) model lives in the paper's refs
//   [11-13], not in its text, so sigma is an input).
// Hole k of a generator call gets centre + sigma * n_k with n_k the Box-Muller triple of
// Philox4x32-10(ctr = (k_lo, 'XRAY', k_hi, 0), key = gen_seed), same uniform mapping as the diffusion stream
// (R13); FP64 arithmetic, z above the back surface mirrored (R12), rounded to FP32.
#pragma once
#include "gc_common.cuh"
#include "gc_integrate.cuh"

namespace gc {

constexpr uint32_t kXrayTag = 0x58524159u;   // 'XRAY': keeps generator counters apart from the diffusion stream

__device__ __forceinline__ void xray_position(uint32_t seed_lo, uint32_t seed_hi, uint64_t k, double cx, double cy, double cz,
                                              double sigma, double thickness, float* __restrict__ out) {
  const uint4 w = philox4x32_10(make_uint4((uint32_t)k, kXrayTag, (uint32_t)(k >> 32), 0u), make_uint2(seed_lo, seed_hi));
  const double ua = ((double)(w.x >> 9) + 0.5) * (1.0 / 8388608.0);
  const double fa = (double)(w.y >> 8) * (1.0 / 16777216.0);
  const double ub = ((double)(w.z >> 9) + 0.5) * (1.0 / 8388608.0);
  const double fb = (double)(w.w >> 8) * (1.0 / 16777216.0);
  const double Ra = sqrt(-2.0 * log(ua)), Rb = sqrt(-2.0 * log(ub));
  double sa, ca;
  sincospi(2.0 * fa, &sa, &ca);
  const double x = cx + sigma * (Ra * ca), y = cy + sigma * (Ra * sa);
  double z = cz + sigma * (Rb * cospi(2.0 * fb));
  if (z > thickness) z = 2.0 * thickness - z;
  out[0] = (float)x; out[1] = (float)y; out[2] = (float)z;
}

// one cloud: n holes, generator indices first_index .. first_index + n
__global__ void __launch_bounds__(kTPB)
k_gen_cloud(float* __restrict__ xyz, uint32_t n, uint64_t first_index, double cx, double cy, double cz, double sigma,
            double thickness, uint32_t seed_lo, uint32_t seed_hi) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  xray_position(seed_lo, seed_hi, first_index + i, cx, cy, cz, sigma, thickness, xyz + 3 * (size_t)i);
}

// a batch of clouds: event e owns carriers [off[e], off[e+1]); centre 3 doubles and sigma per event; generator index =
// first_index + position in the batch.  The event of a carrier is found by bisection of the offsets.
__global__ void __launch_bounds__(kTPB)
k_gen_events(float* __restrict__ xyz, uint32_t n, const uint32_t* __restrict__ off, uint32_t n_events,
             const double* __restrict__ centre, const double* __restrict__ sigma, uint64_t first_index, double thickness,
             uint32_t seed_lo, uint32_t seed_hi) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  uint32_t lo = 0, hi = n_events;                       // largest e with off[e] <= i
  while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (off[mid] <= i) lo = mid; else hi = mid; }
  xray_position(seed_lo, seed_hi, first_index + i, centre[3 * (size_t)lo], centre[3 * (size_t)lo + 1], centre[3 * (size_t)lo + 2],
                sigma[lo], thickness, xyz + 3 * (size_t)i);
}

}  // namespace gc
