// gc_noalloc.cuh — kernels around the allocation-free field evaluation (include/gcoreccd.h gcoreccd_field_noalloc):
// eq. 6 for a caller that may not allocate device memory (code under CUDA-graph capture, tight serving
// loops, harnesses that forbid cudaMalloc).  The field itself is k_field (gc_field.cuh) and the FP64 reduction of its
// chunk partials is k_field_finalize (gc_integrate.cuh), unchanged; what they need besides the caller's input and
// output — positions as structure of arrays, the Ctrl block with the FieldPlan, the partial-sum planes — lives in ONE
// file-scope __device__ array of fixed size (gcoreccd.cu: g_na_scratch), laid out by NaLayout below.
#pragma once
#include "gc_common.cuh"

namespace gc {

constexpr uint32_t kNaMaxCarriers = 16384;                       // = GCORECCD_NOALLOC_MAX_CARRIERS
constexpr uint32_t kNaPartCap = 32u * kNaMaxCarriers;            // floats per partial plane: up to 32 chunks at full size
struct NaLayout {                                                // byte offsets into the scratch array (all 256-aligned)
  static constexpr size_t ctrl = 0;
  static constexpr size_t x = 256;
  static constexpr size_t y = x + sizeof(float) * kNaMaxCarriers;
  static constexpr size_t z = y + sizeof(float) * kNaMaxCarriers;
  static constexpr size_t ep = z + sizeof(float) * kNaMaxCarriers;
  static constexpr size_t bytes = ep + 3u * sizeof(float) * kNaPartCap;      // 6,488,320 B = 6.2 MiB
};

// One warp.  The array keeps the last call's contents: everything a call reads before writing it is set here — the whole
// Ctrl block is cleared (sticky flags, tickets, barrier words of other kernels' conventions), then n_active and the plan.
__global__ void k_na_prepare(Ctrl* __restrict__ ctrl, uint32_t n, PlanArgs pa) {
  uint32_t* w = reinterpret_cast<uint32_t*>(ctrl);
  for (uint32_t k = threadIdx.x; k < sizeof(Ctrl) / 4u; k += 32u) w[k] = 0u;
  __syncwarp();
  const FieldPlan p = plan_search(n, pa);
  if (threadIdx.x == 0) { ctrl->n_active = n; ctrl->n_loaded = n; ctrl->plan = p; }
}

// interleaved x,y,z (the layout of gcoreccd_load_carriers) -> structure of arrays; entries beyond n are never read by
// k_field (it masks on plan.n), so stale positions of an earlier, larger call cannot enter a sum
__global__ void __launch_bounds__(kTPB)
k_na_unpack(const float* __restrict__ xyz, uint32_t n, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  x[i] = xyz[3 * (size_t)i]; y[i] = xyz[3 * (size_t)i + 1]; z[i] = xyz[3 * (size_t)i + 2];
}

}  // namespace gc
