// gc_compact.cuh — step a8 as a kernel of its own: stable stream compaction of the carriers still drifting (not in the
// paper, whose kernel always sums i = 1..N; BASELINE.json north_star (d)).  Used where the survivors are
// known before the compaction starts: the load path (k_unpack), the Coulomb-off multi-step path (k_drift_multi) and
// k_integrate's sharded use; a time step of the main path compacts inside k_advance (gc_advance.cuh).
// Warp ballot + block scan, no Thrust: tile t (kTPB carriers of state B) knows its survivor count from the producer;
// its base offset comes from the single-pass look-back scan of gc_advance.cuh over the tiles' counts (tiles taken in
// ticket order; O(T) in total — round 1 summed tile_count[0..t) in every tile, O(T^2)), the rank inside the tile from
// __ballot_sync/__popc and a scan over the warp totals.  Order is preserved, so a carrier's index never depends on
// timing.  The CTA that FINISHES last publishes the new n_active, advances the step index, accumulates the pair
// counter and computes the next step's FieldPlan.
#pragma once
#include "gc_advance.cuh"
#include "gc_common.cuh"

namespace gc {

// src: m entries of state B (m = n_active for a step, = n for a load); survivors (z > z_well) are appended to
// dst (state A) starting at dst_off.  mode 0: time step (m read from ctrl->n_active, dst_off = 0, step += 1,
// pairs += m^2 unless Coulomb is off);  mode 1: load (m, dst_off given; n_loaded += m);  mode 2: as mode 0 after
// k_drift_multi (step += ctrl->multi_steps, which is cleared).
__global__ void __launch_bounds__(kTPB)
k_compact(SoA B, SoA A, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ tile_count,
          unsigned long long* __restrict__ status, uint32_t m_arg, uint32_t dst_off_arg, int mode, double z_well,
          uint32_t count_pairs, PlanArgs pa) {
  __shared__ uint32_t s_red[kTPB / 32];
  __shared__ uint32_t s_base, s_last, s_tile;
  const uint32_t m = mode != 1 ? ctrl->n_active : m_arg;
  const uint32_t dst_off = mode != 1 ? 0u : dst_off_arg;
  if (m == 0) return;                                     // uniform: every CTA sees the same m; no step is taken
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t stamp = scan_stamp(ctrl->scan_seq);
  if (tid == 0) s_tile = atomicAdd(&ctrl->ticket, 1u);    // tiles in start order: what the look-back waits for is running
  __syncthreads();
  const uint32_t t = s_tile;
  const uint32_t n_tiles = (m + kTPB - 1) / kTPB;

  if (t < n_tiles) {
    // this thread's carrier first: its loads overlap the tile_count reduction below (the kernel is latency bound)
    const uint32_t i = t * kTPB + tid;
    float x = 0.f, y = 0.f, z = 0.f; uint32_t id = 0;
    if (i < m) { x = B.x[i]; y = B.y[i]; z = B.z[i]; id = B.id[i]; }
    const bool keep = i < m && (double)z > z_well;
    // base = sum of the survivor counts of tiles [0, t): single-pass look-back scan
    if (warp == 0) {
      const uint32_t excl = scan_lookback<false>(status, t, stamp, tile_count[t]);
      if (lane == 0) s_base = excl;
    }
    __syncthreads();
    const uint32_t base = dst_off + s_base;

    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    const uint32_t rank_in_warp = __popc(bal & ((1u << lane) - 1u));
    __syncthreads();                                      // s_red reuse
    if (lane == 0) s_red[warp] = __popc(bal);
    __syncthreads();
    uint32_t warp_off = 0;
    for (uint32_t w = 0; w < warp; ++w) warp_off += s_red[w];
    if (keep) {
      const uint32_t d = base + warp_off + rank_in_warp;
      A.x[d] = x; A.y[d] = y; A.z[d] = z; A.id[d] = id;
    }
    if (t == n_tiles - 1 && tid == 0) {
      uint32_t tot = 0;
      for (int w = 0; w < kTPB / 32; ++w) tot += s_red[w];
      ctrl->n_next = base + tot;                          // new n_active (published by the last finisher)
    }
  }

  // ---- last-finisher epilogue -------------------------------------------------------------------
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t ticket = atomicAdd(&ctrl->blocks_done, 1u);
    s_last = (ticket == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (s_last && warp == 0) {
    __threadfence();
    const uint32_t n_new = *((volatile uint32_t*)&ctrl->n_next);
    FieldPlan plan = ctrl->plan;
    if (plan.n != n_new || plan.IB != pa.IB) plan = plan_search(n_new, pa);   // unchanged population: keep the plan
    if (lane == 0) {
      ctrl->plan = plan;
      ctrl->n_active = n_new;
      ctrl->blocks_done = 0;
      ctrl->ticket = 0;
      ctrl->scan_seq += 1;
      if (mode == 0) {
        ctrl->step += 1;
        if (count_pairs) ctrl->pairs += (uint64_t)m * (uint64_t)m;
      } else if (mode == 2) {
        ctrl->step += ctrl->multi_steps;
        ctrl->multi_steps = 0;
      } else {
        ctrl->n_loaded += m;
      }
    }
  }
}

// Recompute the plan when the host switches the field-kernel variant (or after reset / snapshot).
__global__ void k_replan(Ctrl* __restrict__ ctrl, PlanArgs pa, int set_n, uint32_t n_new, int set_step, uint64_t step) {
  if (set_n && threadIdx.x == 0) ctrl->n_active = n_new;
  if (set_step && threadIdx.x == 0) ctrl->step = step;
  __syncwarp();
  const uint32_t n = set_n ? n_new : ctrl->n_active;
  const FieldPlan plan = plan_search(n, pa);
  if (threadIdx.x == 0) ctrl->plan = plan;
}

}  // namespace gc
