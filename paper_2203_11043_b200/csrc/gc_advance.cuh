// gc_advance.cuh — steps a2..a8 in ONE pass over the state (PAPER.md:68 order, then the compaction of north_star (d)):
//   reduce the field partials -> eq. 1 -> |E| -> eq. 2 -> drift -> Philox/Box-Muller diffusion (eqs. 3-4) -> update ->
//   mirror -> collection test + pixel histogram -> STABLE IN-PLACE COMPACTION of the survivors -> n_active, step, plan.
//
// The state is read once and written once (16 B + 16 B per carrier; the separate k_integrate -> tile_count ->
// k_compact pass of round 1 read and wrote it twice and cost a third launch per step).  Compaction is a single-pass
// scan with decoupled look-back over the tiles' survivor counts: tile t publishes its count, then looks back over the
// status words of the tiles before it until it meets one whose inclusive prefix is known.  Tiles are taken in ticket
// order (atomic counter), so every tile a CTA waits for belongs to a CTA that is already running: no deadlock at any
// grid size.  Compaction is IN PLACE: a survivor's destination index is <= its source index, and the slot belongs to a
// tile that published its count — i.e. had its carriers in registers — before this tile could learn its offset.
// Stable (load order preserved) and, like every integer scan, independent of timing: runs stay bit-reproducible.
#pragma once
#include "gc_common.cuh"
#include "gc_integrate.cuh"

namespace gc {

#ifdef GC_TIMING
__device__ long long g_pp[1024][16];              // per CTA: clock64 at probe points of the last step (development builds)
#define GC_P(slot) do { if (threadIdx.x == 0) g_pp[blockIdx.x & 1023][slot] = clock64(); } while (0)
#else
#define GC_P(slot) do { } while (0)
#endif

// status word of a tile: [63:34] stamp of the step | [33:32] kind (1 = count of this tile, 2 = inclusive prefix) | [31:0] value
__device__ __forceinline__ unsigned long long scan_pack(uint32_t stamp, uint32_t kind, uint32_t v) {
  return ((unsigned long long)stamp << 34) | ((unsigned long long)kind << 32) | (unsigned long long)v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Polling loads: relaxed (one L2 round trip, no L1 invalidation per iteration); the consumer fences once after the loop
// where it needs acquire ordering.
__device__ __forceinline__ uint32_t ld_relaxed_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// Publishing a word other CTAs spin on: an atomic exchange executes AT the L2, so the word is visible one trip later.
// A plain (even st.relaxed.gpu) store may sit in the SM's write path: measured 2x longer look-backs than with
// st.release, whose fence drains it at the price of a MEMBAR.
__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v) {
  unsigned long long old;
  asm volatile("atom.relaxed.gpu.global.exch.b64 %0, [%1], %2;" : "=l"(old) : "l"(p), "l"(v) : "memory");
  (void)old;
}
__device__ __forceinline__ uint32_t scan_stamp(uint32_t seq) { return (seq % 0x3ffffffeu) + 1u; }   // 30 bits, never 0

// Executed by ONE full warp of the CTA that owns tile t, after a __syncthreads that follows every thread's loads of the
// tile's carriers.  Publishes `count`, returns the number of survivors in the tiles before t (exclusive prefix), then
// publishes the inclusive prefix.  Memory ordering: everything the look-back communicates is inside the status words,
// so polling is relaxed.  With RELEASE (in-place compaction) the FIRST publish of a tile is a release: it orders the
// tile's loads of its own carriers (all threads', through the barrier) before any later tile — which acts only after
// reading this word — overwrites those slots.  Without (source and destination are different buffers) nothing is.
template <bool RELEASE>
__device__ __forceinline__ uint32_t scan_lookback(unsigned long long* status, uint32_t t, uint32_t stamp, uint32_t count) {
  const uint32_t lane = threadIdx.x & 31u;
  if (t == 0) {
    if (lane == 0) { if (RELEASE) st_release_u64(status, scan_pack(stamp, 2u, count)); else st_relaxed_u64(status, scan_pack(stamp, 2u, count)); }
    return 0u;
  }
  if (lane == 0) { if (RELEASE) st_release_u64(status + t, scan_pack(stamp, 1u, count)); else st_relaxed_u64(status + t, scan_pack(stamp, 1u, count)); }
  uint32_t excl = 0;
  int32_t hi = (int32_t)t - 1;                              // this round looks at tiles hi, hi-1, ..., hi-31
  for (;;) {
    const int32_t idx = hi - (int32_t)lane;
    uint32_t kind = 2u, val = 0u;                           // before tile 0: inclusive prefix 0
    if (idx >= 0) {
      unsigned long long s;
      do { s = ld_relaxed_u64(status + idx); } while ((uint32_t)(s >> 34) != stamp);
      kind = (uint32_t)(s >> 32) & 3u;
      val = (uint32_t)s;
    }
    const uint32_t incl = __ballot_sync(0xffffffffu, kind == 2u);
    if (incl) {                                             // nearest tile whose inclusive prefix is known
      const uint32_t first = (uint32_t)__ffs((int)incl) - 1u;
      excl += __reduce_add_sync(0xffffffffu, lane <= first ? val : 0u);
      break;
    }
    excl += __reduce_add_sync(0xffffffffu, val);
    hi -= 32;
  }
  if (lane == 0) st_relaxed_u64(status + t, scan_pack(stamp, 2u, excl + count));
  return excl;
}

// Two-level scan for a grid whose tiles all run at the same time (the persistent kernel: <= 592 tiles, one per resident
// CTA).  When every tile publishes at once, the look-back above resolves in t / 32 DEPENDENT rounds (only tile 0 knows
// its inclusive prefix at first): measured 7,400 cycles at 256 tiles.  Here tile t = 32 g + r sums the counts of the r
// tiles before it in its group (one round), the last tile of each group publishes the group's total, and every tile adds
// the totals of the g groups before its own (second round): two rounds at any tile count.  Group totals live behind
// the tile words (status[kScanGroupBase + g]).  Executed by one full warp.
constexpr uint32_t kScanGroupBase = 768;                    // tiles < 768; scan_entries >= 1,024 (gcoreccd.cu make_layout)
__device__ __forceinline__ uint32_t scan_two_level(unsigned long long* status, uint32_t t, uint32_t stamp, uint32_t count) {
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t g = t >> 5, r = t & 31u;
  if (lane == 0) st_relaxed_u64(status + t, scan_pack(stamp, 1u, count));
  // both rounds' loads are issued at once; each lane then spins on its own word until it carries this step's stamp
  const unsigned long long* pa = status + (g << 5) + lane;
  const unsigned long long* pg = status + kScanGroupBase + lane;
  unsigned long long a = lane < r ? ld_relaxed_u64(pa) : scan_pack(stamp, 1u, 0u);
  unsigned long long b = lane < g ? ld_relaxed_u64(pg) : scan_pack(stamp, 1u, 0u);
  while ((uint32_t)(a >> 34) != stamp) a = ld_relaxed_u64(pa);
  const uint32_t in_group = __reduce_add_sync(0xffffffffu, (uint32_t)a);
  if (r == 31u && lane == 0) st_relaxed_u64(status + kScanGroupBase + g, scan_pack(stamp, 1u, in_group + count));
  while ((uint32_t)(b >> 34) != stamp) b = ld_relaxed_u64(pg);
  return in_group + __reduce_add_sync(0xffffffffu, (uint32_t)b);
}

// a7..a8 for tile t = carriers [t TQ, t TQ + TQ) of the state, by the first TQ threads of the CTA (TQ <= 256, a multiple of 32;
// ALL threads of the CTA must call): (xf, yf, zf) = this thread's updated carrier, `mine` = it has one, `finite` = the
// update produced finite numbers.  Collection + histogram, survivor ranks, look-back, compacted write into A — the
// buffer the carriers were read from if INPLACE (k_advance: any number of tiles, ticket order), another one otherwise
// (the persistent kernel: all tiles resident).  Returns whether t is the last tile; thread 0 of
// that CTA then holds the new n_active in n_new_out.
template <bool INPLACE>
__device__ __forceinline__ bool commit_tile(const uint32_t TQ, SoA A, uint32_t t, uint32_t n, uint64_t step, uint32_t stamp, bool mine, bool finite,
                                            float xf, float yf, float zf, uint32_t id, Ctrl* ctrl, Sink sink,
                                            unsigned long long* status, const DevParams& P, uint32_t* s_w, uint32_t& n_new_out) {
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  uint32_t coll = 0, over = 0;
  bool keep = false;
  if (mine) {
    if (!finite) atomicOr(&ctrl->nonfinite, 1u);
    if ((double)zf <= P.z_well) { coll = 1; collect(xf, yf, zf, id, step, P, sink, over); }
    else keep = true;
  }
  // s_w: [0, TQ/32) survivors per warp, [8] exclusive prefix of the tile, [9] collected, [10] out of window
  GC_P(4);
  if (tid < 16) s_w[tid] = 0;
  __syncthreads();
  GC_P(5);
  uint32_t rank_in_warp = 0;
  if (tid < TQ) {                                            // whole warps: TQ is a multiple of 32
    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    rank_in_warp = __popc(bal & ((1u << lane) - 1u));
    const uint32_t wc = __popc(__ballot_sync(0xffffffffu, coll)), wo = __popc(__ballot_sync(0xffffffffu, over));
    if (lane == 0) {
      s_w[warp] = __popc(bal);
      if (wc) atomicAdd(&s_w[9], wc);
      if (wo) atomicAdd(&s_w[10], wo);
    }
  }
  __syncthreads();
  GC_P(6);
  if (warp == 0) {
    uint32_t count = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) count += s_w[w];             // warps beyond TQ / 32 hold 0
    const uint32_t excl = INPLACE ? scan_lookback<true>(status, t, stamp, count) : scan_two_level(status, t, stamp, count);
    if (lane == 0) {
      s_w[8] = excl;
      if (s_w[9]) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_w[9]);
      if (s_w[10]) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_w[10]);
      if ((t + 1) * TQ >= n) n_new_out = excl + count;       // the last tile knows the new population
    }
  }
  __syncthreads();
  GC_P(7);
  if (keep) {
    uint32_t off = s_w[8] + rank_in_warp;
    for (uint32_t w = 0; w < warp; ++w) off += s_w[w];
    A.x[off] = xf; A.y[off] = yf; A.z[off] = zf; A.id[off] = id;   // in place: off <= i (see the header)
  }
  return (t + 1) * TQ >= n;
}

// One time step's a2..a8.  Grid = tiles of the host's upper bound on n_active (surplus CTAs take a ticket and leave).
// The CTA that finishes last publishes n_active, step += 1, pairs += n^2 and the next step's FieldPlan.
__global__ void __launch_bounds__(kTPB, 4)
k_advance(SoA A, Ctrl* __restrict__ ctrl, const float* __restrict__ Ep, uint32_t part_cap, Sink sink,
          unsigned long long* __restrict__ status, DevParams P, PlanArgs pa, uint32_t count_pairs) {
  __shared__ uint32_t s_w[16];
  __shared__ uint32_t s_tile, s_last;
  const uint32_t n = ctrl->n_active;                         // only the last finisher writes it, after everybody has read it
  if (n == 0) return;                                        // uniform: no step is taken
  const uint32_t tid = threadIdx.x;
  const uint64_t step = ctrl->step;
  const uint32_t stamp = scan_stamp(ctrl->scan_seq);
  const uint32_t S = ctrl->plan.S, stride = ctrl->plan.stride;
  if (tid == 0) s_tile = atomicAdd(&ctrl->ticket, 1u);
  __syncthreads();
  const uint32_t t = s_tile;
  const uint32_t n_tiles = (n + kTPB - 1) / kTPB;
  uint32_t n_new = 0;
  if (t < n_tiles) {
    const uint32_t i = t * kTPB + tid;
    float x = 0.f, y = 0.f, z = 0.f; uint32_t id = 0;
    double Ex = 0.0, Ey = 0.0, Ez = 0.0;
    if (i < n) {
      x = A.x[i]; y = A.y[i]; z = A.z[i]; id = A.id[i];
      if (!(P.flags & 1u)) {                                 // GCORECCD_COULOMB_OFF
        reduce_partials(Ep + i, part_cap, S, stride, Ex, Ey, Ez);
        Ex *= -P.Kp; Ey *= -P.Kp; Ez *= -P.Kp;               // partials hold sum (r_s - r_t) w
      }
    }
    float xf = 0.f, yf = 0.f, zf = 0.f;
    bool finite = true;
    if (i < n) finite = advance_carrier(x, y, z, id, step, Ex, Ey, Ez, P, xf, yf, zf);
    commit_tile<true>(kTPB, A, t, n, step, stamp, i < n, finite, xf, yf, zf, id, ctrl, sink, status, P, s_w, n_new);
    if (tid == 0 && (t + 1) * kTPB >= n) ctrl->n_next = n_new;
  }
  // ---- last-finisher epilogue
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t done = atomicAdd(&ctrl->blocks_done, 1u);
    s_last = (done == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (s_last && tid < 32) {
    __threadfence();
    const uint32_t n_next = *((volatile uint32_t*)&ctrl->n_next);
    FieldPlan plan = ctrl->plan;
    if (plan.n != n_next || plan.IB != pa.IB) plan = plan_search(n_next, pa);   // unchanged population: keep the plan
    if (tid == 0) {
      ctrl->plan = plan;
      ctrl->n_active = n_next;
      ctrl->blocks_done = 0;
      ctrl->ticket = 0;
      ctrl->scan_seq += 1;
      ctrl->step += 1;
      if (count_pairs) ctrl->pairs += (uint64_t)n * (uint64_t)n;
    }
  }
}

}  // namespace gc
