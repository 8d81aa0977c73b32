// gc_events.cuh — batched independent events: the paper's X-ray workload is MANY small
// clouds (tens to thousands of holes each) whose holes interact only inside their own event,
// and its GPU is "under-utilised" below ~1e3 holes because every step is a train of launches.
//
// B200 design: ONE CTA OWNS ONE EVENT FOR ITS WHOLE LIFE.  The event's state lives in shared memory (up to
// 4,096 holes = 176 KB of the SM's 227 KB), already in the pre-duplicated (x,x,y,y)/(z,z) layout the packed
// field loop consumes; all eight rows a1..a8 of a time step run inside the CTA with two block barriers per
// step and no global-memory traffic except the integer histogram atomics of collected holes.  A persistent
// grid pulls events from a queue (largest first), so hundreds of events are in flight and the FP32 pipes see
// the same packed inner loop as k_field — with zero launches and zero HBM round trips per step.
//
// Per step inside the CTA (PAPER.md:68 order, identical arithmetic to k_field / k_integrate / k_compact):
//   field + integrate:  thread t owns targets {pass*2*NPACK*TPB + p*2*TPB + t + {0,hs}} (the two lanes of pack p; hs = TPB,
//                       less in the last pack, see k_events); it sums eq. 6 over all
//                       sources from shared memory (two-level FP32 accumulation: 256-source tile partials flushed
//                       into a total), then advances each of its targets in FP64 (advance_carrier) into s_next;
//   collect + compact:  each thread takes a contiguous run of s_next, bins the holes with z <= z_well into the
//                       image, block-scans the survivor counts and writes the survivors back, in order (stable),
//                       into the duplicated layout.  step += 1, pairs += n^2.
#pragma once
#include "gc_common.cuh"
#include "gc_field.cuh"
#include "gc_integrate.cuh"
#include <cooperative_groups.h>

namespace gc {

struct EventTable {            // device arrays, one entry per event
  const uint32_t* off;         // first slot of the event in the state arrays (fixed at load)
  uint32_t* cnt;               // holes still drifting, compacted at [off, off + cnt)
  uint64_t* step;              // steps taken so far = index of the event's next step (Philox counter)
};

// Four variants, chosen per event by its size at load (k_events_warp below for the first, k_events for the rest):
constexpr uint32_t kEvCapMicro = 32;       // one WARP per event, state in registers, no block barrier at all
constexpr uint32_t kEvCapTiny  = 128;      // NPACK 1,  64 threads: one pass covers 128 targets, ~12 CTAs (events) per SM
constexpr uint32_t kEvCapSmall = 512;      // NPACK 1, 256 threads: one pass covers 512 targets, 3 CTAs per SM
constexpr uint32_t kEvCapLarge = 4096;     // NPACK 4, 256 threads: 2,048 targets per pass, one CTA per SM

__host__ __device__ constexpr size_t event_smem_bytes(uint32_t cap) {
  // s_xy float4[cap+4] | s_next float4[cap] | s_z float2[cap+4] | s_id u32[cap]
  return (size_t)(cap + 4) * 16 + (size_t)cap * 16 + (size_t)(cap + 4) * 8 + (size_t)cap * 4;
}

// Field of NP packs of this thread against all n sources in shared memory; returns sum (r_s - r_t) w per target.
template <int NP, int TPB>
__device__ __forceinline__ void event_field(const float4* __restrict__ s_xy, const float2* __restrict__ s_z, uint32_t n,
                                            uint32_t i_first, uint32_t p_last, uint32_t hs_last, const float2 eps2v,
                                            float2 (&tx)[NP], float2 (&ty)[NP], float2 (&tz)[NP]) {
  float2 ntx[NP], nty[NP], ntz[NP];
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    const uint32_t i0 = i_first + (uint32_t)p * (2u * TPB), i1 = i0 + ((uint32_t)p == p_last ? hs_last : (uint32_t)TPB);
    // slots >= n hold sentinels or stale data: keep them out of the arithmetic (their result is never used)
    const bool v0 = i0 < n, v1 = i1 < n;
    const float4 a0 = s_xy[v0 ? i0 : 0], a1 = s_xy[v1 ? i1 : 0];
    const float2 b0 = s_z[v0 ? i0 : 0], b1 = s_z[v1 ? i1 : 0];
    ntx[p] = make_float2(-a0.x, -a1.x); nty[p] = make_float2(-a0.z, -a1.z); ntz[p] = make_float2(-b0.x, -b1.x);
    tx[p] = make_float2(0.f, 0.f); ty[p] = tx[p]; tz[p] = tx[p];
  }
  for (uint32_t jt = 0; jt < n; jt += kTile) {
    const int len = (int)min((uint32_t)kTile, (n - jt + 3u) & ~3u);      // tail padded to the unroll factor with sentinels
    float2 ax[NP], ay[NP], az[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) { ax[p] = make_float2(0.f, 0.f); ay[p] = ax[p]; az[p] = ax[p]; }
    const float4* sxy = s_xy + jt;
    const float2* sz = s_z + jt;
#pragma unroll 4
    for (int jj = 0; jj < len; ++jj) interact<NP>(sxy[jj], sz[jj], ntx, nty, ntz, eps2v, ax, ay, az);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      tx[p] = __fadd2_rn(tx[p], ax[p]); ty[p] = __fadd2_rn(ty[p], ay[p]); tz[p] = __fadd2_rn(tz[p], az[p]);
    }
  }
}

// a2..a6 for the 2 NP targets of this thread, results into s_next (x', y', z', id).
template <int NP, int TPB>
__device__ __forceinline__ void event_advance(const float4* __restrict__ s_xy, const float2* __restrict__ s_z,
                                              const uint32_t* __restrict__ s_id, float4* __restrict__ s_next, uint32_t n,
                                              uint32_t i_first, uint32_t p_last, uint32_t hs_last, uint64_t step,
                                              const float2 (&tx)[NP], const float2 (&ty)[NP], const float2 (&tz)[NP],
                                              const DevParams& P, uint32_t& nonfinite) {
#pragma unroll
  for (int p = 0; p < NP; ++p) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t i = i_first + (uint32_t)p * (2u * TPB) + (uint32_t)h * ((uint32_t)p == p_last ? hs_last : (uint32_t)TPB);
      if (i < n) {
        const float x = s_xy[i].x, y = s_xy[i].z, z = s_z[i].x;
        const uint32_t id = s_id[i];
        // partials hold sum (r_s - r_t) w = -S_t
        const double Ex = -P.Kp * (double)(h ? tx[p].y : tx[p].x), Ey = -P.Kp * (double)(h ? ty[p].y : ty[p].x),
                     Ez = -P.Kp * (double)(h ? tz[p].y : tz[p].x);
        float xf, yf, zf;
        if (!advance_carrier(x, y, z, id, step, Ex, Ey, Ez, P, xf, yf, zf)) nonfinite = 1u;
        s_next[i] = make_float4(xf, yf, zf, __uint_as_float(id));
      }
    }
  }
}

template <int NP, int TPB>
__device__ __forceinline__ void event_pass(const float4* s_xy, const float2* s_z, const uint32_t* s_id, float4* s_next,
                                           uint32_t n, uint32_t i_first, uint32_t p_last, uint32_t hs_last, uint64_t step,
                                           const DevParams& P, uint32_t& nonfinite) {
  float2 tx[NP], ty[NP], tz[NP];
  if (!(P.flags & 1u)) {                                     // GCORECCD_COULOMB_OFF
    event_field<NP, TPB>(s_xy, s_z, n, i_first, p_last, hs_last, make_float2(P.eps2, P.eps2), tx, ty, tz);
  } else {
#pragma unroll
    for (int p = 0; p < NP; ++p) { tx[p] = make_float2(0.f, 0.f); ty[p] = tx[p]; tz[p] = tx[p]; }
  }
  event_advance<NP, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, tx, ty, tz, P, nonfinite);
}

// Persistent grid; CTA loop: take the next event of `order[0..n_order)`, run it for up to max_steps more steps
// (or to full collection), store the survivors back.  cap = holes the dynamic shared memory is sized for.
template <int NPACK, int TPB, int MINB>        // NPACK is 1 (tiny / small events) or 4 (large events)
__global__ void __launch_bounds__(TPB, MINB)
k_events(SoA A, EventTable ev, const uint32_t* __restrict__ order, uint32_t n_order, uint32_t* __restrict__ queue,
         Ctrl* __restrict__ ctrl, Sink sink, DevParams P, uint64_t max_steps, uint32_t cap) {
  extern __shared__ __align__(16) unsigned char smem[];
  float4* s_xy = reinterpret_cast<float4*>(smem);                       // (x,x,y,y), cap + 4 entries
  float4* s_next = s_xy + (cap + 4);                                    // (x',y',z',id), cap entries
  float2* s_z = reinterpret_cast<float2*>(s_next + cap);                // (z,z), cap + 4 entries
  uint32_t* s_id = reinterpret_cast<uint32_t*>(s_z + (cap + 4));        // cap entries
  __shared__ uint32_t s_warp[TPB / 32];
  __shared__ uint32_t s_ev, s_coll, s_over;

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  constexpr uint32_t kPass = 2u * NPACK * TPB;                          // targets per pass
  uint32_t nonfinite = 0;

  for (;;) {
    __syncthreads();                                                    // previous event fully retired
    if (tid == 0) { s_ev = atomicAdd(queue, 1u); s_coll = 0; s_over = 0; }
    __syncthreads();
    if (s_ev >= n_order) break;
    const uint32_t e = order[s_ev];
    const uint32_t off = ev.off[e];
    uint32_t n = ev.cnt[e];
    uint64_t step = ev.step[e];
    if (n == 0) continue;
    for (uint32_t i = tid; i < n; i += TPB)
      s_next[i] = make_float4(A.x[off + i], A.y[off + i], A.z[off + i], __uint_as_float(A.id[off + i]));
    __syncthreads();

    uint64_t pairs = 0, done = 0;
    bool first = true;
    for (;;) {
      // ---- a7 + a8: bin the holes that crossed z_well, compact the survivors (stable) into the field layout
      const uint32_t per = (n + TPB - 1) / TPB;
      const uint32_t lo = min(tid * per, n), hi = min(lo + per, n);
      uint32_t keep = 0, coll = 0, over = 0;
      for (uint32_t i = lo; i < hi; ++i) {
        const float4 c = s_next[i];
        if ((double)c.z <= P.z_well) { coll += 1; collect(c.x, c.y, c.z, __float_as_uint(c.w), step, P, sink, over); }
        else keep += 1;
      }
      uint32_t incl = keep;                                             // block exclusive scan of the survivor counts
      for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o); if ((int)lane >= o) incl += v; }
      if (lane == 31) s_warp[warp] = incl;
      const uint32_t wc = __reduce_add_sync(0xffffffffu, coll), wo = __reduce_add_sync(0xffffffffu, over);
      if (lane == 0 && wc) { atomicAdd(&s_coll, wc); if (wo) atomicAdd(&s_over, wo); }
      __syncthreads();
      uint32_t base = 0, total = 0;
#pragma unroll
      for (int w = 0; w < TPB / 32; ++w) { const uint32_t v = s_warp[w]; if (w < (int)warp) base += v; total += v; }
      uint32_t o = base + incl - keep;
      for (uint32_t i = lo; i < hi; ++i) {
        const float4 c = s_next[i];
        if ((double)c.z > P.z_well) {
          s_xy[o] = make_float4(c.x, c.x, c.y, c.y); s_z[o] = make_float2(c.z, c.z); s_id[o] = __float_as_uint(c.w);
          ++o;
        }
      }
      if (tid < 4) {                                                    // sentinels up to the unroll factor
        const uint32_t k = total + tid;
        if (k < ((total + 3u) & ~3u)) { s_xy[k] = make_float4(kSentinel, kSentinel, kSentinel, kSentinel); s_z[k] = make_float2(kSentinel, kSentinel); }
      }
      if (!first) { step += 1; done += 1; if (!(P.flags & 1u)) pairs += (uint64_t)n * (uint64_t)n; }
      first = false;
      n = total;
      __syncthreads();
      if (n == 0 || done >= max_steps) break;

      // ---- a1..a6: field of every hole of the event, then its Euler-Maruyama update, into s_next
      for (uint32_t base_i = 0; base_i < n; base_i += kPass) {
        // Pack p covers targets [base_i + p 2TPB, +2TPB): thread t takes t and t + hs of it.  hs = TPB except in the
        // last live pack, where it shrinks to half the remaining targets (rounded up to a warp), so that both lanes
        // of the packed arithmetic stay busy and an event of <= 32 holes puts one hole on each thread of one warp.
        const uint32_t i_first = base_i + tid;
        const uint32_t m = min(n - base_i, kPass);
        const uint32_t p_last = (m - 1u) / (2u * TPB);
        const uint32_t m_last = m - p_last * (2u * TPB);
        const uint32_t hs_last = min((uint32_t)TPB, max(32u, (((m_last + 1u) >> 1) + 31u) & ~31u));
        const uint32_t np = p_last + ((warp * 32u < hs_last) ? 1u : 0u);   // packs with a live target in this warp (uniform)
        if (np == 0) continue;
        if constexpr (NPACK == 1) {
          event_pass<1, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
        } else {
          if (np == 1) event_pass<1, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else if (np == 2) event_pass<2, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else if (np == 3) event_pass<3, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else event_pass<4, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
        }
      }
      __syncthreads();
    }

    // ---- retire: survivors (if max_steps stopped the event early) back to the state arrays, counters out
    for (uint32_t i = tid; i < n; i += TPB) {
      A.x[off + i] = s_xy[i].x; A.y[off + i] = s_xy[i].z; A.z[off + i] = s_z[i].x; A.id[off + i] = s_id[i];
    }
    if (tid == 0) {
      ev.cnt[e] = n;
      ev.step[e] = step;
      if (s_coll) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_coll);
      if (s_over) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_over);
      if (pairs) atomicAdd((unsigned long long*)&ctrl->pairs, (unsigned long long)pairs);
    }
  }
  if (nonfinite) atomicOr(&ctrl->nonfinite, 1u);
}

// FEW LARGE EVENTS: with one CTA per event and about as many events as SMs, the batch takes as long as its deepest
// event while the SMs of the shallow ones idle (148 x 4,096 holes: 26 % of FP32 peak).  Here a thread-block CLUSTER of
// CL CTAs (CL SMs) owns one event: every CTA keeps the whole state in its own shared memory (the field loop needs all
// sources locally), the passes of 2*NPACK*TPB targets are dealt round-robin to the CTAs, and after the update each CTA
// pulls the other CTAs' new positions through distributed shared memory (two cluster barriers per step).  Collection
// and compaction are repeated identically in every CTA (O(n), cheap); only rank 0 touches the image, the records and
// the counters.  Same arithmetic per pair and per hole as k_events.
template <int NPACK, int TPB, int CL>
__global__ void __launch_bounds__(TPB, 1)
k_events_cluster(SoA A, EventTable ev, const uint32_t* __restrict__ order, uint32_t n_order, uint32_t* __restrict__ queue,
                 Ctrl* __restrict__ ctrl, Sink sink, DevParams P, uint64_t max_steps, uint32_t cap) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const uint32_t rank = cluster.block_rank();
  extern __shared__ __align__(16) unsigned char smem[];
  float4* s_xy = reinterpret_cast<float4*>(smem);                       // (x,x,y,y), cap + 4 entries
  float4* s_next = s_xy + (cap + 4);                                    // (x',y',z',id), cap entries
  float2* s_z = reinterpret_cast<float2*>(s_next + cap);                // (z,z), cap + 4 entries
  uint32_t* s_id = reinterpret_cast<uint32_t*>(s_z + (cap + 4));        // cap entries
  __shared__ uint32_t s_warp[TPB / 32];
  __shared__ uint32_t s_ev, s_coll, s_over;

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  constexpr uint32_t kPass = 2u * NPACK * TPB;                          // targets per pass
  uint32_t nonfinite = 0;

  for (;;) {
    cluster.sync();                                                     // previous event fully retired, in every CTA
    if (tid == 0) {
      s_coll = 0; s_over = 0;
      if (rank == 0) {
        const uint32_t v = atomicAdd(queue, 1u);
        for (uint32_t r = 0; r < CL; ++r) *cluster.map_shared_rank(&s_ev, r) = v;
      }
    }
    cluster.sync();
    if (s_ev >= n_order) break;
    const uint32_t e = order[s_ev];
    const uint32_t off = ev.off[e];
    uint32_t n = ev.cnt[e];
    uint64_t step = ev.step[e];
    if (n == 0) continue;
    for (uint32_t i = tid; i < n; i += TPB)
      s_next[i] = make_float4(A.x[off + i], A.y[off + i], A.z[off + i], __uint_as_float(A.id[off + i]));
    __syncthreads();

    uint64_t pairs = 0, done = 0;
    bool first = true;
    for (;;) {
      // ---- a7 + a8: bin the holes that crossed z_well, compact the survivors (stable) into the field layout
      const uint32_t per = (n + TPB - 1) / TPB;
      const uint32_t lo = min(tid * per, n), hi = min(lo + per, n);
      uint32_t keep = 0, coll = 0, over = 0;
      for (uint32_t i = lo; i < hi; ++i) {
        const float4 c = s_next[i];
        if ((double)c.z <= P.z_well) { coll += 1; if (rank == 0) collect(c.x, c.y, c.z, __float_as_uint(c.w), step, P, sink, over); }
        else keep += 1;
      }
      uint32_t incl = keep;                                             // block exclusive scan of the survivor counts
      for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o); if ((int)lane >= o) incl += v; }
      if (lane == 31) s_warp[warp] = incl;
      const uint32_t wc = __reduce_add_sync(0xffffffffu, coll), wo = __reduce_add_sync(0xffffffffu, over);
      if (lane == 0 && wc) { atomicAdd(&s_coll, wc); if (wo) atomicAdd(&s_over, wo); }
      __syncthreads();
      uint32_t base = 0, total = 0;
#pragma unroll
      for (int w = 0; w < TPB / 32; ++w) { const uint32_t v = s_warp[w]; if (w < (int)warp) base += v; total += v; }
      uint32_t o = base + incl - keep;
      for (uint32_t i = lo; i < hi; ++i) {
        const float4 c = s_next[i];
        if ((double)c.z > P.z_well) {
          s_xy[o] = make_float4(c.x, c.x, c.y, c.y); s_z[o] = make_float2(c.z, c.z); s_id[o] = __float_as_uint(c.w);
          ++o;
        }
      }
      if (tid < 4) {                                                    // sentinels up to the unroll factor
        const uint32_t k = total + tid;
        if (k < ((total + 3u) & ~3u)) { s_xy[k] = make_float4(kSentinel, kSentinel, kSentinel, kSentinel); s_z[k] = make_float2(kSentinel, kSentinel); }
      }
      if (!first) { step += 1; done += 1; if (!(P.flags & 1u)) pairs += (uint64_t)n * (uint64_t)n; }
      first = false;
      n = total;
      __syncthreads();
      if (n == 0 || done >= max_steps) break;

      // ---- a1..a6: field of every hole of the event, then its Euler-Maruyama update, into s_next
      // pass size: an even split of the event over the CTAs, in whole packs of 2 TPB targets, at most kPass
      const uint32_t pass_sz = min(kPass, max(2u * TPB, (((n + CL - 1u) / CL + 2u * TPB - 1u) / (2u * TPB)) * (2u * TPB)));
      for (uint32_t base_i = 0, pass = 0; base_i < n; base_i += pass_sz, ++pass) {
        if (pass % CL != rank) continue;                                  // another CTA of the cluster owns this pass
        // Pack p covers targets [base_i + p 2TPB, +2TPB): thread t takes t and t + hs of it.  hs = TPB except in the
        // last live pack, where it shrinks to half the remaining targets (rounded up to a warp), so that both lanes
        // of the packed arithmetic stay busy and an event of <= 32 holes puts one hole on each thread of one warp.
        const uint32_t i_first = base_i + tid;
        const uint32_t m = min(n - base_i, pass_sz);
        const uint32_t p_last = (m - 1u) / (2u * TPB);
        const uint32_t m_last = m - p_last * (2u * TPB);
        const uint32_t hs_last = min((uint32_t)TPB, max(32u, (((m_last + 1u) >> 1) + 31u) & ~31u));
        const uint32_t np = p_last + ((warp * 32u < hs_last) ? 1u : 0u);   // packs with a live target in this warp (uniform)
        if (np == 0) continue;
        if constexpr (NPACK == 1) {
          event_pass<1, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
        } else {
          if (np == 1) event_pass<1, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else if (np == 2) event_pass<2, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else if (np == 3) event_pass<3, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
          else event_pass<4, TPB>(s_xy, s_z, s_id, s_next, n, i_first, p_last, hs_last, step, P, nonfinite);
        }
      }
      cluster.sync();                                                     // every CTA's new positions are in its s_next
      for (uint32_t base_i = 0, pass = 0; base_i < n; base_i += pass_sz, ++pass) {
        if (pass % CL == rank) continue;
        const float4* remote = cluster.map_shared_rank(s_next, pass % CL);
        const uint32_t hi_i = min(base_i + pass_sz, n);
        for (uint32_t i = base_i + tid; i < hi_i; i += TPB) s_next[i] = remote[i];
      }
      cluster.sync();                                                     // all pulls done before any s_next is rewritten
    }

    // ---- retire (rank 0): survivors (if max_steps stopped the event early) back to the state arrays, counters out
    if (rank != 0) continue;
    for (uint32_t i = tid; i < n; i += TPB) {
      A.x[off + i] = s_xy[i].x; A.y[off + i] = s_xy[i].z; A.z[off + i] = s_z[i].x; A.id[off + i] = s_id[i];
    }
    if (tid == 0) {
      ev.cnt[e] = n;
      ev.step[e] = step;
      if (s_coll) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_coll);
      if (s_over) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_over);
      if (pairs) atomicAdd((unsigned long long*)&ctrl->pairs, (unsigned long long)pairs);
    }
  }
  if (nonfinite) atomicOr(&ctrl->nonfinite, 1u);
}


// Events of at most 32 holes (a 100 eV deposit is 26 holes): ONE WARP OWNS ONE EVENT, one hole per lane,
// the state in registers for the event's whole life; a CTA is four such warps that never synchronise with each other.
// With a CTA per event (k_events<1,64,12>) such an event keeps 26 of 64 threads busy and pays three block barriers per
// step, and the per-hole FP64 update chain (Philox, Box-Muller, eq. 2) that dominates its step has one warp in two to
// hide its latency behind.  Per step: positions to the warp's 384 bytes of shared memory as x[], y[], z[] (dead lanes
// write the sentinel), so one LDS.64 per coordinate brings TWO consecutive sources as a packed pair; the field of lane
// t is accumulated over source pairs with the packed FP32x2 instructions of gc_field.cuh (even sources in the low
// half, odd in the high half, added at the end); advance_carrier as everywhere; collection by ballot, compaction by
// __fns + shuffle (stable).  Same arithmetic per pair and per hole as k_events; only the order of the FP32 field sum
// differs.
__global__ void __launch_bounds__(128)
k_events_warp(SoA A, EventTable ev, const uint32_t* __restrict__ order, uint32_t n_order, uint32_t* __restrict__ queue,
              Ctrl* __restrict__ ctrl, Sink sink, DevParams P, uint64_t max_steps) {
  __shared__ __align__(16) float s_pos[4][3][kEvCapMicro + 2];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  float* sx = s_pos[warp][0];
  float* sy = s_pos[warp][1];
  float* sz = s_pos[warp][2];
  const float2 eps2v = make_float2(P.eps2, P.eps2);
  uint32_t nonfinite = 0;

  for (;;) {
    uint32_t slot = 0;
    if (lane == 0) slot = atomicAdd(queue, 1u);
    slot = __shfl_sync(0xffffffffu, slot, 0);
    if (slot >= n_order) break;
    const uint32_t e = order[slot];
    const uint32_t off = ev.off[e];
    uint32_t n = ev.cnt[e];
    uint64_t step = ev.step[e];
    if (n == 0) continue;
    bool live = lane < n;
    float x = 0.f, y = 0.f, z = 0.f;
    uint32_t id = 0;
    if (live) { x = A.x[off + lane]; y = A.y[off + lane]; z = A.z[off + lane]; id = A.id[off + lane]; }
    uint64_t pairs = 0, done = 0;
    uint32_t n_coll = 0, n_over = 0;
    bool first = true;
    for (;;) {
      // ---- a7 + a8: bin the holes that crossed z_well, compact the survivors (stable)
      const bool crossed = live && (double)z <= P.z_well;
      uint32_t over = 0;
      if (crossed) collect(x, y, z, id, step, P, sink, over);
      n_coll += __popc(__ballot_sync(0xffffffffu, crossed));
      n_over += __popc(__ballot_sync(0xffffffffu, over != 0u));
      const uint32_t bal = __ballot_sync(0xffffffffu, live && !crossed);
      const uint32_t total = __popc(bal);
      const uint32_t src = lane < total ? __fns(bal, 0u, lane + 1u) : lane;     // lane of the (lane+1)-th survivor
      x = __shfl_sync(0xffffffffu, x, src); y = __shfl_sync(0xffffffffu, y, src); z = __shfl_sync(0xffffffffu, z, src);
      id = __shfl_sync(0xffffffffu, id, src);
      live = lane < total;
      if (!first) { step += 1; done += 1; if (!(P.flags & 1u)) pairs += (uint64_t)n * (uint64_t)n; }
      first = false;
      n = total;
      if (n == 0 || done >= max_steps) break;

      // ---- a1: field of lane's hole from all n sources, two sources per packed instruction
      float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax;
      if (!(P.flags & 1u)) {                                 // GCORECCD_COULOMB_OFF
        __syncwarp();                                        // last step's readers are done
        sx[lane] = live ? x : kSentinel; sy[lane] = live ? y : kSentinel; sz[lane] = live ? z : kSentinel;
        if (lane < 2) { sx[32 + lane] = kSentinel; sy[32 + lane] = kSentinel; sz[32 + lane] = kSentinel; }
        __syncwarp();
        const float2 ntx = make_float2(-x, -x), nty = make_float2(-y, -y), ntz = make_float2(-z, -z);
        for (uint32_t j = 0; j < n; j += 2) {
          const float2 px2 = *reinterpret_cast<const float2*>(sx + j), py2 = *reinterpret_cast<const float2*>(sy + j),
                       pz2 = *reinterpret_cast<const float2*>(sz + j);
          const float2 dx = __fadd2_rn(px2, ntx), dy = __fadd2_rn(py2, nty), dz = __fadd2_rn(pz2, ntz);
          float2 r2 = __ffma2_rn(dx, dx, eps2v);
          r2 = __ffma2_rn(dy, dy, r2);
          r2 = __ffma2_rn(dz, dz, r2);
          const float2 inv = make_float2(rsqrt_ftz(r2.x), rsqrt_ftz(r2.y));
          float2 w = __fmul2_rn(inv, inv);
          w = __fmul2_rn(w, inv);
          ax = __ffma2_rn(dx, w, ax); ay = __ffma2_rn(dy, w, ay); az = __ffma2_rn(dz, w, az);
        }
      }
      // ---- a2..a6
      if (live) {
        const double Ex = -P.Kp * (double)(ax.x + ax.y), Ey = -P.Kp * (double)(ay.x + ay.y), Ez = -P.Kp * (double)(az.x + az.y);
        float xf, yf, zf;
        if (!advance_carrier(x, y, z, id, step, Ex, Ey, Ez, P, xf, yf, zf)) nonfinite = 1u;
        x = xf; y = yf; z = zf;
      }
    }
    // ---- retire
    if (live) { A.x[off + lane] = x; A.y[off + lane] = y; A.z[off + lane] = z; A.id[off + lane] = id; }
    if (lane == 0) {
      ev.cnt[e] = n;
      ev.step[e] = step;
      if (n_coll) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)n_coll);
      if (n_over) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)n_over);
      if (pairs) atomicAdd((unsigned long long*)&ctrl->pairs, (unsigned long long)pairs);
    }
  }
  if (nonfinite) atomicOr(&ctrl->nonfinite, 1u);
}

// read_event_carriers: one event's survivors, SoA -> interleaved xyz
__global__ void __launch_bounds__(kTPB)
k_interleave_range(SoA A, uint32_t off, uint32_t n, float* __restrict__ xyz) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  xyz[3 * (size_t)i] = A.x[off + i]; xyz[3 * (size_t)i + 1] = A.y[off + i]; xyz[3 * (size_t)i + 2] = A.z[off + i];
}

// Scheduling hint only (never enters the physics): mean depth of each event, one warp per event.  The host orders
// every queue by the estimated work n^2 x (steps to drift home from that depth), longest first.
__global__ void __launch_bounds__(kTPB)
k_event_depth(SoA A, const uint32_t* __restrict__ off, const uint32_t* __restrict__ cnt, uint32_t n_events,
              float* __restrict__ zmean) {
  const uint32_t e = (blockIdx.x * kTPB + threadIdx.x) >> 5, lane = threadIdx.x & 31u;
  if (e >= n_events) return;
  const uint32_t o = off[e], n = cnt[e];
  float s = 0.f;
  for (uint32_t i = lane; i < n; i += 32) s += A.z[o + i];
  for (int k = 16; k > 0; k >>= 1) s += __shfl_xor_sync(0xffffffffu, s, k);
  if (lane == 0) zmean[e] = n ? s / (float)n : 0.f;
}

// Load path of the batch: interleaved xyz -> state arrays at the same index, ids id_base + index.
__global__ void __launch_bounds__(kTPB)
k_unpack_events(const float* __restrict__ xyz, uint32_t n, SoA A, uint32_t id_base) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  A.x[i] = xyz[3 * (size_t)i]; A.y[i] = xyz[3 * (size_t)i + 1]; A.z[i] = xyz[3 * (size_t)i + 2]; A.id[i] = id_base + i;
}

}  // namespace gc
