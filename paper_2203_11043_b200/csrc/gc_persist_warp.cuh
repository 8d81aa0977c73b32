// gc_persist_warp.cuh — the smallest populations (N_a up to 32 targets per SM: 2,368 / 4,736 holes on 148 SMs):
// MANY TIME STEPS IN ONE LAUNCH, A WARP OWNS ITS TARGETS FOR THE WHOLE STEP, A CTA KEEPS ITS CARRIERS FOR THE WHOLE LAUNCH.
//
// k_steps (gc_persist.cuh) cuts eq. 6 into (row block x source chunk) items like the big field kernel, so every step
// pays: grid barrier -> Ctrl / plan -> loads -> eq. 6 -> chunk partials to L2 -> grid barrier -> partials back from L2
// -> update -> scan -> write.  ncu at 4,096 holes (profiles/r2_persist_ncu.md): the FMA pipe is busy 5.6 of 16.2 us, the
// rest is that serial chain.  Here the roles are turned round.
//   * A warp owns 2 NP targets: all 32 lanes hold the SAME NP packed pairs of targets and each lane takes every 32nd
//     SOURCE from a shared-memory tile, so the whole sum of a target stays inside one warp.  A butterfly of shuffles (in
//     FP64, fixed order) finishes eq. 6 and the warp goes straight on to a2..a8 for its own targets: no chunk partials,
//     no plan, no barrier between the field and the update — ONE grid barrier per step.  One CTA of 8 warps per SM,
//     NP = 1 or 2 by population, and only as many CTAs as the population needs.
//   * A CTA keeps the carriers it was dealt at launch (T = 16 NP of them) and compacts its survivors LOCALLY; it writes
//     them at (prefix of its segment in the state it read) + (rank among its survivors) and stores its survivor count
//     in a word of its own before it arrives at the barrier.  After the barrier every CTA reads all the words (one per
//     thread, once): the population and the prefix of every segment — the scan costs one read instead of two rounds
//     of polling, and the state is dense again as soon as a step collects nobody.  (The first
//     form of this kernel compacted globally with the two-level scan of gc_advance.cuh before the barrier: 6.3 / 13.8 us
//     per step at 1,024 / 4,096 holes against 5.8 / 13.6 us.)
//   * The concatenation of the segments IS the stable compacted order; sources are staged in that order (dense
//     state: index = slot; after a step that collected somebody through a map laid out in shared memory), so every
//     FP32 sum is
//     taken in the order a dense state would give: results do not depend on how a run is cut into launches.
//   * A CTA's targets of the next step are its own survivors: they stay in shared memory, and their Box-Muller
//     chains for the next step are drawn (one KIND of chain per warp: no divergence) while the other CTAs arrive.
//   * Ctrl is read once per launch and written once, at exit, where the segments are copied to their dense places
//     (every CTA holds its own carriers in shared memory, so that needs no further synchronisation).
// Same interact<>, advance_with_normals, collect and Philox counters as every other path; the sum of eq. 6 is taken
// per lane in FP32 (flushed into a per-lane total after every source tile) and over the 32 lanes in FP64.
#pragma once
#include "gc_persist.cuh"

namespace gc {

constexpr int kWsTile = 2048;                  // sources per shared-memory tile, pre-duplicated (x,x,y,y) / (z,z): 48 KB
constexpr int kWsWarps = kTPB / 32;            // warps per CTA
constexpr uint32_t kWsSmemBytes = kWsTile * (sizeof(float4) + sizeof(float2));
constexpr int kSegMaxCtas = 160;               // grid <= SM count (148 on B200)
constexpr uint32_t kSegWordStride = 256;       // count words of step parity p: status[256 p .. 256 p + G)

__device__ __forceinline__ double shfl_xor_f64(double v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }

template <int NP>
__global__ void __launch_bounds__(kTPB, 1)
k_steps_warp(SoA A, SoA B, Ctrl* ctrl, Sink sink, unsigned long long* status, DevParams P, PlanArgs pa, uint32_t n_steps,
            uint32_t n_exit) {
  extern __shared__ __align__(16) unsigned char ws_smem[];
  float4* s_xy = reinterpret_cast<float4*>(ws_smem);
  float2* s_z = reinterpret_cast<float2*>(ws_smem + sizeof(float4) * kWsTile);
  constexpr uint32_t TW = 2 * NP;              // targets per warp
  constexpr uint32_t T = kWsWarps * TW;        // slots per CTA (16 or 32)
  constexpr uint32_t kFull = 0xffffffffu;
  constexpr int kPre = kWsTile / kTPB;         // sources a thread stages per tile
  __shared__ double s_bm[5][T];                // Box-Muller chains Ra, sa, ca, Rb, cb of the CTA's carriers
  __shared__ float s_cx[T], s_cy[T], s_cz[T];  // the CTA's own carriers (front of its segment), this step's targets
  __shared__ uint32_t s_cid[T];
  __shared__ uint32_t s_cnt[kSegMaxCtas], s_pre[kSegMaxCtas + 1], s_start[kSegMaxCtas], s_ct[kWsWarps];
  __shared__ unsigned short s_inv[kSegMaxCtas * 32];   // compacted index -> slot, when the state is not dense
  __shared__ uint32_t s_w[16];
  __shared__ uint32_t s_n;
  __shared__ unsigned long long s_step;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t G = gridDim.x, b = blockIdx.x;
  const uint32_t seq0 = ld_acquire_u32(&ctrl->scan_seq);
  const float2 eps2v = make_float2(P.eps2, P.eps2);
  unsigned long long pairs = 0;                // sum of n^2 over the steps taken (identical in every CTA)
  uint32_t k = 0, arrivals = 0;
  uint32_t n_prev = 0, cnt_own = 0;            // the previous step's population; this CTA's carriers after its last commit

  // Box-Muller chains of the CTA's `cnt` carriers (ids in s_cid) for step `for_step`: one KIND of chain per warp
  auto draw_chains = [&](uint32_t cnt, uint64_t for_step) {
    const uint32_t kq = (warp >> 2) * 32u + lane, kind = warp & 3u;
    if (kq < cnt) {
      const uint4 w = philox_words(P.seed_lo, P.seed_hi, s_cid[kq], for_step);
      if (kind == 0u) s_bm[0][kq] = bm_radius(w.x);
      else if (kind == 1u) { double sa, ca; sincospi(2.0 * bm_fraction(w.y), &sa, &ca); s_bm[1][kq] = sa; s_bm[2][kq] = ca; }
      else if (kind == 2u) s_bm[3][kq] = bm_radius(w.z);
      else s_bm[4][kq] = cospi(2.0 * bm_fraction(w.w));
    }
  };

  for (;; ++k) {
    // the state of step k is segmented in `cur` (dense at k = 0); step k writes the survivors' segments into `nxt`
    const SoA cur = (k & 1u) ? B : A, nxt = (k & 1u) ? A : B;
    // ---- segment counts of state k: from Ctrl at k = 0, else the words the CTAs stored before the barrier just left
    uint32_t c_mine = 0;                                     // thread t < G: carriers in segment t
    if (k == 0) {
      if (tid == 0) {
        s_n = __ldcg(&ctrl->n_active);
        s_step = __ldcg(reinterpret_cast<const unsigned long long*>(&ctrl->step));
      }
      __syncthreads();
      const uint32_t n0 = s_n;
      if (tid < G) c_mine = n0 > tid * T ? min(T, n0 - tid * T) : 0u;
      const uint32_t c0 = n0 > b * T ? min(T, n0 - b * T) : 0u;
      if (tid < c0) {
        s_cx[tid] = __ldcg(A.x + b * T + tid); s_cy[tid] = __ldcg(A.y + b * T + tid); s_cz[tid] = __ldcg(A.z + b * T + tid);
        s_cid[tid] = __ldcg(A.id + b * T + tid);
      }
    } else {
      // (one read, no polling: 22,000 threads polling 148 stamped words instead of an arrival counter were tried and
      // were slower — the words' lines thrash)
      if (tid < G) c_mine = (uint32_t)ld_relaxed_u64(status + ((k - 1u) & 1u) * kSegWordStride + tid);
    }
    // Where segment t of `cur` begins: where its owner wrote it, i.e. at the prefix the owner knew THEN (state k - 1's).
    const uint32_t old_pre_mine = (k > 0 && tid < G) ? s_pre[tid] : 0u;
    // The first source tile is requested at once, as if nobody had been collected in the step before (then `cur` is
    // dense and as long as it was), so that its L2 round trip overlaps the count words': the usual case.
    float px[kPre], py[kPre], pz[kPre];
    const bool spec = k > 0 && cnt_own > 0;
    if (spec) {
#pragma unroll
      for (int u = 0; u < kPre; ++u) {
        const uint32_t j = (uint32_t)u * kTPB + tid;
        const bool ok = j < n_prev;
        px[u] = ok ? __ldcg(cur.x + j) : kSentinel; py[u] = ok ? __ldcg(cur.y + j) : kSentinel; pz[u] = ok ? __ldcg(cur.z + j) : kSentinel;
      }
    }
    GC_T(0);
    // exclusive prefix of the counts: warps 0..4 scan 32 segments each, the chunk totals cross through shared memory
    uint32_t inc = c_mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(kFull, inc, o); if ((int)lane >= o) inc += v; }
    if (lane == 31u) s_ct[warp] = inc;
    __syncthreads();
    uint32_t base = 0, n = 0;
#pragma unroll
    for (int w = 0; w < kWsWarps; ++w) { const uint32_t c = s_ct[w]; if ((uint32_t)w < warp) base += c; n += c; }
    const uint32_t pre_mine = base + inc - c_mine;
    if (tid < G) { s_cnt[tid] = c_mine; s_pre[tid] = pre_mine; s_start[tid] = k > 0 ? old_pre_mine : pre_mine; }
    if (tid == 0) { s_pre[G] = n; s_n = n; }
    __syncthreads();
    GC_T(1);
    // `cur` is dense (slot = compacted index) iff nobody was collected in the step that wrote it: every survivor went to
    // (prefix of its segment) + (rank in its segment), and those prefixes are still the right ones
    const bool dense = k == 0 || n == n_prev;
    if (k == n_steps || n == 0 || n < n_exit) break;         // uniform over the grid; n_exit: a smaller variant takes over
    const uint64_t step = s_step + k;
    const uint32_t cnt = s_cnt[b];                           // this CTA's carriers
    const bool cta_active = cnt > 0;
    pairs += (unsigned long long)n * (unsigned long long)n;
    // compacted index j -> slot of `cur`.  After a step that collected somebody the segments do not abut: a map is laid
    // out in shared memory, one warp per segment at a time (a binary search per source over the prefix table was tried
    // first: 5,700 cycles per 2,048-source tile; this is ~600 per step)
    if (!dense && cta_active) {
      for (uint32_t t0 = warp; t0 < G; t0 += 5u * (uint32_t)kWsWarps) {     // five segments' table entries in flight
        uint32_t c[5], q[5], a[5];
#pragma unroll
        for (int u = 0; u < 5; ++u) {
          const uint32_t t = min(t0 + (uint32_t)u * (uint32_t)kWsWarps, G - 1u);
          c[u] = t0 + (uint32_t)u * (uint32_t)kWsWarps < G ? s_cnt[t] : 0u; q[u] = s_pre[t]; a[u] = s_start[t];
        }
#pragma unroll
        for (int u = 0; u < 5; ++u) if (lane < c[u]) s_inv[q[u] + lane] = (unsigned short)(a[u] + lane);
      }
      __syncthreads();
    }
    auto slot_of = [&](uint32_t j) -> uint32_t { return dense ? j : (uint32_t)s_inv[j]; };
    if (!(spec && dense)) {                                  // somebody was collected (or first step): stage with the table
#pragma unroll
      for (int u = 0; u < kPre; ++u) {
        const uint32_t j = (uint32_t)u * kTPB + tid;
        const bool ok = cta_active && j < n;
        const uint32_t a = ok ? slot_of(j) : 0u;
        px[u] = ok ? __ldcg(cur.x + a) : kSentinel; py[u] = ok ? __ldcg(cur.y + a) : kSentinel; pz[u] = ok ? __ldcg(cur.z + a) : kSentinel;
      }
    }
    n_prev = n;
    if (k == 0 && cta_active && !(P.flags & 2u)) draw_chains(cnt, step);   // later steps: drawn at the end of the step before

    // ---- this warp's targets: slots [warp TW, warp TW + TW) of the CTA's segment, from shared memory
    const uint32_t q0 = warp * TW;
    const bool warp_active = q0 < cnt;
    const bool have = lane < TW && q0 + lane < cnt;
    float x = 0.f, y = 0.f, z = 0.f; uint32_t id = 0;
    if (have) { x = s_cx[q0 + lane]; y = s_cy[q0 + lane]; z = s_cz[q0 + lane]; id = s_cid[q0 + lane]; }
    float2 ntx[NP], nty[NP], ntz[NP], tx[NP], ty[NP], tz[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      ntx[p] = make_float2(-__shfl_sync(kFull, x, 2 * p), -__shfl_sync(kFull, x, 2 * p + 1));
      nty[p] = make_float2(-__shfl_sync(kFull, y, 2 * p), -__shfl_sync(kFull, y, 2 * p + 1));
      ntz[p] = make_float2(-__shfl_sync(kFull, z, 2 * p), -__shfl_sync(kFull, z, 2 * p + 1));
      tx[p] = make_float2(0.f, 0.f); ty[p] = tx[p]; tz[p] = tx[p];
    }
    GC_T(2);
    // ---- a1: every source (in compacted order) against the warp's targets, lane l taking sources l, l + 32, ... of a tile
    for (uint32_t j0 = 0; cta_active && j0 < n; j0 += kWsTile) {
      __syncthreads();                                       // readers of the previous tile are done
#pragma unroll
      for (int u = 0; u < kPre; ++u) {
        const uint32_t s = (uint32_t)u * kTPB + tid;
        s_xy[s] = make_float4(px[u], px[u], py[u], py[u]);
        s_z[s] = make_float2(pz[u], pz[u]);
      }
      __syncthreads();
      if (j0 + kWsTile < n) {                                // next tile into registers while this one is consumed
#pragma unroll
        for (int u = 0; u < kPre; ++u) {
          const uint32_t j = j0 + kWsTile + (uint32_t)u * kTPB + tid;
          const bool ok = j < n;
          const uint32_t a = ok ? slot_of(j) : 0u;
          px[u] = ok ? __ldcg(cur.x + a) : kSentinel; py[u] = ok ? __ldcg(cur.y + a) : kSentinel; pz[u] = ok ? __ldcg(cur.z + a) : kSentinel;
        }
      }
      if (warp_active) {
        const int len = (int)min((uint32_t)kWsTile, (n - j0 + 31u) & ~31u);   // padded with sentinels to whole warps
        float2 ax[NP], ay[NP], az[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) { ax[p] = make_float2(0.f, 0.f); ay[p] = ax[p]; az[p] = ax[p]; }
#pragma unroll 4
        for (int jj = (int)lane; jj < len; jj += 32) interact<NP>(s_xy[jj], s_z[jj], ntx, nty, ntz, eps2v, ax, ay, az);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
          tx[p] = __fadd2_rn(tx[p], ax[p]); ty[p] = __fadd2_rn(ty[p], ay[p]); tz[p] = __fadd2_rn(tz[p], az[p]);
        }
      }
    }
    GC_T(3);
    // ---- the 32 lanes' sums -> every lane, in FP64 (a butterfly: same bits on every lane, same order every run)
    double ex = 0.0, ey = 0.0, ez = 0.0;
    if (warp_active) {
#pragma unroll
      for (int p = 0; p < NP; ++p) {
        double v[6] = {(double)tx[p].x, (double)tx[p].y, (double)ty[p].x, (double)ty[p].y, (double)tz[p].x, (double)tz[p].y};
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
          for (int c = 0; c < 6; ++c) v[c] += shfl_xor_f64(v[c], o);
        }
        if (lane == 2u * p) { ex = v[0]; ey = v[2]; ez = v[4]; }
        if (lane == 2u * p + 1u) { ex = v[1]; ey = v[3]; ez = v[5]; }
      }
    }
    // ---- a2..a6 on one lane per target
    float xf = 0.f, yf = 0.f, zf = 0.f;
    bool finite = true;
    if (have) {
      const uint32_t kq = q0 + lane;
      double nrm[3] = {0.0, 0.0, 0.0};
      if (!(P.flags & 2u)) { nrm[0] = s_bm[0][kq] * s_bm[2][kq]; nrm[1] = s_bm[0][kq] * s_bm[1][kq]; nrm[2] = s_bm[3][kq] * s_bm[4][kq]; }
      finite = advance_with_normals(x, y, z, -P.Kp * ex, -P.Kp * ey, -P.Kp * ez, nrm, P, xf, yf, zf);   // sums hold (r_s - r_t) w
    }
    GC_T(4);
    // ---- a7, a8: collection; the survivors go, in order, to the front of the CTA's segment of `nxt` and stay in
    // shared memory as the next step's targets
    uint32_t coll = 0, over = 0;
    bool keep = false;
    if (have) {
      if (!finite) atomicOr(&ctrl->nonfinite, 1u);
      if ((double)zf <= P.z_well) { coll = 1; collect(xf, yf, zf, id, step, P, sink, over); }
      else keep = true;
    }
    if (tid < 16) s_w[tid] = 0;
    __syncthreads();                                         // (also: every warp has read its targets and chains)
    const uint32_t bal = __ballot_sync(kFull, keep);
    const uint32_t rank_in_warp = __popc(bal & ((1u << lane) - 1u));
    const uint32_t wc = __popc(__ballot_sync(kFull, coll)), wo = __popc(__ballot_sync(kFull, over));
    if (lane == 0) {
      s_w[warp] = __popc(bal);
      if (wc) atomicAdd(&s_w[9], wc);
      if (wo) atomicAdd(&s_w[10], wo);
    }
    __syncthreads();
    uint32_t cnt_new = 0;
#pragma unroll
    for (int w = 0; w < kWsWarps; ++w) cnt_new += s_w[w];
    if (keep) {
      uint32_t r = rank_in_warp;
      for (uint32_t w = 0; w < warp; ++w) r += s_w[w];
      s_cx[r] = xf; s_cy[r] = yf; s_cz[r] = zf; s_cid[r] = id;
      const uint32_t a = s_pre[b] + r;                       // this state's prefix: dense again if nobody is collected
      nxt.x[a] = xf; nxt.y[a] = yf; nxt.z[a] = zf;           // (ids travel with the owner; sources need coordinates only)
    }
    if (tid == 0) {
      if (s_w[9]) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_w[9]);
      if (s_w[10]) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_w[10]);
    }
    GC_T(5);
    // ---- the survivor count goes into this CTA's word (two sets of words, by step parity: a word is rewritten two
    // barriers later, when every CTA has read it), then the CTA arrives at the step's only grid barrier: the arrival's
    // release orders the word and the whole CTA's carriers before it
    if (tid == 0) st_relaxed_u64(status + (k & 1u) * kSegWordStride + b, (unsigned long long)cnt_new);
    cnt_own = cnt_new;
    arrivals += G;
    grid_arrive(&ctrl->bar);
    GC_T(6);
    // while the other CTAs arrive: the next step's normals of the carriers this CTA now holds
    if (cnt_new && !(P.flags & 2u) && k + 1u < n_steps) draw_chains(cnt_new, step + 1u);
    grid_wait(&ctrl->bar, arrivals);
    GC_T(7);
  }

  // ---- exit: state k is segmented in (k odd ? B : A); every CTA holds its own carriers in shared memory and knows
  // every segment's prefix, so it writes them to their dense places in A without reading global memory again.  No CTA
  // reads the state any more (all are past the words of step k - 1), so A may be overwritten in place.
  {
    const uint32_t cnt = s_cnt[b], base = s_pre[b];
    if (k > 0 && tid < cnt) {                                // (k = 0: nothing was stepped, A is as it was)
      A.x[base + tid] = s_cx[tid]; A.y[base + tid] = s_cy[tid]; A.z[base + tid] = s_cz[tid]; A.id[base + tid] = s_cid[tid];
    }
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_w[0] = atomicAdd(&ctrl->bar_exit, 1u) == gridDim.x - 1u ? 1u : 0u;
  }
  __syncthreads();
  if (s_w[0] && tid < 32) {                                  // the last CTA out publishes the launch's outcome
    __threadfence();
    const FieldPlan np = plan_search(s_n, pa);
    if (tid == 0) {
      ctrl->plan = np;
      ctrl->n_active = s_n;
      ctrl->step = s_step + k;
      ctrl->pairs += pairs;
      ctrl->bar = 0;
      ctrl->bar_exit = 0;
      ctrl->scan_seq = seq0 + k;
    }
  }
}

}  // namespace gc
