// gc_persist_warp.cuh — the smallest populations (N_a up to 32 targets per SM: 2,368 / 4,736 holes on 148 SMs):
// MANY TIME STEPS IN ONE LAUNCH, A WARP OWNS ITS TARGETS FOR THE WHOLE STEP.
//
// k_steps (gc_persist.cuh) cuts eq. 6 into (row block x source chunk) items like the big field kernel, so every step
// pays: grid barrier -> Ctrl / plan -> loads -> eq. 6 -> chunk partials to L2 -> grid barrier -> partials back from L2
// -> update -> scan -> write.  ncu at 4,096 holes (profiles/r2_persist_ncu.md): the FMA pipe is busy 5.6 of 16.2 us, the
// rest is that serial chain.  Here the roles are turned round.  Warp w of the grid owns targets [2 NP w, 2 NP (w + 1)):
// all 32 lanes hold the SAME NP packed pairs of targets and each lane takes every 32nd SOURCE from shared memory, so the
// whole sum of a target stays inside one warp.  A butterfly of shuffles (in FP64, fixed order) finishes eq. 6, and the
// warp goes straight on to a2..a8 for its own targets: no chunk partials, no plan, no barrier between the field and the
// update — ONE grid barrier per step.  One CTA per SM, 16 NP targets per CTA, NP = 1 or 2 by population, and only as
// many CTAs as the population needs (a CTA without targets would only slow the barrier down).  The Box-Muller chains of the warp's targets run on separate lanes before the
// source loop (their FP64 latency hides under the other warps' eq. 6), the update on one lane per target.
// Same interact<>, advance_with_normals, collect and Philox counters as every other path; the sum of eq. 6 is taken
// per lane in FP32 (flushed into a per-lane total after every source tile) and over the 32 lanes in FP64.
#pragma once
#include "gc_persist.cuh"

namespace gc {

constexpr int kWsTile = 2048;                  // sources per shared-memory tile, pre-duplicated (x,x,y,y) / (z,z): 48 KB
constexpr int kWsWarps = kTPB / 32;            // warps that OWN targets (8); with SPLIT = 2 eight more share their sources
constexpr uint32_t kWsSmemBytes = kWsTile * (sizeof(float4) + sizeof(float2));

__device__ __forceinline__ double shfl_xor_f64(double v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }

// SPLIT = 2: the CTA has 16 warps; warps w and w + 8 hold the SAME targets and take alternate groups of 32 sources, and
// the second warp's sums cross to the owner through shared memory: four warps per SM sub-partition instead of two.  Built
// to hide latency in the source loop; measured no faster there (16.0k cycles per step at 4,096 holes either way: 32 targets
// x 4,096 sources per SM cost 13k cycles at the operand-read rate of DESIGN.md 6.1) and slower overall, so the host
// instantiates SPLIT = 1.
template <int NP, int SPLIT>
__global__ void __launch_bounds__(kTPB * SPLIT, 1)
k_steps_warp(SoA A, SoA B, Ctrl* ctrl, Sink sink, unsigned long long* status, DevParams P, PlanArgs pa, uint32_t n_steps,
             uint32_t n_exit) {
  extern __shared__ __align__(16) unsigned char ws_smem[];
  float4* s_xy = reinterpret_cast<float4*>(ws_smem);
  float2* s_z = reinterpret_cast<float2*>(ws_smem + sizeof(float4) * kWsTile);
  __shared__ double s_bm[2][5][kWsWarps * 8];    // Box-Muller chains Ra, sa, ca, Rb, cb of the CTA's <= 64 targets: [k & 1] this step's
  __shared__ double s_e[3][kWsWarps * 8];        // SPLIT = 2: the second warp's sums of eq. 6, per target
  constexpr int kThreads = kTPB * SPLIT;
  constexpr int kWsPre = kWsTile / kThreads;     // sources a thread stages per tile
  __shared__ uint32_t s_w[16];
  __shared__ uint32_t s_n;
  __shared__ unsigned long long s_step;
  constexpr uint32_t TW = 2 * NP;              // targets per warp (2, 4 or 8)
  constexpr uint32_t kFull = 0xffffffffu;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t wt = warp % (uint32_t)kWsWarps, ws = warp / (uint32_t)kWsWarps;   // target group, source share
  const uint32_t G = gridDim.x;
  const uint32_t seq0 = ld_acquire_u32(&ctrl->scan_seq);
  const float2 eps2v = make_float2(P.eps2, P.eps2);
  uint32_t arrivals = 0;
  uint32_t k = 0;
  uint32_t n_hi = 0;                           // the previous step's population (0: first step of the launch)
  uint32_t spec_n = 0;                         // population for which s_bm[k & 1] already holds this step's chains (0: none)
  // the state ping-pongs between A and B as in k_steps: no slot is overwritten while another CTA may still read it
  for (; k < n_steps; ++k) {
    const SoA cur = (k & 1u) ? B : A, nxt = (k & 1u) ? A : B;
    if (tid == 0) {
      s_n = __ldcg(&ctrl->n_active);
      s_step = __ldcg(reinterpret_cast<const unsigned long long*>(&ctrl->step));
    }
    // This warp's targets (lane l < TW holds target i0 + l) and the first source tile.  From the second step on they
    // are requested BEFORE Ctrl has arrived, against the previous step's population n_hi >= n (the arrays are padded,
    // the slots exist), and masked once n is known: one L2 round trip per step instead of two.
    const uint32_t i0 = (blockIdx.x * (uint32_t)kWsWarps + wt) * TW;          // the host keeps n <= TW * 8 * G
    const bool cta_hi = blockIdx.x * (uint32_t)kWsWarps * TW < n_hi;
    float x = 0.f, y = 0.f, z = 0.f; uint32_t id = 0;
    float px[kWsPre], py[kWsPre], pz[kWsPre];
    if (n_hi) {
      if (lane < TW && i0 + lane < n_hi) { x = __ldcg(cur.x + i0 + lane); y = __ldcg(cur.y + i0 + lane); z = __ldcg(cur.z + i0 + lane); id = __ldcg(cur.id + i0 + lane); }
#pragma unroll
      for (int u = 0; u < kWsPre; ++u) {
        const uint32_t j = (uint32_t)u * kThreads + tid;
        const bool ok = cta_hi && j < n_hi;
        px[u] = ok ? __ldcg(cur.x + j) : kSentinel; py[u] = ok ? __ldcg(cur.y + j) : kSentinel; pz[u] = ok ? __ldcg(cur.z + j) : kSentinel;
      }
    }
    GC_T(0);
    __syncthreads();
    GC_T(1);
    const uint32_t n = s_n;
    if (n == 0 || n < n_exit) break;                         // uniform over the grid; n_exit: a smaller variant takes over
    const uint64_t step = s_step;
    const uint32_t stamp = scan_stamp(seq0 + k);
    const bool warp_active = i0 < n;
    const bool hold = lane < TW && i0 + lane < n;             // this lane holds a target's coordinates ...
    const bool have = hold && ws == 0u;                      // ... and is the one that advances it
    // (a CTA none of whose warps has a target only takes part in the scan and the barrier)
    const bool cta_active = blockIdx.x * (uint32_t)kWsWarps * TW < n;
    if (n_hi) {
      if (!hold) { x = y = z = 0.f; id = 0; }
#pragma unroll
      for (int u = 0; u < kWsPre; ++u) {
        const bool ok = cta_active && (uint32_t)u * kThreads + tid < n;
        if (!ok) { px[u] = kSentinel; py[u] = kSentinel; pz[u] = kSentinel; }
      }
    } else {
      if (hold) { x = __ldcg(cur.x + i0 + lane); y = __ldcg(cur.y + i0 + lane); z = __ldcg(cur.z + i0 + lane); id = __ldcg(cur.id + i0 + lane); }
#pragma unroll
      for (int u = 0; u < kWsPre; ++u) {
        const uint32_t j = (uint32_t)u * kThreads + tid;
        const bool ok = cta_active && j < n;
        px[u] = ok ? __ldcg(cur.x + j) : kSentinel; py[u] = ok ? __ldcg(cur.y + j) : kSentinel; pz[u] = ok ? __ldcg(cur.z + j) : kSentinel;
      }
    }
    n_hi = n;
    float2 ntx[NP], nty[NP], ntz[NP], tx[NP], ty[NP], tz[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      ntx[p] = make_float2(-__shfl_sync(kFull, x, 2 * p), -__shfl_sync(kFull, x, 2 * p + 1));
      nty[p] = make_float2(-__shfl_sync(kFull, y, 2 * p), -__shfl_sync(kFull, y, 2 * p + 1));
      ntz[p] = make_float2(-__shfl_sync(kFull, z, 2 * p), -__shfl_sync(kFull, z, 2 * p + 1));
      tx[p] = make_float2(0.f, 0.f); ty[p] = tx[p]; tz[p] = tx[p];
    }

    // ---- a5, field-independent half: the four Box-Muller chains (Ra | sa, ca | Rb | cb) of the CTA's T = 8 TW targets.
    // Warp w runs ONE kind of chain (w & 3) for 32 targets (half w >> 2), so no warp diverges over the three code paths
    // and the chains of all targets run side by side; the results cross to the owner lanes through shared memory (the
    // barriers of the source loop below order them).  Skipped when the previous step already drew them while it waited
    // at the grid barrier (see there).
    const uint32_t cb = k & 1u;
    auto draw_chains = [&](uint32_t buf, uint64_t for_step) {
      const uint32_t kq = (warp >> 2) * 32u + lane, kind = warp & 3u;            // target within the CTA, chain kind
      const uint32_t ig = blockIdx.x * (uint32_t)kWsWarps * TW + kq;
      if (kq < (uint32_t)kWsWarps * TW && ig < n) {
        const uint4 w = philox_words(P.seed_lo, P.seed_hi, __ldcg(cur.id + ig), for_step);
        if (kind == 0u) s_bm[buf][0][kq] = bm_radius(w.x);
        else if (kind == 1u) { double sa, ca; sincospi(2.0 * bm_fraction(w.y), &sa, &ca); s_bm[buf][1][kq] = sa; s_bm[buf][2][kq] = ca; }
        else if (kind == 2u) s_bm[buf][3][kq] = bm_radius(w.z);
        else s_bm[buf][4][kq] = cospi(2.0 * bm_fraction(w.w));
      }
    };
    const bool diffuse = cta_active && !(P.flags & 2u);
    if (diffuse && spec_n != n) draw_chains(cb, step);

    GC_T(2);
    // ---- a1: every source against the warp's targets, lane l taking sources l, l + 32, ... of each tile
    for (uint32_t j0 = 0; cta_active && j0 < n; j0 += kWsTile) {
      __syncthreads();                                       // readers of the previous tile are done
#pragma unroll
      for (int u = 0; u < kWsPre; ++u) {
        const uint32_t s = (uint32_t)u * kThreads + tid;
        s_xy[s] = make_float4(px[u], px[u], py[u], py[u]);
        s_z[s] = make_float2(pz[u], pz[u]);
      }
      __syncthreads();
      if (j0 + kWsTile < n) {                                // next tile into registers while this one is consumed
#pragma unroll
        for (int u = 0; u < kWsPre; ++u) {
          const uint32_t j = j0 + kWsTile + (uint32_t)u * kThreads + tid;
          const bool ok = j < n;
          px[u] = ok ? __ldcg(cur.x + j) : kSentinel; py[u] = ok ? __ldcg(cur.y + j) : kSentinel; pz[u] = ok ? __ldcg(cur.z + j) : kSentinel;
        }
      }
      if (warp_active) {
        constexpr uint32_t kStride = 32u * SPLIT;            // sources of a tile go round the SPLIT warps of a target group
        const int len = (int)min((uint32_t)kWsTile, (n - j0 + kStride - 1u) & ~(kStride - 1u));   // padded with sentinels
        float2 ax[NP], ay[NP], az[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) { ax[p] = make_float2(0.f, 0.f); ay[p] = ax[p]; az[p] = ax[p]; }
#pragma unroll (SPLIT >= 2 ? 2 : 4)
        for (int jj = (int)(lane + 32u * ws); jj < len; jj += (int)kStride) interact<NP>(s_xy[jj], s_z[jj], ntx, nty, ntz, eps2v, ax, ay, az);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
          tx[p] = __fadd2_rn(tx[p], ax[p]); ty[p] = __fadd2_rn(ty[p], ay[p]); tz[p] = __fadd2_rn(tz[p], az[p]);
        }
      }
    }

    GC_T(3);
    // ---- the 32 lanes' sums -> every lane, in FP64 (a butterfly: the same bits on every lane, the same order every
    // run); lane l < TW keeps the field of its own target
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
    if (SPLIT > 1) {                                         // the second warp's sums cross to the owner (fixed order: + second)
      if (ws == 1u && hold) { s_e[0][wt * TW + lane] = ex; s_e[1][wt * TW + lane] = ey; s_e[2][wt * TW + lane] = ez; }
      __syncthreads();
      if (have) { ex += s_e[0][wt * TW + lane]; ey += s_e[1][wt * TW + lane]; ez += s_e[2][wt * TW + lane]; }
    }
    // ---- a2..a6 on one lane per target; the normal triple comes from the chain warps
    float xf = 0.f, yf = 0.f, zf = 0.f;
    bool finite = true;
    if (have) {
      const uint32_t kq = wt * TW + lane;
      double nrm[3] = {0.0, 0.0, 0.0};
      if (!(P.flags & 2u)) { nrm[0] = s_bm[cb][0][kq] * s_bm[cb][2][kq]; nrm[1] = s_bm[cb][0][kq] * s_bm[cb][1][kq]; nrm[2] = s_bm[cb][3][kq] * s_bm[cb][4][kq]; }
      finite = advance_with_normals(x, y, z, -P.Kp * ex, -P.Kp * ey, -P.Kp * ez, nrm, P, xf, yf, zf);   // sums hold (r_s - r_t) w
    }

    GC_T(4);
    // ---- a7, a8: collection, then stable compaction: tile = this CTA's 8 TW targets, tiles in CTA order
    uint32_t coll = 0, over = 0;
    bool keep = false;
    if (have) {
      if (!finite) atomicOr(&ctrl->nonfinite, 1u);
      if ((double)zf <= P.z_well) { coll = 1; collect(xf, yf, zf, id, step, P, sink, over); }
      else keep = true;
    }
    if (tid < 16) s_w[tid] = 0;
    __syncthreads();
    const uint32_t bal = __ballot_sync(kFull, keep);
    const uint32_t rank_in_warp = __popc(bal & ((1u << lane) - 1u));
    const uint32_t wc = __popc(__ballot_sync(kFull, coll)), wo = __popc(__ballot_sync(kFull, over));
    if (lane == 0 && ws == 0u) {
      s_w[warp] = __popc(bal);
      if (wc) atomicAdd(&s_w[9], wc);
      if (wo) atomicAdd(&s_w[10], wo);
    }
    __syncthreads();
    if (warp == 0) {
      uint32_t count = 0;
#pragma unroll
      for (int w = 0; w < kWsWarps; ++w) count += s_w[w];
      const uint32_t excl = scan_two_level(status, blockIdx.x, stamp, count);   // every CTA publishes, empty tiles 0
      if (lane == 0) {
        s_w[8] = excl;
        if (s_w[9]) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_w[9]);
        if (s_w[10]) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_w[10]);
        if (blockIdx.x == G - 1u) {                          // the last tile's inclusive prefix is the new population;
          ctrl->n_active = excl + count;                     // every other CTA read Ctrl before it published its count
          ctrl->step = step + 1u;
          ctrl->pairs += (uint64_t)n * (uint64_t)n;
        }
      }
    }
    __syncthreads();
    if (keep) {
      uint32_t off = s_w[8] + rank_in_warp;
      for (uint32_t w = 0; w < warp; ++w) off += s_w[w];
      nxt.x[off] = xf; nxt.y[off] = yf; nxt.z[off] = zf; nxt.id[off] = id;
    }
    GC_T(5);
    arrivals += G;
    grid_arrive(&ctrl->bar);
    GC_T(6);
    // While the other CTAs arrive: if nobody anywhere is collected in this step (the usual case: holes arrive in a burst
    // at the end of an event), the next step finds the same carriers in the same slots, so their normals for step + 1 can
    // be drawn now, in time the CTA would spend polling.  The next step uses them iff its population equals this one's
    // (the population only shrinks, so equal means nobody left), and draws them itself otherwise.
    spec_n = 0;
    if (diffuse && k + 1u < n_steps) { draw_chains(cb ^ 1u, step + 1u); spec_n = n; }
    grid_wait(&ctrl->bar, arrivals);
    GC_T(7);
  }
  // an odd number of steps leaves the state in B: bring it home (every CTA is past the last barrier; B is complete)
  if (k & 1u) {
    if (tid == 0) s_n = __ldcg(&ctrl->n_active);
    __syncthreads();
    const uint32_t n = s_n;
    for (uint32_t i = blockIdx.x * kThreads + tid; i < n; i += gridDim.x * kThreads) {
      A.x[i] = __ldcg(B.x + i); A.y[i] = __ldcg(B.y + i); A.z[i] = __ldcg(B.z + i); A.id[i] = __ldcg(B.id + i);
    }
  }
  // exit: the last CTA out re-arms the barrier, accounts for the scans and leaves a FieldPlan for whoever runs next
  // (eval_field, a two-launch step): this kernel needs none, so Ctrl's plan is stale while it runs
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_w[0] = atomicAdd(&ctrl->bar_exit, 1u) == gridDim.x - 1u ? 1u : 0u;
  }
  __syncthreads();
  if (s_w[0] && tid < 32) {
    __threadfence();
    const FieldPlan np = plan_search(__ldcg(&ctrl->n_active), pa);
    if (tid == 0) {
      ctrl->plan = np;
      ctrl->bar = 0;
      ctrl->bar_exit = 0;
      ctrl->scan_seq = seq0 + k;
    }
  }
}

}  // namespace gc
