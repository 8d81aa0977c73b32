// gc_field.cuh — step a1: all-pairs softened Coulomb field, eq. 6:
//     S_t = sum_{s=1..N_a} (r_t - r_s) / (|r_t - r_s|^2 + eps^2)^{3/2},   E_t = K' S_t
// (t = target = the paper's j, s = source = the paper's i; the s = t term is included and is exactly 0).
//
// Roofline: plain FP32 ALUs (FMA pipe), NOT tensor cores (no dense contraction) and not memory (positions
// are 12 B x N_a, L2 resident).  Per interaction: 3 add, 3 fma (r^2 + eps^2), 1 rsqrt, 2 mul, 3 fma
// = 11 FP32-pipe lane-ops + 1 MUFU, counted as 20 FLOP by the GPU Gems 3 ch. 31 convention.
//
// Design (differs from the paper's kernel, which is one thread = one carrier with a
// blockDim-sized tile and a global-memory E update per tile):
//   * packed FP32x2 arithmetic (FADD2 / FFMA2 / FMUL2, new on sm_100): one instruction works on TWO targets,
//     so the 11 FP32 ops cost 5.5 issue slots per interaction and the FMA pipe, not the scheduler, is the limit;
//   * register blocking: NPACK packs = 2*NPACK targets per thread share every source read;
//   * sources are staged in shared memory pre-duplicated as (x,x,y,y) / (z,z), so one LDS.128 + one LDS.64 with
//     all lanes on the same address (hardware broadcast, conflict free) deliver the packed operands directly;
//   * rsqrt.approx.ftz (MUFU.RSQ) — no denormal fix-up code in the inner loop;
//   * two-level accumulation: per-tile (<= 256 sources) FP32 partials are flushed into per-chunk totals, which
//     keeps the FP32 sum within ~5e-6 of FP64 on track-like geometry (a single running sum fails 1e-4);
//   * the N_a x N_a matrix is cut into (row block, column chunk) items scheduled round-robin over a persistent
//     grid sized to the SM count (gc_common.cuh: FieldPlan) — no wave-quantisation saw-tooth;
//     partial sums go to their own slot and are reduced in fixed order by the integrator.
#pragma once
#include "gc_common.cuh"

namespace gc {

__device__ __forceinline__ float rsqrt_ftz(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// One source against NP packs (2 NP targets): the 11 packed FP32 instructions + 2 MUFU.RSQ of eq. 6.
// sxy = (x,x,y,y), sz = (z,z) of the source; nt* = negated target coordinates; a* += (r_s - r_t) / (r^2+eps^2)^{3/2}.
template <int NP>
__device__ __forceinline__ void interact(const float4 sxy, const float2 sz, const float2 (&ntx)[NP], const float2 (&nty)[NP],
                                         const float2 (&ntz)[NP], const float2 eps2v, float2 (&ax)[NP], float2 (&ay)[NP],
                                         float2 (&az)[NP]) {
  const float2 sx2 = make_float2(sxy.x, sxy.y), sy2 = make_float2(sxy.z, sxy.w);
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    const float2 dx = __fadd2_rn(sx2, ntx[p]);
    const float2 dy = __fadd2_rn(sy2, nty[p]);
    const float2 dz = __fadd2_rn(sz, ntz[p]);
    float2 r2 = __ffma2_rn(dx, dx, eps2v);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    const float2 inv = make_float2(rsqrt_ftz(r2.x), rsqrt_ftz(r2.y));
    float2 w = __fmul2_rn(inv, inv);
    w = __fmul2_rn(w, inv);
    ax[p] = __ffma2_rn(dx, w, ax[p]);
    ay[p] = __ffma2_rn(dy, w, ay[p]);
    az[p] = __ffma2_rn(dz, w, az[p]);
  }
}

template <int NPACK, int TPB>
struct FieldCfg {
  static constexpr int kTargetsPerThread = 2 * NPACK;
  static constexpr int kIB = TPB * kTargetsPerThread;    // targets per row block
};

// Partial sums: Ep is three planes (x,y,z) of part_cap floats each; plane c, chunk s, target i at
// Ep[c*part_cap + s*stride + (i - t0)], [t0, t0+nt) being the targets this rank owns (all of them if unsharded).  The value stored is sum (r_s - r_t) w = -S_t (sign folded by the consumer).
//
// field_items: the work items of `plan` dealt round-robin to this CTA.  Called by k_field (one launch per evaluation)
// and by the persistent multi-step kernel (gc_persist.cuh), in which the state changes between two calls inside ONE
// launch: every load of the state goes to L2 (ld.global.cg), never through the non-coherent path.
template <int NPACK, int TPB, int UNROLL>
__device__ __forceinline__ void field_items(const float* px, const float* py, const float* pz, const FieldPlan& plan, float* Ep,
                                            uint32_t part_cap, float eps2, float4 (&s_xy)[2][TPB], float2 (&s_z)[2][TPB]) {
  constexpr int IB = FieldCfg<NPACK, TPB>::kIB;
  constexpr int kTile = TPB;                            // sources per shared-memory tile: one per thread
  const uint32_t n = plan.n;
  const uint32_t tid = threadIdx.x;
  const uint32_t items = plan.nIB * plan.S;
  const float2 eps2v = make_float2(eps2, eps2);

  for (uint32_t item = blockIdx.x; item < items; item += gridDim.x) {
    const uint32_t ib = item / plan.S, sc = item - ib * plan.S;
    const uint32_t i_base = plan.t0 + ib * IB;             // this rank's share of the targets (whole set if unsharded)
    const uint32_t i_end = plan.t0 + plan.nt;
    const uint32_t j0 = sc * plan.JC;
    const uint32_t j1 = min(j0 + plan.JC, n);

    // first source tile: issued before the target loads so that both L2 round trips overlap
    uint32_t jt = j0;
    float sx, sy, sz;
    {
      const uint32_t j = jt + tid;
      const bool ok = j < j1;
      sx = ok ? __ldcg(px + j) : kSentinel; sy = ok ? __ldcg(py + j) : kSentinel; sz = ok ? __ldcg(pz + j) : kSentinel;
    }

    // this thread's targets, negated: d = r_s + (-r_t)
    float2 ntx[NPACK], nty[NPACK], ntz[NPACK];
    float2 tx[NPACK], ty[NPACK], tz[NPACK];          // per-chunk totals
#pragma unroll
    for (int p = 0; p < NPACK; ++p) {
      const uint32_t i0 = i_base + (p * TPB + tid) * 2u;
      float2 vx = make_float2(0.f, 0.f), vy = vx, vz = vx;
      if (i0 + 1 < i_end) {                           // arrays are padded, but keep padding out of the math
        vx = __ldcg(reinterpret_cast<const float2*>(px + i0));
        vy = __ldcg(reinterpret_cast<const float2*>(py + i0));
        vz = __ldcg(reinterpret_cast<const float2*>(pz + i0));
      } else if (i0 < i_end) {
        vx.x = __ldcg(px + i0); vy.x = __ldcg(py + i0); vz.x = __ldcg(pz + i0);
      }
      ntx[p] = make_float2(-vx.x, -vx.y); nty[p] = make_float2(-vy.x, -vy.y); ntz[p] = make_float2(-vz.x, -vz.y);
      tx[p] = make_float2(0.f, 0.f); ty[p] = tx[p]; tz[p] = tx[p];
    }

    // software pipeline: registers hold tile k+1 while tile k is consumed from shared memory
    int buf = 0;
    __syncthreads();                                  // previous item's readers are done with both buffers
    s_xy[buf][tid] = make_float4(sx, sx, sy, sy);
    s_z[buf][tid] = make_float2(sz, sz);
    __syncthreads();

    for (; jt < j1; jt += kTile) {
      const uint32_t jn = jt + kTile;
      if (jn < j1) {                                  // prefetch the next tile into registers
        const uint32_t j = jn + tid;
        const bool ok = j < j1;
        sx = ok ? __ldcg(px + j) : kSentinel; sy = ok ? __ldcg(py + j) : kSentinel; sz = ok ? __ldcg(pz + j) : kSentinel;
      }
      const int len = (int)min((uint32_t)kTile, (j1 - jt + 3u) & ~3u);   // padded to the unroll factor with sentinels

      float2 ax[NPACK], ay[NPACK], az[NPACK];
#pragma unroll
      for (int p = 0; p < NPACK; ++p) { ax[p] = make_float2(0.f, 0.f); ay[p] = ax[p]; az[p] = ax[p]; }

#pragma unroll UNROLL
      for (int jj = 0; jj < len; ++jj) {
        interact<NPACK>(s_xy[buf][jj], s_z[buf][jj], ntx, nty, ntz, eps2v, ax, ay, az);
      }
      // flush the tile partial into the chunk total (two-level accumulation)
#pragma unroll
      for (int p = 0; p < NPACK; ++p) {
        tx[p] = __fadd2_rn(tx[p], ax[p]); ty[p] = __fadd2_rn(ty[p], ay[p]); tz[p] = __fadd2_rn(tz[p], az[p]);
      }
      if (jn < j1) {
        buf ^= 1;
        s_xy[buf][tid] = make_float4(sx, sx, sy, sy);   // the other buffer: its readers finished one barrier ago
        s_z[buf][tid] = make_float2(sz, sz);
        __syncthreads();
      }
    }

    // chunk result -> its own slot (fixed-order reduction happens in the integrator)
    float* ex = Ep + (size_t)sc * plan.stride;
    float* ey = ex + part_cap;
    float* ez = ey + part_cap;
#pragma unroll
    for (int p = 0; p < NPACK; ++p) {
      const uint32_t i0 = i_base - plan.t0 + (p * TPB + tid) * 2u;   // partial rows are indexed from the share's start
      if (i0 < plan.stride) {                          // stride >= nt, even: the float2 store stays inside the row
        *reinterpret_cast<float2*>(ex + i0) = tx[p];
        *reinterpret_cast<float2*>(ey + i0) = ty[p];
        *reinterpret_cast<float2*>(ez + i0) = tz[p];
      }
    }
  }
}

template <int NPACK, int TPB, int MINB, int UNROLL = 4>
__global__ void __launch_bounds__(TPB, MINB)
k_field(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
        const Ctrl* __restrict__ ctrl, float* __restrict__ Ep, uint32_t part_cap, float eps2) {
  __shared__ float4 s_xy[2][TPB];   // (x,x,y,y) per source
  __shared__ float2 s_z[2][TPB];    // (z,z)
  const FieldPlan plan = ctrl->plan;
  if (plan.n == 0) return;
  field_items<NPACK, TPB, UNROLL>(px, py, pz, plan, Ep, part_cap, eps2, s_xy, s_z);
}

}  // namespace gc
