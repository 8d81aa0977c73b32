// gc_persist.cuh — small populations (N_a up to a few 1e4): MANY TIME STEPS IN ONE LAUNCH.
//
// below ~1e3 charges "the GPU is subutilised" and its run time is flat — every step is a train of
// launches whose latency, not eq. 6, is the cost.  Config 0, config 1 and the tail of every event live there.  Here a
// persistent cooperative grid (every CTA resident, one launch for up to 2^20 steps) loops over
//     field items (eq. 6, the same field_items as k_field)  -> grid barrier ->
//     a2..a8 on tiles of 32..256 carriers, 8..1 threads per carrier (update, collection, in-place look-back compaction)
//     -> grid barrier
// with n_active, the step index and the FieldPlan passed from step to step through the device-resident Ctrl block.
// A step costs two grid barriers (one atomic + one polled L2 line each) instead of three dependent kernel launches.
// The arithmetic per carrier is the code of the one-step kernels (interact<>, advance_carrier, collect), the
// Philox counter is (id, step): a run through this kernel equals a run of single steps up to the FP32 summation order
// of eq. 6 (the chunk partials are summed by several threads per carrier here, in a fixed order).
#pragma once
#include "gc_advance.cuh"
#include "gc_field.cuh"

namespace gc {

// Grid barrier of a cooperative grid, split into ARRIVE and WAIT so that work which does not depend on the other CTAs
// fills the gap.  Arrivals are counted in ONE word (atom.acq_rel: releases this CTA's writes — they precede the
// __syncthreads — and lets the last arriver acquire everybody's); the last arriver then raises one flag PER CTA, 128
// bytes apart, and each CTA polls only its own flag.  With everybody polling the arrival word itself, the polls of
// the early CTAs queue in front of the late arrivals at one L2 slice: measured 19 cycles per CTA per barrier (296 CTAs:
// 5,600 cycles).  `gen` = value the flags take at this barrier (increases by one per barrier, never reused between
// resets); `target` = arrivals expected since the launch began.  Data that crosses the barrier is read with L2-coherent
// loads (ld.global.cg) only.
constexpr uint32_t kFlagStride = 32;                        // uint32 per flag: one 128-byte line each
__device__ __forceinline__ void grid_arrive(uint32_t* bar, uint32_t* flags, uint32_t target, uint32_t gen) {
  __syncthreads();
  if (threadIdx.x < 32) {
    uint32_t last = 0;
    if (threadIdx.x == 0) {
      uint32_t old;
      asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(bar) : "memory");
      last = (old + 1u == target) ? 1u : 0u;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (last) {
      asm volatile("fence.acq_rel.gpu;" ::: "memory");
      for (uint32_t c = threadIdx.x; c < gridDim.x; c += 32)
        asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(flags + (size_t)c * kFlagStride), "r"(gen) : "memory");
    }
  }
}
__device__ __forceinline__ void grid_wait(const uint32_t* flags, uint32_t gen) {
  if (threadIdx.x == 0) {
    const uint32_t* f = flags + (size_t)blockIdx.x * kFlagStride;
    while ((int32_t)(ld_relaxed_u32(f) - gen) < 0) { }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
  }
  __syncthreads();
}

struct PersistShared {
  double e[3][kTPB];          // [component][range q of the chunk partials][carrier c], flattened: index q * TQ + c
  double bm[5][kTPB];         // Box-Muller chains of the tile's carriers: Ra, sa, ca, Rb, cb (index c < TQ)
  uint32_t w[16];
};

// a2..a8 of ONE tile of TQ carriers by the 256 threads of a CTA, R = 256 / TQ threads per carrier, in two halves:
//   pre  (between the arrive and the wait of the field barrier: needs only the carrier itself): load the carrier, run the
//        four Box-Muller chains of its normal triple on up to four threads;
//   post (after the barrier): R threads sum a range of the S chunk partials each, then one thread per carrier runs the
//        field-dependent chain (eq. 1, |E|, eq. 2, update) and the tile is committed.
// A lone warp needs ~2,000 dependent FP64 instructions per carrier for a2..a6 (6-9 us); spread like this the part that
// must wait for the field is the eq. 2 chain alone.
struct Tile {
  uint32_t TQ, R;             // carriers per tile (32, 64, 128 or 256), threads per carrier (256 / TQ)
  float x, y, z; uint32_t id; uint32_t c, q, i; bool have;

  __device__ __forceinline__ void pre(uint32_t tq, const SoA& A, uint32_t t, uint32_t n, uint64_t step, const DevParams& P,
                                      PersistShared& sh) {
    const uint32_t tid = threadIdx.x;
    TQ = tq; R = kTPB / tq;
    c = tid % TQ; q = tid / TQ; i = t * TQ + c;
    have = i < n;
    x = y = z = 0.f; id = 0;
    if (have) { x = __ldcg(A.x + i); y = __ldcg(A.y + i); z = __ldcg(A.z + i); id = __ldcg(A.id + i); }
    if (have && !(P.flags & 2u)) {
      const uint4 w = philox_words(P.seed_lo, P.seed_hi, id, step);
      // chains 0..3 = Ra | (sa, ca) | Rb | cb: one each on threads q = 0..3 (R >= 4), two each (R = 2), all four (R = 1)
      const uint32_t per = R >= 4 ? 1u : 4u / R;
      if (q * per < 4u) {
        BoxMuller b;
        for (uint32_t ch = q * per; ch < q * per + per; ++ch) {
          if (ch == 0) { b.Ra = bm_radius(w.x); sh.bm[0][c] = b.Ra; }
          else if (ch == 1) { sincospi(2.0 * bm_fraction(w.y), &b.sa, &b.ca); sh.bm[1][c] = b.sa; sh.bm[2][c] = b.ca; }
          else if (ch == 2) { b.Rb = bm_radius(w.z); sh.bm[3][c] = b.Rb; }
          else { b.cb = cospi(2.0 * bm_fraction(w.w)); sh.bm[4][c] = b.cb; }
        }
      }
    }
  }

  __device__ __forceinline__ bool post(SoA dst, uint32_t t, uint32_t n, uint64_t step, uint32_t stamp, const FieldPlan& plan,
                                       const float* Ep, uint32_t part_cap, Ctrl* ctrl, Sink sink, unsigned long long* status,
                                       const DevParams& P, PersistShared& sh, uint32_t& n_new) {
    {
      double ex = 0.0, ey = 0.0, ez = 0.0;
      if (have && !(P.flags & 1u)) {
        const uint32_t per = (plan.S + R - 1) / R;
        const uint32_t s0 = min(q * per, plan.S), s1 = min(s0 + per, plan.S);
        const float* e = Ep + i;
        for (uint32_t s = s0; s < s1; s += 4) {
          float vx[4], vy[4], vz[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const bool ok = s + u < s1;
            const size_t o = (size_t)(s + u) * plan.stride;
            vx[u] = ok ? __ldcg(e + o) : 0.f; vy[u] = ok ? __ldcg(e + part_cap + o) : 0.f;
            vz[u] = ok ? __ldcg(e + 2 * (size_t)part_cap + o) : 0.f;
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) { ex += (double)vx[u]; ey += (double)vy[u]; ez += (double)vz[u]; }
        }
      }
      sh.e[0][q * TQ + c] = ex; sh.e[1][q * TQ + c] = ey; sh.e[2][q * TQ + c] = ez;
    }
    __syncthreads();                                         // partial ranges and Box-Muller chains are in shared memory
    float xf = 0.f, yf = 0.f, zf = 0.f;
    bool finite = true;
    const bool mine = have && q == 0;
    if (mine) {
      double E[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        double a = sh.e[k][c];
        for (uint32_t r = 1; r < R; ++r) a += sh.e[k][r * TQ + c];   // ranges in ascending order: fixed summation order
        E[k] = -P.Kp * a;                                           // partials hold sum (r_s - r_t) w
      }
      double nrm[3] = {0.0, 0.0, 0.0};
      if (!(P.flags & 2u)) { nrm[0] = sh.bm[0][c] * sh.bm[2][c]; nrm[1] = sh.bm[0][c] * sh.bm[1][c]; nrm[2] = sh.bm[3][c] * sh.bm[4][c]; }
      finite = advance_with_normals(x, y, z, E[0], E[1], E[2], nrm, P, xf, yf, zf);
    }
    return commit_tile<false>(TQ, dst, t, n, step, stamp, mine, finite, xf, yf, zf, id, ctrl, sink, status, P, sh.w, n_new);
  }
};

#ifdef GC_TIMING
__device__ long long g_dbg[2][64][16];
#define GC_T(slot) do { if (tid == 0 && k < 64 && (blockIdx.x == 0 || blockIdx.x == gridDim.x - 1)) g_dbg[blockIdx.x ? 1 : 0][k][slot] = clock64(); } while (0)
#else
#define GC_T(slot) do { } while (0)
#endif

template <int NPACK, int MINB>
__global__ void __launch_bounds__(kTPB, MINB)
k_steps(SoA A, SoA B, Ctrl* ctrl, float* Ep, uint32_t part_cap, Sink sink, unsigned long long* status, uint32_t* flags,
        DevParams P, PlanArgs pa, uint32_t n_steps) {
  __shared__ float4 s_xy[2][kTPB];
  __shared__ float2 s_z[2][kTPB];
  __shared__ PersistShared sh;
  __shared__ FieldPlan s_plan;
  __shared__ unsigned long long s_step;
  const uint32_t tid = threadIdx.x;
  const uint32_t seq0 = ld_acquire_u32(&ctrl->scan_seq);
  const uint32_t gen0 = ld_acquire_u32(&ctrl->bar_gen);      // written by the previous launch's last CTA
  uint32_t arrivals = 0, gen = gen0;
  uint32_t k = 0;
  // the state ping-pongs between A and B (step k reads one, writes the compacted survivors to the other): no slot is
  // ever overwritten while another CTA may still read it, so the look-back needs no release/acquire ordering
  for (; k < n_steps; ++k) {
    const SoA cur = (k & 1u) ? B : A, nxt = (k & 1u) ? A : B;
    // Ctrl was written by another CTA before the last barrier: ONE thread reads it from L2 and shares it (2,368 warps
    // asking one L2 slice for the same line cost ~1,000 cycles per step)
    if (tid == 0) {
      const uint4* pp = reinterpret_cast<const uint4*>(&ctrl->plan);
      const uint4 a = __ldcg(pp), b = __ldcg(pp + 1);
      const unsigned long long st = __ldcg(reinterpret_cast<const unsigned long long*>(&ctrl->step));
      s_plan.n = a.x; s_plan.nIB = a.y; s_plan.S = a.z; s_plan.JC = a.w;
      s_plan.stride = b.x; s_plan.IB = b.y; s_plan.t0 = b.z; s_plan.nt = b.w;
      s_step = st;
    }
    __syncthreads();
    const FieldPlan plan = s_plan;
    const uint32_t n = plan.n;
    if (n == 0) break;                                       // uniform over the grid
    const uint64_t step = s_step;
    const uint32_t stamp = scan_stamp(seq0 + k);
    // a2..a8 tile size: the smallest that gives every tile a CTA of its own (more threads per carrier = shorter chains)
    const uint32_t G = gridDim.x;
    const int tq = (n + 31u) / 32u <= G ? 32 : (n + 63u) / 64u <= G ? 64 : (n + 127u) / 128u <= G ? 128 : 256;
    const uint32_t t = blockIdx.x;
    const bool owner = t < (n + (uint32_t)tq - 1u) / (uint32_t)tq;     // the host keeps n <= 256 G (persist_max)

    GC_T(0);
    field_items<NPACK, kTPB, 4>(cur.x, cur.y, cur.z, plan, Ep, part_cap, P.eps2, s_xy, s_z);
    GC_T(1);
    arrivals += G; gen += 1;
    grid_arrive(&ctrl->bar, flags, arrivals, gen);
    GC_T(2);

    Tile tile;
    if (owner) tile.pre((uint32_t)tq, cur, t, n, step, P, sh);
    GC_T(3);
    grid_wait(flags, gen);
    GC_T(4);
    if (owner) {
      uint32_t n_new = 0;
      const bool last = tile.post(nxt, t, n, step, stamp, plan, Ep, part_cap, ctrl, sink, status, P, sh, n_new);
      if (last && tid < 32) {                                // the owner of the last tile publishes the next step's control
        n_new = __shfl_sync(0xffffffffu, n_new, 0);
        FieldPlan np = plan;
        if (n_new != n) np = plan_search(n_new, pa);
        if (tid == 0) {
          ctrl->plan = np;
          ctrl->n_active = n_new;
          ctrl->step = step + 1;
          ctrl->pairs += (uint64_t)n * (uint64_t)n;
        }
      }
    }
    GC_T(5);
    arrivals += G; gen += 1;
    grid_arrive(&ctrl->bar, flags, arrivals, gen);
    GC_T(6);
    grid_wait(flags, gen);
    GC_T(7);
  }
  // an odd number of steps leaves the state in B: bring it home (every CTA is past the last barrier; B is complete)
  if (k & 1u) {
    if (tid == 0) s_plan.n = __ldcg(&ctrl->n_active);
    __syncthreads();
    const uint32_t n = s_plan.n;
    for (uint32_t i = blockIdx.x * kTPB + tid; i < n; i += gridDim.x * kTPB) {
      A.x[i] = __ldcg(B.x + i); A.y[i] = __ldcg(B.y + i); A.z[i] = __ldcg(B.z + i); A.id[i] = __ldcg(B.id + i);
    }
  }
  // exit: the last CTA out re-arms the barrier for the next launch and accounts for the steps taken
  if (tid == 0) {
    __threadfence();
    const uint32_t out = atomicAdd(&ctrl->bar_exit, 1u);
    if (out == gridDim.x - 1) {
      ctrl->bar = 0;
      ctrl->bar_exit = 0;
      ctrl->bar_gen = gen;
      ctrl->scan_seq = seq0 + k;
    }
  }
}

}  // namespace gc
