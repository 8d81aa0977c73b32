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
// fills the gap.  `target` = arrivals expected since the launch began (barriers so far x gridDim.x).  One release
// reduction per CTA to arrive (it orders the whole CTA's writes: they precede the __syncthreads), relaxed polling of the
// same word, one fence after the wait; data that crosses the barrier is read with L2-coherent loads (ld.global.cg) only.
// (Tried: one flag line per CTA raised by the last arriver, so that nobody polls the arrival word — slower at every
// size: 10.1 -> 10.6 us per step at 1,024 holes, 18.6 -> 20.2 at 4,096; the second hop costs more than the polls.)
__device__ __forceinline__ void grid_arrive(uint32_t* bar) {
  __syncthreads();
  if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
}
__device__ __forceinline__ void grid_wait(const uint32_t* bar, uint32_t target) {
  if (threadIdx.x == 0) {
    while (ld_relaxed_u32(bar) < target) { }
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
    GC_P(0);
    {
      double ex = 0.0, ey = 0.0, ez = 0.0;
      if (have && !(P.flags & 1u)) {
        const uint32_t per = (plan.S + R - 1) / R;
        const uint32_t s0 = min(q * per, plan.S), s1 = min(s0 + per, plan.S);
        const float* e = Ep + i;
        for (uint32_t s = s0; s < s1; s += 4) {              // 12 loads in flight per round trip; 24 measured slower (3,100 -> 5,900 cycles)
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
    GC_P(1);
    __syncthreads();                                         // partial ranges and Box-Muller chains are in shared memory
    GC_P(2);
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
    GC_P(3);
    return commit_tile<false>(TQ, dst, t, n, step, stamp, mine, finite, xf, yf, zf, id, ctrl, sink, status, P, sh.w, n_new);
  }
};

#ifdef GC_TIMING
__device__ long long g_dbg[2][64][16];
__device__ unsigned long long g_gt[1024][8];      // per CTA: globaltimer (ns) at the phase boundaries of step 8
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define GC_G(slot) do { if (tid == 0 && k == 8) g_gt[blockIdx.x][slot] = gtime(); } while (0)
#else
#define GC_G(slot) do { } while (0)
#endif
#ifdef GC_TIMING
#define GC_T(slot) do { if (tid == 0 && k < 64 && (blockIdx.x == 0 || blockIdx.x == gridDim.x - 1)) g_dbg[blockIdx.x ? 1 : 0][k][slot] = clock64(); } while (0)
#else
#define GC_T(slot) do { } while (0)
#endif

template <int NPACK, int MINB>
__global__ void __launch_bounds__(kTPB, MINB)
k_steps(SoA A, SoA B, Ctrl* ctrl, float* Ep, uint32_t part_cap, Sink sink, unsigned long long* status, DevParams P, PlanArgs pa,
        uint32_t n_steps, uint32_t n_exit) {
  __shared__ float4 s_xy[2][kTPB];
  __shared__ float2 s_z[2][kTPB];
  __shared__ PersistShared sh;
  __shared__ FieldPlan s_plan;
  __shared__ unsigned long long s_step;
  const uint32_t tid = threadIdx.x;
  const uint32_t seq0 = ld_acquire_u32(&ctrl->scan_seq);
  uint32_t arrivals = 0;
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
    if (n == 0 || n < n_exit) break;                         // uniform over the grid; n_exit: a smaller variant takes over
    const uint64_t step = s_step;
    const uint32_t stamp = scan_stamp(seq0 + k);
    // a2..a8 tile size: the smallest that gives every tile a CTA of its own (more threads per carrier = shorter chains)
    const uint32_t G = gridDim.x;
    const int tq = (n + 31u) / 32u <= G ? 32 : (n + 63u) / 64u <= G ? 64 : (n + 127u) / 128u <= G ? 128 : 256;
    const uint32_t t = blockIdx.x;
    const bool owner = t < (n + (uint32_t)tq - 1u) / (uint32_t)tq;     // the host keeps n <= 256 G (persist_max)

    GC_T(0); GC_G(0);
    field_items<NPACK, kTPB, 4>(cur.x, cur.y, cur.z, plan, Ep, part_cap, P.eps2, s_xy, s_z);
    GC_T(1); GC_G(1);
    arrivals += G;
    grid_arrive(&ctrl->bar);
    GC_T(2);

    Tile tile;
    if (owner) tile.pre((uint32_t)tq, cur, t, n, step, P, sh);
    GC_T(3); GC_G(2);
    grid_wait(&ctrl->bar, arrivals);
    GC_T(4); GC_G(3);
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
    GC_T(5); GC_G(4);
    arrivals += G;
    grid_arrive(&ctrl->bar);
    GC_T(6);
    grid_wait(&ctrl->bar, arrivals);
    GC_T(7); GC_G(5);
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
      ctrl->scan_seq = seq0 + k;
    }
  }
}

}  // namespace gc
