// gc_shard.cuh — target sharding over several GPUs.
//
// The muon workload (2e5 .. 1e6 holes) is where the paper's hours went, and eq. 6 shards naturally:
// the fields of different targets are independent given all source positions.  Scheme = replicated state, sharded
// rows: every rank holds the whole active state A (16 B/carrier, <= 16 MB at 1M holes), rank g of G runs a1..a7 for
// the targets of its share [t0, t0+nt) (gc_common.cuh: shard_range) against ALL sources, compacts its survivors
// (a8) into a message, and the messages of all ranks, concatenated in rank order, ARE the next step's state in the
// same stable order a single GPU would produce.  The only exchange per step is that all-gather of 16 B per
// surviving carrier; images and counters stay rank-local and are summed once at the end (integers).
//
// Message layout (bs = entries per coordinate array, a multiple of 256, same on every rank for a given step):
//   [ 256-byte header | x[bs] | y[bs] | z[bs] | id[bs] ]        header = ShardHeader
// k_shard_compact fills it; k_shard_commit reads G of them through a table of G device pointers.  Those pointers
// may be slices of a local all-gather receive buffer (NCCL plumbing) or peer-mapped buffers of the other ranks
// (symmetric memory over NVLink: the gather is then fused into the commit's loads) — the kernel is the same.
// By default no kernel waits on another rank: ordering between ranks is the collective's / the host barrier's job.
// With gcoreccd_set_shard_wait (peer-mapped messages) the commit kernel spins on the headers' `ready` words instead.
#pragma once
#include "gc_common.cuh"

namespace gc {

constexpr uint32_t kShardMaxWorld = 64;
constexpr uint32_t kShardHeaderBytes = 256;

struct ShardHeader {
  uint32_t count;        // survivors in this message
  uint32_t nt;           // targets the rank advanced this step
  uint32_t n_before;     // n_active the step started from (must agree on all ranks)
  uint32_t rank;
  uint64_t step;         // index of the step that produced the message
  unsigned long long ready;   // written LAST, release at system scope: (epoch << 32) | (uint32)(step + 1); see header_ready
};

// Flag synchronisation for peer-mapped messages (symmetric memory over NVLink): with `wait` set, k_shard_commit spins
// on each header's `ready` word until it carries THIS step's value instead of relying on a host-enqueued barrier
// between shard_local and shard_commit.  `epoch` changes at every reset / set_shard (all ranks call them in lockstep),
// so a stale header of an earlier event in the same buffer can never match.  Two message buffers, alternated, are
// enough: a rank overwrites buffer b at step s+2 only after committing step s+1, which needed every peer's message
// of step s+1, which each peer wrote after ITS commit of step s, i.e. after reading buffer b.
__device__ __forceinline__ unsigned long long header_ready(uint32_t epoch, uint64_t step) {
  return ((unsigned long long)epoch << 32) | (unsigned long long)(uint32_t)(step + 1u);
}
__device__ __forceinline__ void header_wait(const char* msg, unsigned long long want) {
  const unsigned long long* p = &reinterpret_cast<const ShardHeader*>(msg)->ready;
  unsigned long long v;
  do { asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); } while (v != want);
}

struct ShardPtrs { const char* p[kShardMaxWorld]; };

__device__ __forceinline__ float* msg_x(char* m) { return reinterpret_cast<float*>(m + kShardHeaderBytes); }
__device__ __forceinline__ const float* msg_x(const char* m) { return reinterpret_cast<const float*>(m + kShardHeaderBytes); }

// a8 for one share: stable compaction of the share's survivors (tiles of state B starting at t0) into the message.
// Same ballot + scan as k_compact; the CTA that finishes last writes the header.  Grid = bs / 256 CTAs.
__global__ void __launch_bounds__(kTPB)
k_shard_compact(SoA B, Ctrl* __restrict__ ctrl, const uint32_t* __restrict__ tile_count, char* __restrict__ msg,
                uint32_t bs, double z_well, uint32_t rank, uint32_t epoch) {
  __shared__ uint32_t s_red[kTPB / 32];
  __shared__ uint32_t s_base, s_last;
  const uint32_t t0 = ctrl->plan.t0, nt = ctrl->plan.nt;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t t = blockIdx.x;
  const uint32_t n_tiles = (nt + kTPB - 1) / kTPB;
  float* mx = msg_x(msg);
  float* my = mx + bs;
  float* mz = my + bs;
  uint32_t* mid = reinterpret_cast<uint32_t*>(mz + bs);

  if (t < n_tiles) {
    const uint32_t k = t * kTPB + tid;
    float x = 0.f, y = 0.f, z = 0.f; uint32_t id = 0;
    if (k < nt) { x = B.x[t0 + k]; y = B.y[t0 + k]; z = B.z[t0 + k]; id = B.id[t0 + k]; }
    const bool keep = k < nt && (double)z > z_well;
    uint32_t part = 0;
    for (uint32_t u = tid; u < t; u += kTPB) part += tile_count[u];
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) s_red[warp] = part;
    __syncthreads();
    if (tid == 0) {
      uint32_t b = 0;
      for (int w = 0; w < kTPB / 32; ++w) b += s_red[w];
      s_base = b;
    }
    __syncthreads();
    const uint32_t base = s_base;
    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    const uint32_t rank_in_warp = __popc(bal & ((1u << lane) - 1u));
    __syncthreads();
    if (lane == 0) s_red[warp] = __popc(bal);
    __syncthreads();
    uint32_t warp_off = 0;
    for (uint32_t w = 0; w < warp; ++w) warp_off += s_red[w];
    if (keep) {
      const uint32_t d = base + warp_off + rank_in_warp;   // < nt <= bs
      mx[d] = x; my[d] = y; mz[d] = z; mid[d] = id;
    }
    if (t == n_tiles - 1 && tid == 0) {
      uint32_t tot = 0;
      for (int w = 0; w < kTPB / 32; ++w) tot += s_red[w];
      ctrl->n_next = base + tot;
    }
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t ticket = atomicAdd(&ctrl->blocks_done, 1u);
    s_last = (ticket == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (s_last && tid == 0) {
    __threadfence();
    ShardHeader* hd = reinterpret_cast<ShardHeader*>(msg);
    hd->count = n_tiles ? *((volatile uint32_t*)&ctrl->n_next) : 0u;
    hd->nt = nt;
    hd->n_before = ctrl->n_active;
    hd->rank = rank;
    hd->step = ctrl->step;
    ctrl->blocks_done = 0;
    ctrl->n_next = 0;
    __threadfence_system();                                  // payload (all CTAs', observed through the ticket) and header
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(&hd->ready), "l"(header_ready(epoch, ctrl->step)) : "memory");
  }
}

// The other half of a8 + the gather: the survivors of all G shares, in rank order, become state A.
// Grid = G x (bs / 256) CTAs; CTA (g, t) copies entries [256 t, 256 t + 256) of message g to A at
// sum_{k<g} count_k.  The last CTA to finish publishes n_active, advances the step index, adds this rank's
// nt x n ordered pairs to the pair counter and plans the next step's share.  A header that disagrees on
// (n_before, step) with this rank's own state means the ranks have diverged: sticky flag, reported as BAD_STATE.
__global__ void __launch_bounds__(kTPB)
k_shard_commit(ShardPtrs bufs, uint32_t world, uint32_t bs, SoA A, Ctrl* __restrict__ ctrl, PlanArgs pa, uint32_t wait,
               uint32_t epoch) {
  __shared__ uint32_t s_base, s_count, s_last;
  const uint32_t tid = threadIdx.x;
  const uint32_t tiles_per = bs / kTPB;
  const uint32_t g = blockIdx.x / tiles_per, t = blockIdx.x - g * tiles_per;
  if (tid == 0) {
    if (wait) {                                              // every message this CTA reads a count or carriers from
      const unsigned long long want = header_ready(epoch, ctrl->step);
      for (uint32_t k = 0; k <= g; ++k) header_wait(bufs.p[k], want);
    }
    uint32_t base = 0;
    for (uint32_t k = 0; k < g; ++k) base += reinterpret_cast<const ShardHeader*>(bufs.p[k])->count;
    const ShardHeader* hd = reinterpret_cast<const ShardHeader*>(bufs.p[g]);
    s_base = base; s_count = hd->count;
    if (t == 0 && (hd->n_before != ctrl->n_active || hd->step != ctrl->step || hd->rank != g)) atomicOr(&ctrl->diverged, 1u);
  }
  __syncthreads();
  const uint32_t k = t * kTPB + tid;
  if (k < s_count) {
    const float* mx = msg_x(bufs.p[g]);
    const float* my = mx + bs;
    const float* mz = my + bs;
    const uint32_t* mid = reinterpret_cast<const uint32_t*>(mz + bs);
    const uint32_t d = s_base + k;
    A.x[d] = mx[k]; A.y[d] = my[k]; A.z[d] = mz[k]; A.id[d] = mid[k];
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t ticket = atomicAdd(&ctrl->blocks_done, 1u);
    s_last = (ticket == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (s_last && tid < 32) {
    __threadfence();
    if (wait) {
      const unsigned long long want = header_ready(epoch, ctrl->step);
      for (uint32_t r = g + 1; r < world; ++r) header_wait(bufs.p[r], want);   // (already seen up to g)
    }
    uint32_t n_new = 0;
    for (uint32_t r = 0; r < world; ++r) n_new += reinterpret_cast<const ShardHeader*>(bufs.p[r])->count;
    const FieldPlan old = ctrl->plan;
    const FieldPlan plan = plan_search(n_new, pa);
    if (tid == 0) {
      ctrl->pairs += (uint64_t)old.nt * (uint64_t)ctrl->n_active;
      ctrl->plan = plan;
      if (ctrl->n_active != 0) ctrl->step += 1;            // a step with nobody drifting is a no-op
      ctrl->n_active = n_new;
      ctrl->blocks_done = 0;
    }
  }
}

}  // namespace gc
