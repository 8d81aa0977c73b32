// gc_common.cuh — device-resident control block, state layout and the field-kernel work plan.
//
// State layout in HBM: structure of arrays, one FP32 array per coordinate plus the carrier
// id, each padded to a multiple of 1024 entries and 256-byte aligned so that vector (64/128-bit) loads and
// bulk copies never straddle an allocation.  Two such sets (A = state at step boundaries, B = scratch the
// integrator writes and the compactor reads).  PAPER.md:84 stores "3N floats"; ids are ours (Philox key).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gc {

constexpr int kTPB        = 256;          // threads per CTA of every kernel
constexpr int kTile       = 256;          // sources per shared-memory tile == carriers per compaction tile
constexpr uint32_t kPartFactor = 16;      // partial-sum chunks a handle can hold at full capacity (gcoreccd.cu make_layout)
constexpr float kSentinel = 1.0e18f;      // padding source: (1e18)^-3 underflows to 0, contribution exactly 0

// Work plan of the field kernel: the N_a x N_a interaction matrix is cut into nIB row blocks
// (IB targets each) times S column chunks (JC sources each); item k = (row block k / S, chunk k % S) goes to
// CTA k % grid.  The plan is a pure function of (n_active, IB, grid, partial capacity); it is computed once per
// step by one warp (plan_search) and stored in Ctrl, so the partial sums are written and reduced in a fixed
// order: runs are bit-reproducible and no float atomics are needed.
struct FieldPlan {
  uint32_t n;        // active carriers the plan was made for
  uint32_t nIB;      // row blocks
  uint32_t S;        // column chunks
  uint32_t JC;       // sources per chunk (multiple of 8)
  uint32_t stride;   // row stride of the partial buffers (n rounded up to 256)
  uint32_t IB;       // targets per row block the plan was made for
  uint32_t t0;       // first target of this rank's share (multiple of 256; 0 when not sharded)
  uint32_t nt;       // targets in the share (= n when not sharded); row blocks and partial rows cover [t0, t0+nt)
};

struct Ctrl {                 // lives in device memory; only kernels write it (plus reset/load on the stream)
  uint32_t n_active;          // carriers still drifting (valid entries of state A)
  uint32_t n_next;            // scratch: survivors counted by the compactor
  uint64_t step;              // index of the NEXT step (Philox counter)
  uint64_t pairs;             // sum over executed steps of n_active^2
  uint64_t n_collected;
  uint64_t n_overflow;        // collected outside the image window
  uint64_t n_loaded;
  uint32_t nonfinite;         // sticky flag
  uint32_t invalid;           // load validation flag
  uint32_t blocks_done;       // "last block finishes" counter of the compactor
  uint32_t multi_steps;       // scratch of the Coulomb-off multi-step kernel: steps the longest-lived carrier took
  FieldPlan plan;             // valid for (n_active, current field variant, shard)
  uint32_t diverged;          // sticky: a shard message disagreed with this rank's (n_active, step) (gc_shard.cuh)
  uint32_t ticket;            // tile tickets of k_advance (look-back needs tiles in start order); 0 between launches
  uint32_t scan_seq;          // executed look-back scans: the stamp that tells this step's status words from stale ones
  uint32_t pad2_[5];
  // second 128-byte line: polled by the persistent kernel's grid barrier, kept away from the line everybody reads
  uint32_t bar;               // arrivals since the launch began; 0 between launches
  uint32_t bar_exit;          // CTAs that left the persistent kernel; 0 between launches
  uint32_t pad3_[30];
};
static_assert(sizeof(Ctrl) == 256, "Ctrl is two 128-byte lines");

struct SoA {                  // one state set
  float* x; float* y; float* z; uint32_t* id;
};

struct DevParams {            // constants uploaded by value with every launch
  double a1_um;               // a1 * 1e-4  (V/cm per um)
  double a2;
  double mu0, inv_Ec, beta, inv_beta;   // eq. 2 with the T terms folded on the host
  const double* mu_tab;       // eq. 2 as piecewise degree-8 interpolants of (1 + r^beta)^(-1/beta), r = E/Ec (gc_integrate.cuh)
  double drift_k;             // 1e-5 * dt
  double sigma_k;             // 2 * 0.1 * (k_B T / q) * dt
  double thickness, z_well;
  double x0, y0, pitch;
  double Kp;                  // K' (V/cm) um^2
  float  eps2;                // softening^2 (clamped to >= 1e-24, R5)
  uint32_t flags;
  uint32_t seed_lo, seed_hi;
  int32_t nx, ny;
};

// eq. 2 table (gc_integrate.cuh mobility): binades 2^kMuEmin <= r < 2^kMuEmax of r = E/Ec, 16 sub-intervals each,
// 9 monomial coefficients per sub-interval
constexpr int kMuEmin = -16, kMuEmax = 16, kMuSub = 16, kMuDeg = 8;
constexpr int kMuTabEntries = (kMuEmax - kMuEmin) * kMuSub * (kMuDeg + 1);

struct Sink {                 // where a collected hole goes (a7)
  uint32_t* image;            // [ny][nx] integer pixel histogram
  float4* fin;                // per-id record (x, y, z at collection, bits(step index)); all-ones = still drifting
  uint32_t fin_cap;           // ids >= fin_cap are binned but not recorded
};

struct PlanArgs { uint32_t IB; uint32_t grid; uint32_t part_cap_entries; uint32_t rank; uint32_t world;
                  uint32_t force_S; };   // force_S > 0: no search, S chunks (the treecode's parts per group, gc_tree.cuh)

// Target sharding: the state is replicated on every rank, the rows of the
// interaction matrix are not.  The n active carriers form ceil(n/256) tiles; rank g of G owns the contiguous tiles
// [floor(g T / G), floor((g+1) T / G)), i.e. targets [t0, t0 + nt).  A pure function of (n, g, G): every rank
// derives every share without communication, and the shares re-balance by themselves as carriers retire.
__host__ __device__ inline void shard_range(uint32_t n, uint32_t rank, uint32_t world, uint32_t& t0, uint32_t& nt) {
  const uint64_t T = ((uint64_t)n + 255u) >> 8;
  const uint64_t a = (T * rank / world) << 8, b = (T * (rank + 1u) / world) << 8;
  const uint64_t lo = a < n ? a : n, hi = b < n ? b : n;
  t0 = (uint32_t)lo; nt = (uint32_t)(hi - lo);
}

#ifdef __CUDACC__
// Executed by ONE full warp.  Static round-robin makespan model: a CTA runs ceil(items/grid) items, each costing
// JC source iterations plus a fixed overhead (target load, first tile, barrier, store ~ kItemOverhead source
// iterations).  Picks the S minimising rounds * (JC + overhead); ties go to the smaller S (fewer partials to
// reduce).  Constraints: >= kMinChunk sources per chunk, S * stride <= partial capacity.
constexpr uint32_t kItemOverhead = 24;
constexpr uint32_t kMinChunk = 32;
__device__ inline FieldPlan plan_search(uint32_t n, PlanArgs a) {
  const uint32_t lane = threadIdx.x & 31u;
  FieldPlan p;
  p.n = n; p.IB = a.IB;
  shard_range(n, a.rank, a.world, p.t0, p.nt);
  p.nIB = (p.nt + a.IB - 1) / a.IB;
  p.stride = (p.nt + 255u) & ~255u;
  p.S = 0; p.JC = 0;
  if (n == 0 || p.nt == 0) return p;
  if (a.force_S) { p.S = a.force_S; p.JC = (((n + p.S - 1) / p.S) + 7u) & ~7u; return p; }
  uint32_t s_max = (n + kMinChunk - 1) / kMinChunk;
  const uint32_t s_cap = a.part_cap_entries / p.stride;
  const uint32_t s_bal = max(64u, (4u * a.grid + p.nIB - 1) / p.nIB);      // beyond ~4 rounds nothing improves
  if (s_max > s_cap) s_max = s_cap;
  if (s_max > s_bal) s_max = s_bal;
  if (s_max < 1u) s_max = 1u;
  uint32_t best_c = 0xffffffffu, best_S = 1;
  for (uint32_t base = 1; base <= s_max; base += 32) {
    const uint32_t S = base + lane;
    if (S <= s_max) {
      const uint32_t JC = (((n + S - 1) / S) + 7u) & ~7u;
      const uint32_t Se = (n + JC - 1) / JC;                                 // chunks actually used
      const uint32_t rounds = (p.nIB * Se + a.grid - 1) / a.grid;
      const uint32_t c = rounds * (JC + kItemOverhead);
      if (c < best_c) { best_c = c; best_S = S; }
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const uint32_t oc = __shfl_xor_sync(0xffffffffu, best_c, o);
    const uint32_t oS = __shfl_xor_sync(0xffffffffu, best_S, o);
    if (oc < best_c || (oc == best_c && oS < best_S)) { best_c = oc; best_S = oS; }
  }
  const uint32_t JC = (((n + best_S - 1) / best_S) + 7u) & ~7u;
  p.JC = JC;
  p.S = (n + JC - 1) / JC;
  return p;
}
#endif

}  // namespace gc
