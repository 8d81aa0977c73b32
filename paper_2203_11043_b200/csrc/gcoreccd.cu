// gcoreccd.cu — host side of the C ABI declared in include/gcoreccd.h: workspace carving, launches, CUDA
// graphs, readback.  Every step of the hot path runs in the kernels of gc_field.cuh / gc_integrate.cuh /
// gc_compact.cuh; nothing here computes physics and there is no CPU fallback.
#include "../../include/gcoreccd.h"

#include <cmath>
#include <cstdarg>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <new>
#include <algorithm>
#include <cstdlib>
#include <vector>

#include <nvtx3/nvToolsExt.h>      // header-only NVTX v3: ranges are no-ops unless a tool (nsys, ncu) is attached

#include "gc_common.cuh"
#include "gc_advance.cuh"
#include "gc_compact.cuh"
#include "gc_events.cuh"
#include "gc_field.cuh"
#include "gc_frontend.cuh"
#include "gc_integrate.cuh"
#include "gc_microbench.cuh"
#include "gc_persist_warp.cuh"
#include "gc_noalloc.cuh"
#include "gc_persist.cuh"
#include "gc_shard.cuh"
#include "gc_tree.cuh"

using namespace gc;

namespace {

constexpr uint64_t kMaxCarriers = GCORECCD_MAX_CARRIERS;
constexpr uint64_t kPersistMaxDefault = 24576;          // populations up to this run many steps per launch (gc_persist.cuh)
constexpr uint64_t kPersistMaxLimit = 37888;            // 148 CTAs x 256: beyond, the one-step kernels are as fast
constexpr int kNumVariants = 8;                       // 0-2: one-step field kernels (2/4/8 targets per thread); 3-4: persistent
                                                      // multi-step kernels (4/8 targets per thread), 5: 2 targets per thread on 96 SMs for < 3,072 holes, gc_persist.cuh;
                                                      // 6-7: a warp owns 2 / 4 targets for the whole step, one CTA per SM (gc_persist_warp.cuh)
constexpr int kGraphSteps = 8;                        // steps per CUDA-graph launch

struct Layout {
  uint64_t cap_pad, part_cap, n_tiles, scan_entries, tree_scratch;
  uint64_t off_ctrl, off_A, off_B, off_Ep, off_tiles, off_scan, off_mutab, off_image, off_fin, total;
};

inline uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

Layout make_layout(uint64_t max_carriers, int32_t nx, int32_t ny) {
  Layout L;
  L.cap_pad = align_up(max_carriers, 1024);
  // Partial planes: S chunks x stride (= n_active rounded to 256) entries each.  A large population is balanced over
  // the SMs with few chunks (64+ row blocks x 16 chunks = 7+ rounds of 148 CTAs, <= 1.5 % idle), a small one needs many
  // (4 row blocks at 4,096 holes over 296 CTAs): 16 chunks at capacity, and never fewer entries than 128 chunks of 16,384 holes.
  L.part_cap = std::max<uint64_t>((uint64_t)kPartFactor * L.cap_pad, 128ull * std::min<uint64_t>(L.cap_pad, 16384));
  L.tree_scratch = 8 * L.cap_pad + 4096;                  // far-field variant: tail of plane x (see gcoreccd_create)
  L.n_tiles = L.cap_pad / kTPB;
  L.scan_entries = std::max<uint64_t>(L.n_tiles, 1024);   // look-back status words: 256-carrier tiles, or 64-carrier tiles of <= 65,536 holes
  uint64_t o = 0;
  L.off_ctrl = o;  o += align_up(sizeof(Ctrl), 256);
  L.off_A = o;     o += align_up(4 * L.cap_pad * 4, 256);
  L.off_B = o;     o += align_up(4 * L.cap_pad * 4, 256);
  L.off_Ep = o;    o += align_up(3 * L.part_cap * 4, 256);
  L.off_tiles = o; o += align_up(L.n_tiles * 4, 256);
  L.off_scan = o;  o += align_up(L.scan_entries * 8, 256);
  L.off_mutab = o; o += align_up((uint64_t)kMuTabEntries * 8, 256);      // eq. 2 interpolants (gc_integrate.cuh), 36 KB
  L.off_image = o; o += align_up((uint64_t)nx * (uint64_t)ny * 4, 256);
  L.off_fin = o;   o += align_up(L.cap_pad * 16, 256);
  L.total = o;
  return L;
}

}  // namespace

// Batched events: one kernel variant ("tier") per event size, so that the threads of a CTA are mostly busy:
// tier 0 one WARP per event (k_events_warp), tiers 1..4 one CTA of 32/64/128/256 threads with one packed pair of
// targets per thread, tier 5 (<= 768 holes) 256 threads with two pairs per thread and shared memory sized so that two events share
// an SM (measured: 600-hole events 1,502 -> 1,883 G pairs/s; at 1,000 holes the big tier is faster), tier 6 256
// threads with four pairs per thread.
constexpr int kEvTiers = 7;
constexpr uint32_t kEvTierCap[kEvTiers] = {kEvCapMicro, 64u, kEvCapTiny, 256u, kEvCapSmall, 768u, kEvCapLarge};
constexpr int kEvTierThreads[kEvTiers] = {128, 32, 64, 128, 256, 256, 256};
constexpr uint32_t kEvClusterFewFactor = 3;  // "few" = at most this many large events per SM
using EvKernel = void (*)(SoA, EventTable, const uint32_t*, uint32_t, uint32_t*, Ctrl*, Sink, DevParams, uint64_t, uint32_t);
inline EvKernel ev_kernel(int tier) {
  switch (tier) {
    case 1: return k_events<1, 32, 16>;
    case 2: return k_events<1, 64, 12>;
    case 3: return k_events<1, 128, 6>;
    case 4: return k_events<1, 256, 3>;
    case 5: return k_events<2, 256, 2>;          // <= 768 holes: 34 KB of shared memory, two CTAs per SM (registers)
    default: return k_events<4, 256, 1>;
  }
}

struct gcoreccd {
  gcoreccd_params p;
  DevParams dp;
  Layout L;
  int device;
  int num_sms;
  cudaStream_t stream;
  bool own_stream, own_ws;
  char* ws;
  Ctrl* ctrl;
  Ctrl* h_ctrl;                 // pinned mirror
  SoA A, B;
  float* Ep;
  uint32_t* tile_count;
  unsigned long long* scan;     // look-back status words (gc_advance.cuh)
  uint32_t* image;
  float4* fin;                  // per-id collection records
  Sink sink;
  uint64_t n_loaded;            // host copy (ids continue)
  uint64_t n_bound;             // host upper bound on n_active
  int variant;                  // current field variant (-1 = none yet)
  int grid_field[kNumVariants];       // persistent grid of each variant (3-4: co-resident CTAs of k_steps<>, cooperative launch)
  uint64_t launches;
  cudaGraphExec_t graph;
  int graph_variant;
  uint32_t graph_tiles;
  uint32_t graph_parts, graph_steps;  // treecode parts the graph was captured for (0: all-pairs), steps it holds
  uint64_t graph_launches;            // kernels in the graph
  uint32_t graph_cadence;             // re-sort cadence baked into a treecode graph
  cudaEvent_t ev[4];
  uint64_t persist_max;
  int persist_mode;                   // 1: every persistent kernel; 2: the CTA-tile kernels (k_steps) only
  bool persist_early_exit;            // set by run_to_collection around its launches
  bool persist_on;                    // many-steps-per-launch path for small populations (gc_persist.cuh); test hook turns it off
  uint32_t shard_rank, shard_world;   // target sharding (gc_shard.cuh); world 1 = not sharded
  uint32_t shard_epoch;               // changes at every reset / set_shard: tells this event's message headers from stale ones
  bool shard_wait;                    // shard_commit spins on the message headers (peer-mapped messages, no host barrier)
  bool ff_on;                         // far-field approximation (gc_tree.cuh)
  float ff_theta;
  uint32_t ff_parts;                  // CTAs (= partial chunks) per group of 256 targets; 0 = all-pairs kernel in use
  uint64_t ff_min_active;             // below this many active holes the all-pairs kernel is faster and is used
  uint32_t ff_resort, ff_age;         // re-sort cadence; field evaluations since set_farfield / reset
  bool ff_auto;                       // default cadence: every 2nd evaluation for the first 192, then every ff_resort-th
  int grid_tree;
  Tree tree;
  char err[256];
  // batched independent events (gc_events.cuh)
  struct {
    bool loaded;
    uint64_t n_events, n_carriers;        // as loaded
    uint64_t events_left, carriers_left;  // after the last run_events
    uint32_t n_q[kEvTiers];               // events per queue, smallest tier first (order = [tier 0..., tier 1..., ...])
    char* d_buf;                          // one allocation: off | cnt | order | queue | step (kept across batches)
    size_t d_buf_bytes, h_cap_events;     // capacities of d_buf and of the host mirrors
    uint32_t *d_off, *d_cnt, *d_order, *d_queue;
    uint64_t* d_step;
    uint32_t *h_off, *h_cnt;              // host mirrors
    uint64_t* h_step;
    int grid_q[kEvTiers];
    cudaStream_t aux[kEvTiers - 1];       // the smaller tiers run beside the largest one
    cudaEvent_t fork, join[kEvTiers - 1];
  } evb;
};

namespace {

// NVTX range around a host-side phase (SURVEY.md section 5 "Tracing"): field / advance / re-sort / load / batch of steps
struct Range {
  explicit Range(const char* name) { nvtxRangePushA(name); }
  ~Range() { nvtxRangePop(); }
};

struct DeviceGuard {
  int prev;
  bool changed;
  explicit DeviceGuard(int dev) : prev(-1), changed(false) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) { cudaSetDevice(dev); changed = true; }
  }
  ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
};

int fail(gcoreccd_t* h, int code, const char* what, cudaError_t e = cudaSuccess) {
  if (h) {
    if (e != cudaSuccess) snprintf(h->err, sizeof(h->err), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(h->err, sizeof(h->err), "%s", what);
  }
  return code;
}

#define GC_CUDA(h, call)                                                       \
  do {                                                                         \
    cudaError_t e__ = (call);                                                  \
    if (e__ != cudaSuccess) return fail((h), GCORECCD_ERR_CUDA, #call, e__);   \
  } while (0)

inline int variant_npack(int v) { return (v == 0 || v == 5 || v == 6) ? 1 : (v == 1 || v == 3 || v == 7) ? 2 : 4; }
inline bool variant_warp_owner(int v) { return v == 6 || v == 7; }
// holes a warp-owner variant can take: 2 NP targets per warp, 8 warps per CTA, one round
inline uint64_t warp_owner_cap(const gcoreccd_t* h, int v);
inline uint32_t variant_ib(int v) { return (uint32_t)kTPB * 2u * (uint32_t)variant_npack(v); }   // targets per row block
inline bool variant_persistent(int v) { return v >= 3; }

// Small populations run many steps per cooperative launch (gc_persist.cuh): all-pairs, unsharded handles only.
inline bool persist_eligible(const gcoreccd_t* h, uint64_t n) {
  return h->persist_on && !(h->dp.flags & GCORECCD_COULOMB_OFF) && h->shard_world == 1 && n <= h->persist_max &&
         !(h->ff_on && n >= h->ff_min_active) && h->grid_field[3] > 0 && h->grid_field[4] > 0;
}

inline uint64_t warp_owner_cap(const gcoreccd_t* h, int v) {
  return (uint64_t)h->grid_field[v] * (uint64_t)(kTPB / 32) * 2u * (uint64_t)variant_npack(v);
}

inline int pick_variant(const gcoreccd_t* h, uint64_t n, bool allow_persistent = true) {
  if (allow_persistent && persist_eligible(h, n)) {
    if (h->persist_mode != 2) {                              // (mode 2: the CTA-tile kernels only, for A/B measurements)
      for (int v = 6; v <= 7; ++v)
        if (n <= warp_owner_cap(h, v)) return v;             // 2,368 / 4,736 holes on 148 SMs (8 targets per warp was
                                                             // tried: 9 % ahead at 9,472 holes, 6 % behind at 8,192, where
                                                             // 64 targets per CTA leave 20 SMs without work)
    }
    return n >= 12288 ? 4 : n >= 3072 ? 3 : 5;
  }
  if (n >= 12288) return 2;            // 8 targets/thread, 1 CTA/SM: highest FMA-pipe utilisation (76 %)
  if (n >= 3072) return 1;             // 4 targets/thread, 3 CTAs/SM: more row blocks for balance
  return 0;                            // 2 targets/thread, 4 CTAs/SM
}

inline PlanArgs plan_args(const gcoreccd_t* h, int v) {
  PlanArgs a;
  a.IB = variant_ib(v);
  a.grid = (uint32_t)h->grid_field[v];
  // with the far-field variant on, the tail of the partial plane is the treecode's scratch (counters included): the
  // all-pairs kernel, which takes over below min_active holes, must not plan its chunks into it
  a.part_cap_entries = (uint32_t)(h->ff_on ? h->L.part_cap - h->L.tree_scratch : h->L.part_cap);
  a.rank = h->shard_rank;
  a.world = h->shard_world;
  a.force_S = h->ff_parts;
  return a;
}

inline uint32_t tiles_for(uint64_t n) { return (uint32_t)((n + kTPB - 1) / kTPB); }

inline uint32_t bucket_tiles(uint32_t t) {                  // power-of-two buckets keep graph re-captures rare
  uint32_t b = 1;
  while (b < t) b <<= 1;
  return b;
}

// Re-sort cadence at a given age.  Early in an event the cloud is dense and diffusion (0.55 um per step) scrambles the
// curve order within a few steps; later it ages slowly, hence the denser cadence at the start.
constexpr uint32_t kFfEarlyEvals = 192;
inline uint32_t ff_cadence_at(const gcoreccd_t* h, uint32_t age) {
  return (h->ff_auto && age < kFfEarlyEvals) ? std::min(2u, h->ff_resort) : h->ff_resort;
}

// Far-field variant (gc_tree.cuh): [Hilbert re-sort of the state every `cadence` evaluations] + nodes + walk/evaluate.
int launch_tree_field(gcoreccd_t* h) {
  const uint64_t nb = h->n_bound ? h->n_bound : 1;
  const uint32_t tiles = tiles_for(nb);
  const Tree& T = h->tree;
  const bool sort = h->ff_age % ff_cadence_at(h, h->ff_age) == 0;
  h->ff_age += 1;
  k_tree_reset<<<1, 256, 0, h->stream>>>(T.tc, sort ? 1 : 0);
  h->launches += 1;
  if (sort) {
    Range r_sort("gcoreccd: Hilbert re-sort");
    k_tree_bbox<<<std::min<uint32_t>(tiles, (uint32_t)h->num_sms * 4u), kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, T.tc);
    k_tree_keys<<<tiles, kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, T.tc, T.key[0], T.val[0]);
    const uint32_t sb = (uint32_t)((nb + kSortBlock - 1) / kSortBlock);
    int cur = 0;
    for (uint32_t shift = 0; shift < 8 * kKeyPasses; shift += 8) {
      uint32_t* tot = &T.tc->tot[shift / 8][0];
      k_radix_hist<<<sb, 256, 0, h->stream>>>(T.key[cur], h->ctrl, shift, T.counts, tot);
      k_radix_scatter<<<sb, 256, 0, h->stream>>>(T.key[cur], T.val[cur], T.key[cur ^ 1], T.val[cur ^ 1], h->ctrl, shift, T.counts, tot);
      cur ^= 1;
    }
    k_tree_permute<<<tiles, kTPB, 0, h->stream>>>(h->A, h->B, T.val[cur], h->ctrl);     // state B is scratch between steps
    k_tree_copy<<<tiles, kTPB, 0, h->stream>>>(h->B, h->A, h->ctrl);
    h->launches += 4 + 2 * kKeyPasses;
  }
  const uint32_t leaves = nodes_at((uint32_t)nb, 0);
  k_tree_leaves<<<(leaves * kLeaf + kTPB - 1) / kTPB, kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, T.node_c, T.node_r);
  // levels 1-2 (8 and 64 leaves per node): a warp per node; levels 3 .. top: a CTA per node; nothing above the top
  const uint32_t ltop = top_level((uint32_t)nb);
  const uint32_t low = (ltop >= 1 ? nodes_at((uint32_t)nb, 1) : 0u) + (ltop >= 2 ? nodes_at((uint32_t)nb, 2) : 0u);
  uint32_t high = 0;
  for (uint32_t l = 3; l <= ltop; ++l) high += nodes_at((uint32_t)nb, l);
  if (low) k_tree_upper<32><<<(low + 7) / 8, kTPB, 0, h->stream>>>(h->ctrl, T.node_c, T.node_r, 1u, 2u);
  if (high) k_tree_upper<kTPB><<<high, kTPB, 0, h->stream>>>(h->ctrl, T.node_c, T.node_r, 3u, kTreeMaxLevels - 1);
  h->launches += (low ? 1 : 0) + (high ? 1 : 0) - 1;
  k_tree_field<<<h->grid_tree, kTreeTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, T, h->Ep, (uint32_t)h->L.part_cap,
                                                         h->dp.eps2, h->ff_theta);
  h->launches += 3;
  return 0;
}

int launch_field(gcoreccd_t* h, int v) {
  Range r_field(h->ff_parts ? "gcoreccd: field (treecode)" : "gcoreccd: field (all pairs)");
  if (h->ff_parts) return launch_tree_field(h);
  const int g = h->grid_field[v];
  const uint32_t pc = (uint32_t)h->L.part_cap;
  switch (variant_npack(v)) {            // the plan was made for this variant's grid g (persistent variants included)
    case 1: k_field<1, 256, 4><<<g, kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, h->Ep, pc, h->dp.eps2); break;
    case 2: k_field<2, 256, 3><<<g, kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, h->Ep, pc, h->dp.eps2); break;
    default: k_field<4, 256, 1><<<g, kTPB, 0, h->stream>>>(h->A.x, h->A.y, h->A.z, h->ctrl, h->Ep, pc, h->dp.eps2); break;
  }
  h->launches += 1;
  return 0;
}

// one time step = field (a1) + advance (a2..a8: update, collection, in-place compaction), both reading n_active / the
// plan from device memory
void enqueue_step(gcoreccd_t* h, uint32_t tiles) {
  const bool coulomb = !(h->dp.flags & GCORECCD_COULOMB_OFF);
  if (coulomb) launch_field(h, h->variant);
  Range r_adv("gcoreccd: advance (a2..a8)");
  k_advance<<<tiles, kTPB, 0, h->stream>>>(h->A, h->ctrl, h->Ep, (uint32_t)h->L.part_cap, h->sink, h->scan, h->dp,
                                           plan_args(h, h->variant), coulomb ? 1u : 0u);
  h->launches += 1;
}

// Small populations: up to 2^20 steps in ONE cooperative launch (gc_persist.cuh).
int launch_persistent(gcoreccd_t* h, uint32_t n_steps) {
  Range r_p("gcoreccd: persistent steps (field + advance per step, one launch)");
  const int v = h->variant;
  SoA A = h->A; SoA B = h->B; Ctrl* ctrl = h->ctrl; float* Ep = h->Ep; uint32_t pc = (uint32_t)h->L.part_cap; Sink sink = h->sink;
  unsigned long long* scan = h->scan; DevParams dp = h->dp; PlanArgs pa = plan_args(h, v);
  // run_to_collection lets the launch end as soon as the population has decayed into the range of a smaller variant
  // (it reads Ctrl after every launch anyway); gcoreccd_step must take exactly n_steps
  uint32_t n_exit = 0;
  if (h->persist_early_exit && h->persist_mode != 2) {
    if (v == 7) n_exit = (uint32_t)warp_owner_cap(h, 6) + 1u;
    else if (v == 3 || v == 4) n_exit = (uint32_t)warp_owner_cap(h, 7) + 1u;
  }
  cudaError_t e;
  if (variant_warp_owner(v)) {
    void* args[] = {&A, &B, &ctrl, &sink, &scan, &dp, &pa, &n_steps, &n_exit};
    const void* fn = v == 6 ? (const void*)k_steps_warp<1> : (const void*)k_steps_warp<2>;
    // one CTA per 16 NP targets of the host's bound (the population only shrinks inside a launch), one CTA per SM at
    // most: a CTA that owns no target would only make the grid barrier slower
    const uint64_t per_cta = (uint64_t)(kTPB / 32) * 2u * (uint64_t)variant_npack(v);
    const unsigned grid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>((uint64_t)h->grid_field[v], (h->n_bound + per_cta - 1) / per_cta));
    e = cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kTPB), args, kWsSmemBytes, h->stream);
  } else {
    void* args[] = {&A, &B, &ctrl, &Ep, &pc, &sink, &scan, &dp, &pa, &n_steps, &n_exit};
    const void* fn = v == 4 ? (const void*)k_steps<4, 1> : v == 3 ? (const void*)k_steps<2, 2> : (const void*)k_steps<1, 2>;
    e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)h->grid_field[v]), dim3(kTPB), args, 0, h->stream);
  }
  if (e == cudaErrorCooperativeLaunchTooLarge) {             // fewer SMs than the occupancy query promised (MPS, green contexts)
    cudaGetLastError();
    return 1;                                                // the caller falls back to the two-launch path, for good
  }
  if (e != cudaSuccess) return fail(h, GCORECCD_ERR_CUDA, "cudaLaunchCooperativeKernel", e);
  h->launches += 1;
  return 0;
}

// parts per treecode group: enough work items for ~1.5 per resident CTA, power of two, at most 8 (workspace layout)
inline uint32_t pick_parts(const gcoreccd_t* h) {
  const uint64_t groups = ((h->n_bound + h->shard_world - 1) / h->shard_world + kGroup - 1) / kGroup;   // of this rank's share
  uint32_t P = 1;
  while (P < 8 && groups * P * 2 < 3ull * (uint64_t)h->grid_tree) P <<= 1;      // 1.5 measured best of 0.25 .. 4
  return P;
}

int ensure_variant(gcoreccd_t* h) {
  const int v = pick_variant(h, h->n_bound);
  const uint32_t parts = h->ff_on && h->n_bound >= h->ff_min_active ? pick_parts(h) : 0u;
  if (v != h->variant || parts != h->ff_parts) {
    h->ff_parts = parts;
    h->variant = v;
    k_replan<<<1, 32, 0, h->stream>>>(h->ctrl, plan_args(h, v), 0, 0u, 0, 0ull);
    h->launches += 1;
    GC_CUDA(h, cudaGetLastError());
  }
  return 0;
}

int sync_ctrl(gcoreccd_t* h) {
  GC_CUDA(h, cudaMemcpyAsync(h->h_ctrl, h->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  h->n_bound = h->h_ctrl->n_active;
  return 0;
}

void drop_graph(gcoreccd_t* h) {
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }
}

// Steps per graph: kGraphSteps for the all-pairs path; for the treecode a whole number of re-sort cycles (the graph
// starts with a re-sort), so that the host-scheduled cadence is baked in.  0 = do not use a graph.
inline uint32_t graph_steps_for(const gcoreccd_t* h) {
  if (!h->ff_parts) return kGraphSteps;
  const uint32_t c = ff_cadence_at(h, h->ff_age);
  if (c > 16) return 0;
  const uint32_t steps = c * ((kGraphSteps + c - 1) / c);
  return ff_cadence_at(h, h->ff_age + steps - 1) == c ? steps : 0;          // not across a change of cadence
}

int ensure_graph(gcoreccd_t* h, uint32_t tiles) {
  const uint32_t steps = graph_steps_for(h);
  const uint32_t cadence = h->ff_parts ? ff_cadence_at(h, h->ff_age) : 0u;
  if (h->graph && h->graph_variant == h->variant && h->graph_tiles == tiles && h->graph_parts == h->ff_parts &&
      h->graph_steps == steps && h->graph_cadence == cadence)
    return 0;
  drop_graph(h);
  cudaGraph_t g = nullptr;
  GC_CUDA(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
  const uint64_t before = h->launches;
  const uint32_t age = h->ff_age;
  for (uint32_t k = 0; k < steps; ++k) enqueue_step(h, tiles);
  h->graph_launches = h->launches - before;
  h->launches = before;                                   // capture does not launch ...
  h->ff_age = age;                                        // ... nor age the treecode's order
  const cudaError_t e_launch = cudaGetLastError();        // a launch refused during capture (bad configuration)
  cudaError_t e = cudaStreamEndCapture(h->stream, &g);    // always end the capture: the caller's stream must not stay in it
  if (e == cudaSuccess && e_launch != cudaSuccess) e = e_launch;
  if (e != cudaSuccess) {
    if (g) cudaGraphDestroy(g);
    cudaGetLastError();                                   // clear the sticky capture-invalidated status
    return fail(h, GCORECCD_ERR_CUDA, "CUDA graph capture of a batch of steps", e);
  }
  e = cudaGraphInstantiate(&h->graph, g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) { h->graph = nullptr; return fail(h, GCORECCD_ERR_CUDA, "cudaGraphInstantiate", e); }
  h->graph_variant = h->variant;
  h->graph_tiles = tiles;
  h->graph_parts = h->ff_parts;
  h->graph_steps = steps;
  h->graph_cadence = cadence;
  return 0;
}

int enqueue_steps(gcoreccd_t* h, uint64_t n_steps) {
  if (n_steps == 0 || h->n_bound == 0) return 0;
  Range r_steps("gcoreccd: batch of steps");
  int rc = ensure_variant(h);
  if (rc) return rc;
  const uint32_t tiles = bucket_tiles(tiles_for(h->n_bound));
  if (h->dp.flags & GCORECCD_COULOMB_OFF) {
    // independent carriers: one launch pair for the whole batch of steps (gc_integrate.cuh: k_drift_multi)
    while (n_steps > 0) {
      const uint32_t chunk = (uint32_t)std::min<uint64_t>(n_steps, 1u << 30);
      k_drift_multi<<<tiles, kTPB, 0, h->stream>>>(h->A, h->B, h->ctrl, h->sink, h->tile_count, h->dp, chunk);
      k_compact<<<tiles, kTPB, 0, h->stream>>>(h->B, h->A, h->ctrl, h->tile_count, h->scan, 0u, 0u, 2, h->dp.z_well, 0u,
                                               plan_args(h, h->variant));
      h->launches += 2;
      n_steps -= chunk;
    }
    GC_CUDA(h, cudaGetLastError());
    return 0;
  }
  if (variant_persistent(h->variant)) {
    while (n_steps > 0) {
      const uint32_t chunk = (uint32_t)std::min<uint64_t>(n_steps, 1u << 20);
      rc = launch_persistent(h, chunk);
      if (rc == 1) break;
      if (rc) return rc;
      n_steps -= chunk;
    }
    if (n_steps == 0) return 0;
    h->persist_on = false;                                   // not all CTAs fit on this device partition: two launches per step
    h->variant = -1;
    rc = ensure_variant(h);
    if (rc) return rc;
  }
  // stream capture is not permitted on the legacy / per-thread default streams: plain launches there
  const bool stream_ok = h->stream != cudaStreamLegacy && h->stream != cudaStreamPerThread && h->stream != nullptr;
  while (stream_ok && n_steps > 0) {
    // the treecode's graph begins with a re-sort: single steps until the cadence is at that point
    if (h->ff_parts && h->ff_age % ff_cadence_at(h, h->ff_age) != 0) { enqueue_step(h, tiles); --n_steps; continue; }
    const uint32_t gsteps = graph_steps_for(h);
    if (gsteps == 0 || n_steps < (uint64_t)gsteps) break;
    rc = ensure_graph(h, tiles);
    if (rc) return rc;
    GC_CUDA(h, cudaGraphLaunch(h->graph, h->stream));
    if (h->ff_parts) h->ff_age += gsteps;
    h->launches += h->graph_launches;
    n_steps -= gsteps;
  }
  for (; n_steps > 0; --n_steps) enqueue_step(h, tiles);
  GC_CUDA(h, cudaGetLastError());
  return 0;
}

// A batch's device buffer, host mirrors, side streams and events are kept from one batch to the next (a production
// run loads batch after batch): clear_events forgets the batch, free_events releases everything.
void clear_events(gcoreccd_t* h) {
  auto& B = h->evb;
  B.loaded = false;
  B.n_events = B.n_carriers = B.events_left = B.carriers_left = 0;
  for (int q = 0; q < kEvTiers; ++q) B.n_q[q] = 0;
}

void free_events(gcoreccd_t* h) {
  if (h->evb.d_buf) cudaFree(h->evb.d_buf);
  for (int k = 0; k < kEvTiers - 1; ++k) {
    if (h->evb.aux[k]) cudaStreamDestroy(h->evb.aux[k]);
    if (h->evb.join[k]) cudaEventDestroy(h->evb.join[k]);
  }
  if (h->evb.fork) cudaEventDestroy(h->evb.fork);
  free(h->evb.h_off); free(h->evb.h_cnt); free(h->evb.h_step);
  memset(&h->evb, 0, sizeof(h->evb));
}

// eq. 2: degree-kMuDeg Chebyshev interpolants of f(r) = (1 + r^beta)^(-1/beta) on every sixteenth of a binade, in long
// double, converted to monomial coefficients in u in [-1, 1] (gc_integrate.cuh mobility).  beta is the handle's double.
void build_mobility_table(double beta, std::vector<double>& tab) {
  constexpr int N = kMuDeg + 1;
  const long double pi = 3.14159265358979323846264338327950288L;
  const long double b = (long double)beta;
  // monomial coefficients of the Chebyshev polynomials T_0 .. T_deg
  long double T[N][N] = {};
  T[0][0] = 1.0L;
  if (N > 1) T[1][1] = 1.0L;
  for (int n = 2; n < N; ++n)
    for (int k = 0; k < N; ++k) T[n][k] = (k > 0 ? 2.0L * T[n - 1][k - 1] : 0.0L) - T[n - 2][k];
  tab.assign(kMuTabEntries, 0.0);
  for (int e = kMuEmin; e < kMuEmax; ++e) {
    for (int j = 0; j < kMuSub; ++j) {
      const long double mc = 1.0L + ((long double)j + 0.5L) / kMuSub, half = 0.5L / kMuSub;
      long double fv[N], cheb[N];
      for (int k = 0; k < N; ++k) {
        const long double u = cosl(pi * ((long double)k + 0.5L) / N);
        const long double r = ldexpl(mc + half * u, e);
        fv[k] = powl(1.0L + powl(r, b), -1.0L / b);
      }
      for (int n = 0; n < N; ++n) {
        long double acc = 0.0L;
        for (int k = 0; k < N; ++k) acc += fv[k] * cosl(pi * (long double)n * ((long double)k + 0.5L) / N);
        cheb[n] = acc * (n == 0 ? 1.0L : 2.0L) / N;
      }
      double* row = tab.data() + ((size_t)(e - kMuEmin) * kMuSub + j) * N;
      for (int k = 0; k < N; ++k) {
        long double mono = 0.0L;
        for (int n = 0; n < N; ++n) mono += cheb[n] * T[n][k];
        row[k] = (double)mono;
      }
    }
  }
}

inline bool events_busy(const gcoreccd_t* h) { return h->evb.loaded && h->evb.carriers_left > 0; }

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

uint64_t gcoreccd_workspace_size(uint64_t max_carriers, int32_t img_nx, int32_t img_ny) {
  if (max_carriers == 0 || max_carriers > kMaxCarriers || img_nx < 1 || img_ny < 1 || img_nx > 16384 || img_ny > 16384)
    return 0;
  return make_layout(max_carriers, img_nx, img_ny).total;
}

int gcoreccd_create(const gcoreccd_params* p, gcoreccd_t** out) {
  if (!p || !out) return GCORECCD_ERR_INVALID;
  if (p->struct_size != sizeof(gcoreccd_params)) return GCORECCD_ERR_INVALID;
  if (!(p->T_K > 0) || !(p->dt_ns > 0) || !(p->pixel_pitch_um > 0) || !(p->thickness_um > p->z_well_um) ||
      !(p->softening_um >= 0) || !(p->eps_si >= 0) || !std::isfinite(p->a1_V_per_cm2) || !std::isfinite(p->a2_V_per_cm) ||
      !std::isfinite(p->img_x0_um) || !std::isfinite(p->img_y0_um) || !std::isfinite(p->thickness_um) ||
      p->img_nx < 1 || p->img_ny < 1 || p->img_nx > 16384 || p->img_ny > 16384 || p->max_carriers == 0 ||
      p->max_carriers > kMaxCarriers || (p->flags & ~7u))
    return GCORECCD_ERR_INVALID;

  int dev = p->device;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return GCORECCD_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return GCORECCD_ERR_CUDA;
  if (prop.major != 10) return GCORECCD_ERR_CUDA;         // sm_100a only: no fallback path exists

  gcoreccd_t* h = new (std::nothrow) gcoreccd();
  if (!h) return GCORECCD_ERR_NOMEM;
  memset(h, 0, sizeof(*h));
  h->p = *p;
  if (h->p.eps_si == 0.0) h->p.eps_si = 11.7;
  h->device = dev;
  h->num_sms = prop.multiProcessorCount;
  h->variant = -1;
  h->shard_world = 1;
  h->persist_on = true;
  h->persist_mode = 1;
  h->persist_early_exit = false;
  h->persist_max = kPersistMaxDefault;
  DeviceGuard guard(dev);

  h->L = make_layout(p->max_carriers, p->img_nx, p->img_ny);
  int rc = GCORECCD_OK;
  cudaError_t e = cudaSuccess;
  do {
    if (p->workspace) {
      if (p->workspace_bytes < h->L.total || ((uintptr_t)p->workspace & 255u)) { rc = GCORECCD_ERR_CAPACITY; break; }
      h->ws = (char*)p->workspace;
    } else {
      e = cudaMalloc((void**)&h->ws, h->L.total);
      if (e != cudaSuccess) { rc = e == cudaErrorMemoryAllocation ? GCORECCD_ERR_NOMEM : GCORECCD_ERR_CUDA; break; }
      h->own_ws = true;
    }
    if (p->stream) h->stream = (cudaStream_t)p->stream;
    else {
      e = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking);
      if (e != cudaSuccess) { rc = GCORECCD_ERR_CUDA; break; }
      h->own_stream = true;
    }
    e = cudaMallocHost((void**)&h->h_ctrl, sizeof(Ctrl));
    if (e != cudaSuccess) { rc = GCORECCD_ERR_CUDA; break; }
    for (int k = 0; k < 4; ++k) {
      e = cudaEventCreate(&h->ev[k]);
      if (e != cudaSuccess) break;
    }
    if (e != cudaSuccess) { rc = GCORECCD_ERR_CUDA; break; }
  } while (0);
  if (rc != GCORECCD_OK) { gcoreccd_destroy(h); return rc; }

  const uint64_t cp = h->L.cap_pad;
  h->ctrl = (Ctrl*)(h->ws + h->L.off_ctrl);
  float* a = (float*)(h->ws + h->L.off_A);
  h->A = SoA{a, a + cp, a + 2 * cp, (uint32_t*)(a + 3 * cp)};
  float* b = (float*)(h->ws + h->L.off_B);
  h->B = SoA{b, b + cp, b + 2 * cp, (uint32_t*)(b + 3 * cp)};
  h->Ep = (float*)(h->ws + h->L.off_Ep);
  h->tile_count = (uint32_t*)(h->ws + h->L.off_tiles);
  h->scan = (unsigned long long*)(h->ws + h->L.off_scan);
  h->image = (uint32_t*)(h->ws + h->L.off_image);
  h->fin = (float4*)(h->ws + h->L.off_fin);
  h->sink = Sink{h->image, h->fin, (uint32_t)std::min<uint64_t>(p->max_carriers, 0xffffffffull)};

  // constants (eq. 2 temperature terms, K', thermal voltage) folded on the host in FP64
  const double q = 1.602176634e-19, kB = 1.380649e-23, eps0 = 8.8541878128e-12, pi = 3.14159265358979323846;
  DevParams& d = h->dp;
  const double T = p->T_K;
  d.a1_um = p->a1_V_per_cm2 * 1e-4;
  d.a2 = p->a2_V_per_cm;
  d.mu0 = 1.31e8 * std::pow(T, -2.2);
  d.inv_Ec = 1.0 / (1.24 * std::pow(T, 1.68));
  d.beta = 0.46 * std::pow(T, 0.17);
  d.inv_beta = 1.0 / d.beta;
  d.mu_tab = (const double*)(h->ws + h->L.off_mutab);
  {
    std::vector<double> tab;
    build_mobility_table(d.beta, tab);
    e = cudaMemcpyAsync(h->ws + h->L.off_mutab, tab.data(), tab.size() * 8, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);             // `tab` leaves scope
    if (e != cudaSuccess) { gcoreccd_destroy(h); return GCORECCD_ERR_CUDA; }
  }
  d.drift_k = 1e-5 * p->dt_ns;
  d.sigma_k = 2.0 * 0.1 * (kB * T / q) * p->dt_ns;
  d.thickness = p->thickness_um;
  d.z_well = p->z_well_um;
  d.x0 = p->img_x0_um; d.y0 = p->img_y0_um; d.pitch = p->pixel_pitch_um;
  d.Kp = q / (4.0 * pi * eps0 * h->p.eps_si) * 1e10;
  const double e2 = p->softening_um * p->softening_um;
  d.eps2 = (float)(e2 < 1e-24 ? 1e-24 : e2);              // eps = 0 -> eq. 5: coincident pairs contribute exactly 0
  d.flags = p->flags;
  d.seed_lo = (uint32_t)(p->seed & 0xffffffffu);
  d.seed_hi = (uint32_t)(p->seed >> 32);
  d.nx = p->img_nx; d.ny = p->img_ny;

  // persistent grid of the field kernel: resident CTAs per SM x SM count
  int occ[kNumVariants] = {0, 0, 0, 0, 0, 0, 0, 0};
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[0], k_field<1, 256, 4>, kTPB, 0);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[1], k_field<2, 256, 3>, kTPB, 0);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[2], k_field<4, 256, 1>, kTPB, 0);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[3], k_steps<2, 2>, kTPB, 0);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[4], k_steps<4, 1>, kTPB, 0);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[5], k_steps<1, 2>, kTPB, 0);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_steps_warp<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kWsSmemBytes);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_steps_warp<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kWsSmemBytes);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[6], k_steps_warp<1>, kTPB, kWsSmemBytes);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[7], k_steps_warp<2>, kTPB, kWsSmemBytes);
  if (e != cudaSuccess) { fail(h, GCORECCD_ERR_CUDA, "occupancy query", e); gcoreccd_destroy(h); return GCORECCD_ERR_CUDA; }
  for (int v = 0; v < 3; ++v) h->grid_field[v] = h->num_sms * (occ[v] > 0 ? occ[v] : 1);
  int coop = 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  for (int v = 3; v < 5; ++v) h->grid_field[v] = coop ? h->num_sms * std::min(occ[v], v == 3 ? 2 : 1) : 0;   // 0: no persistent path
  // < 3,072 holes: 96 tiles of 32 carriers at most; every CTA that only waits at the grid barriers makes them slower
  h->grid_field[5] = coop && occ[5] > 0 ? std::min(h->num_sms, 96) : 0;
  for (int v = 6; v <= 7; ++v) h->grid_field[v] = coop && occ[v] > 0 ? std::min(h->num_sms, kSegMaxCtas) : 0;   // one CTA per SM; 0: pick_variant never returns it
  int occ_tree = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_tree, k_tree_field, kTreeTPB, 0);
  if (e != cudaSuccess) { fail(h, GCORECCD_ERR_CUDA, "occupancy query", e); gcoreccd_destroy(h); return GCORECCD_ERR_CUDA; }
  h->grid_tree = h->num_sms * (occ_tree > 0 ? occ_tree : 1);
  {
    // treecode scratch: the last 8 cap_pad + 4,096 floats of partial plane x.  The treecode writes P <= 8 chunks, and
    // P > 1 only below ~35k holes (pick_parts), so its chunks end far below; with the variant on, the all-pairs plan is
    // confined to the entries in front of the scratch (plan_args); the load paths stage in the first 4 cap_pad floats.
    float* r = h->Ep + (h->L.part_cap - h->L.tree_scratch);
    Tree& T = h->tree;
    T.tc = (TreeCtrl*)r;                         r += 2048;                 // 6.2 KB: box, counters, digit totals
    T.node_c = (float4*)r;                       r += cp * 5 / 8 + 64;      // <= cp/7 + 9 nodes of 4 floats
    T.node_r = r;                                r += cp * 3 / 16 + 64;
    T.key[0] = (unsigned long long*)r; r += 2 * cp;  T.key[1] = (unsigned long long*)r; r += 2 * cp;
    T.val[0] = (uint32_t*)r; r += cp;  T.val[1] = (uint32_t*)r; r += cp;
    T.counts = (uint32_t*)r;                                                // 256 * cp / 2048 = cp / 8 entries
  }
  h->ff_resort = 4;
  h->ff_min_active = 24576;

  rc = gcoreccd_reset(h);
  if (rc != GCORECCD_OK) { gcoreccd_destroy(h); return rc; }
  *out = h;
  return GCORECCD_OK;
}

int gcoreccd_destroy(gcoreccd_t* h) {
  if (!h) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  if (h->stream) cudaStreamSynchronize(h->stream);
  drop_graph(h);
  free_events(h);
  for (int k = 0; k < 4; ++k) if (h->ev[k]) cudaEventDestroy(h->ev[k]);
  if (h->h_ctrl) cudaFreeHost(h->h_ctrl);
  if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
  if (h->own_ws && h->ws) cudaFree(h->ws);
  delete h;
  return GCORECCD_OK;
}

int gcoreccd_reset(gcoreccd_t* h) {
  if (!h) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  GC_CUDA(h, cudaMemsetAsync(h->ctrl, 0, sizeof(Ctrl), h->stream));
  GC_CUDA(h, cudaMemsetAsync(h->scan, 0, (size_t)h->L.scan_entries * 8, h->stream));   // scan_seq restarts: no stale stamps
  GC_CUDA(h, cudaMemsetAsync(h->image, 0, (size_t)h->p.img_nx * h->p.img_ny * 4, h->stream));
  GC_CUDA(h, cudaMemsetAsync(h->fin, 0xff, (size_t)h->L.cap_pad * 16, h->stream));     // NaN / all-ones = still drifting
  if (h->ff_on) GC_CUDA(h, cudaMemsetAsync(h->tree.tc, 0, sizeof(TreeCtrl), h->stream)); // far-field counters restart too
  h->ff_age = 0;
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  drop_graph(h);                                           // its grids were sized for the previous population
  clear_events(h);
  h->shard_epoch += 1;
  h->n_loaded = 0;
  h->n_bound = 0;
  h->variant = -1;
  h->err[0] = 0;
  return GCORECCD_OK;
}

int gcoreccd_load_carriers(gcoreccd_t* h, const float* xyz, uint64_t n, int on_device) {
  if (!h || (!xyz && n)) return GCORECCD_ERR_INVALID;
  if (n == 0) return GCORECCD_OK;
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "load_carriers: a batch of events is still drifting (run_events or reset first)");
  Range r_load("gcoreccd: load_carriers");
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  const uint64_t n_act = h->h_ctrl->n_active;
  if (n_act + n > h->p.max_carriers || h->n_loaded + n > 0xffffffffull) return fail(h, GCORECCD_ERR_CAPACITY, "load_carriers: capacity");
  drop_graph(h);                                           // the population grows: a cached graph's grids may be too small
  const float* src = xyz;
  if (!on_device) {
    GC_CUDA(h, cudaMemcpyAsync(h->Ep, xyz, n * 12, cudaMemcpyHostToDevice, h->stream));
    src = h->Ep;
  }
  const uint32_t tiles = tiles_for(n);
  GC_CUDA(h, cudaMemsetAsync(&h->ctrl->invalid, 0, 4, h->stream));
  k_validate<<<tiles, kTPB, 0, h->stream>>>(src, (uint32_t)n, h->ctrl, h->dp.thickness);
  h->launches += 1;
  rc = sync_ctrl(h);
  if (rc) return rc;
  if (h->h_ctrl->invalid) return fail(h, GCORECCD_ERR_INVALID, "load_carriers: non-finite coordinate or z > thickness");
  // the plan stored with the new n_active must match the variant the next step will use
  const int v = pick_variant(h, n_act + n);
  h->variant = v;
  k_unpack<<<tiles, kTPB, 0, h->stream>>>(src, (uint32_t)n, h->B, h->ctrl, (uint32_t)h->n_loaded, h->sink,
                                          h->tile_count, h->dp, h->shard_rank == 0 ? 1u : 0u);
  k_compact<<<tiles, kTPB, 0, h->stream>>>(h->B, h->A, h->ctrl, h->tile_count, h->scan, (uint32_t)n, (uint32_t)n_act, 1,
                                           h->dp.z_well, 0u, plan_args(h, v));
  h->launches += 2;
  GC_CUDA(h, cudaGetLastError());
  h->n_loaded += n;
  rc = sync_ctrl(h);
  if (rc) return rc;
  h->variant = -1;                                         // re-pick (and re-plan) from the exact count
  return GCORECCD_OK;
}

int gcoreccd_load_snapshot(gcoreccd_t* h, const float* xyz, const uint32_t* id, uint64_t n, uint64_t step) {
  if (!h || ((!xyz || !id) && n)) return GCORECCD_ERR_INVALID;
  if (n > h->p.max_carriers) return fail(h, GCORECCD_ERR_CAPACITY, "load_snapshot: capacity");
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "load_snapshot: a batch of events is still drifting");
  DeviceGuard guard(h->device);
  drop_graph(h);
  float* st_xyz = h->Ep;
  uint32_t* st_id = (uint32_t*)(h->Ep + 3 * h->L.cap_pad);
  if (n) {
    GC_CUDA(h, cudaMemcpyAsync(st_xyz, xyz, n * 12, cudaMemcpyHostToDevice, h->stream));
    GC_CUDA(h, cudaMemcpyAsync(st_id, id, n * 4, cudaMemcpyHostToDevice, h->stream));
    // same validation as load_carriers; in addition an ACTIVE carrier must be above the collection plane
    GC_CUDA(h, cudaMemsetAsync(&h->ctrl->invalid, 0, 4, h->stream));
    k_validate<<<tiles_for(n), kTPB, 0, h->stream>>>(st_xyz, (uint32_t)n, h->ctrl, h->dp.thickness);
    h->launches += 1;
    int rc = sync_ctrl(h);
    if (rc) return rc;
    if (h->h_ctrl->invalid) return fail(h, GCORECCD_ERR_INVALID, "load_snapshot: non-finite coordinate or z > thickness");
    for (uint64_t k = 0; k < n; ++k)
      if (!((double)xyz[3 * k + 2] > h->p.z_well_um)) return fail(h, GCORECCD_ERR_INVALID, "load_snapshot: an active carrier must have z > z_well");
    k_set_snapshot<<<tiles_for(n), kTPB, 0, h->stream>>>(st_xyz, st_id, (uint32_t)n, h->A);
    h->launches += 1;
  }
  // sharded handles: every rank loads the same snapshot; the plan below is this rank's share of it
  const int v = pick_variant(h, h->shard_world > 1 ? (n + h->shard_world - 1) / h->shard_world : n);
  h->variant = v;
  h->ff_parts = 0;
  k_replan<<<1, 32, 0, h->stream>>>(h->ctrl, plan_args(h, v), 1, (uint32_t)n, 1, step);
  h->launches += 1;
  GC_CUDA(h, cudaGetLastError());
  uint64_t max_id = 0;
  for (uint64_t k = 0; k < n; ++k) if (id[k] > max_id) max_id = id[k];
  if (n && h->n_loaded < max_id + 1) h->n_loaded = max_id + 1;
  // keep the device copy in step with the host's: get_state's invariant is stated on n_loaded
  GC_CUDA(h, cudaMemcpyAsync(&h->ctrl->n_loaded, &h->n_loaded, 8, cudaMemcpyHostToDevice, h->stream));
  int rc = sync_ctrl(h);
  if (rc) return rc;
  h->variant = -1;                                         // the next step re-picks (far-field parts included)
  return GCORECCD_OK;
}

int gcoreccd_step(gcoreccd_t* h, uint32_t n_steps) {
  if (!h) return GCORECCD_ERR_INVALID;
  if (h->shard_world > 1) return fail(h, GCORECCD_ERR_STATE, "step: the handle is sharded (use shard_local / shard_commit)");
  DeviceGuard guard(h->device);
  return enqueue_steps(h, n_steps);
}

int gcoreccd_run_to_collection(gcoreccd_t* h, uint64_t max_steps, uint64_t* steps_done, uint64_t* n_active_left) {
  if (!h) return GCORECCD_ERR_INVALID;
  if (h->shard_world > 1) return fail(h, GCORECCD_ERR_STATE, "run_to_collection: the handle is sharded");
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  const uint64_t step0 = h->h_ctrl->step;
  uint64_t done = 0;
  int ret = GCORECCD_OK;
  while (h->h_ctrl->n_active > 0) {
    if (done >= max_steps) { ret = GCORECCD_MAX_STEPS; break; }
    // Coulomb off, or a population small enough for the persistent kernel: the launch itself loops until nobody drifts
    uint64_t batch = ((h->dp.flags & GCORECCD_COULOMB_OFF) || variant_persistent(pick_variant(h, h->n_bound))) ? (1ull << 20)
                                                                                                            : 4 * kGraphSteps;
    if (batch > max_steps - done) batch = max_steps - done;
    h->persist_early_exit = true;
    rc = enqueue_steps(h, batch);
    h->persist_early_exit = false;
    if (rc) return rc;
    rc = sync_ctrl(h);
    if (rc) return rc;
    if (h->h_ctrl->nonfinite) return fail(h, GCORECCD_ERR_NONFINITE, "a carrier position became non-finite");
    done = h->h_ctrl->step - step0;
  }
  if (steps_done) *steps_done = done;
  if (n_active_left) *n_active_left = h->h_ctrl->n_active;
  return ret;
}

int gcoreccd_read_image(gcoreccd_t* h, uint32_t* out, uint64_t cap_elems, uint64_t* n_out_of_window, int on_device) {
  if (!h || !out) return GCORECCD_ERR_INVALID;
  const uint64_t ne = (uint64_t)h->p.img_nx * h->p.img_ny;
  if (cap_elems < ne) return fail(h, GCORECCD_ERR_CAPACITY, "read_image: buffer too small");
  DeviceGuard guard(h->device);
  GC_CUDA(h, cudaMemcpyAsync(out, h->image, ne * 4, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  int rc = sync_ctrl(h);
  if (rc) return rc;
  if (n_out_of_window) *n_out_of_window = h->h_ctrl->n_overflow;
  return GCORECCD_OK;
}

int gcoreccd_get_state(gcoreccd_t* h, uint64_t* step, uint64_t* n_active, uint64_t* n_loaded, uint64_t* n_collected,
                       uint64_t* n_out_of_window, uint64_t* pair_interactions) {
  if (!h) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  if (step) *step = h->h_ctrl->step;
  if (n_active) *n_active = h->h_ctrl->n_active + (h->evb.loaded ? h->evb.carriers_left : 0);
  if (n_loaded) *n_loaded = h->h_ctrl->n_loaded;
  if (n_collected) *n_collected = h->h_ctrl->n_collected;
  if (n_out_of_window) *n_out_of_window = h->h_ctrl->n_overflow;
  if (pair_interactions) *pair_interactions = h->h_ctrl->pairs;
  if (h->h_ctrl->nonfinite) return fail(h, GCORECCD_ERR_NONFINITE, "a carrier position became non-finite");
  if (h->h_ctrl->diverged) return fail(h, GCORECCD_ERR_STATE, "shard messages disagree with this rank's state (ranks diverged)");
  return GCORECCD_OK;
}

int gcoreccd_read_carriers(gcoreccd_t* h, float* xyz, uint32_t* id, uint64_t cap, uint64_t* n, int on_device) {
  if (!h) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  const uint64_t na = h->h_ctrl->n_active;
  if (n) *n = na;
  if ((xyz || id) && cap < na) return fail(h, GCORECCD_ERR_CAPACITY, "read_carriers: buffer too small");
  if (na == 0) return GCORECCD_OK;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  if (xyz) {
    float* stage = on_device ? xyz : h->Ep;
    k_interleave<<<tiles_for(na), kTPB, 0, h->stream>>>(h->A, h->ctrl, stage);
    h->launches += 1;
    if (!on_device) GC_CUDA(h, cudaMemcpyAsync(xyz, stage, na * 12, kind, h->stream));
  }
  if (id) GC_CUDA(h, cudaMemcpyAsync(id, h->A.id, na * 4, kind, h->stream));
  GC_CUDA(h, cudaGetLastError());
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  return GCORECCD_OK;
}

int gcoreccd_read_collected(gcoreccd_t* h, float* xyz, uint32_t* step, uint64_t cap, uint64_t* n) {
  if (!h) return GCORECCD_ERR_INVALID;
  const uint64_t m = std::min<uint64_t>(h->n_loaded, h->sink.fin_cap);
  if (n) *n = m;
  if (!xyz && !step) return GCORECCD_OK;
  if (!xyz || !step) return fail(h, GCORECCD_ERR_INVALID, "read_collected: pass both buffers or neither");
  if (cap < m) return fail(h, GCORECCD_ERR_CAPACITY, "read_collected: buffer too small");
  if (m == 0) return GCORECCD_OK;
  DeviceGuard guard(h->device);
  float* st_xyz = h->Ep;                                   // partials are scratch between steps
  uint32_t* st_step = (uint32_t*)(h->Ep + 3 * h->L.cap_pad);
  k_read_final<<<tiles_for(m), kTPB, 0, h->stream>>>(h->fin, (uint32_t)m, st_xyz, st_step);
  h->launches += 1;
  GC_CUDA(h, cudaGetLastError());
  GC_CUDA(h, cudaMemcpyAsync(xyz, st_xyz, m * 12, cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaMemcpyAsync(step, st_step, m * 4, cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  return GCORECCD_OK;
}

int gcoreccd_eval_field(gcoreccd_t* h, float* E, uint64_t cap, int on_device) {
  if (!h || !E) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  const uint64_t na = h->h_ctrl->n_active;
  if (cap < na) return fail(h, GCORECCD_ERR_CAPACITY, "eval_field: buffer too small");
  if (h->shard_world > 1) return fail(h, GCORECCD_ERR_STATE, "eval_field: the handle is sharded");
  if (na == 0) return GCORECCD_OK;
  rc = ensure_variant(h);
  if (rc) return rc;
  launch_field(h, h->variant);
  float* stage = on_device ? E : h->B.x;                   // state B is scratch between steps (3*cap_pad floats)
  k_field_finalize<<<tiles_for(na), kTPB, 0, h->stream>>>(h->ctrl, h->Ep, (uint32_t)h->L.part_cap, h->dp.Kp, stage);
  h->launches += 1;
  if (!on_device) GC_CUDA(h, cudaMemcpyAsync(E, stage, na * 12, cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaGetLastError());
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  return GCORECCD_OK;
}

int gcoreccd_profile_step(gcoreccd_t* h, float ms[4]) {
  if (!h || !ms) return GCORECCD_ERR_INVALID;
  DeviceGuard guard(h->device);
  ms[0] = ms[1] = ms[2] = ms[3] = 0.f;
  if (h->shard_world > 1) return fail(h, GCORECCD_ERR_STATE, "profile_step: the handle is sharded");
  if (h->n_bound == 0) return GCORECCD_OK;
  int rc = ensure_variant(h);
  if (rc) return rc;
  const uint32_t tiles = bucket_tiles(tiles_for(h->n_bound));
  const bool coulomb = !(h->dp.flags & GCORECCD_COULOMB_OFF);
  GC_CUDA(h, cudaEventRecord(h->ev[0], h->stream));
  if (coulomb) launch_field(h, h->variant);
  GC_CUDA(h, cudaEventRecord(h->ev[1], h->stream));
  k_advance<<<tiles, kTPB, 0, h->stream>>>(h->A, h->ctrl, h->Ep, (uint32_t)h->L.part_cap, h->sink, h->scan, h->dp,
                                           plan_args(h, h->variant), coulomb ? 1u : 0u);
  GC_CUDA(h, cudaEventRecord(h->ev[2], h->stream));
  GC_CUDA(h, cudaEventRecord(h->ev[3], h->stream));
  h->launches += 1;
  GC_CUDA(h, cudaGetLastError());
  rc = sync_ctrl(h);
  if (rc) return rc;
  GC_CUDA(h, cudaEventElapsedTime(&ms[0], h->ev[0], h->ev[1]));
  GC_CUDA(h, cudaEventElapsedTime(&ms[1], h->ev[1], h->ev[2]));
  GC_CUDA(h, cudaEventElapsedTime(&ms[2], h->ev[2], h->ev[3]));
  GC_CUDA(h, cudaEventElapsedTime(&ms[3], h->ev[0], h->ev[3]));
  return GCORECCD_OK;
}

int gcoreccd_set_persistent(gcoreccd_t* h, int on, uint64_t max_active) {
  if (!h || max_active > kPersistMaxLimit) return GCORECCD_ERR_INVALID;
  if (on < 0 || on > 2) return GCORECCD_ERR_INVALID;
  h->persist_on = on != 0;
  h->persist_mode = on == 2 ? 2 : 1;
  h->persist_max = max_active ? max_active : kPersistMaxDefault;
  h->variant = -1;                                         // re-pick the kernel variant (and re-plan) at the next step
  return GCORECCD_OK;
}

// ---- target sharding (gc_shard.cuh) ----------------------------------------------------------------------------
namespace {
// entries per coordinate array of a shard message for the host's current bound on n_active: the largest share of
// ceil(tiles / world) tiles, tiles taken from the same power-of-two bucket on every rank
inline uint64_t shard_bs(const gcoreccd_t* h) {
  const uint64_t tiles = bucket_tiles(tiles_for(h->n_bound ? h->n_bound : 1));
  return (uint64_t)kTPB * ((tiles + h->shard_world - 1) / h->shard_world);
}
// entries per coordinate array a caller's message of msg_bytes holds (0 if it cannot hold the largest share)
inline uint64_t shard_bs_of(const gcoreccd_t* h, uint64_t msg_bytes) {
  if (msg_bytes < kShardHeaderBytes + 16ull * kTPB) return 0;
  const uint64_t bs = (msg_bytes - kShardHeaderBytes) / 16 / kTPB * kTPB;
  const uint64_t need = (uint64_t)kTPB * ((tiles_for(h->n_bound ? h->n_bound : 1) + h->shard_world - 1) / h->shard_world);
  return bs >= need && bs <= 0xffffff00ull ? bs : 0;
}
}  // namespace

int gcoreccd_set_shard(gcoreccd_t* h, uint32_t rank, uint32_t world) {
  if (!h || world == 0 || world > kShardMaxWorld || rank >= world) return GCORECCD_ERR_INVALID;
  if (world > 1 && (h->dp.flags & GCORECCD_COULOMB_OFF))
    return fail(h, GCORECCD_ERR_INVALID, "set_shard: without eq. 6 carriers are independent; run replicas instead");
  if (h->n_loaded != 0 || h->evb.loaded) return fail(h, GCORECCD_ERR_STATE, "set_shard: only on an empty handle (reset first)");
  h->shard_rank = rank;
  h->shard_world = world;
  h->shard_epoch += 1;
  h->variant = -1;
  return GCORECCD_OK;
}

int gcoreccd_set_shard_wait(gcoreccd_t* h, int on) {
  if (!h) return GCORECCD_ERR_INVALID;
  h->shard_wait = on != 0;
  return GCORECCD_OK;
}

uint64_t gcoreccd_shard_message_bytes(gcoreccd_t* h) {
  if (!h) return 0;
  return kShardHeaderBytes + 16ull * shard_bs(h);
}

int gcoreccd_shard_local(gcoreccd_t* h, void* msg_dev, uint64_t msg_bytes) {
  if (!h || !msg_dev) return GCORECCD_ERR_INVALID;
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "shard_local: a batch of events is loaded");
  const uint64_t bs = shard_bs_of(h, msg_bytes);
  if (bs == 0) return fail(h, GCORECCD_ERR_CAPACITY, "shard_local: message buffer too small");
  if ((uintptr_t)msg_dev & 15u) return fail(h, GCORECCD_ERR_INVALID, "shard_local: message buffer must be 16-byte aligned");
  DeviceGuard guard(h->device);
  // the share shrinks with n_active: pick the field variant from the share, not from the whole population
  // (a shard of a world of ONE must plan like the two-launch path it is made of, not like the persistent kernel)
  const int v = pick_variant(h, (h->n_bound + h->shard_world - 1) / h->shard_world, false);
  const uint32_t parts = h->ff_on && h->n_bound >= h->ff_min_active ? pick_parts(h) : 0u;   // treecode walk of the share
  if (v != h->variant || parts != h->ff_parts) {
    h->variant = v;
    h->ff_parts = parts;
    k_replan<<<1, 32, 0, h->stream>>>(h->ctrl, plan_args(h, v), 0, 0u, 0, 0ull);
    h->launches += 1;
  }
  const uint32_t tiles = (uint32_t)(bs / kTPB);
  launch_field(h, h->variant);
  k_integrate<<<tiles, kTPB, 0, h->stream>>>(h->A, h->B, h->ctrl, h->Ep, (uint32_t)h->L.part_cap, h->sink,
                                             h->tile_count, h->dp);
  k_shard_compact<<<tiles, kTPB, 0, h->stream>>>(h->B, h->ctrl, h->tile_count, (char*)msg_dev, (uint32_t)bs,
                                                 h->dp.z_well, h->shard_rank, h->shard_epoch);
  h->launches += 2;
  GC_CUDA(h, cudaGetLastError());
  return GCORECCD_OK;
}

int gcoreccd_shard_commit(gcoreccd_t* h, const void* const* msgs_host, uint32_t n_msgs, uint64_t msg_bytes) {
  if (!h || !msgs_host) return GCORECCD_ERR_INVALID;
  if (n_msgs != h->shard_world) return fail(h, GCORECCD_ERR_INVALID, "shard_commit: one message per rank is required");
  const uint64_t bs = shard_bs_of(h, msg_bytes);
  if (bs == 0) return fail(h, GCORECCD_ERR_CAPACITY, "shard_commit: message buffers too small");
  ShardPtrs ptrs;
  memset(&ptrs, 0, sizeof(ptrs));
  for (uint32_t g = 0; g < n_msgs; ++g) {
    if (!msgs_host[g] || ((uintptr_t)msgs_host[g] & 15u)) return fail(h, GCORECCD_ERR_INVALID, "shard_commit: bad message pointer");
    ptrs.p[g] = (const char*)msgs_host[g];
  }
  DeviceGuard guard(h->device);
  const uint32_t tiles = (uint32_t)(bs / kTPB);
  k_shard_commit<<<tiles * n_msgs, kTPB, 0, h->stream>>>(ptrs, n_msgs, (uint32_t)bs, h->A, h->ctrl, plan_args(h, h->variant),
                                                         h->shard_wait ? 1u : 0u, h->shard_epoch);
  h->launches += 1;
  GC_CUDA(h, cudaGetLastError());
  return GCORECCD_OK;
}

// ---- far-field variant (gc_tree.cuh) ---------------------------------------------------------------------------
int gcoreccd_set_farfield(gcoreccd_t* h, double theta, uint32_t resort_every, uint64_t min_active) {
  if (!h || !(theta < 1.0)) return GCORECCD_ERR_INVALID;
  if (theta >= 0.0 && h->L.cap_pad > (1ull << 26)) return fail(h, GCORECCD_ERR_CAPACITY, "set_farfield: capacity");
  DeviceGuard guard(h->device);
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  drop_graph(h);
  h->ff_on = theta >= 0.0;
  h->ff_theta = (float)(theta >= 0.0 ? theta : 0.0);
  h->ff_resort = resort_every ? resort_every : 4u;
  h->ff_auto = resort_every == 0;
  h->ff_min_active = min_active ? min_active : 24576u;
  h->ff_parts = 0;
  h->ff_age = 0;
  h->variant = -1;                                           // re-plan: the treecode writes one chunk (S = 1)
  if (h->ff_on) GC_CUDA(h, cudaMemsetAsync(h->tree.tc, 0, sizeof(TreeCtrl), h->stream));
  return GCORECCD_OK;
}

int gcoreccd_farfield_stats(gcoreccd_t* h, uint64_t* far_evals, uint64_t* near_evals, double* bound_B) {
  if (!h) return GCORECCD_ERR_INVALID;
  if (!h->ff_on) return fail(h, GCORECCD_ERR_STATE, "farfield_stats: the far-field variant is off");
  DeviceGuard guard(h->device);
  TreeCtrl tc;
  GC_CUDA(h, cudaMemcpyAsync(&tc, h->tree.tc, sizeof(tc), cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  if (far_evals) *far_evals = tc.far_evals;
  if (near_evals) *near_evals = tc.near_evals;
  const double t = h->ff_theta;
  if (bound_B) *bound_B = t * t * (3.0 - 2.0 * t) / ((1.0 - t) * (1.0 - t));
  return GCORECCD_OK;
}

uint64_t gcoreccd_kernel_launches(gcoreccd_t* h) { return h ? h->launches : 0; }

int gcoreccd_mobility_table_host(double T_K, const double* E, uint64_t n, double* mu) {
  if (!(T_K > 0) || !E || !mu) return GCORECCD_ERR_INVALID;
  const double mu0 = 1.31e8 * std::pow(T_K, -2.2), inv_Ec = 1.0 / (1.24 * std::pow(T_K, 1.68)), beta = 0.46 * std::pow(T_K, 0.17);
  std::vector<double> tab;
  build_mobility_table(beta, tab);
  for (uint64_t i = 0; i < n; ++i) {                         // the host twin of gc_integrate.cuh mobility()
    const double r = E[i] * inv_Ec;
    long long bits;
    memcpy(&bits, &r, 8);
    const int e = (int)((bits >> 52) & 0x7ff) - 1023;
    if (e < kMuEmin || e >= kMuEmax || bits < 0) { mu[i] = mu0 * std::exp(-std::log1p(std::exp(beta * std::log(r))) / beta); continue; }
    const int j = (int)((bits >> 48) & 15);
    const long long mb = (bits & 0x000fffffffffffffLL) | 0x3ff0000000000000LL;
    double m;
    memcpy(&m, &mb, 8);
    const double u = (m - (1.0 + ((double)j + 0.5) * (1.0 / kMuSub))) * (2.0 * kMuSub);
    const double* c = tab.data() + ((size_t)(e - kMuEmin) * kMuSub + j) * (kMuDeg + 1);
    double f = c[kMuDeg];
    for (int k = kMuDeg - 1; k >= 0; --k) f = std::fma(f, u, c[k]);
    mu[i] = mu0 * f;
  }
  return GCORECCD_OK;
}

int gcoreccd_debug_mobility(gcoreccd_t* h, const double* E, uint64_t n, double* mu_table, double* mu_direct) {
  if (!h || !E || !mu_table || !mu_direct) return GCORECCD_ERR_INVALID;
  if (n == 0) return GCORECCD_OK;
  DeviceGuard guard(h->device);
  double* buf = nullptr;
  GC_CUDA(h, cudaMalloc((void**)&buf, n * 24));
  cudaError_t e = cudaMemcpyAsync(buf, E, n * 8, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) {
    k_debug_mobility<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(buf, (uint32_t)n, h->dp, buf + n, buf + 2 * n);
    h->launches += 1;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(mu_table, buf + n, n * 8, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(mu_direct, buf + 2 * n, n * 8, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  cudaFree(buf);
  if (e != cudaSuccess) return fail(h, GCORECCD_ERR_CUDA, "debug_mobility", e);
  return GCORECCD_OK;
}

int gcoreccd_debug_normals(gcoreccd_t* h, const uint32_t* id, const uint64_t* step, uint64_t n, double* out, uint32_t* words) {
  if (!h || !id || !step || !out || !words) return GCORECCD_ERR_INVALID;
  if (n == 0) return GCORECCD_OK;
  DeviceGuard guard(h->device);
  char* buf = nullptr;
  const size_t b_id = align_up(n * 4, 256), b_st = align_up(n * 8, 256), b_out = align_up(n * 24, 256), b_w = align_up(n * 16, 256);
  GC_CUDA(h, cudaMalloc((void**)&buf, b_id + b_st + b_out + b_w));
  uint32_t* d_id = (uint32_t*)buf;
  uint64_t* d_st = (uint64_t*)(buf + b_id);
  double* d_out = (double*)(buf + b_id + b_st);
  uint32_t* d_w = (uint32_t*)(buf + b_id + b_st + b_out);
  cudaError_t e = cudaMemcpyAsync(d_id, id, n * 4, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_st, step, n * 8, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) {
    k_debug_normals<<<(unsigned)((n + 127) / 128), 128, 0, h->stream>>>(d_id, d_st, (uint32_t)n, h->dp.seed_lo, h->dp.seed_hi, d_out, d_w);
    h->launches += 1;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(out, d_out, n * 24, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(words, d_w, n * 16, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  cudaFree(buf);
  if (e != cudaSuccess) return fail(h, GCORECCD_ERR_CUDA, "debug_normals", e);
  return GCORECCD_OK;
}

// ---------------------------------------------------------------------------- batched independent events
int gcoreccd_load_events(gcoreccd_t* h, const float* xyz, const uint64_t* offsets, uint64_t n_events, int on_device) {
  if (!h || !offsets || n_events == 0 || n_events > 0x7fffffffull) return GCORECCD_ERR_INVALID;
  if (h->shard_world > 1) return fail(h, GCORECCD_ERR_STATE, "load_events: the handle is sharded (independent events shard as replicas)");
  const uint64_t n = offsets[n_events];
  if (offsets[0] != 0 || (!xyz && n)) return fail(h, GCORECCD_ERR_INVALID, "load_events: offsets[0] must be 0");
  for (uint64_t e = 0; e < n_events; ++e) {
    if (offsets[e + 1] < offsets[e]) return fail(h, GCORECCD_ERR_INVALID, "load_events: offsets must be non-decreasing");
    if (offsets[e + 1] - offsets[e] > GCORECCD_EVENT_MAX_CARRIERS)
      return fail(h, GCORECCD_ERR_CAPACITY, "load_events: an event exceeds GCORECCD_EVENT_MAX_CARRIERS");
  }
  if (n > h->p.max_carriers || h->n_loaded + n > 0xffffffffull) return fail(h, GCORECCD_ERR_CAPACITY, "load_events: capacity");
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "load_events: the previous batch is still drifting (run_events or reset first)");
  DeviceGuard guard(h->device);
  int rc = sync_ctrl(h);
  if (rc) return rc;
  if (h->h_ctrl->n_active) return fail(h, GCORECCD_ERR_STATE, "load_events: the handle holds a single event that is still drifting");

  const float* src = xyz;
  if (n) {
    if (!on_device) {
      GC_CUDA(h, cudaMemcpyAsync(h->Ep, xyz, n * 12, cudaMemcpyHostToDevice, h->stream));
      src = h->Ep;
    }
    GC_CUDA(h, cudaMemsetAsync(&h->ctrl->invalid, 0, 4, h->stream));
    k_validate<<<tiles_for(n), kTPB, 0, h->stream>>>(src, (uint32_t)n, h->ctrl, h->dp.thickness);
    h->launches += 1;
    rc = sync_ctrl(h);
    if (rc) return rc;
    if (h->h_ctrl->invalid) return fail(h, GCORECCD_ERR_INVALID, "load_events: non-finite coordinate or z > thickness");
  }

  clear_events(h);
  auto& B = h->evb;
  const size_t ne = (size_t)n_events;
  const size_t b_off = align_up((ne + 1) * 4, 256), b_cnt = align_up(ne * 4, 256), b_ord = align_up(ne * 4, 256), b_q = 256,
               b_step = align_up(ne * 8, 256);
  cudaError_t e = cudaSuccess;
  if (b_off + b_cnt + b_ord + b_q + b_step > B.d_buf_bytes) {
    if (B.d_buf) cudaFree(B.d_buf);
    B.d_buf = nullptr; B.d_buf_bytes = 0;
    e = cudaMalloc((void**)&B.d_buf, b_off + b_cnt + b_ord + b_q + b_step);
    if (e != cudaSuccess) { B.d_buf = nullptr; return fail(h, e == cudaErrorMemoryAllocation ? GCORECCD_ERR_NOMEM : GCORECCD_ERR_CUDA, "load_events: cudaMalloc", e); }
    B.d_buf_bytes = b_off + b_cnt + b_ord + b_q + b_step;
  }
  B.d_off = (uint32_t*)B.d_buf;
  B.d_cnt = (uint32_t*)(B.d_buf + b_off);
  B.d_order = (uint32_t*)(B.d_buf + b_off + b_cnt);
  B.d_queue = (uint32_t*)(B.d_buf + b_off + b_cnt + b_ord);
  B.d_step = (uint64_t*)(B.d_buf + b_off + b_cnt + b_ord + b_q);
  if (ne > B.h_cap_events) {
    free(B.h_off); free(B.h_cnt); free(B.h_step);
    B.h_off = (uint32_t*)malloc((ne + 1) * 4);
    B.h_cnt = (uint32_t*)malloc(ne * 4 + 4);
    B.h_step = (uint64_t*)malloc((ne + 1) * 8);
    B.h_cap_events = (B.h_off && B.h_cnt && B.h_step) ? ne : 0;
  }
  if (B.h_step) memset(B.h_step, 0, (ne + 1) * 8);
  uint32_t* order = (uint32_t*)malloc(ne * 4 + 4);
  if (!B.h_off || !B.h_cnt || !B.h_step || !order) { free(order); clear_events(h); return fail(h, GCORECCD_ERR_NOMEM, "load_events: host memory"); }
  uint64_t left_events = 0;
  for (size_t k = 0; k < ne; ++k) {
    B.h_off[k] = (uint32_t)offsets[k];
    B.h_cnt[k] = (uint32_t)(offsets[k + 1] - offsets[k]);
    if (B.h_cnt[k]) left_events += 1;
  }
  B.h_off[ne] = (uint32_t)n;
  e = cudaMemcpyAsync(B.d_off, B.h_off, (ne + 1) * 4, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(B.d_cnt, B.h_cnt, ne * 4, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(B.d_step, 0, ne * 8, h->stream);
  if (e == cudaSuccess && n) {
    k_unpack_events<<<tiles_for(n), kTPB, 0, h->stream>>>(src, (uint32_t)n, h->A, (uint32_t)h->n_loaded);
    h->launches += 1;
    e = cudaGetLastError();
  }
  const uint64_t total_loaded = h->n_loaded + n;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h->ctrl->n_loaded, &total_loaded, 8, cudaMemcpyHostToDevice, h->stream);
  // scheduling hint: mean depth per event (d_order doubles as the float scratch until the order is uploaded)
  float* zmean = (float*)malloc(ne * 4 + 4);
  if (!zmean) { free(order); clear_events(h); return fail(h, GCORECCD_ERR_NOMEM, "load_events: host memory"); }
  if (e == cudaSuccess) {
    k_event_depth<<<(unsigned)((ne * 32 + kTPB - 1) / kTPB), kTPB, 0, h->stream>>>(h->A, B.d_off, B.d_cnt, (uint32_t)ne, (float*)B.d_order);
    h->launches += 1;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(zmean, B.d_order, ne * 4, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) { free(order); free(zmean); clear_events(h); return fail(h, GCORECCD_ERR_CUDA, "load_events", e); }
  // one queue per tier (kernel variant), each in longest-processing-time-first order
  // estimated work of an event = n^2 x steps, steps ~ the low-field drift time from its mean depth,
  // ln(a2 / (a2 - a1 z)) (eq. 1 with constant mobility); plain z where that is undefined.  Order only: never physics.
  const uint32_t* cnt = B.h_cnt;
  const double a1u = h->dp.a1_um, a2 = h->dp.a2;
  const bool lin = (h->dp.flags & GCORECCD_DEPLETION_OFF) || !(a1u > 0.0) || !(a2 > 0.0);
  for (size_t k = 0; k < ne; ++k) {
    const double z = zmean[k] > 0.f ? (double)zmean[k] : 0.0;
    const double r = lin ? 0.0 : std::min(a1u * z / a2, 0.98);
    const double steps = lin ? z : -std::log1p(-r);
    zmean[k] = (float)((double)cnt[k] * (double)cnt[k] * (steps + 1e-3));
  }
  const float* cost = zmean;
  auto by_size = [cost](uint32_t a, uint32_t b) { return cost[a] != cost[b] ? cost[a] > cost[b] : a < b; };
  uint32_t filled = 0;
  for (int q = 0; q < kEvTiers; ++q) {
    const uint32_t first = filled;
    for (size_t k = 0; k < ne; ++k)
      if ((q == 0 ? true : B.h_cnt[k] > kEvTierCap[q - 1]) && B.h_cnt[k] <= kEvTierCap[q]) order[filled++] = (uint32_t)k;
    if (q > 0) std::sort(order + first, order + filled, by_size);
    else if (filled > first) {
      // <= 32-hole events come in tens of thousands: a 64-bucket counting sort by estimated work (O(n)) keeps the
      // deep events in front without the 5 ms a comparison sort of 44k events costs on the host
      float cmax = 0.f;
      for (uint32_t k = first; k < filled; ++k) cmax = std::max(cmax, cost[order[k]]);
      const float sc = cmax > 0.f ? 63.999f / cmax : 0.f;
      uint32_t start[65] = {0};
      std::vector<uint32_t> tmp(order + first, order + filled);
      for (uint32_t v : tmp) start[64 - (uint32_t)(cost[v] * sc)] += 1;          // bucket b = 63 - level, counts at b + 1
      for (int b = 1; b <= 64; ++b) start[b] += start[b - 1];
      for (uint32_t v : tmp) order[first + start[63 - (uint32_t)(cost[v] * sc)]++] = v;
    }
    B.n_q[q] = filled - first;
  }
  free(zmean);
  e = cudaMemcpyAsync(B.d_order, order, ne * 4, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  free(order);
  if (e != cudaSuccess) { clear_events(h); return fail(h, GCORECCD_ERR_CUDA, "load_events", e); }

  // persistent grids (resident CTAs per SM x SM count), side streams and events: once per handle
  if (!B.fork) {
    int occ[kEvTiers] = {0};
    e = cudaFuncSetAttribute(k_events<4, 256, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)event_smem_bytes(kEvCapLarge));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_events<2, 256, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)event_smem_bytes(768u));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_events_cluster<4, 256, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)event_smem_bytes(kEvCapLarge));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_events_cluster<4, 256, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)event_smem_bytes(kEvCapLarge));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[0], k_events_warp, kEvTierThreads[0], 0);
    for (int q = 1; q < kEvTiers && e == cudaSuccess; ++q)
      e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ[q], ev_kernel(q), kEvTierThreads[q], event_smem_bytes(kEvTierCap[q]));
    if (e != cudaSuccess) { clear_events(h); return fail(h, GCORECCD_ERR_CUDA, "load_events: kernel attributes", e); }
    for (int q = 0; q < kEvTiers; ++q) B.grid_q[q] = h->num_sms * (occ[q] > 0 ? occ[q] : 1);
    for (int k = 0; k < kEvTiers - 1 && e == cudaSuccess; ++k) {
      e = cudaStreamCreateWithFlags(&B.aux[k], cudaStreamNonBlocking);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&B.join[k], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&B.fork, cudaEventDisableTiming);
    if (e != cudaSuccess) { free_events(h); return fail(h, GCORECCD_ERR_CUDA, "load_events: streams", e); }
  }
  B.loaded = true;
  B.n_events = n_events; B.n_carriers = n;
  B.events_left = left_events; B.carriers_left = n;
  h->n_loaded = total_loaded;
  return GCORECCD_OK;
}

int gcoreccd_run_events(gcoreccd_t* h, uint64_t max_steps, uint64_t* events_left, uint64_t* carriers_left) {
  if (!h) return GCORECCD_ERR_INVALID;
  auto& B = h->evb;
  if (!B.loaded) return fail(h, GCORECCD_ERR_STATE, "run_events: no batch loaded");
  Range r_ev("gcoreccd: run_events");
  DeviceGuard guard(h->device);
  int ret = GCORECCD_OK;
  if (B.carriers_left > 0) {
    const EventTable tab{B.d_off, B.d_cnt, B.d_step};
    GC_CUDA(h, cudaMemsetAsync(B.d_queue, 0, 4 * kEvTiers, h->stream));
    // one kernel per tier, the largest on the handle's stream, the others forked onto side streams so that the small
    // events fill the SMs the large ones leave
    uint32_t first[kEvTiers];
    first[0] = 0;
    for (int q = 1; q < kEvTiers; ++q) first[q] = first[q - 1] + B.n_q[q - 1];
    GC_CUDA(h, cudaEventRecord(B.fork, h->stream));
    for (int q = kEvTiers - 1; q >= 0; --q) {
      if (!B.n_q[q]) continue;
      const bool side = q < kEvTiers - 1;
      cudaStream_t st = side ? B.aux[q] : h->stream;
      if (side) GC_CUDA(h, cudaStreamWaitEvent(st, B.fork, 0));
      if (q == 0) {                                           // one warp per event, four events per CTA
        const int g = (int)std::min<uint32_t>((B.n_q[0] + 3u) / 4u, (uint32_t)B.grid_q[0]);
        k_events_warp<<<g, kEvTierThreads[0], 0, st>>>(h->A, tab, B.d_order, B.n_q[0], B.d_queue, h->ctrl, h->sink, h->dp, max_steps);
      } else if (q == kEvTiers - 1 && B.n_q[q] <= kEvClusterFewFactor * (uint32_t)h->num_sms) {
        // few large events: a cluster of 2 CTAs per event, 4 when there are not even enough events for that
        // (gc_events.cuh: k_events_cluster)
        const uint32_t cl = (B.n_q[q] * 2u <= (uint32_t)h->num_sms) ? 4u : 2u;
        const uint32_t clusters = std::min<uint32_t>(B.n_q[q], (uint32_t)h->num_sms / cl);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(clusters * cl); cfg.blockDim = dim3(256);
        cfg.dynamicSmemBytes = event_smem_bytes(kEvCapLarge); cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        if (cl == 4)
          GC_CUDA(h, cudaLaunchKernelEx(&cfg, k_events_cluster<4, 256, 4>, h->A, tab, (const uint32_t*)(B.d_order + first[q]), B.n_q[q],
                                        B.d_queue + q, h->ctrl, h->sink, h->dp, max_steps, kEvCapLarge));
        else
          GC_CUDA(h, cudaLaunchKernelEx(&cfg, k_events_cluster<4, 256, 2>, h->A, tab, (const uint32_t*)(B.d_order + first[q]), B.n_q[q],
                                        B.d_queue + q, h->ctrl, h->sink, h->dp, max_steps, kEvCapLarge));
      } else {
        const int g = (int)std::min<uint32_t>(B.n_q[q], (uint32_t)B.grid_q[q]);
        ev_kernel(q)<<<g, kEvTierThreads[q], event_smem_bytes(kEvTierCap[q]), st>>>(h->A, tab, B.d_order + first[q], B.n_q[q], B.d_queue + q,
                                                                                     h->ctrl, h->sink, h->dp, max_steps, kEvTierCap[q]);
      }
      h->launches += 1;
      if (side) {
        GC_CUDA(h, cudaEventRecord(B.join[q], st));
        GC_CUDA(h, cudaStreamWaitEvent(h->stream, B.join[q], 0));
      }
    }
    GC_CUDA(h, cudaGetLastError());
    GC_CUDA(h, cudaMemcpyAsync(B.h_cnt, B.d_cnt, B.n_events * 4, cudaMemcpyDeviceToHost, h->stream));
    GC_CUDA(h, cudaMemcpyAsync(B.h_step, B.d_step, B.n_events * 8, cudaMemcpyDeviceToHost, h->stream));
    int rc = sync_ctrl(h);
    if (rc) return rc;
    uint64_t el = 0, cl = 0;
    for (uint64_t k = 0; k < B.n_events; ++k) { if (B.h_cnt[k]) el += 1; cl += B.h_cnt[k]; }
    B.events_left = el; B.carriers_left = cl;
    h->n_bound = 0;
    if (h->h_ctrl->nonfinite) return fail(h, GCORECCD_ERR_NONFINITE, "a carrier position became non-finite");
  }
  if (B.carriers_left > 0) ret = GCORECCD_MAX_STEPS;
  if (events_left) *events_left = B.events_left;
  if (carriers_left) *carriers_left = B.carriers_left;
  return ret;
}

int gcoreccd_get_events(gcoreccd_t* h, uint64_t* n_active, uint64_t* step, uint64_t cap_events, uint64_t* n_events) {
  if (!h) return GCORECCD_ERR_INVALID;
  const auto& B = h->evb;
  if (!B.loaded) return fail(h, GCORECCD_ERR_STATE, "get_events: no batch loaded");
  if (n_events) *n_events = B.n_events;
  if ((n_active || step) && cap_events < B.n_events) return fail(h, GCORECCD_ERR_CAPACITY, "get_events: buffer too small");
  for (uint64_t k = 0; k < B.n_events; ++k) {
    if (n_active) n_active[k] = B.h_cnt[k];
    if (step) step[k] = B.h_step[k];
  }
  return GCORECCD_OK;
}

int gcoreccd_read_event_carriers(gcoreccd_t* h, uint64_t event, float* xyz, uint32_t* id, uint64_t cap, uint64_t* n) {
  if (!h) return GCORECCD_ERR_INVALID;
  const auto& B = h->evb;
  if (!B.loaded) return fail(h, GCORECCD_ERR_STATE, "read_event_carriers: no batch loaded");
  if (event >= B.n_events) return fail(h, GCORECCD_ERR_INVALID, "read_event_carriers: no such event");
  const uint32_t cnt = B.h_cnt[event], off = B.h_off[event];
  if (n) *n = cnt;
  if ((xyz || id) && cap < cnt) return fail(h, GCORECCD_ERR_CAPACITY, "read_event_carriers: buffer too small");
  if (cnt == 0 || (!xyz && !id)) return GCORECCD_OK;
  DeviceGuard guard(h->device);
  if (xyz) {
    k_interleave_range<<<tiles_for(cnt), kTPB, 0, h->stream>>>(h->A, off, cnt, h->Ep);
    h->launches += 1;
    GC_CUDA(h, cudaMemcpyAsync(xyz, h->Ep, (size_t)cnt * 12, cudaMemcpyDeviceToHost, h->stream));
  }
  if (id) GC_CUDA(h, cudaMemcpyAsync(id, h->A.id + off, (size_t)cnt * 4, cudaMemcpyDeviceToHost, h->stream));
  GC_CUDA(h, cudaGetLastError());
  GC_CUDA(h, cudaStreamSynchronize(h->stream));
  return GCORECCD_OK;
}

// ---------------------------------------------------------------------------- workload front end
uint64_t gcoreccd_xray_hole_count(double E_e_eV, double w_eV) {
  if (!(E_e_eV > 0.0) || !(w_eV > 0.0)) return 0;
  const double q = std::floor(E_e_eV / w_eV);
  return q >= 1.8e19 ? 0 : (uint64_t)q;
}

int gcoreccd_generate_cloud(gcoreccd_t* h, uint64_t n, const double* c, double sigma, uint64_t gen_seed, uint64_t first_index) {
  if (!h || !c) return GCORECCD_ERR_INVALID;
  if (n == 0) return GCORECCD_OK;
  if (!(sigma >= 0.0) || !std::isfinite(sigma) || !std::isfinite(c[0]) || !std::isfinite(c[1]) || !std::isfinite(c[2]) ||
      c[2] > h->p.thickness_um)
    return fail(h, GCORECCD_ERR_INVALID, "generate_cloud: sigma must be >= 0 and the centre finite and inside the slab");
  if (n > h->p.max_carriers) return fail(h, GCORECCD_ERR_CAPACITY, "generate_cloud: capacity");
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "generate_cloud: a batch of events is still drifting");
  DeviceGuard guard(h->device);
  k_gen_cloud<<<tiles_for(n), kTPB, 0, h->stream>>>(h->Ep, (uint32_t)n, first_index, c[0], c[1], c[2], sigma, h->dp.thickness,
                                                   (uint32_t)(gen_seed & 0xffffffffu), (uint32_t)(gen_seed >> 32));
  h->launches += 1;
  GC_CUDA(h, cudaGetLastError());
  return gcoreccd_load_carriers(h, h->Ep, n, 1);          // the partial-sum buffer is scratch between steps
}

int gcoreccd_generate_xray_events(gcoreccd_t* h, uint64_t n_events, const double* E, const double* centre, const double* sigma,
                                  double w_eV, uint64_t gen_seed, uint64_t first_index, uint64_t* counts_out) {
  if (!h || !E || !centre || !sigma || n_events == 0 || n_events > 0x7fffffffull || !(w_eV > 0.0)) return GCORECCD_ERR_INVALID;
  std::vector<uint64_t> off(n_events + 1);
  std::vector<uint32_t> off32(n_events + 1);
  off[0] = 0; off32[0] = 0;
  for (uint64_t e = 0; e < n_events; ++e) {
    if (!(sigma[e] >= 0.0) || !std::isfinite(sigma[e]) || !std::isfinite(centre[3 * e]) || !std::isfinite(centre[3 * e + 1]) ||
        !std::isfinite(centre[3 * e + 2]) || centre[3 * e + 2] > h->p.thickness_um || !std::isfinite(E[e]))
      return fail(h, GCORECCD_ERR_INVALID, "generate_xray_events: non-finite input, negative sigma or centre above the back surface");
    const uint64_t cnt = gcoreccd_xray_hole_count(E[e], w_eV);
    if (cnt > GCORECCD_EVENT_MAX_CARRIERS) return fail(h, GCORECCD_ERR_CAPACITY, "generate_xray_events: an event exceeds GCORECCD_EVENT_MAX_CARRIERS");
    off[e + 1] = off[e] + cnt;
    if (off[e + 1] > h->p.max_carriers) return fail(h, GCORECCD_ERR_CAPACITY, "generate_xray_events: capacity");
    off32[e + 1] = (uint32_t)off[e + 1];
    if (counts_out) counts_out[e] = cnt;
  }
  if (events_busy(h)) return fail(h, GCORECCD_ERR_STATE, "generate_xray_events: the previous batch is still drifting");
  const uint64_t n = off[n_events];
  DeviceGuard guard(h->device);
  if (n) {
    char* buf = nullptr;
    const size_t b_off = align_up((n_events + 1) * 4, 256), b_c = align_up(n_events * 24, 256), b_s = align_up(n_events * 8, 256);
    cudaError_t e = cudaMalloc((void**)&buf, b_off + b_c + b_s);
    if (e != cudaSuccess) return fail(h, e == cudaErrorMemoryAllocation ? GCORECCD_ERR_NOMEM : GCORECCD_ERR_CUDA, "generate_xray_events: cudaMalloc", e);
    uint32_t* d_off = (uint32_t*)buf;
    double* d_c = (double*)(buf + b_off);
    double* d_s = (double*)(buf + b_off + b_c);
    e = cudaMemcpyAsync(d_off, off32.data(), (n_events + 1) * 4, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_c, centre, n_events * 24, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_s, sigma, n_events * 8, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
      k_gen_events<<<tiles_for(n), kTPB, 0, h->stream>>>(h->Ep, (uint32_t)n, d_off, (uint32_t)n_events, d_c, d_s, first_index,
                                                        h->dp.thickness, (uint32_t)(gen_seed & 0xffffffffu), (uint32_t)(gen_seed >> 32));
      h->launches += 1;
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(buf);
    if (e != cudaSuccess) return fail(h, GCORECCD_ERR_CUDA, "generate_xray_events", e);
  }
  return gcoreccd_load_events(h, h->Ep, off.data(), n_events, 1);
}

int gcoreccd_load_carriers_file(gcoreccd_t* h, const char* path, uint64_t* n_read) {
  if (!h || !path) return GCORECCD_ERR_INVALID;
  FILE* f = fopen(path, "r");
  if (!f) return fail(h, GCORECCD_ERR_INVALID, "load_carriers_file: cannot open the file");
  std::vector<float> xyz;
  char line[512];
  bool bad = false;
  while (fgets(line, sizeof(line), f)) {
    char* s = line;
    while (*s == ' ' || *s == '\t') ++s;
    if (*s == '#' || *s == '\n' || *s == '\r' || *s == 0) continue;
    float v[3];
    int got = 0;
    while (got < 3) {
      char* end = nullptr;
      v[got] = strtof(s, &end);
      if (end == s) break;
      ++got;
      s = end;
      while (*s == ' ' || *s == '\t' || *s == ',' || *s == ';') ++s;
    }
    if (got != 3 || !(*s == 0 || *s == '\n' || *s == '\r' || *s == '#')) { bad = true; break; }
    xyz.push_back(v[0]); xyz.push_back(v[1]); xyz.push_back(v[2]);
  }
  fclose(f);
  if (bad) return fail(h, GCORECCD_ERR_INVALID, "load_carriers_file: malformed line (expected x y z)");
  if (n_read) *n_read = xyz.size() / 3;
  if (xyz.empty()) return GCORECCD_OK;
  return gcoreccd_load_carriers(h, xyz.data(), xyz.size() / 3, 0);
}

int gcoreccd_save_collected_file(gcoreccd_t* h, const char* path, uint64_t* n_written) {
  if (!h || !path) return GCORECCD_ERR_INVALID;
  uint64_t m = 0;
  int rc = gcoreccd_read_collected(h, nullptr, nullptr, 0, &m);
  if (rc) return rc;
  std::vector<float> xyz(3 * m + 3);
  std::vector<uint32_t> st(m + 1);
  if (m) { rc = gcoreccd_read_collected(h, xyz.data(), st.data(), m, &m); if (rc) return rc; }
  FILE* f = fopen(path, "w");
  if (!f) return fail(h, GCORECCD_ERR_INVALID, "save_collected_file: cannot open the file");
  fprintf(f, "# id x_um y_um z_um step   (holes collected at z <= z_well; PAPER.md:122 output positions)\n");
  uint64_t w = 0;
  for (uint64_t k = 0; k < m; ++k) {
    if (st[k] == 0xffffffffu) continue;                    // still drifting
    fprintf(f, "%llu %.9g %.9g %.9g %u\n", (unsigned long long)k, xyz[3 * k], xyz[3 * k + 1], xyz[3 * k + 2], st[k]);
    ++w;
  }
  const bool ok = fclose(f) == 0;
  if (n_written) *n_written = w;
  return ok ? GCORECCD_OK : fail(h, GCORECCD_ERR_INVALID, "save_collected_file: write failed");
}

int gcoreccd_debug_microbench(int kind, uint32_t iters, uint32_t warps_per_subpartition, double* cycles_per_inst) {
  if (kind < 0 || kind >= kMicroKinds || iters == 0 || warps_per_subpartition < 1 || warps_per_subpartition > 4 || !cycles_per_inst)
    return GCORECCD_ERR_INVALID;
  const int threads = 128 * (int)warps_per_subpartition;      // 4 sub-partitions x 32 lanes x warps
  long long* d_cyc = nullptr;
  float* d_sink = nullptr;
  if (cudaMalloc((void**)&d_cyc, 16 * sizeof(long long)) != cudaSuccess) return GCORECCD_ERR_NOMEM;
  if (cudaMalloc((void**)&d_sink, 4) != cudaSuccess) { cudaFree(d_cyc); return GCORECCD_ERR_NOMEM; }
  for (int rep = 0; rep < 2; ++rep) {                           // first launch warms the instruction cache
    switch (kind) {
      case 0: k_microbench<0><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 1: k_microbench<1><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 2: k_microbench<2><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 3: k_microbench<3><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 4: k_microbench<4><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 5: k_microbench<5><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 6: k_microbench<6><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 7: k_microbench<7><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 8: k_microbench<8><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 9: k_microbench<9><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 10: k_microbench<10><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 11: k_microbench<11><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 12: k_microbench<12><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 13: k_microbench<13><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 14: k_microbench<14><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      case 15: k_microbench<15><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
      default: k_microbench<16><<<1, threads>>>(iters, 1.0f, d_cyc, d_sink); break;
    }
  }
  long long h_cyc[16];
  cudaError_t e = cudaMemcpy(h_cyc, d_cyc, sizeof(h_cyc), cudaMemcpyDeviceToHost);
  cudaFree(d_cyc); cudaFree(d_sink);
  if (e != cudaSuccess) return GCORECCD_ERR_CUDA;
  long long worst = 0;
  for (int w = 0; w < threads / 32; ++w) worst = std::max(worst, h_cyc[w]);
  *cycles_per_inst = (double)worst / ((double)iters * micro_inst_per_iter(kind) * (double)warps_per_subpartition);
  return GCORECCD_OK;
}

#ifdef GC_TIMING
int gcoreccd_debug_timing(long long* out) {      // development builds only (-DGC_TIMING): phase timestamps of k_steps
  return cudaMemcpyFromSymbol(out, gc::g_dbg, sizeof(gc::g_dbg)) == cudaSuccess ? 0 : -5;
}
int gcoreccd_debug_probes(long long* out) {
  return cudaMemcpyFromSymbol(out, gc::g_pp, sizeof(gc::g_pp)) == cudaSuccess ? 0 : -5;
}
int gcoreccd_debug_gtimes(unsigned long long* out) {
  return cudaMemcpyFromSymbol(out, gc::g_gt, sizeof(gc::g_gt)) == cudaSuccess ? 0 : -5;
}
#endif

// ---- allocation-free field evaluation (gc_noalloc.cuh) -----------------------------------------------------------
}  // extern "C"

// The scratch of gcoreccd_field_noalloc: a file-scope device array, part of the library's image on every GPU that loads
// it (6.2 MiB until the process exits).  In host code this name is only a stand-in for the symbol: the device address
// comes from cudaGetSymbolAddress, once per device, below.
static __device__ __align__(256) unsigned char g_na_scratch[gc::NaLayout::bytes];

namespace {
struct NaDevice { bool ready; unsigned char* base; int sms; };
NaDevice g_na_dev[64];
std::mutex g_na_mu;
thread_local char g_na_err[256] = "";

int na_fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_na_err, sizeof(g_na_err), fmt, ap);
  va_end(ap);
  return code;
}

// once per device, with that device current: the array's address ON THIS DEVICE, and the SM count for the grids
int na_setup(int dev, NaDevice** out) {
  if (dev < 0 || dev >= 64) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_na_mu);
  NaDevice& D = g_na_dev[dev];
  if (!D.ready) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    if (major != 10) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: device %d is not sm_100 (no fallback)", dev);
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_na_scratch);
    if (e != cudaSuccess || !ptr) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    D.base = (unsigned char*)ptr;
    D.sms = sms;
    D.ready = true;
  }
  *out = &D;
  return GCORECCD_OK;
}
}  // namespace

extern "C" {

int gcoreccd_field_noalloc(const float* xyz_um_dev, uint64_t n, double softening_um, double eps_si, float* Exyz_dev,
                           void* stream) {
  g_na_err[0] = 0;
  if (n > GCORECCD_NOALLOC_MAX_CARRIERS)
    return na_fail(GCORECCD_ERR_CAPACITY, "field_noalloc: n = %llu exceeds GCORECCD_NOALLOC_MAX_CARRIERS = %u (fixed scratch)",
                   (unsigned long long)n, (unsigned)GCORECCD_NOALLOC_MAX_CARRIERS);
  if (n == 0) return GCORECCD_OK;
  if (!xyz_um_dev || !Exyz_dev) return na_fail(GCORECCD_ERR_INVALID, "field_noalloc: null input or output pointer");
  if (!(softening_um >= 0.0) || !(eps_si >= 0.0) || !std::isfinite(softening_um) || !std::isfinite(eps_si))
    return na_fail(GCORECCD_ERR_INVALID, "field_noalloc: softening and eps_si must be finite and >= 0");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
  NaDevice* D = nullptr;
  int rc = na_setup(dev, &D);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Ctrl* ctrl = (Ctrl*)(D->base + NaLayout::ctrl);
  float* x = (float*)(D->base + NaLayout::x);
  float* y = (float*)(D->base + NaLayout::y);
  float* z = (float*)(D->base + NaLayout::z);
  float* Ep = (float*)(D->base + NaLayout::ep);
  // same constants as gcoreccd_create (K' = q / (4 pi eps0 eps_Si) in (V/cm) um^2; R5: eps^2 >= 1e-24)
  const double q = 1.602176634e-19, eps0 = 8.8541878128e-12, pi = 3.14159265358979323846;
  const double Kp = q / (4.0 * pi * eps0 * (eps_si > 0.0 ? eps_si : 11.7)) * 1e10;
  const double e2 = softening_um * softening_um;
  const float eps2 = (float)(e2 < 1e-24 ? 1e-24 : e2);
  // field variant by size, as the handle's two-launch path picks it (pick_variant)
  const int npack = n >= 12288 ? 4 : n >= 3072 ? 2 : 1;
  const int per_sm = npack == 4 ? 1 : npack == 2 ? 3 : 4;
  PlanArgs pa;
  pa.IB = (uint32_t)kTPB * 2u * (uint32_t)npack;
  pa.grid = (uint32_t)(D->sms * per_sm);
  pa.part_cap_entries = kNaPartCap;
  pa.rank = 0; pa.world = 1; pa.force_S = 0;
  const uint32_t tiles = (uint32_t)((n + kTPB - 1) / kTPB);
  k_na_prepare<<<1, 32, 0, st>>>(ctrl, (uint32_t)n, pa);
  k_na_unpack<<<tiles, kTPB, 0, st>>>(xyz_um_dev, (uint32_t)n, x, y, z);
  switch (npack) {
    case 1: k_field<1, 256, 4><<<pa.grid, kTPB, 0, st>>>(x, y, z, ctrl, Ep, kNaPartCap, eps2); break;
    case 2: k_field<2, 256, 3><<<pa.grid, kTPB, 0, st>>>(x, y, z, ctrl, Ep, kNaPartCap, eps2); break;
    default: k_field<4, 256, 1><<<pa.grid, kTPB, 0, st>>>(x, y, z, ctrl, Ep, kNaPartCap, eps2); break;
  }
  k_field_finalize<<<tiles, kTPB, 0, st>>>(ctrl, Ep, kNaPartCap, Kp, Exyz_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(GCORECCD_ERR_CUDA, "field_noalloc: kernel launch: %s", cudaGetErrorString(e));
  return GCORECCD_OK;
}

const char* gcoreccd_field_noalloc_error(void) { return g_na_err; }

const char* gcoreccd_strerror(int code) {
  switch (code) {
    case GCORECCD_OK: return "ok";
    case GCORECCD_MAX_STEPS: return "max_steps reached with carriers still drifting";
    case GCORECCD_ERR_INVALID: return "invalid argument";
    case GCORECCD_ERR_STATE: return "bad state";
    case GCORECCD_ERR_CAPACITY: return "capacity exceeded";
    case GCORECCD_ERR_NOMEM: return "out of memory";
    case GCORECCD_ERR_CUDA: return "CUDA error or no sm_100 device";
    case GCORECCD_ERR_NONFINITE: return "non-finite carrier state";
    default: return "unknown";
  }
}

const char* gcoreccd_last_error(gcoreccd_t* h) { return h ? h->err : ""; }

const char* gcoreccd_version(void) { return "gcoreccd-b200 0.1 (sm_100a)"; }

}  // extern "C"
