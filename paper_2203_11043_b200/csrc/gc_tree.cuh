// gc_tree.cuh — far-field approximation of eq. 6 (second half; "O(N^2)", 92).
// A VARIANT, off by default and reported separately from the exact all-pairs metric: gcoreccd_set_farfield(theta).
//
// Method (a GPU treecode over an implicit tree; nothing of it is in the paper, whose kernel is all-pairs):
//   1. every `resort` steps the active carriers are reordered along a 48-bit Hilbert curve of their bounding box
//      (LSD radix sort written here: block histograms, one scan, stable warp-match scatter; no Thrust/CUB);
//   2. every step an implicit 8-ary tree is laid over that order: the level-l node k is the run of 8*8^l consecutive
//      carriers starting at k*8*8^l; a node stores its hole count m, its centre of charge c (the dipole about c
//      vanishes) and the radius a of the smallest ball about c holding its members (computed from the CURRENT
//      positions, so the nodes stay valid between re-sorts, only less compact);
//   3. every 256 consecutive targets (a "group") walk the tree level by level from the lowest level with <= 64 nodes: a
//      node is ACCEPTED when  a <= theta * |x_t - c|  for EVERY target t of the group (decided exactly, through boxes of
//      256 / 32 / 8 targets and then the targets themselves: tree_accept) and enters the group's far list as one
//      pseudo-hole of charge m at c; otherwise it is opened (it joins the frontier whose children are the next level's
//      candidates) or, at the leaf level, its 8 holes enter the near list and are summed exactly;
//   4. the lists are consumed by the same packed FP32x2 inner loop as k_field (weighted by m for pseudo-holes).
//
// Error bound (stated, and checked against the FP64 oracle in tests/test_gpu_farfield.py): for one accepted node,
// expanding grad(1/|x - s|) about c, the monopole term is kept, the dipole terms cancel in the sum over the node,
// and the rest is bounded by  (m K'/d^2) * sum_{k>=2} (k+1) (a/d)^k  =  (m K'/d^2) * t^2 (3 - 2t)/(1 - t)^2, t = a/d
// <= theta.  Hence  |E_approx - E_exact|_j  <=  B(theta) * sum_{accepted nodes} m K'/d_j^2  <=  B(theta) * sum_i
// K'/|r_ij|^2-like field-magnitude sum (the sum of the MAGNITUDES of the far pair fields, not of the net field),
// B(theta) = theta^2 (3 - 2 theta)/(1 - theta)^2.  Softening (eps = 1e-3 um) enters at relative order eps^2/d^2.
// The near field is exact.  theta = 0 accepts nothing: the result is the exact sum in a different order.
#pragma once
#include "gc_common.cuh"
#include "gc_field.cuh"

namespace gc {

constexpr uint32_t kLeaf = 8;              // carriers per level-0 node (32 and 16 measured slower: more exact near field)
constexpr uint32_t kFan = 8;               // children per node
constexpr uint32_t kTreeMaxLevels = 9;     // 8 * 8^8 = 2^27 > 2^26
constexpr uint32_t kGroup = 256;           // targets per traversal group = one level-1 node
constexpr int kTreeTPB = 128;              // threads of k_tree_field: one packed pair of targets each
constexpr uint32_t kFarCap = 1024, kNearCap = 768, kFrontCap = 2048;
constexpr int kCPT = 2;                    // candidates per thread and batch of the walk
constexpr uint32_t kBatch = kCPT * kTreeTPB;
constexpr uint32_t kTopNodes = 64;         // the walk starts at the lowest level with at most this many nodes
constexpr uint32_t kSortBlock = 2048;      // keys per block of the radix passes (256 threads x 8)

struct TreeCtrl {                          // device resident, next to the tree arrays
  uint32_t lo[3], hi[3];                   // bounding box, order-preserving integer images of the floats
  uint32_t next_group;                     // dynamic work counter of k_tree_field
  uint32_t pad_;
  unsigned long long far_evals, near_evals;  // interactions actually evaluated (pseudo-hole and exact)
  uint32_t tot[6][256];                    // radix sort: global digit totals of each pass (order-independent)
};

struct Tree {                              // device pointers carved from the workspace
  TreeCtrl* tc;
  float4* node_c;                          // (cx, cy, cz, m), all levels concatenated, level 0 first
  float* node_r;
  unsigned long long* key[2];              // radix sort double buffers: 48-bit curve keys ...
  uint32_t* val[2];                        // ... and the carrier index they came from
  uint32_t* counts;                        // [blocks][256] digit histograms
};

__host__ __device__ inline uint32_t level_size(uint32_t l) { return kLeaf << (3u * l); }
__host__ __device__ inline uint32_t nodes_at(uint32_t n, uint32_t l) {
  const uint64_t s = (uint64_t)kLeaf << (3u * l);
  return (uint32_t)(((uint64_t)n + s - 1) / s);
}
__host__ __device__ inline uint32_t level_offset(uint32_t n, uint32_t l) {
  uint32_t o = 0;
  for (uint32_t k = 0; k < l; ++k) o += nodes_at(n, k);
  return o;
}

__device__ __forceinline__ uint32_t f2ord(float f) {
  const uint32_t b = __float_as_uint(f);
  return b ^ ((b >> 31) ? 0xffffffffu : 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t o) {
  return __uint_as_float(o ^ ((o >> 31) ? 0x80000000u : 0xffffffffu));
}

__global__ void k_tree_reset(TreeCtrl* __restrict__ tc, int reset_box) {
  if (threadIdx.x == 0) {
    tc->next_group = 0;
    if (reset_box) {
      for (int c = 0; c < 3; ++c) { tc->lo[c] = 0xffffffffu; tc->hi[c] = 0u; }
    }
  }
  if (reset_box)                                            // a re-sort follows: clear the digit totals
    for (uint32_t k = threadIdx.x; k < 6u * 256u; k += blockDim.x) (&tc->tot[0][0])[k] = 0u;
}

__global__ void __launch_bounds__(kTPB)
k_tree_bbox(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
            const Ctrl* __restrict__ ctrl, TreeCtrl* __restrict__ tc) {
  const uint32_t n = ctrl->n_active;
  uint32_t lo[3] = {0xffffffffu, 0xffffffffu, 0xffffffffu}, hi[3] = {0u, 0u, 0u};
  for (uint32_t i = blockIdx.x * kTPB + threadIdx.x; i < n; i += gridDim.x * kTPB) {
    const uint32_t v[3] = {f2ord(px[i]), f2ord(py[i]), f2ord(pz[i])};
#pragma unroll
    for (int c = 0; c < 3; ++c) { lo[c] = min(lo[c], v[c]); hi[c] = max(hi[c], v[c]); }
  }
  __shared__ uint32_t s_lo[3][kTPB / 32], s_hi[3][kTPB / 32];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = __reduce_min_sync(0xffffffffu, lo[c]);
    hi[c] = __reduce_max_sync(0xffffffffu, hi[c]);
  }
  if ((threadIdx.x & 31u) == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) { s_lo[c][threadIdx.x >> 5] = lo[c]; s_hi[c][threadIdx.x >> 5] = hi[c]; }
  }
  __syncthreads();
  if (threadIdx.x < 3) {                                    // one atomic pair per coordinate and CTA, not per warp
    uint32_t a = s_lo[threadIdx.x][0], b = s_hi[threadIdx.x][0];
    for (int w = 1; w < kTPB / 32; ++w) { a = min(a, s_lo[threadIdx.x][w]); b = max(b, s_hi[threadIdx.x][w]); }
    atomicMin(&tc->lo[threadIdx.x], a); atomicMax(&tc->hi[threadIdx.x], b);
  }
}

constexpr uint32_t kKeyBits = 16;          // bits per axis: 65,536^3 cells (a 1,350 um track resolves to 0.02 um)
constexpr uint32_t kKeyPasses = 6;         // 48-bit keys, 8 bits per radix pass

__device__ __forceinline__ unsigned long long spread3(uint32_t v) {     // 16 bits -> every third bit of 48
  unsigned long long x = v & 0xffffull;
  x = (x | (x << 32)) & 0x001f00000000ffffull;
  x = (x | (x << 16)) & 0x001f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

// 48-bit space-filling-curve key on a cubic grid of 65,536^3 cells spanning the largest extent of the bounding box.
__global__ void __launch_bounds__(kTPB)
k_tree_keys(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
            const Ctrl* __restrict__ ctrl, const TreeCtrl* __restrict__ tc, unsigned long long* __restrict__ key,
            uint32_t* __restrict__ val) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  const float x0 = ord2f(tc->lo[0]), y0 = ord2f(tc->lo[1]), z0 = ord2f(tc->lo[2]);
  const float ext = fmaxf(fmaxf(ord2f(tc->hi[0]) - x0, ord2f(tc->hi[1]) - y0), fmaxf(ord2f(tc->hi[2]) - z0, 1e-30f));
  constexpr float kCells = (float)((1u << kKeyBits) - 1u);
  const float sc = kCells / ext;
  const uint32_t qx = (uint32_t)fminf(fmaxf((px[i] - x0) * sc, 0.f), kCells);
  const uint32_t qy = (uint32_t)fminf(fmaxf((py[i] - y0) * sc, 0.f), kCells);
  const uint32_t qz = (uint32_t)fminf(fmaxf((pz[i] - z0) * sc, 0.f), kCells);
  // Hilbert index of the cell (Skilling's axes-to-transpose transform, AIP Conf. Proc. 707, 2004): consecutive
  // indices are always face-adjacent cells, so a run of consecutive carriers is spatially compact — a Morton run
  // is not (it jumps at octant boundaries), and loose runs inflate the exact near field of step 3.
  uint32_t X0 = qx, X1 = qy, X2 = qz;
  for (uint32_t Q = 1u << (kKeyBits - 1); Q > 1u; Q >>= 1) {
    const uint32_t Pm = Q - 1u;
    if (X0 & Q) X0 ^= Pm;
    if (X1 & Q) X0 ^= Pm; else { const uint32_t t = (X0 ^ X1) & Pm; X0 ^= t; X1 ^= t; }
    if (X2 & Q) X0 ^= Pm; else { const uint32_t t = (X0 ^ X2) & Pm; X0 ^= t; X2 ^= t; }
  }
  X1 ^= X0; X2 ^= X1;
  uint32_t t = 0;
  for (uint32_t Q = 1u << (kKeyBits - 1); Q > 1u; Q >>= 1) if (X2 & Q) t ^= Q - 1u;
  X0 ^= t; X1 ^= t; X2 ^= t;
  key[i] = (spread3(X0) << 2) | (spread3(X1) << 1) | spread3(X2);
  val[i] = i;
}

// ---- LSD radix sort, 8 bits per pass, keys + values; stable ------------------------------------------------------
__global__ void __launch_bounds__(256)
k_radix_hist(const unsigned long long* __restrict__ key, const Ctrl* __restrict__ ctrl, uint32_t shift, uint32_t* __restrict__ counts,
             uint32_t* __restrict__ tot) {
  __shared__ uint32_t s_h[256];
  const uint32_t n = ctrl->n_active;
  const uint32_t nb = (n + kSortBlock - 1) / kSortBlock;
  if (blockIdx.x >= nb) return;
  s_h[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * kSortBlock;
  for (uint32_t k = threadIdx.x; k < kSortBlock; k += 256) {
    const uint32_t i = base + k;
    if (i < n) atomicAdd(&s_h[(uint32_t)(key[i] >> shift) & 255u], 1u);
  }
  __syncthreads();
  counts[blockIdx.x * 256u + threadIdx.x] = s_h[threadIdx.x];             // block-major: [block][digit]
  if (s_h[threadIdx.x]) atomicAdd(&tot[threadIdx.x], s_h[threadIdx.x]);      // integer: order-independent
}

__global__ void __launch_bounds__(256)
k_radix_scatter(const unsigned long long* __restrict__ key_in, const uint32_t* __restrict__ val_in, unsigned long long* __restrict__ key_out,
                uint32_t* __restrict__ val_out, const Ctrl* __restrict__ ctrl, uint32_t shift,
                const uint32_t* __restrict__ counts, const uint32_t* __restrict__ tot) {
  __shared__ uint32_t s_wh[8][256];       // per-warp digit counts of the current round
  __shared__ uint32_t s_run[256];         // digits already placed by this block
  const uint32_t n = ctrl->n_active;
  const uint32_t nb = (n + kSortBlock - 1) / kSortBlock;
  if (blockIdx.x >= nb) return;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  // where this block's keys of digit d go: (keys of smaller digits anywhere) + (keys of digit d in earlier blocks).
  // No separate scan kernel: the digit totals come from the histogram pass, the prefix over the earlier blocks is summed
  // here from the block-major count table.
  {
    const uint32_t v = tot[tid];
    uint32_t inc = v;
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (uint32_t)o) inc += t; }
    if (lane == 31) s_wh[0][warp] = inc;
    __syncthreads();
    uint32_t base = inc - v;
    for (uint32_t w = 0; w < warp; ++w) base += s_wh[0][w];
    __syncthreads();
    uint32_t a0 = 0, a1 = 0, a2 = 0, a3 = 0;                 // thread d sums digit d over the earlier blocks: coalesced
    uint32_t b = 0;                                         // across threads, independent loads along b
    for (; b + 4 <= blockIdx.x; b += 4) {
      a0 += counts[(b + 0) * 256u + tid]; a1 += counts[(b + 1) * 256u + tid];
      a2 += counts[(b + 2) * 256u + tid]; a3 += counts[(b + 3) * 256u + tid];
    }
    for (; b < blockIdx.x; ++b) a0 += counts[b * 256u + tid];
    s_run[tid] = base + a0 + a1 + a2 + a3;
    __syncthreads();
  }
  const uint32_t base = blockIdx.x * kSortBlock;
  for (uint32_t r = 0; r < kSortBlock / 256; ++r) {
    for (int w = 0; w < 8; ++w) s_wh[w][tid] = 0;
    __syncthreads();
    const uint32_t i = base + r * 256 + tid;
    const bool ok = i < n;
    const unsigned long long k = ok ? key_in[i] : 0ull;
    const uint32_t v = ok ? val_in[i] : 0u;
    const uint32_t d = ok ? ((uint32_t)(k >> shift) & 255u) : 256u + lane;          // invalid lanes match nobody
    const uint32_t m = __match_any_sync(0xffffffffu, d);
    const uint32_t rank = __popc(m & ((1u << lane) - 1u));
    if (ok && rank == 0) s_wh[warp][d] = __popc(m);
    __syncthreads();
    // exclusive prefix over the 8 warps for digit `tid`, plus the running base
    uint32_t acc = s_run[tid];
    for (int w = 0; w < 8; ++w) { const uint32_t c = s_wh[w][tid]; s_wh[w][tid] = acc; acc += c; }
    __syncthreads();
    if (ok) {
      const uint32_t pos = s_wh[warp][d] + rank;
      key_out[pos] = k; val_out[pos] = v;
    }
    __syncthreads();
    s_run[tid] = acc;
  }
}

// reorder the state along the sorted permutation: dst[i] = src[val[i]]
__global__ void __launch_bounds__(kTPB)
k_tree_permute(SoA src, SoA dst, const uint32_t* __restrict__ val, const Ctrl* __restrict__ ctrl) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  const uint32_t s = val[i];
  dst.x[i] = src.x[s]; dst.y[i] = src.y[s]; dst.z[i] = src.z[s]; dst.id[i] = src.id[s];
}
__global__ void __launch_bounds__(kTPB)
k_tree_copy(SoA src, SoA dst, const Ctrl* __restrict__ ctrl) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  dst.x[i] = src.x[i]; dst.y[i] = src.y[i]; dst.z[i] = src.z[i]; dst.id[i] = src.id[i];
}

// ---- nodes -------------------------------------------------------------------------------------------------------
// Level 0: kLeaf lanes per leaf: m, centre of charge, radius of the members about it.
__global__ void __launch_bounds__(kTPB)
k_tree_leaves(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
              const Ctrl* __restrict__ ctrl, float4* __restrict__ node_c, float* __restrict__ node_r) {
  const uint32_t n = ctrl->n_active;
  const uint32_t gt = blockIdx.x * kTPB + threadIdx.x;
  const uint32_t leaf = gt / kLeaf, sub = gt % kLeaf;
  const bool live = leaf < nodes_at(n, 0);                // whole warps stay for the shuffles
  const uint32_t i0 = live ? leaf * kLeaf : 0u;
  const uint32_t i = i0 + sub;
  const bool ok = live && i < n;
  const float x0 = live ? px[i0] : 0.f, y0 = live ? py[i0] : 0.f, z0 = live ? pz[i0] : 0.f;   // sums relative to the first member
  const float dx = ok ? px[i] - x0 : 0.f, dy = ok ? py[i] - y0 : 0.f, dz = ok ? pz[i] - z0 : 0.f;
  float sx = dx, sy = dy, sz = dz;
#pragma unroll
  for (int o = kLeaf / 2; o > 0; o >>= 1) {
    sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o); sz += __shfl_xor_sync(0xffffffffu, sz, o);
  }
  const uint32_t m = live ? min(kLeaf, n - i0) : 1u;
  const float inv = 1.0f / (float)m;
  const float cx = sx * inv, cy = sy * inv, cz = sz * inv;           // relative to (x0,y0,z0)
  float r2 = ok ? (dx - cx) * (dx - cx) + (dy - cy) * (dy - cy) + (dz - cz) * (dz - cz) : 0.f;
#pragma unroll
  for (int o = kLeaf / 2; o > 0; o >>= 1) r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, o));
  if (live && sub == 0) {
    node_c[leaf] = make_float4(x0 + cx, y0 + cy, z0 + cz, (float)m);
    // the stored centre is rounded to FP32 (<= 1 ulp per coordinate): widen the radius accordingly
    node_r[leaf] = sqrtf(r2) * 1.000001f + 2e-7f * (fabsf(x0) + fabsf(y0) + fabsf(z0));
  }
}

// Level of the walk's start: the lowest level with at most kTopNodes nodes.  Higher levels are never visited.
__host__ __device__ inline uint32_t top_level(uint32_t n) {
  uint32_t l = 0;
  while (l + 1 < kTreeMaxLevels && nodes_at(n, l) > kTopNodes) ++l;
  return l;
}

// Levels 1 .. top_level, straight from the leaves: centre = count-weighted mean of the leaves' centres (FP64),
// radius = max over leaves of |c_leaf - c| + r_leaf (a valid, slightly generous ball; tighter than nesting level by
// level).  TPN threads per node: a warp for levels [l_lo, l_hi] = [1, 2] (8 and 64 leaves), a CTA above.
template <int TPN>
__global__ void __launch_bounds__(kTPB)
k_tree_upper(const Ctrl* __restrict__ ctrl, float4* __restrict__ node_c, float* __restrict__ node_r, uint32_t l_lo,
             uint32_t l_hi) {
  constexpr int kWarps = TPN / 32;
  __shared__ double s_s[4][kTPB / 32];
  __shared__ float s_r[kTPB / 32];
  __shared__ float s_c[3];
  const uint32_t n = ctrl->n_active;
  const uint32_t ltop = top_level(n);
  if (l_hi > ltop) l_hi = ltop;
  // which (level, k) is this thread group?
  uint32_t b = (blockIdx.x * kTPB + threadIdx.x) / TPN, l = l_lo;
  bool live = false;
  for (; l <= l_hi; ++l) {
    const uint32_t c = nodes_at(n, l);
    if (b < c) { live = true; break; }
    b -= c;
  }
  if (TPN > 32 && !live) return;                             // whole CTA; warps of the TPN = 32 variant exit below
  if (TPN == 32 && !live) return;                            // whole warp
  const uint32_t per = 1u << (3u * l);                       // leaves per node at this level
  const uint32_t n_leaves = nodes_at(n, 0);
  const uint32_t f0 = b * per, f1 = min(f0 + per, n_leaves);
  const uint32_t tid = threadIdx.x % TPN, lane = threadIdx.x & 31u, warp = tid >> 5;
  const float4 ref = node_c[f0];
  double sx = 0, sy = 0, sz = 0, sm = 0;
  for (uint32_t f = f0 + tid; f < f1; f += TPN) {
    const float4 c = node_c[f];
    sx += (double)c.w * (double)(c.x - ref.x); sy += (double)c.w * (double)(c.y - ref.y); sz += (double)c.w * (double)(c.z - ref.z);
    sm += (double)c.w;
  }
  for (int o = 16; o > 0; o >>= 1) {
    sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o);
    sz += __shfl_xor_sync(0xffffffffu, sz, o); sm += __shfl_xor_sync(0xffffffffu, sm, o);
  }
  if (kWarps > 1) {
    if (lane == 0) { s_s[0][warp] = sx; s_s[1][warp] = sy; s_s[2][warp] = sz; s_s[3][warp] = sm; }
    __syncthreads();
    sx = sy = sz = sm = 0;
    for (int w = 0; w < kWarps; ++w) { sx += s_s[0][w]; sy += s_s[1][w]; sz += s_s[2][w]; sm += s_s[3][w]; }
  }
  const float cx = (float)((double)ref.x + sx / sm), cy = (float)((double)ref.y + sy / sm), cz = (float)((double)ref.z + sz / sm);
  float r = 0.f;
  for (uint32_t f = f0 + tid; f < f1; f += TPN) {
    const float4 c = node_c[f];
    const float dx = c.x - cx, dy = c.y - cy, dz = c.z - cz;
    r = fmaxf(r, sqrtf(dx * dx + dy * dy + dz * dz) * 1.000001f + node_r[f]);
  }
  for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, o));
  if (kWarps > 1) {
    if (lane == 0) s_r[warp] = r;
    __syncthreads();
    r = s_r[0];
    for (int w = 1; w < kWarps; ++w) r = fmaxf(r, s_r[w]);
  }
  (void)s_c;
  if (tid == 0) {
    const uint32_t idx = level_offset(n, l) + b;
    node_c[idx] = make_float4(cx, cy, cz, (float)sm);
    node_r[idx] = r + 2e-7f * (fabsf(cx) + fabsf(cy) + fabsf(cz));
  }
}

// ---- traversal + evaluation ----------------------------------------------------------------------------------------
// One source (hole, or pseudo-hole of charge m) against this thread's packed pair of targets: the inner loop of
// gc_field.cuh with one more FMUL2 for the charge.
template <bool WEIGHTED>
__device__ __forceinline__ void interact_w(const float4 sxy, const float2 sz, const float2 sm, const float2 ntx, const float2 nty,
                                           const float2 ntz, const float2 eps2v, float2& ax, float2& ay, float2& az) {
  const float2 dx = __fadd2_rn(make_float2(sxy.x, sxy.y), ntx);
  const float2 dy = __fadd2_rn(make_float2(sxy.z, sxy.w), nty);
  const float2 dz = __fadd2_rn(sz, ntz);
  float2 r2 = __ffma2_rn(dx, dx, eps2v);
  r2 = __ffma2_rn(dy, dy, r2);
  r2 = __ffma2_rn(dz, dz, r2);
  const float2 inv = make_float2(rsqrt_ftz(r2.x), rsqrt_ftz(r2.y));
  float2 w = __fmul2_rn(inv, inv);
  w = __fmul2_rn(w, inv);
  if (WEIGHTED) w = __fmul2_rn(w, sm);
  ax = __ffma2_rn(dx, w, ax);
  ay = __ffma2_rn(dy, w, ay);
  az = __ffma2_rn(dz, w, az);
}

struct TreeShared {
  float4 xy[256];
  float2 z[256];
  float2 m[256];
  uint32_t far[kFarCap];
  uint2 near[kNearCap];
  uint32_t pref[kNearCap + 1];
  uint32_t front[2][kFrontCap];
  uint32_t wcnt[2][kCPT][kTreeTPB / 32][3];
  float4 tgt[kGroup];          // the group's targets (sentinel where the group is ragged)
  float box1[6];               // box of the whole group (lo xyz, hi xyz)
  float box8[8][6];            // boxes of 32 targets
  float box32[32][6];          // boxes of 8 targets
  uint32_t group;
};

__device__ __forceinline__ float box_d2(const float (&b)[6], const float4 c) {
  const float dx = fmaxf(fmaxf(b[0] - c.x, c.x - b[3]), 0.f), dy = fmaxf(fmaxf(b[1] - c.y, c.y - b[4]), 0.f),
              dz = fmaxf(fmaxf(b[2] - c.z, c.z - b[5]), 0.f);
  return dx * dx + dy * dy + dz * dz;
}

// True iff every target of the group is at least R = a / theta from the node's centre c (R < 0: never).
__device__ __forceinline__ bool tree_accept(const TreeShared& S, const float4 c, const float R) {
  if (!(R >= 0.f)) return false;
  const float R2 = R * R * 1.000004f;                        // rounding of the distances below
  if (box_d2(S.box1, c) >= R2) return true;                  // far from the whole group: the common case
  for (int b = 0; b < 8; ++b) {
    if (box_d2(S.box8[b], c) >= R2) continue;
    for (int q = 4 * b; q < 4 * b + 4; ++q) {
      if (box_d2(S.box32[q], c) >= R2) continue;
      for (int t = 8 * q; t < 8 * q + 8; ++t) {
        const float4 x = S.tgt[t];
        const float dx = x.x - c.x, dy = x.y - c.y, dz = x.z - c.z;
        if (dx * dx + dy * dy + dz * dz < R2) return false;
      }
    }
  }
  return true;
}

template <bool WEIGHTED>
__device__ __forceinline__ void tree_eval_tile(const TreeShared& S, int len, const float2 ntx, const float2 nty, const float2 ntz,
                                               const float2 eps2v, float2& tx, float2& ty, float2& tz) {
  float2 ax = make_float2(0.f, 0.f), ay = ax, az = ax;
#pragma unroll 8
  for (int jj = 0; jj < len; ++jj) interact_w<WEIGHTED>(S.xy[jj], S.z[jj], S.m[jj], ntx, nty, ntz, eps2v, ax, ay, az);
  tx = __fadd2_rn(tx, ax); ty = __fadd2_rn(ty, ay); tz = __fadd2_rn(tz, az);       // two-level accumulation
}

// A group's work is split P ways: CTA ("part") p walks only the subtrees of the top-level nodes k = p (mod P) and
// evaluates what it finds; the P partial sums go to P chunks that the integrator adds in fixed order.  This keeps 148
// SMs busy when there are few groups and breaks up the occasional heavy group.  (Splitting the TILES of identical
// lists instead balanced the parts better but repeated the whole walk P times: slower once leaves hold 8 holes.)
// Callers guarantee a block barrier between the last list append and the flush; n_far / n_near are the (uniform)
// register copies of the list lengths and are reset here.
__device__ __forceinline__ void tree_flush_far(TreeShared& S, const Tree& T, uint32_t& n_far, const float2 ntx, const float2 nty,
                                               const float2 ntz, const float2 eps2v, float2& tx, float2& ty, float2& tz) {
  const uint32_t tid = threadIdx.x;
  const uint32_t nf = n_far;
  for (uint32_t base = 0; base < nf; base += 256) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t slot = tid + h * kTreeTPB, q = base + slot;
      float4 c = make_float4(kSentinel, kSentinel, kSentinel, 0.f);
      if (q < nf) c = T.node_c[S.far[q]];
      S.xy[slot] = make_float4(c.x, c.x, c.y, c.y); S.z[slot] = make_float2(c.z, c.z); S.m[slot] = make_float2(c.w, c.w);
    }
    __syncthreads();
    const int len = (int)min(256u, (nf - base + 7u) & ~7u);
    tree_eval_tile<true>(S, len, ntx, nty, ntz, eps2v, tx, ty, tz);
    __syncthreads();
  }
  if (tid == 0 && nf) atomicAdd(&T.tc->far_evals, (unsigned long long)nf * kGroup);
  n_far = 0;
}

__device__ __forceinline__ void tree_flush_near(TreeShared& S, const Tree& T, uint32_t& n_near, const float* __restrict__ px,
                                                const float* __restrict__ py, const float* __restrict__ pz, const float2 ntx,
                                                const float2 nty, const float2 ntz, const float2 eps2v, float2& tx, float2& ty,
                                                float2& tz) {
  const uint32_t tid = threadIdx.x, lane = tid & 31u;
  const uint32_t nn = n_near;
  if (tid < 32) {                                          // exclusive prefix of the range lengths, one warp
    uint32_t run = 0;
    for (uint32_t b = 0; b < nn; b += 32) {
      const uint32_t v = b + lane < nn ? S.near[b + lane].y : 0u;
      uint32_t inc = v;
      for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (uint32_t)o) inc += t; }
      if (b + lane < nn) S.pref[b + lane] = run + inc - v;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) S.pref[nn] = run;
  }
  __syncthreads();
  const uint32_t total = S.pref[nn];
  for (uint32_t base = 0; base < total; base += 256) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t slot = tid + h * kTreeTPB, q = base + slot;
      float x = kSentinel, y = kSentinel, z = kSentinel;
      if (q < total) {
        uint32_t lo = 0, hi = nn;                          // largest r with pref[r] <= q
        while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (S.pref[mid] <= q) lo = mid; else hi = mid; }
        const uint32_t i = S.near[lo].x + (q - S.pref[lo]);
        x = px[i]; y = py[i]; z = pz[i];
      }
      S.xy[slot] = make_float4(x, x, y, y); S.z[slot] = make_float2(z, z);
    }
    __syncthreads();
    const int len = (int)min(256u, (total - base + 7u) & ~7u);
    tree_eval_tile<false>(S, len, ntx, nty, ntz, eps2v, tx, ty, tz);
    __syncthreads();
  }
  if (tid == 0 && total) atomicAdd(&T.tc->near_evals, (unsigned long long)total * kGroup);
  n_near = 0;
}

// Field of every active carrier by the treecode; result in the first plan.S chunks of the partial planes, in the
// same convention as k_field: sum over sources of (r_s - r_t) w.  Persistent grid, groups handed out dynamically (the
// result of a group does not depend on which CTA computes it: list order and summation order are fixed).
__global__ void __launch_bounds__(kTreeTPB, 6)
k_tree_field(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
             const Ctrl* __restrict__ ctrl, Tree T, float* __restrict__ Ep, uint32_t part_cap, float eps2, float theta) {
  __shared__ TreeShared S;
  const uint32_t n = ctrl->n_active;
  if (n == 0) return;
  const uint32_t stride = ctrl->plan.stride;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t t0 = ctrl->plan.t0, t_end = t0 + ctrl->plan.nt;   // this rank's share of the targets (all, if unsharded)
  const uint32_t n_groups = (ctrl->plan.nt + kGroup - 1) / kGroup;
  const uint32_t P = max(ctrl->plan.S, 1u);                  // parts per group = partial chunks (set by the planner)
  uint32_t cnt[kTreeMaxLevels], off[kTreeMaxLevels];
  uint32_t ltop = 0;
  {
    uint32_t o = 0;
    bool found = false;
#pragma unroll
    for (uint32_t l = 0; l < kTreeMaxLevels; ++l) {
      cnt[l] = nodes_at(n, l); off[l] = o; o += cnt[l];
      if (!found && (cnt[l] <= kTopNodes || l + 1 == kTreeMaxLevels)) { ltop = l; found = true; }
    }
  }
  const float2 eps2v = make_float2(eps2, eps2);
  const float inv_theta = theta > 0.f ? 1.0f / theta * 1.000001f : 0.f;      // rounded up: never accepts more than a <= theta d
  constexpr uint32_t kInvalid = 0xffffffffu;

  for (;;) {
    if (tid == 0) S.group = atomicAdd(&T.tc->next_group, 1u);      // dynamic: with ~1.5 items per CTA, fetching ahead
    __syncthreads();                                                // (tried) costs more in balance than it hides
    const uint32_t item = S.group;
    if (item >= n_groups * P) break;
    const uint32_t g = item / P;
    const uint32_t part = item - g * P;
    // this thread's packed pair of targets, negated
    const uint32_t i0 = t0 + g * kGroup + 2u * tid;
    float2 vx = make_float2(0.f, 0.f), vy = vx, vz = vx;
    if (i0 + 1 < t_end) {
      vx = *reinterpret_cast<const float2*>(px + i0); vy = *reinterpret_cast<const float2*>(py + i0);
      vz = *reinterpret_cast<const float2*>(pz + i0);
    } else if (i0 < t_end) { vx.x = px[i0]; vy.x = py[i0]; vz.x = pz[i0]; }
    const float2 ntx = make_float2(-vx.x, -vx.y), nty = make_float2(-vy.x, -vy.y), ntz = make_float2(-vz.x, -vz.y);
    float2 tx = make_float2(0.f, 0.f), ty = tx, tz = tx;
    // Acceptance needs  a <= theta |x_t - c|  for EVERY target t of the group.  It is decided exactly, through a
    // small hierarchy over the group's own targets: 8 boxes of 32 targets, 32 boxes of 8, then the targets themselves
    // (tree_accept).  A single box (or ball) about the group would not do: where the occupancy is sparse the curve
    // leaves the cloud and re-enters it elsewhere, a run of 256 holes is then two distant pieces, and everything in
    // between would be swallowed into its exact near field.
    {
      const bool v0 = i0 < t_end, v1 = i0 + 1 < t_end;
      S.tgt[2 * tid] = v0 ? make_float4(vx.x, vy.x, vz.x, 0.f) : make_float4(kSentinel, kSentinel, kSentinel, 0.f);
      S.tgt[2 * tid + 1] = v1 ? make_float4(vx.y, vy.y, vz.y, 0.f) : make_float4(kSentinel, kSentinel, kSentinel, 0.f);
      float lo[3] = {v0 ? vx.x : 3e18f, v0 ? vy.x : 3e18f, v0 ? vz.x : 3e18f};
      float hi[3] = {v0 ? vx.x : -3e18f, v0 ? vy.x : -3e18f, v0 ? vz.x : -3e18f};
      if (v1) {
        lo[0] = fminf(lo[0], vx.y); lo[1] = fminf(lo[1], vy.y); lo[2] = fminf(lo[2], vz.y);
        hi[0] = fmaxf(hi[0], vx.y); hi[1] = fmaxf(hi[1], vy.y); hi[2] = fmaxf(hi[2], vz.y);
      }
#pragma unroll
      for (int o = 1; o <= 8; o <<= 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o)); hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
        }
        if (o == 2 && (lane & 3u) == 0) {                    // 4 lanes = 8 targets
#pragma unroll
          for (int c = 0; c < 3; ++c) { S.box32[tid >> 2][c] = lo[c]; S.box32[tid >> 2][3 + c] = hi[c]; }
        }
      }
      if ((lane & 15u) == 0) {                               // 16 lanes = 32 targets
#pragma unroll
        for (int c = 0; c < 3; ++c) { S.box8[tid >> 4][c] = lo[c]; S.box8[tid >> 4][3 + c] = hi[c]; }
      }
    }
    __syncthreads();
    if (tid < 3) {
      float lo = S.box8[0][tid], hi = S.box8[0][3 + tid];
      for (int b = 1; b < 8; ++b) { lo = fminf(lo, S.box8[b][tid]); hi = fmaxf(hi, S.box8[b][3 + tid]); }
      S.box1[tid] = lo; S.box1[3 + tid] = hi;
    }
    __syncthreads();
    // Level-by-level walk.  A frontier holds the OPENED nodes of the level above (one entry each); their children
    // k = 8 p + c are the candidates of this level.  At the top level the candidates are this part's share of its
    // nodes.  The list lengths live in registers, identical in every thread (each derives them from the per-warp
    // counts), so a batch of 256 candidates costs ONE barrier (three with shared-memory counters: the barrier after
    // the divergent acceptance test was the largest single stall of the kernel).
    uint32_t n_far = 0, n_near = 0, n_front_cur = 0, n_front_next = 0, par = 0;
    int cur = 0;
    for (uint32_t l = ltop;; --l) {
      const uint32_t n_cand = l == ltop ? cnt[ltop] : n_front_cur * kFan;
      const uint32_t lsize = level_size(l);
      for (uint32_t base = 0; base < n_cand; base += kBatch) {
        if (n_far + kBatch > kFarCap) { __syncthreads(); tree_flush_far(S, T, n_far, ntx, nty, ntz, eps2v, tx, ty, tz); }
        if (n_near + kBatch > kNearCap) { __syncthreads(); tree_flush_near(S, T, n_near, px, py, pz, ntx, nty, ntz, eps2v, tx, ty, tz); }
        const bool room = l > 0 && n_front_next + kBatch <= kFrontCap;
        uint32_t k[kCPT], b1[kCPT], b2[kCPT], b3[kCPT];
        float4 c[kCPT];
        float r[kCPT];
#pragma unroll
        for (int u = 0; u < kCPT; ++u) {                    // both candidates' node loads are in flight together
          const uint32_t q = base + u * kTreeTPB + tid;
          k[u] = kInvalid;
          if (q < n_cand) {
            k[u] = l == ltop ? q : S.front[cur][q >> 3] * kFan + (q & 7u);
            if (k[u] >= cnt[l] || (l == ltop && k[u] % P != part)) k[u] = kInvalid;   // this part's share of the top level
          }
          if (k[u] != kInvalid) { c[u] = T.node_c[off[l] + k[u]]; r[u] = T.node_r[off[l] + k[u]]; }
        }
        int cat[kCPT];                                      // 1 far, 2 near (exact), 3 open
#pragma unroll
        for (int u = 0; u < kCPT; ++u) {
          cat[u] = 0;
          if (k[u] != kInvalid) {
            if (theta > 0.f && tree_accept(S, c[u], r[u] * inv_theta)) cat[u] = 1;
            else cat[u] = room ? 3 : 2;                     // no room to open: sum the whole node exactly (always valid)
          }
          b1[u] = __ballot_sync(0xffffffffu, cat[u] == 1); b2[u] = __ballot_sync(0xffffffffu, cat[u] == 2);
          b3[u] = __ballot_sync(0xffffffffu, cat[u] == 3);
          if (lane == 0) {
            S.wcnt[par][u][warp][0] = __popc(b1[u]); S.wcnt[par][u][warp][1] = __popc(b2[u]); S.wcnt[par][u][warp][2] = __popc(b3[u]);
          }
        }
        __syncthreads();
        const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
        for (int u = 0; u < kCPT; ++u) {                    // list order: (u, warp, lane) — fixed, hence reproducible sums
          uint32_t o1 = n_far, o2 = n_near, o3 = n_front_next;
#pragma unroll
          for (uint32_t w = 0; w < kTreeTPB / 32; ++w) {
            const uint32_t c1 = S.wcnt[par][u][w][0], c2 = S.wcnt[par][u][w][1], c3 = S.wcnt[par][u][w][2];
            if (w < warp) { o1 += c1; o2 += c2; o3 += c3; }
            n_far += c1; n_near += c2; n_front_next += c3;
          }
          if (cat[u] == 1) S.far[o1 + __popc(b1[u] & lt)] = off[l] + k[u];
          else if (cat[u] == 2) {
            const uint32_t start = k[u] * lsize;
            S.near[o2 + __popc(b2[u] & lt)] = make_uint2(start, min(lsize, n - start));
          } else if (cat[u] == 3) S.front[cur ^ 1][o3 + __popc(b3[u] & lt)] = k[u];
        }
        par ^= 1u;                                          // double-buffered counts: the next batch may write at once
      }
      if (l == 0) break;
      __syncthreads();                                      // the next level's frontier is complete
      n_front_cur = n_front_next; n_front_next = 0;
      cur ^= 1;
    }
    __syncthreads();
    tree_flush_far(S, T, n_far, ntx, nty, ntz, eps2v, tx, ty, tz);
    tree_flush_near(S, T, n_near, px, py, pz, ntx, nty, ntz, eps2v, tx, ty, tz);

    if (i0 - t0 < stride) {                                   // partial rows are indexed from the share's start
      float* e = Ep + (size_t)part * stride + (i0 - t0);
      *reinterpret_cast<float2*>(e) = tx;
      *reinterpret_cast<float2*>(e + part_cap) = ty;
      *reinterpret_cast<float2*>(e + 2 * (size_t)part_cap) = tz;
    }
  }
}

}  // namespace gc
