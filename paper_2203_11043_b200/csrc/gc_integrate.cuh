// gc_integrate.cuh — steps a2..a7 fused in one kernel (PAPER.md:68 order):
//   reduce the field partials in fixed order -> E_Coul = K' S (eq. 6) -> + depletion field (eq. 1) -> |E| ->
//   mobility (eq. 2) -> drift (v = mu E) -> Philox4x32-10 + Box-Muller diffusion (eqs. 3-4) -> update ->
//   mirror at the back surface -> collection test -> integer atomic pixel histogram.
// O(N) and bandwidth/latency bound; the per-carrier arithmetic is done in FP64 (B200 runs FP64 at half the
// FP32 rate, and this kernel is < 0.1 % of a step at large N) so that a carrier's new position is the
// correctly rounded FP32 value of the same FP64 expression the oracle evaluates; only E_Coul carries FP32
// summation error.  State is stored FP32.
#pragma once
#include "gc_common.cuh"

namespace gc {

// ---------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  Counter = (id, 0, step_lo, step_hi), key = (seed_lo, seed_hi).
// Written independently of oracle/goracle.c (DESIGN.md §3 R13).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}

// u = ((w>>9)+0.5) 2^-23 in (0,1); f = (w>>8) 2^-24 in [0,1): exactly representable in FP32 and FP64.
// n = (R_a cos 2 pi f_a, R_a sin 2 pi f_a, R_b cos 2 pi f_b), R = sqrt(-2 ln u).
// The draw is written as four independent chains (R_a | sin, cos | R_b | cos) so that the small-population kernel
// (gc_persist.cuh) can give each to a thread of its own; one thread running all four computes the same bits.
struct BoxMuller { double Ra, sa, ca, Rb, cb; };
__device__ __forceinline__ uint4 philox_words(uint32_t seed_lo, uint32_t seed_hi, uint32_t id, uint64_t step) {
  return philox4x32_10(make_uint4(id, 0u, (uint32_t)step, (uint32_t)(step >> 32)), make_uint2(seed_lo, seed_hi));
}
__device__ __forceinline__ double bm_radius(uint32_t w) {
  const double u = ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0);
  return sqrt(-2.0 * log(u));
}
__device__ __forceinline__ double bm_fraction(uint32_t w) { return (double)(w >> 8) * (1.0 / 16777216.0); }
__device__ __forceinline__ void bm_chain(const uint4 w, int chain, BoxMuller& b) {   // chain 0..3, or -1 = all
  if (chain == 0 || chain < 0) b.Ra = bm_radius(w.x);
  if (chain == 1 || chain < 0) sincospi(2.0 * bm_fraction(w.y), &b.sa, &b.ca);
  if (chain == 2 || chain < 0) b.Rb = bm_radius(w.z);
  if (chain == 3 || chain < 0) b.cb = cospi(2.0 * bm_fraction(w.w));
}
__device__ __forceinline__ void philox_normals(uint32_t seed_lo, uint32_t seed_hi, uint32_t id, uint64_t step,
                                               double n[3], uint4* words) {
  const uint4 w = philox_words(seed_lo, seed_hi, id, step);
  BoxMuller b;
  bm_chain(w, -1, b);
  n[0] = b.Ra * b.ca; n[1] = b.Ra * b.sa; n[2] = b.Rb * b.cb;
  if (words) *words = w;
}

// eq. 2 with the temperature terms folded on the host: mu = mu0 f(r), f(r) = (1 + r^beta)^(-1/beta), r = E/Ec.
//
// Direct evaluation is mu0 exp(-log1p(exp(beta log r)) / beta): four FP64 transcendentals in series, ~2,400 cycles of
// dependent instructions on a lone warp — the longest link of the per-carrier chain that bounds a small population's
// step and a small event's step (gc_persist.cuh, gc_events.cuh).  f is analytic away from r = 0 and r^beta = -1, so on
// a sixteenth of a binade it is reproduced to < 1e-19 relative by its degree-8 Chebyshev interpolant (nearest
// singularity at 128 half-widths: error ~ 128^-9); gcoreccd_create tabulates those interpolants in long double for
// 2^-16 <= r < 2^16 (E from 0.08 V/cm to 3e8 V/cm at 140 K) as monomial coefficients in u in [-1, 1].  Evaluation: exponent and
// the top four mantissa bits select the row, u is exact, eight FMAs: ~150 cycles, rounding error ~2 ulp — the same
// class as the four chained libm calls it replaces, ten orders below what the FP32 state resolves.  Outside the table
// (r = 0, tiny, huge, NaN) the direct form runs.  mobility_direct is also what tests/ compare the table with.
__device__ __forceinline__ double mobility_direct(double E, const DevParams& P) {
  const double t = exp(P.beta * log(E * P.inv_Ec));          // E = 0: log = -inf, exp = 0, mu = mu0
  return P.mu0 * exp(-P.inv_beta * log1p(t));
}
__device__ __forceinline__ double mobility(double E, const DevParams& P) {
  const double r = E * P.inv_Ec;
  const long long bits = __double_as_longlong(r);
  const int e = (int)((bits >> 52) & 0x7ff) - 1023;
  if (e < kMuEmin || e >= kMuEmax || bits < 0) return mobility_direct(E, P);
  const int j = (int)((bits >> 48) & 15);
  const double m = __longlong_as_double((bits & 0x000fffffffffffffLL) | 0x3ff0000000000000LL);   // mantissa in [1, 2)
  const double u = (m - (1.0 + ((double)j + 0.5) * (1.0 / kMuSub))) * (2.0 * kMuSub);         // exact, in [-1, 1)
  const double* c = P.mu_tab + ((e - kMuEmin) * kMuSub + j) * (kMuDeg + 1);
  double f = __ldg(c + kMuDeg);
#pragma unroll
  for (int k = kMuDeg - 1; k >= 0; --k) f = fma(f, u, __ldg(c + k));
  return P.mu0 * f;
}

// a7: half-open pixel bins, floor, in FP64 on the stored FP32 position (exactly reproducible); the final position
// and the index of the crossing step are recorded per carrier id ("output positions").
__device__ __forceinline__ void collect(float x, float y, float z, uint32_t id, uint64_t step, const DevParams& P,
                                        const Sink& sink, uint32_t& n_over) {
  const double fx = floor(((double)x - P.x0) / P.pitch);
  const double fy = floor(((double)y - P.y0) / P.pitch);
  if (fx >= 0.0 && fx < (double)P.nx && fy >= 0.0 && fy < (double)P.ny)
    atomicAdd(sink.image + (size_t)fy * (size_t)P.nx + (size_t)fx, 1u);
  else
    n_over += 1u;
  if (id < sink.fin_cap) sink.fin[id] = make_float4(x, y, z, __uint_as_float((uint32_t)step));
}

// Sum of the S column-chunk partials of one target, in FP64 and in fixed (ascending chunk) order.  The loads of
// a batch of kRedBatch chunks are issued together before any is consumed: the loop is bound by L2 latency, and a
// load -> convert -> add chain per chunk would serialise S round trips.
constexpr int kRedBatch = 8;
__device__ __forceinline__ void reduce_partials(const float* __restrict__ e, uint32_t part_cap, uint32_t S, uint32_t stride,
                                                double& Ex, double& Ey, double& Ez) {
  const float* ey = e + part_cap;
  const float* ez = ey + part_cap;
  for (uint32_t s0 = 0; s0 < S; s0 += kRedBatch) {
    float vx[kRedBatch], vy[kRedBatch], vz[kRedBatch];
#pragma unroll
    for (int u = 0; u < kRedBatch; ++u) {
      const bool ok = s0 + u < S;
      const size_t o = (size_t)(s0 + u) * stride;
      vx[u] = ok ? __ldg(e + o) : 0.f; vy[u] = ok ? __ldg(ey + o) : 0.f; vz[u] = ok ? __ldg(ez + o) : 0.f;
    }
#pragma unroll
    for (int u = 0; u < kRedBatch; ++u) { Ex += (double)vx[u]; Ey += (double)vy[u]; Ez += (double)vz[u]; }
  }
}

// a2..a6 for one carrier: (Ex,Ey,Ez) is its Coulomb field in V/cm (eq. 6), nrm its normal triple (unused with
// DIFFUSION_OFF); returns the new FP32 position, i.e. the correctly rounded value of the FP64 expression the oracle
// evaluates.  False if the result is not finite.
__device__ __forceinline__ bool advance_with_normals(float x, float y, float z, double Ex, double Ey, double Ez, const double nrm[3],
                                                     const DevParams& P, float& xf, float& yf, float& zf) {
  if (!(P.flags & 4u)) Ez += P.a1_um * (double)z - P.a2;     // eq. 1
  const double Emag = sqrt(Ex * Ex + Ey * Ey + Ez * Ez);
  const double mu = mobility(Emag, P);                       // eq. 2
  const double kd = P.drift_k * mu;                          // 1e-5 mu dt
  double dx = kd * Ex, dy = kd * Ey, dz = kd * Ez;
  if (!(P.flags & 2u)) {                                     // eqs. 3-4
    const double sigma = sqrt(P.sigma_k * mu);
    dx += sigma * nrm[0]; dy += sigma * nrm[1]; dz += sigma * nrm[2];
  }
  const double xn = (double)x + dx, yn = (double)y + dy;
  double zn = (double)z + dz;
  if (zn > P.thickness) zn = 2.0 * P.thickness - zn;         // specular back surface
  xf = (float)xn; yf = (float)yn; zf = (float)zn;
  return isfinite(xf) && isfinite(yf) && isfinite(zf);
}

__device__ __forceinline__ bool advance_carrier(float x, float y, float z, uint32_t id, uint64_t step, double Ex, double Ey,
                                                double Ez, const DevParams& P, float& xf, float& yf, float& zf) {
  double nrm[3] = {0.0, 0.0, 0.0};
  if (!(P.flags & 2u)) philox_normals(P.seed_lo, P.seed_hi, id, step, nrm, nullptr);
  return advance_with_normals(x, y, z, Ex, Ey, Ez, nrm, P, xf, yf, zf);
}

// Block-level tally of (collected, overflow) and the survivor count of this tile.
__device__ __forceinline__ void tally(uint32_t coll, uint32_t over, uint32_t keep, Ctrl* ctrl, uint32_t* tile_count) {
  __shared__ uint32_t s_c[3];
  if (threadIdx.x < 3) s_c[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t wc = __popc(__ballot_sync(0xffffffffu, coll)), wo = __popc(__ballot_sync(0xffffffffu, over)),
                 wk = __popc(__ballot_sync(0xffffffffu, keep));
  if ((threadIdx.x & 31u) == 0) {
    if (wc) atomicAdd(&s_c[0], wc);
    if (wo) atomicAdd(&s_c[1], wo);
    if (wk) atomicAdd(&s_c[2], wk);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (s_c[0]) atomicAdd((unsigned long long*)&ctrl->n_collected, (unsigned long long)s_c[0]);
    if (s_c[1]) atomicAdd((unsigned long long*)&ctrl->n_overflow, (unsigned long long)s_c[1]);
    tile_count[blockIdx.x] = s_c[2];
  }
}

// One thread per carrier; tile = kTPB carriers; reads state A + partials, writes state B (same index) and
// the tile's survivor count.  Grid is sized from the host's upper bound on n_active; surplus CTAs exit.
__global__ void __launch_bounds__(kTPB, 4)      // 64 registers: 4 CTAs/SM, 151,552 carriers in one wave on 148 SMs
k_integrate(SoA A, SoA B, Ctrl* __restrict__ ctrl, const float* __restrict__ Ep, uint32_t part_cap,
            Sink sink, uint32_t* __restrict__ tile_count, DevParams P) {
  const uint32_t t0 = ctrl->plan.t0, nt = ctrl->plan.nt;     // this rank's share: [0, n_active) unless sharded
  const uint32_t k = blockIdx.x * kTPB + threadIdx.x;        // index inside the share (= partial-sum row)
  if (blockIdx.x * kTPB >= nt) return;
  const uint32_t i = t0 + k;
  const uint64_t step = ctrl->step;
  uint32_t coll = 0, over = 0, keep = 0;
  if (k < nt) {
    const float x = A.x[i], y = A.y[i], z = A.z[i];
    const uint32_t id = A.id[i];
    double Ex = 0.0, Ey = 0.0, Ez = 0.0;
    if (!(P.flags & 1u)) {                                   // GCORECCD_COULOMB_OFF
      reduce_partials(Ep + k, part_cap, ctrl->plan.S, ctrl->plan.stride, Ex, Ey, Ez);
      Ex *= -P.Kp; Ey *= -P.Kp; Ez *= -P.Kp;                 // partials hold sum (r_s - r_t) w
    }
    float xf, yf, zf;
    if (!advance_carrier(x, y, z, id, step, Ex, Ey, Ez, P, xf, yf, zf)) atomicOr(&ctrl->nonfinite, 1u);
    B.x[i] = xf; B.y[i] = yf; B.z[i] = zf; B.id[i] = id;
    if ((double)zf <= P.z_well) { coll = 1; uint32_t o = 0; collect(xf, yf, zf, id, step, P, sink, o); over = o; }
    else keep = 1;
  }
  tally(coll, over, keep, ctrl, tile_count);
}

// Coulomb OFF (the O(N) mode): without eq. 6 the carriers are independent, so one launch takes
// every carrier through up to n_steps steps (or to collection) instead of one launch train per step.  Same
// advance_carrier, same Philox counters (id, step): bit-identical to n_steps single steps.  The step index advances
// by the steps the longest-lived carrier needed (a step with nobody drifting is a no-op), via ctrl->multi_steps.
__global__ void __launch_bounds__(kTPB, 4)
k_drift_multi(SoA A, SoA B, Ctrl* __restrict__ ctrl, Sink sink, uint32_t* __restrict__ tile_count, DevParams P,
              uint32_t n_steps) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (blockIdx.x * kTPB >= n) return;
  const uint64_t step0 = ctrl->step;
  uint32_t coll = 0, over = 0, keep = 0, taken = 0;
  if (i < n) {
    float x = A.x[i], y = A.y[i], z = A.z[i];
    const uint32_t id = A.id[i];
    bool bad = false;
    for (uint32_t k = 0; k < n_steps; ++k) {
      float xf, yf, zf;
      if (!advance_carrier(x, y, z, id, step0 + k, 0.0, 0.0, 0.0, P, xf, yf, zf)) bad = true;
      x = xf; y = yf; z = zf;
      taken = k + 1;
      if ((double)z <= P.z_well) { coll = 1; uint32_t o = 0; collect(x, y, z, id, step0 + k, P, sink, o); over = o; break; }
      if (bad) break;                                        // non-finite: stop here, the flag below reports it
    }
    if (bad) atomicOr(&ctrl->nonfinite, 1u);
    B.x[i] = x; B.y[i] = y; B.z[i] = z; B.id[i] = id;
    keep = coll ? 0u : 1u;
  }
  const uint32_t wmax = __reduce_max_sync(0xffffffffu, taken);
  if ((threadIdx.x & 31u) == 0 && wmax) atomicMax(&ctrl->multi_steps, wmax);
  tally(coll, over, keep, ctrl, tile_count);
}

// Load path: unpack interleaved xyz into state B at [0,n), assign ids n_loaded + k, collect z <= z_well.
__global__ void __launch_bounds__(kTPB)
k_unpack(const float* __restrict__ xyz, uint32_t n, SoA B, Ctrl* __restrict__ ctrl, uint32_t id_base,
         Sink sink, uint32_t* __restrict__ tile_count, DevParams P, uint32_t record) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  uint32_t coll = 0, over = 0, keep = 0;
  const uint64_t step = ctrl->step;
  if (i < n) {
    const float x = xyz[3 * (size_t)i], y = xyz[3 * (size_t)i + 1], z = xyz[3 * (size_t)i + 2];
    B.x[i] = x; B.y[i] = y; B.z[i] = z; B.id[i] = id_base + i;
    // sharded runs load the same holes on every rank: only rank 0 (record = 1) bins the ones collected at load
    if ((double)z <= P.z_well) { if (record) { coll = 1; uint32_t o = 0; collect(x, y, z, id_base + i, step, P, sink, o); over = o; } }
    else keep = 1;
  }
  tally(coll, over, keep, ctrl, tile_count);
}

// Load validation: any non-finite coordinate or z above the back surface sets ctrl->invalid.
__global__ void __launch_bounds__(kTPB)
k_validate(const float* __restrict__ xyz, uint32_t n, Ctrl* __restrict__ ctrl, double thickness) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  const float x = xyz[3 * (size_t)i], y = xyz[3 * (size_t)i + 1], z = xyz[3 * (size_t)i + 2];
  if (!(isfinite(x) && isfinite(y) && isfinite(z)) || (double)z > thickness) atomicOr(&ctrl->invalid, 1u);
}

// eval_field epilogue: E = -K' * sum_s partial, interleaved Ex,Ey,Ez.
__global__ void __launch_bounds__(kTPB)
k_field_finalize(const Ctrl* __restrict__ ctrl, const float* __restrict__ Ep, uint32_t part_cap, double Kp,
                 float* __restrict__ out) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  double Ex = 0.0, Ey = 0.0, Ez = 0.0;
  reduce_partials(Ep + i, part_cap, ctrl->plan.S, ctrl->plan.stride, Ex, Ey, Ez);
  out[3 * (size_t)i] = (float)(-Kp * Ex); out[3 * (size_t)i + 1] = (float)(-Kp * Ey); out[3 * (size_t)i + 2] = (float)(-Kp * Ez);
}

// read_carriers: SoA -> interleaved xyz
__global__ void __launch_bounds__(kTPB)
k_interleave(SoA A, const Ctrl* __restrict__ ctrl, float* __restrict__ xyz) {
  const uint32_t n = ctrl->n_active;
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  xyz[3 * (size_t)i] = A.x[i]; xyz[3 * (size_t)i + 1] = A.y[i]; xyz[3 * (size_t)i + 2] = A.z[i];
}

// read_collected: per-id records -> interleaved xyz (NaN while drifting) and the crossing step (all-ones likewise)
__global__ void __launch_bounds__(kTPB)
k_read_final(const float4* __restrict__ fin, uint32_t n, float* __restrict__ xyz, uint32_t* __restrict__ step) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  const float4 f = fin[i];
  xyz[3 * (size_t)i] = f.x; xyz[3 * (size_t)i + 1] = f.y; xyz[3 * (size_t)i + 2] = f.z;
  step[i] = __float_as_uint(f.w);
}

// load_snapshot: replace the active set
__global__ void __launch_bounds__(kTPB)
k_set_snapshot(const float* __restrict__ xyz, const uint32_t* __restrict__ id, uint32_t n, SoA A) {
  const uint32_t i = blockIdx.x * kTPB + threadIdx.x;
  if (i >= n) return;
  A.x[i] = xyz[3 * (size_t)i]; A.y[i] = xyz[3 * (size_t)i + 1]; A.z[i] = xyz[3 * (size_t)i + 2]; A.id[i] = id[i];
}

// test hook: eq. 2 as the kernels evaluate it (table) and by the direct form
__global__ void k_debug_mobility(const double* __restrict__ E, uint32_t n, DevParams P, double* __restrict__ mu_table,
                                 double* __restrict__ mu_direct) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  mu_table[i] = mobility(E[i], P);
  mu_direct[i] = mobility_direct(E[i], P);
}

__global__ void k_debug_normals(const uint32_t* __restrict__ id, const uint64_t* __restrict__ step, uint32_t n,
                                uint32_t seed_lo, uint32_t seed_hi, double* __restrict__ out, uint32_t* __restrict__ words) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double nrm[3]; uint4 w;
  philox_normals(seed_lo, seed_hi, id[i], step[i], nrm, &w);
  out[3 * i] = nrm[0]; out[3 * i + 1] = nrm[1]; out[3 * i + 2] = nrm[2];
  words[4 * i] = w.x; words[4 * i + 1] = w.y; words[4 * i + 2] = w.z; words[4 * i + 3] = w.w;
}

}  // namespace gc
