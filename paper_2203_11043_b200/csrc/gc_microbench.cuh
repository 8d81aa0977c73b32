// gc_microbench.cuh — instruction-throughput probes behind DESIGN.md 6.1 / 6.8 (tracked so that those numbers can be
// regenerated: `python bench.py --microbench`).  Not on the hot path.  One CTA on one SM, `warps` warps per SM
// sub-partition, each running 8 independent dependency chains of one instruction kind; the figure reported is cycles
// per warp-instruction per sub-partition (2.0 = a packed FP32x2 instruction at full lane rate: 32 lanes x 2 values on
// 32 FP32 lanes; 1.0 for a scalar FP32 instruction; 2.0 for FP64 at 16 lanes per sub-partition).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gc {

enum MicroKind {
  kMicroFfma2Three = 0,     // d = a * b + c, three distinct register pairs per instruction (eq. 6's accumulates d.w + a)
  kMicroFfma2Two = 1,       // d = a * a + c (eq. 6's r^2 chain: dx.dx + r2)
  kMicroFfma2Shared = 2,    // d = s * b + c with s shared by consecutive instructions (operand-reuse cache)
  kMicroFadd2 = 3,
  kMicroFmul2 = 4,
  kMicroFfmaScalarThree = 5,
  kMicroFfmaScalarShared = 6,
  kMicroDfma = 7,           // FP64 pipe: the bound of k_advance
  kMicroRsqrt = 8,          // MUFU.RSQ
  kMicroFieldMix = 9,       // the 11 packed instructions + 2 MUFU of one eq. 6 interaction pair, from registers
  kMicroF2F64to32 = 10,     // cvt.rn.f32.f64: which pipe converts, and how fast (FP64-pipe offload experiment)
  kMicroF2F32to64 = 11,     // cvt.f64.f32
  kMicroDadd = 12,
  kMicroField64 = 13,       // one eq. 6 interaction per lane on the FP64 pipe: 3 DADD + 3 DFMA + F2F + MUFU + 2 FMUL + F2F + 3 DFMA
  kMicroFieldMixD1 = 14,    // eq. 6 mix on 8 packs (16 FP32 targets) + 1 FP64-pipe target per lane, interleaved
  kMicroFieldMixD2 = 15,    // ... + 2 FP64-pipe targets
  kMicroFieldMixD4 = 16,    // ... + 4 FP64-pipe targets
  kMicroKinds = 17
};

// one source against one target on the FP64 pipe: differences, r^2 and the accumulates in FP64, w = r^-3 through the FP32
// MUFU.RSQ (relative error 2e-7: the same w the FP32 path uses)
__device__ __forceinline__ void interact64(const double sx, const double sy, const double sz, const double ntx, const double nty,
                                           const double ntz, const double eps2, double& ax, double& ay, double& az) {
  const double dx = sx + ntx, dy = sy + nty, dz = sz + ntz;
  double r2 = fma(dx, dx, eps2);
  r2 = fma(dy, dy, r2);
  r2 = fma(dz, dz, r2);
  float r2f, inv;
  asm("cvt.rn.f32.f64 %0, %1;" : "=f"(r2f) : "d"(r2));
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(r2f));
  const float wf = (inv * inv) * inv;
  double w;
  asm("cvt.f64.f32 %0, %1;" : "=d"(w) : "f"(wf));
  ax = fma(dx, w, ax);
  ay = fma(dy, w, ay);
  az = fma(dz, w, az);
}

template <int KIND>
__global__ void __launch_bounds__(512, 1) k_microbench(uint32_t iters, float seed, long long* cycles, float* sink) {
  float2 a[8], b[8], c[8];
  double da[8], db[8], dc[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    a[k] = make_float2(seed + 0.001f * (float)(threadIdx.x + k), seed * 0.5f + (float)k);
    b[k] = make_float2(1.0f + 1e-6f * (float)k, 1.0f - 1e-6f * (float)(threadIdx.x & 7));
    c[k] = make_float2(0.25f * (float)k, 0.125f);
    da[k] = (double)a[k].x; db[k] = (double)b[k].x; dc[k] = (double)c[k].x;
  }
  const float2 sh = make_float2(seed, seed + 1.0f);
  const double dsz = (double)seed * 0.75;
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (KIND == kMicroFfma2Three) c[k] = __ffma2_rn(a[k], b[k], c[k]);
        else if (KIND == kMicroFfma2Two) c[k] = __ffma2_rn(a[k], a[k], c[k]);
        else if (KIND == kMicroFfma2Shared) c[k] = __ffma2_rn(sh, b[k], c[k]);
        else if (KIND == kMicroFadd2) c[k] = __fadd2_rn(a[k], c[k]);
        else if (KIND == kMicroFmul2) c[k] = __fmul2_rn(b[k], c[k]);
        else if (KIND == kMicroFfmaScalarThree) { c[k].x = __fmaf_rn(a[k].x, b[k].x, c[k].x); c[k].y = __fmaf_rn(a[k].y, b[k].y, c[k].y); }
        else if (KIND == kMicroFfmaScalarShared) { c[k].x = __fmaf_rn(sh.x, b[k].x, c[k].x); c[k].y = __fmaf_rn(sh.x, b[k].y, c[k].y); }
        else if (KIND == kMicroDfma) dc[k] = fma(da[k], db[k], dc[k]);
        else if (KIND == kMicroRsqrt) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(c[k].x)); c[k].x = y + 1.5f; }
        else if (KIND == kMicroF2F64to32) { float y; asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(y) : "d"(dc[k])); dc[k] = da[k]; c[k].x += y; }
        else if (KIND == kMicroF2F32to64) { double y; asm volatile("cvt.f64.f32 %0, %1;" : "=d"(y) : "f"(c[k].x)); dc[k] = y; }
        else if (KIND == kMicroDadd) dc[k] = da[k] + dc[k];
        else if (KIND == kMicroField64) interact64((double)sh.x, (double)sh.y, db[k], da[k], db[(k + 1) & 7], da[(k + 3) & 7], 1e-6, dc[k], da[k], db[k]);
        else {                                      // one source against target pack k: eq. 6 as in gc_field.cuh interact<>
          const float2 dx = __fadd2_rn(sh, a[k]), dy = __fadd2_rn(sh, b[k]), dz = __fadd2_rn(make_float2(sh.y, sh.x), a[k]);
          float2 r2 = __ffma2_rn(dx, dx, make_float2(1e-6f, 1e-6f));
          r2 = __ffma2_rn(dy, dy, r2);
          r2 = __ffma2_rn(dz, dz, r2);
          float ix, iy;
          asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(ix) : "f"(r2.x));
          asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(iy) : "f"(r2.y));
          const float2 inv = make_float2(ix, iy);
          float2 w = __fmul2_rn(inv, inv);
          w = __fmul2_rn(w, inv);
          c[k] = __ffma2_rn(dx, w, c[k]);
          a[k] = __ffma2_rn(dy, w, a[k]);
          b[k] = __ffma2_rn(dz, w, b[k]);
          constexpr int ND = KIND == kMicroFieldMixD1 ? 1 : KIND == kMicroFieldMixD2 ? 2 : KIND == kMicroFieldMixD4 ? 4 : 0;
          if (ND > 0 && (k % (8 / (ND > 0 ? ND : 1))) == 0) {
            const int q = k / (8 / (ND > 0 ? ND : 1));
            interact64((double)sh.x, (double)sh.y, dsz, da[q], db[q], da[q + 4], 1e-6, dc[q], dc[q + 4], db[q + 4]);
          }
        }
      }
    }
  }
  const long long t1 = clock64();
  float acc = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) acc += c[k].x + c[k].y + a[k].x + b[k].y + (float)dc[k] + (float)da[k] + (float)db[k];
  if (acc == 123.456f) sink[0] = acc;                // keeps the chains alive
  if ((threadIdx.x & 31u) == 0) cycles[threadIdx.x >> 5] = t1 - t0;
}

// instructions of the probed kind per warp per outer iteration (4 x 8 chains; scalar kinds issue two per chain;
// the field mix issues 11 packed + 2 MUFU per chain)
inline double micro_inst_per_iter(int kind) {
  if (kind == kMicroFfmaScalarThree || kind == kMicroFfmaScalarShared) return 64.0;
  if (kind == kMicroFieldMix) return 32.0 * 11.0;    // reported per PACKED instruction; MUFU rides along
  if (kind >= kMicroFieldMixD1) return 4.0;          // reported per round of 8 packs (+ 1 / 2 / 4 FP64 targets) per lane
  return 32.0;                                       // kMicroField64: per interaction (its 9 FP64 + 2 F2F + 3 FP32 ride along)
}

}  // namespace gc
