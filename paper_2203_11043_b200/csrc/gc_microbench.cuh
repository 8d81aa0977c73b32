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
  kMicroKinds = 10
};

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
        }
      }
    }
  }
  const long long t1 = clock64();
  float acc = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) acc += c[k].x + c[k].y + a[k].x + b[k].y + (float)dc[k];
  if (acc == 123.456f) sink[0] = acc;                // keeps the chains alive
  if ((threadIdx.x & 31u) == 0) cycles[threadIdx.x >> 5] = t1 - t0;
}

// instructions of the probed kind per warp per outer iteration (4 x 8 chains; scalar kinds issue two per chain;
// the field mix issues 11 packed + 2 MUFU per chain)
inline double micro_inst_per_iter(int kind) {
  if (kind == kMicroFfmaScalarThree || kind == kMicroFfmaScalarShared) return 64.0;
  if (kind == kMicroFieldMix) return 32.0 * 11.0;    // reported per PACKED instruction; MUFU rides along
  return 32.0;
}

}  // namespace gc
