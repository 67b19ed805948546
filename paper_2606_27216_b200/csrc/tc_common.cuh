// Small device helpers shared by the tensor-core kernels (kernels_tc128.cu, kernels_tc64.cu):
// bf16 packing, packed fp32x2 arithmetic, fix-ups of one element of a packed register chunk.
#pragma once
#include <cuda_bf16.h>
#include <stdint.h>

namespace himuon {
namespace tc {

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// ---- packed fp32x2 arithmetic (FADD2 / FMUL2 / FFMA2 on sm_100) --------------------------------
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk2(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f2 pk2u(uint32_t lo, uint32_t hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi)); return r; }
__device__ __forceinline__ void upk2(f2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void upk2u(f2 v, uint32_t& lo, uint32_t& hi) { asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(v)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ uint32_t cvt_bf16x2(f2 v) {
  float lo, hi;
  upk2(v, lo, hi);
  return pack_bf16(lo, hi);
}

// Replace one bf16 of a packed 16-column chunk: word `idx` (0..7, or 8 for none) becomes (word & keep) | val.
__device__ __forceinline__ void set_one(uint32_t (&p)[8], int idx, uint32_t keep, uint32_t val) {
#pragma unroll
  for (int j = 0; j < 8; ++j) p[j] = (j == idx) ? ((p[j] & keep) | val) : p[j];
}
__device__ __forceinline__ void pack16(const uint32_t (&r)[16], uint32_t (&p)[8]) {
#pragma unroll
  for (int j = 0; j < 8; ++j) p[j] = pack_bf16(__uint_as_float(r[2 * j]), __uint_as_float(r[2 * j + 1]));
}

// ---- e4m3 operands (the F8 variants of kernels_tc128.cu, kernels_tc256.cu) ----------------------------------
// four fp32 (two packed pairs) -> four e4m3 bytes, element 0 in the low byte
__device__ __forceinline__ uint32_t cvt_e4m3x4(f2 v01, f2 v23) {
  float a, b, c, d;
  upk2(v01, a, b);
  upk2(v23, c, d);
  uint32_t r;
  asm("{\n\t.reg .b16 lo, hi;\n\tcvt.rn.satfinite.e4m3x2.f32 lo, %2, %1;\n\tcvt.rn.satfinite.e4m3x2.f32 hi, %4, %3;\n\t"
      "mov.b32 %0, {lo, hi};\n\t}"
      : "=r"(r) : "f"(a), "f"(b), "f"(c), "f"(d));
  return r;
}
// 16 accumulator columns, scaled by k -> 16 e4m3 (4 words)
__device__ __forceinline__ void pack16_e4m3(const uint32_t (&r)[16], f2 k2, uint32_t (&p)[4]) {
#pragma unroll
  for (int j = 0; j < 4; ++j)
    p[j] = cvt_e4m3x4(mul2(pk2u(r[4 * j], r[4 * j + 1]), k2), mul2(pk2u(r[4 * j + 2], r[4 * j + 3]), k2));
}
// Replace one byte of a packed 16-column chunk: word `idx` (0..3, or 4 for none) becomes (word & keep) | val.
__device__ __forceinline__ void set_one4(uint32_t (&p)[4], int idx, uint32_t keep, uint32_t val) {
#pragma unroll
  for (int j = 0; j < 4; ++j) p[j] = (j == idx) ? ((p[j] & keep) | val) : p[j];
}

}  // namespace tc
}  // namespace himuon
