// quant_math.cuh -- the NVFP4 scale / code arithmetic of DESIGN.md Q1-Q4, device side.
// Every float operation is an explicit round-to-nearest intrinsic (__fdiv_rn,
// __fmul_rn) so that no FMA contraction or approximate reciprocal can change a bit
// (reading O-5).  The grid conversions are the hardware cvt.rn.satfinite forms.
#pragma once
#include <cfloat>
#include <stdint.h>

namespace ft {

struct TensorScale {
  float g_enc, g_dec;
};

// Q3: g_enc = 2688 / amax_t, 1 if amax_t == 0, clamped to FLT_MAX; g_dec = 1 / g_enc.
__device__ __forceinline__ TensorScale tensor_scale(float amax_t) {
  TensorScale s;
  s.g_enc = (amax_t == 0.0f) ? 1.0f : __fdiv_rn(2688.0f, amax_t);
  if (isinf(s.g_enc)) s.g_enc = FLT_MAX;
  s.g_dec = __fdiv_rn(1.0f, s.g_enc);
  return s;
}

// float >= 0 -> E4M3 byte, RNE, satfinite (Q2)
__device__ __forceinline__ uint32_t f32_to_e4m3(float t) {
  uint16_t packed;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(packed) : "f"(0.0f), "f"(t));
  return (uint32_t)(packed & 0xFF);
}
__device__ __forceinline__ float e4m3_to_f32(uint32_t b) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)b));
  return __half2float(__ushort_as_half((unsigned short)(h2 & 0xFFFF)));
}

// Q4 per block: returns the scale byte and enc_b.
__device__ __forceinline__ void block_scale(float amax_b, const TensorScale& ts, uint32_t& sf8,
                                            float& enc_b) {
  float t = __fmul_rn(__fdiv_rn(amax_b, 6.0f), ts.g_enc);
  t = fminf(t, 448.0f);
  sf8 = f32_to_e4m3(t);
  const float sf = e4m3_to_f32(sf8);
  const float prod = __fmul_rn(sf, ts.g_dec);
  enc_b = (sf8 == 0) ? 0.0f : __fdiv_rn(1.0f, prod);
}

// 8 floats -> 8 E2M1 codes packed in a uint32 (element 0 in bits 0-3), Q1 + Q5
__device__ __forceinline__ uint32_t f32x8_to_e2m1(float x0, float x1, float x2, float x3,
                                                  float x4, float x5, float x6, float x7) {
  uint32_t r;
  asm("{\n\t.reg .b8 b0, b1, b2, b3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b0, %2, %1;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b1, %4, %3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b2, %6, %5;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b3, %8, %7;\n\t"
      "mov.b32 %0, {b0, b1, b2, b3};\n\t}"
      : "=r"(r)
      : "f"(x0), "f"(x1), "f"(x2), "f"(x3), "f"(x4), "f"(x5), "f"(x6), "f"(x7));
  return r;
}

// max |.| over the eight bf16 values held in a uint4 (exact)
__device__ __forceinline__ float amax_bf16x8(const uint4& v) {
  const uint32_t m = 0x7FFF7FFFu;
  uint32_t a = v.x & m, b = v.y & m, c = v.z & m, d = v.w & m;
  __nv_bfloat162 ha = *reinterpret_cast<__nv_bfloat162*>(&a);
  __nv_bfloat162 hb = *reinterpret_cast<__nv_bfloat162*>(&b);
  __nv_bfloat162 hc = *reinterpret_cast<__nv_bfloat162*>(&c);
  __nv_bfloat162 hd = *reinterpret_cast<__nv_bfloat162*>(&d);
  __nv_bfloat162 mx = __hmax2(__hmax2(ha, hb), __hmax2(hc, hd));
  return fmaxf(__low2float(mx), __high2float(mx));
}

// quantize the eight bf16 values of a uint4 with enc_b -> 8 codes (uint32)
__device__ __forceinline__ uint32_t quant_bf16x8(const uint4& v, float enc_b) {
  float f[8];
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __fmul_rn(__uint_as_float(w[i] << 16), enc_b);
    f[2 * i + 1] = __fmul_rn(__uint_as_float(w[i] & 0xFFFF0000u), enc_b);
  }
  return f32x8_to_e2m1(f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7]);
}

// ---- leaner forms for the hot kernel (bit-identical results)
// max |.| over eight bf16: max.xorsign.abs keeps max(|a|,|b|) in the magnitude bits
__device__ __forceinline__ uint32_t absmax2_bf16(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.xorsign.abs.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
// amax of a 1x16 block held in two uint4; exact (bf16 magnitudes order like their bit patterns)
__device__ __forceinline__ float amax_block16(const uint4& a, const uint4& b) {
  uint32_t m = absmax2_bf16(absmax2_bf16(absmax2_bf16(a.x, a.y), absmax2_bf16(a.z, a.w)),
                            absmax2_bf16(absmax2_bf16(b.x, b.y), absmax2_bf16(b.z, b.w)));
  m &= 0x7FFF7FFFu;
  const uint32_t best = max(m & 0xFFFFu, m >> 16);
  return __uint_as_float(best << 16);
}
// two fp32 products with one instruction (each a single IEEE round-to-nearest multiply)
__device__ __forceinline__ void mul2_rn(float& x0, float& x1, float s) {
  uint64_t a, b, d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(x0), "f"(x1));
  asm("mov.b64 %0, {%1, %1};" : "=l"(b) : "f"(s));
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(x0), "=f"(x1) : "l"(d));
}
__device__ __forceinline__ uint32_t quant_bf16x8_fast(const uint4& v, float enc_b) {
  float f[8];
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __uint_as_float(w[i] << 16);
    f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    mul2_rn(f[2 * i], f[2 * i + 1], enc_b);
  }
  return f32x8_to_e2m1(f[0], f[1], f[2], f[3], f[4], f[5], f[6], f[7]);
}
// enc_b of Q4 depends only on the scale byte and the tensor's g_dec: at most 127 values per
// tensor.  Entry i of the table is computed with the same two IEEE operations.
__device__ __forceinline__ float enc_of_sf8(uint32_t sf8, float g_dec) {
  const float prod = __fmul_rn(e4m3_to_f32(sf8), g_dec);
  return (sf8 == 0) ? 0.0f : __fdiv_rn(1.0f, prod);
}
// x / 6 for a bf16-valued x, correctly rounded, in three instructions: one Newton step on
// x * fl(1/6) with exact residual.  Equal to the IEEE quotient for every finite non-negative bf16 x
// (all 32 640 of them, subnormal quotients included): tests/test_host_logic.py proves it in exact
// rational arithmetic.  The general-purpose __fdiv_rn is ~12 instructions with a slow-path branch.
__device__ __forceinline__ float div6_bf16(float x) {
  const float c = 0.16666667163372039795f;   // fl(1/6)
  const float q0 = __fmul_rn(x, c);
  const float r = __fmaf_rn(-6.0f, q0, x);
  return __fmaf_rn(r, c, q0);
}
__device__ __forceinline__ uint32_t block_sf8(float amax_b, float g_enc) {
  float t = __fmul_rn(div6_bf16(amax_b), g_enc);
  return f32_to_e4m3(fminf(t, 448.0f));
}

// byte offset of scale (row r, 16-wide block c) in FT_SF_TILE128x4 (include/fourtune.h)
__host__ __device__ __forceinline__ int64_t sf_tile_offset(int64_t r, int64_t c, int64_t nblk) {
  const int64_t tiles_c = (nblk + 3) / 4;
  return ((r / 128) * tiles_c + c / 4) * 512 + (r % 32) * 16 + ((r % 128) / 32) * 4 + (c % 4);
}

}  // namespace ft
