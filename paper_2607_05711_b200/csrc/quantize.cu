// quantize.cu -- a0 (tensor amax), a6 (offline weight quantize + pack) and the
// generic block quantizer.  The hot fused quantize + down-projection kernel (a1/a3)
// is in quantize_fused.cu.
#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

// ------------------------------------------------------------------ a0: amax
// max |x| of n bf16 values.  |x| of a finite bf16 orders like its low 15 bits, so
// the reduction runs on integers and atomicMax on the float's bit pattern is exact.
__global__ void __launch_bounds__(256) k_amax(const uint4* __restrict__ x, int64_t n_vec,
                                              const uint16_t* __restrict__ tail, int n_tail,
                                              unsigned int* __restrict__ out_bits) {
  pdl_wait();      // behind the clear kernel of the quantize call (no-op without a programmatic edge)
  pdl_trigger();
  const uint32_t m = 0x7FFF7FFFu;
  uint32_t acc = 0;  // two 15-bit maxima packed; compared per half with vmax
  // a CTA walks 32 KB tiles (256 threads x 8 x 16 bytes); the 8 loads of a thread are issued
  // back to back so 32 KB per CTA are in flight
  const int64_t n_tiles = (n_vec + 2047) / 2048;
  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t base = tile * 2048 + threadIdx.x;
    uint4 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int64_t i = base + j * 256;
      v[j] = make_uint4(0, 0, 0, 0);
      if (i < n_vec) asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                                  : "=r"(v[j].x), "=r"(v[j].y), "=r"(v[j].z), "=r"(v[j].w) : "l"(x + i));
    }
#pragma unroll
    for (int j = 0; j < 8; ++j)
      acc = __vmaxu2(acc, __vmaxu2(__vmaxu2(v[j].x & m, v[j].y & m), __vmaxu2(v[j].z & m, v[j].w & m)));
  }
  if (blockIdx.x == 0 && threadIdx.x < n_tail) acc = __vmaxu2(acc, (uint32_t)(tail[threadIdx.x] & 0x7FFF));
  uint32_t best = max(acc & 0xFFFFu, acc >> 16);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
  __shared__ uint32_t s_best[8];
  if ((threadIdx.x & 31) == 0) s_best[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) best = max(best, s_best[w]);
    atomicMax(out_bits, best << 16);  // bf16 bits -> float bits; non-negative floats order as uints
  }
}

// zero_first: the target word is not known to be zero (ft_tensor_amax): a memset node precedes the kernel.
// pdl: a kernel of the same call directly precedes the launch (never together with zero_first: a memset
// predecessor gets no programmatic edge).
int launch_amax(const void* x_bf16, int64_t n, float* amax_out, cudaStream_t st, bool zero_first, bool pdl) {
  if (zero_first) FT_CUDA_TRY(cudaMemsetAsync(amax_out, 0, sizeof(float), st));
  if (n == 0) return FT_OK;
  const int64_t n_vec = n / 8;
  const int n_tail = (int)(n % 8);
  int64_t blocks = ceil_div(n_vec, 2048);
  const int64_t cap = (int64_t)sm_count() * 6;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)blocks, 1, 1);
  cfg.blockDim = dim3(256, 1, 1);
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (!zero_first && pdl && pdl_enabled()) ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_amax, reinterpret_cast<const uint4*>(x_bf16), n_vec,
                                 reinterpret_cast<const uint16_t*>(x_bf16) + n_vec * 8, n_tail,
                                 reinterpret_cast<unsigned int*>(amax_out)));
  return FT_OK;
}

// ------------------------------------------------ clears with a programmatic edge
// Two buffers zeroed by one kernel launched with the programmatic-stream-serialization attribute: in
// a CUDA graph a memset node is a full dependency on both sides, this is a kernel that sets itself up
// while its predecessor drains and lets its successor do the same.  Sizes in bytes, multiples of 16.
__global__ void __launch_bounds__(256) k_clear2(uint4* a, int64_t na, uint4* b, int64_t nb) {
  pdl_wait();
  pdl_trigger();
  const int64_t nthr = (int64_t)gridDim.x * 256, me = (int64_t)blockIdx.x * 256 + threadIdx.x;
  for (int64_t i = me; i < na; i += nthr) a[i] = make_uint4(0, 0, 0, 0);
  for (int64_t i = me; i < nb; i += nthr) b[i] = make_uint4(0, 0, 0, 0);
}

int launch_clear2(void* a, size_t a_bytes, void* b, size_t b_bytes, cudaStream_t st) {
  const int64_t na = (int64_t)(a_bytes / 16), nb = (int64_t)(b_bytes / 16);
  int64_t blocks = ceil_div(na + nb, 256 * 4);
  if (blocks > 2 * sm_count()) blocks = 2 * sm_count();
  if (blocks < 1) blocks = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)blocks, 1, 1);
  cfg.blockDim = dim3(256, 1, 1);
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_clear2, reinterpret_cast<uint4*>(a), na, reinterpret_cast<uint4*>(b), nb));
  return FT_OK;
}

// ------------------------------------------- generic quantizer (a6, offline path)
// One thread per 16-element row segment.  BR = 16: the 16 lanes of a half-warp own
// the 16 rows of one 16x16 block and share its amax by shuffles.  BR = 1: 1x16 blocks.
template <int BR>
__global__ void __launch_bounds__(256) k_quantize_generic(
    const uint4* __restrict__ x, int64_t rows, int64_t cols, const float* __restrict__ amax_t,
    uint8_t* __restrict__ codes, uint8_t* __restrict__ sf, float* __restrict__ g_dec_out,
    int sf_layout) {
  const int64_t nblk = cols / 16;
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const TensorScale ts = tensor_scale(*amax_t);
  if (t == 0) *g_dec_out = ts.g_dec;
  int64_t row, bc;
  if (BR == 16) {
    const int64_t i = t % 16, blk = t / 16;
    bc = blk % nblk;
    row = (blk / nblk) * 16 + i;
  } else {
    bc = t % nblk;
    row = t / nblk;
  }
  const bool live = row < rows;  // rows % BR == 0, so a half-warp is live or dead as a whole
  uint4 v0 = make_uint4(0, 0, 0, 0), v1 = v0;
  if (live) {
    const uint4* p = x + (row * cols + bc * 16) / 8;
    v0 = __ldg(p);
    v1 = __ldg(p + 1);
  }
  float amax_b = fmaxf(amax_bf16x8(v0), amax_bf16x8(v1));
  if (BR == 16) {
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) amax_b = fmaxf(amax_b, __shfl_xor_sync(0xffffffffu, amax_b, o));
  }
  uint32_t sf8;
  float enc_b;
  block_scale(amax_b, ts, sf8, enc_b);
  if (!live) return;
  uint2 c;
  c.x = quant_bf16x8(v0, enc_b);
  c.y = quant_bf16x8(v1, enc_b);
  *reinterpret_cast<uint2*>(codes + row * (cols / 2) + bc * 8) = c;
  if (sf_layout == FT_SF_TILE128x4) {
    sf[sf_tile_offset(row, bc, nblk)] = (uint8_t)sf8;
  } else if (BR == 1 || (row % 16) == 0) {
    sf[(row / BR) * nblk + bc] = (uint8_t)sf8;
  }
}

// ------------------------------- stochastic rounding of the element codes (NEXT-4 variant, O-6')
// Philox4x32-10 (Salmon et al., SC'11): counter (c0..c3), key (k0, k1), ten rounds.  Written from the paper's
// round function; the oracle has its own copy (no shared code), both pinned by the published known answers.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}
// v -> the E2M1 neighbour below |v| or the one above, the latter iff u * (hi - lo) < |v| - lo with u = (word >> 8) *
// 2^-24; returned as a float on the grid carrying v's sign (the hardware convert then packs it exactly).  Every
// operation is exact in fp32: lo is |v| with all but the top mantissa bit cleared (the grid above 1 has one mantissa
// bit), hi - lo a power of two, |v| - lo within a factor of two of |v|.
__device__ __forceinline__ float e2m1_sr(float v, uint32_t word) {
  const float mag = fabsf(v);
  const uint32_t b = __float_as_uint(mag);
  const float u = __uint2float_rn(word >> 8) * 5.9604644775390625e-8f;   // 24 bits: exact
  float lo, step;
  if (mag >= 1.0f) {
    lo = __uint_as_float(b & 0xFFC00000u);
    step = __uint_as_float((b & 0x7F800000u) - 0x00800000u);
  } else {
    lo = mag >= 0.5f ? 0.5f : 0.0f;
    step = 0.5f;
  }
  const float r = (__fmul_rn(u, step) < __fsub_rn(mag, lo)) ? __fadd_rn(lo, step) : lo;   // >= 6 saturates in the convert
  return copysignf(r, v);
}

// One thread per 1x16 block: the scales exactly as in the nearest-rounding quantizer (Q3, Q4), the codes by
// e2m1_sr on x_i * enc_b with the uniform of element idx = row * cols + col: word idx % 4 of
// philox4x32_10(counter = offset + idx / 4, key = seed).
__global__ void __launch_bounds__(256) k_quantize_sr(
    const uint4* __restrict__ x, int64_t rows, int64_t cols, const float* __restrict__ amax_t,
    uint8_t* __restrict__ codes, uint8_t* __restrict__ sf, float* __restrict__ g_dec_out, int sf_layout,
    uint64_t seed, uint64_t offset) {
  const int64_t nblk = cols / 16;
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const TensorScale ts = tensor_scale(__ldg(amax_t));
  const int64_t bc = t % nblk, row = t / nblk;
  if (row >= rows) return;
  if (t == 0) *g_dec_out = ts.g_dec;
  const uint4* src = x + (row * cols + bc * 16) / 8;
  const uint4 v0 = __ldg(src), v1 = __ldg(src + 1);
  const float amax_b = fmaxf(amax_bf16x8(v0), amax_bf16x8(v1));
  uint32_t sf8;
  float enc_b;
  block_scale(amax_b, ts, sf8, enc_b);
  const uint32_t w[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
  const uint64_t ctr0 = offset + (uint64_t)(row * cols + bc * 16) / 4;
  const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
  uint32_t packed[2];
#pragma unroll
  for (int q = 0; q < 4; ++q) {       // four elements (two words of the block) per Philox call
    const uint64_t ctr = ctr0 + q;
    const uint4 rnd = philox4x32_10(make_uint4((uint32_t)ctr, (uint32_t)(ctr >> 32), 0u, 0u), key);
    const uint32_t wa = w[2 * q], wb = w[2 * q + 1];
    const float f0 = e2m1_sr(__fmul_rn(__uint_as_float(wa << 16), enc_b), rnd.x);
    const float f1 = e2m1_sr(__fmul_rn(__uint_as_float(wa & 0xFFFF0000u), enc_b), rnd.y);
    const float f2 = e2m1_sr(__fmul_rn(__uint_as_float(wb << 16), enc_b), rnd.z);
    const float f3 = e2m1_sr(__fmul_rn(__uint_as_float(wb & 0xFFFF0000u), enc_b), rnd.w);
    uint32_t two;
    asm("{\n\t.reg .b8 b0, b1;\n\t"
        "cvt.rn.satfinite.e2m1x2.f32 b0, %2, %1;\n\t"
        "cvt.rn.satfinite.e2m1x2.f32 b1, %4, %3;\n\t"
        "mov.b32 %0, {b0, b1, 0, 0};\n\t}"
        : "=r"(two) : "f"(f0), "f"(f1), "f"(f2), "f"(f3));
    if (q & 1) packed[q >> 1] |= two << 16;
    else packed[q >> 1] = two;
  }
  *reinterpret_cast<uint2*>(codes + row * (cols / 2) + bc * 8) = make_uint2(packed[0], packed[1]);
  if (sf_layout == FT_SF_TILE128x4) sf[sf_tile_offset(row, bc, nblk)] = (uint8_t)sf8;
  else sf[row * nblk + bc] = (uint8_t)sf8;
}

int launch_quantize_sr(const void* x, int64_t rows, int64_t cols, const float* amax_t, ft_qtensor* out,
                       uint64_t seed, uint64_t offset, cudaStream_t st) {
  const int64_t threads = rows * (cols / 16);
  if (out->sf_layout == FT_SF_TILE128x4)
    FT_CUDA_TRY(cudaMemsetAsync(out->sf, 0, ft_sf_bytes(rows, cols, 1, FT_SF_TILE128x4), st));
  k_quantize_sr<<<(unsigned)ceil_div(threads, 256), 256, 0, st>>>(reinterpret_cast<const uint4*>(x), rows, cols, amax_t,
                                                                  out->codes, out->sf, out->tensor_dec_scale,
                                                                  out->sf_layout, seed, offset);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

int launch_quantize_generic(const void* x, int64_t rows, int64_t cols, const float* amax_t,
                            ft_qtensor* out, cudaStream_t st) {
  const int64_t threads = rows * (cols / 16);
  const unsigned blocks = (unsigned)ceil_div(threads, 256);
  if (out->sf_layout == FT_SF_TILE128x4)
    FT_CUDA_TRY(cudaMemsetAsync(out->sf, 0, ft_sf_bytes(rows, cols, out->block_rows, FT_SF_TILE128x4), st));
  if (out->block_rows == 16)
    k_quantize_generic<16><<<blocks, 256, 0, st>>>(reinterpret_cast<const uint4*>(x), rows, cols,
                                                   amax_t, out->codes, out->sf,
                                                   out->tensor_dec_scale, out->sf_layout);
  else
    k_quantize_generic<1><<<blocks, 256, 0, st>>>(reinterpret_cast<const uint4*>(x), rows, cols,
                                                  amax_t, out->codes, out->sf,
                                                  out->tensor_dec_scale, out->sf_layout);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

// --------------------------------------------------------- a6: weight re-packing
// Q(R) [N x K/2 bytes] -> Q(R)^T [K x N/2 bytes]: a transposition of 4-bit elements (the same codes
// serve forward and backward; nothing is re-quantized).  Used offline by ft_pack_weight and, with single-copy weights
// (SURVEY NEXT-5), once per backward by ft_weight_transpose_codes, so it is written for the HBM roofline: a CTA
// moves a tile of 256 x 256 elements (32 KB); both its reads and its writes are whole 128-byte row pieces.
//   warp w, lane t: the 32 rows n = 32 w .. 32 w + 31, the word t of each (elements k = 8 t .. 8 t + 7): four 8x8
//   element blocks, each transposed in registers by three butterfly stages (PRMT for the 16- and 8-bit stages,
//   LOP3 for the 4-bit one); the lane then owns, for each of its 8 output rows k, 16 contiguous bytes (32 elements
//   n) -> one 16-byte store into the staged output tile, chunk index XOR (t & 7) against bank conflicts;
//   then every output row leaves as eight 16-byte pieces written by eight neighbouring lanes.
__device__ __forceinline__ void nibble_transpose8x8(uint32_t (&a)[8]) {
#pragma unroll
  for (int i = 0; i < 4; ++i) {   // swap the off-diagonal 4x4 blocks
    const uint32_t x = a[i], y = a[i + 4];
    a[i] = __byte_perm(x, y, 0x5410);
    a[i + 4] = __byte_perm(x, y, 0x7632);
  }
#pragma unroll
  for (int b = 0; b < 8; b += 4)
#pragma unroll
    for (int i = b; i < b + 2; ++i) {   // 2x2 blocks inside each 4x4
      const uint32_t x = a[i], y = a[i + 2];
      a[i] = __byte_perm(x, y, 0x6240);
      a[i + 2] = __byte_perm(x, y, 0x7351);
    }
#pragma unroll
  for (int i = 0; i < 8; i += 2) {     // single elements inside each 2x2
    const uint32_t x = a[i], y = a[i + 1];
    a[i] = (x & 0x0F0F0F0Fu) | ((y & 0x0F0F0F0Fu) << 4);
    a[i + 1] = ((x >> 4) & 0x0F0F0F0Fu) | (y & 0xF0F0F0F0u);
  }
}

__global__ void __launch_bounds__(256) k_transpose_codes(const uint8_t* __restrict__ src,
                                                         uint8_t* __restrict__ dst, int64_t N,
                                                         int64_t K) {
  __shared__ __align__(16) uint8_t tile[256 * 128];   // [k][n / 2], 16-byte chunks swizzled by (k >> 3) & 7
  const int64_t n0 = (int64_t)blockIdx.y * 256, k0 = (int64_t)blockIdx.x * 256;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool k_ok = k0 + lane * 8 < K;
  uint32_t out[8][4];
#pragma unroll
  for (int g = 0; g < 4; ++g) {        // 8x8 block g: rows n = 32 warp + 8 g + i
    uint32_t a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int64_t n = n0 + warp * 32 + g * 8 + i;
      a[i] = (k_ok && n < N) ? __ldg(reinterpret_cast<const uint32_t*>(src + n * (K / 2) + k0 / 2) + lane) : 0u;
    }
    nibble_transpose8x8(a);
#pragma unroll
    for (int j = 0; j < 8; ++j) out[j][g] = a[j];
  }
#pragma unroll
  for (int j = 0; j < 8; ++j)          // row k = 8 lane + j, chunk = warp (32 elements n each)
    *reinterpret_cast<uint4*>(tile + (lane * 8 + j) * 128 + ((warp ^ (lane & 7)) << 4)) =
        make_uint4(out[j][0], out[j][1], out[j][2], out[j][3]);
  __syncthreads();
  const int c = threadIdx.x & 7;
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const int k = it * 32 + (threadIdx.x >> 3);
    if (k0 + k < K && n0 + c * 32 < N)
      *reinterpret_cast<uint4*>(dst + (k0 + k) * (N / 2) + n0 / 2 + c * 16) =
          *reinterpret_cast<const uint4*>(tile + k * 128 + ((c ^ ((k >> 3) & 7)) << 4));
  }
}

int launch_transpose_codes(const uint8_t* src, uint8_t* dst, int64_t N, int64_t K, cudaStream_t st) {
  dim3 grid((unsigned)ceil_div(K, 256), (unsigned)ceil_div(N, 256));
  k_transpose_codes<<<grid, 256, 0, st>>>(src, dst, N, K);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

// Expand S[N/16][K/16] to per-row TILE128x4 scales for both orientations:
//   fwd  : rows n, blocks along K :  sf(n, kb) = S[n/16][kb]
//   dgrad: rows k, blocks along N :  sf(k, nb) = S[nb][k/16]
__global__ void __launch_bounds__(256) k_expand_sf(const uint8_t* __restrict__ S, int64_t N,
                                                   int64_t K, uint8_t* __restrict__ sf_fwd,
                                                   uint8_t* __restrict__ sf_bwd) {
  const int64_t nb16 = N / 16, kb16 = K / 16;
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (sf_fwd != nullptr && t < N * kb16) {
    const int64_t n = t / kb16, kb = t % kb16;
    sf_fwd[sf_tile_offset(n, kb, kb16)] = S[(n / 16) * kb16 + kb];
  }
  if (sf_bwd != nullptr && t < K * nb16) {
    const int64_t k = t / nb16, nb = t % nb16;
    sf_bwd[sf_tile_offset(k, nb, nb16)] = S[nb * kb16 + k / 16];
  }
}

// The scales of a weight operand [rows x cols] (16x16 blocks) cut to output tiles of `ntile` rows
// (ft_qtensor::sf_ntile): one thread per output byte.  transposed == 0: scale(row, kb) = S[row/16][kb] with S
// [rows/16][cols/16]; transposed == 1 (the dgrad operand, rows = K, cols = N): scale(row, nb) = S[nb][row/16]
// with S [cols/16][rows/16].
__global__ void __launch_bounds__(256) k_expand_sf_ntile(const uint8_t* __restrict__ S, int64_t rows, int64_t cols,
                                                         int ntile, int transposed, uint8_t* __restrict__ out) {
  const int64_t k64 = cols / 64, tiles = (rows + ntile - 1) / ntile;
  const int64_t total = tiles * k64 * 1024;
  const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= total) return;
  const int64_t grp = o / 512;                 // (nt * k64 + ks) * 2 + half
  const int within = (int)(o % 512);
  const int half = (int)(grp & 1);
  const int64_t ks = (grp >> 1) % k64, nt = (grp >> 1) / k64;
  const int l = within / 16, gi = (within % 16) / 4, c = within % 4;
  const int rt = half * 128 + gi * 32 + l;     // row inside the tile
  const int64_t row = nt * ntile + rt;
  uint8_t v = 0;
  if (rt < ntile && row < rows) {
    const int64_t kb = ks * 4 + c;
    v = transposed ? S[kb * (rows / 16) + row / 16] : S[(row / 16) * (cols / 16) + kb];
  }
  out[o] = v;
}

int launch_pack_weight(const ft_qtensor* rk, ft_qtensor* rk_tiled, ft_qtensor* rn,
                       cudaStream_t st) {
  const int64_t N = rk->rows, K = rk->cols;
  const int rc_t = launch_transpose_codes(rk->codes, rn->codes, N, K, st);
  if (rc_t != FT_OK) return rc_t;
  FT_CUDA_TRY(cudaMemsetAsync(rn->sf, 0, ft_sf_bytes(K, N, 16, FT_SF_TILE128x4), st));
  if (rk_tiled != nullptr)
    FT_CUDA_TRY(cudaMemsetAsync(rk_tiled->sf, 0, ft_sf_bytes(N, K, 16, FT_SF_TILE128x4), st));
  const int64_t tmax = (N * (K / 16) > K * (N / 16)) ? N * (K / 16) : K * (N / 16);
  k_expand_sf<<<(unsigned)ceil_div(tmax, 256), 256, 0, st>>>(
      rk->sf, N, K, rk_tiled ? rk_tiled->sf : nullptr, rn->sf);
  FT_CUDA_TRY(cudaGetLastError());
  if (rk_tiled != nullptr && rk_tiled->sf_ntile != nullptr && rk_tiled->ntile > 0) {
    const int64_t total = ceil_div(N, rk_tiled->ntile) * (K / 64) * 1024;
    k_expand_sf_ntile<<<(unsigned)ceil_div(total, 256), 256, 0, st>>>(rk->sf, N, K, rk_tiled->ntile, 0, rk_tiled->sf_ntile);
    FT_CUDA_TRY(cudaGetLastError());
  }
  if (rn->sf_ntile != nullptr && rn->ntile > 0) {
    const int64_t total = ceil_div(K, rn->ntile) * (N / 64) * 1024;
    k_expand_sf_ntile<<<(unsigned)ceil_div(total, 256), 256, 0, st>>>(rk->sf, K, N, rn->ntile, 1, rn->sf_ntile);
    FT_CUDA_TRY(cudaGetLastError());
  }
  FT_CUDA_TRY(cudaMemcpyAsync(rn->tensor_dec_scale, rk->tensor_dec_scale, sizeof(float),
                              cudaMemcpyDeviceToDevice, st));
  if (rk_tiled != nullptr && rk_tiled->tensor_dec_scale != rk->tensor_dec_scale &&
      rk_tiled->tensor_dec_scale != nullptr)
    FT_CUDA_TRY(cudaMemcpyAsync(rk_tiled->tensor_dec_scale, rk->tensor_dec_scale, sizeof(float),
                                cudaMemcpyDeviceToDevice, st));
  return FT_OK;
}

}  // namespace ft
