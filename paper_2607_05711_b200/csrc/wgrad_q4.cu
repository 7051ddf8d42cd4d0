// wgrad_q4.cu -- a5 with 4-bit saved activations (O-12'):
//     dA[f, j] (+)= g_dec * sum_m ( E2M1(code[m, f]) * sf[m, f/16] ) * P[m, r_s + j]
// Eq. 4 with the X of dA = X^T (G B^T) taken as dequant(Q(X)): the codes and scales
// that ft_linear_fwd produced anyway are what the layer keeps for backward (0.5625 instead of 2 bytes
// per activation element; the activation side of PAPER.md:197-207).  Same skeleton as k_wgrad (wgrad.cu):
// a CTA owns 128 features x one slice of M, walks it in 64-row chunks, one thread issues four
// tcgen05.mma kind::f16 per chunk with both operands MN-major into a TMEM accumulator.  The difference is
// where the A operand comes from: TMA stages the chunk's codes (64 rows x 64 bytes) and its two 512-byte
// scale tiles; eight warps expand them to bf16 in the swizzled layout the MMA reads.  E2M1 x E4M3 has at
// most six significant bits, so e2m1 * sf is EXACT in f16 and in bf16: the dequantizer rounds nothing,
// and the tensor scale g_dec is one fp32 multiply on the drained accumulator.
#include <cuda_fp16.h>

#include "common.cuh"

namespace ft {

int launch_clear2(void* a, size_t a_bytes, void* b, size_t b_bytes, cudaStream_t st);

constexpr int WQ_F = 128;
constexpr int WQ_MC = 64;
constexpr int WQ_STAGES = 3;
constexpr int WQ_THREADS = 384;                // warp 0 TMA, 1 MMA, 2 TMEM owner, 4-11 dequantize
constexpr int WQ_IN_BYTES = 2 * WQ_MC * 128;   // two 64-feature boxes of bf16
constexpr int WQ_LG_BYTES = WQ_MC * 128;       // one 64-column group of P
constexpr int WQ_CODE_BYTES = WQ_MC * 64;      // 64 rows x 128 fp4
constexpr int WQ_SF_BYTES = 1024;              // two 128-row x 4-block scale tiles

struct WqParams {
  int64_t M, F;
  int r_s;
  int chunks_per_cta;
  int direct;
  int late_wait;              // 1: everything this kernel reads or clears was complete before its predecessor
                              //    triggered (see launch_wgrad_q4): run beside the predecessor and wait for
                              //    it at the END, so that "this kernel is complete" still implies "everything
                              //    before it in the stream is complete" for whatever is launched next
  int64_t sf_tiles_per_row;   // ceil(F / 64)
  const uint8_t* sf;          // FT_SF_TILE128x4
  const float* g_dec;
  float* out;
};

__device__ __forceinline__ void red_add_v4_q(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
               : "memory");
}

// two E2M1 codes (one byte, element 2j in bits 0-3) -> f16x2, low half = element 2j
__device__ __forceinline__ uint32_t e2m1x2_to_f16x2(uint32_t byte) {
  uint32_t d;
  asm("{\n\t.reg .b8 lo, hi;\n\t.reg .b16 t;\n\t"
      "cvt.u16.u32 t, %1;\n\t"
      "mov.b16 {lo, hi}, t;\n\t"
      "cvt.rn.f16x2.e2m1x2 %0, lo;\n\t}"
      : "=r"(d)
      : "r"(byte));
  return d;
}
// one E4M3 byte -> the same value in both halves of an f16x2
__device__ __forceinline__ uint32_t e4m3_to_f16x2_bcast(uint32_t byte) {
  uint32_t d;
  const uint16_t two = (uint16_t)(byte | (byte << 8));
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(d) : "h"(two));
  return d;
}
// f16x2 -> bf16x2 (exact for the values here)
__device__ __forceinline__ uint32_t f16x2_to_bf16x2(uint32_t h2) {
  const __half2 h = *reinterpret_cast<const __half2*>(&h2);
  const float lo = __low2float(h), hi = __high2float(h);
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

template <int R>
__global__ void __launch_bounds__(WQ_THREADS, 2)
k_wgrad_q4(const __grid_constant__ CUtensorMap map_codes, const __grid_constant__ CUtensorMap map_l,
           const WqParams p) {
  constexpr int NG = (R + 63) / 64;
  constexpr int STAGE_BYTES = WQ_IN_BYTES + NG * WQ_LG_BYTES + WQ_CODE_BYTES + WQ_SF_BYTES;
  constexpr int RAW_OFF = WQ_IN_BYTES + NG * WQ_LG_BYTES;
  constexpr uint32_t TMEM_COLS = R <= 32 ? 32 : (R <= 64 ? 64 : 128);
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t raw_bar[WQ_STAGES], cvt_bar[WQ_STAGES], empty_bar[WQ_STAGES], acc_bar;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t f0 = (int32_t)blockIdx.x * WQ_F;
  const int64_t chunks_total = (p.M + WQ_MC - 1) / WQ_MC;
  const int64_t c_begin = (int64_t)blockIdx.y * p.chunks_per_cta;
  int n_chunks = (int)min((int64_t)p.chunks_per_cta, chunks_total - c_begin);
  if (n_chunks < 0) n_chunks = 0;
  const bool two_tiles = (int64_t)f0 + 64 < p.F;

  if (tid == 0) {
    prefetch_tmap(&map_codes);
    prefetch_tmap(&map_l);
    for (int s = 0; s < WQ_STAGES; ++s) {
      mbar_init(&raw_bar[s], 1);
      mbar_init(&cvt_bar[s], 8);     // one arrival per dequantizer warp
      mbar_init(&empty_bar[s], 1);   // MMA commit
    }
    mbar_init(&acc_bar, 1);
    fence_mbar_init();
  }
  if (warp == 2) {
    tmem_alloc(&tmem_base_s, TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  if (!p.late_wait) pdl_wait();   // P and Q(X) come from kernels before this one (no-op without a programmatic edge)
  pdl_trigger();

  if (warp == 0) {
    if (elect_one()) {   // ---- TMA producer: codes, scale tiles, P
      const uint32_t sf_bytes = two_tiles ? 1024u : 512u;
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WQ_STAGES;
        mbar_wait(&empty_bar[s], ((it / WQ_STAGES) & 1) ^ 1);
        uint8_t* base = smem + s * STAGE_BYTES;
        const int64_t m0 = (c_begin + it) * WQ_MC;
        mbar_expect_tx(&raw_bar[s], WQ_CODE_BYTES + sf_bytes + NG * WQ_LG_BYTES);
        tma_load_2d(base + RAW_OFF, &map_codes, &raw_bar[s], f0 / 2, (int32_t)m0);
        bulk_load_1d(base + RAW_OFF + WQ_CODE_BYTES,
                     p.sf + ((m0 / 128) * p.sf_tiles_per_row + f0 / 64) * 512, sf_bytes, &raw_bar[s]);
#pragma unroll
        for (int g = 0; g < NG; ++g)
          tma_load_2d(base + WQ_IN_BYTES + g * WQ_LG_BYTES, &map_l, &raw_bar[s], p.r_s + g * 64, (int32_t)m0);
      }
    }
  } else if (warp == 1) {
    if (elect_one()) {   // ---- MMA issuer: acc[128 f x R] += Xq[64 m, 128 f]^T * P[64 m, R]
      constexpr uint32_t idesc = idesc_bf16(WQ_F, R) | (1u << 15) | (1u << 16);  // A and B MN-major
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WQ_STAGES;
        mbar_wait(&raw_bar[s], (it / WQ_STAGES) & 1);   // P landed
        mbar_wait(&cvt_bar[s], (it / WQ_STAGES) & 1);   // A expanded
        tc_fence_after();
        const uint32_t in_u = smem_u32(smem + s * STAGE_BYTES);
        const uint32_t l_u = in_u + WQ_IN_BYTES;
#pragma unroll
        for (int k = 0; k < 4; ++k)
          mma_bf16(tmem_base, make_smem_desc(in_u + k * 2048, 1024, WQ_MC * 128, 2),
                   make_smem_desc(l_u + k * 2048, 1024, WQ_LG_BYTES, 2), idesc, (it | k) != 0);
        tc_commit(&empty_bar[s]);
      }
      tc_commit(&acc_bar);
    }
  } else if (warp >= 4) {
    // ---- dequantizer: thread = one 1x16 block at a time, two per chunk.  Eight consecutive threads
    // cover one row's 128 features, a warp four rows.
    const int t = tid - 128;
    for (int it = 0; it < n_chunks; ++it) {
      const int s = it % WQ_STAGES;
      mbar_wait(&raw_bar[s], (it / WQ_STAGES) & 1);
      uint8_t* base = smem + s * STAGE_BYTES;
      const uint8_t* codes = base + RAW_OFF;
      const uint8_t* sft = codes + WQ_CODE_BYTES;
      const int64_t m0 = (c_begin + it) * WQ_MC;
      const int half = (int)((m0 >> 6) & 1);   // which 64 rows of the 128-row scale tile
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int q = i * 256 + t;
        const int row = q >> 3, b = q & 7;
        uint32_t w[8];
        // rows beyond M and features beyond F: zeros (their scale bytes are not defined)
        if (m0 + row < p.M && (int64_t)f0 + b * 16 < p.F) {
          const uint2 c = *reinterpret_cast<const uint2*>(codes + row * 64 + b * 8);
          const uint32_t sfb = sft[(b >> 2) * 512 + (row & 31) * 16 + (half * 2 + (row >> 5)) * 4 + (b & 3)];
          const uint32_t sf2 = e4m3_to_f16x2_bcast(sfb);
          const __half2 sfh = *reinterpret_cast<const __half2*>(&sf2);
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const uint32_t byte = ((j < 4 ? c.x : c.y) >> ((j & 3) * 8)) & 0xFFu;
            const uint32_t v2 = e2m1x2_to_f16x2(byte);
            const __half2 pr = __hmul2(*reinterpret_cast<const __half2*>(&v2), sfh);   // exact
            w[j] = f16x2_to_bf16x2(*reinterpret_cast<const uint32_t*>(&pr));
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) w[j] = 0u;
        }
        // SWIZZLE_128B: 16-byte unit u of row `row` lives at unit u ^ (row % 8)
        uint8_t* dst = base + (b >> 2) * (WQ_MC * 128) + row * 128;
        const int u0 = (b & 3) * 2;
        *reinterpret_cast<uint4*>(dst + ((u0 ^ (row & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
        *reinterpret_cast<uint4*>(dst + (((u0 + 1) ^ (row & 7)) << 4)) = make_uint4(w[4], w[5], w[6], w[7]);
      }
      fence_proxy_async();   // generic-proxy stores -> visible to the tensor core's reads
      __syncwarp();
      if (lane == 0) mbar_arrive(&cvt_bar[s]);
    }
  }
  __syncwarp();

  if (warp < 4 && n_chunks > 0) {   // ---- drain: thread = feature (TMEM lane), R fp32 columns, x g_dec
    mbar_wait(&acc_bar, 0);
    tc_fence_after();
    const float g_dec = *p.g_dec;
    const int64_t f = (int64_t)f0 + warp * 32 + lane;
#pragma unroll
    for (int c0 = 0; c0 < R; c0 += 16) {
      uint32_t v[16];
      asm volatile(
          "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
          "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
          : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
            "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
          : "r"(tmem_base + ((uint32_t)(warp * 32) << 16) + c0)
          : "memory");
      tmem_ld_wait();
      if (f < p.F) {
        float* o = p.out + f * R + c0;
        float x[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) x[j] = __fmul_rn(__uint_as_float(v[j]), g_dec);
        if (p.direct) {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<float4*>(o + j) = make_float4(x[j], x[j + 1], x[j + 2], x[j + 3]);
        } else {
#pragma unroll
          for (int j = 0; j < 16; j += 4) red_add_v4_q(o + j, x[j], x[j + 1], x[j + 2], x[j + 3]);
        }
      }
    }
    tc_fence_before();
  }
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, TMEM_COLS);
  }
  if (p.late_wait) pdl_wait();
}

template <int R>
static int launch_wq(const CUtensorMap* maps, const WqParams& p, dim3 grid, bool pdl, cudaStream_t st) {
  constexpr int NG = (R + 63) / 64;
  const int smem = WQ_STAGES * (WQ_IN_BYTES + NG * WQ_LG_BYTES + WQ_CODE_BYTES + WQ_SF_BYTES) + 1024;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad_q4<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  // two CTAs per SM need the largest carveout (the default one fits a single CTA of this size)
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad_q4<R>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                   cudaSharedmemCarveoutMaxShared));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(WQ_THREADS, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (pdl && pdl_enabled()) ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_wgrad_q4<R>, maps[0], maps[1], p));
  return FT_OK;
}

// dA [K x r] (+)= dequant(Q(X))^T P[:, r_s:].  codes [M x K/2], sf FT_SF_TILE128x4 over [M x K/16],
// g_dec device float.  accumulate == 0 and a single M slice: plain stores; otherwise dA is cleared by
// a small kernel first (accumulate == 0) and the slices combine with fp32 reductions.
// beside_prev: the launch directly follows a kernel of the same call that (a) neither writes anything
// this kernel touches nor reads dA and (b) passes griddepcontrol.wait in every CTA before it triggers its
// dependents -- then all earlier work of the stream is complete when this kernel starts; it fills the SMs as
// that kernel's CTAs retire and waits for it only before it exits (every CTA of the predecessor is
// resident by then, so the wait cannot deadlock).
int launch_wgrad_q4(const uint8_t* codes, const uint8_t* sf, const float* g_dec, int64_t M, int64_t K,
                    const void* p_saved, int r_t, int r_s, int r, float* dA, int accumulate, bool beside_prev,
                    cudaStream_t st) {
  CUtensorMap maps[2];
  int rc = make_tensor_map_2d(&maps[0], codes, 1, (uint64_t)K / 2, (uint64_t)M, (uint64_t)K / 2, 64, WQ_MC,
                              Swizzle::None);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&maps[1], p_saved, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, WQ_MC,
                          Swizzle::B128);
  if (rc != FT_OK) return rc;
  const int64_t chunks = ceil_div(M, WQ_MC);
  const int64_t f_tiles = ceil_div(K, WQ_F);
  int64_t slices = (int64_t)2 * sm_count() / f_tiles;   // one wave of two resident CTAs per SM
  if (slices > chunks / 4) slices = chunks / 4;   // at least 4 chunks (256 rows) per slice
  if (slices < 1) slices = 1;
  WqParams p;
  p.M = M;
  p.F = K;
  p.r_s = r_s;
  p.chunks_per_cta = (int)ceil_div(chunks, slices);
  const unsigned sl = (unsigned)ceil_div(chunks, p.chunks_per_cta);
  p.direct = (sl == 1 && !accumulate) ? 1 : 0;
  p.sf_tiles_per_row = ceil_div(K, 64);
  p.sf = sf;
  p.g_dec = g_dec;
  p.out = dA;
  bool pdl = beside_prev && accumulate != 0;
  p.late_wait = pdl ? 1 : 0;
  if (!accumulate && !p.direct) {
    rc = launch_clear2(dA, (size_t)K * r * sizeof(float), nullptr, 0, st);
    if (rc != FT_OK) return rc;
    pdl = true;
  }
  const dim3 grid((unsigned)f_tiles, sl, 1);
  switch (r) {
    case 16: return launch_wq<16>(maps, p, grid, pdl, st);
    case 32: return launch_wq<32>(maps, p, grid, pdl, st);
    case 48: return launch_wq<48>(maps, p, grid, pdl, st);
    case 64: return launch_wq<64>(maps, p, grid, pdl, st);
    case 80: return launch_wq<80>(maps, p, grid, pdl, st);
    case 96: return launch_wq<96>(maps, p, grid, pdl, st);
    case 112: return launch_wq<112>(maps, p, grid, pdl, st);
    case 128: return launch_wq<128>(maps, p, grid, pdl, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
