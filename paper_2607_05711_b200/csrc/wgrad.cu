// wgrad.cu -- a5: LoRA weight gradients (Eq. 4)
//     out[f, j] (+)= sum_m In[m, f] * L[m, r_s + j]        f < F, j < r
// used twice: dA = X^T (G B^T) with In = X, L = P;  dB^T = G^T (X A) with In = G, L = H.
// HBM-bound: In is read exactly once.  A CTA owns 128 features x one slice of M and walks it in
// 64-row chunks that TMA stages (SWIZZLE_128B) through an mbarrier ring.  One thread issues
// tcgen05.mma kind::f16 (M = 128 features, N = r, K = 16 rows, four per chunk) with BOTH
// operands MN-major -- the staged chunks are used as they lie in memory, nothing is transposed
// by the SM -- into a TMEM accumulator; four warps drain it and combine the M slices with
// fp32 vector red.global.add.
#include "common.cuh"

namespace ft {

constexpr int WG_F = 128;
constexpr int WG_MC = 64;
constexpr int WG_STAGES = 4;
constexpr int WG_THREADS = 128;
constexpr int WG_IN_BYTES = 2 * WG_MC * 128;  // two 64-feature boxes
constexpr int WG_LG_BYTES = WG_MC * 128;      // one 64-column group of L

struct WgParams {
  int64_t M, F;
  int r_s, r;
  int chunks_per_cta;
  float* out;
};

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
               : "memory");
}

template <int R>
__global__ void __launch_bounds__(WG_THREADS, 2)
k_wgrad(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_l,
        const WgParams p) {
  constexpr int NG = (R + 63) / 64;
  constexpr int STAGE_BYTES = WG_IN_BYTES + NG * WG_LG_BYTES;
  constexpr uint32_t TMEM_COLS = R <= 32 ? 32 : (R <= 64 ? 64 : 128);
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[WG_STAGES], empty_bar[WG_STAGES], acc_bar;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t f0 = (int32_t)blockIdx.x * WG_F;
  const int64_t chunks_total = (p.M + WG_MC - 1) / WG_MC;
  const int64_t c_begin = (int64_t)blockIdx.y * p.chunks_per_cta;
  int n_chunks = (int)min((int64_t)p.chunks_per_cta, chunks_total - c_begin);
  if (n_chunks < 0) n_chunks = 0;

  if (tid == 0) {
    prefetch_tmap(&map_in);
    prefetch_tmap(&map_l);
    for (int s = 0; s < WG_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
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

  if (warp == 0) {
    if (elect_one()) {   // ---- TMA producer
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WG_STAGES;
        mbar_wait(&empty_bar[s], ((it / WG_STAGES) & 1) ^ 1);
        uint8_t* base = smem + s * STAGE_BYTES;
        const int32_t m0 = (int32_t)((c_begin + it) * WG_MC);
        mbar_expect_tx(&full_bar[s], STAGE_BYTES);
        tma_load_2d(base, &map_in, &full_bar[s], f0, m0);
        tma_load_2d(base + WG_MC * 128, &map_in, &full_bar[s], f0 + 64, m0);
#pragma unroll
        for (int g = 0; g < NG; ++g)
          tma_load_2d(base + WG_IN_BYTES + g * WG_LG_BYTES, &map_l, &full_bar[s], p.r_s + g * 64, m0);
      }
    }
  } else if (warp == 1) {
    if (elect_one()) {   // ---- MMA issuer: acc[128 f x R] += In[64 m, 128 f]^T * L[64 m, R]
      constexpr uint32_t idesc = idesc_bf16(WG_F, R) | (1u << 15) | (1u << 16);  // A and B MN-major
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WG_STAGES;
        mbar_wait(&full_bar[s], (it / WG_STAGES) & 1);
        tc_fence_after();
        const uint32_t in_u = smem_u32(smem + s * STAGE_BYTES);
        const uint32_t l_u = in_u + WG_IN_BYTES;
#pragma unroll
        for (int k = 0; k < 4; ++k)   // 16 rows of m per MMA = two 8-row swizzle groups = 2048 bytes
          mma_bf16(tmem_base, make_smem_desc(in_u + k * 2048, 1024, WG_MC * 128, 2),
                   make_smem_desc(l_u + k * 2048, 1024, WG_LG_BYTES, 2), idesc, (it | k) != 0);
        tc_commit(&empty_bar[s]);
      }
      tc_commit(&acc_bar);
    }
  }
  __syncwarp();

  if (n_chunks > 0) {   // ---- drain: thread = feature (TMEM lane), R fp32 columns
    mbar_wait(&acc_bar, 0);
    tc_fence_after();
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
#pragma unroll
        for (int j = 0; j < 16; j += 4)
          red_add_v4(o + j, __uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]),
                     __uint_as_float(v[j + 3]));
      }
    }
    tc_fence_before();
  }
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, TMEM_COLS);
  }
}

template <int R>
static int launch_wg(const CUtensorMap& mi, const CUtensorMap& ml, const WgParams& p, unsigned gy,
                     cudaStream_t st) {
  constexpr int NG = (R + 63) / 64;
  const int smem = WG_STAGES * (WG_IN_BYTES + NG * WG_LG_BYTES) + 1024;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  dim3 grid((unsigned)ceil_div(p.F, WG_F), gy, 1);
  k_wgrad<R><<<grid, WG_THREADS, smem, st>>>(mi, ml, p);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

int launch_wgrad(const void* in_bf16, int64_t M, int64_t F, const void* lr_bf16, int r_t, int r_s, int r,
                 float* out, cudaStream_t st) {
  CUtensorMap mi, ml;
  int rc = make_tensor_map_2d(&mi, in_bf16, 2, (uint64_t)F, (uint64_t)M, (uint64_t)F * 2, 64, WG_MC,
                              Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&ml, lr_bf16, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, WG_MC,
                          Swizzle::B128);
  if (rc != FT_OK) return rc;
  const int64_t f_tiles = ceil_div(F, WG_F), chunks = ceil_div(M, WG_MC);
  // M slices: about two resident CTAs per SM, at least 4 chunks per slice
  int64_t slices = ceil_div((int64_t)2 * sm_count(), f_tiles);
  if (slices > chunks / 4) slices = chunks / 4;
  if (slices < 1) slices = 1;
  WgParams p;
  p.M = M;
  p.F = F;
  p.r_s = r_s;
  p.r = r;
  p.chunks_per_cta = (int)ceil_div(chunks, slices);
  p.out = out;
  const unsigned gy = (unsigned)ceil_div(chunks, p.chunks_per_cta);
  switch (r) {
    case 16: return launch_wg<16>(mi, ml, p, gy, st);
    case 32: return launch_wg<32>(mi, ml, p, gy, st);
    case 48: return launch_wg<48>(mi, ml, p, gy, st);
    case 64: return launch_wg<64>(mi, ml, p, gy, st);
    case 80: return launch_wg<80>(mi, ml, p, gy, st);
    case 96: return launch_wg<96>(mi, ml, p, gy, st);
    case 112: return launch_wg<112>(mi, ml, p, gy, st);
    case 128: return launch_wg<128>(mi, ml, p, gy, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
