// gemm.cu -- a2 / a4: block-scaled 4-bit GEMM with the low-rank up-projection fused
// into the same accumulator:
//
//     out[m, n] = bf16( alpha * ( sum_k e_a[m,k] sf_a[m,k/16] e_b[n,k] sf_b[n,k/16]
//                                 + sum_j Hs[m,j] U[n,j] ) ),   alpha = g_dec_a * g_dec_b
//
// a: Q(X) or Q(G) [M x K], b: Q(R) [N x K] (K-major both), Hs = bf16(H * fl(1 / alpha)) [M x r_t],
// U [N x r_t] (O-10').  One persistent CTA per SM, warp-specialised:
//   warp 0   : TMA producer (codes by tensor map, scale tiles by 1-D bulk copy)
//   warp 1   : tcgen05 issuer -- tcgen05.cp (scales -> TMEM), tcgen05.mma
//              kind::mxf4nvf4 (K = 64 per instruction), then kind::f16 for the low-rank
//              chunks staged through the same ring; accumulator in TMEM
//   warp 2   : TMEM allocator
//   warps 4-7: epilogue -- tcgen05.ld, * alpha, bf16, global store
#include "common.cuh"
#include "../../include/fourtune_debug.h"

namespace ft {

constexpr int G_BM = 128;
constexpr int G_BK = 256;             // fp4 elements per stage = 128 bytes per row
constexpr int G_THREADS = 256;
constexpr int G_A_BYTES = G_BM * 128; // 16 KB
constexpr int G_SFA_BYTES = 4 * 512;  // four 128x4 scale tiles

template <int BN>
struct GemmCfg {
  static constexpr int B_BYTES = BN * 128;
  static constexpr int SFB_ROWT = (BN == 192) ? 2 : BN / 128;
  static constexpr int SFB_BYTES = SFB_ROWT * 4 * 512;
  static constexpr int STAGE_BYTES = G_A_BYTES + B_BYTES + G_SFA_BYTES + SFB_BYTES;
  static constexpr int STAGES = (BN == 256) ? 4 : (BN == 192 ? 4 : 6);
  static constexpr int ACC_STAGES = (2 * BN + 64 <= 512) ? 2 : 1;
  static constexpr int SF_COL = ACC_STAGES * BN;       // first TMEM column of the scale area
  static constexpr int SMEM = STAGES * STAGE_BYTES + 1024;
};

struct GemmParams {
  int64_t M, N, K;
  int r_t;
  const uint8_t* sfa;
  const uint8_t* sfb;
  const float* g_dec_a;
  const float* g_dec_b;
  __nv_bfloat16* out;
};

template <int BN>
__global__ void __launch_bounds__(G_THREADS, 1)
k_gemm4(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
        const __grid_constant__ CUtensorMap map_h, const __grid_constant__ CUtensorMap map_u,
        const GemmParams p) {
  using C = GemmCfg<BN>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[C::STAGES], empty_bar[C::STAGES];
  __shared__ uint64_t acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t tiles_m = (p.M + G_BM - 1) / G_BM, tiles_n = (p.N + BN - 1) / BN;
  const int64_t n_tiles = tiles_m * tiles_n;
  const int k4 = (int)((p.K + G_BK - 1) / G_BK);  // fp4 stages per tile
  const int klr = (p.r_t + 63) / 64;              // low-rank stages per tile
  const int kiters = k4 + klr;
  const int64_t sf_tiles_k = p.K / 64;            // 512-byte scale tiles per 128 rows
  const int64_t sfb_row_tiles = (p.N + 127) / 128;

  if (threadIdx.x == 0) {
    prefetch_tmap(&map_a);
    prefetch_tmap(&map_b);
    if (p.r_t > 0) {
      prefetch_tmap(&map_h);
      prefetch_tmap(&map_u);
    }
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(&acc_full[s], 1);
      mbar_init(&acc_empty[s], 4);
    }
    fence_mbar_init();
  }
  if (warp == 2) {
    tmem_alloc(&tmem_base_s, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    // ===================================================== TMA producer
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int64_t mt = tile % tiles_m, nt = tile / tiles_m;
        const int32_t m0 = (int32_t)(mt * G_BM), n0 = (int32_t)(nt * BN);
        const int64_t sfb_rt0 = n0 / 128;
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t* sa = smem + stage * C::STAGE_BYTES;
          uint8_t* sb = sa + G_A_BYTES;
          if (kt < k4) {
            const int atoms = (int)min((int64_t)4, sf_tiles_k - (int64_t)kt * 4);
            int rts = C::SFB_ROWT;
            if (sfb_rt0 + rts > sfb_row_tiles) rts = (int)(sfb_row_tiles - sfb_rt0);
            mbar_expect_tx(&full_bar[stage], G_A_BYTES + C::B_BYTES + atoms * 512 * (1 + rts));
            tma_load_2d(sa, &map_a, &full_bar[stage], kt * 128, m0);
            tma_load_2d(sb, &map_b, &full_bar[stage], kt * 128, n0);
            uint8_t* ssfa = sb + C::B_BYTES;
            uint8_t* ssfb = ssfa + G_SFA_BYTES;
            bulk_load_1d(ssfa, p.sfa + (mt * sf_tiles_k + (int64_t)kt * 4) * 512, atoms * 512,
                         &full_bar[stage]);
            for (int j = 0; j < rts; ++j)
              bulk_load_1d(ssfb + j * 2048, p.sfb + ((sfb_rt0 + j) * sf_tiles_k + (int64_t)kt * 4) * 512,
                           atoms * 512, &full_bar[stage]);
          } else {
            const int c0 = (kt - k4) * 64;
            mbar_expect_tx(&full_bar[stage], G_A_BYTES + C::B_BYTES);
            tma_load_2d(sa, &map_h, &full_bar[stage], c0, m0);
            tma_load_2d(sb, &map_u, &full_bar[stage], c0, n0);
          }
          if (++stage == C::STAGES) {
            stage = 0;
            phase ^= 1;
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer
    if (elect_one()) {
      constexpr uint32_t idesc4 = idesc_nvf4(G_BM, BN);
      constexpr uint32_t idesc16 = idesc_bf16(G_BM, BN);
      const uint32_t sfa_t = tmem_base + C::SF_COL;       // 16 columns: 4 per K=64 step
      const uint32_t sfb_t = tmem_base + C::SF_COL + 16;  // 32 columns: 8 per K=64 step
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int64_t nt = tile / tiles_m;
        const uint32_t sfb_shift = (uint32_t)(((nt * BN) % 128) / 32);  // BN = 192: odd tiles start mid scale tile
        mbar_wait(&acc_empty[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_t = tmem_base + acc * BN;
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * C::STAGE_BYTES);
          const uint32_t sb = sa + G_A_BYTES;
          if (kt < k4) {
            const int nk = (int)min((int64_t)4, sf_tiles_k - (int64_t)kt * 4);
            const uint32_t ssfa = sb + C::B_BYTES, ssfb = ssfa + G_SFA_BYTES;
            for (int k = 0; k < nk; ++k) {
              tc_cp_sf(sfa_t + 4 * k, make_smem_desc(ssfa + k * 512, 128, 0, 0));
#pragma unroll
              for (int j = 0; j < C::SFB_ROWT; ++j)
                tc_cp_sf(sfb_t + 8 * k + 4 * j, make_smem_desc(ssfb + j * 2048 + k * 512, 128, 0, 0));
            }
            for (int k = 0; k < nk; ++k) {
              mma_nvf4(d_t, make_smem_desc(sa + k * 32, 1024, 0, 2), make_smem_desc(sb + k * 32, 1024, 0, 2),
                       idesc4, sfa_t + 4 * k, sfb_t + 8 * k + sfb_shift, (kt | k) != 0);
            }
          } else {
            const int cols = min(64, p.r_t - (kt - k4) * 64);
            for (int k = 0; k < cols / 16; ++k)
              mma_bf16(d_t, make_smem_desc(sa + k * 32, 1024, 0, 2), make_smem_desc(sb + k * 32, 1024, 0, 2),
                       idesc16, 1u);
          }
          tc_commit(&empty_bar[stage]);
          if (kt == kiters - 1) tc_commit(&acc_full[acc]);
          if (++stage == C::STAGES) {
            stage = 0;
            phase ^= 1;
          }
        }
        if (++acc == C::ACC_STAGES) {
          acc = 0;
          acc_phase ^= 1;
        }
      }
    }
  } else if (warp >= 4) {
    // ===================================================== epilogue
    const int q = warp - 4;  // TMEM lane quarter this warp may read
    const float alpha = __fmul_rn(__ldg(p.g_dec_a), __ldg(p.g_dec_b));
    int acc = 0;
    uint32_t acc_phase = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      const int64_t mt = tile % tiles_m, nt = tile / tiles_m;
      const int64_t row = mt * G_BM + q * 32 + lane;
      const int64_t n0 = nt * BN;
      mbar_wait(&acc_full[acc], acc_phase);
      tc_fence_after();
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BN;
      __nv_bfloat16* orow = p.out + row * p.N + n0;
#pragma unroll 1
      for (int c = 0; c < BN / 32; ++c) {
        uint32_t v[32];
        tmem_ld32(t0 + c * 32, v);
        tmem_ld_wait();
        if (row < p.M && n0 + c * 32 < p.N) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            uint4 o;
            o.x = pack_bf16x2(__uint_as_float(v[8 * i + 0]) * alpha, __uint_as_float(v[8 * i + 1]) * alpha);
            o.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]) * alpha, __uint_as_float(v[8 * i + 3]) * alpha);
            o.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]) * alpha, __uint_as_float(v[8 * i + 5]) * alpha);
            o.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]) * alpha, __uint_as_float(v[8 * i + 7]) * alpha);
            *reinterpret_cast<uint4*>(orow + c * 32 + i * 8) = o;
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&acc_empty[acc]);
      if (++acc == C::ACC_STAGES) {
        acc = 0;
        acc_phase ^= 1;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

template <int BN>
static int launch_gemm4_bn(const CUtensorMap& ma, const CUtensorMap& mb, const CUtensorMap& mh,
                           const CUtensorMap& mu, const GemmParams& p, cudaStream_t st) {
  using C = GemmCfg<BN>;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_gemm4<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  const int64_t n_tiles = ceil_div(p.M, G_BM) * ceil_div(p.N, BN);
  const unsigned grid = (unsigned)(n_tiles < sm_count() ? n_tiles : sm_count());
  k_gemm4<BN><<<grid, G_THREADS, C::SMEM, st>>>(ma, mb, mh, mu, p);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

int launch_gemm4_pair(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                      const void* lr_a_scaled, const void* lr_b, int r_t, void* out_bf16, bool lr_late, cudaStream_t st);
int g_force_bn = 0;  // test/bench hook: 0 = CTA-pair kernel (default), else 1-CTA kernel with this N tile
extern int g_pair_bn;   // gemm_pair.cu: 0 = tile width chosen per shape, else forced

template <int BN>
static int setup_and_launch(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                            const void* lr_a, const void* lr_b, int r_t, void* out, cudaStream_t st) {
  CUtensorMap ma, mb, mh, mu;
  int rc = make_tensor_map_2d(&ma, a->codes, 1, (uint64_t)K / 2, (uint64_t)M, (uint64_t)K / 2, 128, G_BM,
                              Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&mb, b->codes, 1, (uint64_t)K / 2, (uint64_t)N, (uint64_t)K / 2, 128, BN,
                          Swizzle::B128);
  if (rc != FT_OK) return rc;
  if (r_t > 0) {
    rc = make_tensor_map_2d(&mh, lr_a, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, G_BM, Swizzle::B128);
    if (rc != FT_OK) return rc;
    rc = make_tensor_map_2d(&mu, lr_b, 2, (uint64_t)r_t, (uint64_t)N, (uint64_t)r_t * 2, 64, BN, Swizzle::B128);
    if (rc != FT_OK) return rc;
  } else {
    mh = ma;
    mu = mb;
  }
  GemmParams p;
  p.M = M;
  p.N = N;
  p.K = K;
  p.r_t = r_t;
  p.sfa = a->sf;
  p.sfb = b->sf;
  p.g_dec_a = a->tensor_dec_scale;
  p.g_dec_b = b->tensor_dec_scale;
  p.out = reinterpret_cast<__nv_bfloat16*>(out);
  return launch_gemm4_bn<BN>(ma, mb, mh, mu, p, st);
}

// lr_late: the launch directly follows k_finalize_h of the same call, which writes nothing the GEMM reads
// except lr_a_scaled: the pair kernel may start beside it (gemm_pair.cu); the 1-CTA kernels ignore it
int launch_gemm4(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                 const void* lr_a_scaled, const void* lr_b, int r_t, void* out_bf16, bool lr_late, cudaStream_t st) {
  const int bn = g_force_bn;
  if (bn == 0) return launch_gemm4_pair(a, b, M, N, K, lr_a_scaled, lr_b, r_t, out_bf16, lr_late, st);
  if (bn == 256) return setup_and_launch<256>(a, b, M, N, K, lr_a_scaled, lr_b, r_t, out_bf16, st);
  if (bn == 192) return setup_and_launch<192>(a, b, M, N, K, lr_a_scaled, lr_b, r_t, out_bf16, st);
  return setup_and_launch<128>(a, b, M, N, K, lr_a_scaled, lr_b, r_t, out_bf16, st);
}

}  // namespace ft

extern "C" int ft_debug_set_gemm_tile_n(int bn) {
  if (bn == 1224 || bn == 1240 || bn == 1256) {   // the CTA-pair kernel with a forced tile width
    ft::g_force_bn = 0;
    ft::g_pair_bn = bn - 1000;
    return FT_OK;
  }
  if (bn != 0 && bn != 128 && bn != 192 && bn != 256) return FT_ERR_INVALID_ARG;
  ft::g_force_bn = bn;
  ft::g_pair_bn = 0;
  return FT_OK;
}
