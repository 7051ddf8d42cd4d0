// wgrad.cu -- a5: LoRA weight gradients (Eq. 4)
//     out[f, j] (+)= sum_m In[m, f] * L[m, r_s + j]        f < F, j < r
// used twice: dA = X^T (G B^T) with In = X, L = P;  dB^T = G^T (X A) with In = G, L = H.
// HBM-bound (reads In once).  A CTA owns 128 features x one slice of M and walks it in
// 64-row chunks staged by TMA (SWIZZLE_128B, 4-deep ring); 8 warps x 16 features run
// mma.sync m16n8k16 with A taken transposed from the staged chunk (ldmatrix.trans);
// slices are combined with fp32 red.global.add.
#include "common.cuh"

namespace ft {

constexpr int WG_F = 128;
constexpr int WG_MC = 64;
constexpr int WG_STAGES = 4;
constexpr int WG_THREADS = 256;
constexpr int WG_IN_BYTES = 2 * WG_MC * 128;  // two 64-feature boxes
constexpr int WG_LG_BYTES = WG_MC * 128;      // one 64-column group of L

struct WgParams {
  int64_t M, F;
  int r_s, r;
  int chunks_per_cta;
  float* out;
};

__device__ __forceinline__ void wg_ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                             uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void wg_mma(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                       uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, "
      "{%8, %9}, {%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

template <int R>
__global__ void __launch_bounds__(WG_THREADS, 1)
k_wgrad(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_l,
        const WgParams p) {
  constexpr int NG = (R + 63) / 64;
  constexpr int NT = R / 8;
  constexpr int STAGE_BYTES = WG_IN_BYTES + NG * WG_LG_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[WG_STAGES];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t f0 = (int32_t)blockIdx.x * WG_F;
  const int64_t chunks_total = (p.M + WG_MC - 1) / WG_MC;
  const int64_t c_begin = (int64_t)blockIdx.y * p.chunks_per_cta;
  int n_chunks = (int)min((int64_t)p.chunks_per_cta, chunks_total - c_begin);
  if (n_chunks < 0) n_chunks = 0;

  if (tid == 0) {
    prefetch_tmap(&map_in);
    prefetch_tmap(&map_l);
    for (int s = 0; s < WG_STAGES; ++s) mbar_init(&full_bar[s], 1);
    fence_mbar_init();
  }
  __syncthreads();
  auto issue = [&](int it) {
    const int s = it % WG_STAGES;
    uint8_t* base = smem + s * STAGE_BYTES;
    const int32_t m0 = (int32_t)((c_begin + it) * WG_MC);
    mbar_expect_tx(&full_bar[s], STAGE_BYTES);
    tma_load_2d(base, &map_in, &full_bar[s], f0, m0);
    tma_load_2d(base + WG_MC * 128, &map_in, &full_bar[s], f0 + 64, m0);
#pragma unroll
    for (int g = 0; g < NG; ++g)
      tma_load_2d(base + WG_IN_BYTES + g * WG_LG_BYTES, &map_l, &full_bar[s], p.r_s + g * 64, m0);
  };
  if (tid == 0)
    for (int it = 0; it < WG_STAGES && it < n_chunks; ++it) issue(it);

  float acc[NT][4];
#pragma unroll
  for (int j = 0; j < NT; ++j) acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f;
  // warp -> features [16*warp, 16*warp+16): box = warp / 4, 16-byte chunks 2*(warp%4), +1
  const int box = warp >> 2, fc = (warp & 3) * 2;

  for (int it = 0; it < n_chunks; ++it) {
    const int s = it % WG_STAGES;
    mbar_wait(&full_bar[s], (it / WG_STAGES) & 1);
    const uint32_t in_u = smem_u32(smem + s * STAGE_BYTES) + box * (WG_MC * 128);
    const uint32_t l_u = smem_u32(smem + s * STAGE_BYTES) + WG_IN_BYTES;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      uint32_t a0, a1, a2, a3;
      {
        const int i = lane >> 3;
        const int mr = ks * 16 + (lane & 7) + (i >> 1) * 8;
        const int c = fc + (i & 1);
        wg_ldsm_x4_t(in_u + mr * 128 + ((c ^ (mr & 7)) << 4), a0, a1, a2, a3);
      }
#pragma unroll
      for (int j = 0; j < NT; j += 2) {
        const int kr = ks * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int nt = j + (lane >> 4);
        uint32_t b0, b1, b2, b3;
        wg_ldsm_x4_t(l_u + (nt >> 3) * WG_LG_BYTES + kr * 128 + (((nt & 7) ^ (kr & 7)) << 4), b0, b1, b2, b3);
        wg_mma(acc[j], a0, a1, a2, a3, b0, b1);
        if (j + 1 < NT) wg_mma(acc[j + 1], a0, a1, a2, a3, b2, b3);
      }
    }
    __syncthreads();
    if (tid == 0 && it + WG_STAGES < n_chunks) issue(it + WG_STAGES);
  }

  if (n_chunks > 0) {
    const int g = lane >> 2, t = lane & 3;
    const int64_t f = (int64_t)f0 + warp * 16 + g;
#pragma unroll
    for (int j = 0; j < NT; ++j) {
      const int c = j * 8 + 2 * t;
      if (f < p.F) {
        atomicAdd(p.out + f * R + c, acc[j][0]);
        atomicAdd(p.out + f * R + c + 1, acc[j][1]);
      }
      if (f + 8 < p.F) {
        atomicAdd(p.out + (f + 8) * R + c, acc[j][2]);
        atomicAdd(p.out + (f + 8) * R + c + 1, acc[j][3]);
      }
    }
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
  // M slices: about two waves of CTAs, at least 4 chunks per slice
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
    case 8: return launch_wg<8>(mi, ml, p, gy, st);
    case 16: return launch_wg<16>(mi, ml, p, gy, st);
    case 32: return launch_wg<32>(mi, ml, p, gy, st);
    case 48: return launch_wg<48>(mi, ml, p, gy, st);
    case 64: return launch_wg<64>(mi, ml, p, gy, st);
    case 96: return launch_wg<96>(mi, ml, p, gy, st);
    case 128: return launch_wg<128>(mi, ml, p, gy, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
