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

int launch_clear2(void* a, size_t a_bytes, void* b, size_t b_bytes, cudaStream_t st);

constexpr int WG_F = 128;
constexpr int WG_MC = 64;
constexpr int WG_STAGES = 4;
constexpr int WG_THREADS = 128;
constexpr int WG_IN_BYTES = 2 * WG_MC * 128;  // two 64-feature boxes
constexpr int WG_LG_BYTES = WG_MC * 128;      // one 64-column group of L

struct WgParams {      // two problems in one launch: [0] dA = X^T P_lora, [1] dB^T = G^T H_lora
  int64_t M;
  int64_t F[2];
  int r_s, r;
  int chunks_per_cta[2];
  int direct[2];       // 1: a single M slice owns the output, plain stores (no zero-fill needed)
  float* out[2];
  unsigned int* amax_bits[2];   // non-null: atomicMax target for max |In| (bf16 bits << 16), pre-zeroed
  int late_wait;                // 1: nothing this launch touches depends on its predecessor, which passes
                                //    griddepcontrol.wait in every CTA before triggering: start beside it and
                                //    wait for it at the END (completion stays transitive for the next launch)
  float4* zero_fill;            // non-null: buffer this launch clears for a LATER launch (zero_fill_n4 float4s)
  int64_t zero_fill_n4;
};

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
               : "memory");
}

template <int R>
__global__ void __launch_bounds__(WG_THREADS, 2)
k_wgrad(const __grid_constant__ CUtensorMap map_in0, const __grid_constant__ CUtensorMap map_l0,
        const __grid_constant__ CUtensorMap map_in1, const __grid_constant__ CUtensorMap map_l1,
        const WgParams p) {
  const int z = blockIdx.z;
  if (p.zero_fill != nullptr) {   // grid-stride clear, every CTA of the launch (before any early return)
    pdl_wait();                   // launched with a programmatic edge: nothing is written before the predecessor ends
    const int64_t nthr = (int64_t)gridDim.x * gridDim.y * gridDim.z * WG_THREADS;
    const int64_t me = ((int64_t)(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * WG_THREADS + threadIdx.x;
    for (int64_t i = me; i < p.zero_fill_n4; i += nthr) p.zero_fill[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const CUtensorMap& map_in = z == 0 ? map_in0 : map_in1;
  const CUtensorMap& map_l = z == 0 ? map_l0 : map_l1;
  const int64_t F = p.F[z];
  const int cpc = p.chunks_per_cta[z];
  // CTAs beyond this problem's feature tiles or M slices have nothing to do (uniform per CTA)
  if ((int64_t)blockIdx.x * WG_F >= F || (int64_t)blockIdx.y * cpc >= (p.M + WG_MC - 1) / WG_MC) return;
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
  const int64_t c_begin = (int64_t)blockIdx.y * cpc;
  int n_chunks = (int)min((int64_t)cpc, chunks_total - c_begin);
  if (n_chunks < 0) n_chunks = 0;

  if (tid == 0) {
    prefetch_tmap(&map_in);
    prefetch_tmap(&map_l);
    for (int s = 0; s < WG_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], p.amax_bits[z] != nullptr ? 3 : 1);   // MMA commit (+ the two amax warps)
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
  if (!p.late_wait) pdl_wait();   // dA reads P, written by the kernels before it (no-op without a programmatic edge)
  pdl_trigger();

  if (warp == 0) {
    if (elect_one()) {   // ---- TMA producer
      // the pass that also finds max |G| is followed by the quantize pass over the same G: ask L2 to keep it
      const bool keep = p.amax_bits[z] != nullptr;
      const uint64_t pol = l2_policy_evict_last();
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WG_STAGES;
        mbar_wait(&empty_bar[s], ((it / WG_STAGES) & 1) ^ 1);
        uint8_t* base = smem + s * STAGE_BYTES;
        const int32_t m0 = (int32_t)((c_begin + it) * WG_MC);
        mbar_expect_tx(&full_bar[s], STAGE_BYTES);
        if (keep) {
          tma_load_2d_hint(base, &map_in, &full_bar[s], f0, m0, pol);
          tma_load_2d_hint(base + WG_MC * 128, &map_in, &full_bar[s], f0 + 64, m0, pol);
        } else {
          tma_load_2d(base, &map_in, &full_bar[s], f0, m0);
          tma_load_2d(base + WG_MC * 128, &map_in, &full_bar[s], f0 + 64, m0);
        }
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
  } else if (p.amax_bits[z] != nullptr) {
    // ---- warps 2-3: max |In| over the staged chunks (|bf16| orders like its low 15 bits)
    const uint32_t m = 0x7FFF7FFFu;
    uint32_t acc = 0;
    const int t64 = tid - 64;
    for (int it = 0; it < n_chunks; ++it) {
      const int s = it % WG_STAGES;
      mbar_wait(&full_bar[s], (it / WG_STAGES) & 1);
      const uint4* src = reinterpret_cast<const uint4*>(smem + s * STAGE_BYTES);
#pragma unroll 4
      for (int j = 0; j < WG_IN_BYTES / 16 / 64; ++j) {
        const uint4 v = src[t64 + j * 64];
        acc = __vmaxu2(acc, __vmaxu2(__vmaxu2(v.x & m, v.y & m), __vmaxu2(v.z & m, v.w & m)));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty_bar[s]);
    }
    uint32_t best = max(acc & 0xFFFFu, acc >> 16);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if (lane == 0 && best != 0) atomicMax(p.amax_bits[z], best << 16);
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
      if (f < F) {
        float* o = p.out[z] + f * R + c0;
        if (p.direct[z]) {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4*>(o + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
        } else {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            red_add_v4(o + j, __uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]),
                       __uint_as_float(v[j + 3]));
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
static int launch_wg(const CUtensorMap* maps, const WgParams& p, dim3 grid, bool pdl, cudaStream_t st) {
  constexpr int NG = (R + 63) / 64;
  const int smem = WG_STAGES * (WG_IN_BYTES + NG * WG_LG_BYTES) + 1024;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(WG_THREADS, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (pdl && pdl_enabled()) ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_wgrad<R>, maps[0], maps[1], maps[2], maps[3], p));
  return FT_OK;
}

// which = 1: dA [K x r] = X^T P[:, r_s:];  which = 2: dBt [N x r] = G^T H[:, r_s:];  which = 3: both in
// ONE launch (blockIdx.z picks the problem).  accumulate == 0 and a single M slice: plain stores;
// otherwise the buffers are zeroed first (accumulate == 0) and the slices combine with fp32 reductions.
// amax_g (which & 2 only): pre-zeroed word that receives the bit pattern of max |G|.
int launch_wgrad(int which, const void* x, const void* g, int64_t M, int64_t K, int64_t N, const void* p_saved,
                 const void* h_saved, int r_t, int r_s, int r, float* dA, float* dBt, int accumulate,
                 unsigned int* amax_g, float* zero_fill, int64_t zero_fill_n, bool after_kernel, bool beside_prev,
                 cudaStream_t st) {
  CUtensorMap maps[4];
  const void* in_all[2] = {x, g};
  const void* lr_all[2] = {p_saved, h_saved};
  const int64_t F_all[2] = {K, N};
  float* out_all[2] = {dA, dBt};
  WgParams p;
  p.M = M;
  p.r_s = r_s;
  p.r = r;
  p.zero_fill = reinterpret_cast<float4*>(zero_fill);
  p.zero_fill_n4 = zero_fill_n / 4;   // K * r, r % 16 == 0
  const int64_t chunks = ceil_div(M, WG_MC);
  // the enabled problems, compacted into z = 0 .. nz-1
  int sel[2], nz = 0;
  for (int z = 0; z < 2; ++z)
    if (which & (1 << z)) sel[nz++] = z;
  int64_t f_tiles_total = 0;
  for (int i = 0; i < nz; ++i) f_tiles_total += ceil_div(F_all[sel[i]], WG_F);
  // M slices: one wave of two resident CTAs per SM over all feature tiles (rounded DOWN: a second,
  // mostly empty wave costs more than slightly longer slices), at least 8 chunks (512 rows) each
  int64_t slices = (int64_t)2 * sm_count() / f_tiles_total;
  if (slices > chunks / 8) slices = chunks / 8;
  if (slices < 1) slices = 1;
  unsigned gx = 0, gy = 0;
  void* clr[2] = {nullptr, nullptr};
  size_t clr_bytes[2] = {0, 0};
  int nclr = 0;
  for (int i = 0; i < 2; ++i) {
    const int z = i < nz ? sel[i] : sel[0];
    int rc = make_tensor_map_2d(&maps[2 * i], in_all[z], 2, (uint64_t)F_all[z], (uint64_t)M, (uint64_t)F_all[z] * 2, 64,
                                WG_MC, Swizzle::B128);
    if (rc != FT_OK) return rc;
    rc = make_tensor_map_2d(&maps[2 * i + 1], lr_all[z], 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, WG_MC,
                            Swizzle::B128);
    if (rc != FT_OK) return rc;
    p.F[i] = F_all[z];
    p.chunks_per_cta[i] = (int)ceil_div(chunks, slices);
    const unsigned sl = (unsigned)ceil_div(chunks, p.chunks_per_cta[i]);
    p.direct[i] = (sl == 1 && !accumulate) ? 1 : 0;
    p.out[i] = out_all[z];
    p.amax_bits[i] = z == 1 ? amax_g : nullptr;
    if (i >= nz) continue;
    if (!accumulate && !p.direct[i]) {   // cleared below by one kernel with programmatic edges
      clr[nclr] = out_all[z];
      clr_bytes[nclr++] = (size_t)F_all[z] * r * sizeof(float);
    }
    const unsigned ft = (unsigned)ceil_div(F_all[z], WG_F);
    if (ft > gx) gx = ft;
    if (sl > gy) gy = sl;
  }
  const dim3 grid(gx, gy, (unsigned)nz);
  if (nclr > 0) {
    int rc = launch_clear2(clr[0], clr_bytes[0], clr[1], clr_bytes[1], st);
    if (rc != FT_OK) return rc;
    after_kernel = true;
  }
  // after_kernel: the launch directly follows a kernel of the same call (the clear above, or the caller's
  // previous launch with accumulate set): it may set itself up while that kernel drains
  const bool pdl = after_kernel && (accumulate != 0 || nclr > 0 || (p.direct[0] && (nz == 1 || p.direct[1])));
  // beside_prev (caller's promise, see WgParams::late_wait): only without a clear kernel in between and
  // without a zero-fill job, whose wait comes first
  p.late_wait = (beside_prev && pdl && nclr == 0 && zero_fill == nullptr) ? 1 : 0;
  switch (r) {
    case 16: return launch_wg<16>(maps, p, grid, pdl, st);
    case 32: return launch_wg<32>(maps, p, grid, pdl, st);
    case 48: return launch_wg<48>(maps, p, grid, pdl, st);
    case 64: return launch_wg<64>(maps, p, grid, pdl, st);
    case 80: return launch_wg<80>(maps, p, grid, pdl, st);
    case 96: return launch_wg<96>(maps, p, grid, pdl, st);
    case 112: return launch_wg<112>(maps, p, grid, pdl, st);
    case 128: return launch_wg<128>(maps, p, grid, pdl, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
