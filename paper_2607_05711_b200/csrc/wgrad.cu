// wgrad.cu -- a5: LoRA weight gradients (Eq. 4)
//     out[f, j] (+)= sum_m In[m, f] * L[m, r_s + j]        f < F, j < r
// used twice: dA = X^T (G B^T) with In = X, L = P;  dB^T = G^T (X A) with In = G, L = H.
// HBM-bound: In is read exactly once.  A CTA owns 128 features x one slice of M and walks it in
// 64-row chunks that TMA stages (SWIZZLE_128B) through an mbarrier ring.  One thread issues
// tcgen05.mma kind::f16 (M = 128 features, N = r, K = 16 rows, four per chunk) with BOTH
// operands MN-major -- the staged chunks are used as they lie in memory, nothing is transposed
// by the SM -- into a TMEM accumulator; four warps drain it.  The M slices of one feature tile (at most 8) are
// the CTAs of one thread-block cluster (1, slices, 1): each parks its fp32 partial tile in its own shared
// memory, and after a cluster barrier every CTA sums an equal share of the tile over distributed shared memory,
// in slice order, and writes (or adds to) the output.  No clear kernel, no atomics on the data, no workspace,
// the same bits on every run.  (Round 1 combined the slices with red.global.add into a pre-cleared output: a
// clear launch per call and an unordered sum.  Slots in global memory with an arrival counter per tile -- the
// scheme of the quantize kernel -- cost 20 us per step here: the last arriver's sum is a chain of L2 round trips.)
#include <cstdio>
#include <cstdlib>

#include "common.cuh"

namespace ft {

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
  float* out[2];
  unsigned int* amax_bits[2];   // non-null: atomicMax target for max |In| (bf16 bits << 16), pre-zeroed
  int late_wait;                // 1: nothing this launch touches depends on its predecessor, which passes
                                //    griddepcontrol.wait in every CTA before triggering: start beside it and
                                //    wait for it at the END (completion stays transitive for the next launch)
  int n_slices;                 // M slices = CTAs per cluster (gridDim.y); every slice has work
  int accumulate;               // add to the output instead of overwriting it
};

__device__ __forceinline__ float4 ld_cluster_f4(uint32_t cluster_addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(cluster_addr) : "memory");
  return v;
}

template <int R>
__global__ void __launch_bounds__(WG_THREADS, 2)
k_wgrad(const __grid_constant__ CUtensorMap map_in0, const __grid_constant__ CUtensorMap map_l0,
        const __grid_constant__ CUtensorMap map_in1, const __grid_constant__ CUtensorMap map_l1,
        const WgParams p) {
  const int z = blockIdx.z;
  const CUtensorMap& map_in = z == 0 ? map_in0 : map_in1;
  const CUtensorMap& map_l = z == 0 ? map_l0 : map_l1;
  const int64_t F = p.F[z];
  const int cpc = p.chunks_per_cta[z];
  // CTAs beyond this problem's feature tiles have nothing to do (uniform per cluster: a cluster spans blockIdx.y
  // only).  Every M slice has work: the host sizes gridDim.y = ceil(chunks / chunks_per_cta).
  if ((int64_t)blockIdx.x * WG_F >= F) return;
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

  {   // ---- drain: thread = feature (TMEM lane), R fp32 columns
    mbar_wait(&acc_bar, 0);   // every MMA has completed: the ring's shared memory is free
    tc_fence_after();
    const int fl = warp * 32 + lane;
    const int64_t f = (int64_t)f0 + fl;
    const int ns = p.n_slices;
    // several slices: park the partial tile in this CTA's shared memory (the ring's: every warp must be done with
    // the staged chunks first -- the amax warps read them too), layout [column quad][feature][4 floats]
    if (ns > 1) __syncthreads();
    float* park = reinterpret_cast<float*>(smem);
#pragma unroll
    for (int c0 = 0; c0 < R; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + c0, v);
      tmem_ld_wait();
      if (ns > 1) {
#pragma unroll
        for (int j = 0; j < 16; j += 4)
          *reinterpret_cast<uint4*>(park + ((c0 + j) / 4 * WG_F + fl) * 4) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
      } else if (f < F) {
        float4* o = reinterpret_cast<float4*>(p.out[z] + f * R + c0);
#pragma unroll
        for (int j = 0; j < 16; j += 4) {
          float4 a = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]),
                                 __uint_as_float(v[j + 3]));
          if (p.accumulate) {
            const float4 old = o[j / 4];
            a.x += old.x;
            a.y += old.y;
            a.z += old.z;
            a.w += old.w;
          }
          o[j / 4] = a;
        }
      }
    }
    tc_fence_before();
    if (ns > 1) {
      // the cluster = the M slices of this feature tile.  After the barrier slice s sums column quads
      // s, s + ns, ... of the tile over all slices' shared memory, in slice order, and owns those outputs.
      cluster_sync();
      const uint32_t rank = cluster_ctarank();
      const uint32_t park_u = smem_u32(park);
#pragma unroll 1
      for (int q = (int)rank; q < R / 4; q += ns) {
        const uint32_t off = park_u + (uint32_t)((q * WG_F + fl) * 16);
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int s0 = 0; s0 < ns; s0 += 4) {
          float4 v[4];
#pragma unroll
          for (int j = 0; j < 4; ++j)
            v[j] = (s0 + j < ns) ? ld_cluster_f4(map_to_cta(off, (uint32_t)(s0 + j))) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            acc.x += v[j].x;
            acc.y += v[j].y;
            acc.z += v[j].z;
            acc.w += v[j].w;
          }
        }
        if (f < F) {
          float4* o = reinterpret_cast<float4*>(p.out[z] + f * R + q * 4);
          if (p.accumulate) {
            const float4 old = *o;
            acc.x += old.x;
            acc.y += old.y;
            acc.z += old.z;
            acc.w += old.w;
          }
          *o = acc;
        }
      }
      cluster_sync();   // no slice leaves (and frees its shared memory) while a peer still reads it
    }
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
  const int smem = WG_STAGES * (WG_IN_BYTES + NG * WG_LG_BYTES) + 1024;   // >= the 128 x R fp32 parked tile
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(WG_THREADS, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  int na = 0;
  if (grid.y > 1) {   // the M slices of a feature tile form one cluster
    attr[na].id = cudaLaunchAttributeClusterDimension;
    attr[na].val.clusterDim.x = 1;
    attr[na].val.clusterDim.y = grid.y;
    attr[na].val.clusterDim.z = 1;
    ++na;
  }
  if (pdl && pdl_enabled()) {
    attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = attr;
  cfg.numAttrs = na;
  if (getenv("FT_DEBUG_OCC") != nullptr) {
    int ncl = -1, nb = -1;
    cudaOccupancyMaxActiveClusters(&ncl, k_wgrad<R>, &cfg);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_wgrad<R>, WG_THREADS, smem);
    fprintf(stderr, "k_wgrad<%d> grid (%u,%u,%u) smem %d: max active clusters %d, blocks/SM %d\n", R, grid.x, grid.y, grid.z,
            smem, ncl, nb);
  }
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_wgrad<R>, maps[0], maps[1], maps[2], maps[3], p));
  return FT_OK;
}

// which = 1: dA [K x r] = X^T P[:, r_s:];  which = 2: dBt [N x r] = G^T H[:, r_s:];  which = 3: both in
// ONE launch (blockIdx.z picks the problem).  The M slices (at most 8, the portable cluster size) of a feature
// tile are one cluster and combine over distributed shared memory in slice order.
// amax_g (which & 2 only): zero word that receives the bit pattern of max |G|.
// after_kernel: the launch directly follows a kernel of the same call (programmatic edge allowed).
// beside_prev: see WgParams::late_wait (the caller's promise).
int launch_wgrad(int which, const void* x, const void* g, int64_t M, int64_t K, int64_t N, const void* p_saved,
                 const void* h_saved, int r_t, int r_s, int r, float* dA, float* dBt, int accumulate,
                 unsigned int* amax_g, bool after_kernel, bool beside_prev, cudaStream_t st) {
  CUtensorMap maps[4];
  const void* in_all[2] = {x, g};
  const void* lr_all[2] = {p_saved, h_saved};
  const int64_t F_all[2] = {K, N};
  float* out_all[2] = {dA, dBt};
  WgParams p;
  p.M = M;
  p.r_s = r_s;
  p.r = r;
  p.accumulate = accumulate;
  const int64_t chunks = ceil_div(M, WG_MC);
  // the enabled problems, compacted into z = 0 .. nz-1
  int sel[2], nz = 0;
  for (int z = 0; z < 2; ++z)
    if (which & (1 << z)) sel[nz++] = z;
  int64_t f_tiles_total = 0;
  for (int i = 0; i < nz; ++i) f_tiles_total += ceil_div(F_all[sel[i]], WG_F);
  // M slices: one wave of two resident CTAs per SM over all feature tiles (rounded DOWN: a second,
  // mostly empty wave costs more than slightly longer slices), at least 8 chunks (512 rows) each, at most 8
  int64_t slices = (int64_t)2 * sm_count() / f_tiles_total;
  if (slices > chunks / 8) slices = chunks / 8;
  if (slices > 8) slices = 8;
  if (slices < 1) slices = 1;
  const int cpc = (int)ceil_div(chunks, slices);
  const unsigned sl = (unsigned)ceil_div(chunks, cpc);   // every slice has at least one chunk
  p.n_slices = (int)sl;
  unsigned gx = 0;
  for (int i = 0; i < 2; ++i) {
    const int z = i < nz ? sel[i] : sel[0];
    int rc = make_tensor_map_2d(&maps[2 * i], in_all[z], 2, (uint64_t)F_all[z], (uint64_t)M, (uint64_t)F_all[z] * 2, 64,
                                WG_MC, Swizzle::B128);
    if (rc != FT_OK) return rc;
    rc = make_tensor_map_2d(&maps[2 * i + 1], lr_all[z], 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, WG_MC,
                            Swizzle::B128);
    if (rc != FT_OK) return rc;
    p.F[i] = F_all[z];
    p.chunks_per_cta[i] = cpc;
    p.out[i] = out_all[z];
    p.amax_bits[i] = z == 1 ? amax_g : nullptr;
    if (i >= nz) continue;
    const unsigned ft = (unsigned)ceil_div(F_all[z], WG_F);
    if (ft > gx) gx = ft;
  }
  const dim3 grid(gx, sl, (unsigned)nz);
  const bool pdl = after_kernel;
  p.late_wait = (beside_prev && pdl) ? 1 : 0;
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
