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

constexpr int WG_MC = 64;         // rows of M per ring stage
constexpr int WG_THREADS = 128;
constexpr int WG_LG_BYTES = WG_MC * 128;      // one 64-column group of L
// A CTA owns FW = 256 features (two MMA halves of 128; 512 contiguous bytes per row of In) and a ring as deep as
// shared memory allows (5 x 40 KB for r <= 64): the runtime co-schedules ONE CTA per SM of a cluster kernel that
// allocates tensor memory, so the bytes in flight come from the ring, not from a second CTA.
// What bounds the pass (round 2, measured): ~3.7-3.9 TB/s whatever was tried -- 128- or 256-feature tiles, 3 to 6
// stages, 108 to 432 CTAs in flight (a workspace-slot variant with three CTAs per SM), no MMAs and no amax work at
// all (same time), whole-row L2 prefetches ahead of the strip loads (slower), strips started at rotated rows (same).
// A strip walking DOWN the rows takes 256-512 bytes from each DRAM page; the quantize kernel, which walks ALONG
// the rows with the same TMA boxes, reaches 5.9 TB/s.
template <int R, int FW>
struct WgCfg {
  static constexpr int NG = (R + 63) / 64;
  static constexpr int HALVES = FW / 128;                    // MMA halves of 128 features
  static constexpr int IN_BYTES = (FW / 64) * WG_MC * 128;   // FW / 64 boxes of 64 features x 64 rows
  static constexpr int STAGE_BYTES = IN_BYTES + NG * WG_LG_BYTES;
  static constexpr int DEEP = (226 * 1024) / STAGE_BYTES > 6 ? 6 : (226 * 1024) / STAGE_BYTES;
  static constexpr int STAGES = DEEP;
  static constexpr int SMEM = STAGES * STAGE_BYTES + 1024;
  static constexpr uint32_t HALF_COLS = R <= 32 ? 32 : (R <= 64 ? 64 : 128);   // TMEM columns of one 128-feature half
  static_assert(FW == 256, "feature tile");
};

struct WgParams {      // two problems in one launch: [0] dA = X^T P_lora, [1] dB^T = G^T H_lora
  int64_t M;
  int64_t F[2];
  int r_s, r;
  int chunks_per_cta;
  float* out[2];
  unsigned int* amax_bits[2];   // non-null: atomicMax target for max |In| (bf16 bits << 16), pre-zeroed
  int late_wait;                // 1: nothing this launch touches depends on its predecessor, which passes
                                //    griddepcontrol.wait in every CTA before triggering: start beside it and
                                //    wait for it at the END (completion stays transitive for the next launch)
  int n_slices;                 // M slices (gridDim.y); every slice has work
  int accumulate;               // add to the output instead of overwriting it
#ifdef FT_TRACE
  int dbg;                      // development builds: 1 = no MMAs, 2 = no amax fold
#endif
};

__device__ __forceinline__ float4 ld_cluster_f4(uint32_t cluster_addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(cluster_addr) : "memory");
  return v;
}

template <int R, int FW>
__global__ void __launch_bounds__(WG_THREADS, 1)
k_wgrad(const __grid_constant__ CUtensorMap map_in0, const __grid_constant__ CUtensorMap map_l0,
        const __grid_constant__ CUtensorMap map_in1, const __grid_constant__ CUtensorMap map_l1,
        const WgParams p) {
  using Cfg = WgCfg<R, FW>;
  constexpr int NG = Cfg::NG, HALVES = Cfg::HALVES, STAGE_BYTES = Cfg::STAGE_BYTES, WG_STAGES = Cfg::STAGES;
  constexpr int IN_BYTES = Cfg::IN_BYTES;
  constexpr uint32_t HALF_COLS = Cfg::HALF_COLS;
  constexpr uint32_t TMEM_COLS = HALVES * HALF_COLS < 32 ? 32 : HALVES * HALF_COLS;
  const int z = blockIdx.z;
  const CUtensorMap& map_in = z == 0 ? map_in0 : map_in1;
  const CUtensorMap& map_l = z == 0 ? map_l0 : map_l1;
  const int64_t F = p.F[z];
  const int cpc = p.chunks_per_cta;
  // CTAs beyond this problem's feature tiles have nothing to do (uniform per cluster: a cluster spans blockIdx.y
  // only).  Every M slice has work: the host sizes gridDim.y = ceil(chunks / chunks_per_cta).
  if ((int64_t)blockIdx.x * FW >= F) return;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[WG_STAGES], empty_bar[WG_STAGES], acc_bar;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t f0 = (int32_t)blockIdx.x * FW;
  const int64_t chunks_total = (p.M + WG_MC - 1) / WG_MC;
  const int64_t c_begin = (int64_t)blockIdx.y * cpc;
  const int n_chunks = (int)min((int64_t)cpc, chunks_total - c_begin);   // >= 1

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
#pragma unroll
        for (int b = 0; b < FW / 64; ++b) {
          if (keep) tma_load_2d_hint(base + b * (WG_MC * 128), &map_in, &full_bar[s], f0 + b * 64, m0, pol);
          else tma_load_2d(base + b * (WG_MC * 128), &map_in, &full_bar[s], f0 + b * 64, m0);
        }
#pragma unroll
        for (int g = 0; g < NG; ++g)
          tma_load_2d(base + IN_BYTES + g * WG_LG_BYTES, &map_l, &full_bar[s], p.r_s + g * 64, m0);
      }
    }
  } else if (warp == 1) {
    if (elect_one()) {   // ---- MMA issuer: acc_h[128 f x R] += In[64 m, 128 f of half h]^T * L[64 m, R]
      constexpr uint32_t idesc = idesc_bf16(128, R) | (1u << 15) | (1u << 16);  // A and B MN-major
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WG_STAGES;
        mbar_wait(&full_bar[s], (it / WG_STAGES) & 1);
        tc_fence_after();
        const uint32_t in_u = smem_u32(smem + s * STAGE_BYTES);
        const uint32_t l_u = in_u + IN_BYTES;
#ifdef FT_TRACE
        if (p.dbg & 1) {
          tc_commit(&empty_bar[s]);
          continue;
        }
#endif
#pragma unroll
        for (int hf = 0; hf < HALVES; ++hf)
#pragma unroll
          for (int k = 0; k < 4; ++k)   // 16 rows of m per MMA = two 8-row swizzle groups = 2048 bytes
            mma_bf16(tmem_base + hf * HALF_COLS, make_smem_desc(in_u + hf * (2 * WG_MC * 128) + k * 2048, 1024, WG_MC * 128, 2),
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
      for (int j = 0; j < IN_BYTES / 16 / 64; ++j) {
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

  {   // ---- drain: thread = feature (TMEM lane) of each 128-feature half, R fp32 columns
    mbar_wait(&acc_bar, 0);   // every MMA has completed: the ring's shared memory is free
    tc_fence_after();
    const int fl = warp * 32 + lane;
    const int ns = p.n_slices;
    constexpr int QH = R / 4;   // column quads per half
    const bool via_cluster = ns > 1;
    // several slices: park the partial tile in this CTA's shared memory (the ring's: every warp must be done with the staged
    // chunks first -- the amax warps read them too), layout [half][column quad][feature][4 floats]
    if (via_cluster) __syncthreads();
    float* park = reinterpret_cast<float*>(smem);
#pragma unroll
    for (int hf = 0; hf < HALVES; ++hf) {
      const int64_t f = (int64_t)f0 + hf * 128 + fl;
#pragma unroll
      for (int c0 = 0; c0 < R; c0 += 16) {
        uint32_t v[16];
        tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + hf * HALF_COLS + c0, v);
        tmem_ld_wait();
        if (via_cluster) {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4*>(park + ((hf * QH + (c0 + j) / 4) * 128 + fl) * 4) =
                make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
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
    }
    tc_fence_before();
    if (via_cluster) {
      // the cluster = the M slices of this feature tile.  After the barrier slice s sums column quads
      // s, s + ns, ... (of the HALVES x R / 4 of the tile) over all slices' shared memory, in slice order, and owns
      // those outputs.
      cluster_sync();
      const uint32_t rank = cluster_ctarank();
      const uint32_t park_u = smem_u32(park);
#pragma unroll 1
      for (int qi = (int)rank; qi < HALVES * QH; qi += ns) {
        const int hf = qi / QH, q = qi % QH;
        const int64_t f = (int64_t)f0 + hf * 128 + fl;
        const uint32_t off = park_u + (uint32_t)((qi * 128 + fl) * 16);
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

// one-time per-device setup: shared-memory opt-in and the largest carveout
template <int R, int FW>
static int wg_prepare() {
  static bool done[FT_MAX_DEVICES] = {};
  const int dev = current_device();
  if (dev >= 0 && dev < FT_MAX_DEVICES && done[dev]) return FT_OK;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad<R, FW>, cudaFuncAttributeMaxDynamicSharedMemorySize, WgCfg<R, FW>::SMEM));
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad<R, FW>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                   cudaSharedmemCarveoutMaxShared));
  if (dev >= 0 && dev < FT_MAX_DEVICES) done[dev] = true;
  return FT_OK;
}

// how many clusters (1, s, 1) the device holds at once (cached per device and s): a grid that does
// not fit in one wave runs its last clusters alone
template <int R>
static int wg_max_active_clusters(int s) {
  static int cached[FT_MAX_DEVICES][9] = {};
  const int dev = current_device();
  const bool ok = dev >= 0 && dev < FT_MAX_DEVICES && s >= 1 && s <= 8;
  if (ok && cached[dev][s] != 0) return cached[dev][s];
  if (wg_prepare<R, 256>() != FT_OK) return 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1, (unsigned)s, 1);
  cfg.blockDim = dim3(WG_THREADS, 1, 1);
  cfg.dynamicSmemBytes = WgCfg<R, 256>::SMEM;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 1;
  attr[0].val.clusterDim.y = (unsigned)s;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, k_wgrad<R, 256>, &cfg) != cudaSuccess || n < 1) {
    (void)cudaGetLastError();
    n = sm_count() / s;   // one CTA per SM, perfect packing: a guess that only sizes the slices
    if (n < 1) n = 1;
  }
  if (ok) cached[dev][s] = n;
  return n;
}

template <int R, int FW>
static int launch_wg(const CUtensorMap* maps, const WgParams& p, dim3 grid, bool pdl, cudaStream_t st) {
  int rc = wg_prepare<R, FW>();
  if (rc != FT_OK) return rc;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(WG_THREADS, 1, 1);
  cfg.dynamicSmemBytes = WgCfg<R, FW>::SMEM;
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
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_wgrad<R, FW>, maps[0], maps[1], maps[2], maps[3], p));
  return FT_OK;
}

static int wg_clusters_for(int r, int s) {
  switch (r) {
    case 16: return wg_max_active_clusters<16>(s);
    case 32: return wg_max_active_clusters<32>(s);
    case 48: return wg_max_active_clusters<48>(s);
    case 64: return wg_max_active_clusters<64>(s);
    case 80: return wg_max_active_clusters<80>(s);
    case 96: return wg_max_active_clusters<96>(s);
    case 112: return wg_max_active_clusters<112>(s);
    case 128: return wg_max_active_clusters<128>(s);
    default: return 1;
  }
}

template <int FW>
static int launch_wg_r(int r, const CUtensorMap* maps, const WgParams& p, dim3 grid, bool pdl, cudaStream_t st) {
  switch (r) {
    case 16: return launch_wg<16, FW>(maps, p, grid, pdl, st);
    case 32: return launch_wg<32, FW>(maps, p, grid, pdl, st);
    case 48: return launch_wg<48, FW>(maps, p, grid, pdl, st);
    case 64: return launch_wg<64, FW>(maps, p, grid, pdl, st);
    case 80: return launch_wg<80, FW>(maps, p, grid, pdl, st);
    case 96: return launch_wg<96, FW>(maps, p, grid, pdl, st);
    case 112: return launch_wg<112, FW>(maps, p, grid, pdl, st);
    case 128: return launch_wg<128, FW>(maps, p, grid, pdl, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

// which = 1: dA [K x r] = X^T P[:, r_s:];  which = 2: dBt [N x r] = G^T H[:, r_s:];  which = 3: both in
// ONE launch (blockIdx.z picks the problem).  The M slices (at most 8, the portable cluster size) of a feature
// tile are one cluster and combine over distributed shared memory in slice order: no clear kernel, no atomics on
// the data, no workspace, a fixed order of additions.
// amax_g (which & 2 only): zero word that receives the bit pattern of max |G|.
// after_kernel: the launch directly follows a kernel of the same call (programmatic edge allowed).
// beside_prev: see WgParams::late_wait (the caller's promise).
int launch_wgrad(int which, const void* x, const void* g, int64_t M, int64_t K, int64_t N, const void* p_saved,
                 const void* h_saved, int r_t, int r_s, int r, float* dA, float* dBt, int accumulate,
                 unsigned int* amax_g, bool after_kernel, bool beside_prev, cudaStream_t st) {
  constexpr int FW = 256;
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
  for (int i = 0; i < nz; ++i) f_tiles_total += ceil_div(F_all[sel[i]], FW);
  // M slices = cluster size, at most 8, at least 4 chunks (256 rows) each: the count s that minimises
  // waves(s) x chunks per slice, where waves(s) = clusters of the launch / clusters of size s the device holds at
  // once (one CTA per SM, and clusters of 3 or more strand a few SMs: 148, 74, 45, 33, 26, 22, 15, 15 on B200) --
  // a launch that spills into a second wave runs its last clusters alone
  int64_t max_slices = chunks / 4;
  if (max_slices > 8) max_slices = 8;
  if (max_slices < 1) max_slices = 1;
  int64_t slices = 1, best_cost = -1;
  for (int64_t s = 1; s <= max_slices; ++s) {
    const int64_t cap = wg_clusters_for(r, (int)s);
    const int64_t cost = ceil_div(f_tiles_total, cap) * ceil_div(chunks, s);
    if (best_cost < 0 || cost < best_cost) {
      best_cost = cost;
      slices = s;
    }
  }
  const int cpc = (int)ceil_div(chunks, slices);
  const unsigned sl = (unsigned)ceil_div(chunks, cpc);   // every slice has at least one chunk
  p.n_slices = (int)sl;
  p.chunks_per_cta = cpc;
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
    p.out[i] = out_all[z];
    p.amax_bits[i] = z == 1 ? amax_g : nullptr;
    if (i >= nz) continue;
    const unsigned ft = (unsigned)ceil_div(F_all[z], FW);
    if (ft > gx) gx = ft;
  }
  const dim3 grid(gx, sl, (unsigned)nz);
  const bool pdl = after_kernel;
  p.late_wait = (beside_prev && pdl) ? 1 : 0;
#ifdef FT_TRACE
  p.dbg = getenv("FT_WG_DBG") ? atoi(getenv("FT_WG_DBG")) : 0;
  if (p.dbg & 2) p.amax_bits[0] = p.amax_bits[1] = nullptr;
#endif
  return launch_wg_r<256>(r, maps, p, grid, pdl, st);
}

}  // namespace ft
