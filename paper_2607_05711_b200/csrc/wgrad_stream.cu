// wgrad_stream.cu -- a5 inside ft_linear_bwd: the two LoRA weight-gradient passes of Eq. 4
//     out[f, j] (+)= sum_m In[m, f] * L[m, r_s + j]        f < F, j < r
// as the one-call backward schedules them: dB^T = G^T (X A) FIRST (it also yields max |G|, the a0 of the backward,
// and clears dA for the last launch), dA = X^T (G B^T) LAST (it needs P; it starts beside the dgrad GEMM's tail).
// Same arithmetic as wgrad.cu (TMA-staged 64-row chunks, tcgen05.mma kind::f16 with both operands MN-major, TMEM
// accumulator); what differs is how the pass is laid over the SMs and how the M slices meet:
//   * a CTA owns 128 features x one M slice, 128 threads, a 4-deep ring (~100 KB): TWO CTAs per SM, all of them
//     resident in one wave (slices = 2 SMs / feature tiles, rounded down).  wgrad.cu's cluster kernel is held to one
//     CTA per SM by the runtime (a cluster kernel that allocates tensor memory) and to 45 clusters of three at C2:
//     108 CTAs on 148 SMs, 25.6 us for the dB^T pass against 19.7 us for this shape (ncu, same box, round 2);
//     and a dA kernel of small CTAs finds room beside the retiring CTAs of the GEMM in front of it.
//   * dB^T: every slice stores its fp32 partial tile to its own slot in the workspace; k_finalize_h of the quantize
//     pass that follows -- it runs beside the dgrad GEMM anyway -- adds the slots in slice order (SumJob,
//     quantize_fused.cu).  No clear kernel, no atomics, the same bits on every run.  With accumulate set the slices
//     add to the caller's buffer with red.global.add instead (nothing to clear).
//   * dA: the last kernel of the call has nobody behind it to add slots; its slices meet by red.global.add.v4.f32
//     in a buffer that the dB^T launch cleared on its way (order of the additions not fixed: DESIGN.md O-17).
// ft_lora_wgrad (the standalone call, no workspace) keeps wgrad.cu's cluster kernel.
#include <cstdlib>

#include "common.cuh"

namespace ft {

constexpr int WS_F = 128;
constexpr int WS_MC = 64;
constexpr int WS_STAGES = 4;
constexpr int WS_THREADS = 128;
constexpr int WS_IN_BYTES = 2 * WS_MC * 128;  // two 64-feature boxes
constexpr int WS_LG_BYTES = WS_MC * 128;      // one 64-column group of L

enum { WS_OUT_STORE = 0, WS_OUT_RED = 1, WS_OUT_SLOTS = 2 };

struct WgsParams {
  int64_t M, F;
  int r_s;
  int chunks_per_cta;
  int mode;                     // WS_OUT_*: one slice stores; slices add with fp32 reductions; slices store to slots
  float* out;                   // [F x R] (STORE, RED) or [slices x F x R] (SLOTS)
  unsigned int* amax_bits;      // non-null: atomicMax target for max |In| (bf16 bits << 16), pre-zeroed
  int late_wait;                // 1: nothing this launch touches depends on its predecessor, which passes
                                //    griddepcontrol.wait in every CTA before triggering: start beside it and
                                //    wait for it at the END (completion stays transitive for the next launch)
  float4* zero_fill;            // non-null: buffer this launch clears for a LATER launch (zero_fill_n4 float4s)
  int64_t zero_fill_n4;
#ifdef FT_TRACE
  int dbg;                      // development builds: 1 = no MMAs, 2 = no amax fold, 4 = no L2 hint
#endif
};

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
               : "memory");
}

template <int R>
__global__ void __launch_bounds__(WS_THREADS, 2)
k_wgrad_s(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_l, const WgsParams p) {
  if (p.zero_fill != nullptr) {   // grid-stride clear by every CTA of the launch
    pdl_wait();                   // nothing is written before the predecessor has ended
    const int64_t nthr = (int64_t)gridDim.x * gridDim.y * WS_THREADS;
    const int64_t me = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * WS_THREADS + threadIdx.x;
    for (int64_t i = me; i < p.zero_fill_n4; i += nthr) p.zero_fill[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  constexpr int NG = (R + 63) / 64;
  constexpr int STAGE_BYTES = WS_IN_BYTES + NG * WS_LG_BYTES;
  constexpr uint32_t TMEM_COLS = R <= 32 ? 32 : (R <= 64 ? 64 : 128);
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[WS_STAGES], empty_bar[WS_STAGES], acc_bar;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t f0 = (int32_t)blockIdx.x * WS_F;
  const int64_t chunks_total = (p.M + WS_MC - 1) / WS_MC;
  const int64_t c_begin = (int64_t)blockIdx.y * p.chunks_per_cta;
  const int n_chunks = (int)min((int64_t)p.chunks_per_cta, chunks_total - c_begin);   // >= 1: the host sizes gridDim.y

  if (tid == 0) {
    prefetch_tmap(&map_in);
    prefetch_tmap(&map_l);
    for (int s = 0; s < WS_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], p.amax_bits != nullptr ? 3 : 1);   // MMA commit (+ the two amax warps)
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
#ifdef FT_TRACE
      const bool keep = p.amax_bits != nullptr && !(p.dbg & 4);
#else
      const bool keep = p.amax_bits != nullptr;
#endif
      const uint64_t pol = l2_policy_evict_last();
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WS_STAGES;
        mbar_wait(&empty_bar[s], ((it / WS_STAGES) & 1) ^ 1);
        uint8_t* base = smem + s * STAGE_BYTES;
        const int32_t m0 = (int32_t)((c_begin + it) * WS_MC);
        mbar_expect_tx(&full_bar[s], STAGE_BYTES);
        if (keep) {
          tma_load_2d_hint(base, &map_in, &full_bar[s], f0, m0, pol);
          tma_load_2d_hint(base + WS_MC * 128, &map_in, &full_bar[s], f0 + 64, m0, pol);
        } else {
          tma_load_2d(base, &map_in, &full_bar[s], f0, m0);
          tma_load_2d(base + WS_MC * 128, &map_in, &full_bar[s], f0 + 64, m0);
        }
#pragma unroll
        for (int g = 0; g < NG; ++g)
          tma_load_2d(base + WS_IN_BYTES + g * WS_LG_BYTES, &map_l, &full_bar[s], p.r_s + g * 64, m0);
      }
    }
  } else if (warp == 1) {
    if (elect_one()) {   // ---- MMA issuer: acc[128 f x R] += In[64 m, 128 f]^T * L[64 m, R]
      constexpr uint32_t idesc = idesc_bf16(WS_F, R) | (1u << 15) | (1u << 16);  // A and B MN-major
      for (int it = 0; it < n_chunks; ++it) {
        const int s = it % WS_STAGES;
        mbar_wait(&full_bar[s], (it / WS_STAGES) & 1);
        tc_fence_after();
        const uint32_t in_u = smem_u32(smem + s * STAGE_BYTES);
        const uint32_t l_u = in_u + WS_IN_BYTES;
#ifdef FT_TRACE
        if (!(p.dbg & 1))
#endif
#pragma unroll
        for (int k = 0; k < 4; ++k)   // 16 rows of m per MMA = two 8-row swizzle groups = 2048 bytes
          mma_bf16(tmem_base, make_smem_desc(in_u + k * 2048, 1024, WS_MC * 128, 2),
                   make_smem_desc(l_u + k * 2048, 1024, WS_LG_BYTES, 2), idesc, (it | k) != 0);
        tc_commit(&empty_bar[s]);
      }
      tc_commit(&acc_bar);
    }
  } else if (p.amax_bits != nullptr) {
    // ---- warps 2-3: max |In| over the staged chunks (|bf16| orders like its low 15 bits)
    const uint32_t m = 0x7FFF7FFFu;
    uint32_t acc = 0;
    const int t64 = tid - 64;
    for (int it = 0; it < n_chunks; ++it) {
      const int s = it % WS_STAGES;
      mbar_wait(&full_bar[s], (it / WS_STAGES) & 1);
      const uint4* src = reinterpret_cast<const uint4*>(smem + s * STAGE_BYTES);
#ifdef FT_TRACE
      if (!(p.dbg & 2))
#endif
#pragma unroll 4
      for (int j = 0; j < WS_IN_BYTES / 16 / 64; ++j) {
        const uint4 v = src[t64 + j * 64];
        acc = __vmaxu2(acc, __vmaxu2(__vmaxu2(v.x & m, v.y & m), __vmaxu2(v.z & m, v.w & m)));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty_bar[s]);
    }
    uint32_t best = max(acc & 0xFFFFu, acc >> 16);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if (lane == 0 && best != 0) atomicMax(p.amax_bits, best << 16);
  }
  __syncwarp();

  {   // ---- drain: thread = feature (TMEM lane), R fp32 columns
    mbar_wait(&acc_bar, 0);
    tc_fence_after();
    const int64_t f = (int64_t)f0 + warp * 32 + lane;
    float* o = p.out + (p.mode == WS_OUT_SLOTS ? (int64_t)blockIdx.y * p.F * R : 0) + f * R;
#pragma unroll
    for (int c0 = 0; c0 < R; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + c0, v);
      tmem_ld_wait();
      if (f < p.F) {
        if (p.mode != WS_OUT_RED) {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4*>(o + c0 + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
        } else {
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            red_add_v4(o + c0 + j, __uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]),
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
static int launch_wgs(const CUtensorMap& mi, const CUtensorMap& ml, const WgsParams& p, dim3 grid, bool pdl, cudaStream_t st) {
  constexpr int NG = (R + 63) / 64;
  const int smem = WS_STAGES * (WS_IN_BYTES + NG * WS_LG_BYTES) + 1024;
  FT_CUDA_TRY(cudaFuncSetAttribute(k_wgrad_s<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(WS_THREADS, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (pdl && pdl_enabled()) ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_wgrad_s<R>, mi, ml, p));
  return FT_OK;
}

// One gradient: out [F x r] (+)= In[M x F]^T L[M x r_t][:, r_s:].
//   slots == NULL: the slices add into `out` with fp32 reductions; the caller guarantees that `out` is zero (or holds
//     what is to be accumulated into) by the time this kernel's CTAs drain -- e.g. via an earlier launch's zero_fill.
//   slots != NULL (capacity slot_capacity_floats): more than one slice -> each stores its partial to slots
//     [slice][F x r] and *n_slots = slices: the caller has them added in slice order (SumJob); one slice -> plain
//     stores to `out`, *n_slots = 0.
//   amax_in: pre-zeroed word that receives the bit pattern of max |In|.
//   zero_fill: a buffer of zero_fill_n floats this launch clears on its way (for a later launch's reductions).
//   after_kernel / beside_prev: as in launch_wgrad (programmatic edge; late wait).
int launch_wgrad_stream(const void* in, const void* l, int64_t M, int64_t F, int r_t, int r_s, int r, float* out,
                        float* slots, size_t slot_capacity_floats, int* n_slots, unsigned int* amax_in,
                        float* zero_fill, int64_t zero_fill_n, bool after_kernel, bool beside_prev, cudaStream_t st) {
  CUtensorMap mi, ml;
  int rc = make_tensor_map_2d(&mi, in, 2, (uint64_t)F, (uint64_t)M, (uint64_t)F * 2, 64, WS_MC, Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&ml, l, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, WS_MC, Swizzle::B128);
  if (rc != FT_OK) return rc;
  const int64_t chunks = ceil_div(M, WS_MC);
  const int64_t f_tiles = ceil_div(F, WS_F);
  // M slices: one wave of two resident CTAs per SM over all feature tiles (rounded DOWN: a second, mostly empty
  // wave costs more than slightly longer slices), at least 8 chunks (512 rows) each
  int64_t slices = (int64_t)2 * sm_count() / f_tiles;
  if (slices > chunks / 8) slices = chunks / 8;
  if (slices < 1) slices = 1;
  if (slots != nullptr)   // never more slots than the workspace region holds
    while (slices > 1 && (size_t)slices * (size_t)F * (size_t)r > slot_capacity_floats) --slices;
  WgsParams p = {};
  p.M = M;
  p.F = F;
  p.r_s = r_s;
  p.chunks_per_cta = (int)ceil_div(chunks, slices);
  const unsigned sl = (unsigned)ceil_div(chunks, (int64_t)p.chunks_per_cta);
  if (slots != nullptr) {
    p.mode = sl > 1 ? WS_OUT_SLOTS : WS_OUT_STORE;
    p.out = sl > 1 ? slots : out;
    if (n_slots != nullptr) *n_slots = sl > 1 ? (int)sl : 0;
  } else {
    p.mode = WS_OUT_RED;
    p.out = out;
  }
  p.amax_bits = amax_in;
  p.zero_fill = reinterpret_cast<float4*>(zero_fill);
  p.zero_fill_n4 = zero_fill_n / 4;   // F' * r, r % 16 == 0
#ifdef FT_TRACE
  p.dbg = getenv("FT_WG_DBG") ? atoi(getenv("FT_WG_DBG")) : 0;
#endif
  const bool pdl = after_kernel;
  p.late_wait = (beside_prev && pdl && zero_fill == nullptr) ? 1 : 0;
  const dim3 grid((unsigned)f_tiles, sl, 1);
  switch (r) {
    case 16: return launch_wgs<16>(mi, ml, p, grid, pdl, st);
    case 32: return launch_wgs<32>(mi, ml, p, grid, pdl, st);
    case 48: return launch_wgs<48>(mi, ml, p, grid, pdl, st);
    case 64: return launch_wgs<64>(mi, ml, p, grid, pdl, st);
    case 80: return launch_wgs<80>(mi, ml, p, grid, pdl, st);
    case 96: return launch_wgs<96>(mi, ml, p, grid, pdl, st);
    case 112: return launch_wgs<112>(mi, ml, p, grid, pdl, st);
    case 128: return launch_wgs<128>(mi, ml, p, grid, pdl, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
