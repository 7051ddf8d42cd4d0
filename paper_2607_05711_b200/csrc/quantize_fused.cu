// quantize_fused.cu -- a1 / a3: one pass over X (or G) that emits the NVFP4 codes,
// the block scales and the low-rank down-projection H = X * D ("fuse
// ... quantization and down-projection").
//
// Decomposition: a CTA owns 128 rows x (cols / SPLIT) columns and walks them in
// 128 x 64 chunks that TMA stages into shared memory (SWIZZLE_128B) through a
// 4-deep mbarrier ring.  From one staged chunk
//   - 256 threads quantize: thread (row = tid/2, half = tid%2) owns two 1x16 blocks;
//   - 8 warps run mma.sync m16n8k16 (bf16 -> fp32) on their 16 rows against the
//     64 x r_t slice of D staged beside it.
// The SPLIT CTAs of a 128-row tile form a thread-block cluster (1, SPLIT, 1); their
// fp32 partial H tiles are summed through distributed shared memory, so H is
// complete in one pass with no atomics and no second kernel.
#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

constexpr int QF_ROWS = 128;    // rows per CTA
constexpr int QF_KC = 64;       // columns per chunk (128 bytes of bf16 = one swizzle row)
constexpr int QF_STAGES = 4;
constexpr int QF_THREADS = 256;
constexpr int QF_X_BYTES = QF_ROWS * QF_KC * 2;  // 16 KB
constexpr int QF_DG_BYTES = QF_KC * 128;         // one 64-column group of D: 8 KB

struct QFParams {
  int64_t rows, cols;
  const float* amax_t;
  uint8_t* codes;
  uint8_t* sf;
  float* g_dec_out;
  int sf_layout;
  __nv_bfloat16* h_out;         // [rows x r_t] or null
  __nv_bfloat16* hs_out;        // [rows x r_t] or null
  const float* other_dec_scale; // for hs_out
  int split;                    // CTAs per row tile (cluster size)
};

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                        uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                          uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void mma_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                          uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, "
      "{%8, %9}, {%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;"
               ::: "memory");
}
__device__ __forceinline__ float ld_dsmem_f32(uint32_t local_addr, uint32_t cta_rank) {
  uint32_t remote;
  float v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local_addr), "r"(cta_rank));
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(remote));
  return v;
}

// R_T: width of the projection (0 = quantize only).  NG = 64-column groups of D.
template <int R_T>
__global__ void __launch_bounds__(QF_THREADS, 1)
k_quantize_fused(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_d,
                 const QFParams p) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr int NT = R_T / 8;
  constexpr int STAGE_BYTES = QF_X_BYTES + NG * QF_DG_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment for the 128-byte swizzle atoms
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[QF_STAGES];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t row0 = (int64_t)blockIdx.x * QF_ROWS;
  const int split = p.split;
  const int64_t chunks_total = p.cols / QF_KC;
  const int n_chunks = (int)(chunks_total / split);
  const int64_t chunk0 = (int64_t)blockIdx.y * n_chunks;

  if (tid == 0) {
    prefetch_tmap(&map_x);
    if (R_T > 0) prefetch_tmap(&map_d);
    for (int s = 0; s < QF_STAGES; ++s) mbar_init(&full_bar[s], 1);
    fence_mbar_init();
  }
  __syncthreads();

  auto issue = [&](int it) {
    const int s = it % QF_STAGES;
    uint8_t* base = smem + s * STAGE_BYTES;
    const int32_t kcol = (int32_t)((chunk0 + it) * QF_KC);
    mbar_expect_tx(&full_bar[s], STAGE_BYTES);
    tma_load_2d(base, &map_x, &full_bar[s], kcol, (int32_t)row0);
#pragma unroll
    for (int g = 0; g < NG; ++g)
      tma_load_2d(base + QF_X_BYTES + g * QF_DG_BYTES, &map_d, &full_bar[s], g * 64, kcol);
  };
  if (tid == 0) {
    for (int it = 0; it < QF_STAGES && it < n_chunks; ++it) issue(it);
  }

  const TensorScale ts = tensor_scale(__ldg(p.amax_t));
  if (blockIdx.x == 0 && blockIdx.y == 0 && tid == 0) *p.g_dec_out = ts.g_dec;

  // quantizer role of this thread
  const int q_row = tid >> 1, q_half = tid & 1;
  const int64_t q_grow = row0 + q_row;
  const bool q_live = q_grow < p.rows;
  const int64_t nblk = p.cols / 16;
  // projection role: warp -> rows 16*warp .. +15
  float acc[NT > 0 ? NT : 1][4];
#pragma unroll
  for (int j = 0; j < (NT > 0 ? NT : 1); ++j) acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f;

  for (int it = 0; it < n_chunks; ++it) {
    const int s = it % QF_STAGES;
    const uint32_t parity = (it / QF_STAGES) & 1;
    mbar_wait(&full_bar[s], parity);
    const uint8_t* xs = smem + s * STAGE_BYTES;
    const int64_t kcol = (chunk0 + it) * QF_KC;

    // ---- quantize two 1x16 blocks (32 elements = 4 x 16-byte chunks of this row)
    {
      const uint8_t* rowp = xs + q_row * 128;
      const int sw = q_row & 7;
      uint4 v[4];
#pragma unroll
      for (int i = 0; i < 4; ++i)
        v[i] = *reinterpret_cast<const uint4*>(rowp + (((q_half * 4 + i) ^ sw) << 4));
      uint32_t sf8a, sf8b;
      float enca, encb;
      block_scale(fmaxf(amax_bf16x8(v[0]), amax_bf16x8(v[1])), ts, sf8a, enca);
      block_scale(fmaxf(amax_bf16x8(v[2]), amax_bf16x8(v[3])), ts, sf8b, encb);
      uint4 c;
      c.x = quant_bf16x8(v[0], enca);
      c.y = quant_bf16x8(v[1], enca);
      c.z = quant_bf16x8(v[2], encb);
      c.w = quant_bf16x8(v[3], encb);
      uint32_t sfpair = sf8a | (sf8b << 8);
      const uint32_t other = __shfl_xor_sync(0xffffffffu, sfpair, 1);
      if (q_live) {
        *reinterpret_cast<uint4*>(p.codes + q_grow * (p.cols / 2) + (kcol + q_half * 32) / 2) = c;
        if (q_half == 0) {
          const uint32_t word = sfpair | (other << 16);
          const int64_t kb0 = kcol / 16;
          const int64_t off = (p.sf_layout == FT_SF_TILE128x4) ? sf_tile_offset(q_grow, kb0, nblk)
                                                               : q_grow * nblk + kb0;
          *reinterpret_cast<uint32_t*>(p.sf + off) = word;
        }
      }
    }

    // ---- projection: acc += X[16 rows, 64 k] * D[64 k, r_t]
    if constexpr (R_T > 0) {
      const uint32_t xs_u = smem_u32(xs);
      const uint32_t ds_u = xs_u + QF_X_BYTES;
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) {
        uint32_t a0, a1, a2, a3;
        {
          const int r = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
          const int c = ks * 2 + (lane >> 4);
          ldsm_x4(xs_u + r * 128 + ((c ^ (r & 7)) << 4), a0, a1, a2, a3);
        }
#pragma unroll
        for (int j = 0; j < NT; j += 2) {
          const int kr = ks * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
          const int nt = j + (lane >> 4);
          uint32_t b0, b1, b2, b3;
          ldsm_x4_t(ds_u + (nt >> 3) * QF_DG_BYTES + kr * 128 + (((nt & 7) ^ (kr & 7)) << 4), b0, b1,
                    b2, b3);
          mma_16816(acc[j], a0, a1, a2, a3, b0, b1);
          if (j + 1 < NT) mma_16816(acc[j + 1], a0, a1, a2, a3, b2, b3);
        }
      }
    }
    __syncthreads();  // every thread is done with stage s
    if (tid == 0 && it + QF_STAGES < n_chunks) issue(it + QF_STAGES);
  }

  // ---- cluster reduction of the partial H tiles and output
  if constexpr (R_T > 0) {
    float* part = reinterpret_cast<float*>(smem);  // [128][R_T] fp32, reuses the ring
    {
      const int g = lane >> 2, t = lane & 3;
#pragma unroll
      for (int j = 0; j < NT; ++j) {
        const int r = warp * 16 + g, c = j * 8 + 2 * t;
        *reinterpret_cast<float2*>(part + r * R_T + c) = make_float2(acc[j][0], acc[j][1]);
        *reinterpret_cast<float2*>(part + (r + 8) * R_T + c) = make_float2(acc[j][2], acc[j][3]);
      }
    }
    if (split > 1) cluster_sync_all(); else __syncthreads();
    const int rows_per = QF_ROWS / split;
    const int r_begin = (int)blockIdx.y * rows_per;
    float alpha = 1.0f;
    if (p.hs_out != nullptr) alpha = __fmul_rn(ts.g_dec, __ldg(p.other_dec_scale));
    const uint32_t part_u = smem_u32(part);
    for (int e = tid; e < rows_per * (R_T / 2); e += QF_THREADS) {
      const int r = r_begin + e / (R_T / 2), c = (e % (R_T / 2)) * 2;
      float s0 = 0.f, s1 = 0.f;
      if (split > 1) {
        for (int q = 0; q < split; ++q) {
          s0 += ld_dsmem_f32(part_u + (r * R_T + c) * 4, q);
          s1 += ld_dsmem_f32(part_u + (r * R_T + c + 1) * 4, q);
        }
      } else {
        s0 = part[r * R_T + c];
        s1 = part[r * R_T + c + 1];
      }
      const int64_t gr = row0 + r;
      if (gr < p.rows) {
        if (p.h_out != nullptr)
          *reinterpret_cast<uint32_t*>(p.h_out + gr * R_T + c) = pack_bf16x2(s0, s1);
        if (p.hs_out != nullptr)
          *reinterpret_cast<uint32_t*>(p.hs_out + gr * R_T + c) =
              pack_bf16x2(__fdiv_rn(s0, alpha), __fdiv_rn(s1, alpha));
      }
    }
    if (split > 1) cluster_sync_all();  // keep this CTA's smem alive until all peers have read it
  }
}

template <int R_T>
static int launch_qf(const CUtensorMap& mx, const CUtensorMap& md, const QFParams& p,
                     cudaStream_t st) {
  constexpr int NG = (R_T + 63) / 64;
  const int smem = QF_STAGES * (QF_X_BYTES + NG * QF_DG_BYTES) + 1024;
  static_assert(QF_ROWS * (R_T > 0 ? R_T : 1) * 4 <= QF_STAGES * (QF_X_BYTES + NG * QF_DG_BYTES),
                "partial H tile must fit in the ring");
  FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)ceil_div(p.rows, QF_ROWS), (unsigned)p.split, 1);
  cfg.blockDim = dim3(QF_THREADS, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 1;
  attr[0].val.clusterDim.y = (unsigned)p.split;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_quantize_fused<R_T>, mx, md, p));
  return FT_OK;
}

// choose the cluster size: smallest power of two <= 8 that divides the chunk count
// and gives >= ~0.9 waves of CTAs, else the largest that divides.
static int choose_split(int64_t rows, int64_t cols) {
  const int64_t tiles = ceil_div(rows, QF_ROWS), chunks = cols / QF_KC;
  const int sms = sm_count();
  int best = 1;
  for (int s = 1; s <= 8; s *= 2) {
    if (chunks % s != 0) break;
    best = s;
    if (tiles * s >= (int64_t)(0.9 * sms)) break;
  }
  return best;
}

int launch_quantize_fused(const void* x, int64_t rows, int64_t cols, const float* amax_t,
                          const ft_proj* proj, ft_qtensor* out, cudaStream_t st) {
  const int r_t = proj ? proj->r_t : 0;
  CUtensorMap mx, md;
  int rc = make_tensor_map_2d(&mx, x, 2, (uint64_t)cols, (uint64_t)rows, (uint64_t)cols * 2, QF_KC,
                              QF_ROWS, Swizzle::B128);
  if (rc != FT_OK) return rc;
  if (r_t > 0) {
    rc = make_tensor_map_2d(&md, proj->down, 2, (uint64_t)r_t, (uint64_t)cols, (uint64_t)r_t * 2, 64,
                            QF_KC, Swizzle::B128);
    if (rc != FT_OK) return rc;
  } else {
    md = mx;
  }
  QFParams p;
  p.rows = rows;
  p.cols = cols;
  p.amax_t = amax_t;
  p.codes = out->codes;
  p.sf = out->sf;
  p.g_dec_out = out->tensor_dec_scale;
  p.sf_layout = out->sf_layout;
  p.h_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out) : nullptr;
  p.hs_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out_scaled) : nullptr;
  p.other_dec_scale = proj ? proj->other_dec_scale : nullptr;
  p.split = choose_split(rows, cols);
  // padding rows of the last 128-row scale tile must read as zero
  if (out->sf_layout == FT_SF_TILE128x4 && rows % 128 != 0) {
    const int64_t tiles_c = ceil_div(cols / 16, 4);
    FT_CUDA_TRY(cudaMemsetAsync(out->sf + (rows / 128) * tiles_c * 512, 0, tiles_c * 512, st));
  }
  switch (r_t) {
    case 0: return launch_qf<0>(mx, md, p, st);
    case 16: return launch_qf<16>(mx, md, p, st);
    case 32: return launch_qf<32>(mx, md, p, st);
    case 48: return launch_qf<48>(mx, md, p, st);
    case 64: return launch_qf<64>(mx, md, p, st);
    case 80: return launch_qf<80>(mx, md, p, st);
    case 96: return launch_qf<96>(mx, md, p, st);
    case 112: return launch_qf<112>(mx, md, p, st);
    case 128: return launch_qf<128>(mx, md, p, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
