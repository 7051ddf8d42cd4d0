// quantize_fused.cu -- a1 / a3: one pass over X (or G) that emits the NVFP4 codes,
// the block scales and the low-rank down-projection H = X * D ("fuse
// ... quantization and down-projection").
//
// Decomposition: a CTA owns 128 rows x (cols / SPLIT) columns and walks them in
// 128 x 64 chunks that TMA stages into shared memory (SWIZZLE_128B) through a
// 3/4-deep mbarrier ring.  From one staged chunk
//   - 512 threads quantize: thread (row = tid/4, quarter = tid%4) owns one 1x16 block;
//   - one thread issues tcgen05.mma kind::f16 (M = 128, N = r_t, K = 16, four per chunk):
//     A = the staged chunk itself (K-major, the TMA swizzle is the UMMA canonical layout),
//     B = the 64 x r_t slice of D staged beside it (MN-major), accumulator in tensor memory.
//     The staged bytes are read once by the tensor core instead of once per warp by ldmatrix.
// Two CTAs are resident per SM (32 warps): the per-block scale arithmetic is a long
// dependent chain (three IEEE divisions) and needs the warps to hide its latency.
// The SPLIT CTAs of a 128-row tile form a thread-block cluster (1, SPLIT, 1); their
// fp32 partial H tiles are summed through distributed shared memory, so H is
// complete in one pass with no atomics and no second kernel.
#include <cstdio>
#include <cstdlib>

#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

constexpr int QF_ROWS = 128;    // rows per CTA
constexpr int QF_KC = 64;       // columns per chunk (128 bytes of bf16 = one swizzle row)
constexpr int QF_THREADS = 512;
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

__device__ __forceinline__ float2 ld_dsmem_f32x2(uint32_t local_addr, uint32_t cta_rank) {
  uint32_t remote;
  float2 v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local_addr), "r"(cta_rank));
  asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(remote));
  return v;
}

// R_T: width of the projection (0 = quantize only).  NG = 64-column groups of D.
template <int R_T>
__global__ void __launch_bounds__(QF_THREADS, 2)
k_quantize_fused(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_d,
                 const QFParams p) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr uint32_t TMEM_COLS = R_T <= 32 ? 32 : (R_T <= 64 ? 64 : 128);
  constexpr int QF_STAGES = (NG == 2) ? 3 : 4;
  constexpr int STAGE_BYTES = QF_X_BYTES + NG * QF_DG_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment for the 128-byte swizzle atoms
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_bar[4], empty_bar[4];
  __shared__ float enc_tab[128];
  __shared__ uint64_t acc_bar;
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t row0 = (int64_t)blockIdx.x * QF_ROWS;
  const int split = p.split;
  const int64_t chunks_total = p.cols / QF_KC;
  const int n_chunks = (int)((chunks_total - blockIdx.y + split - 1) / split);  // interleaved, may be uneven
  // chunk `it` of this CTA is global chunk it * split + blockIdx.y: the CTAs of a cluster walk
  // the columns interleaved, so together they touch split * 128 contiguous bytes of each row at
  // about the same time (DRAM page locality) instead of `split` far-apart 128-byte pieces.

  if (tid == 0) {
    prefetch_tmap(&map_x);
    if (R_T > 0) prefetch_tmap(&map_d);
    for (int s = 0; s < QF_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], QF_THREADS / 32 + (R_T > 0 ? 1 : 0));  // every warp (+ the MMA commit)
    }
    mbar_init(&acc_bar, 1);
    fence_mbar_init();
  }
  if (R_T > 0 && warp == 2) {
    tmem_alloc(&tmem_base_s, TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  auto issue = [&](int it) {
    const int s = it % QF_STAGES;
    uint8_t* base = smem + s * STAGE_BYTES;
    const int32_t kcol = (int32_t)(((int64_t)it * split + blockIdx.y) * QF_KC);
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
  if (tid < 128) enc_tab[tid] = enc_of_sf8((uint32_t)tid, ts.g_dec);
  __syncthreads();

  // quantizer role of this thread
  const int q_row = tid >> 2, q_quarter = tid & 3;
  const int64_t q_grow = row0 + q_row;
  const bool q_live = q_grow < p.rows;
  const int64_t nblk = p.cols / 16;
  const uint32_t q_smem_base = smem_u32(smem) + q_row * 128;
  const uint32_t q_smem_off0 = q_smem_base + (((q_quarter * 2) ^ (q_row & 7)) << 4);
  const uint32_t q_smem_off1 = q_smem_base + (((q_quarter * 2 + 1) ^ (q_row & 7)) << 4);
  // output cursors: chunk `it` is global chunk it * split + blockIdx.y
  uint8_t* q_codes = p.codes + q_grow * (p.cols / 2) + ((int64_t)blockIdx.y * QF_KC + q_quarter * 16) / 2;
  const int64_t q_codes_step = (int64_t)split * (QF_KC / 2);
  uint8_t* q_sf = p.sf + ((p.sf_layout == FT_SF_TILE128x4) ? sf_tile_offset(q_grow, (int64_t)blockIdx.y * 4, nblk)
                                                           : q_grow * nblk + (int64_t)blockIdx.y * 4);
  const int64_t q_sf_step = (p.sf_layout == FT_SF_TILE128x4) ? (int64_t)split * 512 : (int64_t)split * 4;
  for (int it = 0; it < n_chunks; ++it) {
    const int s = it % QF_STAGES;
    const uint32_t parity = (it / QF_STAGES) & 1;
    // refill, one iteration late: warp 0 re-arms the slot of chunk it-1 once every warp has
    // released it; no block-wide barrier, so the other warps run ahead through the ring
    if (warp == 0 && it > 0) {
      if (lane == 0 && it - 1 + QF_STAGES < n_chunks) {
        mbar_wait(&empty_bar[(it - 1) % QF_STAGES], ((it - 1) / QF_STAGES) & 1);
        issue(it - 1 + QF_STAGES);
      }
      __syncwarp();
    }
    mbar_wait(&full_bar[s], parity);

    // ---- quantize one 1x16 block (two 16-byte chunks of this row)
    {
      uint4 v0, v1;
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(v0.x), "=r"(v0.y), "=r"(v0.z), "=r"(v0.w) : "r"(q_smem_off0 + s * STAGE_BYTES));
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(v1.x), "=r"(v1.y), "=r"(v1.z), "=r"(v1.w) : "r"(q_smem_off1 + s * STAGE_BYTES));
      const uint32_t sf8 = block_sf8(amax_block16(v0, v1), ts.g_enc);
      const float enc = enc_tab[sf8];
      uint2 c;
      c.x = quant_bf16x8_fast(v0, enc);
      c.y = quant_bf16x8_fast(v1, enc);
      // gather the row's four scale bytes into the quarter-0 lane
      uint32_t w = sf8 << (8 * q_quarter);
      w |= __shfl_xor_sync(0xffffffffu, w, 1);
      w |= __shfl_xor_sync(0xffffffffu, w, 2);
      if (q_live) {
        *reinterpret_cast<uint2*>(q_codes) = c;
        if (q_quarter == 0) *reinterpret_cast<uint32_t*>(q_sf) = w;
      }
      q_codes += q_codes_step;
      q_sf += q_sf_step;
    }

    // ---- projection: acc[128 x r_t] += X[128, 64 k] * D[64 k, r_t], issued by one thread
    if constexpr (R_T > 0) {
      if (warp == 1) {
        if (lane == 0) {
          tc_fence_after();
          const uint32_t xs_u = smem_u32(smem) + s * STAGE_BYTES;
          const uint32_t ds_u = xs_u + QF_X_BYTES;
          constexpr uint32_t idesc = idesc_bf16(QF_ROWS, R_T) | (1u << 16);  // B is MN-major
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mma_bf16(tmem_base_s, make_smem_desc(xs_u + k * 32, 1024, 0, 2),
                     make_smem_desc(ds_u + k * 2048, 1024, QF_DG_BYTES, 2), idesc, (it | k) != 0);
          tc_commit(&empty_bar[s]);                       // slot free once the MMAs have read it
          if (it == n_chunks - 1) tc_commit(&acc_bar);    // accumulator complete
        }
        __syncwarp();
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[s]);  // this warp is done with stage s
  }
  __syncthreads();  // every warp has consumed every stage: the ring can be reused below

  // ---- cluster reduction of the partial H tiles and output
  if constexpr (R_T > 0) {
    float* part = reinterpret_cast<float*>(smem);  // [128][R_T] fp32, reuses the ring
    if (warp < 4) {   // warp w may read TMEM lanes 32w .. 32w+31 = rows of the tile
      mbar_wait(&acc_bar, 0);
      tc_fence_after();
      const int r = warp * 32 + lane;
#pragma unroll
      for (int c0 = 0; c0 < R_T; c0 += 16) {
        uint32_t v[16];
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
              "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
            : "r"(tmem_base_s + ((uint32_t)(warp * 32) << 16) + c0)
            : "memory");
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; j += 4)   // rotate the 16-byte pieces by row to spread the banks
          *reinterpret_cast<uint4*>(part + r * R_T + c0 + ((j + 4 * (r & 3)) & 15)) =
              make_uint4(v[(j + 4 * (r & 3)) & 15], v[(j + 4 * (r & 3) + 1) & 15], v[(j + 4 * (r & 3) + 2) & 15],
                         v[(j + 4 * (r & 3) + 3) & 15]);
      }
      tc_fence_before();
    }
    if (split > 1) cluster_sync_all(); else __syncthreads();
    const int rows_per = (QF_ROWS + split - 1) / split;
    const int r_begin = (int)blockIdx.y * rows_per;
    float alpha = 1.0f;
    if (p.hs_out != nullptr) alpha = __fmul_rn(ts.g_dec, __ldg(p.other_dec_scale));
    const uint32_t part_u = smem_u32(part);
    for (int e = tid; e < rows_per * (R_T / 2); e += QF_THREADS) {
      const int r = r_begin + e / (R_T / 2), c = (e % (R_T / 2)) * 2;
      if (r >= QF_ROWS) break;
      float s0 = 0.f, s1 = 0.f;
      if (split > 1) {
        float2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q)   // all remote loads in flight before the first add
          if (q < split) v[q] = ld_dsmem_f32x2(part_u + (r * R_T + c) * 4, q);
#pragma unroll
        for (int q = 0; q < 8; ++q)
          if (q < split) {
            s0 += v[q].x;
            s1 += v[q].y;
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
    if (warp == 2) {
      tc_fence_after();
      tmem_dealloc(tmem_base_s, TMEM_COLS);
    }
  }
}

template <int R_T>
static int choose_split(int64_t rows, int64_t cols, int smem);

template <int R_T>
static int launch_qf(const CUtensorMap& mx, const CUtensorMap& md, const QFParams& p_in,
                     cudaStream_t st) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr int QF_STAGES = (NG == 2) ? 3 : 4;
  const int smem = QF_STAGES * (QF_X_BYTES + NG * QF_DG_BYTES) + 1024;
  static_assert(QF_ROWS * (R_T > 0 ? R_T : 1) * 4 <= QF_STAGES * (QF_X_BYTES + NG * QF_DG_BYTES),
                "partial H tile must fit in the ring");
  FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                   cudaSharedmemCarveoutMaxShared));
  QFParams p = p_in;
  p.split = choose_split<R_T>(p.rows, p.cols, smem);
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

// Cluster size (= K split) of the fused kernel: any 1..8.  Clusters are co-scheduled inside a
// GPC, so not every size packs the chip equally; ask the driver how many clusters of each size
// fit at once and minimise  waves * chunks-per-CTA  (ties: the larger split = more warps).
template <int R_T>
static int choose_split(int64_t rows, int64_t cols, int smem) {
  const int64_t tiles = ceil_div(rows, QF_ROWS), chunks = cols / QF_KC;
  if (const char* e = getenv("FT_QF_SPLIT")) {
    const int v = atoi(e);
    if (v > 0 && v <= 8 && v <= chunks) return v;
  }
  static int max_active[9] = {0};   // per instantiation; device properties do not change
  int best = 1;
  double best_cost = 1e30;
  for (int s = 1; s <= 8 && s <= chunks; ++s) {
    if (max_active[s] == 0) {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(1, (unsigned)s, 1);
      cfg.blockDim = dim3(QF_THREADS, 1, 1);
      cfg.dynamicSmemBytes = smem;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = 1;
      attr[0].val.clusterDim.y = (unsigned)s;
      attr[0].val.clusterDim.z = 1;
      cfg.attrs = attr;
      cfg.numAttrs = 1;
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, k_quantize_fused<R_T>, &cfg) != cudaSuccess || n < 1) {
        (void)cudaGetLastError();
        n = -1;
      }
      max_active[s] = n;
    }
    if (max_active[s] < 1) continue;
    const double waves = (double)ceil_div(tiles, max_active[s]);
    const double cost = waves * (double)ceil_div(chunks, s) + 1.5;   // + a fixed head/tail per CTA
    if (cost <= best_cost) {
      best_cost = cost;
      best = s;
    }
  }
  if (getenv("FT_QF_DEBUG")) {
    fprintf(stderr, "[qf] r_t=%d rows=%ld cols=%ld split=%d max_active:", R_T, (long)rows, (long)cols, best);
    for (int s = 1; s <= 8; ++s) fprintf(stderr, " %d", max_active[s]);
    fprintf(stderr, "\n");
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
  p.split = 1;
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
