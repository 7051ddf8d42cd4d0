// quantize_fused.cu -- a1 / a3 (and a0 folded in): one kernel that emits the NVFP4 codes, the
// block scales and the low-rank down-projection H = X * D of a bf16 matrix (PAPER.md:110,
// "fuse ... quantization and down-projection").
//
// Decomposition.  The matrix is cut into 128-row x 64-column chunks (16 KB), numbered row tile
// major.  CTA i of a persistent grid owns the contiguous chunk range [i*TC/G, (i+1)*TC/G): every
// CTA has the same number of chunks (+-1) whatever the shape -- no row-tile x split quantisation --
// and a range touches at most two row tiles when it is no longer than a row of chunks.
// From one TMA-staged chunk (SWIZZLE_128B)
//   - 512 threads quantize: thread (row = tid/4, quarter = tid%4) owns one 1x16 block;
//   - one thread issues tcgen05.mma kind::f16 (M = 128, N = r_t, K = 16, four per chunk):
//     A = the staged chunk itself (K-major), B = the 64 x r_t slice of D staged in its own ring
//     (MN-major), accumulator in tensor memory.
// Warps 0-15 quantize, warp 16 is the TMA producer, warp 17 the tcgen05 issuer (a quantizer warp that
// also issues the MMAs is ~400 cycles slower per chunk than its peers and sets the pace of the ring).
// At the end of a row-tile segment the fp32 partial H tile goes TMEM -> plain vector stores into the
// segment's own 128 x r_t slot of the workspace (slot = CTA index + row tile: unique, and the slots of
// one row tile are consecutive).  Once every slot is written, each row's slots are summed in CTA order
// and leave as bf16 H and Hs = H * (1 / alpha): no atomics on the data, a fixed summation order.
// Measured and dropped: fp32 reductions into one accumulator (REDG issues at ~1.3 cycles per lane and
// word: 10 k cycles per 128 x 64 tile) and a last-arriver CTA finishing a whole row tile alone (a
// 9-17 k-cycle tail on 36 of 296 CTAs).
//
// Two modes, one kernel template:
//   streaming (amax known): chunks stream through a 4-deep ring, two CTAs per SM (48 registers: 18
//     warps put 10 on one SM sub-partition, 10 x 32 x 48 fits its 16 K registers); the slot sums are
//     done by k_finalize_h, launched behind it with a programmatic edge.  A grid barrier inside the
//     kernel would need a cooperative launch, and the runtime admits one CTA per SM of a kernel that
//     allocates tensor memory.
//   single pass (amax not known, tensor <= 12 chunks per SM = 29 MB on 148 SMs): one CTA per SM, every
//     chunk stays resident in shared memory; phase 1 finds the tensor amax (and runs the projection
//     MMAs) as the chunks land, a grid-wide barrier publishes it, phase 2 quantizes from shared
//     memory, a second grid barrier precedes the slot sums (each CTA an equal share of the rows); it is
//     split-phase: a CTA arrives as soon as its slots are written (before phase 2) and waits after
//     phase 2, when every CTA has long arrived.
//     The tensor is read from HBM exactly once and the separate amax kernel (a0) disappears.
//     Launched cooperatively (all CTAs co-resident); the barrier spin traps after 2 s instead of hanging.
#include <cstdio>
#include <cstdlib>

#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

constexpr int QF_ROWS = 128;    // rows per chunk
constexpr int QF_KC = 64;       // columns per chunk (128 bytes of bf16 = one swizzle row)
constexpr int QF_QTHREADS = 512;              // quantizer threads (warps 0-15)
constexpr int QF_THREADS = QF_QTHREADS + 64;  // + warp 16: TMA producer, warp 17: tcgen05 issuer
constexpr int QF_X_BYTES = QF_ROWS * QF_KC * 2;  // 16 KB
constexpr int QF_DG_BYTES = QF_KC * 128;         // one 64-column group of D: 8 KB
constexpr int QF_MAX_NX = 12;   // resident chunks per CTA in single-pass mode
constexpr int QF_MAX_ND = 4;
constexpr int QF_MAX_GRID = WS_MAX_QUANT_CTAS;   // the workspace has one slot per CTA + one per row tile

struct QFParams {
  int64_t rows, cols;
  const float* amax_in;         // streaming: tensor amax (device)
  uint32_t* amax_bits;          // single pass: zeroed word, receives the amax bit pattern
  uint32_t* grid_bar;           // two zeroed arrival counters: [0] amax published (single pass), [1] slots written
  float* slots;                 // [(grid + row tiles) x 128 x r_t] fp32 partial H tiles (not zeroed)
  uint8_t* codes;
  uint8_t* sf;
  float* g_dec_out;
  int sf_layout;
  __nv_bfloat16* h_out;         // [rows x r_t] or null
  __nv_bfloat16* hs_out;        // [rows x r_t] or null
  const float* other_dec_scale; // for hs_out
  int single;                   // 1: single-pass mode
  int nx, nd;                   // ring depths (single pass: nx = max chunks per CTA)
  int chunks_per_tile;          // C = cols / 64
  int64_t total_chunks;         // TC = row tiles * C
};

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ uint64_t globaltimer_ns() {
  uint64_t t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// R_T: width of the projection (0 = quantize only).  NG = 64-column groups of D.
// Registers: 18 warps land 5/5/4/4 on the four SM sub-partitions (16 K registers each), so two resident
// CTAs put 10 warps on one of them: 10 x 32 x 48 = 15 360 fits, 56 per thread (what
// __launch_bounds__(576, 2) would allow) does not, and the streaming kernel would silently run one
// CTA per SM.
template <int R_T, bool SINGLE>
__global__ void __launch_bounds__(QF_THREADS) __maxnreg__(SINGLE ? 96 : 48)
k_quantize_fused(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_d,
                 const QFParams p) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr uint32_t ACC_COLS = R_T <= 32 ? 32 : (R_T <= 64 ? 64 : 128);
  constexpr int D_BYTES = NG * QF_DG_BYTES;
  constexpr int NXS = NG == 2 ? 3 : 4;     // streaming mode: ring depth (X chunk + D slice per stage)
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment for the 128-byte swizzle atoms
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_x[QF_MAX_NX], empty_x[QF_MAX_ND], full_d[QF_MAX_ND], empty_d[QF_MAX_ND];
  __shared__ uint64_t acc_full[2], acc_free[2];
  __shared__ float enc_tab[128];
  __shared__ uint32_t tmem_base_s, s_red[QF_QTHREADS / 32], s_amax;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t c_begin = (int64_t)blockIdx.x * p.total_chunks / gridDim.x;
  const int n = (int)(((int64_t)blockIdx.x + 1) * p.total_chunks / gridDim.x - c_begin);   // >= 1 (grid <= TC)
  const int C = p.chunks_per_tile;
  const uint32_t xs_u = smem_u32(smem);
  const uint32_t ds_u = xs_u + (uint32_t)p.nx * QF_X_BYTES;

  if (tid == 0) {
    prefetch_tmap(&map_x);
    if (R_T > 0) prefetch_tmap(&map_d);
    for (int s = 0; s < QF_MAX_NX; ++s) mbar_init(&full_x[s], 1);
    for (int s = 0; s < QF_MAX_ND; ++s) {
      mbar_init(&empty_x[s], QF_QTHREADS / 32 + (R_T > 0 ? 1 : 0));  // every quantizer warp (+ the MMA commit)
      mbar_init(&full_d[s], 1);
      mbar_init(&empty_d[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&acc_full[a], 1);   // tcgen05.commit of a segment's last MMA
      mbar_init(&acc_free[a], 4);   // the four drain warps
    }
    fence_mbar_init();
  }
  if (R_T > 0 && warp == 2) {
    tmem_alloc(&tmem_base_s, 2 * ACC_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();      // streaming mode inside ft_linear_bwd: the amax comes from the dB^T kernel before us
  pdl_trigger();   // the kernel that follows may set itself up while this one runs (it waits for our end)

  // chunk `it` of this CTA is global chunk c_begin + it = (row tile t, column chunk kc)
  auto issue_x = [&](int it, int slot) {
    const int64_t c = c_begin + it;
    const int t = (int)(c / C), kc = (int)(c % C);
    mbar_expect_tx(&full_x[slot], QF_X_BYTES);
    tma_load_2d(smem + slot * QF_X_BYTES, &map_x, &full_x[slot], kc * QF_KC, t * QF_ROWS);
  };
  auto issue_d = [&](int it, int slot) {
    const int kc = (int)((c_begin + it) % C);
    mbar_expect_tx(&full_d[slot], D_BYTES);
#pragma unroll
    for (int g = 0; g < NG; ++g)
      tma_load_2d(smem + p.nx * QF_X_BYTES + slot * D_BYTES + g * QF_DG_BYTES, &map_d, &full_d[slot], g * 64,
                  kc * QF_KC);
  };
  // the four MMAs of one chunk: acc[128 x r_t] (+)= X[128, 64 k] * D[64 k, r_t]
  auto issue_mma = [&](uint32_t x_u, uint32_t d_u, uint32_t acc, bool first) {
    constexpr uint32_t idesc = idesc_bf16(QF_ROWS, R_T > 0 ? R_T : 16) | (1u << 16);  // B is MN-major
#pragma unroll
    for (int k = 0; k < 4; ++k)
      mma_bf16(acc, make_smem_desc(x_u + k * 32, 1024, 0, 2), make_smem_desc(d_u + k * 2048, 1024, QF_DG_BYTES, 2),
               idesc, !(first && k == 0));
  };

  // quantizer role of this thread: one 1x16 block (two 16-byte pieces of a swizzled row) per chunk
  const int q_row = tid >> 2, q_quarter = tid & 3;
  const uint32_t q_off0 = q_row * 128 + (((q_quarter * 2) ^ (q_row & 7)) << 4);
  const uint32_t q_off1 = q_off0 ^ 16;
  const bool sf_tiled = p.sf_layout == FT_SF_TILE128x4;
  // output cursor (32-bit byte offsets; the host rejects tensors whose codes exceed 4 GB): advanced
  // one chunk at a time, no per-chunk index arithmetic
  int o_t = (int)(c_begin / C), o_kc = (int)(c_begin % C);
  uint32_t o_co, o_so;
  bool o_live;
  {
    const uint32_t nblk = (uint32_t)(p.cols / 16), half_cols = (uint32_t)(p.cols / 2);
    const uint32_t grow = (uint32_t)o_t * QF_ROWS + q_row;
    o_live = (int64_t)grow < p.rows;
    o_co = grow * half_cols + o_kc * 32 + q_quarter * 8;
    o_so = sf_tiled ? ((uint32_t)o_t * C + o_kc) * 512 + (q_row & 31) * 16 + (q_row >> 5) * 4 : grow * nblk + o_kc * 4;
  }
  auto advance_out = [&]() {
    o_co += 32;
    o_so += sf_tiled ? 512 : 4;
    if (++o_kc == C) {     // row tile change: 128 rows down, C chunks back
      o_kc = 0;
      ++o_t;
      o_co += 127u * (uint32_t)(p.cols / 2);
      if (!sf_tiled) o_so += 127u * (uint32_t)(p.cols / 16);
      o_live = (int64_t)o_t * QF_ROWS + q_row < p.rows;
    }
  };
  auto load_block = [&](uint32_t x_u, uint4& v0, uint4& v1) {
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v0.x), "=r"(v0.y), "=r"(v0.z), "=r"(v0.w) : "r"(x_u + q_off0));
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v1.x), "=r"(v1.y), "=r"(v1.z), "=r"(v1.w) : "r"(x_u + q_off1));
  };
  const uint32_t enc_u = smem_u32(enc_tab), full_u = smem_u32(full_x), empty_u = smem_u32(empty_x);
  // release_u: shared address of the slot's empty barrier, or 0 (single-pass mode: nothing to release).
  // The slot is handed back as soon as the block is in registers (the amax tree consumes all eight
  // loaded words, so the loads have completed), not after the ~100 instructions of arithmetic and the
  // stores: the ring looks deeper to the producer.
  auto quantize_chunk = [&](uint32_t x_u, float g_enc, uint32_t release_u) {
    uint4 v0, v1;
    load_block(x_u, v0, v1);
    const float amax_b = amax_block16(v0, v1);
    if (release_u != 0) {
      __syncwarp();
      if (lane == 0) mbar_arrive_u32(release_u);
    }
    const uint32_t sf8 = block_sf8(amax_b, g_enc);
    float enc;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(enc) : "r"(enc_u + sf8 * 4));
    uint2 c;
    c.x = quant_bf16x8_fast(v0, enc);
    c.y = quant_bf16x8_fast(v1, enc);
    // gather the row's four scale bytes into the quarter-0 lane
    uint32_t w = sf8 << (8 * q_quarter);
    w |= __shfl_xor_sync(0xffffffffu, w, 1);
    w |= __shfl_xor_sync(0xffffffffu, w, 2);
    if (o_live) {
      *reinterpret_cast<uint2*>(p.codes + o_co) = c;
      if (q_quarter == 0) *reinterpret_cast<uint32_t*>(p.sf + o_so) = w;
    }
  };

  // barrier of the 16 quantizer warps only (the producer and the issuer warp run free)
  auto qsync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(QF_QTHREADS) : "memory"); };

  // ---- projection bookkeeping.  A "segment" is this CTA's run of chunks inside one row tile; its
  // fp32 partial H tile accumulates in TMEM accumulator (segment & 1).
  // drain: TMEM -> the segment's slot in the workspace, by warps 0-3, with no block-wide barrier (the
  // other warps keep quantizing).
  auto drain_segment = [&](int t, int seg) {
    const int a = seg & 1;
    if (warp < 4) {   // warp w may read TMEM lanes 32w .. 32w+31 = rows of the tile
      mbar_wait(&acc_full[a], (uint32_t)(seg >> 1) & 1);
      tc_fence_after();
      // slot layout [column quad q = c / 4][row][4 floats]: a warp's store instruction covers 512
      // contiguous bytes (full sectors), and so does a warp's load in the finalizer
      float* dst = p.slots + ((int64_t)blockIdx.x + t) * (QF_ROWS * R_T) + (warp * 32 + lane) * 4;
#pragma unroll 1
      for (int c0 = 0; c0 < R_T; c0 += 16) {
        uint32_t v[16];
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
              "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
            : "r"(tmem_base_s + ((uint32_t)(warp * 32) << 16) + a * ACC_COLS + c0)
            : "memory");
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; j += 4)
          *reinterpret_cast<uint4*>(dst + (c0 + j) / 4 * (QF_ROWS * 4)) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&acc_free[a]);   // the accumulator may be overwritten
    }
  };
  // After the grid barrier every partial H tile is in its slot.  CTA i completes rows
  // [i * rows / G, (i + 1) * rows / G): fp32 sum of the row tile's slots in CTA order (fixed order:
  // the result does not depend on timing) -> bf16 H and Hs = H * (1 / alpha).
  auto finalize_share = [&](float inv_alpha) {
    constexpr int QUADS = R_T > 0 ? R_T / 4 : 1;
    constexpr int SLOT_F4 = QF_ROWS * (R_T > 0 ? R_T : 4) / 4;
    const int64_t TC = p.total_chunks, G = gridDim.x;
    const int64_t r_begin = (int64_t)blockIdx.x * p.rows / G;
    const int nrows = (int)(((int64_t)blockIdx.x + 1) * p.rows / G - r_begin);
    // item e -> (row e % nrows, column quad e / nrows): neighbouring threads read neighbouring rows
    for (int e = tid; e < nrows * QUADS; e += QF_QTHREADS) {
      const int64_t gr = r_begin + e % nrows;
      const int q = e / nrows;
      const int t = (int)(gr / QF_ROWS), r = (int)(gr % QF_ROWS);
      // the CTAs whose ranges meet row tile t: owner(c) = floor(((c + 1) * G - 1) / TC)
      const int i_lo = (int)((((int64_t)t * C + 1) * G - 1) / TC);
      const int i_hi = (int)((((int64_t)(t + 1) * C) * G - 1) / TC);
      const float4* src = reinterpret_cast<const float4*>(p.slots) + ((int64_t)i_lo + t) * SLOT_F4 + q * QF_ROWS + r;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int i = i_lo; i <= i_hi; i += 4) {   // four loads in flight, added in order
        float4 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          v[j] = (i + j <= i_hi) ? __ldcg(src + (int64_t)j * SLOT_F4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc.x += v[j].x;
          acc.y += v[j].y;
          acc.z += v[j].z;
          acc.w += v[j].w;
        }
        src += 4 * (int64_t)SLOT_F4;
      }
      if (p.h_out != nullptr)
        *reinterpret_cast<uint2*>(p.h_out + gr * R_T + q * 4) =
            make_uint2(pack_bf16x2(acc.x, acc.y), pack_bf16x2(acc.z, acc.w));
      if (p.hs_out != nullptr)
        *reinterpret_cast<uint2*>(p.hs_out + gr * R_T + q * 4) =
            make_uint2(pack_bf16x2(__fmul_rn(acc.x, inv_alpha), __fmul_rn(acc.y, inv_alpha)),
                       pack_bf16x2(__fmul_rn(acc.z, inv_alpha), __fmul_rn(acc.w, inv_alpha)));
    }
  };

  if constexpr (!SINGLE) {
    // =========================================================== streaming mode (amax known)
    // a stage = the X chunk and its D slice; both land on full_x[slot] (issue_d is given that barrier)
    const uint64_t pol_stream = l2_policy_evict_first();
    auto issue_stage = [&](int it, int slot) {
      const int64_t c = c_begin + it;
      const int t = (int)(c / C), kc = (int)(c % C);
      mbar_expect_tx(&full_x[slot], QF_X_BYTES + (R_T > 0 ? D_BYTES : 0));
      // streaming mode reads its tensor for the last time: evict-first, so that what the pass before left
      // in L2 (the dB^T pass over the same G) is not displaced by lines nobody reads again
      tma_load_2d_hint(smem + slot * QF_X_BYTES, &map_x, &full_x[slot], kc * QF_KC, t * QF_ROWS, pol_stream);
      if constexpr (R_T > 0) {
#pragma unroll
        for (int g = 0; g < NG; ++g)
          tma_load_2d(smem + NXS * QF_X_BYTES + slot * D_BYTES + g * QF_DG_BYTES, &map_d, &full_x[slot], g * 64,
                      kc * QF_KC);
      }
    };
    const TensorScale ts = tensor_scale(__ldg(p.amax_in));
    if (blockIdx.x == 0 && tid == 0) *p.g_dec_out = ts.g_dec;
    if (tid < 128) enc_tab[tid] = enc_of_sf8((uint32_t)tid, ts.g_dec);
    __syncthreads();

    if (warp == 16) {
      // ===== TMA producer: keeps the ring full; a slot is re-armed once the 16 quantizer warps and
      // the MMAs that read it have released it
      if (lane == 0) {
        int sx = 0;
        uint32_t phx = 0;
        for (int it = 0; it < n; ++it) {
          if (it >= NXS) mbar_wait(&empty_x[sx], phx ^ 1);
          issue_stage(it, sx);
          if (++sx == NXS) {
            sx = 0;
            phx ^= 1;
          }
        }
      }
    } else if (warp == 17) {
      // ===== tcgen05 issuer: never waits for an MMA to complete, the MMAs of successive chunks pipeline
      if constexpr (R_T > 0) {
        if (lane == 0) {
          int sx = 0, kc = o_kc, seg = 0;
          uint32_t phx = 0;
          bool first = true;
          for (int it = 0; it < n; ++it) {
            const bool seg_end = (kc == C - 1) || (it == n - 1);
            mbar_wait(&full_x[sx], phx);
            if (first && seg >= 2) mbar_wait(&acc_free[seg & 1], (uint32_t)((seg >> 1) - 1) & 1);
            tc_fence_after();
            issue_mma(xs_u + sx * QF_X_BYTES, ds_u + sx * D_BYTES, tmem_base_s + (seg & 1) * ACC_COLS, first);
            tc_commit(&empty_x[sx]);                      // slot free once the MMAs have read it
            first = false;
            if (seg_end) {
              tc_commit(&acc_full[seg & 1]);              // this segment's accumulator is complete
              ++seg;
              first = true;
            }
            if (++kc == C) kc = 0;
            if (++sx == NXS) {
              sx = 0;
              phx ^= 1;
            }
          }
        }
      }
    } else {
      // ===== quantizer warps
      int seg = 0;
      int sx = 0;            // ring slot of chunk `it`
      uint32_t phx = 0;      // and its barrier parity
      for (int it = 0; it < n; ++it) {
        mbar_wait_u32(full_u + sx * 8, phx);
        quantize_chunk(xs_u + sx * QF_X_BYTES, ts.g_enc, empty_u + sx * 8);
        if constexpr (R_T > 0) {
          if ((o_kc == C - 1) || (it == n - 1)) {   // end of a row-tile segment
            drain_segment(o_t, seg);
            ++seg;
          }
        }
        advance_out();
        if (++sx == NXS) {
          sx = 0;
          phx ^= 1;
        }
      }
      // the partial H tiles are in their slots; k_finalize_h (next launch) sums them.  A grid barrier
      // here would need a cooperative launch, and the runtime admits only ONE CTA per SM of a kernel
      // that allocates tensor memory (it cannot see that two 128-column allocations fit).
    }
  } else {
    // =========================================================== single-pass mode
    const int nd = p.nd;
    const int n0 = min(n, C - o_kc);                         // chunks in the first row tile
    if (warp == 16) {
      // ===== TMA producer: the whole range stays resident; the D slices go through a small ring
      if (lane == 0) {
        for (int it = 0; it < n; ++it) issue_x(it, it);
        if constexpr (R_T > 0) {
          int sd = 0;
          uint32_t phd = 0;
          for (int it = 0; it < n; ++it) {
            if (it >= nd) mbar_wait(&empty_d[sd], phd ^ 1);
            issue_d(it, sd);
            if (++sd == nd) {
              sd = 0;
              phd ^= 1;
            }
          }
        }
      }
    } else if (warp == 17) {
      // ===== tcgen05 issuer: the projection MMAs as the chunks land (row-tile segment 0 / 1)
      if constexpr (R_T > 0) {
        if (lane == 0) {
          int sd = 0;
          uint32_t phd = 0;
          for (int it = 0; it < n; ++it) {
            const int sg = it < n0 ? 0 : 1;
            mbar_wait(&full_x[it], 0);
            mbar_wait(&full_d[sd], phd);
            tc_fence_after();
            issue_mma(xs_u + it * QF_X_BYTES, ds_u + sd * D_BYTES, tmem_base_s + sg * ACC_COLS,
                      it == 0 || it == n0);
            tc_commit(&empty_d[sd]);
            if (it == n0 - 1 || it == n - 1) tc_commit(&acc_full[sg]);
            if (++sd == nd) {
              sd = 0;
              phd ^= 1;
            }
          }
        }
      }
    } else {
    // ===== quantizer warps
    // ---- phase 1: tensor amax as the chunks land
    uint32_t m2 = 0;
    for (int it = 0; it < n; ++it) {
      mbar_wait(&full_x[it], 0);
      uint4 v0, v1;
      load_block(xs_u + it * QF_X_BYTES, v0, v1);
      m2 = absmax2_bf16(m2, absmax2_bf16(absmax2_bf16(absmax2_bf16(v0.x, v0.y), absmax2_bf16(v0.z, v0.w)),
                                         absmax2_bf16(absmax2_bf16(v1.x, v1.y), absmax2_bf16(v1.z, v1.w))));
    }
    m2 &= 0x7FFF7FFFu;
    uint32_t best = max(m2 & 0xFFFFu, m2 >> 16);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if (lane == 0) s_red[warp] = best;
    qsync();
    if (tid == 0) {
      for (int w = 1; w < QF_QTHREADS / 32; ++w) best = max(best, s_red[w]);
      atomicMax(p.amax_bits, best << 16);   // bf16 bits -> float bits; non-negative floats order as uints
      __threadfence();
      atomicAdd(p.grid_bar, 1u);
    }
    // ---- partial H tiles out while the other CTAs arrive
    if constexpr (R_T > 0) {
      drain_segment(o_t, 0);
      if (n > n0) drain_segment(o_t + 1, 1);
      // split-phase second barrier: ARRIVE now (this CTA's slots are written), wait only after phase 2 --
      // by then every CTA has long arrived and the wait costs one poll instead of a barrier round trip
      if (warp < 4) {
        asm volatile("bar.sync 2, 128;" ::: "memory");   // the four draining warps
        if (tid == 0) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p.grid_bar + 1) : "memory");
      }
    }
    // ---- grid-wide barrier: every CTA has published its amax
    if (tid == 0) {
      const uint64_t t0 = globaltimer_ns();
      while (ld_acquire_u32(p.grid_bar) < gridDim.x) {
        if (globaltimer_ns() - t0 > 2000000000ull) __trap();   // co-residency broken: fail, do not hang
      }
      s_amax = ld_acquire_u32(p.amax_bits);
    }
    qsync();
    const TensorScale ts = tensor_scale(__uint_as_float(s_amax));
    float inv_alpha = 1.0f;
    if (R_T > 0 && p.hs_out != nullptr) inv_alpha = __fdiv_rn(1.0f, __fmul_rn(ts.g_dec, __ldg(p.other_dec_scale)));
    if (blockIdx.x == 0 && tid == 0) *p.g_dec_out = ts.g_dec;
    if (tid < 128) enc_tab[tid] = enc_of_sf8((uint32_t)tid, ts.g_dec);
    qsync();
    // ---- phase 2: quantize from shared memory
    for (int it = 0; it < n; ++it) {
      quantize_chunk(xs_u + it * QF_X_BYTES, ts.g_enc, 0);
      advance_out();
    }
    if constexpr (R_T > 0) {
      if (tid == 0) {   // every CTA's slots are written (they arrived before their phase 2)
        const uint64_t t0 = globaltimer_ns();
        while (ld_acquire_u32(p.grid_bar + 1) < gridDim.x) {
          if (globaltimer_ns() - t0 > 2000000000ull) __trap();
        }
      }
      qsync();
      finalize_share(inv_alpha);
    }
    }
  }

  if constexpr (R_T > 0) {
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
      tc_fence_after();
      tmem_dealloc(tmem_base_s, 2 * ACC_COLS);
    }
  }
}

// Streaming mode's second step: H[row] = sum of the row tile's slots, in CTA order, -> bf16 H and
// Hs = H * (1 / alpha).  One thread per (row, column quad); neighbouring threads read neighbouring rows
// of a slot (layout [quad][row][4]).  G = grid size of the quantize launch that filled the slots.
template <int R_T>
__global__ void __launch_bounds__(256) k_finalize_h(const QFParams p, int G) {
  constexpr int QUADS = R_T / 4;
  constexpr int SLOT_F4 = QF_ROWS * R_T / 4;
  pdl_wait();      // the slots and g_dec come from the quantize kernel before us
  pdl_trigger();
  float inv_alpha = 1.0f;   // Hs = bf16(H * (1 / alpha)), alpha = g_dec(this) * g_dec(other)
  if (p.hs_out != nullptr) inv_alpha = __fdiv_rn(1.0f, __fmul_rn(__ldcg(p.g_dec_out), __ldg(p.other_dec_scale)));
  const int C = p.chunks_per_tile;
  const int64_t TC = p.total_chunks;
  // thread -> (tile t, quad q, row r) with r fastest
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  const int r = (int)(e % QF_ROWS);
  const int q = (int)((e / QF_ROWS) % QUADS);
  const int64_t t = e / (QF_ROWS * QUADS);
  const int64_t gr = t * QF_ROWS + r;
  if (gr >= p.rows) return;
  // the CTAs whose ranges meet row tile t: owner(c) = floor(((c + 1) * G - 1) / TC)
  const int i_lo = (int)(((t * C + 1) * G - 1) / TC);
  const int i_hi = (int)((((t + 1) * C) * G - 1) / TC);
  const float4* src = reinterpret_cast<const float4*>(p.slots) + (i_lo + t) * SLOT_F4 + q * QF_ROWS + r;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  constexpr int BATCH = 12;   // loads in flight; a row tile rarely has more contributors than that
  for (int i = i_lo; i <= i_hi; i += BATCH) {   // added in CTA order whatever the batching
    float4 v[BATCH];
#pragma unroll
    for (int j = 0; j < BATCH; ++j)
      v[j] = (i + j <= i_hi) ? __ldcg(src + (int64_t)j * SLOT_F4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int j = 0; j < BATCH; ++j) {
      acc.x += v[j].x;
      acc.y += v[j].y;
      acc.z += v[j].z;
      acc.w += v[j].w;
    }
    src += BATCH * (int64_t)SLOT_F4;
  }
  if (p.h_out != nullptr)
    *reinterpret_cast<uint2*>(p.h_out + gr * R_T + q * 4) = make_uint2(pack_bf16x2(acc.x, acc.y), pack_bf16x2(acc.z, acc.w));
  if (p.hs_out != nullptr)
    *reinterpret_cast<uint2*>(p.hs_out + gr * R_T + q * 4) =
        make_uint2(pack_bf16x2(__fmul_rn(acc.x, inv_alpha), __fmul_rn(acc.y, inv_alpha)),
                   pack_bf16x2(__fmul_rn(acc.z, inv_alpha), __fmul_rn(acc.w, inv_alpha)));
}

int launch_amax(const void* x_bf16, int64_t n, float* amax_out, cudaStream_t st, bool zero_first);
int launch_clear2(void* a, size_t a_bytes, void* b, size_t b_bytes, cudaStream_t st);

// true if launch_quantize_fused would take the single-pass route (amax inside the kernel) for this tensor
bool quantize_single_pass_fits(int64_t rows, int64_t cols, int r_t);

static int g_qf_mode = 0;   // 0 auto, 1 never single pass, 2 (= auto; single pass whenever it fits)
void set_quantize_mode(int mode) { g_qf_mode = mode; }

template <int R_T>
static int launch_qf(const CUtensorMap& mx, const CUtensorMap& md, QFParams p, const void* x, const float* amax_t,
                     bool after_kernel, bool* finalize_last, cudaStream_t st) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr int D_BYTES = NG * QF_DG_BYTES;
  constexpr int SMEM_MAX = 227 * 1024 - 2048;   // minus the static shared memory (barriers, table)
  const int nsm = sm_count();
  const int64_t TC = p.total_chunks;
  const int C = p.chunks_per_tile;
  static bool attr_set = false;
  if (!attr_set) {
    FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
    FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
    FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T, false>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                     cudaSharedmemCarveoutMaxShared));
    attr_set = true;
  }
  // ---- single pass: the tensor amax is not known and every CTA can keep its whole range resident
  if (amax_t == nullptr && g_qf_mode != 1) {
    const int64_t G = TC < nsm ? TC : (nsm < QF_MAX_GRID ? nsm : QF_MAX_GRID);
    const int64_t n_max = ceil_div(TC, G);
    const int nd = R_T == 0 ? 0 : (NG == 2 ? 2 : 3);
    int smem = (int)n_max * QF_X_BYTES + nd * D_BYTES + 1024;
    if (smem < 512 * R_T + 1024) smem = 512 * R_T + 1024;   // the finalizer stages two bf16 tiles in the ring
    if (n_max <= QF_MAX_NX && smem <= SMEM_MAX && (R_T == 0 || n_max <= C)) {
      p.single = 1;
      p.nx = (int)n_max;
      p.nd = nd > 0 ? nd : 1;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)G, 1, 1);
      cfg.blockDim = dim3(QF_THREADS, 1, 1);
      cfg.dynamicSmemBytes = smem;
      cfg.stream = st;
      cudaLaunchAttribute attr[2];
      attr[0].id = cudaLaunchAttributeCooperative;   // the grid barrier needs every CTA resident
      attr[0].val.cooperative = 1;
      attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[1].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = attr;
      static bool coop_pdl_ok = true;   // cooperative + programmatic edge: tried once, dropped if refused
      cfg.numAttrs = (after_kernel && pdl_enabled() && coop_pdl_ok) ? 2 : 1;
      cudaError_t e = cudaLaunchKernelEx(&cfg, k_quantize_fused<R_T, true>, mx, md, p);
      if (e != cudaSuccess && cfg.numAttrs == 2) {
        (void)cudaGetLastError();
        coop_pdl_ok = false;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, k_quantize_fused<R_T, true>, mx, md, p);
      }
      if (e == cudaSuccess) return FT_OK;
      if (e != cudaErrorCooperativeLaunchTooLarge && e != cudaErrorNotSupported) {
        g_last_cuda_error = (int)e;
        return FT_ERR_CUDA;
      }
      (void)cudaGetLastError();   // cannot be co-resident here: two passes instead
    }
  }
  // ---- streaming: amax first (unless the caller supplied it), then a 2-CTA/SM ring kernel
  if (amax_t == nullptr) {
    int rc = launch_amax(x, p.rows * p.cols, reinterpret_cast<float*>(p.amax_bits), st, /*zero_first=*/false);
    if (rc != FT_OK) return rc;
    amax_t = reinterpret_cast<const float*>(p.amax_bits);
  }
  p.single = 0;
  p.amax_in = amax_t;
  p.nx = NG == 2 ? 3 : 4;   // = NXS of the kernel
  p.nd = p.nx;
  const int smem = p.nx * QF_X_BYTES + (R_T == 0 ? 0 : p.nd * D_BYTES) + 1024;
  int64_t cap = (int64_t)nsm * 2;   // two CTAs per SM (48 registers, <= 97 KB, 128 TMEM columns each)
  if (cap > QF_MAX_GRID) cap = QF_MAX_GRID;
  const int grid = (int)(TC < cap ? TC : cap);
  {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid, 1, 1);
    cfg.blockDim = dim3(QF_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (after_kernel && pdl_enabled()) ? 1 : 0;   // directly behind the dB^T kernel: no memset between
    FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_quantize_fused<R_T, false>, mx, md, p));
  }
  if constexpr (R_T > 0) {
    // partial H tiles -> H, Hs; programmatic edge: it sets itself up while the quantize kernel drains
    const int64_t items = ceil_div(p.rows, QF_ROWS) * QF_ROWS * (R_T / 4);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ceil_div(items, 256), 1, 1);
    cfg.blockDim = dim3(256, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_finalize_h<(R_T > 0 ? R_T : 16)>, p, grid));
    if (finalize_last != nullptr) *finalize_last = true;   // the caller's GEMM may start beside it (gemm_pair.cu)
  }
  return FT_OK;
}

bool quantize_single_pass_fits(int64_t rows, int64_t cols, int r_t) {
  if (g_qf_mode == 1) return false;
  const int nsm = sm_count();
  const int64_t C = cols / QF_KC, TC = ceil_div(rows, QF_ROWS) * C;
  const int64_t G = TC < nsm ? TC : (nsm < QF_MAX_GRID ? nsm : QF_MAX_GRID);
  const int64_t n_max = ceil_div(TC, G);
  const int NG = (r_t + 63) / 64;
  const int nd = r_t == 0 ? 0 : (NG == 2 ? 2 : 3);
  const int64_t smem = n_max * QF_X_BYTES + (int64_t)nd * NG * QF_DG_BYTES + 1024;
  return n_max <= QF_MAX_NX && smem <= 227 * 1024 - 2048 && (r_t == 0 || n_max <= C);
}

// Workspace use (offsets from ws_layout, common.cuh): the zero region holds the amax word and the two
// grid-barrier counters; it is cleared here with one 256-byte memset node.  The partial-H slots behind
// it need no clearing.
int launch_quantize_fused(const void* x, int64_t rows, int64_t cols, const float* amax_t, const ft_proj* proj,
                          ft_qtensor* out, void* workspace, bool zero_region_cleared, bool* finalize_last,
                          cudaStream_t st) {
  const int r_t = proj ? proj->r_t : 0;
  if (finalize_last != nullptr) *finalize_last = false;
  CUtensorMap mx, md;
  int rc = make_tensor_map_2d(&mx, x, 2, (uint64_t)cols, (uint64_t)rows, (uint64_t)cols * 2, QF_KC, QF_ROWS,
                              Swizzle::B128);
  if (rc != FT_OK) return rc;
  if (r_t > 0) {
    rc = make_tensor_map_2d(&md, proj->down, 2, (uint64_t)r_t, (uint64_t)cols, (uint64_t)r_t * 2, 64, QF_KC,
                            Swizzle::B128);
    if (rc != FT_OK) return rc;
  } else {
    md = mx;
  }
  if (rows * (cols / 2) >= ((int64_t)1 << 32)) return FT_ERR_UNSUPPORTED_SHAPE;   // 32-bit output cursors
  const WsLayout w = ws_layout(rows, r_t);
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  QFParams p = {};
  p.rows = rows;
  p.cols = cols;
  p.amax_in = amax_t;
  p.amax_bits = reinterpret_cast<uint32_t*>(ws + w.amax_off);
  p.grid_bar = reinterpret_cast<uint32_t*>(ws + w.bar_off);
  p.slots = reinterpret_cast<float*>(ws + w.slots_off);
  p.codes = out->codes;
  p.sf = out->sf;
  p.g_dec_out = out->tensor_dec_scale;
  p.sf_layout = out->sf_layout;
  p.h_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out) : nullptr;
  p.hs_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out_scaled) : nullptr;
  p.other_dec_scale = proj ? proj->other_dec_scale : nullptr;
  p.chunks_per_tile = (int)(cols / QF_KC);
  p.total_chunks = ceil_div(rows, QF_ROWS) * (cols / QF_KC);
  bool after_kernel = zero_region_cleared;   // a kernel of ours directly precedes the quantize launch
  if (!zero_region_cleared && (amax_t == nullptr || r_t > 0)) {
    // the control words are cleared by a small kernel with programmatic edges, not a memset node
    rc = launch_clear2(ws + w.zero_off, w.zero_bytes, nullptr, 0, st);
    if (rc != FT_OK) return rc;
    after_kernel = true;
  }
  // padding rows of the last 128-row scale tile must read as zero
  if (out->sf_layout == FT_SF_TILE128x4 && rows % 128 != 0) {
    const int64_t tiles_c = ceil_div(cols / 16, 4);
    FT_CUDA_TRY(cudaMemsetAsync(out->sf + (rows / 128) * tiles_c * 512, 0, tiles_c * 512, st));
  }
  // a memset of ours in front of the kernel (below) breaks the programmatic chain
  if (out->sf_layout == FT_SF_TILE128x4 && rows % 128 != 0) after_kernel = false;
  switch (r_t) {
    case 0: return launch_qf<0>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 16: return launch_qf<16>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 32: return launch_qf<32>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 48: return launch_qf<48>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 64: return launch_qf<64>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 80: return launch_qf<80>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 96: return launch_qf<96>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 112: return launch_qf<112>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    case 128: return launch_qf<128>(mx, md, p, x, amax_t, after_kernel, finalize_last, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft
