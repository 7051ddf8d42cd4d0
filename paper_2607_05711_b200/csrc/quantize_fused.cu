// quantize_fused.cu -- a1 / a3 (and a0 folded in): one kernel that emits the NVFP4 codes, the
// block scales and the low-rank down-projection H = X * D of a bf16 matrix (PAPER.md:110,
// "fuse ... quantization and down-projection").
//
// Decomposition.  The matrix is cut into 128-row x 64-column chunks (16 KB), numbered row tile
// major.  CTA i of a persistent grid (one CTA per SM) owns the contiguous chunk range
// [i*TC/G, (i+1)*TC/G): every CTA has the same number of chunks (+-1) whatever the shape -- no
// row-tile x split quantisation -- and a range touches at most two row tiles when it is no longer than
// a row of chunks.  From one TMA-staged chunk (SWIZZLE_128B)
//   - 256 threads quantize: thread (row = tid/2, half = tid%2) owns TWO adjacent 1x16 blocks (32
//     contiguous elements: four 16-byte shared loads, one 16-byte store of codes, the row's four
//     scale bytes gathered by one shuffle);
//   - one thread issues tcgen05.mma kind::f16 (M = 128, N = r_t, K = 16, four per chunk):
//     A = the staged chunk itself (K-major), B = the 64 x r_t slice of D (MN-major), accumulator in
//     tensor memory.
// Warp roles (22 warps): 0-15 quantize, in two groups of eight that take alternate chunks; 16 TMA
// producer; 17 tcgen05 issuer (a quantizer warp that also issues the MMAs is ~400 cycles slower per chunk
// than its peers and sets the pace of the ring); 18-21 drain: at the end of a row-tile segment they move
// the fp32 partial H tile TMEM -> plain vector stores into the segment's own 128 x r_t slot of the
// workspace (slot = CTA index + row tile: unique, and the slots of one row tile are consecutive).  The
// quantizer warps never wait for a drain (round 1 and the first build of round 2 drained with quantizer
// warps: the ring stalls for the 1-2 us of every drain; with a projection the main loop now ends when the
// projection-less one does).  k_finalize_h, launched behind the kernel with a programmatic edge, sums every
// row over its slots in CTA order and writes bf16 H and Hs = H * (1 / alpha): no atomics on the data, a
// fixed summation order (the same bits on every run), thousands of threads with one L2 round trip each.  Its
// blocks run beside this kernel: a CTA counts itself in for a row tile (control word, release) once its slot is
// stored and the tensor scale written, a finalize block starts when its tile's count is complete, and the
// GEMM that follows runs its 4-bit stages beside whatever is left of it (gemm_pair.cu, lr_late).  Measured in round 2 and
// dropped (profiles/r02_experiments.md, B2): the sums inside this kernel -- by the CTA whose arrival completes
// a row tile (36 finalizers, each a chain of L2 round trips: 6-11 us of tail at C2), or by every CTA behind a
// grid barrier (imbalance + drain + fence + poll + sum: 6-8 us of tail that nothing can overlap); fp32
// reductions into one accumulator (REDG issues at ~1.3 cycles per lane and word).
//
// Two modes, one kernel template:
//   streaming (amax known): chunks stream through a ring as deep as shared memory allows (9 stages of
//     24 KB with a projection of rank <= 64).
//   single pass (amax not known, tensor <= 12 chunks per SM = 29 MB on 148 SMs): every chunk stays resident
//     in shared memory; phase 1 finds the tensor amax (and runs the projection MMAs) as the chunks land, a
//     first grid barrier publishes it, phase 2 quantizes from shared memory.  The tensor is read from HBM
//     exactly once and the separate amax kernel (a0) disappears.  Launched cooperatively (co-residency is
//     the runtime's promise); the barrier spin traps after 2 s instead of hanging.
//
// Control words (common.cuh: WsLayout): the amax words, the barrier counter and the exit counter are zero
// between calls; the last CTA to leave puts them back, so no clear kernel runs per call.
#include <cstdio>
#include <cstdlib>

#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

constexpr int QF_ROWS = 128;    // rows per chunk
constexpr int QF_KC = 64;       // columns per chunk (128 bytes of bf16 = one swizzle row)
constexpr int QF_X_BYTES = QF_ROWS * QF_KC * 2;  // 16 KB
constexpr int QF_DG_BYTES = QF_KC * 128;         // one 64-column group of D: 8 KB
constexpr int QF_MAX_NX = 12;   // ring slots / resident chunks per CTA
constexpr int QF_MAX_ND = 4;    // single pass: ring of D slices
constexpr int QF_MAX_GRID = WS_MAX_QUANT_CTAS;   // the workspace has one slot per CTA + one per row tile
constexpr int QF_QWARPS = 16;                    // quantizer warps: two groups of eight
constexpr int QF_QTHREADS = QF_QWARPS * 32;
constexpr int QF_W_PRODUCER = 16, QF_W_ISSUER = 17, QF_W_DRAIN = 18;
constexpr int QF_THREADS = (QF_W_DRAIN + 4) * 32;   // 704

struct QFParams {
  int64_t rows, cols;
  const float* amax_in;         // streaming: tensor amax (device)
  uint32_t* ctl;                // control words of the workspace (WS_CTL_*), or null (amax given, no projection)
  uint32_t* tile_cnt;           // per-row-tile arrival counters (WS_CTL_TILE_CNT), or null: k_finalize_h waits for the grid
  uint32_t* tile_done;          // per-row-tile count of finished finalize blocks
  float* slots;                 // [(grid + row tiles) x 128 x r_t] fp32 partial H tiles (not zeroed)
  uint8_t* codes;
  uint8_t* sf;
  float* g_dec_out;
  int sf_layout;
  __nv_bfloat16* h_out;         // [rows x r_t] or null
  __nv_bfloat16* hs_out;        // [rows x r_t] or null
  const float* other_dec_scale; // for hs_out
  int nx, nd;                   // ring depths (single pass: nx = max chunks per CTA)
  int chunks_per_tile;          // C = cols / 64
  int64_t total_chunks;         // TC = row tiles * C
#ifdef FT_TRACE
  unsigned long long* trace;    // development builds only: 8 globaltimer stamps per CTA
  int dbg;                      // 1 = no D-slice loads, 2 = no MMAs, 4 = no slot stores (timing only)
#endif
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
#ifdef FT_TRACE
unsigned long long* g_qf_trace = nullptr;
#define QF_STAMP(i) do { if (p.trace != nullptr && threadIdx.x == 0) p.trace[blockIdx.x * 8 + (i)] = globaltimer_ns(); } while (0)
#else
#define QF_STAMP(i) do { } while (0)
#endif

// R_T: width of the projection (0 = quantize only).  NG = 64-column groups of D.
template <int R_T, bool SINGLE>
__global__ void __launch_bounds__(QF_THREADS, 1)
k_quantize_fused(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_d,
                 const QFParams p) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr uint32_t ACC_COLS = R_T <= 32 ? 32 : (R_T <= 64 ? 64 : 128);
  constexpr int D_BYTES = NG * QF_DG_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment for the 128-byte swizzle atoms
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t full_x[QF_MAX_NX], empty_x[QF_MAX_NX], full_d[QF_MAX_ND], empty_d[QF_MAX_ND];
  __shared__ uint64_t acc_full[2], acc_free[2], gdec_bar;
  __shared__ float enc_tab[128];
  __shared__ uint32_t tmem_base_s, s_red[QF_QWARPS], s_amax;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t c_begin = (int64_t)blockIdx.x * p.total_chunks / gridDim.x;
  const int n = (int)(((int64_t)blockIdx.x + 1) * p.total_chunks / gridDim.x - c_begin);   // >= 1 (grid <= TC)
  const int C = p.chunks_per_tile;
  const int NX = p.nx;
  const uint32_t xs_u = smem_u32(smem);
  const uint32_t ds_u = xs_u + (uint32_t)NX * QF_X_BYTES;
  uint32_t* const bar_amax = p.ctl + WS_CTL_BAR / 4;

  if (tid == 0) {
    prefetch_tmap(&map_x);
    if (R_T > 0) prefetch_tmap(&map_d);
    for (int s = 0; s < QF_MAX_NX; ++s) {
      mbar_init(&full_x[s], 1);
      mbar_init(&empty_x[s], QF_QWARPS / 2 + (R_T > 0 ? 1 : 0));  // the eight warps of one group (+ the MMA commit)
    }
    for (int s = 0; s < QF_MAX_ND; ++s) {
      mbar_init(&full_d[s], 1);
      mbar_init(&empty_d[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&acc_full[a], 1);   // tcgen05.commit of a segment's last MMA
      mbar_init(&acc_free[a], 4);   // the four drain warps
    }
    mbar_init(&gdec_bar, 1);        // this CTA has written the tensor scale (the drain warps publish their slots after it)
    fence_mbar_init();
  }
  if (R_T > 0 && warp == QF_W_ISSUER) {
    tmem_alloc(&tmem_base_s, 2 * ACC_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  QF_STAMP(0);
  pdl_wait();      // streaming mode inside ft_linear_bwd: the amax comes from the dB^T kernel before us
  pdl_trigger();   // the kernel that follows may set itself up while this one runs (it waits for our end)
  QF_STAMP(1);

  // the four MMAs of one chunk: acc[128 x r_t] (+)= X[128, 64 k] * D[64 k, r_t]
  auto issue_mma = [&](uint32_t x_u, uint32_t d_u, uint32_t acc, bool first) {
    constexpr uint32_t idesc = idesc_bf16(QF_ROWS, R_T > 0 ? R_T : 16) | (1u << 16);  // B is MN-major
#pragma unroll
    for (int k = 0; k < 4; ++k)
      mma_bf16(acc, make_smem_desc(x_u + k * 32, 1024, 0, 2), make_smem_desc(d_u + k * 2048, 1024, QF_DG_BYTES, 2),
               idesc, !(first && k == 0));
  };

  // ---- geometry of this CTA's range: segment s = its run of chunks inside row tile t0 + s
  const int t0 = (int)(c_begin / C), kc0 = (int)(c_begin % C);
  const int n0 = min(n, C - kc0);                           // chunks in the first row tile
  const int nseg = 1 + (n - n0 + C - 1) / C;

  auto spin_until = [&](const uint32_t* word, uint32_t target) {
    const uint64_t t_start = globaltimer_ns();
    while (ld_acquire_u32(word) < target) {
      if (globaltimer_ns() - t_start > 2000000000ull) __trap();   // co-residency broken: fail, do not hang
    }
  };

  if (warp == QF_W_PRODUCER) {
    // =========================================================== TMA producer
    if (lane == 0) {
      if constexpr (!SINGLE) {
        // a stage = the X chunk and its D slice, both on full_x[slot].  Streaming mode reads its tensor for the
        // last time: evict-first, so that what the pass before left in L2 (the dB^T pass over the same G) is not
        // displaced by lines nobody reads again
        const uint64_t pol_stream = l2_policy_evict_first();
        int kc = kc0, t = t0, sx = 0;
        uint32_t phx = 0;
        for (int it = 0; it < n; ++it) {
          if (it >= NX) mbar_wait(&empty_x[sx], phx ^ 1);
#ifdef FT_TRACE
          if (p.dbg & 1) {
            mbar_expect_tx(&full_x[sx], QF_X_BYTES);
            tma_load_2d_hint(smem + sx * QF_X_BYTES, &map_x, &full_x[sx], kc * QF_KC, t * QF_ROWS, pol_stream);
          } else
#endif
          {
          mbar_expect_tx(&full_x[sx], QF_X_BYTES + (R_T > 0 ? D_BYTES : 0));
          tma_load_2d_hint(smem + sx * QF_X_BYTES, &map_x, &full_x[sx], kc * QF_KC, t * QF_ROWS, pol_stream);
          }
#ifdef FT_TRACE
          if (!(p.dbg & 1))
#endif
          if constexpr (R_T > 0) {
#pragma unroll
            for (int g = 0; g < NG; ++g)
              tma_load_2d(smem + NX * QF_X_BYTES + sx * D_BYTES + g * QF_DG_BYTES, &map_d, &full_x[sx], g * 64,
                          kc * QF_KC);
          }
          if (++kc == C) {
            kc = 0;
            ++t;
          }
          if (++sx == NX) {
            sx = 0;
            phx ^= 1;
          }
        }
      } else {
        // the whole range stays resident; the D slices go through a small ring
        int kc = kc0, t = t0;
        for (int it = 0; it < n; ++it) {
          mbar_expect_tx(&full_x[it], QF_X_BYTES);
          tma_load_2d(smem + it * QF_X_BYTES, &map_x, &full_x[it], kc * QF_KC, t * QF_ROWS);
          if (++kc == C) {
            kc = 0;
            ++t;
          }
        }
        if constexpr (R_T > 0) {
          const int nd = p.nd;
          int sd = 0, kd = kc0;
          uint32_t phd = 0;
          for (int it = 0; it < n; ++it) {
            if (it >= nd) mbar_wait(&empty_d[sd], phd ^ 1);
            mbar_expect_tx(&full_d[sd], D_BYTES);
#pragma unroll
            for (int g = 0; g < NG; ++g)
              tma_load_2d(smem + NX * QF_X_BYTES + sd * D_BYTES + g * QF_DG_BYTES, &map_d, &full_d[sd], g * 64,
                          kd * QF_KC);
            if (++kd == C) kd = 0;
            if (++sd == nd) {
              sd = 0;
              phd ^= 1;
            }
          }
        }
      }
    }
  } else if (warp == QF_W_ISSUER) {
    // =========================================================== tcgen05 issuer: never waits for an MMA to
    // complete, the MMAs of successive chunks pipeline
    if constexpr (R_T > 0) {
      if (lane == 0) {
        int sx = 0, sd = 0, kc = kc0, seg = 0;
        uint32_t phx = 0, phd = 0;
        bool first = true;
        for (int it = 0; it < n; ++it) {
          const bool seg_end = (kc == C - 1) || (it == n - 1);
          if constexpr (!SINGLE) {
            mbar_wait(&full_x[sx], phx);
          } else {
            mbar_wait(&full_x[it], 0);
            mbar_wait(&full_d[sd], phd);
          }
          if (first && seg >= 2) mbar_wait(&acc_free[seg & 1], (uint32_t)((seg >> 1) - 1) & 1);
          tc_fence_after();
          if constexpr (!SINGLE) {
#ifdef FT_TRACE
            if (!(p.dbg & 2))
#endif
            issue_mma(xs_u + sx * QF_X_BYTES, ds_u + sx * D_BYTES, tmem_base_s + (seg & 1) * ACC_COLS, first);
            tc_commit(&empty_x[sx]);                      // slot free once the MMAs have read it
          } else {
            issue_mma(xs_u + it * QF_X_BYTES, ds_u + sd * D_BYTES, tmem_base_s + (seg & 1) * ACC_COLS, first);
            tc_commit(&empty_d[sd]);
          }
          first = false;
          if (seg_end) {
            tc_commit(&acc_full[seg & 1]);                // this segment's accumulator is complete
            ++seg;
            first = true;
          }
          if (++kc == C) kc = 0;
          if (++sx == NX) {
            sx = 0;
            phx ^= 1;
          }
          if (++sd == p.nd) {
            sd = 0;
            phd ^= 1;
          }
        }
      }
    }
  } else if (warp >= QF_W_DRAIN) {
    // =========================================================== drain warps: TMEM -> the segment's slot.
    // Warp w may read TMEM lanes 32 (w % 4) .. + 31 = rows of the tile.
    if constexpr (R_T > 0) {
      const int dq = warp & 3;
      // the slot of segment seg is complete in memory and the tensor scale written: count this CTA in for row tile
      // t0 + seg (release; k_finalize_h acquires the count)
      auto publish = [&](int seg) {
        asm volatile("bar.sync 2, 128;" ::: "memory");   // the four drain warps have stored their parts
        if (warp == QF_W_DRAIN && lane == 0) {
          mbar_wait(&gdec_bar, 0);
          __threadfence();
          asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p.tile_cnt + t0 + seg) : "memory");
        }
      };
      for (int seg = 0; seg < nseg; ++seg) {
        const int a = seg & 1;
        mbar_wait(&acc_full[a], (uint32_t)(seg >> 1) & 1);
        tc_fence_after();
        // slot layout [column quad q = c / 4][row][4 floats]: a warp's store instruction covers 512
        // contiguous bytes (full sectors), and so does a warp's load in the finalizer
        float* dst = p.slots + ((int64_t)blockIdx.x + t0 + seg) * (QF_ROWS * R_T) + (dq * 32 + lane) * 4;
#pragma unroll 1
        for (int c0 = 0; c0 < R_T; c0 += 16) {
          uint32_t v[16];
          tmem_ld16(tmem_base_s + ((uint32_t)(dq * 32) << 16) + a * ACC_COLS + c0, v);
          tmem_ld_wait();
#ifdef FT_TRACE
          if (!(p.dbg & 4))
#endif
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4*>(dst + (c0 + j) / 4 * (QF_ROWS * 4)) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&acc_free[a]);   // the accumulator may be overwritten
        if (!SINGLE && p.tile_cnt != nullptr) publish(seg);
      }
      // the partial H tiles are in their slots; k_finalize_h (next launch) sums a row tile as soon as all its slots
      // are published.  Single pass: the tensor scale is known only behind the grid barrier, the segments (at most
      // three) are published then.
      if (SINGLE && p.tile_cnt != nullptr)
        for (int seg = 0; seg < nseg; ++seg) publish(seg);
    }
  } else {
    // =========================================================== quantizer warps: two groups of eight, group g
    // takes the chunks it = g, g + 2, ...  Thread role: two adjacent 1x16 blocks (four 16-byte pieces of a
    // swizzled row) per chunk.  A warp's load instruction covers 16 rows x 2 halves; every quarter-warp touches
    // eight distinct 16-byte columns of the 128-byte swizzle row: conflict-free.
    const int grp = warp >> 3;
    const int qt = tid & 255;
    const int q_row = qt >> 1, q_half = qt & 1;
    const uint32_t q_base = q_row * 128;
    const uint32_t q_x = q_row & 7;
    const bool sf_tiled = p.sf_layout == FT_SF_TILE128x4;
    // output cursor (32-bit byte offsets; the host rejects tensors whose codes exceed 4 GB): advanced
    // one chunk at a time, no per-chunk index arithmetic
    int o_t = t0, o_kc = kc0;
    uint32_t o_co, o_so;
    bool o_live;
    {
      const uint32_t nblk = (uint32_t)(p.cols / 16), half_cols = (uint32_t)(p.cols / 2);
      const uint32_t grow = (uint32_t)o_t * QF_ROWS + q_row;
      o_live = (int64_t)grow < p.rows;
      o_co = grow * half_cols + o_kc * 32 + q_half * 16;
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
    auto load_blocks = [&](uint32_t x_u, uint4 (&v)[4]) {
#pragma unroll
      for (int i = 0; i < 4; ++i)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v[i].x), "=r"(v[i].y), "=r"(v[i].z), "=r"(v[i].w)
                     : "r"(x_u + q_base + ((((uint32_t)(q_half * 4 + i)) ^ q_x) << 4)));
    };
    const uint32_t enc_u = smem_u32(enc_tab), full_u = smem_u32(full_x), empty_u = smem_u32(empty_x);
    // release_u: shared address of the slot's empty barrier, or 0 (single-pass mode: nothing to release).
    // The slot is handed back as soon as the blocks are in registers (the amax trees consume all sixteen
    // loaded words, so the loads have completed), not after the arithmetic and the stores: the ring looks
    // deeper to the producer.
    auto quantize_chunk = [&](uint32_t x_u, float g_enc, uint32_t release_u) {
      uint4 v[4];
      load_blocks(x_u, v);
      const float amax_a = amax_block16(v[0], v[1]);
      const float amax_b = amax_block16(v[2], v[3]);
      if (release_u != 0) {
        __syncwarp();
        if (lane == 0) mbar_arrive_u32(release_u);
      }
      const uint32_t sf_a = block_sf8(amax_a, g_enc), sf_b = block_sf8(amax_b, g_enc);
      float enc_a, enc_b;
      asm volatile("ld.shared.f32 %0, [%1];" : "=f"(enc_a) : "r"(enc_u + sf_a * 4));
      asm volatile("ld.shared.f32 %0, [%1];" : "=f"(enc_b) : "r"(enc_u + sf_b * 4));
      uint4 c;
      c.x = quant_bf16x8_fast(v[0], enc_a);
      c.y = quant_bf16x8_fast(v[1], enc_a);
      c.z = quant_bf16x8_fast(v[2], enc_b);
      c.w = quant_bf16x8_fast(v[3], enc_b);
      // the row's four scale bytes: this thread's two and its neighbour's (lane ^ 1) two
      uint32_t w = (sf_a | (sf_b << 8)) << (16 * q_half);
      w |= __shfl_xor_sync(0xffffffffu, w, 1);
      if (o_live) {
        *reinterpret_cast<uint4*>(p.codes + o_co) = c;
        if (q_half == 0) *reinterpret_cast<uint32_t*>(p.sf + o_so) = w;
      } else if (sf_tiled && q_half == 0) {
        *reinterpret_cast<uint32_t*>(p.sf + o_so) = 0u;   // padding rows of the last 128-row scale tile read as zero
      }
    };
    // barrier of the quantizer warps only (the other warps run free)
    auto qsync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(QF_QTHREADS) : "memory"); };

    TensorScale ts;
    if constexpr (!SINGLE) {
      // ---- streaming mode (amax known)
      ts = tensor_scale(__ldcg(p.amax_in));
      if (tid == 0) {   // every CTA writes the (same) tensor scale: whoever sees this CTA's slots published sees it too
        *p.g_dec_out = ts.g_dec;
        mbar_arrive(&gdec_bar);
      }
      if (tid < 128) enc_tab[tid] = enc_of_sf8((uint32_t)tid, ts.g_dec);
      qsync();
      if (grp == 1) advance_out();
      // chunk it lives in ring slot it % NX, parity (it / NX) & 1
      int sx = grp % NX;
      uint32_t phx = (uint32_t)(grp / NX) & 1;
      for (int it = grp; it < n; it += 2) {
        mbar_wait_u32(full_u + sx * 8, phx);
        quantize_chunk(xs_u + sx * QF_X_BYTES, ts.g_enc, empty_u + sx * 8);
        advance_out();
        advance_out();
        sx += 2;
        if (sx >= NX) {
          sx -= NX;
          phx ^= 1;
        }
      }
    } else {
      // ---- single-pass mode, phase 1: tensor amax as the chunks land
      uint32_t m2 = 0;
      for (int it = grp; it < n; it += 2) {
        mbar_wait(&full_x[it], 0);
        uint4 v[4];
        load_blocks(xs_u + it * QF_X_BYTES, v);
#pragma unroll
        for (int i = 0; i < 4; ++i)
          m2 = absmax2_bf16(m2, absmax2_bf16(absmax2_bf16(v[i].x, v[i].y), absmax2_bf16(v[i].z, v[i].w)));
      }
      m2 &= 0x7FFF7FFFu;
      uint32_t best = max(m2 & 0xFFFFu, m2 >> 16);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
      if (lane == 0) s_red[warp] = best;
      QF_STAMP(2);
      qsync();
      if (tid == 0) {
        for (int w = 1; w < QF_QWARPS; ++w) best = max(best, s_red[w]);
        atomicMax(p.ctl + WS_CTL_AMAX / 4, best << 16);   // bf16 bits -> float bits; non-negative floats order as uints
        __threadfence();
        atomicAdd(bar_amax, 1u);
        // ---- first grid barrier: every CTA has published its amax (the drain warps write the slots meanwhile)
        spin_until(bar_amax, gridDim.x);
        s_amax = ld_acquire_u32(p.ctl + WS_CTL_AMAX / 4);
      }
      QF_STAMP(3);
      qsync();
      ts = tensor_scale(__uint_as_float(s_amax));
      if (tid == 0) {
        *p.g_dec_out = ts.g_dec;
        mbar_arrive(&gdec_bar);
      }
      if (tid < 128) enc_tab[tid] = enc_of_sf8((uint32_t)tid, ts.g_dec);
      qsync();
      // ---- phase 2: quantize from shared memory
      if (grp == 1) advance_out();
      for (int it = grp; it < n; it += 2) {
        quantize_chunk(xs_u + it * QF_X_BYTES, ts.g_enc, 0);
        advance_out();
        advance_out();
      }
      QF_STAMP(4);
    }
  }
  QF_STAMP(5);

  if constexpr (R_T > 0) tc_fence_before();
  __syncthreads();
  if constexpr (R_T > 0) {
    if (warp == QF_W_ISSUER) {
      tc_fence_after();
      tmem_dealloc(tmem_base_s, 2 * ACC_COLS);
    }
  }
  QF_STAMP(6);
  // the last CTA to leave puts the shared control words back to zero (every CTA has read them by now)
  if (tid == 0 && p.ctl != nullptr) {
    __threadfence();
    if (atomicAdd(p.ctl + WS_CTL_EXIT / 4, 1u) == gridDim.x - 1) {
      p.ctl[WS_CTL_AMAX / 4] = 0u;
      p.ctl[WS_CTL_BAR / 4] = 0u;
      p.ctl[WS_CTL_AMAX_EXT / 4] = 0u;
      p.ctl[WS_CTL_EXIT / 4] = 0u;
    }
  }
}

// The second step: H[row] = sum of the row tile's slots -> bf16 H and Hs = H * (1 / alpha).  Block = one column quad of
// one 128-row tile: thread (r, part) adds the slots i_lo + part, i_lo + part + P, ... of its row (one batch of loads
// in flight: a single L2 round trip for up to 8 P contributors), the P partial sums of a row meet in shared memory
// and are added in part order: a fixed association whatever the timing (the same bits on every run).  Neighbouring
// threads read neighbouring rows of a slot (layout [quad][row][4]).  G = grid size of the quantize launch that filled
// the slots; P = blockDim.y (1 when a row tile has at most 8 contributors, as on the large shapes).
template <int R_T>
__global__ void __launch_bounds__(1024) k_finalize_h(const QFParams p, int G, const SumJob job) {
  constexpr int SLOT_F4 = QF_ROWS * R_T / 4;
  extern __shared__ float4 s_part[];   // [P][QF_ROWS], P > 1 only
  const bool flags = p.tile_cnt != nullptr;
  // flags: this kernel's blocks may run BESIDE the quantize kernel and start a row tile's sum as soon as all its
  // slots are published; they wait for that kernel as a whole only before they exit (completion stays transitive:
  // the GEMM behind us needs its codes and scales).  No flags: wait for it here.
  if (!flags) pdl_wait();
  pdl_trigger();
  if (job.n_slots > 0) {   // side job (ft_linear_bwd: the M slices of dB^T, written two kernels ago): slot order
    const int64_t nthr = (int64_t)gridDim.x * gridDim.y * blockDim.x * blockDim.y;
    const int64_t me = (((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    for (int64_t i = me; i < job.n4; i += nthr) {
      float4 a = __ldcg(job.slots + i);
      for (int sidx = 1; sidx < job.n_slots; ++sidx) {
        const float4 o = __ldcg(job.slots + (int64_t)sidx * job.n4 + i);
        a.x += o.x;
        a.y += o.y;
        a.z += o.z;
        a.w += o.w;
      }
      job.out[i] = a;
    }
  }
  const int C = p.chunks_per_tile;
  const int64_t TC = p.total_chunks;
  const int r = threadIdx.x, part = threadIdx.y, P = blockDim.y;
  const int q = blockIdx.x;
  const int64_t t = blockIdx.y;
  const int64_t gr = t * QF_ROWS + r;
  // the CTAs whose ranges meet row tile t: owner(c) = floor(((c + 1) * G - 1) / TC)
  const int i_lo = (int)(((t * C + 1) * G - 1) / TC);
  const int i_hi = (int)((((t + 1) * C) * G - 1) / TC);
  if (flags) {
    if (r == 0 && part == 0) {
      const uint32_t want = (uint32_t)(i_hi - i_lo + 1);
      const uint64_t t_start = globaltimer_ns();
      while (ld_acquire_u32(p.tile_cnt + t) < want) {
        __nanosleep(64);
        if (globaltimer_ns() - t_start > 2000000000ull) __trap();   // fail, do not hang
      }
    }
    __syncthreads();
  }
  float inv_alpha = 1.0f;   // Hs = bf16(H * (1 / alpha)), alpha = g_dec(this) * g_dec(other)
  if (p.hs_out != nullptr) inv_alpha = __fdiv_rn(1.0f, __fmul_rn(__ldcg(p.g_dec_out), __ldg(p.other_dec_scale)));
  const float4* src = reinterpret_cast<const float4*>(p.slots) + (i_lo + t) * SLOT_F4 + q * QF_ROWS + r;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  constexpr int BATCH = 8;   // loads in flight per thread
  for (int i = i_lo + part; i <= i_hi; i += BATCH * P) {   // this part's slots, in CTA order
    float4 v[BATCH];
#pragma unroll
    for (int j = 0; j < BATCH; ++j)
      v[j] = (i + j * P <= i_hi) ? __ldcg(src + (int64_t)(i - i_lo + j * P) * SLOT_F4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int j = 0; j < BATCH; ++j) {
      acc.x += v[j].x;
      acc.y += v[j].y;
      acc.z += v[j].z;
      acc.w += v[j].w;
    }
  }
  if (P > 1) {
    s_part[part * QF_ROWS + r] = acc;
    __syncthreads();
    if (part == 0)
      for (int k = 1; k < P; ++k) {
        const float4 o = s_part[k * QF_ROWS + r];
        acc.x += o.x;
        acc.y += o.y;
        acc.z += o.z;
        acc.w += o.w;
      }
  }
  if (part == 0 && gr < p.rows) {
    if (p.h_out != nullptr)
      *reinterpret_cast<uint2*>(p.h_out + gr * R_T + q * 4) = make_uint2(pack_bf16x2(acc.x, acc.y), pack_bf16x2(acc.z, acc.w));
    if (p.hs_out != nullptr)
      *reinterpret_cast<uint2*>(p.hs_out + gr * R_T + q * 4) =
          make_uint2(pack_bf16x2(__fmul_rn(acc.x, inv_alpha), __fmul_rn(acc.y, inv_alpha)),
                     pack_bf16x2(__fmul_rn(acc.z, inv_alpha), __fmul_rn(acc.w, inv_alpha)));
  }
  if (flags) {
    __syncthreads();   // every thread of the block has read its slots
    if (r == 0 && part == 0) {
      // the last block of this row tile puts its two counters back to zero for the next call
      if (atomicAdd(p.tile_done + t, 1u) == gridDim.x - 1) {
        p.tile_cnt[t] = 0u;
        p.tile_done[t] = 0u;
      }
    }
    pdl_wait();   // "this grid complete" implies "the quantize kernel complete"
  }
}

int launch_amax(const void* x_bf16, int64_t n, float* amax_out, cudaStream_t st, bool zero_first, bool pdl);

static int g_qf_mode = 0;      // 0 auto, 1 never single pass, 2 (= auto; single pass whenever it fits)
void set_quantize_mode(int mode) { g_qf_mode = mode; }

constexpr int QF_SMEM_MAX = 227 * 1024 - 2560;   // minus the static shared memory (barriers, table)

// single pass: nx resident chunks + a ring of nd D slices; returns false if the tensor does not fit
static bool single_pass_geometry(int64_t rows, int64_t cols, int r_t, int nsm, int64_t* G_out, int* nx, int* nd,
                                 int* smem) {
  const int64_t C = cols / QF_KC, TC = ceil_div(rows, QF_ROWS) * C;
  const int64_t G = TC < nsm ? TC : nsm;
  const int64_t n_max = ceil_div(TC, G);
  const int NG = (r_t + 63) / 64;
  const int d = r_t == 0 ? 0 : (NG == 2 ? 2 : 3);
  const int64_t bytes = n_max * QF_X_BYTES + (int64_t)d * NG * QF_DG_BYTES + 1024;
  if (n_max > QF_MAX_NX || bytes > QF_SMEM_MAX || (r_t > 0 && n_max > C)) return false;
  *G_out = G;
  *nx = (int)(n_max < 2 ? 2 : n_max);
  *nd = d > 0 ? d : 1;
  *smem = (int)bytes + (n_max < 2 ? QF_X_BYTES : 0);
  return true;
}

template <int R_T>
static int launch_qf(const CUtensorMap& mx, const CUtensorMap& md, QFParams p, const void* x, const float* amax_t,
                     bool after_kernel, bool* finalize_last, const SumJob& job, cudaStream_t st) {
  constexpr int NG = (R_T + 63) / 64;
  constexpr int D_BYTES = NG * QF_DG_BYTES;
  const int nsm = sm_count() < QF_MAX_GRID ? sm_count() : QF_MAX_GRID;
  const int dev = current_device();
  const bool dev_ok = dev >= 0 && dev < FT_MAX_DEVICES;
  const int64_t TC = p.total_chunks;
  static bool attr_set[FT_MAX_DEVICES] = {};
  if (dev_ok && !attr_set[dev]) {
    FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, QF_SMEM_MAX));
    FT_CUDA_TRY(cudaFuncSetAttribute(k_quantize_fused<R_T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, QF_SMEM_MAX));
    attr_set[dev] = true;
  }
  // Both modes: one CTA per SM; the single-pass kernel has a grid barrier and is launched cooperatively
  // (co-residency is then the runtime's promise).  A programmatic edge on top is tried once per device and dropped
  // if the runtime refuses the combination.
  static bool coop_pdl_refused[FT_MAX_DEVICES] = {};
  auto launch = [&](auto kernel, unsigned grid, int smem, bool barrier) -> cudaError_t {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(QF_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (barrier) {
      attr[na].id = cudaLaunchAttributeCooperative;
      attr[na].val.cooperative = 1;
      ++na;
    }
    const bool want_pdl = after_kernel && pdl_enabled() && !(barrier && dev_ok && coop_pdl_refused[dev]);
    if (want_pdl) {
      attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[na].val.programmaticStreamSerializationAllowed = 1;
      ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, mx, md, p);
    if (e != cudaSuccess && barrier && want_pdl) {
      (void)cudaGetLastError();
      if (dev_ok) coop_pdl_refused[dev] = true;
      cfg.numAttrs = 1;
      e = cudaLaunchKernelEx(&cfg, kernel, mx, md, p);
    }
    return e;
  };
  // partial H tiles -> H, Hs; programmatic edge: it sets itself up while the quantize kernel drains
  auto finalize = [&](int grid) -> int {
    if constexpr (R_T > 0) {
      const int64_t tiles = ceil_div(p.rows, QF_ROWS);
      const int64_t contributors = ceil_div((int64_t)grid, tiles) + 1;   // CTAs whose ranges meet one row tile
      int parts = (int)ceil_div(contributors, 8);
      if (parts > 8) parts = 8;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)(R_T / 4), (unsigned)tiles, 1);
      cfg.blockDim = dim3(QF_ROWS, (unsigned)parts, 1);
      cfg.dynamicSmemBytes = parts > 1 ? (size_t)parts * QF_ROWS * sizeof(float4) : 0;   // none on the large shapes: the
      cfg.stream = st;                                                                    // blocks fit beside the quantize CTAs
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[0].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = attr;
      cfg.numAttrs = pdl_enabled() ? 1 : 0;
      FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_finalize_h<(R_T > 0 ? R_T : 16)>, p, grid, job));
      // The caller's GEMM may start beside k_finalize_h (gemm_pair.cu, lr_late) only if every finalize block has waited
      // for the quantize grid BEFORE it lets its dependents go, i.e. without the tile counters: with them the blocks
      // trigger at once and wait at their end, and a GEMM that skipped its own wait could read codes still being written.
      if (finalize_last != nullptr) *finalize_last = p.tile_cnt == nullptr;
    }
    return FT_OK;
  };
  // ---- single pass: the tensor amax is not known and every CTA can keep its whole range resident
  if (amax_t == nullptr && g_qf_mode != 1) {
    int64_t G;
    int smem;
    if (single_pass_geometry(p.rows, p.cols, R_T, nsm, &G, &p.nx, &p.nd, &smem)) {
      const cudaError_t e = launch(k_quantize_fused<R_T, true>, (unsigned)G, smem, true);
      if (e == cudaSuccess) return finalize((int)G);
      if (e != cudaErrorCooperativeLaunchTooLarge && e != cudaErrorNotSupported) {
        g_last_cuda_error = (int)e;
        return FT_ERR_CUDA;
      }
      (void)cudaGetLastError();   // cannot be co-resident here: two passes instead
    }
  }
  // ---- streaming: amax first (unless the caller supplied it), then the ring kernel
  if (amax_t == nullptr) {
    float* word = reinterpret_cast<float*>(p.ctl + WS_CTL_AMAX / 4);   // zero by the workspace invariant
    int rc = launch_amax(x, p.rows * p.cols, word, st, /*zero_first=*/false, /*pdl=*/after_kernel);
    if (rc != FT_OK) return rc;
    amax_t = word;
    after_kernel = true;
  }
  p.amax_in = amax_t;
  // Streaming: nearly every row tile is completed by a CTA whose range ENDS in it, so the sums cannot start before
  // the kernel's end whatever the protocol.  A caller that chains a GEMM (finalize_last != NULL) is better served by
  // the grid-wide wait + lr_late (the GEMM's 4-bit stages run beside the sums); a stand-alone call by the counters
  // (the finalize blocks are resident and start the moment the last slot lands).
  if (finalize_last != nullptr) {
    p.tile_cnt = nullptr;
    p.tile_done = nullptr;
  }
  const int stage = QF_X_BYTES + (R_T == 0 ? 0 : D_BYTES);
  int nxs = (QF_SMEM_MAX - 1024) / stage;          // as deep as shared memory allows: 9 x 24 KB, 7 x 32 KB, 12 x 16 KB
  if (nxs > QF_MAX_NX) nxs = QF_MAX_NX;
  p.nx = nxs;
  p.nd = nxs;
  const int smem = nxs * stage + 1024;
  const unsigned grid = (unsigned)(TC < nsm ? TC : nsm);
  const cudaError_t e = launch(k_quantize_fused<R_T, false>, grid, smem, false);
  if (e != cudaSuccess) {
    g_last_cuda_error = (int)e;
    return FT_ERR_CUDA;
  }
  return finalize((int)grid);
}

bool quantize_single_pass_fits(int64_t rows, int64_t cols, int r_t) {
  if (g_qf_mode == 1) return false;
  int64_t G;
  int nx, nd, smem;
  const int nsm = sm_count() < QF_MAX_GRID ? sm_count() : QF_MAX_GRID;
  return single_pass_geometry(rows, cols, r_t, nsm, &G, &nx, &nd, &smem);
}

// after_kernel: a kernel of the same call directly precedes this launch in the stream (programmatic edge allowed).
// finalize_last (may be NULL): set when the last launch is k_finalize_h, which writes only H and Hs (and the side job).
// side_job (may be NULL; needs a projection, i.e. a k_finalize_h launch): a slot sum that kernel runs as well.
int launch_quantize_fused(const void* x, int64_t rows, int64_t cols, const float* amax_t, const ft_proj* proj,
                          ft_qtensor* out, void* workspace, bool after_kernel, bool* finalize_last,
                          const SumJob* side_job, cudaStream_t st) {
  const int r_t = proj ? proj->r_t : 0;
  if (side_job != nullptr && side_job->n_slots > 0 && r_t == 0) return FT_ERR_INVALID_ARG;
  const SumJob job = side_job != nullptr ? *side_job : SumJob{nullptr, nullptr, 0, 0};
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
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  QFParams p = {};
  p.rows = rows;
  p.cols = cols;
  p.amax_in = amax_t;
  p.ctl = reinterpret_cast<uint32_t*>(ws);
  const bool tile_flags = ws != nullptr && r_t > 0 && ceil_div(rows, QF_ROWS) <= WS_CTL_MAX_TILES;
  p.tile_cnt = tile_flags ? reinterpret_cast<uint32_t*>(ws + WS_CTL_TILE_CNT) : nullptr;
  p.tile_done = tile_flags ? reinterpret_cast<uint32_t*>(ws + WS_CTL_TILE_DONE) : nullptr;
  p.slots = ws ? reinterpret_cast<float*>(ws + ws_layout(rows, r_t).slots_off) : nullptr;
  p.codes = out->codes;
  p.sf = out->sf;
  p.g_dec_out = out->tensor_dec_scale;
  p.sf_layout = out->sf_layout;
  p.h_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out) : nullptr;
  p.hs_out = proj ? reinterpret_cast<__nv_bfloat16*>(proj->out_scaled) : nullptr;
  p.other_dec_scale = proj ? proj->other_dec_scale : nullptr;
  p.chunks_per_tile = (int)(cols / QF_KC);
  p.total_chunks = ceil_div(rows, QF_ROWS) * (cols / QF_KC);
#ifdef FT_TRACE
  p.trace = g_qf_trace;
  p.dbg = getenv("FT_QF_DBG") ? atoi(getenv("FT_QF_DBG")) : 0;
#endif
  switch (r_t) {
    case 0: return launch_qf<0>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 16: return launch_qf<16>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 32: return launch_qf<32>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 48: return launch_qf<48>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 64: return launch_qf<64>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 80: return launch_qf<80>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 96: return launch_qf<96>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 112: return launch_qf<112>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    case 128: return launch_qf<128>(mx, md, p, x, amax_t, after_kernel, finalize_last, job, st);
    default: return FT_ERR_UNSUPPORTED_SHAPE;
  }
}

}  // namespace ft

#ifdef FT_TRACE
extern "C" int ft_debug_set_quantize_trace(unsigned long long* device_buffer) {
  ft::g_qf_trace = device_buffer;
  return 0;
}
#endif
