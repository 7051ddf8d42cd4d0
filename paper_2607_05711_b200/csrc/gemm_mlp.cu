// gemm_mlp.cu -- NEXT-1, MLP fusion (sec. 3.3: "we fuse the first fully connected (FC1) GEMM
// with the subsequent FC2 quantization kernel ... intermediate results [are] consumed immediately without
// materializing large tensors in global memory").  The FC1 GEMM of gemm_pair.cu (CTA pairs, 256 x 192 tiles, scale
// columns of their own) with a different epilogue: instead of writing bf16 Y1 it
//   - rounds y1 = bf16(alpha * acc), applies GeLU (tanh form as u sigmoid(2 t), fp32) and rounds z = bf16(gelu(y1));
//   - quantizes z AND y1 in 1x16 blocks along N1 (FC2's reduction dim) with the caller's tensor amax (delayed
//     scaling, reading O-16 of DESIGN.md): codes and tile-layout scales of Q(Z) -- FC2's A operand -- and of Q(Y1),
//     the pre-activation GeLU's backward consumes;
//   - stages the bf16 z tile in shared memory and the issuing thread multiplies it with the [192 x r2] slice of
//     FC2's down-projection D_f2 (tcgen05.mma kind::f16, cta_group::2, M = 256, N = r2, K = 16 x 12) into a THIRD
//     tensor-memory accumulator: H2 = Z D_f2 accumulates over the tiles a pair runs inside one 256-row tile and is
//     drained to a slot of the workspace at the end of that run (k_finalize_h2 sums the slots, as for the quantize
//     kernel); the low-rank branches of FC2 thus consume the bf16 Z (reading O-10 unchanged), which never exists
//     in global memory;
//   - tracks max |z| and max |y1| (this step's amax, for the next step's scaling).
// Tile order: tiles are numbered 256-row tile major and a pair owns a CONTIGUOUS range (at most two row tiles when
// the range is no longer than a row of tiles), so that H2 partials are flushed once or twice per pair.
// TMEM: two 192-column accumulators, 16 scale columns, r2 <= 112 columns of H2: 512.
// 12 epilogue warps (the epilogue is ~19 instructions per element: the MMAs of a tile take ~5.6 k cycles).
// Shared memory: 4 ring stages of 34 KB, the 48 KB z tile, the 24 KB D_f2 slice (this CTA's r2 / 2 columns).
#include <cstdio>
#include <cstdlib>

#include "common.cuh"
#include "quant_math.cuh"

namespace ft {

constexpr int ML_BM = 256, ML_BN = 192;
constexpr int ML_THREADS = 512;          // 4 control warps + 12 epilogue warps (three groups, one 64-column unit each)
constexpr int ML_A_BYTES = 128 * 128;
constexpr int ML_B_BYTES = (ML_BN / 2) * 128;
constexpr int ML_SFA_BYTES = 4 * 512;
constexpr int ML_SFB_BYTES = 2 * 4 * 512;
constexpr int ML_STAGE_BYTES = ML_A_BYTES + ML_B_BYTES + ML_SFA_BYTES + ML_SFB_BYTES;   // 34 KB
constexpr int ML_STAGES = 4;
constexpr int ML_Z_BYTES = 3 * 128 * 128;     // three 64-column boxes of the z tile (this CTA's 128 rows)
constexpr int ML_D2_BYTES = 3 * 64 * 128;     // 192 rows of D_f2 x this CTA's (<= 64) columns
constexpr int ML_SMEM = ML_STAGES * ML_STAGE_BYTES + ML_Z_BYTES + ML_D2_BYTES + 1024;
constexpr uint32_t ML_SF_COL = 2 * ML_BN;     // 384
constexpr uint32_t ML_H2_COL = 2 * ML_BN + 16;   // 400

struct MlpParams {
  int64_t M, N, K;          // FC1: [M x K] x [N x K]^T, N = N1
  int r_t, r2;              // low-rank width of FC1 (its up-projection stage) and of FC2 (the H2 accumulator)
  const float* g_dec_a;     // X
  const float* g_dec_b;     // R1
  const float* z_amax_in;   // delayed-scaling amax of Z and Y1 (device)
  const float* y1_amax_in;
  uint8_t* codes_z;         // [M x N/2]
  uint8_t* sf_z;            // FT_SF_TILE128x4 over [M x N/16]
  float* g_dec_z;
  uint8_t* codes_y1;
  uint8_t* sf_y1;
  float* g_dec_y1;
  unsigned int* z_amax_out;   // zero words (or NULL): receive the bit patterns of max |z|, max |y1|
  unsigned int* y1_amax_out;
  __nv_bfloat16* z_dbg;       // NULL in production: bf16 copies of Z and Y1 for the staged parity comparison
  __nv_bfloat16* y1_dbg;
  float* slots;               // [(pairs + row tiles) x 256 x r2] fp32 partial H2 tiles, layout [quad][row][4]
#ifdef FT_TRACE
  int dbg;                    // development builds: 1 = no GeLU, 2 = no quantizer arithmetic, 4 = no H2 MMAs, 8 = no stores
#endif
};

// sigmoid(2 t) with t = sqrt(2/pi) (u + 0.044715 u^3): 0.5 (1 + tanh t) without the cancellation of 1 + tanh for
// negative u.  exp2 and the reciprocal by the hardware approximations (2^-22 relative: far below half a bf16 ulp,
// the precision of the results that are kept).
__device__ __forceinline__ float gelu_sigmoid_f32(float u) {
  const float t2 = -2.0f * 1.4426950408889634f * 0.7978845608028654f * fmaf(0.044715f * u * u, u, u);   // -2 t log2(e)
  float e, s;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(t2));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(1.0f + e));
  return s;
}
// GeLU, tanh form: 0.5 u (1 + tanh t) = u sigmoid(2 t)
__device__ __forceinline__ float gelu_tanh_f32(float u) { return u * gelu_sigmoid_f32(u); }

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(ML_THREADS, 1)
k_gemm4_mlp(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
            const __grid_constant__ CUtensorMap map_sfa, const __grid_constant__ CUtensorMap map_sfb,
            const __grid_constant__ CUtensorMap map_h, const __grid_constant__ CUtensorMap map_u,
            const __grid_constant__ CUtensorMap map_d2, const MlpParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* const zs = smem + ML_STAGES * ML_STAGE_BYTES;     // the staged bf16 z tile: three SW128 boxes
  uint8_t* const d2s = zs + ML_Z_BYTES;                       // D_f2 slice: three boxes of 64 rows x 128 B
  __shared__ uint64_t full_bar[ML_STAGES], empty_bar[ML_STAGES];
  __shared__ uint64_t acc_full[2], acc_empty[2], z_full, z_free, d2_full, h2_full;
  __shared__ float enc_z[128], enc_y[128];
  __shared__ uint32_t tmem_base_s;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int64_t tiles_m = (p.M + ML_BM - 1) / ML_BM, tiles_n = p.N / ML_BN;
  const int64_t T = tiles_m * tiles_n;
  const int64_t pair_id = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int64_t t_begin = pair_id * T / n_pairs;
  const int n_local = (int)((pair_id + 1) * T / n_pairs - t_begin);   // >= 1 (pairs <= tiles)
  const int k4 = (int)((p.K + 255) / 256);
  const int klr = (p.r_t + 63) / 64;
  const int kiters = k4 + klr;
  const int64_t sf_tiles_k = p.K / 64;
  // local tile i = global tile t_begin + i = (row tile mt, column tile nt); a segment = the run inside one row tile
  auto seg_end = [&](int i) { return ((t_begin + i) % tiles_n) == tiles_n - 1 || i == n_local - 1; };

  const TensorScale ts_z = tensor_scale(__ldg(p.z_amax_in)), ts_y = tensor_scale(__ldg(p.y1_amax_in));
  if (threadIdx.x == 0) {
    prefetch_tmap(&map_a);
    prefetch_tmap(&map_b);
    prefetch_tmap(&map_sfa);
    prefetch_tmap(&map_sfb);
    prefetch_tmap(&map_d2);
    for (int s = 0; s < ML_STAGES; ++s) {
      mbar_init(&full_bar[s], 2);   // the leader's two producer threads
      mbar_init(&empty_bar[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&acc_full[a], 1);
      mbar_init(&acc_empty[a], 24);   // 12 epilogue warps x 2 CTAs (used in the leader only)
    }
    mbar_init(&z_full, 24);           // the z tile of both CTAs is staged (leader only)
    mbar_init(&z_free, 1);            // the H2 MMAs have read it (commit, both CTAs)
    mbar_init(&d2_full, 1);           // D_f2 slice landed (leader only)
    mbar_init(&h2_full, 1);           // a segment's H2 accumulator is complete (commit, both CTAs)
    fence_mbar_init();
    if (blockIdx.x == 0) {
      *p.g_dec_z = ts_z.g_dec;
      *p.g_dec_y1 = ts_y.g_dec;
    }
  }
  if (threadIdx.x < 128) {
    enc_z[threadIdx.x] = enc_of_sf8(threadIdx.x, ts_z.g_dec);
    enc_y[threadIdx.x] = enc_of_sf8(threadIdx.x, ts_y.g_dec);
  }
  if (warp == 2) {
    tmem_alloc2(&tmem_base_s, 512);
    tmem_relinquish2();
  }
  tc_fence_before();
  cluster_sync();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  pdl_wait();      // everything this kernel reads comes from the quantize pass before it (and k_finalize_h: Hs)
  pdl_trigger();

  if (warp == 0 || warp == 3) {
    // ===================================================== TMA producers (both CTAs): warp 0 loads A (X codes, Hs) and its
    // scales, warp 3 loads B (weight codes, U) with its scales and the D_f2 slices.  A thread pays ~95 cycles per TMA
    // instruction it issues: four per stage from one thread were 600 of the K loop's cycles per stage (gemm_pair.cu).
    if (elect_one()) {
      const bool load_a = warp == 0;
      int stage = 0;
      uint32_t phase = 0;
      // The D_f2 slice of tile j goes into the single slice buffer once the H2 MMAs of tile j - 1 have read it (z_free).
      // Those are issued after the K loop of tile j, so the load is placed ML_STAGES ring stages into tile j + 1: by
      // then the issuer has consumed a stage of tile j + 1 and z_free(j - 1) has fired -- the wait never stalls the ring
      // (at the head of the tile the producer sat on z_free while the ring ran empty, once per tile).
      auto load_d2 = [&](int j) {
        if (j >= 1) mbar_wait(&z_free, (uint32_t)(j - 1) & 1);
        const int64_t nt = (t_begin + j) % tiles_n;
        const uint32_t bar = map_to_cta(smem_u32(&d2_full), 0);
        if (leader) mbar_expect_tx(&d2_full, 2 * ML_D2_BYTES);
        for (int u = 0; u < 3; ++u)
          tma_load_2d_pair(d2s + u * 8192, &map_d2, bar, (int32_t)(rank * (p.r2 / 2)), (int32_t)(nt * ML_BN + u * 64));
      };
      const int kt_d2 = min(ML_STAGES, kiters - 1);
      for (int i = 0; i <= n_local; ++i) {
        if (i == n_local) {
          if (!load_a) load_d2(i - 1);
          break;
        }
        const int64_t tile = t_begin + i;
        const int64_t mt = tile / tiles_n, nt = tile % tiles_n;
        const int32_t m0 = (int32_t)(mt * ML_BM + rank * 128);
        const int32_t nb0 = (int32_t)(nt * ML_BN + rank * (ML_BN / 2));
        const int32_t sfa_row = (int32_t)((mt * 2 + rank) * sf_tiles_k), sfb_row = (int32_t)(nt * sf_tiles_k);
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t* sa = smem + stage * ML_STAGE_BYTES;
          uint8_t* sb = sa + ML_A_BYTES;
          const uint32_t bar = map_to_cta(smem_u32(&full_bar[stage]), 0);
          if (kt < k4) {
            if (load_a) {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * (ML_A_BYTES + ML_SFA_BYTES));
              tma_load_2d_pair(sa, &map_a, bar, kt * 128, m0);
              tma_load_2d_pair(sb + ML_B_BYTES, &map_sfa, bar, 0, sfa_row + kt * 4);
            } else {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * (ML_B_BYTES + ML_SFB_BYTES));
              tma_load_2d_pair(sb, &map_b, bar, kt * 128, nb0);
              tma_load_2d_pair(sb + ML_B_BYTES + ML_SFA_BYTES, &map_sfb, bar, 0, sfb_row + kt * 4);
            }
          } else {
            const int c0 = (kt - k4) * 64;
            if (load_a) {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * ML_A_BYTES);
              tma_load_2d_pair(sa, &map_h, bar, c0, m0);
            } else {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * ML_B_BYTES);
              tma_load_2d_pair(sb, &map_u, bar, c0, nb0);
            }
          }
          if (++stage == ML_STAGES) {
            stage = 0;
            phase ^= 1;
          }
          if (!load_a && kt == kt_d2 && i >= 1) load_d2(i - 1);
        }
      }
    }
  } else if (warp == 1 && leader) {
    // ===================================================== MMA issuer (leader only)
    if (elect_one()) {
      constexpr uint32_t idesc4 = idesc_nvf4(ML_BM, ML_BN), idesc16 = idesc_bf16(ML_BM, ML_BN);
      const uint32_t idesc_h2 = idesc_bf16(ML_BM, p.r2) | (1u << 16);   // B (the D_f2 slice) is MN-major
      const uint32_t sfa_t = tmem_base + ML_SF_COL, sfb_t = sfa_t + 8, h2_t = tmem_base + ML_H2_COL;
      const uint32_t zs_u = smem_u32(zs), d2_u = smem_u32(d2s);
      // H2 (+)= z tile [256 x 192] * D_f2 slice [192 x r2]: 12 MMAs of K = 16 on the staged tile of local tile j
#ifdef FT_TRACE
      long long tr_k = 0, tr_zw = 0, tr_dw = 0, tr_h2 = 0, tr_acc = 0, tr_t = clock64();
      const long long tr_start = tr_t;
#define MLP_TR(x) do { const long long now_ = clock64(); (x) += now_ - tr_t; tr_t = now_; } while (0)
#else
#define MLP_TR(x) do { } while (0)
#endif
      auto h2_step = [&](int j) {
        mbar_wait(&z_full, (uint32_t)j & 1);
        MLP_TR(tr_zw);
        mbar_wait(&d2_full, (uint32_t)j & 1);
        MLP_TR(tr_dw);
        tc_fence_after();
        const bool first = j == 0 || seg_end(j - 1);
#ifdef FT_TRACE
        if (!(p.dbg & 4))
#endif
#pragma unroll
        for (int u = 0; u < 3; ++u)
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mma_bf16_pair(h2_t, make_smem_desc(zs_u + u * 16384 + k * 32, 1024, 0, 2),
                          make_smem_desc(d2_u + u * 8192 + k * 2048, 1024, 8192, 2), idesc_h2,
                          (first && u == 0 && k == 0) ? 0u : 1u);
        tc_commit_pair(&z_free, 3);                 // the z tile and the slice may be overwritten
        if (seg_end(j)) tc_commit_pair(&h2_full, 3);   // the row tile's partial H2 is complete
        MLP_TR(tr_h2);
      };
      int stage = 0;
      uint32_t phase = 0;
      for (int i = 0; i < n_local; ++i) {
        const int a = i & 1;
        const uint32_t acc_t = tmem_base + a * ML_BN;
        mbar_wait(&acc_empty[a], (((uint32_t)i >> 1) & 1) ^ 1);   // tile i-2 drained
        tc_fence_after();
        MLP_TR(tr_acc);
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * ML_STAGE_BYTES);
          const uint32_t sb = sa + ML_A_BYTES;
          if (kt < k4) {
            const int nk = (int)min((int64_t)4, sf_tiles_k - (int64_t)kt * 4);
            const uint32_t ssfa = sb + ML_B_BYTES, ssfb = ssfa + ML_SFA_BYTES;
            const uint64_t da = make_smem_desc(sa, 1024, 0, 2), db = make_smem_desc(sb, 1024, 0, 2);
            const uint64_t dfa = make_smem_desc(ssfa, 128, 0, 0), dfb = make_smem_desc(ssfb, 128, 0, 0);
            for (int k = 0; k < nk; ++k) {
              tc_cp_sf_pair(sfa_t, dfa + (uint64_t)(k * 32));
              tc_cp_sf_pair(sfb_t, dfb + (uint64_t)(k * 64));
              tc_cp_sf_pair(sfb_t + 4, dfb + (uint64_t)(k * 64 + 32));
              mma_nvf4_pair(acc_t, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc4, sfa_t, sfb_t, (kt | k) != 0);
            }
          } else {
            const int cols = min(64, p.r_t - (kt - k4) * 64);
            for (int k = 0; k < cols / 16; ++k)
              mma_bf16_pair(acc_t, make_smem_desc(sa + k * 32, 1024, 0, 2),
                            make_smem_desc(sb + k * 32, 1024, 0, 2), idesc16, 1u);
          }
          tc_commit_pair(&empty_bar[stage], 3);
          if (kt == kiters - 1) tc_commit_pair(&acc_full[a], 3);
          if (++stage == ML_STAGES) {
            stage = 0;
            phase ^= 1;
          }
        }
        MLP_TR(tr_k);
        if (i >= 1) h2_step(i - 1);   // the z tile of the tile before is staged by now (its epilogue ran beside this tile)
      }
      h2_step(n_local - 1);
#ifdef FT_TRACE
      if (pair_id == 0 || pair_id == 41)
        printf("mlp pair %d: %d tiles, per tile: acc_empty wait %.0f, K loop %.0f, z_full wait %.0f, d2_full wait %.0f, H2 issue %.0f; total %lld cycles\n",
               (int)pair_id, n_local, (double)tr_acc / n_local, (double)tr_k / n_local, (double)tr_zw / n_local, (double)tr_dw / n_local,
               (double)tr_h2 / n_local, clock64() - tr_start);
#endif
    }
  } else if (warp >= 4) {
    // ===================================================== epilogue (both CTAs, own 128 rows)
    // Three groups of four warps (a warp may read the TMEM lane quarter warp % 4); group g takes the 64-column unit g
    // of the 192-column accumulator, in two halves of 32 columns.  Thread = one row of the tile.  (Two groups with
    // two and one unit: 144 us at C3 -- a warp's 2 500 dependent instructions per tile set the pace, not the MMAs.)
    const int q = warp & 3;
    const int grp = (warp - 4) >> 2;
    const int et = (threadIdx.x - 128) & 127;  // 0..127 = row of this CTA's half tile
    const float alpha = __fmul_rn(__ldg(p.g_dec_a), __ldg(p.g_dec_b));
    const uint32_t enc_z_u = smem_u32(enc_z), enc_y_u = smem_u32(enc_y);
    const int64_t half_cols = p.N / 2, sf_tiles_n = p.N / 64;
    uint32_t amax_z2 = 0, amax_y2 = 0;   // running max of the bf16 magnitudes, two per word
    int seg = 0;                         // segments whose H2 accumulator this thread has drained
#ifdef FT_TRACE
    long long e_accw = 0, e_ld = 0, e_zfw = 0, e_math = 0, e_drain = 0;
#endif
    // drain the H2 accumulator of the row tile mt to this pair's slot: 16-column pieces alternate between the groups
    auto drain_h2 = [&](int64_t mt) {
      mbar_wait(&h2_full, (uint32_t)seg & 1);
      tc_fence_after();
      float* dst = p.slots + (pair_id + mt) * (int64_t)(ML_BM * p.r2) + (rank * 128 + q * 32 + lane) * 4;
      for (int c0 = grp * 16; c0 < p.r2; c0 += 48) {
        uint32_t v[16];
        tmem_ld16(tmem_base + ((uint32_t)(q * 32) << 16) + ML_H2_COL + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; j += 4)
          *reinterpret_cast<uint4*>(dst + (int64_t)((c0 + j) / 4) * (ML_BM * 4)) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
      }
      tc_fence_before();
      ++seg;
    };
    for (int i = 0; i < n_local; ++i) {
      const int a = i & 1;
      const int64_t tile = t_begin + i;
      const int64_t mt = tile / tiles_n, nt = tile % tiles_n;
      const int64_t row = mt * ML_BM + rank * 128 + et;
      const bool live = row < p.M;
#ifdef FT_TRACE
      long long e_t = clock64();
#define EPI_TR(x) do { const long long now_ = clock64(); (x) += now_ - e_t; e_t = now_; } while (0)
#else
#define EPI_TR(x) do { } while (0)
#endif
      mbar_wait(&acc_full[a], ((uint32_t)i >> 1) & 1);
      tc_fence_after();
      EPI_TR(e_accw);
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + a * ML_BN;
      {
        const int u = grp;
        uint8_t* zrow = zs + u * 16384 + et * 128;
        uint32_t cz[4], cy[4], sfz = 0, sfy = 0;
        uint4 cz_lo = make_uint4(0, 0, 0, 0), cy_lo = cz_lo;
#pragma unroll 1
        for (int hh = 0; hh < 2; ++hh) {     // two halves of 32 columns: 32 accumulator words in registers at a time
          uint32_t v[32];
          tmem_ld32(t0 + u * 64 + hh * 32, v);
          tmem_ld_wait();
          // the H2 MMAs of the tile before must have read the staged z before it is overwritten
          if (hh == 0) EPI_TR(e_ld);
          if (hh == 0 && i >= 1) mbar_wait(&z_free, (uint32_t)(i - 1) & 1);
          if (hh == 0) EPI_TR(e_zfw);
          if (hh == 1) {   // this warp's part of the accumulator is in registers: hand it back
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
          }
#pragma unroll
          for (int bb = 0; bb < 2; ++bb) {       // two 1x16 blocks of the half
            const int b = hh * 2 + bb;
            uint32_t yb[8], zb[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              yb[j] = pack_bf16x2(__uint_as_float(v[16 * bb + 2 * j]) * alpha, __uint_as_float(v[16 * bb + 2 * j + 1]) * alpha);
#if defined(FT_MLP_CT) && (FT_MLP_CT & 1)
              zb[j] = yb[j];   // development builds: no GeLU at all (compile time)
#else
              zb[j] = pack_bf16x2(gelu_tanh_f32(__uint_as_float(yb[j] << 16)), gelu_tanh_f32(__uint_as_float(yb[j] & 0xFFFF0000u)));
#endif
#ifdef FT_TRACE
              if (p.dbg & 1) zb[j] = yb[j];
#endif
            }
            const uint4 y0 = make_uint4(yb[0], yb[1], yb[2], yb[3]), y1 = make_uint4(yb[4], yb[5], yb[6], yb[7]);
            const uint4 z0 = make_uint4(zb[0], zb[1], zb[2], zb[3]), z1 = make_uint4(zb[4], zb[5], zb[6], zb[7]);
            // z goes to the staged tile (the A operand of the H2 MMAs): two 16-byte pieces of the swizzled row
            *reinterpret_cast<uint4*>(zrow + (((2 * b) ^ (et & 7)) << 4)) = z0;
            *reinterpret_cast<uint4*>(zrow + (((2 * b + 1) ^ (et & 7)) << 4)) = z1;
#if defined(FT_MLP_CT) && (FT_MLP_CT & 2)
            cz[2 * bb] = z0.x; cz[2 * bb + 1] = z1.x; cy[2 * bb] = y0.x; cy[2 * bb + 1] = y1.x;   // no quantizer at all
            continue;
#endif
            const float az = amax_block16(z0, z1), ay = amax_block16(y0, y1);
            amax_z2 = __vmaxu2(amax_z2, __float_as_uint(az) >> 16);
            amax_y2 = __vmaxu2(amax_y2, __float_as_uint(ay) >> 16);
            const uint32_t sz = block_sf8(az, ts_z.g_enc), sy = block_sf8(ay, ts_y.g_enc);
            float ez, ey;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(ez) : "r"(enc_z_u + sz * 4));
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(ey) : "r"(enc_y_u + sy * 4));
#ifdef FT_TRACE
            if (p.dbg & 2) {
              cz[2 * bb] = z0.x; cz[2 * bb + 1] = z1.x; cy[2 * bb] = y0.x; cy[2 * bb + 1] = y1.x;
            } else
#endif
            {
            cz[2 * bb] = quant_bf16x8_fast(z0, ez);
            cz[2 * bb + 1] = quant_bf16x8_fast(z1, ez);
            cy[2 * bb] = quant_bf16x8_fast(y0, ey);
            cy[2 * bb + 1] = quant_bf16x8_fast(y1, ey);
            }
            sfz |= sz << (8 * b);
            sfy |= sy << (8 * b);
            if (p.z_dbg != nullptr && live) {   // parity tests only: bf16 copies for the staged comparison
              const int64_t o = row * p.N + nt * ML_BN + u * 64 + b * 16;
              *reinterpret_cast<uint4*>(p.z_dbg + o) = z0;
              *reinterpret_cast<uint4*>(p.z_dbg + o + 8) = z1;
              *reinterpret_cast<uint4*>(p.y1_dbg + o) = y0;
              *reinterpret_cast<uint4*>(p.y1_dbg + o + 8) = y1;
            }
          }
          // codes: the unit's 32 bytes per row and tensor leave as ONE 256-bit store -- a full sector per lane (two
          // 16-byte stores per sector cost twice the L1 transactions: 23 us of the kernel at C3)
          if (hh == 0) {
            cz_lo = make_uint4(cz[0], cz[1], cz[2], cz[3]);
            cy_lo = make_uint4(cy[0], cy[1], cy[2], cy[3]);
          } else
#ifdef FT_TRACE
          if (!(p.dbg & 8))
#endif
          if (live) {
            const int64_t co = row * half_cols + (nt * ML_BN + u * 64) / 2;
            st_global_v8(p.codes_z + co, cz_lo, make_uint4(cz[0], cz[1], cz[2], cz[3]));
            st_global_v8(p.codes_y1 + co, cy_lo, make_uint4(cy[0], cy[1], cy[2], cy[3]));
          }
        }
        // scales: one word per row, unit and tensor in the tile layout
        const int64_t so = ((row >> 7) * sf_tiles_n + nt * 3 + u) * 512 + (row & 31) * 16 + ((row & 127) >> 5) * 4;
        if (live) {
          *reinterpret_cast<uint32_t*>(p.sf_z + so) = sfz;
          *reinterpret_cast<uint32_t*>(p.sf_y1 + so) = sfy;
        } else if (row < ((p.M + 127) & ~(int64_t)127)) {   // padding rows of the last 128-row scale tile read as zero
          *reinterpret_cast<uint32_t*>(p.sf_z + so) = 0u;
          *reinterpret_cast<uint32_t*>(p.sf_y1 + so) = 0u;
        }
      }
      // the H2 accumulator of a row tile that ended with the tile before must be out before the H2 MMAs of THIS
      // tile (which follow this warp's z_full arrival) overwrite it
      EPI_TR(e_math);
      if (i >= 1 && seg_end(i - 1)) drain_h2((t_begin + i - 1) / tiles_n);
      EPI_TR(e_drain);
      fence_proxy_async();   // the staged z is read by the tensor core (async proxy)
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&z_full), 0));
    }
    drain_h2((t_begin + n_local - 1) / tiles_n);
#ifdef FT_TRACE
    if (pair_id == 0 && rank == 0 && (warp == 4 || warp == 9) && lane == 0)
      printf("mlp epilogue warp %d: per tile: acc_full wait %.0f, first tmem load %.0f, z_free wait %.0f, math+stores %.0f, drain_h2 %.0f\n",
             warp, (double)e_accw / n_local, (double)e_ld / n_local, (double)e_zfw / n_local, (double)e_math / n_local, (double)e_drain / n_local);
#endif
    // this step's tensor amax of Z and Y1 (for the next step's scaling)
    if (p.z_amax_out != nullptr) {
      uint32_t bz = max(amax_z2 & 0xFFFFu, amax_z2 >> 16), by = max(amax_y2 & 0xFFFFu, amax_y2 >> 16);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        bz = max(bz, __shfl_xor_sync(0xffffffffu, bz, o));
        by = max(by, __shfl_xor_sync(0xffffffffu, by, o));
      }
      if (lane == 0) {
        if (bz != 0) atomicMax(p.z_amax_out, bz << 16);
        if (by != 0) atomicMax(p.y1_amax_out, by << 16);
      }
    }
  }

  tc_fence_before();
  cluster_sync();   // no CTA of the pair exits (or frees TMEM) while its peer still uses it
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc2(tmem_base, 512);
  }
}

// H2[row] = sum of the row tile's slots in pair order -> bf16 H2 and Hs2 = H2 * (1 / alpha2), alpha2 = g_dec(Z) *
// g_dec(R2).  One thread per (row, column quad); a 256-row tile has ~4 contributing pairs.  Fixed order of additions.
__global__ void __launch_bounds__(256) k_finalize_h2(const float* __restrict__ slots, int64_t rows, int r2, int64_t tiles_n,
                                                     int64_t T, int64_t P, const float* g_dec_z, const float* g_dec_r2,
                                                     __nv_bfloat16* __restrict__ h_out, __nv_bfloat16* __restrict__ hs_out) {
  pdl_wait();
  pdl_trigger();
  const int quads = r2 / 4;
  const int64_t slot_f4 = (int64_t)ML_BM * r2 / 4;
  const int r = threadIdx.x, q = blockIdx.x;
  const int64_t mt = blockIdx.y;
  const int64_t gr = mt * ML_BM + r;
  (void)quads;
  // the pairs whose ranges meet row tile mt: owner(tile) = floor(((tile + 1) * P - 1) / T)
  const int i_lo = (int)(((mt * tiles_n + 1) * P - 1) / T);
  const int i_hi = (int)((((mt + 1) * tiles_n) * P - 1) / T);
  const float4* src = reinterpret_cast<const float4*>(slots) + (i_lo + mt) * slot_f4 + (int64_t)q * ML_BM + r;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  constexpr int BATCH = 8;
  for (int i = i_lo; i <= i_hi; i += BATCH) {
    float4 v[BATCH];
#pragma unroll
    for (int j = 0; j < BATCH; ++j)
      v[j] = (i + j <= i_hi) ? __ldcg(src + (int64_t)(i - i_lo + j) * slot_f4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int j = 0; j < BATCH; ++j) {
      acc.x += v[j].x;
      acc.y += v[j].y;
      acc.z += v[j].z;
      acc.w += v[j].w;
    }
  }
  if (gr >= rows) return;
  const float inv_alpha = __fdiv_rn(1.0f, __fmul_rn(__ldcg(g_dec_z), __ldg(g_dec_r2)));
  if (h_out != nullptr)
    *reinterpret_cast<uint2*>(h_out + gr * r2 + q * 4) = make_uint2(pack_bf16x2(acc.x, acc.y), pack_bf16x2(acc.z, acc.w));
  *reinterpret_cast<uint2*>(hs_out + gr * r2 + q * 4) =
      make_uint2(pack_bf16x2(__fmul_rn(acc.x, inv_alpha), __fmul_rn(acc.y, inv_alpha)),
                 pack_bf16x2(__fmul_rn(acc.z, inv_alpha), __fmul_rn(acc.w, inv_alpha)));
}

// dY1 = bf16( dZ * gelu'(dequant(Q(Y1))) ): GeLU's backward on the 4-bit saved pre-activation (reading O-16).
// One thread per 1x16 block: 32 bytes of dZ, 8 bytes of codes, one scale byte (tile layout).
__global__ void __launch_bounds__(256) k_gelu_bwd_q4(const uint4* __restrict__ dz, const uint8_t* __restrict__ codes,
                                                     const uint8_t* __restrict__ sf, const float* __restrict__ g_dec,
                                                     uint4* __restrict__ out, int64_t rows, int64_t cols) {
  const int64_t nblk = cols / 16;
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= rows * nblk) return;
  const int64_t row = t / nblk, bc = t % nblk;
  const float scale = e4m3_to_f32(sf[sf_tile_offset(row, bc, nblk)]) * __ldg(g_dec);
  const uint2 c = *reinterpret_cast<const uint2*>(codes + row * (cols / 2) + bc * 8);
  const uint4 g0 = __ldg(dz + t * 2), g1 = __ldg(dz + t * 2 + 1);
  const uint32_t gw[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
  const uint32_t cw[2] = {c.x, c.y};
  uint32_t o[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {   // two elements per word of dZ, one byte of codes
    const uint32_t byte = (cw[j >> 2] >> (8 * (j & 3))) & 0xFFu;
    float y[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t code = (byte >> (4 * h)) & 0xFu;
      const uint32_t m = code & 7u;
      // E2M1 magnitudes 0, .5, 1, 1.5, 2, 3, 4, 6
      const float mag = m < 2 ? 0.5f * m : __uint_as_float(((m >> 1) + 126u) << 23 | (m & 1u) << 22);
      y[h] = (code & 8u) ? -mag * scale : mag * scale;
    }
    float r[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      // gelu(u) = u s, s = sigmoid(2 t):  gelu' = s + u s (1 - s) 2 t',  t' = sqrt(2/pi) (1 + 3 * 0.044715 u^2)
      const float u = y[h], sg = gelu_sigmoid_f32(u);
      const float grad = sg + u * sg * (1.0f - sg) * (2.0f * 0.7978845608028654f) * (1.0f + 0.134145f * u * u);
      const float gv = h == 0 ? __uint_as_float(gw[j] << 16) : __uint_as_float(gw[j] & 0xFFFF0000u);
      r[h] = gv * grad;
    }
    o[j] = pack_bf16x2(r[0], r[1]);
  }
  out[t * 2] = make_uint4(o[0], o[1], o[2], o[3]);
  out[t * 2 + 1] = make_uint4(o[4], o[5], o[6], o[7]);
}

int launch_gelu_bwd_q4(const void* dz, const ft_qtensor* qy1, void* out, cudaStream_t st) {
  const int64_t blocks = qy1->rows * (qy1->cols / 16);
  k_gelu_bwd_q4<<<(unsigned)ceil_div(blocks, 256), 256, 0, st>>>(reinterpret_cast<const uint4*>(dz), qy1->codes, qy1->sf,
                                                                 qy1->tensor_dec_scale, reinterpret_cast<uint4*>(out),
                                                                 qy1->rows, qy1->cols);
  FT_CUDA_TRY(cudaGetLastError());
  return FT_OK;
}

// FC1 GEMM with the fused GeLU / quantize / FC2-down-projection epilogue, then the sums of the H2 partials.
// a = Q(X) [M x K], b = Q(R1) [N1 x K] with sf_ntile cut to 192; lr_a = Hs1 [M x r_t], lr_b = U_t1 [N1 x r_t];
// d2 = D_f2 [N1 x r2]; qz / qy1: outputs (codes, TILE128x4 scales, tensor scales); h2 / hs2 [M x r2]; slots:
// mlp_slot_bytes() of scratch.  Requirements: N1 % 192 == 0, K % 64 == 0, 16 <= r2 <= 112, r2 % 16 == 0.
int launch_gemm4_mlp(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N1, int64_t K, const void* lr_a,
                     const void* lr_b, int r_t, const void* d2, int r2, const float* g_dec_r2, const float* z_amax_in,
                     const float* y1_amax_in, ft_qtensor* qz, ft_qtensor* qy1, unsigned int* z_amax_out,
                     unsigned int* y1_amax_out, void* z_dbg, void* y1_dbg, void* h2, void* hs2, float* slots,
                     cudaStream_t st) {
  if (N1 % ML_BN != 0 || K % 64 != 0 || r2 < 16 || r2 > 112 || r2 % 16 != 0) return FT_ERR_UNSUPPORTED_SHAPE;
  if (b->sf_ntile == nullptr || b->ntile != ML_BN) return FT_ERR_INVALID_ARG;
  CUtensorMap ma, mb, msa, msb, mh, mu, md2;
  int rc = make_tensor_map_2d(&ma, a->codes, 1, (uint64_t)K / 2, (uint64_t)M, (uint64_t)K / 2, 128, 128, Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&mb, b->codes, 1, (uint64_t)K / 2, (uint64_t)N1, (uint64_t)K / 2, 128, ML_BN / 2, Swizzle::B128);
  if (rc != FT_OK) return rc;
  const uint64_t tk = (uint64_t)K / 64;
  rc = make_tensor_map_2d(&msa, a->sf, 4, 128, (uint64_t)ceil_div(M, 128) * tk, 512, 128, 4, Swizzle::None);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&msb, b->sf_ntile, 4, 256, (uint64_t)(N1 / ML_BN) * tk, 1024, 256, 4, Swizzle::None);
  if (rc != FT_OK) return rc;
  if (r_t > 0) {
    rc = make_tensor_map_2d(&mh, lr_a, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, 128, Swizzle::B128);
    if (rc != FT_OK) return rc;
    rc = make_tensor_map_2d(&mu, lr_b, 2, (uint64_t)r_t, (uint64_t)N1, (uint64_t)r_t * 2, 64, ML_BN / 2, Swizzle::B128);
    if (rc != FT_OK) return rc;
  } else {
    mh = ma;
    mu = mb;
  }
  rc = make_tensor_map_2d(&md2, d2, 2, (uint64_t)r2, (uint64_t)N1, (uint64_t)r2 * 2, 64, 64, Swizzle::B128);
  if (rc != FT_OK) return rc;
  MlpParams p;
  p.M = M;
  p.N = N1;
  p.K = K;
  p.r_t = r_t;
  p.r2 = r2;
  p.g_dec_a = a->tensor_dec_scale;
  p.g_dec_b = b->tensor_dec_scale;
  p.z_amax_in = z_amax_in;
  p.y1_amax_in = y1_amax_in;
  p.codes_z = qz->codes;
  p.sf_z = qz->sf;
  p.g_dec_z = qz->tensor_dec_scale;
  p.codes_y1 = qy1->codes;
  p.sf_y1 = qy1->sf;
  p.g_dec_y1 = qy1->tensor_dec_scale;
  p.z_amax_out = z_amax_out;
  p.y1_amax_out = y1_amax_out;
  p.z_dbg = reinterpret_cast<__nv_bfloat16*>(z_dbg);
  p.y1_dbg = reinterpret_cast<__nv_bfloat16*>(y1_dbg);
  p.slots = slots;
#ifdef FT_TRACE
  p.dbg = getenv("FT_MLP_DBG") ? atoi(getenv("FT_MLP_DBG")) : 0;
#endif
  FT_CUDA_TRY(cudaFuncSetAttribute(k_gemm4_mlp, cudaFuncAttributeMaxDynamicSharedMemorySize, ML_SMEM));
  const int64_t tiles_m = ceil_div(M, ML_BM), tiles_n = N1 / ML_BN, T = tiles_m * tiles_n;
  const int64_t max_pairs = sm_count() / 2;
  const int64_t pairs = T < max_pairs ? T : max_pairs;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2u * (unsigned)pairs, 1, 1);
  cfg.blockDim = dim3(ML_THREADS, 1, 1);
  cfg.dynamicSmemBytes = ML_SMEM;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_gemm4_mlp, ma, mb, msa, msb, mh, mu, md2, p));
  cudaLaunchConfig_t cf = {};
  cf.gridDim = dim3((unsigned)(r2 / 4), (unsigned)tiles_m, 1);
  cf.blockDim = dim3(ML_BM, 1, 1);
  cf.stream = st;
  cf.attrs = attr;
  cf.numAttrs = pdl_enabled() ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cf, k_finalize_h2, (const float*)slots, M, r2, tiles_n, T, pairs,
                                 (const float*)qz->tensor_dec_scale, g_dec_r2, reinterpret_cast<__nv_bfloat16*>(h2),
                                 reinterpret_cast<__nv_bfloat16*>(hs2)));
  return FT_OK;
}

}  // namespace ft
