// gemm_pair.cu -- a2 / a4 on CTA pairs: the same computation as gemm.cu,
//     out = bf16( alpha * ( GEMM4(a, b) + Hs * U^T ) ),
// with tcgen05.mma.cta_group::2: the two CTAs of a cluster (2,1,1) own one 256 x BN output
// tile.  Each CTA stages its own 128 rows of A and its own BN/2-row half of B, so a CTA moves
// 128 + BN/2 operand rows through its shared memory per 128 x BN of output.  Ring: 5 stages of one K = 256 step.
// What paces the main loop (round 2, clock64 around the issuing thread's waits and FT_TRACE ablations,
// profiles/r02_experiments.md B6, B7): the single issuing thread spends ~530 cycles per stage whatever the tile width
// (a barrier wait of >= 100, 16 tcgen05 instructions, a multicast commit, the loop) against 512 (BN = 256) or 448
// (BN = 224) cycles of MMA; on top of that the forward pass, which writes a 256 x 224 tile every 13 stages, waits
// ~80 cycles per stage longer for its operands while the output is being stored (no stores: 69 k instead of 80 k
// cycles for the C2 forward launch).  Not the limit, each measured: the TMA unit (76-86 B/clk per SM in a probe, the
// loop needs 59-74), one thread issuing all loads (two threads: -2 %), the scale columns shared by the four K=64
// steps (own columns per step: no change), a sixth stage.
//
//   warp 0, 3: TMA producers (both CTAs; completion bytes land on the LEADER's full barrier): warp 0 loads A and
//              its scales, warp 3 loads B and its scales
//   warp 1   : tcgen05 issuer (leader CTA only): tcgen05.cp of the scale tiles, MMAs, commits
//              multicast to both CTAs' barriers
//   warp 2   : TMEM allocator (cta_group::2, both CTAs)
//   warps 4-11: epilogue of this CTA's 128 rows, two groups of four warps that take alternate 64-column
//              units of the accumulator: tcgen05.ld, * alpha, bf16, 256-bit global stores of the thread's own row
// TMEM: TWO BN-column fp32 accumulators, used alternately, so the epilogue of tile i overlaps the MMAs of
// tile i+1.  The block scales need 16 more columns (one K=64 step: 4 for A, 8 for B).
//   BN = 256: the accumulators fill all 512 columns, and the scales live in the first 16 columns of the
//     accumulator that is NOT being accumulated into -- the one the epilogue is draining -- which the
//     epilogue reads first and hands over at once (sf_free).  The tensor pipe drains between tiles: the next
//     tile's first scale copy waits for last MMA -> commit -> epilogue read -> remote arrive (~1.9 k cycles per
//     tile, 19 % of a K = 3072 tile).
//   BN = 224 / 192: 2 BN + 64 <= 512, the scales have columns of their own (16 per K=64 step of a stage) and the
//     issuer runs from one tile into the next without a hand-over.  The weight scales then come in a layout cut to the tile width
//     (ft_qtensor::sf_ntile, built offline by ft_pack_weight): tile nt, K=64 step ks -> two 512-byte
//     tcgen05.cp sources (rows 0-127 and 128-BN-1 of the tile), so one TMA box serves a K=256 stage.
//     N need not be a multiple of BN: the last tile of a row runs its MMAs with N_eff = N - nt BN (a multiple
//     of 32), B rows past N are zero-filled by TMA, the store is clipped.
// The scale copies are issued per K=64 step, three tcgen05.cp in front of each MMA (same rate as copying a
// whole stage up front: the FP4 probe's mode 1).
#include <cstdio>
#include <cstdlib>

#include "common.cuh"

namespace ft {

constexpr int P_BM = 256;              // pair tile rows (128 per CTA)
constexpr int P_THREADS = 384;         // 4 control warps + 8 epilogue warps
constexpr int P_A_BYTES = 128 * 128;   // 128 rows x 256 fp4 (or 64 bf16)
constexpr int P_SFA_BYTES = 4 * 512;   // this CTA's 128 rows, four K=64 steps
constexpr int P_SFB_BYTES = 2 * 4 * 512;  // all BN columns of the tile (two 128-row scale tiles per step)

template <int BN>
struct PairCfg {
  static constexpr bool OVERLAY = BN == 256;           // scale columns overlaid on the draining accumulator
  static constexpr int B_ROWS = BN / 2;                // rows of B staged per CTA
  static constexpr int B_BYTES = B_ROWS * 128;
  static constexpr int STAGE_BYTES = P_A_BYTES + B_BYTES + P_SFA_BYTES + P_SFB_BYTES;
  // ring depth 5 (a sixth stage, which fits for BN <= 224 now that the epilogue needs no staging, changes nothing)
  static constexpr int STAGES = 5;
  static constexpr int SMEM = STAGES * STAGE_BYTES + 1024;
  static constexpr uint32_t SF_COL = OVERLAY ? 0 : 2 * BN;   // TMEM column of the scales (OVERLAY: per tile)
  static constexpr bool SF_PER_STEP = !OVERLAY && 2 * BN + 64 <= 512;   // 16 scale columns for each K=64 step of a stage
  static_assert(BN % 16 == 0 && BN <= 256 && (OVERLAY || 2 * BN + 16 <= 512), "tile width");
  static_assert(STAGE_BYTES % 1024 == 0, "stage buffers stay 1024-byte aligned");
};

struct PairParams {
  int64_t M, N, K;
  int r_t;
  int lr_late;   // 1: only the low-rank operand Hs depends on the kernel in front (k_finalize_h), see below
  const float* g_dec_a;
  const float* g_dec_b;
  __nv_bfloat16* out;   // [M x N]: the epilogue stores rows straight from registers
  int out_align32;      // out is 32-byte aligned: 256-bit stores (else pairs of 128-bit ones)
#ifdef FT_TRACE
  int dbg;       // development builds: 1 = no scale loads, 2 = no epilogue work (timing only, wrong results)
#endif
};

template <int BN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(P_THREADS, 1)
k_gemm4_pair(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
             const __grid_constant__ CUtensorMap map_sfa, const __grid_constant__ CUtensorMap map_sfb,
             const __grid_constant__ CUtensorMap map_h, const __grid_constant__ CUtensorMap map_u,
             const PairParams p) {
  using Cfg = PairCfg<BN>;
  constexpr bool OVERLAY = Cfg::OVERLAY;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  constexpr int P_STAGES = Cfg::STAGES;
  __shared__ uint64_t full_bar[P_STAGES], empty_bar[P_STAGES];
  __shared__ uint64_t acc_full[2], acc_empty[2], sf_free[2];
  __shared__ uint32_t tmem_base_s;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  const int64_t tiles_m = (p.M + P_BM - 1) / P_BM, tiles_n = (p.N + BN - 1) / BN;
  const int64_t n_tiles = tiles_m * tiles_n;
  const int64_t pair_id = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int k4 = (int)((p.K + 255) / 256);
  const int klr = (p.r_t + 63) / 64;
  const int kiters = k4 + klr;
  const int64_t sf_tiles_k = p.K / 64;
  // width of tile column nt: BN, or what is left of N (a multiple of 16: N % 64 == 0, BN % 16 == 0)
  auto n_eff_of = [&](int64_t nt) { return (int)min((int64_t)BN, p.N - nt * BN); };

  if (threadIdx.x == 0) {
    prefetch_tmap(&map_a);
    prefetch_tmap(&map_b);
    prefetch_tmap(&map_sfa);
    prefetch_tmap(&map_sfb);
    for (int s = 0; s < P_STAGES; ++s) {
      mbar_init(&full_bar[s], 2);   // the leader's two producer threads arrive once each (with the pair's byte counts)
      mbar_init(&empty_bar[s], 1);  // one multicast commit per use
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&acc_full[a], 1);
      mbar_init(&acc_empty[a], 16);   // 8 epilogue warps x 2 CTAs (used in the leader only)
      mbar_init(&sf_free[a], 8);      // OVERLAY: the 4 warps of group 0 x 2 CTAs: first 16 columns read
    }
    fence_mbar_init();
  }
  if (warp == 2) {
    tmem_alloc2(&tmem_base_s, 512);
    tmem_relinquish2();
  }
  tc_fence_before();
  cluster_sync();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  // Programmatic edge to the kernel in front.  Normally everything this kernel reads comes from it: wait, then
  // let the next kernel set itself up.  lr_late: the kernel in front is k_finalize_h, which writes only the
  // low-rank operand Hs (and H), and every one of ITS CTAs has passed its own wait before this grid could
  // start -- so the quantize kernel before it had completed, and with it the codes, scales and tensor scales.
  // The 4-bit stages of the first tile then run beside k_finalize_h; each producer waits just before its first
  // Hs load and triggers the dependents only there (the dA kernel behind us reads P, also written by
  // k_finalize_h).  INVARIANT the host keeps (launch_gemm4_pair's only lr_late caller is linear_pass in api.cu):
  // the launch directly in front of this one is k_finalize_h of the same call, with a programmatic edge.
  if (!p.lr_late) {
    pdl_wait();
    pdl_trigger();
  }

  if (warp == 0 || warp == 3) {
    // ===================================================== TMA producers (both CTAs): warp 0 loads A and its scales,
    // warp 3 loads B and its scales.  One thread pays ~95 cycles per TMA instruction it issues (plus ~40 for the
    // expect-arrive and >= 55 for the wait): five loads per K=256 stage from one thread are ~600 cycles of issue
    // against 512 cycles of MMA (profiles/r02_experiments.md B7).  Two threads in different warps issue side by side.
    if (elect_one()) {
      const bool load_a = warp == 0;
      int stage = 0;
      uint32_t phase = 0;
      bool lr_waited = !p.lr_late;
      for (int64_t tile = pair_id; tile < n_tiles; tile += n_pairs) {
        const int64_t mt = tile % tiles_m, nt = tile / tiles_m;
        const int n_eff = n_eff_of(nt);
        const int32_t m0 = (int32_t)(mt * P_BM + rank * 128);            // this CTA's rows of A
        const int32_t nb0 = (int32_t)(nt * BN + rank * (n_eff / 2));     // this CTA's half of B
        const int32_t sfa_row = (int32_t)((mt * 2 + rank) * sf_tiles_k);
        const int32_t sfb_row = (int32_t)((OVERLAY ? nt * 2 : nt) * sf_tiles_k);
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t* sa = smem + stage * Cfg::STAGE_BYTES;
          uint8_t* sb = sa + P_A_BYTES;
          const uint32_t bar = map_to_cta(smem_u32(&full_bar[stage]), 0);  // the leader's barrier
          if (kt < k4) {
#ifdef FT_TRACE
            if (p.dbg & 1) {
              if (load_a) {
                if (leader) mbar_expect_tx(&full_bar[stage], 2 * P_A_BYTES);
                tma_load_2d_pair(sa, &map_a, bar, kt * 128, m0);
              } else {
                if (leader) mbar_expect_tx(&full_bar[stage], 2 * Cfg::B_BYTES);
                tma_load_2d_pair(sb, &map_b, bar, kt * 128, nb0);
              }
            } else
#endif
            if (load_a) {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * (P_A_BYTES + P_SFA_BYTES));
              tma_load_2d_pair(sa, &map_a, bar, kt * 128, m0);
              tma_load_2d_pair(sb + Cfg::B_BYTES, &map_sfa, bar, 0, sfa_row + kt * 4);
            } else {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * (Cfg::B_BYTES + P_SFB_BYTES));
              tma_load_2d_pair(sb, &map_b, bar, kt * 128, nb0);
              uint8_t* ssfb = sb + Cfg::B_BYTES + P_SFA_BYTES;
              if constexpr (OVERLAY) {   // standard layout: the tile's two 128-row scale tiles
                tma_load_2d_pair(ssfb, &map_sfb, bar, 0, sfb_row + kt * 4);
                tma_load_2d_pair(ssfb + 2048, &map_sfb, bar, 0, sfb_row + (int32_t)sf_tiles_k + kt * 4);
              } else {                   // layout cut to the tile: [nt][k64][2][512 B], one box of 4 steps
                tma_load_2d_pair(ssfb, &map_sfb, bar, 0, sfb_row + kt * 4);
              }
            }
          } else {
            const int c0 = (kt - k4) * 64;
            if (load_a) {
              if (!lr_waited) {   // first Hs load of this CTA: k_finalize_h must be complete
                pdl_wait();
                pdl_trigger();
                lr_waited = true;
              }
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * P_A_BYTES);
              tma_load_2d_pair(sa, &map_h, bar, c0, m0);
            } else {
              if (leader) mbar_expect_tx(&full_bar[stage], 2 * Cfg::B_BYTES);
              tma_load_2d_pair(sb, &map_u, bar, c0, nb0);
            }
          }
          if (++stage == P_STAGES) {
            stage = 0;
            phase ^= 1;
          }
        }
      }
    }
  } else if (warp == 1 && leader) {
    // ===================================================== MMA issuer (leader only)
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      int i = 0;   // local tile index: accumulator i & 1
#ifdef FT_TRACE
      long long tr_wait = 0, tr_issue = 0, tr_commit = 0, tr_tile = 0, tr_gap = 0, tr_t = clock64();
      const long long tr_start = tr_t;
      int tr_n = 0;
#endif
      for (int64_t tile = pair_id; tile < n_tiles; tile += n_pairs, ++i) {
        const int a = i & 1;
#ifdef FT_TRACE
        { const long long now = clock64(); tr_gap += now - tr_t; tr_t = now; }
#endif
        const int n_eff = n_eff_of(tile / tiles_m);
        const uint32_t idesc4 = idesc_nvf4(P_BM, n_eff), idesc16 = idesc_bf16(P_BM, n_eff);
        const uint32_t acc_t = tmem_base + a * BN;
        // scales: 4 columns for A, 8 for B.  OVERLAY: in the first 16 columns of the other accumulator
        const uint32_t sfa_t = tmem_base + (OVERLAY ? (uint32_t)((a ^ 1) * 256) : Cfg::SF_COL);
        const uint32_t sfb_t = sfa_t + 8;
        mbar_wait(&acc_empty[a], (((uint32_t)i >> 1) & 1) ^ 1);              // tile i-2 drained
        if constexpr (OVERLAY) {
          if (i > 0) mbar_wait(&sf_free[a ^ 1], (((uint32_t)(i - 1)) >> 1) & 1);  // tile i-1: columns 0-15 read
        }
        tc_fence_after();
#ifdef FT_TRACE
        { const long long now = clock64(); tr_tile += now - tr_t; tr_t = now; }
#endif
        // One K stage = wait for the operands, 4 x (3 scale copies + 1 MMA), commit.  The issuing thread's own
        // instruction stream paces the main loop (~530 cycles per stage against 448-512 cycles of MMA: a barrier
        // wait, ~45 uniform-datapath instructions, a commit), so the loop over the full 4-bit stages is kept as small
        // as it can be: the ragged last stage and the low-rank stages are separate loops behind it.
        auto end_stage = [&](bool last) {
          tc_commit_pair(&empty_bar[stage], 3);            // frees the slot in both CTAs
          if (last) tc_commit_pair(&acc_full[a], 3);
          if (++stage == P_STAGES) {
            stage = 0;
            phase ^= 1;
          }
        };
        auto stage4 = [&](int nk, uint32_t first_acc) {     // a 4-bit stage of nk K=64 steps
          const uint32_t sa = smem_u32(smem + stage * Cfg::STAGE_BYTES);
          const uint32_t sb = sa + P_A_BYTES;
          const uint32_t ssfa = sb + Cfg::B_BYTES, ssfb = ssfa + P_SFA_BYTES;
          // one descriptor per operand and stage; the K=64 steps advance the 16-byte address field by a
          // constant (the stage buffers are 1024-byte aligned, the field cannot carry)
          const uint64_t da = make_smem_desc(sa, 1024, 0, 2), db = make_smem_desc(sb, 1024, 0, 2);
          const uint64_t dfa = make_smem_desc(ssfa, 128, 0, 0), dfb = make_smem_desc(ssfb, 128, 0, 0);
          // B scales of step k: OVERLAY: 512 B at k * 512 of each of the two 2 KB scale tiles;
          // else 1 KB (both halves) at k * 1024
          // BN <= 224: every K=64 step of a stage has its own 16 scale columns (2 BN + 64 <= 512), so the copies of
          // step k + 1 need not wait until the MMA of step k has read its scales (measured: no difference)
          auto step = [&](int k, uint32_t acc) {
            if constexpr (OVERLAY) {
              tc_cp_sf_pair(sfa_t, dfa + (uint64_t)(k * 32));
              tc_cp_sf_pair(sfb_t, dfb + (uint64_t)(k * 32));
              tc_cp_sf_pair(sfb_t + 4, dfb + (uint64_t)(128 + k * 32));
              mma_nvf4_pair(acc_t, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc4, sfa_t, sfb_t, acc);
            } else {
              const uint32_t fa = sfa_t + (Cfg::SF_PER_STEP ? 16 * k : 0), fb = fa + 8;
              tc_cp_sf_pair(fa, dfa + (uint64_t)(k * 32));
              tc_cp_sf_pair(fb, dfb + (uint64_t)(k * 64));
              tc_cp_sf_pair(fb + 4, dfb + (uint64_t)(k * 64 + 32));
              mma_nvf4_pair(acc_t, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc4, fa, fb, acc);
            }
          };
          if (nk == 4) {   // straight-line code
            step(0, first_acc);
            step(1, 1u);
            step(2, 1u);
            step(3, 1u);
          } else {
            for (int k = 0; k < nk; ++k) step(k, k == 0 ? first_acc : 1u);
          }
        };
        const int k4_full = (int)(p.K / 256);       // full 4-bit stages; k4 - k4_full (0 or 1) ragged ones
        uint32_t acc_flag = 0;
#pragma unroll 1
        for (int kt = 0; kt < k4_full; ++kt) {      // ---- the hot loop
#ifdef FT_TRACE
          { const long long now = clock64(); tr_gap += now - tr_t; tr_t = now; }
#endif
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
#ifdef FT_TRACE
          { const long long now = clock64(); tr_wait += now - tr_t; tr_t = now; ++tr_n; }
#endif
          stage4(4, acc_flag);
          acc_flag = 1;
#ifdef FT_TRACE
          { const long long now = clock64(); tr_issue += now - tr_t; tr_t = now; }
#endif
          end_stage(kt == kiters - 1);
#ifdef FT_TRACE
          { const long long now = clock64(); tr_commit += now - tr_t; tr_t = now; }
#endif
        }
        if (k4_full < k4) {                         // ---- ragged last 4-bit stage (K % 256 != 0)
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          stage4((int)(sf_tiles_k - (int64_t)k4_full * 4), acc_flag);
          end_stage(k4 == kiters);
        }
#pragma unroll 1
        for (int kt = k4; kt < kiters; ++kt) {      // ---- low-rank stages: Hs [128 x 64] x U [BN/2 x 64] chunks
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * Cfg::STAGE_BYTES);
          const uint32_t sb = sa + P_A_BYTES;
          const int cols = min(64, p.r_t - (kt - k4) * 64);
          for (int k = 0; k < cols / 16; ++k)
            mma_bf16_pair(acc_t, make_smem_desc(sa + k * 32, 1024, 0, 2),
                          make_smem_desc(sb + k * 32, 1024, 0, 2), idesc16, 1u);
          end_stage(kt == kiters - 1);
        }
      }
#ifdef FT_TRACE
      if (pair_id == 0 || pair_id == 41)
        printf("pair %d BN %d: stages %d, per stage: wait_full %.0f issue %.0f commit+loop %.0f gap %.0f; per tile hand-over %.0f; sum %lld total %lld cycles\n",
               (int)pair_id, BN, tr_n, (double)tr_wait / tr_n, (double)tr_issue / tr_n, (double)tr_commit / tr_n, (double)tr_gap / tr_n,
               (double)tr_tile / (i > 0 ? i : 1), tr_wait + tr_issue + tr_commit + tr_gap + tr_tile, clock64() - tr_start);
#endif
    }
  } else if (warp >= 4) {
    // ===================================================== epilogue (both CTAs, own 128 rows)
    // TMEM -> registers -> swizzled shared memory -> TMA store.  Two groups of four warps (a warp may read
    // the TMEM lane quarter warp % 4); group g takes the 64-column units g, g + 2, ... of the accumulator
    // (the last unit of a 224-wide or ragged tile is 32 columns: its own tensor map, 64-byte swizzle), through
    // its own 16 KB staging box.  The accumulator is released as soon as a warp has its last unit in registers.
    const int q = warp & 3;
    const int grp = (warp - 4) >> 2;
    const int et = (threadIdx.x - 128) & 127;  // 0..127 = row of this CTA's half tile
    const float alpha = __fmul_rn(__ldg(p.g_dec_a), __ldg(p.g_dec_b));
    int i = 0;   // local tile index, as in the MMA issuer
    for (int64_t tile = pair_id; tile < n_tiles; tile += n_pairs, ++i) {
      const int a = i & 1;
      const int64_t mt = tile % tiles_m, nt = tile / tiles_m;
      const int n_eff = n_eff_of(nt);
      const int32_t row0 = (int32_t)(mt * P_BM + rank * 128);
      const int32_t n0 = (int32_t)(nt * BN);
      mbar_wait(&acc_full[a], ((uint32_t)i >> 1) & 1);
      tc_fence_after();
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + a * BN;
      // units of this group that hold columns of the tile: u = grp, grp + 2, ... with u * 64 < n_eff
      const int n_units = (n_eff + 63) / 64;
      const int last_u = n_units - 1 - ((n_units - 1 - grp) & 1);   // this group's last unit (< grp: none)
      bool released = false;
#ifdef FT_TRACE
      if (p.dbg & 2) {   // timing only: no drain, no stores
        if (OVERLAY && grp == 0) {
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&sf_free[a]), 0));
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
        continue;
      }
#endif
#pragma unroll 1
      for (int u = grp; u < n_units; u += 2) {
        const int c0 = u * 64;
        const int w = min(64, n_eff - c0);   // unit width: 64, or what is left of the tile (a multiple of 16)
        uint32_t v[64];
        if (OVERLAY && u == 0) {
          // columns 0-15 of this accumulator are the next tile's scale-factor buffer: read them first and
          // hand them over, so the next tile's MMAs (other accumulator) start while the rest drains
          tmem_ld16(t0, *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
          tmem_ld_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&sf_free[a]), 0));
          if (w > 16) tmem_ld16(t0 + 16, *reinterpret_cast<uint32_t(*)[16]>(&v[16]));
        } else if (w >= 32) {
          tmem_ld32(t0 + c0, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        } else {
          tmem_ld16(t0 + c0, *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
        }
        if (w == 64) tmem_ld32(t0 + c0 + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        else if (w == 48) tmem_ld16(t0 + c0 + 32, *reinterpret_cast<uint32_t(*)[16]>(&v[32]));
        tmem_ld_wait();
        if (u == last_u) {   // this warp's part of the accumulator is in registers: hand it back
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
          released = true;
        }
        // bf16( alpha * acc ): a thread holds up to 64 consecutive columns of one row = 128 bytes, stored as
        // 256-bit pieces: every store instruction fills whole 32-byte sectors.  (Staging the tile in shared memory
        // for a TMA store put the output through the shared-memory ports and the TMA unit that the operand loads
        // need: the forward pass, one 256 x 224 tile per 13 stages, ran 21 % slower for it.)
        const int64_t grow = (int64_t)row0 + et;
#ifdef FT_TRACE
        if (p.dbg & 4) {   // timing only: TMEM read, no conversion, no stores (keep the registers alive)
          uint32_t x = 0;
#pragma unroll
          for (int j = 0; j < 64; ++j) x ^= v[j];
          if (x == 0x12345677u) p.out[0] = __float2bfloat16(1.0f);
          continue;
        }
#endif
        if (grow < p.M) {
          __nv_bfloat16* dst = p.out + grow * p.N + n0 + c0;
          const int pieces = w / 16;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if (j < pieces) {
              uint4 lo, hi;
              lo.x = pack_bf16x2(__uint_as_float(v[16 * j + 0]) * alpha, __uint_as_float(v[16 * j + 1]) * alpha);
              lo.y = pack_bf16x2(__uint_as_float(v[16 * j + 2]) * alpha, __uint_as_float(v[16 * j + 3]) * alpha);
              lo.z = pack_bf16x2(__uint_as_float(v[16 * j + 4]) * alpha, __uint_as_float(v[16 * j + 5]) * alpha);
              lo.w = pack_bf16x2(__uint_as_float(v[16 * j + 6]) * alpha, __uint_as_float(v[16 * j + 7]) * alpha);
              hi.x = pack_bf16x2(__uint_as_float(v[16 * j + 8]) * alpha, __uint_as_float(v[16 * j + 9]) * alpha);
              hi.y = pack_bf16x2(__uint_as_float(v[16 * j + 10]) * alpha, __uint_as_float(v[16 * j + 11]) * alpha);
              hi.z = pack_bf16x2(__uint_as_float(v[16 * j + 12]) * alpha, __uint_as_float(v[16 * j + 13]) * alpha);
              hi.w = pack_bf16x2(__uint_as_float(v[16 * j + 14]) * alpha, __uint_as_float(v[16 * j + 15]) * alpha);
#ifdef FT_TRACE
              if (p.dbg & 8) {   // timing only: conversion, no stores
                if ((lo.x ^ hi.w) == 0x12345677u) p.out[1] = __float2bfloat16(1.0f);
              } else if (p.dbg & 16) {   // timing only: the same stores into a per-CTA region that stays in L2
                st_global_v8(p.out + ((int64_t)(blockIdx.x * 128 + et)) * p.N + c0 + 16 * j, lo, hi);
              } else
#endif
              if (p.out_align32) {
                st_global_v8(dst + 16 * j, lo, hi);
              } else {
                *reinterpret_cast<uint4*>(dst + 16 * j) = lo;
                *reinterpret_cast<uint4*>(dst + 16 * j + 8) = hi;
              }
            }
          }
        }
      }
      if (!released) {   // a ragged tile with no unit for this group
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
      }
    }
  }

  if (p.lr_late) pdl_wait();   // every thread: "this grid complete" implies "k_finalize_h complete" (no-op if passed)
  tc_fence_before();
  cluster_sync();   // no CTA of the pair exits (or frees TMEM) while its peer still uses it
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc2(tmem_base, 512);
  }
}

int g_pair_bn = 0;   // test / bench hook: 0 = choose per shape, else force this pair tile width

// Tile width of the pair kernel for a shape: 256, or the width `ntile_avail` (224 / 240) the weight's tile-cut scales
// were packed for.  Cost model of the persistent schedule (profiles/r02_experiments.md B6): rounds of n_pairs
// tiles; a K=256 stage costs the issuing thread ~530 cycles or the MMAs' 4 x BN/2, whichever is more; BN = 256 pays
// the ~1.7 k-cycle hand-over of the overlaid scale columns per tile, the others ~270.
static double pair_cost(int bn, int64_t M, int64_t N, int64_t K, int r_t, int64_t pairs) {
  const double stage4 = 4.0 * (bn / 2) > 530.0 ? 4.0 * (bn / 2) : 530.0;
  double lr = 0.0;   // low-rank stages: up to four K=16 bf16 MMAs of BN/2 cycles each, or the thread's ~300
  for (int c = 0; c < r_t; c += 64) {
    const double mma = ((r_t - c < 64 ? r_t - c : 64) / 16) * (bn / 2.0);
    lr += mma > 300.0 ? mma : 300.0;
  }
  const double per_tile = (double)ceil_div(K, 256) * stage4 + lr + (bn == 256 ? 1700.0 : 270.0);
  const int64_t tiles = ceil_div(M, P_BM) * ceil_div(N, bn);   // a ragged last column tile costs a whole tile's issue time
  return (double)ceil_div(tiles, pairs) * per_tile;
}
static int choose_pair_bn(int64_t M, int64_t N, int64_t K, int r_t, int ntile_avail) {
  if (g_pair_bn != 0) return g_pair_bn;
  if (ntile_avail != 224 && ntile_avail != 240) return 256;
  const int64_t pairs = sm_count() / 2;
  return pair_cost(ntile_avail, M, N, K, r_t, pairs) < pair_cost(256, M, N, K, r_t, pairs) ? ntile_avail : 256;
}
// the tile-cut scale layout worth packing for a weight that will meet M tokens: 224, 240, or 0 (256-wide tiles win)
int best_pair_ntile(int64_t M, int64_t N, int64_t K, int r_t) {
  const int64_t pairs = sm_count() / 2;
  const double c256 = pair_cost(256, M, N, K, r_t, pairs);
  // a width that would leave a 16-column last tile is not run (launch_gemm4_pair): never worth packing for
  const double c224 = N % 224 == 16 ? 2.0 * c256 : pair_cost(224, M, N, K, r_t, pairs);
  const double c240 = N % 240 == 16 ? 2.0 * c256 : pair_cost(240, M, N, K, r_t, pairs);
  if (c256 <= c224 && c256 <= c240) return 0;
  return c240 < c224 ? 240 : 224;
}

template <int BN>
static int launch_pair_bn(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                          const void* lr_a, const void* lr_b, int r_t, void* out, bool lr_late, cudaStream_t st) {
  using Cfg = PairCfg<BN>;
  CUtensorMap ma, mb, msa, msb, mh, mu;
  int rc = make_tensor_map_2d(&ma, a->codes, 1, (uint64_t)K / 2, (uint64_t)M, (uint64_t)K / 2, 128, 128,
                              Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&mb, b->codes, 1, (uint64_t)K / 2, (uint64_t)N, (uint64_t)K / 2, 128, Cfg::B_ROWS,
                          Swizzle::B128);
  if (rc != FT_OK) return rc;
  // scale tiles: [row_tiles * K/64] tiles of 512 bytes = 128 uint32; one box = four K=64 steps
  const uint64_t tk = (uint64_t)K / 64;
  rc = make_tensor_map_2d(&msa, a->sf, 4, 128, (uint64_t)ceil_div(M, 128) * tk, 512, 128, 4, Swizzle::None);
  if (rc != FT_OK) return rc;
  if (Cfg::OVERLAY)
    rc = make_tensor_map_2d(&msb, b->sf, 4, 128, (uint64_t)ceil_div(N, 128) * tk, 512, 128, 4, Swizzle::None);
  else   // [n tiles * K/64] rows of 1024 bytes (both 128-row halves of one K=64 step)
    rc = make_tensor_map_2d(&msb, b->sf_ntile, 4, 256, (uint64_t)ceil_div(N, BN) * tk, 1024, 256, 4, Swizzle::None);
  if (rc != FT_OK) return rc;
  if (r_t > 0) {
    rc = make_tensor_map_2d(&mh, lr_a, 2, (uint64_t)r_t, (uint64_t)M, (uint64_t)r_t * 2, 64, 128, Swizzle::B128);
    if (rc != FT_OK) return rc;
    rc = make_tensor_map_2d(&mu, lr_b, 2, (uint64_t)r_t, (uint64_t)N, (uint64_t)r_t * 2, 64, Cfg::B_ROWS, Swizzle::B128);
    if (rc != FT_OK) return rc;
  } else {
    mh = ma;
    mu = mb;
  }
  PairParams p;
  p.M = M;
  p.N = N;
  p.K = K;
  p.r_t = r_t;
  p.lr_late = (lr_late && r_t > 0 && pdl_enabled()) ? 1 : 0;
  p.g_dec_a = a->tensor_dec_scale;
  p.g_dec_b = b->tensor_dec_scale;
  p.out = reinterpret_cast<__nv_bfloat16*>(out);
  p.out_align32 = (reinterpret_cast<uintptr_t>(out) & 31) == 0 ? 1 : 0;
#ifdef FT_TRACE
  p.dbg = getenv("FT_GEMM_DBG") ? atoi(getenv("FT_GEMM_DBG")) : 0;
#endif
  FT_CUDA_TRY(cudaFuncSetAttribute(k_gemm4_pair<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM));
  const int64_t n_tiles = ceil_div(M, P_BM) * ceil_div(N, BN);
  const int64_t max_pairs = sm_count() / 2;
  const unsigned grid = 2u * (unsigned)(n_tiles < max_pairs ? n_tiles : max_pairs);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid, 1, 1);
  cfg.blockDim = dim3(P_THREADS, 1, 1);
  cfg.dynamicSmemBytes = Cfg::SMEM;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_gemm4_pair<BN>, ma, mb, msa, msb, mh, mu, p));
  return FT_OK;
}

// lr_late: the launch directly in front of this one is k_finalize_h of the same call (see the kernel)
int launch_gemm4_pair(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                      const void* lr_a, const void* lr_b, int r_t, void* out, bool lr_late, cudaStream_t st) {
  const int avail = (b->sf_ntile != nullptr) ? b->ntile : 0;
  int bn = choose_pair_bn(M, N, K, r_t, avail);
  if (bn != 256 && bn != avail) bn = 256;   // no scale layout for that width: the 256-wide kernel takes the standard one
  // a last column tile of 16 columns would be an MMA of N = 16 across the pair (8 rows of B per CTA): below what the
  // instruction takes with M = 256.  256-wide tiles leave multiples of 64.
  if (bn != 256 && N % bn == 16) bn = 256;
  if (bn == 224) return launch_pair_bn<224>(a, b, M, N, K, lr_a, lr_b, r_t, out, lr_late, st);
  if (bn == 240) return launch_pair_bn<240>(a, b, M, N, K, lr_a, lr_b, r_t, out, lr_late, st);
  return launch_pair_bn<256>(a, b, M, N, K, lr_a, lr_b, r_t, out, lr_late, st);
}

}  // namespace ft
