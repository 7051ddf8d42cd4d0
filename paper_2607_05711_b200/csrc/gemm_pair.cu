// gemm_pair.cu -- a2 / a4 on CTA pairs: the same computation as gemm.cu,
//     out = bf16( alpha * ( GEMM4(a, b) + Hs * U^T ) ),
// with tcgen05.mma.cta_group::2: the two CTAs of a cluster (2,1,1) own one 256 x BN output
// tile.  Each CTA stages its own 128 rows of A and its own BN/2-row half of B, so a CTA moves
// 128 + BN/2 operand rows through its shared memory per 128 x BN of output: the main loop is bound
// by shared-memory traffic, not by the tensor pipe, and the pair halves the
// bytes per MAC.  Ring: 5 stages; the epilogue stages through one 16 KB box per warp group.
//
//   warp 0   : TMA producer (both CTAs; completion bytes land on the LEADER's full barrier)
//   warp 1   : tcgen05 issuer (leader CTA only): tcgen05.cp of the scale tiles, MMAs, commits
//              multicast to both CTAs' barriers
//   warp 2   : TMEM allocator (cta_group::2, both CTAs)
//   warps 4-11: epilogue of this CTA's 128 rows, two groups of four warps that take alternate 64-column
//              units of the accumulator: tcgen05.ld, * alpha, bf16, swizzled smem, TMA store
// TMEM: TWO BN-column fp32 accumulators, used alternately, so the epilogue of tile i overlaps the MMAs of
// tile i+1.  The block scales need 16 more columns (one K=64 step: 4 for A, 8 for B).
//   BN = 256: the accumulators fill all 512 columns, and the scales live in the first 16 columns of the
//     accumulator that is NOT being accumulated into -- the one the epilogue is draining -- which the
//     epilogue reads first and hands over at once (sf_free).  The tensor pipe drains between tiles: the next
//     tile's first scale copy waits for last MMA -> commit -> epilogue read -> remote arrive (~1.9 k cycles per
//     tile, 19 % of a K = 3072 tile).
//   BN = 224 / 192: 2 BN + 16 <= 512, the scales have columns of their own and the issuer runs from one tile
//     into the next without a hand-over.  The weight scales then come in a layout cut to the tile width
//     (ft_qtensor::sf_ntile, built offline by ft_pack_weight): tile nt, K=64 step ks -> two 512-byte
//     tcgen05.cp sources (rows 0-127 and 128-BN-1 of the tile), so one TMA box serves a K=256 stage.
//     N need not be a multiple of BN: the last tile of a row runs its MMAs with N_eff = N - nt BN (a multiple
//     of 32), B rows past N are zero-filled by TMA, the store is clipped.
// The scale copies are issued per K=64 step, three tcgen05.cp in front of each MMA (same rate as copying a
// whole stage up front: the FP4 probe's mode 1).
#include "common.cuh"

namespace ft {

constexpr int P_BM = 256;              // pair tile rows (128 per CTA)
constexpr int P_THREADS = 384;         // 4 control warps + 8 epilogue warps
constexpr int P_A_BYTES = 128 * 128;   // 128 rows x 256 fp4 (or 64 bf16)
constexpr int P_SFA_BYTES = 4 * 512;   // this CTA's 128 rows, four K=64 steps
constexpr int P_SFB_BYTES = 2 * 4 * 512;  // all BN columns of the tile (two 128-row scale tiles per step)
constexpr int P_STAGES = 5;
constexpr int P_OUT_BYTES = 128 * 128;     // one staged output box: 128 rows x 64 bf16

template <int BN>
struct PairCfg {
  static constexpr bool OVERLAY = BN == 256;           // scale columns overlaid on the draining accumulator
  static constexpr int B_ROWS = BN / 2;                // rows of B staged per CTA
  static constexpr int B_BYTES = B_ROWS * 128;
  static constexpr int STAGE_BYTES = P_A_BYTES + B_BYTES + P_SFA_BYTES + P_SFB_BYTES;
  static constexpr int SMEM = P_STAGES * STAGE_BYTES + 2 * P_OUT_BYTES + 1024;
  static constexpr uint32_t SF_COL = OVERLAY ? 0 : 2 * BN;   // TMEM column of the scales (OVERLAY: per tile)
  static_assert(BN % 32 == 0 && BN <= 256 && (OVERLAY || 2 * BN + 16 <= 512), "tile width");
  static_assert(STAGE_BYTES % 1024 == 0, "stage buffers stay 1024-byte aligned");
};

struct PairParams {
  int64_t M, N, K;
  int r_t;
  int lr_late;   // 1: only the low-rank operand Hs depends on the kernel in front (k_finalize_h), see below
  const float* g_dec_a;
  const float* g_dec_b;
};

template <int BN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(P_THREADS, 1)
k_gemm4_pair(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
             const __grid_constant__ CUtensorMap map_sfa, const __grid_constant__ CUtensorMap map_sfb,
             const __grid_constant__ CUtensorMap map_h, const __grid_constant__ CUtensorMap map_u,
             const __grid_constant__ CUtensorMap map_out, const __grid_constant__ CUtensorMap map_out32,
             const PairParams p) {
  using Cfg = PairCfg<BN>;
  constexpr bool OVERLAY = Cfg::OVERLAY;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
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
  // width of tile column nt: BN, or what is left of N (a multiple of 32: N % 64 == 0, BN % 32 == 0)
  auto n_eff_of = [&](int64_t nt) { return (int)min((int64_t)BN, p.N - nt * BN); };

  if (threadIdx.x == 0) {
    prefetch_tmap(&map_a);
    prefetch_tmap(&map_b);
    prefetch_tmap(&map_sfa);
    prefetch_tmap(&map_sfb);
    for (int s = 0; s < P_STAGES; ++s) {
      mbar_init(&full_bar[s], 1);   // leader's producer arrives once (with the pair's byte count)
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

  if (warp == 0) {
    // ===================================================== TMA producer (both CTAs)
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      bool lr_waited = !p.lr_late;
      for (int64_t tile = pair_id; tile < n_tiles; tile += n_pairs) {
        const int64_t mt = tile % tiles_m, nt = tile / tiles_m;
        const int n_eff = n_eff_of(nt);
        const int32_t m0 = (int32_t)(mt * P_BM + rank * 128);            // this CTA's rows of A
        const int32_t nb0 = (int32_t)(nt * BN + rank * (n_eff / 2));     // this CTA's half of B
        const int64_t sfa_rt = mt * 2 + rank;
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          uint8_t* sa = smem + stage * Cfg::STAGE_BYTES;
          uint8_t* sb = sa + P_A_BYTES;
          const uint32_t bar = map_to_cta(smem_u32(&full_bar[stage]), 0);  // the leader's barrier
          if (kt < k4) {
            if (leader) mbar_expect_tx(&full_bar[stage], 2 * Cfg::STAGE_BYTES);
            tma_load_2d_pair(sa, &map_a, bar, kt * 128, m0);
            tma_load_2d_pair(sb, &map_b, bar, kt * 128, nb0);
            uint8_t* ssfa = sb + Cfg::B_BYTES;
            uint8_t* ssfb = ssfa + P_SFA_BYTES;
            tma_load_2d_pair(ssfa, &map_sfa, bar, 0, (int32_t)(sfa_rt * sf_tiles_k + kt * 4));
            if constexpr (OVERLAY) {   // standard layout: the tile's two 128-row scale tiles
              tma_load_2d_pair(ssfb, &map_sfb, bar, 0, (int32_t)(nt * 2 * sf_tiles_k + kt * 4));
              tma_load_2d_pair(ssfb + 2048, &map_sfb, bar, 0, (int32_t)((nt * 2 + 1) * sf_tiles_k + kt * 4));
            } else {                   // layout cut to the tile: [nt][k64][2][512 B], one box of 4 steps
              tma_load_2d_pair(ssfb, &map_sfb, bar, 0, (int32_t)(nt * sf_tiles_k + kt * 4));
            }
          } else {
            if (!lr_waited) {   // first Hs load of this CTA: k_finalize_h must be complete
              pdl_wait();
              pdl_trigger();
              lr_waited = true;
            }
            const int c0 = (kt - k4) * 64;
            if (leader) mbar_expect_tx(&full_bar[stage], 2 * (P_A_BYTES + Cfg::B_BYTES));
            tma_load_2d_pair(sa, &map_h, bar, c0, m0);
            tma_load_2d_pair(sb, &map_u, bar, c0, nb0);
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
      for (int64_t tile = pair_id; tile < n_tiles; tile += n_pairs, ++i) {
        const int a = i & 1;
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
        for (int kt = 0; kt < kiters; ++kt) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * Cfg::STAGE_BYTES);
          const uint32_t sb = sa + P_A_BYTES;
          if (kt < k4) {
            const int nk = (int)min((int64_t)4, sf_tiles_k - (int64_t)kt * 4);
            const uint32_t ssfa = sb + Cfg::B_BYTES, ssfb = ssfa + P_SFA_BYTES;
            // one descriptor per operand and stage; the K=64 steps advance the 16-byte address field by a
            // constant (the stage buffers are 1024-byte aligned, the field cannot carry)
            const uint64_t da = make_smem_desc(sa, 1024, 0, 2), db = make_smem_desc(sb, 1024, 0, 2);
            const uint64_t dfa = make_smem_desc(ssfa, 128, 0, 0), dfb = make_smem_desc(ssfb, 128, 0, 0);
            // B scales of step k: OVERLAY: 512 B at k * 512 of each of the two 2 KB scale tiles;
            // else 1 KB (both halves) at k * 1024
            auto step = [&](int k) {
              tc_cp_sf_pair(sfa_t, dfa + (uint64_t)(k * 32));
              if constexpr (OVERLAY) {
                tc_cp_sf_pair(sfb_t, dfb + (uint64_t)(k * 32));
                tc_cp_sf_pair(sfb_t + 4, dfb + (uint64_t)(128 + k * 32));
              } else {
                tc_cp_sf_pair(sfb_t, dfb + (uint64_t)(k * 64));
                tc_cp_sf_pair(sfb_t + 4, dfb + (uint64_t)(k * 64 + 32));
              }
              mma_nvf4_pair(acc_t, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc4, sfa_t, sfb_t, (kt | k) != 0);
            };
            if (nk == 4) {   // every stage but a ragged last one: straight-line code
              step(0);
              step(1);
              step(2);
              step(3);
            } else {
              for (int k = 0; k < nk; ++k) step(k);
            }
          } else {
            const int cols = min(64, p.r_t - (kt - k4) * 64);
            for (int k = 0; k < cols / 16; ++k)
              mma_bf16_pair(acc_t, make_smem_desc(sa + k * 32, 1024, 0, 2),
                            make_smem_desc(sb + k * 32, 1024, 0, 2), idesc16, 1u);
          }
          tc_commit_pair(&empty_bar[stage], 3);            // frees the slot in both CTAs
          if (kt == kiters - 1) tc_commit_pair(&acc_full[a], 3);
          if (++stage == P_STAGES) {
            stage = 0;
            phase ^= 1;
          }
        }
      }
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
    uint8_t* buf = smem + P_STAGES * Cfg::STAGE_BYTES + grp * P_OUT_BYTES;
    auto group_sync = [&]() {
      if (grp == 0) asm volatile("bar.sync 1, 128;" ::: "memory");
      else asm volatile("bar.sync 2, 128;" ::: "memory");
    };
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
#pragma unroll 1
      for (int u = grp; u < n_units; u += 2) {
        const int c0 = u * 64;
        const bool narrow = n_eff - c0 <= 32;   // a 32-column unit (only the last one of a 224-wide or ragged tile)
        uint32_t v[64];
        if (OVERLAY && u == 0) {
          // columns 0-15 of this accumulator are the next tile's scale-factor buffer: read them first and
          // hand them over, so the next tile's MMAs (other accumulator) start while the rest drains
          tmem_ld16(t0, *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
          tmem_ld_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&sf_free[a]), 0));
          tmem_ld16(t0 + 16, *reinterpret_cast<uint32_t(*)[16]>(&v[16]));
        } else {
          tmem_ld32(t0 + c0, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        }
        if (!narrow) tmem_ld32(t0 + c0 + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tmem_ld_wait();
        if (u == last_u) {   // this warp's part of the accumulator is in registers: hand it back
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
          released = true;
        }
        if (et == 0) tma_store_wait_read<0>();   // the store that last used this group's box has read it
        group_sync();
        if (!narrow) {
          uint8_t* rowp = buf + et * 128;      // 128-byte rows, 128-byte swizzle
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            uint4 o;
            o.x = pack_bf16x2(__uint_as_float(v[8 * j + 0]) * alpha, __uint_as_float(v[8 * j + 1]) * alpha);
            o.y = pack_bf16x2(__uint_as_float(v[8 * j + 2]) * alpha, __uint_as_float(v[8 * j + 3]) * alpha);
            o.z = pack_bf16x2(__uint_as_float(v[8 * j + 4]) * alpha, __uint_as_float(v[8 * j + 5]) * alpha);
            o.w = pack_bf16x2(__uint_as_float(v[8 * j + 6]) * alpha, __uint_as_float(v[8 * j + 7]) * alpha);
            *reinterpret_cast<uint4*>(rowp + ((j ^ (et & 7)) << 4)) = o;
          }
        } else {
          uint8_t* rowp = buf + et * 64;       // 64-byte rows, 64-byte swizzle
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 o;
            o.x = pack_bf16x2(__uint_as_float(v[8 * j + 0]) * alpha, __uint_as_float(v[8 * j + 1]) * alpha);
            o.y = pack_bf16x2(__uint_as_float(v[8 * j + 2]) * alpha, __uint_as_float(v[8 * j + 3]) * alpha);
            o.z = pack_bf16x2(__uint_as_float(v[8 * j + 4]) * alpha, __uint_as_float(v[8 * j + 5]) * alpha);
            o.w = pack_bf16x2(__uint_as_float(v[8 * j + 6]) * alpha, __uint_as_float(v[8 * j + 7]) * alpha);
            *reinterpret_cast<uint4*>(rowp + ((j ^ ((et >> 1) & 3)) << 4)) = o;
          }
        }
        fence_proxy_async();
        group_sync();
        if (et == 0) {
          tma_store_2d(narrow ? &map_out32 : &map_out, buf, n0 + c0, row0);
          tma_store_commit();
        }
      }
      if (!released) {   // a ragged tile with no unit for this group
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&acc_empty[a]), 0));
      }
    }
    if (et == 0) tma_store_wait<0>();
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

// Tile width for an [M x N] output with reduction length K and a rank-r_t stage, from a cost model of the
// persistent schedule: rounds of n_pairs tiles, each tile K/64 MMAs of BN/2 cycles (+ the low-rank MMAs) plus,
// for BN = 256, the ~1.9 k-cycle hand-over of the overlaid scale columns; narrower tiles move ~4 % more operand
// bytes per MAC through shared memory.
static int choose_pair_bn(int64_t M, int64_t N, int64_t K, int r_t, int ntile_avail) {
  if (g_pair_bn != 0) return g_pair_bn;
  if (ntile_avail != 224) return 256;
  const int64_t pairs = sm_count() / 2;
  auto cost = [&](int bn) {
    const double per_tile = (double)(K / 64 + (r_t + 15) / 16) * (bn / 2) * (bn == 256 ? 1.0 : 1.04) +
                            (bn == 256 ? 1900.0 : 250.0);
    const int64_t tiles_m = ceil_div(M, P_BM), full_n = N / bn, rest = N - full_n * bn;
    const int64_t full_tiles = tiles_m * full_n;
    const double rounds_full = (double)ceil_div(full_tiles, pairs);
    // the ragged column of tiles runs in the slack of the last round if there is any
    const int64_t slack = (int64_t)rounds_full * pairs - full_tiles;
    const int64_t spill = tiles_m > slack ? tiles_m - slack : 0;
    const double ragged = rest == 0 ? 0.0 : (double)ceil_div(spill, pairs) * rest / bn;
    return (rounds_full + ragged) * per_tile;
  };
  return cost(224) < cost(256) ? 224 : 256;
}

template <int BN>
static int launch_pair_bn(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                          const void* lr_a, const void* lr_b, int r_t, void* out, bool lr_late, cudaStream_t st) {
  using Cfg = PairCfg<BN>;
  CUtensorMap ma, mb, msa, msb, mh, mu, mo, mo32;
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
  rc = make_tensor_map_2d(&mo, out, 2, (uint64_t)N, (uint64_t)M, (uint64_t)N * 2, 64, 128, Swizzle::B128);
  if (rc != FT_OK) return rc;
  rc = make_tensor_map_2d(&mo32, out, 2, (uint64_t)N, (uint64_t)M, (uint64_t)N * 2, 32, 128, Swizzle::B64);
  if (rc != FT_OK) return rc;
  PairParams p;
  p.M = M;
  p.N = N;
  p.K = K;
  p.r_t = r_t;
  p.lr_late = (lr_late && r_t > 0 && pdl_enabled()) ? 1 : 0;
  p.g_dec_a = a->tensor_dec_scale;
  p.g_dec_b = b->tensor_dec_scale;
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
  FT_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_gemm4_pair<BN>, ma, mb, msa, msb, mh, mu, mo, mo32, p));
  return FT_OK;
}

// lr_late: the launch directly in front of this one is k_finalize_h of the same call (see the kernel)
int launch_gemm4_pair(const ft_qtensor* a, const ft_qtensor* b, int64_t M, int64_t N, int64_t K,
                      const void* lr_a, const void* lr_b, int r_t, void* out, bool lr_late, cudaStream_t st) {
  const int avail = (b->sf_ntile != nullptr) ? b->ntile : 0;
  int bn = choose_pair_bn(M, N, K, r_t, avail);
  if (bn != 256 && bn != avail) bn = 256;   // no scale layout for that width: the 256-wide kernel takes the standard one
  if (bn == 224) return launch_pair_bn<224>(a, b, M, N, K, lr_a, lr_b, r_t, out, lr_late, st);
  return launch_pair_bn<256>(a, b, M, N, K, lr_a, lr_b, r_t, out, lr_late, st);
}

}  // namespace ft
