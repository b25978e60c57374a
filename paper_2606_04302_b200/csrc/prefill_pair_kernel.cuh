// prefill_pair_kernel.cuh -- one CTA of a prefill CTA pair (head_dim 128, tcgen05 cta_group::2) as a device function,
// shared by prefill_umma2.cu (its own kernel) and mixed_fused.cu.  See prefill_umma2.cu for the design notes.
#pragma once
#include <cuda_fp16.h>

#include "prefill_common.cuh"

namespace lazy {
namespace {

constexpr int kStages = 4;              // K and V ring depth per CTA
constexpr int kHalfPages = kPagesPerTile / 2;

struct PairCfg {                        // head_dim 128
  static constexpr int D = 128;
  static constexpr int Q_TILE = 2 * kHalfBytes;                 // 128 rows x 128 dims
  static constexpr int K_SLAB = (kTileRows / 2) * 128;          // 64 keys x 64 dims
  static constexpr int K_STAGE = 2 * K_SLAB;                    // this CTA's 64 keys of a tile, 128 dims
  static constexpr int V_STAGE = kTileRows * 128;               // 128 keys x this CTA's 64 dims
  static constexpr int CS_ROW_BYTES = D / 2 * 8;
  static constexpr int CS_STAGE = kHalfPages * CS_ROW_BYTES;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = 2 * Q_TILE;
  static constexpr int OFF_V = OFF_K + kStages * K_STAGE;
  static constexpr int OFF_CS = OFF_V + kStages * V_STAGE;
  static constexpr int OFF_BAR = OFF_CS + kStages * CS_STAGE;
  static constexpr int NUM_BARS = 48;
  static constexpr int OFF_TMEM = OFF_BAR + NUM_BARS * 8;
  static constexpr int OFF_SIGN = OFF_TMEM + 16;                // ring of 8 tiles x 8 pages (sign / page start)
  static constexpr int OFF_SC = OFF_SIGN + 8 * kPagesPerTile * 4;   // FP8 pages: [stage][4 K pages | 8 V pages][16] row scales
  static constexpr int SC_STAGE = (kHalfPages + kPagesPerTile) * 64;
  static constexpr int SMEM_BYTES = OFF_SC + kStages * SC_STAGE + 1024;   // + alignment slack
};

// barrier indices.  (L): only the leader CTA's copy is used, threads of both CTAs arrive on it.
// t = Q tile of the CTA (0, 1); h = half of a KV tile's keys (see "key halves" in the kernel).
enum : int {
  P_QFULL = 0,      // +t     TMA -> softmax WG t                                   (local)
  P_QREADY = 2,     // +t     softmax WG t of both CTAs (8 warps) -> MMA            (L)
  P_KFULL = 4,      // +s     TMA (K boxes + table rows) -> rotate WG               (local)
  P_KREADY = 8,     // +s     rotate WGs of both CTAs (8 warps) -> MMA              (L)
  P_KEMPTY = 12,    // +s     MMA commit (multicast) -> TMA of both CTAs
  P_VFULL = 16,     // +s     V boxes of both CTAs -> MMA                           (L)
  P_VEMPTY = 20,    // +s     MMA commit (multicast) -> TMA of both CTAs
  P_VLASTFULL = 24, //        last tile's V boxes -> this CTA's fixer               (local, one shot)
  P_VFIXED = 25,    //        fixers of both CTAs -> MMA                            (L, last tile only)
  P_SFULL = 26,     // +2t+h  MMA commit (multicast) -> softmax WG t: S half h is in TMEM
  P_PREADY = 30,    // +2t+h  softmax WG t of both CTAs -> MMA: P half h is in TMEM (L)
  P_PVDONE = 34,    // +2t+h  MMA commit (multicast) -> softmax WG t: O_t += P_h V has completed (slow path only)
  P_OFULL = 38,     // +t     MMA commit (multicast) -> softmax WG t (epilogue)
  P_VLOCAL = 40,    // +s     FP8 pages: this CTA's V boxes (codes + scales) -> its rotate WG (local)
  P_VREADY = 44,    // +s     FP8 pages: rotate WGs of both CTAs (8 warps) -> MMA: V tile dequantised     (L)
};

// FP8 pages: 8 E4M3 codes (two words) -> 8 fp32 values, exact
__device__ __forceinline__ void pair_e4m3x8_to_f32(uint2 v, float2 (&x)[4]) {
  const uint32_t h[4] = {ptx::e4m3x2_lo_to_f16x2(v.x), ptx::e4m3x2_hi_to_f16x2(v.x), ptx::e4m3x2_lo_to_f16x2(v.y),
                         ptx::e4m3x2_hi_to_f16x2(v.y)};
#pragma unroll
  for (int w = 0; w < 4; ++w) x[w] = __half22float2(*reinterpret_cast<const __half2*>(&h[w]));
}
__device__ __forceinline__ uint2 pair_lds64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}

// byte offset of 16-byte chunk `ci` of row `row` (0..63) inside a K half-stage (two 64-row slabs, 128B swizzle)
__device__ __forceinline__ uint32_t kchunk_off(int row, int ci) {
  return (ci >> 3) * PairCfg::K_SLAB + row * 128 + (((ci & 7) ^ (row & 7)) << 4);
}

// The body of one CTA of a pair; `pair` is the pair's work-item index.  prefill_pair_kernel maps it to blockIdx.x / 2;
// the fused mixed-step kernel (mixed_fused.cu) runs the same body on the CTAs behind its decode CTAs.
// F8: LAZY_KV_FP8_E4M3 pages.  As in prefill_umma.cu, a page's codes land (plain rows) at the start of the page's own
// region of the bf16 stage and the rotate warpgroup writes the bf16 tile over them: this CTA's 4 pages of K dequantised
// and rotated, its 64-column slab of all 8 pages of V dequantised (rows past the sequence cleared -- there is no tail
// fixer).  V boxes report to a LOCAL barrier; the leader's MMA warp waits for VREADY (8 rotate warps) instead of VFULL.
template <int KM, bool F8 = false>
__device__ __forceinline__ void prefill_pair_cta(const CUtensorMap& tmap_q, const CUtensorMap& tmap_k,
                                                 const CUtensorMap& tmap_v, const PrefillArgs& a, const int pair,
                                                 unsigned char* smem_raw) {
  using C = PairCfg;
  constexpr int D = C::D;
  constexpr bool kNoRotate = KM == LAZY_K_ABSOLUTE || KM == kKmAlibi;   // the K tile goes to the MMA as it landed
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t smem_base = ptx::smem_u32(smem);
  const uint32_t sQ = smem_base + C::OFF_Q, sK = smem_base + C::OFF_K, sV = smem_base + C::OFF_V;
  const uint32_t sCS = smem_base + C::OFF_CS;
  const uint32_t bars = smem_base + C::OFF_BAR;
  auto bar = [&](int idx) { return bars + 8u * idx; };                  // this CTA's copy
  auto lbar = [&](int idx) { return ptx::mapa(bars + 8u * idx, 0); };   // the leader's copy (cluster address)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_TMEM);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int rank = (int)ptx::cluster_ctarank();
  const Shape sh = a.sh;
  const int group = sh.group, TPT = a.tokens_per_tile, TPC = 2 * TPT;

  // ---- work item of the PAIR: (request, kv head, block of 4*TPT query tokens); this CTA takes half of the block ----
  // (the blocks of one (request, kv head) stay adjacent: they share K/V through the L2; the last block, which sees the
  // most keys under the causal mask, goes first).  Every early exit below is taken by both CTAs of the pair.
  const int pblk = a.mblocks - 1 - pair % a.mblocks;
  const int hk = (pair / a.mblocks) % sh.Hkv;
  const int r = pair / (a.mblocks * sh.Hkv);
  const int q_begin = a.cu_q_lens[r];
  const int n_q = a.cu_q_lens[r + 1] - q_begin;
  const int L = a.seq_lens[r];
  const int i0p = pblk * 2 * TPC;
  if (i0p >= n_q) return;
  const int i0 = i0p + rank * TPC;                  // may be >= n_q: this CTA then only serves its K / V halves
  const int i_end = min(i0 + TPC, n_q);
  if (L <= 0) {                                     // degenerate: rows of an empty sequence are zeros
    const int n = max(0, i_end - i0) * group * (D / 8);
    for (int x = tid; x < n; x += kPrefillThreads) {
      int ch = x % (D / 8), g = (x / (D / 8)) % group, i = i0 + x / (D / 8 * group);
      reinterpret_cast<uint4*>(a.out + ((size_t)(q_begin + i) * sh.Hq + hk * group + g) * D)[ch] = make_uint4(0, 0, 0, 0);
    }
    return;
  }
  const int kv_len = max(1, min(L, L - n_q + min(i0p + 2 * TPC, n_q)));   // keys visible to the pair's last query row
  const int n_kv = (kv_len + kTileRows - 1) / kTileRows;
  const int num_pages = (L + kPageSize - 1) / kPageSize;
  const int* bt = a.block_table + (size_t)r * sh.table_stride;
  const int* ppos = a.page_pos + (size_t)r * sh.table_stride;

  // barrier x is initialised by thread x of warp 0 (one thread doing all 48 took ~0.5 us of every item's prologue);
  // arrival counts: 8 = the four warps of a warpgroup in both CTAs, 2 = the two fixers, 1 = a TMA / commit arrival
  if (warp == 0) {
    for (int x = lane; x < C::NUM_BARS; x += 32) {
      const bool eight = (x >= P_QREADY && x < P_QREADY + 2) || (x >= P_KREADY && x < P_KREADY + kStages) ||
                         (x >= P_PREADY && x < P_PREADY + 4) || (x >= P_VREADY && x < P_VREADY + kStages);
      ptx::mbar_init(bar(x), eight ? 8 : x == P_VFIXED ? 2 : 1);
    }
    ptx::fence_mbar_init();
  }
  if (warp == 13) {
    ptx::tmem_alloc_pair<512>(ptx::smem_u32(tmem_slot));
    ptx::tmem_relinquish_pair();
  }
  ptx::tc_fence_before();
  ptx::cluster_sync();                               // barriers of both CTAs initialised before any remote arrive
  ptx::tc_fence_after();
  const uint32_t tbase = *tmem_slot;

  if (warp >= 12) {
    ptx::setmaxnreg_dec<kRegsMisc>();
    if (warp == 12) {
      // ================================ TMA producer ========================================================
      if (lane == 0) { ptx::prefetch_tmap(&tmap_q); ptx::prefetch_tmap(&tmap_k); ptx::prefetch_tmap(&tmap_v); }
      if (lane < 2) {
        const int t = lane;
        ptx::mbar_arrive_expect_tx(bar(P_QFULL + t), 2 * group * TPT * 128);
#pragma unroll
        for (int h = 0; h < 2; ++h)
          tma_load_4d(sQ + t * C::Q_TILE + h * kHalfBytes, &tmap_q, bar(P_QFULL + t), h * 64, 0, hk,
                      q_begin + i0 + t * TPT);
      }
      // lanes 0-7: K box (slab, page 4*rank + pgl) and, for slab 0, the page's table row; lanes 8-15: V box of page
      // pg (this CTA's 64-column slab).  Table entries travel through a 3-deep shift register (tile j+2 -> j+1 -> j).
      const bool is_k = lane < 8, is_v = lane >= 8 && lane < 16;
      const int half = (lane >> 2) & 1, pgl = lane & 3, pg = is_k ? kHalfPages * rank + pgl : (lane & 7);
      auto entry = [&](int tile, int& page, int& pos) {
        const int idx = tile * kPagesPerTile + pg;
        page = 0; pos = 0;
        if (lane < 16 && tile < n_kv && idx < num_pages) {
          page = bt[idx];
          pos = ppos[idx];
          if (KM == LAZY_K_STORED_POS) pos -= a.stored_pos[page];
        }
      };
      int page_next, pos_next, page_n2, pos_n2;
      entry(0, page_next, pos_next);
      entry(1, page_n2, pos_n2);
      int* s_sign = reinterpret_cast<int*>(smem + C::OFF_SIGN);
      for (int j = 0; j < n_kv; ++j) {
        const int s = j & (kStages - 1), ph = (j / kStages) & 1;
        const int page = page_next;
        const int p0 = pos_next < 0 ? -pos_next : pos_next;      // negative only for LAZY_K_STORED_POS
        const int p0_sign = pos_next < 0 ? -1 : 1;
        page_next = page_n2; pos_next = pos_n2;
        entry(j + 2, page_n2, pos_n2);
        const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);     // pages of the tile that exist
        const int npk = max(0, min(kHalfPages, npv - kHalfPages * rank));      // ... of this CTA's K half
        const int row0 = (page * sh.Hkv + hk) * kPageSize;
        ptx::mbar_wait_sleep(bar(P_KEMPTY + s), ph ^ 1);
        if (KM == LAZY_K_STORED_POS && is_v) s_sign[(j & 7) * kPagesPerTile + pg] = p0_sign;
        if (KM == kKmAlibi && is_v) s_sign[(j & 7) * kPagesPerTile + pg] = p0;
        __syncwarp();
        const uint32_t sSC = smem_base + C::OFF_SC + s * C::SC_STAGE;
        if (lane == 0)
          ptx::mbar_arrive_expect_tx(bar(P_KFULL + s), npk * ((F8 ? kPageSize * 128 + 64 : 2 * kPageSize * 128) +
                                                              (kNoRotate ? 0 : C::CS_ROW_BYTES)));
        __syncwarp();
        if (is_k && pgl < npk) {
          if (!F8) ptx::tma_load_2d(sK + s * C::K_STAGE + half * C::K_SLAB + pgl * (kPageSize * 128), &tmap_k,
                                    bar(P_KFULL + s), half * 64, row0);
          if (F8 && half == 0) {                    // one box of 16 rows x 128 code bytes, and the rows' scales
            ptx::tma_load_2d(sK + s * C::K_STAGE + pgl * (kPageSize * 128), &tmap_k, bar(P_KFULL + s), 0, row0);
            ptx::bulk_load_1d(sSC + pgl * 64, a.k_scale + row0, 64, bar(P_KFULL + s));
          }
          if (half == 0 && !kNoRotate)
            ptx::bulk_load_1d(sCS + s * C::CS_STAGE + pgl * C::CS_ROW_BYTES, a.cs + (size_t)p0 * (D / 2),
                              C::CS_ROW_BYTES, bar(P_KFULL + s));
        }
        ptx::mbar_wait_sleep(bar(P_VEMPTY + s), ph ^ 1);
        const uint32_t vdst = sV + s * C::V_STAGE + (lane & 7) * (kPageSize * 128);
        if (F8) {
          // this CTA's 64 code bytes of each row of every page of the tile + the rows' scales, to the local barrier
          if (lane == 0) ptx::mbar_arrive_expect_tx(bar(P_VLOCAL + s), npv * (kPageSize * 64 + 64));
          __syncwarp();
          if (is_v && (lane & 7) < npv) {
            ptx::tma_load_2d(vdst, &tmap_v, bar(P_VLOCAL + s), rank * 64, row0);
            ptx::bulk_load_1d(sSC + (kHalfPages + (lane & 7)) * 64, a.v_scale + row0, 64, bar(P_VLOCAL + s));
          }
        } else if (j < n_kv - 1) {
          // bytes of both CTAs are counted on the leader's barrier; the leader announces them (a peer box that lands
          // first only drives the pending-byte count negative for a moment)
          if (lane == 0 && rank == 0) ptx::mbar_arrive_expect_tx(bar(P_VFULL + s), 2 * npv * kPageSize * 128);
          __syncwarp();
          if (is_v && (lane & 7) < npv) ptx::tma_load_2d_pair(vdst, &tmap_v, lbar(P_VFULL + s), rank * 64, row0);
        } else {
          // last tile: the boxes report to this CTA's own one-shot barrier, the fixer cleans the tail rows and then
          // tells the leader
          if (lane == 0) ptx::mbar_arrive_expect_tx(bar(P_VLASTFULL), npv * kPageSize * 128);
          __syncwarp();
          if (is_v && (lane & 7) < npv) ptx::tma_load_2d(vdst, &tmap_v, bar(P_VLASTFULL), rank * 64, row0);
        }
      }
    } else if (warp == 13) {
      // ================================ MMA issuer (leader CTA only) ========================================
      // The whole warp walks the loop convergently and ONE elected lane issues, so that every operand of
      // tcgen05.mma / tcgen05.commit is warp-uniform and lives in uniform registers.
      //
      // Key halves.  S_t = Q_t Khat^T of a 128-key tile is issued as TWO MMAs of N = 64: half h takes rows 32h..32h+31
      // of each CTA's 64-key K stage, i.e. keys {32h..32h+31} u {64+32h..64+32h+31} of the tile, into columns
      // 64h..64h+63 of S_t (P_h is packed over the first 32 of them).  O_t += P_h V follows with the matching V rows.
      // What this buys: the columns of half h are free again as soon as PV_h has run, so QK_h of the NEXT tile is
      // issued right behind it, while the softmax warpgroup is still busy with the other half.  S is therefore
      // (nearly) always waiting when a warpgroup comes back for it, and the softmax -> PV -> QK -> softmax chain that
      // paced the kernel (with S_t of N = 128 aliased by P_t it could not be cut) is gone.  The price is the Q operand
      // read twice per tile (N = 64 MMAs are shared-memory-bound: ~40 instead of 32 cycles per k-step).
      if (rank == 0) {
        constexpr uint32_t IDESC_QK = ptx::umma_idesc_bf16(256, 64, 0, 0);
        constexpr uint32_t IDESC_PV = ptx::umma_idesc_bf16(256, D, 0, 1);       // B = V is MN-major
        const uint32_t tb = __shfl_sync(0xffffffffu, tbase, 0);
        const int nkv = __shfl_sync(0xffffffffu, n_kv, 0);
        const bool leader = ptx::elect_one();
        auto qk = [&](int t, int s, int h) {
          if (leader) {
            const uint32_t qa = sQ + t * C::Q_TILE, ka = sK + s * C::K_STAGE + h * (32 * 128);
#pragma unroll
            for (int k = 0; k < D / 16; ++k)
              ptx::umma_ss_pair(tb + t * 128 + h * 64,
                                ptx::umma_desc_sw128(qa + (k >> 2) * kHalfBytes + (k & 3) * 32, 0, 1024),
                                ptx::umma_desc_sw128(ka + (k >> 2) * C::K_SLAB + (k & 3) * 32, 0, 1024), IDESC_QK, k > 0);
          }
        };
        auto pv = [&](int t, int s, int h, uint32_t acc) {
          if (leader) {
            const uint32_t va = sV + s * C::V_STAGE + h * (32 * 128);
#pragma unroll
            for (int k = 0; k < 4; ++k)                       // keys 32h + 16k (k < 2), 64 + 32h + 16(k-2) (k >= 2)
              ptx::umma_ts_pair(tb + 256 + t * 128, tb + t * 128 + h * 64 + k * 8,
                                ptx::umma_desc_sw128(va + ((k & 1) * 16 + (k >> 1) * 64) * 128, kHalfBytes, 1024), IDESC_PV,
                                acc | (uint32_t)(k > 0));
          }
        };
        auto commit = [&](int idx) { if (leader) ptx::umma_commit_pair(bar(idx)); };
        ptx::mbar_wait_acquire_cluster(bar(P_KREADY + 0), 0);
        for (int t = 0; t < 2; ++t) {
          ptx::mbar_wait_acquire_cluster(bar(P_QREADY + t), 0);
          ptx::tc_fence_after();
          for (int h = 0; h < 2; ++h) { qk(t, 0, h); commit(P_SFULL + 2 * t + h); }
        }
        commit(P_KEMPTY + 0);
        // Hand-offs are taken in the fixed order (tile 0, half 0), (tile 1, half 0), (tile 0, half 1), (tile 1, half 1):
        // the two Q tiles stay in lockstep, so the K / V rings -- which only turn when BOTH tiles have consumed a
        // stage -- keep flowing.  (Serving whichever tile was ready first let one softmax warpgroup run a full ring
        // ahead of the other; the kernel then alternated between bursts of one tile and refill latencies: 668 TFLOP/s.)
        for (int j = 0; j < nkv; ++j) {
          const int s = j & (kStages - 1), sn = (j + 1) & (kStages - 1);
          if (F8) ptx::mbar_wait_acquire_cluster(bar(P_VREADY + s), (j / kStages) & 1);
          else if (j == nkv - 1) ptx::mbar_wait_acquire_cluster(bar(P_VFIXED), 0);
          else ptx::mbar_wait(bar(P_VFULL + s), (j / kStages) & 1);
#pragma unroll
          for (int h = 0; h < 2; ++h) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
              ptx::mbar_wait_tmem(bar(P_PREADY + 2 * t + h), j & 1);
              ptx::tc_fence_after();
              pv(t, s, h, (uint32_t)(j > 0 || h > 0));
              commit(P_PVDONE + 2 * t + h);
              if (h == 1 && t == 1) commit(P_VEMPTY + s);
              if (j + 1 < nkv) {
                if (h == 0 && t == 0) {
                  ptx::mbar_wait_acquire_cluster(bar(P_KREADY + sn), ((j + 1) / kStages) & 1);
                  ptx::tc_fence_after();
                }
                qk(t, sn, h);
                commit(P_SFULL + 2 * t + h);
                if (h == 1 && t == 1) commit(P_KEMPTY + sn);
              } else if (h == 1) {
                commit(P_OFULL + t);
              }
            }
          }
        }
        __syncwarp();
      }
    } else if (warp == 14 && !F8) {
      // ================================ V tail fixer ========================================================
      // zeroes the rows >= seq_len of this CTA's slab of the last V tile, so that poisoned bytes never reach PV
      const int jl = n_kv - 1;
      ptx::mbar_wait_sleep(bar(P_VLASTFULL), 0);
      const int rows_valid = min(kTileRows, L - jl * kTileRows);
      if (rows_valid < kTileRows) {
        const uint32_t vb = sV + (jl & (kStages - 1)) * C::V_STAGE + rows_valid * 128;
        for (int x = lane; x < (kTileRows - rows_valid) * 8; x += 32) ptx::sts128(vb + x * 16, make_uint4(0, 0, 0, 0));
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster_release(lbar(P_VFIXED));
    }
  } else if (warp >= 8) {
    // ================================ K-rotate warpgroup ======================================================
    // this CTA's 64 keys of every tile.  thread = (page, token group tg, chunk pair c = 8 rotation pairs): it takes the
    // tokens tg, tg+4, tg+8, tg+12 of the page.  The page's table row w = e^{i p0 theta_j} is read once, composed with
    // e^{i tg theta_j}, and the tokens are walked with z <- z * e^{i 4 theta_j} (at most 3 fp32 complex products from
    // a table value).  Lane -> (c, tg) is chosen so that the 8 lanes of a quarter warp (one shared-memory wavefront of
    // a 16-byte access) hold the four c of one parity x two ADJACENT tokens: their table chunks are 4 distinct
    // 16-byte words (broadcast across the two tokens; chunk pairs c and c+1 would collide, they sit 256 B apart), and
    // their K chunks, swizzled by (row & 7), fall into disjoint bank groups because adjacent rows differ in parity.
    // (FP8 pages: the warpgroup holds a page's codes of both tiles: 2*128*168 + 128*136 + 128*40 = 65536)
    if (F8) ptx::setmaxnreg_inc<136>();
    else ptx::setmaxnreg_dec<kRegsRotate>();
    constexpr int TOK = 4;
    const int wtid = tid - 256;
    const int i = wtid >> 5;                        // page of this CTA's half tile
    const int c = 2 * (lane & 3) + ((lane >> 3) & 1);
    const int tg = ((lane >> 2) & 1) + 2 * (lane >> 4);
    float2 u0c[4], u0s[4], u1c[4], u1s[4];          // e^{i tg theta_j}, e^{i 4 theta_j} for this thread's 8 pairs
    if (KM == LAZY_K_UNROTATED) {
      const float4* r0 = reinterpret_cast<const float4*>(a.cs + (size_t)tg * (D / 2));
      const float4* r1 = reinterpret_cast<const float4*>(a.cs + (size_t)4 * (D / 2));
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const float4 v0 = __ldg(r0 + cs_f4_index<D>(c, x)), v1 = __ldg(r1 + cs_f4_index<D>(c, x));
        u0c[x] = make_float2(v0.x, v0.y); u0s[x] = make_float2(v0.z, v0.w);
        u1c[x] = make_float2(v1.x, v1.y); u1s[x] = make_float2(v1.z, v1.w);
      }
    }
    const int* s_sign = reinterpret_cast<const int*>(smem + C::OFF_SIGN);
    for (int j = 0; j < n_kv; ++j) {
      const int s = j & (kStages - 1);
      const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
      const int npk = max(0, min(kHalfPages, npv - kHalfPages * rank));
      const uint32_t kb = sK + s * C::K_STAGE;
      const uint32_t cb = sCS + s * C::CS_STAGE;
      ptx::mbar_wait(bar(P_KFULL + s), (j / kStages) & 1);
      if (F8) {
        // ---- K: this CTA's 4 pages; thread = (page i, tokens tg + 4tt, pairs 8c..8c+7); a warp serves one page
        const uint32_t sc = smem_base + C::OFF_SC + s * C::SC_STAGE;
        const uint32_t land = kb + i * (kPageSize * 128) + tg * 128 + 8 * c;     // codes of (page i, token tg, dims 8c..)
        uint2 ra[TOK], rb[TOK];
        float scl[TOK];
        float2 zc[4], zs[4];
        if (i < npk) {
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint4 v = ptx::lds128(cb + i * C::CS_ROW_BYTES + 16 * cs_f4_index<D>(c, x));
            const float2 wc = make_float2(f32(v.x), f32(v.y)), ws = make_float2(f32(v.z), f32(v.w));
            zc[x] = __ffma2_rn(neg2(ws), u0s[x], __fmul2_rn(wc, u0c[x]));
            zs[x] = __ffma2_rn(wc, u0s[x], __fmul2_rn(ws, u0c[x]));
          }
#pragma unroll
          for (int tt = 0; tt < TOK; ++tt) {
            ra[tt] = pair_lds64(land + 4 * tt * 128);
            rb[tt] = pair_lds64(land + 4 * tt * 128 + 64);
            scl[tt] = __int_as_float(ptx::lds32(sc + i * 64 + (tg + 4 * tt) * 4));
          }
        }
        __syncwarp();                               // the page's codes are in registers: overwrite them
        if (i < npk) {
          const int row0 = i * kPageSize + tg;
#pragma unroll
          for (int tt = 0; tt < TOK; ++tt) {
            float2 x1[4], x2[4];
            pair_e4m3x8_to_f32(ra[tt], x1);
            pair_e4m3x8_to_f32(rb[tt], x2);
            const float2 sk2 = make_float2(scl[tt], scl[tt]);
            uint4 va, vb;
            uint32_t* aw = reinterpret_cast<uint32_t*>(&va);
            uint32_t* bw = reinterpret_cast<uint32_t*>(&vb);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
              const float2 cc = __fmul2_rn(zc[w], sk2), ss = __fmul2_rn(zs[w], sk2);
              const float2 y1 = __ffma2_rn(neg2(x2[w]), ss, __fmul2_rn(x1[w], cc));
              const float2 y2 = __ffma2_rn(x2[w], cc, __fmul2_rn(x1[w], ss));
              aw[w] = ptx::pack_bf16(y1.x, y1.y);
              bw[w] = ptx::pack_bf16(y2.x, y2.y);
            }
            ptx::sts128(kb + kchunk_off(row0 + 4 * tt, c), va);
            ptx::sts128(kb + kchunk_off(row0 + 4 * tt, c + 8), vb);
            if (tt + 1 < TOK) {
#pragma unroll
              for (int x = 0; x < 4; ++x) {
                const float2 wc = zc[x], ws = zs[x];
                zc[x] = __ffma2_rn(neg2(ws), u1s[x], __fmul2_rn(wc, u1c[x]));
                zs[x] = __ffma2_rn(wc, u1s[x], __fmul2_rn(ws, u1c[x]));
              }
            }
          }
        }
        ptx::fence_proxy_async();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_release(lbar(P_KREADY + s));
        // ---- V: this CTA's 64-column slab of all 8 pages; thread = (page vp, token vt): 64 codes -> one 128-byte row
        const int vp = wtid >> 4, vt = wtid & 15;
        const int vrow = vp * kPageSize + vt;
        const uint32_t vs_ = sV + s * C::V_STAGE;
        ptx::mbar_wait(bar(P_VLOCAL + s), (j / kStages) & 1);
        const bool live = vp < npv && j * kTileRows + vrow < L;
        uint4 cv[4];
        float sv = 0.f;
        if (live) {
#pragma unroll
          for (int x = 0; x < 4; ++x) cv[x] = ptx::lds128(vs_ + vp * (kPageSize * 128) + vt * 64 + 16 * x);
          sv = __int_as_float(ptx::lds32(sc + (kHalfPages + vp) * 64 + vt * 4));
        }
        __syncwarp();
        if (vp < npv || j == n_kv - 1) {            // pages that do not exist are cleared on the last tile only
          const float2 sv2 = make_float2(sv, sv);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            uint4 o0 = make_uint4(0, 0, 0, 0), o1 = make_uint4(0, 0, 0, 0);
            if (live) {
              float2 f0[4], f1[4];
              pair_e4m3x8_to_f32(make_uint2(cv[x].x, cv[x].y), f0);
              pair_e4m3x8_to_f32(make_uint2(cv[x].z, cv[x].w), f1);
              uint32_t* w0 = reinterpret_cast<uint32_t*>(&o0);
              uint32_t* w1 = reinterpret_cast<uint32_t*>(&o1);
#pragma unroll
              for (int w = 0; w < 4; ++w) {
                const float2 y0 = __fmul2_rn(f0[w], sv2), y1 = __fmul2_rn(f1[w], sv2);
                w0[w] = ptx::pack_bf16(y0.x, y0.y);
                w1[w] = ptx::pack_bf16(y1.x, y1.y);
              }
            }
            ptx::sts128(vs_ + vrow * 128 + (((2 * x) ^ (vrow & 7)) << 4), o0);
            ptx::sts128(vs_ + vrow * 128 + (((2 * x + 1) ^ (vrow & 7)) << 4), o1);
          }
        }
        ptx::fence_proxy_async();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_release(lbar(P_VREADY + s));
        continue;
      }
      if (!kNoRotate && i < npk) {
        float2 zc[4], zs[4];                        // e^{i (p0+t) theta_j}, or e^{i Delta theta_j} of the page
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          const uint4 v = ptx::lds128(cb + i * C::CS_ROW_BYTES + 16 * cs_f4_index<D>(c, x));
          zc[x] = make_float2(f32(v.x), f32(v.y));
          zs[x] = make_float2(f32(v.z), f32(v.w));
        }
        if (KM == LAZY_K_UNROTATED) {               // first token of the thread: z = w * u0
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const float2 wc = zc[x], ws = zs[x];
            zc[x] = __ffma2_rn(neg2(ws), u0s[x], __fmul2_rn(wc, u0c[x]));
            zs[x] = __ffma2_rn(wc, u0s[x], __fmul2_rn(ws, u0c[x]));
          }
        } else {                                    // one relative rotation for the whole page (may be negative)
          const float sgn = (float)s_sign[(j & 7) * kPagesPerTile + kHalfPages * rank + i];
#pragma unroll
          for (int x = 0; x < 4; ++x) zs[x] = __fmul2_rn(zs[x], make_float2(sgn, sgn));
        }
        const int row0 = i * kPageSize + tg;
        uint4 va[TOK], vb[TOK];
#pragma unroll
        for (int tt = 0; tt < TOK; ++tt) {
          va[tt] = ptx::lds128(kb + kchunk_off(row0 + 4 * tt, c));
          vb[tt] = ptx::lds128(kb + kchunk_off(row0 + 4 * tt, c + 8));
        }
#pragma unroll
        for (int tt = 0; tt < TOK; ++tt) {
          rotate8_packed(va[tt], vb[tt], zc, zs);
          ptx::sts128(kb + kchunk_off(row0 + 4 * tt, c), va[tt]);
          ptx::sts128(kb + kchunk_off(row0 + 4 * tt, c + 8), vb[tt]);
          if (KM == LAZY_K_UNROTATED && tt + 1 < TOK) {          // next token (4 further): z <- z * e^{i 4 theta_j}
#pragma unroll
            for (int x = 0; x < 4; ++x) {
              const float2 wc = zc[x], ws = zs[x];
              zc[x] = __ffma2_rn(neg2(ws), u1s[x], __fmul2_rn(wc, u1c[x]));
              zs[x] = __ffma2_rn(wc, u1s[x], __fmul2_rn(ws, u1c[x]));
            }
          }
        }
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster_release(lbar(P_KREADY + s));
    }
  } else {
    // ================================ softmax warpgroups ======================================================
    ptx::setmaxnreg_inc<F8 ? 168 : kRegsSoftmax>();
    const int t = warp >> 2;
    const int row = tid - t * 128;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tbase + t * 128 + lane_base, tO = tbase + 256 + t * 128 + lane_base;
    const int tokl = row / group, g = row - tokl * group;
    const int i = i0 + t * TPT + tokl;
    const int sq = L - n_q + i;
    const bool valid = tokl < TPT && i < n_q && sq >= 0;
    const int lim_row = max(0, L - n_q + min(i, n_q - 1));
    const int lim_min = max(0, L - n_q + min(i0 + t * TPT, n_q - 1));

    // ---- Q tile: rotate by the query position, fold in log2(e)/sqrt(D), in place ----------------------------
    // the row's cos/sin (one table row: D/4 16-byte chunks) is pulled into the L2 BEFORE waiting for the Q tile and read
    // chunk by chunk behind the wait.  (Holding the whole row in 128 registers across the wait -- all loads in flight
    // at once -- made ptxas spill it to local memory: cfg 5's short items ran 10 % slower, 85.3 -> 76.7 us.)
    const float4* csp = reinterpret_cast<const float4*>(a.cs);
    if (valid && KM != kKmAlibi) {
      const int pos = ppos[sq / kPageSize] + sq % kPageSize;
      csp = reinterpret_cast<const float4*>(a.cs + (size_t)pos * (D / 2));
      if (g == 0) {
#pragma unroll
        for (int x = 0; x < D / 4; x += 8) asm volatile("prefetch.global.L2 [%0];" ::"l"(csp + x));
      }
    }
    ptx::mbar_wait(bar(P_QFULL + t), 0);
    {
      const uint32_t qb = sQ + t * C::Q_TILE;
      if (valid) {
        uint4 src[D / 8];                           // LAZY_ROPE_INTERLEAVED: the whole row first (in-place hazard)
        if (a.q_interleaved) {
#pragma unroll
          for (int c = 0; c < D / 8; ++c) src[c] = ptx::lds128(qb + chunk_off(row, c));
        }
#pragma unroll
        for (int c = 0; c < D / 16; ++c) {
          float co[8], si[8];
          if (KM == kKmAlibi) {                     // no rotation: scale only
#pragma unroll
            for (int e = 0; e < 8; ++e) { co[e] = sh.scale_log2; si[e] = 0.f; }
          } else {
#pragma unroll
            for (int x = 0; x < 4; ++x) {
              const float4 v = __ldg(csp + cs_f4_index<D>(c, x));
              co[2 * x] = v.x * sh.scale_log2; co[2 * x + 1] = v.y * sh.scale_log2;
              si[2 * x] = v.z * sh.scale_log2; si[2 * x + 1] = v.w * sh.scale_log2;
            }
          }
          const uint32_t pa = qb + chunk_off(row, c), pb = qb + chunk_off(row, c + D / 16);
          uint4 va, vb;
          if (!a.q_interleaved) {
            va = ptx::lds128(pa); vb = ptx::lds128(pb);
          } else {                                  // model words (x1_j, x2_j) -> x1 chunk and x2 chunk of pairs 8c..8c+7
            const uint4 s0 = src[2 * c], s1 = src[2 * c + 1];
            va.x = __byte_perm(s0.x, s0.y, 0x5410u); va.y = __byte_perm(s0.z, s0.w, 0x5410u);
            va.z = __byte_perm(s1.x, s1.y, 0x5410u); va.w = __byte_perm(s1.z, s1.w, 0x5410u);
            vb.x = __byte_perm(s0.x, s0.y, 0x7632u); vb.y = __byte_perm(s0.z, s0.w, 0x7632u);
            vb.z = __byte_perm(s1.x, s1.y, 0x7632u); vb.w = __byte_perm(s1.z, s1.w, 0x7632u);
          }
          rotate8(va, vb, co, si);
          ptx::sts128(pa, va);
          ptx::sts128(pb, vb);
        }
      } else {
#pragma unroll
        for (int c = 0; c < D / 8; ++c) ptx::sts128(qb + chunk_off(row, c), make_uint4(0, 0, 0, 0));
      }
    }
    ptx::fence_proxy_async();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive_cluster_release(lbar(P_QREADY + t));

    float alibi_slope = 0.f;                                   // kKmAlibi: this row's slope (log2 units), position
    int alibi_pos_q = 0;
    float2 alibi_d2[kPageSize / 2];                            // slope * t for the in-page offsets, as pairs
    if (KM == kKmAlibi && valid) {
      alibi_slope = a.alibi[hk * group + g];
      alibi_pos_q = ppos[sq / kPageSize] + sq % kPageSize;
    }
    if (KM == kKmAlibi) {
#pragma unroll
      for (int x = 0; x < kPageSize / 2; ++x)
        alibi_d2[x] = make_float2(alibi_slope * (float)(2 * x), alibi_slope * (float)(2 * x + 1));
    }
    // Online softmax with optimistic exponentials (see prefill_umma.cu), one key half at a time: columns c of half h
    // are the keys key(c) = 32h + c (c < 32), 64 + 32h + (c - 32) (c >= 32) of the tile.  The two warpgroups run free.
    constexpr float kDanger = 20.f;
    float m_used = -INFINITY, l_run = 0.f;
    for (int j = 0; j < n_kv; ++j) {
      const bool edge = j * kTileRows + kTileRows - 1 > lim_min;   // tile touches the causal edge / the tail
      const int lim_col = lim_row - j * kTileRows;            // key of the tile visible iff key <= lim_col
      const int* pstart = reinterpret_cast<const int*>(smem + C::OFF_SIGN) + (j & 7) * kPagesPerTile;
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
        uint32_t sreg[64];                                    // this row of S half (fp32 bits); P is packed over it
        const uint32_t tSh = tS + 64 * hf;
        ptx::mbar_wait(bar(P_SFULL + 2 * t + hf), j & 1);
        ptx::tc_fence_after();
        ptx::tmem_ld32(tSh, sreg);
        ptx::tmem_ld32(tSh + 32, sreg + 32);
        float abase[4];                                       // kKmAlibi: slope * (page start - m) of the half's 4 pages
        if (KM == kKmAlibi) {
#pragma unroll
          for (int pg = 0; pg < 4; ++pg)
            abase[pg] = alibi_slope * (float)(pstart[2 * hf + (pg & 1) + 4 * (pg >> 1)] - alibi_pos_q);
        }
        ptx::tmem_wait_ld();
        if (KM == kKmAlibi) {
          // S += slope * (n - m), n = page start + t: the in-page part slope * t goes to the elements here, the
          // per-page part abase[] into the maxima and into the constant of the exponential
#pragma unroll
          for (int x = 0; x < 64; x += 2) {
            const float2 v = __fadd2_rn(make_float2(f32(sreg[x]), f32(sreg[x + 1])), alibi_d2[(x & 15) >> 1]);
            sreg[x] = __float_as_uint(v.x);
            sreg[x + 1] = __float_as_uint(v.y);
          }
        }
        if (edge) {
#pragma unroll
          for (int x = 0; x < 64; ++x)
            if (32 * hf + x + (x >= 32 ? 32 : 0) > lim_col) sreg[x] = 0xff800000u;   // -inf replaces the value (NaN-safe)
        }
        const bool first = j == 0 && hf == 0;
        // O and l move to a new reference maximum.  The last PV issued for this Q tile (the other half: of this tile
        // for h = 1, of the previous tile for h = 0) must have completed before O is touched.
        auto rescale_to = [&](float m_new) {
          ptx::mbar_wait(bar(P_PVDONE + 2 * t + (hf ^ 1)), (hf == 1 ? j : j - 1) & 1);
          ptx::tc_fence_after();
          const float f = ex2(m_used - m_new);
          m_used = m_new;
          l_run *= f;
#pragma unroll 1
          for (int c = 0; c < D / 16; ++c) {
            uint32_t rr[16];
            ptx::tmem_ld16(tO + c * 16, rr);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int x = 0; x < 16; ++x) rr[x] = __float_as_uint(f32(rr[x]) * f);
            ptx::tmem_st16(tO + c * 16, rr);
          }
          ptx::tmem_wait_st();
        };
        // The exact maximum first: for the very first half (key 0 is always visible), and always under ALiBi, whose
        // bias grows by slope * 128 from tile to tile by construction -- an optimistic reference would be stale every
        // tile (lazy rescale: only when the maximum grew by more than 2^8).
        constexpr bool kExactMax = KM == kKmAlibi;
        if (first || kExactMax) {
          float r0 = -INFINITY, r1 = -INFINITY;
#pragma unroll
          for (int pg = 0; pg < 4; ++pg) {
            float a0 = -INFINITY, a1 = -INFINITY;
#pragma unroll
            for (int x = 16 * pg; x < 16 * pg + 16; x += 4) {
              a0 = fmaxf(fmaxf(a0, f32(sreg[x + 0])), f32(sreg[x + 1]));
              a1 = fmaxf(fmaxf(a1, f32(sreg[x + 2])), f32(sreg[x + 3]));
            }
            if (KM == kKmAlibi) r0 = fmaxf(r0, fmaxf(a0, a1) + abase[pg]);
            else { r0 = fmaxf(r0, a0); r1 = fmaxf(r1, a1); }
          }
          const float mx = fmaxf(r0, r1);
          if (first) m_used = mx;
          else if (__any_sync(0xffffffffu, mx > m_used + 8.f)) rescale_to(fmaxf(m_used, mx));
        }
        // P = 2^(S - m_used), packed in place; the half's own maximum is taken alongside
        const float2 negm = make_float2(-m_used, -m_used);
        float2 sum0 = make_float2(0.f, 0.f), sum1 = make_float2(0.f, 0.f);
        float mx0 = -INFINITY, mx1 = -INFINITY, mxa = -INFINITY;
#pragma unroll
        for (int x = 0; x < 32; x += 2) {
          const float s0 = f32(sreg[2 * x]), s1 = f32(sreg[2 * x + 1]), s2 = f32(sreg[2 * x + 2]), s3 = f32(sreg[2 * x + 3]);
          const float2 nm = KM == kKmAlibi ? make_float2(abase[x >> 3] - m_used, abase[x >> 3] - m_used) : negm;
          const float2 v0 = __fadd2_rn(make_float2(s0, s1), nm);
          const float2 v1 = __fadd2_rn(make_float2(s2, s3), nm);
          mx0 = fmaxf(fmaxf(mx0, s0), s1);
          mx1 = fmaxf(fmaxf(mx1, s2), s3);
          const float2 p0 = make_float2(ex2(v0.x), ex2(v0.y));
          const float2 p1 = make_float2(ex2(v1.x), ex2(v1.y));
          sum0 = __fadd2_rn(sum0, p0);
          sum1 = __fadd2_rn(sum1, p1);
          sreg[x] = ptx::pack_bf16(p0.x, p0.y);
          sreg[x + 1] = ptx::pack_bf16(p1.x, p1.y);
          if (KM == kKmAlibi && (x & 7) == 6) {               // end of a page: fold its per-page bias into the maximum
            mxa = fmaxf(mxa, fmaxf(mx0, mx1) + abase[x >> 3]);
            mx0 = -INFINITY; mx1 = -INFINITY;
          }
        }
        const float mxh = KM == kKmAlibi ? mxa : fmaxf(mx0, mx1);
        float hsum = (sum0.x + sum0.y) + (sum1.x + sum1.y);
        const bool slow = !first && !kExactMax && __any_sync(0xffffffffu, mxh > m_used + kDanger);
        if (slow) {
          // Slow path (a score beyond 2^kDanger of m_used): O and l move to the new maximum and this half of P is
          // rebuilt 16 columns (one page) at a time straight from S in TMEM.
          rescale_to(fmaxf(m_used, mxh));
          hsum = 0.f;
#pragma unroll 1
          for (int c = 0; c < 4; ++c) {
            const int key0 = 32 * hf + 16 * (c & 1) + 64 * (c >> 1);     // first key of this page of the half
            uint32_t rr[16], pk[8];
            ptx::tmem_ld16(tSh + 16 * c, rr);
            ptx::tmem_wait_ld();
            float off = -m_used;
            if (KM == kKmAlibi) off += alibi_slope * (float)(pstart[key0 >> 4] - alibi_pos_q);
#pragma unroll
            for (int x = 0; x < 16; x += 2) {
              float v0 = f32(rr[x]) + off, v1 = f32(rr[x + 1]) + off;
              if (KM == kKmAlibi) { v0 += alibi_slope * (float)x; v1 += alibi_slope * (float)(x + 1); }
              if (key0 + x > lim_col) v0 = -INFINITY;         // lim_col >= 127 on interior tiles
              if (key0 + x + 1 > lim_col) v1 = -INFINITY;
              const float q0 = ex2(v0), q1 = ex2(v1);
              hsum += q0 + q1;
              pk[x >> 1] = ptx::pack_bf16(q0, q1);
            }
            ptx::tmem_st8(tSh + 8 * c, pk);
          }
        }
        l_run += hsum;
        if (!slow) ptx::tmem_st32(tSh, sreg);                 // P_h (bf16 pairs) over the first 32 columns of S_h
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_tmem(lbar(P_PREADY + 2 * t + hf));
      }
    }

    // ---- epilogue (a9): normalise, round to bf16, store the row -------------------------------------------
    ptx::mbar_wait(bar(P_OFULL + t), 0);
    ptx::tc_fence_after();
    const float inv = 1.f / l_run;
    __nv_bfloat16* orow = a.out + ((size_t)(q_begin + i) * sh.Hq + hk * group + g) * D;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
      uint32_t rr[32];
      ptx::tmem_ld32(tO + c * 32, rr);
      ptx::tmem_wait_ld();
      if (valid) {
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          uint4 o;
          o.x = ptx::pack_bf16(f32(rr[8 * x + 0]) * inv, f32(rr[8 * x + 1]) * inv);
          o.y = ptx::pack_bf16(f32(rr[8 * x + 2]) * inv, f32(rr[8 * x + 3]) * inv);
          o.z = ptx::pack_bf16(f32(rr[8 * x + 4]) * inv, f32(rr[8 * x + 5]) * inv);
          o.w = ptx::pack_bf16(f32(rr[8 * x + 6]) * inv, f32(rr[8 * x + 7]) * inv);
          reinterpret_cast<uint4*>(orow + c * 32)[x] = o;
        }
      }
    }
  }

  // neither CTA may leave (its shared memory and TMEM are operands of the pair's MMAs) before both are done
  ptx::tc_fence_before();
  ptx::cluster_sync();
  if (warp == 13) ptx::tmem_dealloc_pair<512>(tbase);
}

}  // namespace
}  // namespace lazy
