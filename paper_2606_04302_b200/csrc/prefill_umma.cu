// prefill_umma.cu -- lazy_attn_prefill: tiled flash-attention on tcgen05/TMEM over position-free paged K.
//
// Path rows: a1 metadata fetch, a2 page gather (TMA, 128B-swizzled 16-token boxes), a3/a4 RoPE
// on the SMEM K tile in fp32 (and once per CTA on the Q tile), a5 QK^T and a7 PV on the 5th-gen tensor cores
// (tcgen05.mma, accumulators in TMEM), a6 mask + online softmax in fp32, a9 epilogue.
//
// What is computed: PAPER.md Eq. 4 (L94-106) with deferred RoPE (L108): K is stored un-rotated; each K tile is
// rotated ONCE per tile on chip by the absolute angle of its tokens before the MMA (Fig. 3b),
// Q is rotated once per CTA.  Angles: (p0 + t) * theta_j composed as e^{i p0 theta_j} (one table row per page,
// fp64-built) times e^{i t theta_j} (t < 16, constants in registers) -- stateless, absolute-index (L455).
//
// CTA = 2 Q tiles of 128 rows (GQA group packed into M: row = token*group + head-in-group, so one rotated K tile
// serves every head of the group) x KV tiles of 128 tokens (8 pages).  16 warps:
//   warps 0-3 / 4-7 : softmax warpgroup of Q tile 0 / 1 (thread = row; S from TMEM, P bf16 back into TMEM over S)
//   warps 8-11      : K-rotate warpgroup (SMEM tile in place, generic proxy -> fence.proxy.async -> MMA)
//   warp 12         : TMA producer (block-table fetch, K/V page boxes, Q tiles)
//   warp 13         : MMA issuer (one lane): S_t = Q_t Khat^T (SS), O_t += P_t V (A from TMEM, V MN-major)
//   warp 14         : V tail fixer (zeroes rows >= seq_len of the last tile so poisoned bytes never reach PV)
// TMEM (512 columns): S0 | S1 | O0 | O1, P_t aliases the first 64 columns of S_t.
#include <climits>

#include <cuda_fp16.h>

#include "prefill_common.cuh"

namespace lazy {
namespace {

template <int D>
struct PrefillCfg {
  static constexpr int NH = D / 64;                 // 128-byte column slabs per row
  static constexpr int TILE_BYTES = NH * kHalfBytes;
  static constexpr int CPR = D / 16;                // rotation chunk-pairs (8 pairs each) per row
  static constexpr int CS_ROW_BYTES = D / 2 * 8;    // one table row: D/2 (cos, sin) float2
  static constexpr int CS_STAGE_BYTES = kPagesPerTile * CS_ROW_BYTES;
  static constexpr int OFF_Q = 0;                   // 2 tiles
  static constexpr int OFF_K = 2 * TILE_BYTES;      // 2 stages
  static constexpr int OFF_V = 4 * TILE_BYTES;      // 2 stages
  static constexpr int OFF_CS = 6 * TILE_BYTES;     // 2 stages of 8 table rows (e^{i p0 theta_j} per page)
  static constexpr int OFF_BAR = OFF_CS + 2 * CS_STAGE_BYTES;
  static constexpr int NUM_BARS = 28;
  static constexpr int OFF_TMEM = OFF_BAR + NUM_BARS * 8;
  static constexpr int OFF_SIGN = OFF_TMEM + 16;    // ring of 4 tiles x 8 pages: sign of the page's relative offset
                                                    // (LAZY_K_STORED_POS) or its logical start (ALiBi)
  static constexpr int OFF_SC = OFF_SIGN + 4 * kPagesPerTile * 4;   // FP8 pages: [stage][K, V][page][16] row scales
  static constexpr int SMEM_BYTES = OFF_SC + 2 * 2 * kPagesPerTile * 64 + 1024;   // + alignment slack
};

// barrier indices
enum : int {
  B_QFULL = 0,    // +t   TMA -> softmax WG t
  B_QREADY = 2,   // +t   softmax WG t (4 warps) -> MMA
  B_KFULL = 4,    // +s   TMA (K boxes + table rows) -> rotate WG
  B_KREADY = 6,   // +s   rotate WG (4 warps) -> MMA
  B_KEMPTY = 8,   // +s   MMA commit -> TMA
  B_VFULL = 10,   // +s   TMA -> MMA, fixer
  B_VEMPTY = 12,  // +s   MMA commit -> TMA
  B_VFIXED = 14,  //      fixer -> MMA (last tile only)
  B_VLAST = 15,   //      TMA -> fixer: the last tile's V loads have been issued (one shot)
  B_SFULL = 16,   // +t   MMA commit -> softmax WG t
  B_PREADY = 18,  // +t   softmax WG t (4 warps) -> MMA
  B_OFULL = 20,   // +t   MMA commit -> softmax WG t (epilogue)
  B_PHALF = 22,   // +t   softmax WG t (4 warps) -> MMA: first half of P (keys 0..63) is in TMEM
  B_PVH = 24,     // +t   MMA commit -> softmax WG t: PV over the first half of P has completed (slow path only)
  B_VREADY = 26,  // +s   FP8 pages: rotate WG (4 warps) -> MMA: the V tile has been dequantised to bf16
};

// FP8 pages: 8 E4M3 codes (two words) -> 8 fp32 values, exact
__device__ __forceinline__ void e4m3x8_to_f32(uint2 v, float2 (&x)[4]) {
  const uint32_t h[4] = {ptx::e4m3x2_lo_to_f16x2(v.x), ptx::e4m3x2_hi_to_f16x2(v.x), ptx::e4m3x2_lo_to_f16x2(v.y),
                         ptx::e4m3x2_hi_to_f16x2(v.y)};
#pragma unroll
  for (int w = 0; w < 4; ++w) x[w] = __half22float2(*reinterpret_cast<const __half2*>(&h[w]));
}
__device__ __forceinline__ uint2 lds64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}

// F8: LAZY_KV_FP8_E4M3 pages.  A page's E4M3 codes land (TMA, un-swizzled rows of D bytes) at the
// start of the page's own 2 KB region of the bf16 tile; the rotate warpgroup reads ALL codes of the page into
// registers, and then writes the bf16 tile over them: K dequantised (code x the token's scale) and rotated in one
// pass, V dequantised -- and the rows past the end of the sequence cleared, which is the tail fixer's job on bf16
// pages.  The tensor cores see exactly the bf16 tiles they see on bf16 pages.
template <int D, int KM, bool F8>
__global__ void __launch_bounds__(kPrefillThreads, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v, const PrefillArgs a) {
  using C = PrefillCfg<D>;
  constexpr bool kNoRotate = KM == LAZY_K_ABSOLUTE || KM == kKmAlibi;   // the K tile goes to the MMA as it landed
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t smem_base = ptx::smem_u32(smem);
  const uint32_t sQ = smem_base + C::OFF_Q, sK = smem_base + C::OFF_K, sV = smem_base + C::OFF_V;
  const uint32_t sCS = smem_base + C::OFF_CS;
  const uint32_t bars = smem_base + C::OFF_BAR;
  auto bar = [&](int idx) { return bars + 8u * idx; };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_TMEM);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const Shape sh = a.sh;
  const int group = sh.group, TPT = a.tokens_per_tile, TPC = 2 * TPT;

  // ---- work item: (request, kv head, block of 2*TPT query tokens) -------------------------------------------
  // the m-blocks of one (request, kv head) stay adjacent (they share K/V through the L2); the last one, which sees
  // the most keys under the causal mask, goes first
  const int mblk = a.mblocks - 1 - blockIdx.x % a.mblocks;
  const int hk = (blockIdx.x / a.mblocks) % sh.Hkv;
  const int r = blockIdx.x / (a.mblocks * sh.Hkv);
  const int q_begin = a.cu_q_lens[r];
  const int n_q = a.cu_q_lens[r + 1] - q_begin;
  const int L = a.seq_lens[r];
  const int i0 = mblk * TPC;
  if (i0 >= n_q) return;
  const int i_end = min(i0 + TPC, n_q);
  if (L <= 0) {                                     // degenerate: rows of an empty sequence are zeros
    const int n = (i_end - i0) * group * (D / 8);
    for (int x = tid; x < n; x += kPrefillThreads) {
      int ch = x % (D / 8), g = (x / (D / 8)) % group, i = i0 + x / (D / 8 * group);
      reinterpret_cast<uint4*>(a.out + ((size_t)(q_begin + i) * sh.Hq + hk * group + g) * D)[ch] = make_uint4(0, 0, 0, 0);
    }
    return;
  }
  const int kv_len = max(1, min(L, L - n_q + i_end));      // keys visible to the last query row of this CTA
  const int n_kv = (kv_len + kTileRows - 1) / kTileRows;
  const int num_pages = (L + kPageSize - 1) / kPageSize;
  const int* bt = a.block_table + (size_t)r * sh.table_stride;
  const int* ppos = a.page_pos + (size_t)r * sh.table_stride;

  if (tid == 0) {
    for (int x = 0; x < 2; ++x) {
      ptx::mbar_init(bar(B_VREADY + x), 4);
      ptx::mbar_init(bar(B_QFULL + x), 1);  ptx::mbar_init(bar(B_QREADY + x), 4);
      ptx::mbar_init(bar(B_KFULL + x), 1);  ptx::mbar_init(bar(B_KREADY + x), 4);
      ptx::mbar_init(bar(B_KEMPTY + x), 1); ptx::mbar_init(bar(B_VFULL + x), 1);
      ptx::mbar_init(bar(B_VEMPTY + x), 1); ptx::mbar_init(bar(B_SFULL + x), 1);
      ptx::mbar_init(bar(B_PREADY + x), 4); ptx::mbar_init(bar(B_OFULL + x), 1);
      ptx::mbar_init(bar(B_PHALF + x), 4);  ptx::mbar_init(bar(B_PVH + x), 1);
    }
    ptx::mbar_init(bar(B_VFIXED), 1);
    ptx::mbar_init(bar(B_VLAST), 1);
    ptx::fence_mbar_init();
  }
  if (warp == 13) {
    ptx::tmem_alloc<512>(ptx::smem_u32(tmem_slot));
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tbase = *tmem_slot;

  if (warp >= 12) {
    ptx::setmaxnreg_dec<kRegsMisc>();
    if (warp == 12) {
      // ================================ TMA producer ========================================================
      if (lane == 0) { ptx::prefetch_tmap(&tmap_q); ptx::prefetch_tmap(&tmap_k); ptx::prefetch_tmap(&tmap_v); }
      if (lane < 2) {
        const int t = lane;
        ptx::mbar_arrive_expect_tx(bar(B_QFULL + t), C::NH * group * TPT * 128);
#pragma unroll
        for (int h = 0; h < C::NH; ++h)
          tma_load_4d(sQ + t * C::TILE_BYTES + h * kHalfBytes, &tmap_q, bar(B_QFULL + t), h * 64, 0, hk,
                      q_begin + i0 + t * TPT);
      }
      // lane -> (K or V, column slab, page of the tile); the K lanes of slab 0 also fetch the page's table row
      const int kvsel = lane >> 4, half = (lane >> 3) & 1, pg = lane & 7;
      const bool lane_on = half < C::NH;
      // table entries travel through a 3-deep shift register (tile j+2 -> j+1 -> j), so neither the table loads nor
      // the dependent stored-position lookup sit on the issue path.  (A cp.async.bulk.prefetch.tensor of the next
      // tile's boxes into L2 was tried here and cost 25%: the TMA unit is better left to the real loads.)
      auto entry = [&](int tile, int& page, int& pos) {
        const int idx = tile * kPagesPerTile + pg;
        page = 0; pos = 0;
        if (tile < n_kv && idx < num_pages) {
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
        const int s = j & 1, ph = (j >> 1) & 1;
        const int page = page_next;
        const int p0 = pos_next < 0 ? -pos_next : pos_next;      // negative only for LAZY_K_STORED_POS
        const int p0_sign = pos_next < 0 ? -1 : 1;
        page_next = page_n2; pos_next = pos_n2;
        entry(j + 2, page_n2, pos_n2);
        const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
        const int row0 = (page * sh.Hkv + hk) * kPageSize;
        const uint32_t dst = s * C::TILE_BYTES + half * kHalfBytes + pg * (kPageSize * 128);
        ptx::mbar_wait_sleep(bar(B_KEMPTY + s), ph ^ 1);
        if (KM == LAZY_K_STORED_POS && lane < kPagesPerTile) s_sign[(j & 3) * kPagesPerTile + pg] = p0_sign;
        if (KM == kKmAlibi && lane < kPagesPerTile) s_sign[(j & 3) * kPagesPerTile + pg] = p0;
        __syncwarp();
        const uint32_t sSC = smem_base + C::OFF_SC + s * (2 * kPagesPerTile * 64) + pg * 64;
        if (lane == 0)
          ptx::mbar_arrive_expect_tx(bar(B_KFULL + s), npv * ((F8 ? kPageSize * D + 64 : C::NH * kPageSize * 128) +
                                                              (kNoRotate ? 0 : C::CS_ROW_BYTES)));
        __syncwarp();
        if (kvsel == 0 && lane_on && pg < npv) {
          if (!F8) ptx::tma_load_2d(sK + dst, &tmap_k, bar(B_KFULL + s), half * 64, row0);
          if (F8 && half == 0) {
            ptx::tma_load_2d(sK + dst, &tmap_k, bar(B_KFULL + s), 0, row0);
            ptx::bulk_load_1d(sSC, a.k_scale + row0, 64, bar(B_KFULL + s));
          }
          if (half == 0 && !kNoRotate)
            ptx::bulk_load_1d(sCS + s * C::CS_STAGE_BYTES + pg * C::CS_ROW_BYTES, a.cs + (size_t)p0 * (D / 2),
                              C::CS_ROW_BYTES, bar(B_KFULL + s));
        }
        ptx::mbar_wait_sleep(bar(B_VEMPTY + s), ph ^ 1);
        if (lane == 0)
          ptx::mbar_arrive_expect_tx(bar(B_VFULL + s), npv * (F8 ? kPageSize * D + 64 : C::NH * kPageSize * 128));
        __syncwarp();
        if (kvsel == 1 && lane_on && pg < npv) {
          if (!F8) ptx::tma_load_2d(sV + dst, &tmap_v, bar(B_VFULL + s), half * 64, row0);
          if (F8 && half == 0) {
            ptx::tma_load_2d(sV + dst, &tmap_v, bar(B_VFULL + s), 0, row0);
            ptx::bulk_load_1d(sSC + kPagesPerTile * 64, a.v_scale + row0, 64, bar(B_VFULL + s));
          }
        }
        if (!F8 && j == n_kv - 1) {
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(bar(B_VLAST));
        }
      }
    } else if (warp == 13) {
      // ================================ MMA issuer ==========================================================
      // The whole warp walks the loop convergently and ONE elected lane issues: every operand of tcgen05.mma /
      // tcgen05.commit is then provably warp-uniform and lives in uniform registers.  (Issuing from inside
      // `if (lane == 0)` with opaque operands made the compiler wrap each MMA in an ELECT / R2UR / BRA.U.ANY
      // waterfall loop, ~16 dependent instructions per MMA: the issue thread, not the tensor pipe, set the pace.)
      constexpr uint32_t IDESC_QK = ptx::umma_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t IDESC_PV = ptx::umma_idesc_bf16(128, D, 0, 1);       // B = V is MN-major
      const uint32_t tb = __shfl_sync(0xffffffffu, tbase, 0);
      const int nkv = __shfl_sync(0xffffffffu, n_kv, 0);
      const bool leader = ptx::elect_one();
      auto qk = [&](int t, int s) {
        if (leader) {
          const uint32_t qa = sQ + t * C::TILE_BYTES, ka = sK + s * C::TILE_BYTES;
#pragma unroll
          for (int k = 0; k < D / 16; ++k) {
            const uint32_t off = (k >> 2) * kHalfBytes + (k & 3) * 32;
            ptx::umma_ss(tb + t * 128, ptx::umma_desc_sw128(qa + off, 0, 1024),
                         ptx::umma_desc_sw128(ka + off, 0, 1024), IDESC_QK, k > 0);
          }
        }
      };
      auto pv = [&](int t, int s, uint32_t acc, int k0, int k1) {
        if (leader) {
          const uint32_t va = sV + s * C::TILE_BYTES;
#pragma unroll
          for (int k = k0; k < k1; ++k)
            ptx::umma_ts(tb + 256 + t * 128, tb + t * 128 + k * 8,
                         ptx::umma_desc_sw128(va + k * 2048, kHalfBytes, 1024), IDESC_PV, acc | (uint32_t)(k > 0));
        }
      };
      auto commit = [&](int idx) { if (leader) ptx::umma_commit(bar(idx)); };
      ptx::mbar_wait(bar(B_KREADY + 0), 0);
      for (int t = 0; t < 2; ++t) {
        ptx::mbar_wait(bar(B_QREADY + t), 0);
        ptx::tc_fence_after();
        qk(t, 0);
        commit(B_SFULL + t);
      }
      commit(B_KEMPTY + 0);
      for (int j = 0; j < nkv; ++j) {
        const int s = j & 1;
        ptx::mbar_wait(bar((F8 ? B_VREADY : B_VFULL) + s), (j >> 1) & 1);
        if (!F8 && j == nkv - 1) ptx::mbar_wait(bar(B_VFIXED), 0);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          // PV starts on the first 64 keys while the softmax warpgroup is still exponentiating the other 64
          ptx::mbar_wait(bar(B_PHALF + t), j & 1);
          ptx::tc_fence_after();
          pv(t, s, j > 0, 0, kTileRows / 32);
          commit(B_PVH + t);
          ptx::mbar_wait(bar(B_PREADY + t), j & 1);
          ptx::tc_fence_after();
          pv(t, s, 1u, kTileRows / 32, kTileRows / 16);
          if (t == 1) commit(B_VEMPTY + s);
          if (j + 1 < nkv) {
            if (t == 0) {
              ptx::mbar_wait(bar(B_KREADY + (s ^ 1)), ((j + 1) >> 1) & 1);
              ptx::tc_fence_after();
            }
            qk(t, s ^ 1);
            commit(B_SFULL + t);
            if (t == 1) commit(B_KEMPTY + (s ^ 1));
          } else {
            commit(B_OFULL + t);
          }
        }
      }
      __syncwarp();
    } else if (warp == 14 && !F8) {
      // ================================ V tail fixer ========================================================
      // The fixer is not part of the V ring's full/empty hand-shake, so it must not walk the ring's phases (a lagging
      // observer would alias parities).  It sleeps on a one-shot barrier until the producer has ISSUED the last tile's
      // V loads: from then on VFULL[s] is in that tile's phase and cannot advance (the MMA warp waits for VFIXED).
      const int jl = n_kv - 1;
      ptx::mbar_wait_sleep(bar(B_VLAST), 0);
      ptx::mbar_wait_sleep(bar(B_VFULL + (jl & 1)), (jl >> 1) & 1);
      const int rows_valid = min(kTileRows, L - jl * kTileRows);
      if (rows_valid < kTileRows) {
        const int per_half = (kTileRows - rows_valid) * 8;          // 16-byte chunks to clear per column slab
        const uint32_t vb = sV + (jl & 1) * C::TILE_BYTES + rows_valid * 128;
        for (int x = lane; x < per_half * C::NH; x += 32)
          ptx::sts128(vb + (x / per_half) * kHalfBytes + (x % per_half) * 16, make_uint4(0, 0, 0, 0));
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar(B_VFIXED));
    }
  } else if (warp >= 8) {
    // ================================ K-rotate warpgroup ======================================================
    // thread = (page of the tile, group of CPR consecutive tokens, chunk pair c = 8 rotation pairs): it reads the
    // page's table row w = e^{i p0 theta_j} ONCE, composes it with the group's first in-page offset and then walks
    // its tokens with the one-step recurrence z <- z * e^{i theta_j} (at most 7 fp32 complex products away from a
    // table value built in fp64: ~4e-7 relative, PAPER.md L455's drift concern does not arise).  This takes the
    // per-token table reads (64 KB of LDS per tile, 2-way bank-conflicted) out of the shared-memory pipe, which the
    // tensor cores' operand fetches already load to ~40 % (profiles/r2_prefill_smem_attribution.md).
    // FP8 pages: the rotate warpgroup holds a page's codes of both tiles: 2*128*168 + 128*136 + 128*40 = 65536
    if (F8) ptx::setmaxnreg_inc<136>();
    else ptx::setmaxnreg_dec<kRegsRotate>();
    constexpr int TOK = C::CPR;                     // tokens per thread (16 threads serve a page)
    const int wtid = tid - 256;
    const int i = wtid >> 4;                        // page of the tile
    const int t0 = ((wtid & 15) / C::CPR) * TOK, c = wtid % C::CPR;
    float2 u0c[4], u0s[4], u1c[4], u1s[4];          // e^{i t0 theta_j}, e^{i theta_j} for this thread's 8 pairs
    if (KM == LAZY_K_UNROTATED) {
      const float4* r0 = reinterpret_cast<const float4*>(a.cs + (size_t)t0 * (D / 2));
      const float4* r1 = reinterpret_cast<const float4*>(a.cs + (size_t)1 * (D / 2));
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const float4 v0 = __ldg(r0 + cs_f4_index<D>(c, x)), v1 = __ldg(r1 + cs_f4_index<D>(c, x));
        u0c[x] = make_float2(v0.x, v0.y); u0s[x] = make_float2(v0.z, v0.w);
        u1c[x] = make_float2(v1.x, v1.y); u1s[x] = make_float2(v1.z, v1.w);
      }
    }
    const int* s_sign = reinterpret_cast<const int*>(smem + C::OFF_SIGN);
    for (int j = 0; j < n_kv; ++j) {
      const int s = j & 1;
      const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
      const uint32_t kb = sK + s * C::TILE_BYTES;
      const uint32_t cb = sCS + s * C::CS_STAGE_BYTES;
      ptx::mbar_wait(bar(B_KFULL + s), (j >> 1) & 1);
      if (F8) {
        // ---- FP8 pages: dequantise + rotate K, then dequantise V, each over its own landing area ----------------
        const uint32_t sc = smem_base + C::OFF_SC + s * (2 * kPagesPerTile * 64) + i * 64 + t0 * 4;
        const uint32_t land = i * (kPageSize * 128) + t0 * D + 8 * c;   // codes of (page i, token t0, dims 8c..)
        uint2 ra[TOK], rb[TOK];
        float scl[TOK];
        float2 zc[4], zs[4];
        if (i < npv) {
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint4 v = ptx::lds128(cb + i * C::CS_ROW_BYTES + 16 * cs_f4_index<D>(c, x));
            const float2 wc = make_float2(f32(v.x), f32(v.y)), ws = make_float2(f32(v.z), f32(v.w));
            zc[x] = __ffma2_rn(neg2(ws), u0s[x], __fmul2_rn(wc, u0c[x]));     // z = w * u0: the group's first token
            zs[x] = __ffma2_rn(wc, u0s[x], __fmul2_rn(ws, u0c[x]));
          }
#pragma unroll
          for (int tt = 0; tt < TOK; ++tt) {
            ra[tt] = lds64(kb + land + tt * D);
            rb[tt] = lds64(kb + land + tt * D + D / 2);
            scl[tt] = __int_as_float(ptx::lds32(sc + tt * 4));
          }
        }
        __syncwarp();                               // the 16 threads of a page have read its codes: overwrite them
        if (i < npv) {
#pragma unroll
          for (int tt = 0; tt < TOK; ++tt) {
            float2 x1[4], x2[4];
            e4m3x8_to_f32(ra[tt], x1);
            e4m3x8_to_f32(rb[tt], x2);
            const float2 sk2 = make_float2(scl[tt], scl[tt]);
            uint4 va, vb;
            uint32_t* aw = reinterpret_cast<uint32_t*>(&va);
            uint32_t* bw = reinterpret_cast<uint32_t*>(&vb);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
              const float2 cc = __fmul2_rn(zc[w], sk2), ss = __fmul2_rn(zs[w], sk2);   // the token's scale rides on z
              const float2 y1 = __ffma2_rn(neg2(x2[w]), ss, __fmul2_rn(x1[w], cc));
              const float2 y2 = __ffma2_rn(x2[w], cc, __fmul2_rn(x1[w], ss));
              aw[w] = ptx::pack_bf16(y1.x, y1.y);
              bw[w] = ptx::pack_bf16(y2.x, y2.y);
            }
            const int row = i * kPageSize + t0 + tt;
            ptx::sts128(kb + chunk_off(row, c), va);
            ptx::sts128(kb + chunk_off(row, c + C::CPR), vb);
            if (tt + 1 < TOK) {                     // next token: z <- z * e^{i theta_j}
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
        if (lane == 0) ptx::mbar_arrive(bar(B_KREADY + s));
        // ---- V: code x the token's scale -> bf16; rows at or past seq_len become zeros (never multiplied)
        const uint32_t vb_ = sV + s * C::TILE_BYTES;
        ptx::mbar_wait(bar(B_VFULL + s), (j >> 1) & 1);
        const int rows_valid = L - j * kTileRows;   // >= 128 on interior tiles
        if (i < npv) {
#pragma unroll
          for (int tt = 0; tt < TOK; ++tt) {
            ra[tt] = lds64(vb_ + land + tt * D);
            rb[tt] = lds64(vb_ + land + tt * D + D / 2);
            scl[tt] = __int_as_float(ptx::lds32(sc + kPagesPerTile * 64 + tt * 4));
          }
        }
        __syncwarp();
#pragma unroll
        for (int tt = 0; tt < TOK; ++tt) {
          const int row = i * kPageSize + t0 + tt;
          uint4 va = make_uint4(0, 0, 0, 0), vb = make_uint4(0, 0, 0, 0);
          if (i < npv && row < rows_valid) {
            float2 x1[4], x2[4];
            e4m3x8_to_f32(ra[tt], x1);
            e4m3x8_to_f32(rb[tt], x2);
            const float2 sv2 = make_float2(scl[tt], scl[tt]);
            uint32_t* aw = reinterpret_cast<uint32_t*>(&va);
            uint32_t* bw = reinterpret_cast<uint32_t*>(&vb);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
              const float2 y1 = __fmul2_rn(x1[w], sv2), y2 = __fmul2_rn(x2[w], sv2);
              aw[w] = ptx::pack_bf16(y1.x, y1.y);
              bw[w] = ptx::pack_bf16(y2.x, y2.y);
            }
          }
          if (i < npv || j == n_kv - 1) {           // pages that do not exist are cleared on the last tile only
            ptx::sts128(vb_ + chunk_off(row, c), va);
            ptx::sts128(vb_ + chunk_off(row, c + C::CPR), vb);
          }
        }
        ptx::fence_proxy_async();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(B_VREADY + s));
        continue;
      }
      if (!kNoRotate && i < npv) {
        float2 zc[4], zs[4];                        // e^{i (p0+t) theta_j}, or e^{i Delta theta_j} of the page
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          const uint4 v = ptx::lds128(cb + i * C::CS_ROW_BYTES + 16 * cs_f4_index<D>(c, x));
          zc[x] = make_float2(f32(v.x), f32(v.y));
          zs[x] = make_float2(f32(v.z), f32(v.w));
        }
        if (KM == LAZY_K_UNROTATED) {               // first token of the group: z = w * u0
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const float2 wc = zc[x], ws = zs[x];
            zc[x] = __ffma2_rn(neg2(ws), u0s[x], __fmul2_rn(wc, u0c[x]));
            zs[x] = __ffma2_rn(wc, u0s[x], __fmul2_rn(ws, u0c[x]));
          }
        } else {                                    // one relative rotation for the whole page (may be negative)
          const float sgn = (float)s_sign[(j & 3) * kPagesPerTile + i];
#pragma unroll
          for (int x = 0; x < 4; ++x) zs[x] = __fmul2_rn(zs[x], make_float2(sgn, sgn));
        }
        const int row0 = i * kPageSize + t0;
#pragma unroll
        for (int tb = 0; tb < TOK; tb += 4) {
          uint4 va[4], vb[4];
#pragma unroll
          for (int tt = 0; tt < 4; ++tt) {
            va[tt] = ptx::lds128(kb + chunk_off(row0 + tb + tt, c));
            vb[tt] = ptx::lds128(kb + chunk_off(row0 + tb + tt, c + C::CPR));
          }
#pragma unroll
          for (int tt = 0; tt < 4; ++tt) {
            rotate8_packed(va[tt], vb[tt], zc, zs);
            ptx::sts128(kb + chunk_off(row0 + tb + tt, c), va[tt]);
            ptx::sts128(kb + chunk_off(row0 + tb + tt, c + C::CPR), vb[tt]);
            if (KM == LAZY_K_UNROTATED && tb + tt + 1 < TOK) {      // next token: z <- z * e^{i theta_j}
#pragma unroll
              for (int x = 0; x < 4; ++x) {
                const float2 wc = zc[x], ws = zs[x];
                zc[x] = __ffma2_rn(neg2(ws), u1s[x], __fmul2_rn(wc, u1c[x]));
                zs[x] = __ffma2_rn(wc, u1s[x], __fmul2_rn(ws, u1c[x]));
              }
            }
          }
        }
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar(B_KREADY + s));
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
    // chunk by chunk behind the wait (a 128-register copy of the row held across the wait was spilled by ptxas)
    const float4* csp = reinterpret_cast<const float4*>(a.cs);
    if (valid && KM != kKmAlibi) {
      const int pos = ppos[sq / kPageSize] + sq % kPageSize;
      csp = reinterpret_cast<const float4*>(a.cs + (size_t)pos * (D / 2));
      if (g == 0) {
#pragma unroll
        for (int x = 0; x < D / 4; x += 8) asm volatile("prefetch.global.L2 [%0];" ::"l"(csp + x));
      }
    }
    ptx::mbar_wait(bar(B_QFULL + t), 0);
    {
      const uint32_t qb = sQ + t * C::TILE_BYTES;
      if (valid) {
        uint4 src[2 * C::CPR];                      // LAZY_ROPE_INTERLEAVED: the whole row first (in-place hazard)
        if (a.q_interleaved) {
#pragma unroll
          for (int c = 0; c < 2 * C::CPR; ++c) src[c] = ptx::lds128(qb + chunk_off(row, c));
        }
#pragma unroll
        for (int c = 0; c < C::CPR; ++c) {
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
          const uint32_t pa = qb + chunk_off(row, c), pb = qb + chunk_off(row, c + C::CPR);
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
        for (int c = 0; c < 2 * C::CPR; ++c) ptx::sts128(qb + chunk_off(row, c), make_uint4(0, 0, 0, 0));
      }
    }
    ptx::fence_proxy_async();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar(B_QREADY + t));

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
    // Online softmax with OPTIMISTIC exponentials.  The output is O / l whatever reference value m the exponentials
    // use (floating point keeps relative precision at any scale), so after the first tile -- whose exact row max
    // becomes m_used -- a tile's P = 2^(S - m_used) is computed straight away with the m_used already at hand, and
    // the tile's own maximum is taken alongside (it has no consumer on the critical path).  Only if a score
    // exceeds m_used by more than kDanger (P > 2^20: never with sane inputs after the first 128 keys) the warp takes
    // the slow path: it brings O and l to the new maximum and recomputes that half of P.  This takes the
    // load-then-max phase (~600 cycles per tile) out of the softmax -> PV -> QK -> softmax chain that sets the
    // kernel's pace.
    constexpr float kDanger = 20.f;
    float m_used = -INFINITY, l_run = 0.f;
    if (t == 1) ptx::named_bar_arrive(2, 256);                            // tile 0 goes first
    for (int j = 0; j < n_kv; ++j) {
      uint32_t sreg[128];                                     // this row of S (fp32 bits); P is packed over it in place
      ptx::mbar_wait(bar(B_SFULL + t), j & 1);
      ptx::tc_fence_after();
      float abase[kPagesPerTile];                             // kKmAlibi: slope * (page start - m) of the tile's pages
#pragma unroll
      for (int c = 0; c < 4; ++c) ptx::tmem_ld32(tS + c * 32, sreg + c * 32);
      if (KM == kKmAlibi) {
        const int* pstart = reinterpret_cast<const int*>(smem + C::OFF_SIGN) + (j & 3) * kPagesPerTile;
#pragma unroll
        for (int pg = 0; pg < kPagesPerTile; ++pg) abase[pg] = alibi_slope * (float)(pstart[pg] - alibi_pos_q);
      }
      const bool edge = j * kTileRows + kTileRows - 1 > lim_min;   // tile touches the causal edge / the tail: rare
      const int lim_col = lim_row - j * kTileRows;            // column visible iff col <= lim_col
      // columns 64hf .. 64hf+63 as they enter the softmax: ALiBi's in-page part slope * t added (S += slope * (n - m),
      // n = page start + t; the per-page part abase[] is folded into the maxima and into the exponential's constant),
      // masked columns replaced by -inf (never multiplied: poisoned bytes past the tail may be NaN)
      auto prep_half = [&](int hf) {
        if (KM == kKmAlibi) {
#pragma unroll
          for (int x = 64 * hf; x < 64 * hf + 64; x += 2) {
            const float2 v = __fadd2_rn(make_float2(f32(sreg[x]), f32(sreg[x + 1])), alibi_d2[(x & 15) >> 1]);
            sreg[x] = __float_as_uint(v.x);
            sreg[x + 1] = __float_as_uint(v.y);
          }
        }
        if (edge) {
#pragma unroll
          for (int x = 64 * hf; x < 64 * hf + 64; ++x)
            if (x > lim_col) sreg[x] = 0xff800000u;
        }
      };
      ptx::tmem_wait_ld();
      prep_half(0);
      prep_half(1);
      // The exact row max first: on the first tile (column 0 is always visible), and always under ALiBi, whose bias
      // grows by slope * 128 from tile to tile by construction -- an optimistic reference would be stale every tile.
      if (j == 0 || KM == kKmAlibi) {
        float r0 = -INFINITY, r1 = -INFINITY;
#pragma unroll
        for (int pg = 0; pg < kPagesPerTile; ++pg) {
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
        if (j == 0) {
          m_used = mx;
        } else if (__any_sync(0xffffffffu, mx > m_used + 8.f)) {   // PV(j-1) has completed: S(j) was committed after it
          const float m_new = fmaxf(m_used, mx);
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
        }
      }
      ptx::named_bar_sync(2 + t, 256);                                   // my turn on the MUFU
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
        // P = 2^(S - m_used) for this half, packed in place; the half's own maximum is taken alongside
        const float2 negm = make_float2(-m_used, -m_used);
        float2 sum0 = make_float2(0.f, 0.f), sum1 = make_float2(0.f, 0.f);
        float mx0 = -INFINITY, mx1 = -INFINITY, mxa = -INFINITY;
#pragma unroll
        for (int x = 32 * hf; x < 32 * hf + 32; x += 2) {
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
        const bool slow = j > 0 && KM != kKmAlibi && __any_sync(0xffffffffu, mxh > m_used + kDanger);
        if (slow) {
          // Slow path (a score beyond 2^kDanger of m_used).  O and l -- which hold the tiles < j, and keys 0..63 of
          // this tile once the first half of PV has completed -- move to the new maximum; then this half of P is
          // rebuilt 16 columns at a time straight from S in TMEM (P half 0 sits in columns 0..31, so the S columns
          // still to be read are intact) and written back to TMEM from here.
          if (hf == 1) {
            ptx::mbar_wait(bar(B_PVH + t), j & 1);
            ptx::tc_fence_after();
          }
          const float m_new = fmaxf(m_used, mxh);
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
          hsum = 0.f;
          const int* pstart = reinterpret_cast<const int*>(smem + C::OFF_SIGN) + (j & 3) * kPagesPerTile;
#pragma unroll 1
          for (int c = 0; c < 4; ++c) {
            const int col0 = 64 * hf + 16 * c;                // one page of the tile
            uint32_t rr[16], pk[8];
            ptx::tmem_ld16(tS + col0, rr);
            ptx::tmem_wait_ld();
            float off = -m_used;
            if (KM == kKmAlibi) off += alibi_slope * (float)(pstart[col0 >> 4] - alibi_pos_q);
#pragma unroll
            for (int x = 0; x < 16; x += 2) {
              float v0 = f32(rr[x]) + off, v1 = f32(rr[x + 1]) + off;
              if (KM == kKmAlibi) { v0 += alibi_slope * (float)x; v1 += alibi_slope * (float)(x + 1); }
              if (col0 + x > lim_col) v0 = -INFINITY;         // lim_col >= 127 on interior tiles
              if (col0 + x + 1 > lim_col) v1 = -INFINITY;
              const float q0 = ex2(v0), q1 = ex2(v1);
              hsum += q0 + q1;
              pk[x >> 1] = ptx::pack_bf16(q0, q1);
            }
            ptx::tmem_st8(tS + (col0 >> 1), pk);
          }
        }
        l_run += hsum;
        if (hf == 1) ptx::named_bar_arrive(2 + (t ^ 1), 256);                 // the other tile's turn
        if (!slow) ptx::tmem_st32(tS + 32 * hf, sreg + 32 * hf);   // P (bf16 pairs) over the first 64 columns of S
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar((hf == 0 ? B_PHALF : B_PREADY) + t));
      }
    }

    if (t == 0) ptx::named_bar_sync(2, 256);                              // consume tile 1's last hand-off
    // ---- epilogue (a9): normalise, round to bf16, store the row -------------------------------------------
    ptx::mbar_wait(bar(B_OFULL + t), 0);
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

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 13) ptx::tmem_dealloc<512>(tbase);
}

}  // namespace

template <int D, int KM, bool F8 = false>
static int launch_prefill_t(const lazy_handle* h, const PrefillArgs& args, int grid, cudaStream_t stream) {
  using C = PrefillCfg<D>;
  auto kern = prefill_umma_kernel<D, KM, F8>;
  // per launch: the attribute is per device, and a process may hold handles on several devices
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess)
    return LAZY_ERR_CUDA;
  const CUtensorMap* mq = reinterpret_cast<const CUtensorMap*>(h->tmap_pq);
  const CUtensorMap* mk = reinterpret_cast<const CUtensorMap*>(h->tmap_pk);
  const CUtensorMap* mv = reinterpret_cast<const CUtensorMap*>(h->tmap_pv);
  kern<<<grid, kPrefillThreads, C::SMEM_BYTES, stream>>>(*mq, *mk, *mv, args);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

int launch_prefill(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                   const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                   const int32_t* cu_q_lens, int num_reqs, int total_q, int max_q_len, void* out,
                   cudaStream_t stream) {
  const lazy_config& c = h->cfg;
  const int group = c.num_q_heads / c.num_kv_heads;
  const int tpt = kTileRows / group;                 // query tokens per 128-row tile
  const long long rows = (long long)c.num_pages * c.num_kv_heads * kPageSize;
  const bool fp8 = c.dtype == LAZY_KV_FP8_E4M3;
  const bool fp8_pair = fp8 && c.head_dim == 128 && !(c.flags & LAZY_FLAG_PREFILL_ONE_CTA);
  if (h->tmap_pk_ptr != k_cache) {
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_pk, k_cache, rows, c.head_dim, kPageSize, false, c.head_dim)
              : encode_pool_tmap(h->tmap_pk, k_cache, rows, c.head_dim, kPageSize)))
      return LAZY_ERR_CUDA;
    h->tmap_pk_ptr = k_cache;
  }
  if (h->tmap_pv_ptr != v_cache) {
    // (FP8 pages on CTA pairs: a CTA takes its own 64 code bytes of every V row)
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_pv, v_cache, rows, c.head_dim, kPageSize, false, fp8_pair ? 64 : c.head_dim)
              : encode_pool_tmap(h->tmap_pv, v_cache, rows, c.head_dim, kPageSize)))
      return LAZY_ERR_CUDA;
    h->tmap_pv_ptr = v_cache;
  }
  if (h->tmap_pq_ptr != q || h->tmap_pq_rows != total_q) {
    if (!encode_q_tmap(h->tmap_pq, q, total_q, c.num_q_heads, c.num_kv_heads, c.head_dim, tpt)) return LAZY_ERR_CUDA;
    h->tmap_pq_ptr = q;
    h->tmap_pq_rows = total_q;
  }
  PrefillArgs a;
  a.block_table = block_table;
  a.page_pos = page_logical_pos;
  a.seq_lens = seq_lens;
  a.cu_q_lens = cu_q_lens;
  a.out = static_cast<__nv_bfloat16*>(out);
  a.cs = h->ws.cs;
  a.stored_pos = h->page_stored_pos;
  a.alibi = h->ws.alibi;
  a.num_reqs = num_reqs;
  a.q_interleaved = c.rope_style == LAZY_ROPE_INTERLEAVED;
  a.mblocks = (max_q_len + 2 * tpt - 1) / (2 * tpt);
  a.tokens_per_tile = tpt;
  a.sh = h->shape;
  a.k_scale = h->k_scale;
  a.v_scale = h->v_scale;
  if (fp8 && !fp8_pair) {
    // FP8 pages at head_dim 64 (and the A/B arm at 128) run on the one-CTA kernel
    const long long grid = (long long)a.mblocks * c.num_kv_heads * num_reqs;
    if (grid <= 0 || grid > INT_MAX) return LAZY_ERR_INVALID;
    return c.head_dim == 128 ? launch_prefill_t<128, LAZY_K_UNROTATED, true>(h, a, (int)grid, stream)
                             : launch_prefill_t<64, LAZY_K_UNROTATED, true>(h, a, (int)grid, stream);
  }
  if (c.head_dim == 128 && !(c.flags & LAZY_FLAG_PREFILL_ONE_CTA)) {
    // CTA pairs (prefill_umma2.cu): a pair covers 4 * tpt query tokens
    a.mblocks = (max_q_len + 4 * tpt - 1) / (4 * tpt);
    const long long pgrid = 2LL * a.mblocks * c.num_kv_heads * num_reqs;
    if (pgrid <= 0 || pgrid > INT_MAX) return LAZY_ERR_INVALID;
    const int km = c.rope_style == LAZY_POS_ALIBI ? kKmAlibi : c.k_storage;
    return launch_prefill_pair(h, a, km, (int)pgrid, stream);
  }
  const long long grid = (long long)a.mblocks * c.num_kv_heads * num_reqs;
  if (grid <= 0 || grid > INT_MAX) return LAZY_ERR_INVALID;
  const int g = (int)grid;
  if (c.rope_style == LAZY_POS_ALIBI)
    return c.head_dim == 128 ? launch_prefill_t<128, kKmAlibi>(h, a, g, stream)
                             : launch_prefill_t<64, kKmAlibi>(h, a, g, stream);
  if (c.head_dim == 128) {
    if (c.k_storage == LAZY_K_STORED_POS) return launch_prefill_t<128, LAZY_K_STORED_POS>(h, a, g, stream);
    if (c.k_storage == LAZY_K_ABSOLUTE) return launch_prefill_t<128, LAZY_K_ABSOLUTE>(h, a, g, stream);
    return launch_prefill_t<128, LAZY_K_UNROTATED>(h, a, g, stream);
  }
  if (c.k_storage == LAZY_K_STORED_POS) return launch_prefill_t<64, LAZY_K_STORED_POS>(h, a, g, stream);
  if (c.k_storage == LAZY_K_ABSOLUTE) return launch_prefill_t<64, LAZY_K_ABSOLUTE>(h, a, g, stream);
  return launch_prefill_t<64, LAZY_K_UNROTATED>(h, a, g, stream);
}

}  // namespace lazy
