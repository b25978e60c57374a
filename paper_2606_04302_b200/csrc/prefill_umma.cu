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

#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {
namespace {

constexpr int kPrefillThreads = 512;
constexpr int kTileRows = 128;          // rows of a Q tile == keys of a KV tile
constexpr int kHalfBytes = kTileRows * 128;   // one 64-column (128-byte) slab of a 128-row tile
constexpr int kPagesPerTile = kTileRows / kPageSize;
constexpr float kRescaleThreshold = 8.f;      // log2 units: O is rescaled only when the row max grew by > 2^8

template <int D>
struct PrefillCfg {
  static constexpr int NH = D / 64;                 // 128-byte column slabs per row
  static constexpr int TILE_BYTES = NH * kHalfBytes;
  static constexpr int CPR = D / 16;                // rotation chunk-pairs (8 pairs each) per row
  static constexpr int OFF_Q = 0;                   // 2 tiles
  static constexpr int OFF_K = 2 * TILE_BYTES;      // 2 stages
  static constexpr int OFF_V = 4 * TILE_BYTES;      // 2 stages
  static constexpr int OFF_BAR = 6 * TILE_BYTES;
  static constexpr int NUM_BARS = 24;
  static constexpr int OFF_TMEM = OFF_BAR + NUM_BARS * 8;
  static constexpr int SMEM_BYTES = OFF_TMEM + 16 + 1024;   // + alignment slack
};

// barrier indices
enum : int {
  B_QFULL = 0,    // +t   TMA -> softmax WG t
  B_QREADY = 2,   // +t   softmax WG t (4 warps) -> MMA
  B_KFULL = 4,    // +s   TMA -> rotate WG
  B_KREADY = 6,   // +s   rotate WG (4 warps) -> MMA
  B_KEMPTY = 8,   // +s   MMA commit -> TMA
  B_VFULL = 10,   // +s   TMA -> MMA, fixer
  B_VEMPTY = 12,  // +s   MMA commit -> TMA
  B_VFIXED = 14,  //      fixer -> MMA (last tile only)
  B_SFULL = 16,   // +t   MMA commit -> softmax WG t
  B_PREADY = 18,  // +t   softmax WG t (4 warps) -> MMA
  B_OFULL = 20,   // +t   MMA commit -> softmax WG t (epilogue)
};

struct PrefillArgs {
  const int* block_table;
  const int* page_pos;
  const int* seq_lens;
  const int* cu_q_lens;
  __nv_bfloat16* out;
  const float2* cs;
  int num_reqs;
  int mblocks;          // CTAs per (request, kv head)
  int tokens_per_tile;  // 128 / group
  Shape sh;
};

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const void* tmap, uint32_t bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// (cos, sin) of the 8 rotation pairs j = 8c .. 8c+7 from one row of the table (layout: cs_index in ptx_util.cuh):
// four 16-byte loads, each holding (cos j, sin j, cos j+1, sin j+1).
template <int D>
__device__ __forceinline__ void load_cs8(const float2* __restrict__ cs_row, int c, float (&co)[8], float (&si)[8]) {
  constexpr int JT = D / 8;
  const int j0 = 8 * c, tq = j0 / JT, k0 = (j0 % JT) / 2;
  const float4* p = reinterpret_cast<const float4*>(cs_row);
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    float4 v = __ldg(p + (k0 + x) * 4 + tq);
    co[2 * x] = v.x; si[2 * x] = v.y; co[2 * x + 1] = v.z; si[2 * x + 1] = v.w;
  }
}

// byte offset of 16-byte chunk `ci` (8 dims: 8ci .. 8ci+7) of row `row` inside a 128-row, 128B-swizzled tile
__device__ __forceinline__ uint32_t chunk_off(int row, int ci) {
  return (ci >> 3) * kHalfBytes + row * 128 + (((ci & 7) ^ (row & 7)) << 4);
}

// rotate 8 pairs held as two 16-byte chunks (x1 = dims j, x2 = dims j + D/2) by (co, si), scale, round to bf16
__device__ __forceinline__ void rotate8(uint4& a, uint4& b, const float (&co)[8], const float (&si)[8], float scale) {
  uint32_t* aw = reinterpret_cast<uint32_t*>(&a);
  uint32_t* bw = reinterpret_cast<uint32_t*>(&b);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float a0 = ptx::bf16_lo(aw[w]), a1 = ptx::bf16_hi(aw[w]);
    float b0 = ptx::bf16_lo(bw[w]), b1 = ptx::bf16_hi(bw[w]);
    float c0 = co[2 * w] * scale, s0 = si[2 * w] * scale, c1 = co[2 * w + 1] * scale, s1 = si[2 * w + 1] * scale;
    aw[w] = ptx::pack_bf16(a0 * c0 - b0 * s0, a1 * c1 - b1 * s1);
    bw[w] = ptx::pack_bf16(a0 * s0 + b0 * c0, a1 * s1 + b1 * c1);
  }
}

template <int D>
__global__ void __launch_bounds__(kPrefillThreads, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v, const PrefillArgs a) {
  using C = PrefillCfg<D>;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t smem_base = ptx::smem_u32(smem);
  const uint32_t sQ = smem_base + C::OFF_Q, sK = smem_base + C::OFF_K, sV = smem_base + C::OFF_V;
  const uint32_t bars = smem_base + C::OFF_BAR;
  auto bar = [&](int idx) { return bars + 8u * idx; };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_TMEM);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const Shape sh = a.sh;
  const int group = sh.group, TPT = a.tokens_per_tile, TPC = 2 * TPT;

  // ---- work item: (request, kv head, block of 2*TPT query tokens) -------------------------------------------
  const int mblk = blockIdx.x % a.mblocks;
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
      ptx::mbar_init(bar(B_QFULL + x), 1);  ptx::mbar_init(bar(B_QREADY + x), 4);
      ptx::mbar_init(bar(B_KFULL + x), 1);  ptx::mbar_init(bar(B_KREADY + x), 4);
      ptx::mbar_init(bar(B_KEMPTY + x), 1); ptx::mbar_init(bar(B_VFULL + x), 1);
      ptx::mbar_init(bar(B_VEMPTY + x), 1); ptx::mbar_init(bar(B_SFULL + x), 1);
      ptx::mbar_init(bar(B_PREADY + x), 4); ptx::mbar_init(bar(B_OFULL + x), 1);
    }
    ptx::mbar_init(bar(B_VFIXED), 1);
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

  if (warp == 12) {
    // ================================ TMA producer ==========================================================
    if (lane == 0) { ptx::prefetch_tmap(&tmap_q); ptx::prefetch_tmap(&tmap_k); ptx::prefetch_tmap(&tmap_v); }
    if (lane < 2) {
      const int t = lane;
      ptx::mbar_arrive_expect_tx(bar(B_QFULL + t), C::NH * group * TPT * 128);
#pragma unroll
      for (int h = 0; h < C::NH; ++h)
        tma_load_4d(sQ + t * C::TILE_BYTES + h * kHalfBytes, &tmap_q, bar(B_QFULL + t), h * 64, 0, hk,
                    q_begin + i0 + t * TPT);
    }
    const int kvsel = lane >> 4, half = (lane >> 3) & 1, pg = lane & 7;
    const bool lane_on = half < C::NH;
    int page_next = (pg < num_pages) ? bt[pg] : 0;
    for (int j = 0; j < n_kv; ++j) {
      const int s = j & 1, ph = (j >> 1) & 1;
      const int page = page_next;
      if (j + 1 < n_kv) {
        const int idx = (j + 1) * kPagesPerTile + pg;
        page_next = idx < num_pages ? bt[idx] : 0;
      }
      const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
      const int row0 = (page * sh.Hkv + hk) * kPageSize;
      const uint32_t dst = s * C::TILE_BYTES + half * kHalfBytes + pg * (kPageSize * 128);
      ptx::mbar_wait(bar(B_KEMPTY + s), ph ^ 1);
      if (lane == 0) ptx::mbar_arrive_expect_tx(bar(B_KFULL + s), npv * C::NH * kPageSize * 128);
      __syncwarp();
      if (kvsel == 0 && lane_on && pg < npv) ptx::tma_load_2d(sK + dst, &tmap_k, bar(B_KFULL + s), half * 64, row0);
      ptx::mbar_wait(bar(B_VEMPTY + s), ph ^ 1);
      if (lane == 0) ptx::mbar_arrive_expect_tx(bar(B_VFULL + s), npv * C::NH * kPageSize * 128);
      __syncwarp();
      if (kvsel == 1 && lane_on && pg < npv) ptx::tma_load_2d(sV + dst, &tmap_v, bar(B_VFULL + s), half * 64, row0);
    }
  } else if (warp == 13) {
    // ================================ MMA issuer (one lane) =================================================
    if (lane == 0) {
      constexpr uint32_t IDESC_QK = ptx::umma_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t IDESC_PV = ptx::umma_idesc_bf16(128, D, 0, 1);     // B = V is MN-major
      auto qk = [&](int t, int s) {
#pragma unroll
        for (int k = 0; k < D / 16; ++k) {
          const uint32_t off = (k >> 2) * kHalfBytes + (k & 3) * 32;
          ptx::umma_ss(tbase + t * 128, ptx::umma_desc_sw128(sQ + t * C::TILE_BYTES + off, 0, 1024),
                       ptx::umma_desc_sw128(sK + s * C::TILE_BYTES + off, 0, 1024), IDESC_QK, k > 0);
        }
      };
      auto pv = [&](int t, int s, uint32_t acc) {
#pragma unroll
        for (int k = 0; k < kTileRows / 16; ++k)
          ptx::umma_ts(tbase + 256 + t * 128, tbase + t * 128 + k * 8,
                       ptx::umma_desc_sw128(sV + s * C::TILE_BYTES + k * 2048, kHalfBytes, 1024), IDESC_PV,
                       acc | (uint32_t)(k > 0));
      };
      ptx::mbar_wait(bar(B_KREADY + 0), 0);
      for (int t = 0; t < 2; ++t) {
        ptx::mbar_wait(bar(B_QREADY + t), 0);
        ptx::tc_fence_after();
        qk(t, 0);
        ptx::umma_commit(bar(B_SFULL + t));
      }
      ptx::umma_commit(bar(B_KEMPTY + 0));
      for (int j = 0; j < n_kv; ++j) {
        const int s = j & 1;
        ptx::mbar_wait(bar(B_VFULL + s), (j >> 1) & 1);
        if (j == n_kv - 1) ptx::mbar_wait(bar(B_VFIXED), 0);
        for (int t = 0; t < 2; ++t) {
          ptx::mbar_wait(bar(B_PREADY + t), j & 1);
          ptx::tc_fence_after();
          pv(t, s, j > 0);
          if (t == 1) ptx::umma_commit(bar(B_VEMPTY + s));
          if (j + 1 < n_kv) {
            if (t == 0) {
              ptx::mbar_wait(bar(B_KREADY + (s ^ 1)), ((j + 1) >> 1) & 1);
              ptx::tc_fence_after();
            }
            qk(t, s ^ 1);
            ptx::umma_commit(bar(B_SFULL + t));
            if (t == 1) ptx::umma_commit(bar(B_KEMPTY + (s ^ 1)));
          } else {
            ptx::umma_commit(bar(B_OFULL + t));
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 14) {
    // ================================ V tail fixer ==========================================================
    for (int j = 0; j < n_kv; ++j) ptx::mbar_wait(bar(B_VFULL + (j & 1)), (j >> 1) & 1);
    const int jl = n_kv - 1;
    const int rows_valid = min(kTileRows, L - jl * kTileRows);
    if (rows_valid < kTileRows) {
      const int n = (kTileRows - rows_valid) * 8 * C::NH;       // 16-byte chunks to clear
      unsigned char* vb = smem + C::OFF_V + (jl & 1) * C::TILE_BYTES;
      for (int x = lane; x < n; x += 32) {
        const int h = x / ((kTileRows - rows_valid) * 8), y = x % ((kTileRows - rows_valid) * 8);
        *reinterpret_cast<uint4*>(vb + h * kHalfBytes + rows_valid * 128 + y * 16) = make_uint4(0, 0, 0, 0);
      }
    }
    ptx::fence_proxy_async();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar(B_VFIXED));
  } else if (warp >= 8 && warp < 12) {
    // ================================ K-rotate warpgroup ====================================================
    constexpr int TPP = 16 * C::CPR;                // threads per page
    constexpr int PPP = 128 / TPP;                  // pages per pass
    constexpr int PASSES = kPagesPerTile / PPP;
    const int wtid = tid - 256;
    const int pp_ = wtid / TPP, t = (wtid % TPP) / C::CPR, c = wtid % C::CPR;
    float uc[8], us[8];                             // e^{i t theta_j}: in-page offset, fixed per thread
    load_cs8<D>(a.cs + (size_t)t * (D / 2), c, uc, us);
    for (int j = 0; j < n_kv; ++j) {
      const int s = j & 1;
      const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
      int p0s[PASSES];
#pragma unroll
      for (int ps = 0; ps < PASSES; ++ps) {
        const int i = ps * PPP + pp_;
        p0s[ps] = (i < npv) ? ppos[j * kPagesPerTile + i] : 0;
      }
      float wc[2][8], ws[2][8];                     // e^{i p0 theta_j} of the page being / about to be rotated
      load_cs8<D>(a.cs + (size_t)p0s[0] * (D / 2), c, wc[0], ws[0]);
      ptx::mbar_wait(bar(B_KFULL + s), (j >> 1) & 1);
      unsigned char* kb = smem + C::OFF_K + s * C::TILE_BYTES;
#pragma unroll
      for (int ps = 0; ps < PASSES; ++ps) {
        if (ps + 1 < PASSES) load_cs8<D>(a.cs + (size_t)p0s[ps + 1] * (D / 2), c, wc[(ps + 1) & 1], ws[(ps + 1) & 1]);
        const int i = ps * PPP + pp_;
        if (i < npv) {
          float zc[8], zs[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            zc[e] = wc[ps & 1][e] * uc[e] - ws[ps & 1][e] * us[e];
            zs[e] = ws[ps & 1][e] * uc[e] + wc[ps & 1][e] * us[e];
          }
          const int row = i * kPageSize + t;
          uint4* pa = reinterpret_cast<uint4*>(kb + chunk_off(row, c));
          uint4* pb = reinterpret_cast<uint4*>(kb + chunk_off(row, c + C::CPR));
          uint4 va = *pa, vb = *pb;
          rotate8(va, vb, zc, zs, 1.0f);
          *pa = va; *pb = vb;
        }
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar(B_KREADY + s));
    }
  } else if (warp < 8) {
    // ================================ softmax warpgroups ====================================================
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
    ptx::mbar_wait(bar(B_QFULL + t), 0);
    {
      unsigned char* qb = smem + C::OFF_Q + t * C::TILE_BYTES;
      if (valid) {
        const int pos = ppos[sq / kPageSize] + sq % kPageSize;
        const float2* cs_row = a.cs + (size_t)pos * (D / 2);
#pragma unroll
        for (int c = 0; c < C::CPR; ++c) {
          float co[8], si[8];
          load_cs8<D>(cs_row, c, co, si);
          uint4* pa = reinterpret_cast<uint4*>(qb + chunk_off(row, c));
          uint4* pb = reinterpret_cast<uint4*>(qb + chunk_off(row, c + C::CPR));
          uint4 va = *pa, vb = *pb;
          rotate8(va, vb, co, si, sh.scale_log2);
          *pa = va; *pb = vb;
        }
      } else {
#pragma unroll
        for (int c = 0; c < 2 * C::CPR; ++c)
          *reinterpret_cast<uint4*>(qb + chunk_off(row, c)) = make_uint4(0, 0, 0, 0);
      }
    }
    ptx::fence_proxy_async();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar(B_QREADY + t));

    float m_used = -INFINITY, l_run = 0.f;
    for (int j = 0; j < n_kv; ++j) {
      ptx::mbar_wait(bar(B_SFULL + t), j & 1);
      ptx::tc_fence_after();
      const int lim_col = lim_row - j * kTileRows;            // column visible iff col <= lim_col
      const bool need_mask = j * kTileRows + kTileRows - 1 > lim_min;
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t rr[32];
        ptx::tmem_ld32(tS + c * 32, rr);
        ptx::tmem_wait_ld();
#pragma unroll
        for (int x = 0; x < 32; ++x) {
          float v = __uint_as_float(rr[x]);
          if (need_mask && c * 32 + x > lim_col) v = -INFINITY;
          mx = fmaxf(mx, v);
        }
      }
      const float m_new = fmaxf(m_used, mx);
      if (j == 0) {
        m_used = m_new;
      } else {
        const bool grow = m_new > m_used + kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {                  // PV(j-1) has completed: S(j) was committed after it
          const float f = grow ? ex2(m_used - m_new) : 1.f;
          if (grow) m_used = m_new;
          l_run *= f;
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t rr[32];
            ptx::tmem_ld32(tO + c * 32, rr);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int x = 0; x < 32; ++x) rr[x] = __float_as_uint(__uint_as_float(rr[x]) * f);
            ptx::tmem_st32(tO + c * 32, rr);
          }
          ptx::tmem_wait_st();
        }
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t rr[32], pk[16];
        ptx::tmem_ld32(tS + c * 32, rr);
        ptx::tmem_wait_ld();
#pragma unroll
        for (int x = 0; x < 16; ++x) {
          float v0 = __uint_as_float(rr[2 * x]), v1 = __uint_as_float(rr[2 * x + 1]);
          if (need_mask && c * 32 + 2 * x > lim_col) v0 = -INFINITY;
          if (need_mask && c * 32 + 2 * x + 1 > lim_col) v1 = -INFINITY;
          const float p0 = ex2(v0 - m_used), p1 = ex2(v1 - m_used);
          l_run += p0 + p1;
          pk[x] = ptx::pack_bf16(p0, p1);
        }
        ptx::tmem_st16(tS + c * 16, pk);                      // P over the already-consumed part of S
      }
      ptx::tmem_wait_st();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar(B_PREADY + t));
    }

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
          o.x = ptx::pack_bf16(__uint_as_float(rr[8 * x + 0]) * inv, __uint_as_float(rr[8 * x + 1]) * inv);
          o.y = ptx::pack_bf16(__uint_as_float(rr[8 * x + 2]) * inv, __uint_as_float(rr[8 * x + 3]) * inv);
          o.z = ptx::pack_bf16(__uint_as_float(rr[8 * x + 4]) * inv, __uint_as_float(rr[8 * x + 5]) * inv);
          o.w = ptx::pack_bf16(__uint_as_float(rr[8 * x + 6]) * inv, __uint_as_float(rr[8 * x + 7]) * inv);
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

template <int D>
static int launch_prefill_t(const lazy_handle* h, const PrefillArgs& args, int grid, cudaStream_t stream) {
  using C = PrefillCfg<D>;
  static bool attr_set = false;
  auto kern = prefill_umma_kernel<D>;
  if (!attr_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess)
      return LAZY_ERR_CUDA;
    attr_set = true;
  }
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
  if (h->tmap_pk_ptr != k_cache) {
    if (!encode_pool_tmap(h->tmap_pk, k_cache, rows, c.head_dim, kPageSize)) return LAZY_ERR_CUDA;
    h->tmap_pk_ptr = k_cache;
  }
  if (h->tmap_pv_ptr != v_cache) {
    if (!encode_pool_tmap(h->tmap_pv, v_cache, rows, c.head_dim, kPageSize)) return LAZY_ERR_CUDA;
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
  a.num_reqs = num_reqs;
  a.mblocks = (max_q_len + 2 * tpt - 1) / (2 * tpt);
  a.tokens_per_tile = tpt;
  a.sh = h->shape;
  const long long grid = (long long)a.mblocks * c.num_kv_heads * num_reqs;
  if (grid <= 0 || grid > INT_MAX) return LAZY_ERR_INVALID;
  return c.head_dim == 128 ? launch_prefill_t<128>(h, a, (int)grid, stream)
                           : launch_prefill_t<64>(h, a, (int)grid, stream);
}

}  // namespace lazy
