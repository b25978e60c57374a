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

// Optional timeline probe (compile with -DLAZY_TRACE): one mid-grid CTA records clock64() at the hand-offs of 16
// consecutive KV iterations into a device array read back by lazy_debug_trace().  Off in the product build.
#ifdef LAZY_TRACE
__device__ long long g_trace[16 * 16];
#define LAZY_TR(slot) do { if (blockIdx.x == 300 && j >= 10 && j < 26) g_trace[(j - 10) * 16 + (slot)] = clock64(); } while (0)
#else
#define LAZY_TR(slot) do { } while (0)
#endif

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
  static constexpr int NUM_BARS = 24;
  static constexpr int OFF_TMEM = OFF_BAR + NUM_BARS * 8;
  static constexpr int OFF_SIGN = OFF_TMEM + 16;    // ring of 4 tiles x 8 pages: sign of the page's relative offset
                                                    // (LAZY_K_STORED_POS) or its logical start (ALiBi)
  static constexpr int SMEM_BYTES = OFF_SIGN + 4 * kPagesPerTile * 4 + 1024;   // + alignment slack
};

// register budgets per warpgroup (setmaxnreg; 2*128*184 + 128*104 + 128*40 = 65536)
constexpr int kRegsSoftmax = 184, kRegsRotate = 104, kRegsMisc = 40;

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
  B_SFULL = 16,   // +t   MMA commit -> softmax WG t
  B_PREADY = 18,  // +t   softmax WG t (4 warps) -> MMA
  B_OFULL = 20,   // +t   MMA commit -> softmax WG t (epilogue)
  B_PHALF = 22,   // +t   softmax WG t (4 warps) -> MMA: first half of P (keys 0..63) is in TMEM
};

struct PrefillArgs {
  const int* block_table;
  const int* page_pos;
  const int* seq_lens;
  const int* cu_q_lens;
  __nv_bfloat16* out;
  const float2* cs;
  const int* stored_pos;   // LAZY_K_STORED_POS: [num_pages] position each physical page was stored at
  const float* alibi;      // kKmAlibi: [Hq] slopes * log2(e)
  const unsigned char* k_pool;   // raw pool pointers: only the L2 prefetch warp uses them (loads go through TMA)
  const unsigned char* v_pool;
  int num_reqs;
  int q_interleaved;    // LAZY_ROPE_INTERLEAVED: q arrives with pairs (2j, 2j+1); de-interleaved while it is rotated
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
__device__ __forceinline__ float f32(uint32_t x) { return __uint_as_float(x); }

// 2^x for a PAIR of elements on the FMA pipe instead of the MUFU (ex2.approx runs at 16/clk/SM and is as loaded as
// the tensor pipe in this kernel): Cody-Waite split x = floor(x) + f with a round-down magic-number
// add, degree-3 polynomial for 2^f on [0,1) (max relative error 8.8e-5, far inside P's bf16 rounding 2^-9), exponent
// inserted with one integer shift-add.  x is clamped to >= -126 (covers -inf of masked columns: result 2^-126 ~ 0).
// Softmax ping-pong (FA3-style named-barrier hand-off between the two softmax warpgroups): 0 = free running,
// 1 = the whole softmax of a tile is exclusive, 2 = only the exponential phase is exclusive.
#ifndef LAZY_PINGPONG
#define LAZY_PINGPONG 2
#endif
// L2 prefetch distance in KV tiles (warp 15; 0 = off: measured 2-4 % slower at 1-3 tiles)
#ifndef LAZY_L2_AHEAD
#define LAZY_L2_AHEAD 0
#endif
#ifndef LAZY_POLY_EVERY
#define LAZY_POLY_EVERY 0   // every LAZY_POLY_EVERY-th group of 4 columns takes this path (0 = never: measured slower)
#endif
__device__ __forceinline__ float2 ex2_poly2(float2 v) {
  v.x = fmaxf(v.x, -126.f);
  v.y = fmaxf(v.y, -126.f);
  unsigned long long vv, rr;
  asm("mov.b64 %0, {%1, %2};" : "=l"(vv) : "f"(v.x), "f"(v.y));
  asm("add.rm.ftz.f32x2 %0, %1, %2;" : "=l"(rr) : "l"(vv), "l"(0x4b4000004b400000ull));   // + 1.5 * 2^23, round down
  float2 xr;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(xr.x), "=f"(xr.y) : "l"(rr));
  const float2 fl = __fadd2_rn(xr, make_float2(-12582912.f, -12582912.f));               // floor(x)
  const float2 f = __ffma2_rn(fl, make_float2(-1.f, -1.f), v);                           // x - floor(x) in [0, 1)
  float2 p = __ffma2_rn(make_float2(0.077119089663028717f, 0.077119089663028717f), f,
                        make_float2(0.227564394474029541f, 0.227564394474029541f));
  p = __ffma2_rn(p, f, make_float2(0.695146143436431885f, 0.695146143436431885f));
  p = __ffma2_rn(p, f, make_float2(1.f, 1.f));
  return make_float2(__int_as_float(__float_as_int(p.x) + (__float_as_int(xr.x) << 23)),
                     __int_as_float(__float_as_int(p.y) + (__float_as_int(xr.y) << 23)));
}

// Index (in 16-byte units) inside a table row of the chunk holding (cos j, cos j+1, sin j, sin j+1), j = 8c + 2x
// (row layout: cs_cos_index in ptx_util.cuh).
template <int D>
__device__ __forceinline__ int cs_f4_index(int c, int x) {
  constexpr int JT = D / 8;
  const int j0 = 8 * c;
  return ((j0 % JT) / 2 + x) * 4 + j0 / JT;
}
// (cos, sin) of the 8 rotation pairs j = 8c .. 8c+7 from one table row in global memory / in shared memory.
template <int D>
__device__ __forceinline__ void load_cs8(const float2* __restrict__ cs_row, int c, float (&co)[8], float (&si)[8]) {
  const float4* p = reinterpret_cast<const float4*>(cs_row);
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    float4 v = __ldg(p + cs_f4_index<D>(c, x));
    co[2 * x] = v.x; co[2 * x + 1] = v.y; si[2 * x] = v.z; si[2 * x + 1] = v.w;
  }
}
template <int D>
__device__ __forceinline__ void load_cs8_smem(uint32_t row_addr, int c, float (&co)[8], float (&si)[8]) {
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    uint4 v = ptx::lds128(row_addr + 16 * cs_f4_index<D>(c, x));
    co[2 * x] = f32(v.x); co[2 * x + 1] = f32(v.y); si[2 * x] = f32(v.z); si[2 * x + 1] = f32(v.w);
  }
}

// byte offset of 16-byte chunk `ci` (8 dims: 8ci .. 8ci+7) of row `row` inside a 128-row, 128B-swizzled tile
__device__ __forceinline__ uint32_t chunk_off(int row, int ci) {
  return (ci >> 3) * kHalfBytes + row * 128 + (((ci & 7) ^ (row & 7)) << 4);
}

// rotate 8 pairs held as two 16-byte chunks (x1 = dims j, x2 = dims j + D/2) by (co, si), round to bf16
__device__ __forceinline__ void rotate8(uint4& a, uint4& b, const float (&co)[8], const float (&si)[8]) {
  uint32_t* aw = reinterpret_cast<uint32_t*>(&a);
  uint32_t* bw = reinterpret_cast<uint32_t*>(&b);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float a0 = ptx::bf16_lo(aw[w]), a1 = ptx::bf16_hi(aw[w]);
    float b0 = ptx::bf16_lo(bw[w]), b1 = ptx::bf16_hi(bw[w]);
    aw[w] = ptx::pack_bf16(a0 * co[2 * w] - b0 * si[2 * w], a1 * co[2 * w + 1] - b1 * si[2 * w + 1]);
    bw[w] = ptx::pack_bf16(a0 * si[2 * w] + b0 * co[2 * w], a1 * si[2 * w + 1] + b1 * co[2 * w + 1]);
  }
}

// KM = lazy_config.k_storage.  LAZY_K_UNROTATED: K tile rotated by the absolute angle of its tokens.
// LAZY_K_STORED_POS (Eq. 5): K tile rotated once by the page's relative offset
// D = p0 - stored[page] (one table row per page, no in-page composition).  LAZY_K_ABSOLUTE: the K tile goes to
// the MMA as it landed (the "rotation compiled out" arm of the overhead ablation, Fig. 5).  kKmAlibi
// (PAPER.md L221): nothing is rotated; the softmax warpgroups add slope[head] * (n - m) to S, with the key position
// n = page start + t taken from a small per-tile ring the producer fills.
// Same rotation on packed f32x2 lanes (FMUL2 / FFMA2: half the FMA-pipe issue slots).  zc[w], zs[w] hold the
// (cos, sin) of the two pairs whose x1 / x2 elements are the bf16 halves of word w of a / b.
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }
__device__ __forceinline__ void rotate8_packed(uint4& a, uint4& b, const float2 (&zc)[4], const float2 (&zs)[4]) {
  uint32_t* aw = reinterpret_cast<uint32_t*>(&a);
  uint32_t* bw = reinterpret_cast<uint32_t*>(&b);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const float2 x1 = make_float2(ptx::bf16_lo(aw[w]), ptx::bf16_hi(aw[w]));
    const float2 x2 = make_float2(ptx::bf16_lo(bw[w]), ptx::bf16_hi(bw[w]));
    const float2 y1 = __ffma2_rn(neg2(x2), zs[w], __fmul2_rn(x1, zc[w]));
    const float2 y2 = __ffma2_rn(x2, zc[w], __fmul2_rn(x1, zs[w]));
    aw[w] = ptx::pack_bf16(y1.x, y1.y);
    bw[w] = ptx::pack_bf16(y2.x, y2.y);
  }
}

template <int D, int KM>
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
      ptx::mbar_init(bar(B_PHALF + x), 4);
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
        if (lane == 0)
          ptx::mbar_arrive_expect_tx(bar(B_KFULL + s), npv * (C::NH * kPageSize * 128 +
                                                              (kNoRotate ? 0 : C::CS_ROW_BYTES)));
        __syncwarp();
        if (kvsel == 0 && lane_on && pg < npv) {
          ptx::tma_load_2d(sK + dst, &tmap_k, bar(B_KFULL + s), half * 64, row0);
          if (half == 0 && !kNoRotate)
            ptx::bulk_load_1d(sCS + s * C::CS_STAGE_BYTES + pg * C::CS_ROW_BYTES, a.cs + (size_t)p0 * (D / 2),
                              C::CS_ROW_BYTES, bar(B_KFULL + s));
        }
        ptx::mbar_wait_sleep(bar(B_VEMPTY + s), ph ^ 1);
        if (lane == 0) ptx::mbar_arrive_expect_tx(bar(B_VFULL + s), npv * C::NH * kPageSize * 128);
        __syncwarp();
        if (kvsel == 1 && lane_on && pg < npv) ptx::tma_load_2d(sV + dst, &tmap_v, bar(B_VFULL + s), half * 64, row0);
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
        ptx::mbar_wait(bar(B_VFULL + s), (j >> 1) & 1);
        if (j == nkv - 1) ptx::mbar_wait(bar(B_VFIXED), 0);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          // PV starts on the first 64 keys while the softmax warpgroup is still exponentiating the other 64
          ptx::mbar_wait(bar(B_PHALF + t), j & 1);
          ptx::tc_fence_after();
          pv(t, s, j > 0, 0, kTileRows / 32);
          ptx::mbar_wait(bar(B_PREADY + t), j & 1);
          ptx::tc_fence_after();
          if (leader) LAZY_TR(8 + 3 * t);
          pv(t, s, 1u, kTileRows / 32, kTileRows / 16);
          if (t == 1) commit(B_VEMPTY + s);
          if (j + 1 < nkv) {
            if (t == 0) {
              ptx::mbar_wait(bar(B_KREADY + (s ^ 1)), ((j + 1) >> 1) & 1);
              ptx::tc_fence_after();
              if (leader) LAZY_TR(9);
            }
            qk(t, s ^ 1);
            commit(B_SFULL + t);
            if (leader) LAZY_TR(10 + 3 * t);
            if (t == 1) commit(B_KEMPTY + (s ^ 1));
          } else {
            commit(B_OFULL + t);
          }
        }
      }
      __syncwarp();
    } else if (warp == 14) {
      // ================================ V tail fixer ========================================================
      for (int j = 0; j < n_kv; ++j) ptx::mbar_wait_sleep(bar(B_VFULL + (j & 1)), (j >> 1) & 1);
      const int jl = n_kv - 1;
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
    } else if (LAZY_L2_AHEAD > 0) {
      // ================================ L2 prefetcher (warp 15) =============================================
      // touches the K and V pages of tile j + LAZY_L2_AHEAD with plain prefetch instructions (LSU path, not the
      // TMA unit), throttled by the arrival of tile j, so that the TMA gather of a freed stage hits the L2
      const int pgi = lane & 7, part = lane >> 3;   // lane -> (page of the tile, K lo / K hi / V lo / V hi half)
      constexpr int kHalfPage = kPageSize * D;      // bytes of half a (page, head) tile
      for (int j = 0; j < n_kv; ++j) {
        const int idx = (j + LAZY_L2_AHEAD) * kPagesPerTile + pgi;
        if (j + LAZY_L2_AHEAD < n_kv && idx < num_pages) {
          const unsigned char* p = (part < 2 ? a.k_pool : a.v_pool) +
                                   ((size_t)bt[idx] * sh.Hkv + hk) * (2 * kHalfPage) + (part & 1) * kHalfPage;
#pragma unroll
          for (int l = 0; l < kHalfPage / 128; ++l)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p + 128 * l));
        }
        ptx::mbar_wait_sleep(bar(B_KFULL + (j & 1)), (j >> 1) & 1);
      }
    }
  } else if (warp >= 8) {
    // ================================ K-rotate warpgroup ======================================================
    ptx::setmaxnreg_dec<kRegsRotate>();
    constexpr int TPP = 16 * C::CPR;                // threads per page
    constexpr int PPP = 128 / TPP;                  // pages per pass
    constexpr int PASSES = kPagesPerTile / PPP;
    const int wtid = tid - 256;
    const int pp_ = wtid / TPP, t = (wtid % TPP) / C::CPR, c = wtid % C::CPR;
    float2 uc[4], us[4];                            // e^{i t theta_j}: in-page offset, fixed per thread
    if (KM == LAZY_K_UNROTATED) {
      const float4* urow = reinterpret_cast<const float4*>(a.cs + (size_t)t * (D / 2));
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const float4 v = __ldg(urow + cs_f4_index<D>(c, x));
        uc[x] = make_float2(v.x, v.y);
        us[x] = make_float2(v.z, v.w);
      }
    }
    const int* s_sign = reinterpret_cast<const int*>(smem + C::OFF_SIGN);
    for (int j = 0; j < n_kv; ++j) {
      const int s = j & 1;
      const int npv = min(kPagesPerTile, num_pages - j * kPagesPerTile);
      const uint32_t kb = sK + s * C::TILE_BYTES;
      const uint32_t cb = sCS + s * C::CS_STAGE_BYTES;
      ptx::mbar_wait(bar(B_KFULL + s), (j >> 1) & 1);
      if (wtid == 0) LAZY_TR(6);
#pragma unroll
      for (int ps = 0; ps < PASSES; ++ps) {
        const int i = ps * PPP + pp_;
        if (!kNoRotate && i < npv) {
          float2 zc[4], zs[4];                      // e^{i (p0+t) theta_j}, or e^{i Delta theta_j} of the page
          const int row = i * kPageSize + t;
          const uint32_t pa = kb + chunk_off(row, c), pb = kb + chunk_off(row, c + C::CPR);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint4 v = ptx::lds128(cb + i * C::CS_ROW_BYTES + 16 * cs_f4_index<D>(c, x));
            zc[x] = make_float2(f32(v.x), f32(v.y));
            zs[x] = make_float2(f32(v.z), f32(v.w));
          }
          uint4 va = ptx::lds128(pa), vb = ptx::lds128(pb);
          if (KM == LAZY_K_UNROTATED) {             // compose with the in-page offset: z = w * u
#pragma unroll
            for (int x = 0; x < 4; ++x) {
              const float2 wc = zc[x], ws = zs[x];
              zc[x] = __ffma2_rn(neg2(ws), us[x], __fmul2_rn(wc, uc[x]));
              zs[x] = __ffma2_rn(wc, us[x], __fmul2_rn(ws, uc[x]));
            }
          } else {                                  // one relative rotation for the whole page (may be negative)
            const float sgn = (float)s_sign[(j & 3) * kPagesPerTile + i];
#pragma unroll
            for (int x = 0; x < 4; ++x) zs[x] = __fmul2_rn(zs[x], make_float2(sgn, sgn));
          }
          rotate8_packed(va, vb, zc, zs);
          ptx::sts128(pa, va);
          ptx::sts128(pb, vb);
        }
      }
      ptx::fence_proxy_async();
      __syncwarp();
      if (wtid == 0) LAZY_TR(7);
      if (lane == 0) ptx::mbar_arrive(bar(B_KREADY + s));
    }
  } else {
    // ================================ softmax warpgroups ======================================================
    ptx::setmaxnreg_inc<kRegsSoftmax>();
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
      const uint32_t qb = sQ + t * C::TILE_BYTES;
      if (valid) {
        const int pos = ppos[sq / kPageSize] + sq % kPageSize;
        const float2* cs_row = a.cs + (size_t)pos * (D / 2);
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
            load_cs8<D>(cs_row, c, co, si);
#pragma unroll
            for (int e = 0; e < 8; ++e) { co[e] *= sh.scale_log2; si[e] *= sh.scale_log2; }
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
    float m_used = -INFINITY, l_run = 0.f;
    if (LAZY_PINGPONG && t == 1) ptx::named_bar_arrive(2, 256);          // tile 0 goes first
    for (int j = 0; j < n_kv; ++j) {
      uint32_t sreg[128];                                     // this row of S (fp32 bits), later packed P
      ptx::mbar_wait(bar(B_SFULL + t), j & 1);
      if (LAZY_PINGPONG == 1) ptx::named_bar_sync(2 + t, 256);             // my turn
      ptx::tc_fence_after();
      if (row == 0) LAZY_TR(3 * t);
      float abase[kPagesPerTile];                             // kKmAlibi: slope * (page start - m) of the tile's pages
      float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
      auto max_chunk = [&](int c) {                           // running row max over columns 32c .. 32c+31
#pragma unroll
        for (int x = 32 * c; x < 32 * c + 32; x += 8) {
          mx0 = fmaxf(fmaxf(mx0, f32(sreg[x + 0])), f32(sreg[x + 1]));
          mx1 = fmaxf(fmaxf(mx1, f32(sreg[x + 2])), f32(sreg[x + 3]));
          mx2 = fmaxf(fmaxf(mx2, f32(sreg[x + 4])), f32(sreg[x + 5]));
          mx3 = fmaxf(fmaxf(mx3, f32(sreg[x + 6])), f32(sreg[x + 7]));
        }
      };
      const bool edge = j * kTileRows + kTileRows - 1 > lim_min;   // tile touches the causal edge / the tail: rare
      if (KM != kKmAlibi && !edge) {
        // interior tile: the TMEM load of chunk c+1 is in flight while the max of chunk c is taken
        ptx::tmem_ld32(tS, sreg);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          ptx::tmem_wait_ld();
          if (c + 1 < 4) ptx::tmem_ld32(tS + (c + 1) * 32, sreg + (c + 1) * 32);
          max_chunk(c);
        }
      } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) ptx::tmem_ld32(tS + c * 32, sreg + c * 32);
        ptx::tmem_wait_ld();
        if (KM == kKmAlibi) {
          // S += slope * (n - m), n = page start + t: only the in-page part slope * t is added to the elements
          // (one packed add per pair); the per-page part abase[page] = slope * (page start - m) is folded into the
          // page maxima below and into the constant of the exponential
          const int* pstart = reinterpret_cast<const int*>(smem + C::OFF_SIGN) + (j & 3) * kPagesPerTile;
#pragma unroll
          for (int pg = 0; pg < kPagesPerTile; ++pg) {
            abase[pg] = alibi_slope * (float)(pstart[pg] - alibi_pos_q);
#pragma unroll
            for (int x = 0; x < kPageSize; x += 2) {
              const float2 v = __fadd2_rn(make_float2(f32(sreg[16 * pg + x]), f32(sreg[16 * pg + x + 1])),
                                          alibi_d2[x / 2]);
              sreg[16 * pg + x] = __float_as_uint(v.x);
              sreg[16 * pg + x + 1] = __float_as_uint(v.y);
            }
          }
        }
        if (edge) {
          const int lim_col = lim_row - j * kTileRows;        // column visible iff col <= lim_col
#pragma unroll
          for (int x = 0; x < 128; ++x)
            if (x > lim_col) sreg[x] = 0xff800000u;           // -inf replaces the value (NaN-safe)
        }
        if (KM == kKmAlibi) {
#pragma unroll
          for (int pg = 0; pg < kPagesPerTile; ++pg) {
            float a0 = -INFINITY, a1 = -INFINITY;
#pragma unroll
            for (int x = 16 * pg; x < 16 * pg + 16; x += 4) {
              a0 = fmaxf(fmaxf(a0, f32(sreg[x + 0])), f32(sreg[x + 1]));
              a1 = fmaxf(fmaxf(a1, f32(sreg[x + 2])), f32(sreg[x + 3]));
            }
            mx0 = fmaxf(mx0, fmaxf(a0, a1) + abase[pg]);
          }
        } else {
#pragma unroll
          for (int c = 0; c < 4; ++c) max_chunk(c);
        }
      }
      const float m_new = fmaxf(m_used, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)));
      if (j == 0) {
        m_used = m_new;
      } else {
        const bool grow = m_new > m_used + kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {                  // PV(j-1) has completed: S(j) was committed after it
          const float f = grow ? ex2(m_used - m_new) : 1.f;
          if (grow) m_used = m_new;
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
      if (row == 0) LAZY_TR(3 * t + 1);
      if (LAZY_PINGPONG == 2) ptx::named_bar_sync(2 + t, 256);             // my turn on the MUFU
      const float2 negm = make_float2(-m_used, -m_used);
      float2 sum0 = make_float2(0.f, 0.f), sum1 = make_float2(0.f, 0.f);
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
#pragma unroll
        for (int x = 32 * hf; x < 32 * hf + 32; x += 2) {
          const float2 nm = KM == kKmAlibi ? make_float2(abase[x >> 3] - m_used, abase[x >> 3] - m_used) : negm;
          const float2 v0 = __fadd2_rn(make_float2(f32(sreg[2 * x]), f32(sreg[2 * x + 1])), nm);
          const float2 v1 = __fadd2_rn(make_float2(f32(sreg[2 * x + 2]), f32(sreg[2 * x + 3])), nm);
          float2 p0, p1;
          if (LAZY_POLY_EVERY > 0 && (x / 2) % (LAZY_POLY_EVERY > 0 ? LAZY_POLY_EVERY : 1) == LAZY_POLY_EVERY - 1) {
            p0 = ex2_poly2(v0);
            p1 = ex2_poly2(v1);
          } else {
            p0 = make_float2(ex2(v0.x), ex2(v0.y));
            p1 = make_float2(ex2(v1.x), ex2(v1.y));
          }
          sum0 = __fadd2_rn(sum0, p0);
          sum1 = __fadd2_rn(sum1, p1);
          sreg[x] = ptx::pack_bf16(p0.x, p0.y);
          sreg[x + 1] = ptx::pack_bf16(p1.x, p1.y);
        }
        if (hf == 1 && LAZY_PINGPONG) ptx::named_bar_arrive(2 + (t ^ 1), 256);   // the other tile's turn
        ptx::tmem_st32(tS + 32 * hf, sreg + 32 * hf);         // P (bf16 pairs) over the first 64 columns of S
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncwarp();
        if (hf == 0 && lane == 0) ptx::mbar_arrive(bar(B_PHALF + t));
      }
      l_run += (sum0.x + sum0.y) + (sum1.x + sum1.y);
      if (row == 0) LAZY_TR(3 * t + 2);
      if (lane == 0) ptx::mbar_arrive(bar(B_PREADY + t));
    }

    if (LAZY_PINGPONG && t == 0) ptx::named_bar_sync(2, 256);            // consume tile 1's last hand-off
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

template <int D, int KM>
static int launch_prefill_t(const lazy_handle* h, const PrefillArgs& args, int grid, cudaStream_t stream) {
  using C = PrefillCfg<D>;
  static bool attr_set = false;
  auto kern = prefill_umma_kernel<D, KM>;
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

#ifdef LAZY_TRACE
extern "C" int lazy_debug_trace(long long* host_out) {
  return cudaMemcpyFromSymbol(host_out, g_trace, sizeof(long long) * 256) == cudaSuccess ? 0 : -1;
}
#endif

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
  a.stored_pos = h->page_stored_pos;
  a.alibi = h->ws.alibi;
  a.k_pool = static_cast<const unsigned char*>(k_cache);
  a.v_pool = static_cast<const unsigned char*>(v_cache);
  a.num_reqs = num_reqs;
  a.q_interleaved = c.rope_style == LAZY_ROPE_INTERLEAVED;
  a.mblocks = (max_q_len + 2 * tpt - 1) / (2 * tpt);
  a.tokens_per_tile = tpt;
  a.sh = h->shape;
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
