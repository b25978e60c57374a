// prefill_common.cuh -- pieces shared by the two prefill kernels (prefill_umma.cu: one CTA per tile pair;
// prefill_umma2.cu: CTA pairs with tcgen05 cta_group::2): kernel arguments, the 128B-swizzled tile addressing,
// the cos/sin table chunk order and the fp32 rotation of 8 pairs.
#pragma once
#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {

struct PrefillArgs {
  const int* block_table;
  const int* page_pos;
  const int* seq_lens;
  const int* cu_q_lens;
  __nv_bfloat16* out;
  const float2* cs;
  const int* stored_pos;   // LAZY_K_STORED_POS: [num_pages] position each physical page was stored at
  const float* alibi;      // kKmAlibi: [Hq] slopes * log2(e)
  const float* k_scale;    // LAZY_KV_FP8_E4M3: [num_pages][Hkv][16] per-row scales of the code pools
  const float* v_scale;
  int num_reqs;
  int q_interleaved;    // LAZY_ROPE_INTERLEAVED: q arrives with pairs (2j, 2j+1); de-interleaved while it is rotated
  int mblocks;          // CTAs (pair kernel: CTA pairs) per (request, kv head)
  int tokens_per_tile;  // 128 / group
  Shape sh;
};

// prefill_umma2.cu: head_dim 128 on CTA pairs; `a.mblocks` counts pairs per (request, kv head), `grid` = 2 CTAs per pair
int launch_prefill_pair(const lazy_handle* h, const PrefillArgs& a, int km, int grid, cudaStream_t stream);

namespace {

constexpr int kPrefillThreads = 512;
constexpr int kTileRows = 128;          // rows of a Q tile == keys of a KV tile
constexpr int kHalfBytes = kTileRows * 128;   // one 64-column (128-byte) slab of a 128-row tile
constexpr int kPagesPerTile = kTileRows / kPageSize;

// register budgets per warpgroup (setmaxnreg; 2*128*184 + 128*104 + 128*40 = 65536)
constexpr int kRegsSoftmax = 184, kRegsRotate = 104, kRegsMisc = 40;


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

// Index (in 16-byte units) inside a table row of the chunk holding (cos j, cos j+1, sin j, sin j+1), j = 8c + 2x
// (row layout: cs_cos_index in ptx_util.cuh).
template <int D>
__device__ __forceinline__ int cs_f4_index(int c, int x) {
  constexpr int JT = D / 8;
  const int j0 = 8 * c;
  return ((j0 % JT) / 2 + x) * 4 + j0 / JT;
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

}  // namespace
}  // namespace lazy
