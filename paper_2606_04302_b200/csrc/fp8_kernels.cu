// fp8_kernels.cu -- LAZY_KV_FP8_E4M3 pages: the quantising lazy_cache_write and the simple
// row-wise attention kernel over FP8 pages (LAZY_FLAG_ROWWISE_KERNELS debugging path).
//
// Format (include/lazy_attn.h): a page holds OCP FP8 E4M3 codes of the un-rotated K row / of the V row
// divided by one fp32 scale per (page, kv head, token).  Still "purely content-based keys and values":
// nothing position-dependent is stored, so a quantised page is reusable at any logical offset.
//
//  * cache_write_fp8 : one warp per (token, kv head, K or V) row.  amax by warp shuffles, scale = amax / 448 and the
//    quotients x / scale with IEEE fp32 division (__fdiv_rn), codes by cvt.rn.satfinite.e4m3x2.f32 -- the decisions
//    that produce integers are taken in fp32 exactly as the oracle states them, so codes and scales are bit-exact.
//  * rowwise_attn_fp8 : basic_kernels.cu's row-wise kernel reading dequantised elements (code value x scale).
#include <cuda_fp8.h>

#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {

namespace {

__device__ __forceinline__ float e4m3_to_float(uint8_t c) {
  const __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)c, __NV_E4M3);   // exact: e4m3 is a subset of f16
  return __half2float(*reinterpret_cast<const __half*>(&h));
}

template <int D>
__global__ void __launch_bounds__(256)
cache_write_fp8_kernel(const __nv_bfloat16* __restrict__ k_new, const __nv_bfloat16* __restrict__ v_new,
                       const long long* __restrict__ slot_mapping, long long num_rows, int Hkv, int deinterleave,
                       uint8_t* __restrict__ k_codes, uint8_t* __restrict__ v_codes, float* __restrict__ k_scale,
                       float* __restrict__ v_scale) {
  constexpr int PER = D / 32;                       // elements per lane: 4 (D = 128) or 2 (D = 64)
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= num_rows) return;
  const int which = (int)(w & 1);                   // 0 = K, 1 = V
  const long long row = w >> 1;
  const int head = (int)(row % Hkv);
  const long long tok = row / Hkv;
  const long long slot = slot_mapping[tok];
  if (slot < 0) return;
  const long long page = slot / kPageSize;
  const int off = (int)(slot % kPageSize);
  const __nv_bfloat16* src = (which ? v_new : k_new) + (tok * Hkv + head) * D + lane * PER;
  float x[PER];
  if (deinterleave && which == 0) {
    // LAZY_ROPE_INTERLEAVED: stored dim d' < D/2 is model dim 2d', stored dim D/2 + d' is model dim 2d' + 1 (the row's
    // values, hence its scale, are the same set: still position-free)
    const __nv_bfloat16* rowp = k_new + (tok * Hkv + head) * D;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
      const int d = lane * PER + i;
      x[i] = __bfloat162float(rowp[d < D / 2 ? 2 * d : 2 * (d - D / 2) + 1]);
    }
  } else if (PER == 4) {
    const uint2 v = *reinterpret_cast<const uint2*>(src);
    x[0] = ptx::bf16_lo(v.x); x[1] = ptx::bf16_hi(v.x); x[PER - 2] = ptx::bf16_lo(v.y); x[PER - 1] = ptx::bf16_hi(v.y);
  } else {
    const uint32_t v = *reinterpret_cast<const uint32_t*>(src);
    x[0] = ptx::bf16_lo(v); x[1] = ptx::bf16_hi(v);
  }
  float amax = 0.f;
#pragma unroll
  for (int i = 0; i < PER; ++i) amax = fmaxf(amax, fabsf(x[i]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  float scale = __fdiv_rn(amax, 448.f);
  if (!(scale > 0.f)) scale = 1.f;
  const long long srow = (page * Hkv + head) * kPageSize + off;
  uint8_t* dst = (which ? v_codes : k_codes) + srow * D + lane * PER;
  uint32_t packed = 0;
#pragma unroll
  for (int i = 0; i < PER; i += 2) {
    const float2 y = make_float2(__fdiv_rn(x[i], scale), __fdiv_rn(x[i + 1], scale));
    packed |= (uint32_t)__nv_cvt_float2_to_fp8x2(y, __NV_SATFINITE, __NV_E4M3) << (8 * i);
  }
  if (PER == 4) *reinterpret_cast<uint32_t*>(dst) = packed;
  else *reinterpret_cast<uint16_t*>(dst) = (uint16_t)packed;
  if (lane == 0) (which ? v_scale : k_scale)[srow] = scale;
}

// Row-wise attention over FP8 pages (debug path): PER = D/64 rotation pairs per lane, lane owns j = lane*PER + i.
template <int D>
__global__ void __launch_bounds__(128)
rowwise_attn_fp8_kernel(const __nv_bfloat16* __restrict__ q, const uint8_t* __restrict__ k_codes,
                        const uint8_t* __restrict__ v_codes, const float* __restrict__ k_scale,
                        const float* __restrict__ v_scale, const int* __restrict__ block_table,
                        const int* __restrict__ page_pos, const int* __restrict__ seq_lens,
                        const int* __restrict__ cu_q_lens, int num_reqs, Shape sh, const float2* __restrict__ cs,
                        int q_interleaved, __nv_bfloat16* __restrict__ out) {
  constexpr int HALF = D / 2;
  constexpr int PER = D / 64;
  const int row = blockIdx.x;
  const int hq = blockIdx.y;
  const int hk = hq / sh.group;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int r, i, n_q;
  if (cu_q_lens == nullptr) { r = row; i = 0; n_q = 1; }
  else {
    int lo = 0, hi = num_reqs;
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (cu_q_lens[mid] <= row) lo = mid; else hi = mid; }
    r = lo; i = row - cu_q_lens[r]; n_q = cu_q_lens[r + 1] - cu_q_lens[r];
    if (row >= cu_q_lens[num_reqs]) return;
  }
  const int L = seq_lens[r];
  __nv_bfloat16* o_ptr = out + ((size_t)row * sh.Hq + hq) * D;
  if (L <= 0) {
    for (int d = threadIdx.x; d < D; d += blockDim.x) o_ptr[d] = __float2bfloat16(0.f);
    return;
  }
  const int sq = L - n_q + i;
  const int* bt = block_table + (size_t)r * sh.table_stride;
  const int* pp = page_pos + (size_t)r * sh.table_stride;
  const int pos_q = pp[sq / kPageSize] + sq % kPageSize;
  float q1[PER], q2[PER];
  {
    const __nv_bfloat16* qp = q + ((size_t)row * sh.Hq + hq) * D;
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      int j = lane * PER + e;
      float a = __bfloat162float(qp[q_interleaved ? 2 * j : j]);
      float b = __bfloat162float(qp[q_interleaved ? 2 * j + 1 : j + HALF]);
      float2 t = cs_load(cs + (size_t)pos_q * HALF, j, D);
      q1[e] = (a * t.x - b * t.y) * sh.scale_log2;
      q2[e] = (a * t.y + b * t.x) * sh.scale_log2;
    }
  }
  float m = -INFINITY, l = 0.f, o1[PER], o2[PER];
#pragma unroll
  for (int e = 0; e < PER; ++e) { o1[e] = 0.f; o2[e] = 0.f; }
  for (int s = warp; s <= sq; s += 4) {
    const int slot = s / kPageSize, t = s % kPageSize;
    const int page = bt[slot];
    const int pos = pp[slot] + t;
    const size_t srow = ((size_t)page * sh.Hkv + hk) * kPageSize + t;
    const size_t base = srow * D;
    const float sk = k_scale[srow], sv = v_scale[srow];
    float dot = 0.f, v1[PER], v2[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      int j = lane * PER + e;
      float a = e4m3_to_float(k_codes[base + j]) * sk, b = e4m3_to_float(k_codes[base + j + HALF]) * sk;
      float2 tcs = cs_load(cs + (size_t)pos * HALF, j, D);
      dot += q1[e] * (a * tcs.x - b * tcs.y) + q2[e] * (a * tcs.y + b * tcs.x);
      v1[e] = e4m3_to_float(v_codes[base + j]) * sv;
      v2[e] = e4m3_to_float(v_codes[base + j + HALF]) * sv;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
    float m_new = fmaxf(m, dot);
    float corr = exp2f(m - m_new);
    float p = exp2f(dot - m_new);
    l = l * corr + p;
#pragma unroll
    for (int e = 0; e < PER; ++e) { o1[e] = o1[e] * corr + p * v1[e]; o2[e] = o2[e] * corr + p * v2[e]; }
    m = m_new;
  }
  __shared__ float sm_m[4], sm_l[4], sm_o[4][D];
  if (lane == 0) { sm_m[warp] = m; sm_l[warp] = l; }
#pragma unroll
  for (int e = 0; e < PER; ++e) { sm_o[warp][lane * PER + e] = o1[e]; sm_o[warp][lane * PER + e + HALF] = o2[e]; }
  __syncthreads();
  float mm = fmaxf(fmaxf(sm_m[0], sm_m[1]), fmaxf(sm_m[2], sm_m[3]));
  float w[4], lsum = 0.f;
#pragma unroll
  for (int k = 0; k < 4; ++k) { w[k] = (sm_m[k] == -INFINITY) ? 0.f : exp2f(sm_m[k] - mm); lsum += w[k] * sm_l[k]; }
  for (int d = threadIdx.x; d < D; d += blockDim.x) {
    float acc = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc += w[k] * sm_o[k][d];
    o_ptr[d] = __float2bfloat16(acc / lsum);
  }
}

}  // namespace

int launch_cache_write_fp8(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                           int num_tokens, void* k_cache, void* v_cache, cudaStream_t stream) {
  const long long rows = 2LL * num_tokens * h->cfg.num_kv_heads;
  const int threads = 256;
  const long long blocks = (rows * 32 + threads - 1) / threads;
  auto kn = static_cast<const __nv_bfloat16*>(k_new);
  auto vn = static_cast<const __nv_bfloat16*>(v_new);
  auto sm = reinterpret_cast<const long long*>(slot_mapping);
  auto kc = static_cast<uint8_t*>(k_cache);
  auto vc = static_cast<uint8_t*>(v_cache);
  const int deint = h->cfg.rope_style == LAZY_ROPE_INTERLEAVED;
  if (h->cfg.head_dim == 128)
    cache_write_fp8_kernel<128><<<(unsigned)blocks, threads, 0, stream>>>(kn, vn, sm, rows, h->cfg.num_kv_heads, deint, kc, vc,
                                                                          h->k_scale, h->v_scale);
  else
    cache_write_fp8_kernel<64><<<(unsigned)blocks, threads, 0, stream>>>(kn, vn, sm, rows, h->cfg.num_kv_heads, deint, kc, vc,
                                                                         h->k_scale, h->v_scale);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

int launch_rowwise_fp8(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                       const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                       const int32_t* cu_q_lens, int num_reqs, int total_q, void* out, cudaStream_t stream) {
  dim3 grid(total_q, h->cfg.num_q_heads);
  auto qp = static_cast<const __nv_bfloat16*>(q);
  auto kp = static_cast<const uint8_t*>(k_cache);
  auto vp = static_cast<const uint8_t*>(v_cache);
  auto op = static_cast<__nv_bfloat16*>(out);
  if (h->cfg.head_dim == 128)
    rowwise_attn_fp8_kernel<128><<<grid, 128, 0, stream>>>(qp, kp, vp, h->k_scale, h->v_scale, block_table,
                                                           page_logical_pos, seq_lens, cu_q_lens, num_reqs, h->shape,
                                                           h->ws.cs, h->cfg.rope_style == LAZY_ROPE_INTERLEAVED, op);
  else
    rowwise_attn_fp8_kernel<64><<<grid, 128, 0, stream>>>(qp, kp, vp, h->k_scale, h->v_scale, block_table,
                                                          page_logical_pos, seq_lens, cu_q_lens, num_reqs, h->shape,
                                                          h->ws.cs, h->cfg.rope_style == LAZY_ROPE_INTERLEAVED, op);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

}  // namespace lazy
