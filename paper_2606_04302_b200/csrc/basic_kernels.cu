// basic_kernels.cu -- RoPE table build, lazy_cache_write, and the simple row-wise attention kernel.
//
//  * build_cs_table : cs[pos][j] = (cos, sin)(pos * theta^(-2j/D)), angles formed and reduced in fp64 so the
//    fp32 table entries are correctly rounded at any position (stateless rotation from the
//    absolute index; L138/L173: cos/sin loaded from a table).
//  * cache_write    : un-rotated K/V rows -> pages, 16-byte vectorised.
//  * rowwise_attn   : one CTA per (query row, q head), keys strided over 4 warps, K rotated by its absolute
//    angle from the table, online softmax.  It follows PAPER.md Eq. 4 (L94-106) directly and is kept as the
//    LAZY_FLAG_ROWWISE_KERNELS debugging path; the production kernels are decode_splitkv.cu / prefill_umma.cu.
#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {

__global__ void build_cs_table_kernel(float2* __restrict__ cs, int max_position, int half, double theta, int D) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)max_position * half;
  if (idx >= total) return;
  int j = (int)(idx % half);
  long long pos = idx / half;
  double inv_freq = pow(theta, -2.0 * (double)j / (double)D);
  double s, c;
  sincos((double)pos * inv_freq, &s, &c);
  cs[pos * half + cs_index(j, D)] = make_float2((float)c, (float)s);
}

int launch_build_tables(lazy_handle* h, cudaStream_t stream) {
  int half = h->cfg.head_dim / 2;
  long long total = (long long)h->cfg.max_position * half;
  int threads = 256;
  long long blocks = (total + threads - 1) / threads;
  build_cs_table_kernel<<<(unsigned)blocks, threads, 0, stream>>>(h->ws.cs, h->cfg.max_position, half,
                                                                 h->cfg.rope_theta, h->cfg.head_dim);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------
// cache write: one thread moves one 16-byte chunk of K and the matching chunk of V.
// chunk index c in [0, T*Hkv*D/8): token = c / (Hkv*D/8), head = (c / (D/8)) % Hkv, part = c % (D/8).
__global__ void cache_write_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                   const long long* __restrict__ slot_mapping, long long num_chunks,
                                   int Hkv, int chunks_per_row, uint4* __restrict__ k_cache,
                                   uint4* __restrict__ v_cache) {
  long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= num_chunks) return;
  int part = (int)(c % chunks_per_row);
  long long row = c / chunks_per_row;
  int head = (int)(row % Hkv);
  long long tok = row / Hkv;
  long long slot = slot_mapping[tok];
  if (slot < 0) return;
  long long page = slot / kPageSize;
  int off = (int)(slot % kPageSize);
  long long dst = (((page * Hkv + head) * kPageSize) + off) * chunks_per_row + part;
  k_cache[dst] = k_new[c];
  v_cache[dst] = v_new[c];
}

int launch_cache_write(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                       int num_tokens, void* k_cache, void* v_cache, cudaStream_t stream) {
  int chunks_per_row = h->cfg.head_dim / 8;
  long long num_chunks = (long long)num_tokens * h->cfg.num_kv_heads * chunks_per_row;
  int threads = 256;
  long long blocks = (num_chunks + threads - 1) / threads;
  cache_write_kernel<<<(unsigned)blocks, threads, 0, stream>>>(
      static_cast<const uint4*>(k_new), static_cast<const uint4*>(v_new),
      reinterpret_cast<const long long*>(slot_mapping), num_chunks, h->cfg.num_kv_heads, chunks_per_row,
      static_cast<uint4*>(k_cache), static_cast<uint4*>(v_cache));
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------
// Row-wise attention (debug path).  PER = D/64 rotation pairs per lane: lane owns j = lane*PER + i.
template <int D>
__global__ void __launch_bounds__(128)
rowwise_attn_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k_cache,
                    const __nv_bfloat16* __restrict__ v_cache, const int* __restrict__ block_table,
                    const int* __restrict__ page_pos, const int* __restrict__ seq_lens,
                    const int* __restrict__ cu_q_lens, int num_reqs, Shape sh, const float2* __restrict__ cs,
                    __nv_bfloat16* __restrict__ out) {
  constexpr int HALF = D / 2;
  constexpr int PER = D / 64;
  const int row = blockIdx.x;
  const int hq = blockIdx.y;
  const int hk = hq / sh.group;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // locate the request of this row
  int r, i, n_q;
  if (cu_q_lens == nullptr) { r = row; i = 0; n_q = 1; }
  else {
    int lo = 0, hi = num_reqs;          // largest r with cu[r] <= row
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
  const int sq = L - n_q + i;           // sequence index of the query token
  const int* bt = block_table + (size_t)r * sh.table_stride;
  const int* pp = page_pos + (size_t)r * sh.table_stride;
  const int pos_q = pp[sq / kPageSize] + sq % kPageSize;

  // rotated query, pre-scaled by log2(e)/sqrt(D)
  float q1[PER], q2[PER];
  {
    const __nv_bfloat16* qp = q + ((size_t)row * sh.Hq + hq) * D;
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      int j = lane * PER + e;
      float a = __bfloat162float(qp[j]), b = __bfloat162float(qp[j + HALF]);
      float2 t = cs[(size_t)pos_q * HALF + cs_index(j, D)];
      q1[e] = (a * t.x - b * t.y) * sh.scale_log2;
      q2[e] = (a * t.y + b * t.x) * sh.scale_log2;
    }
  }
  float m = -INFINITY, l = 0.f, o1[PER], o2[PER];
#pragma unroll
  for (int e = 0; e < PER; ++e) { o1[e] = 0.f; o2[e] = 0.f; }

  for (int s = warp; s <= sq; s += 4) {
    int slot = s / kPageSize, t = s % kPageSize;
    int page = bt[slot];
    int pos = pp[slot] + t;
    size_t base = (((size_t)page * sh.Hkv + hk) * kPageSize + t) * D;
    float dot = 0.f, v1[PER], v2[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      int j = lane * PER + e;
      float a = __bfloat162float(k_cache[base + j]), b = __bfloat162float(k_cache[base + j + HALF]);
      float2 tcs = cs[(size_t)pos * HALF + cs_index(j, D)];
      dot += q1[e] * (a * tcs.x - b * tcs.y) + q2[e] * (a * tcs.y + b * tcs.x);
      v1[e] = __bfloat162float(v_cache[base + j]);
      v2[e] = __bfloat162float(v_cache[base + j + HALF]);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
    float m_new = fmaxf(m, dot);
    float corr = exp2f(m - m_new);       // m = -inf on the first key -> 0
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

int launch_rowwise(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                   const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                   const int32_t* cu_q_lens, int num_reqs, int total_q, int /*max_q_len*/, void* out,
                   cudaStream_t stream) {
  dim3 grid(total_q, h->cfg.num_q_heads);
  auto qp = static_cast<const __nv_bfloat16*>(q);
  auto kp = static_cast<const __nv_bfloat16*>(k_cache);
  auto vp = static_cast<const __nv_bfloat16*>(v_cache);
  auto op = static_cast<__nv_bfloat16*>(out);
  if (h->cfg.head_dim == 128)
    rowwise_attn_kernel<128><<<grid, 128, 0, stream>>>(qp, kp, vp, block_table, page_logical_pos, seq_lens,
                                                       cu_q_lens, num_reqs, h->shape, h->ws.cs, op);
  else
    rowwise_attn_kernel<64><<<grid, 128, 0, stream>>>(qp, kp, vp, block_table, page_logical_pos, seq_lens,
                                                      cu_q_lens, num_reqs, h->shape, h->ws.cs, op);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

}  // namespace lazy
