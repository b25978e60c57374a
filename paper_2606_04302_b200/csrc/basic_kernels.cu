// basic_kernels.cu -- RoPE table build, lazy_cache_write, and the simple row-wise attention kernel.
//
//  * build_cs_table : cs[pos][j] = (cos, sin)(pos * theta^(-2j/D)), angles formed and reduced in fp64 so the
//    fp32 table entries are correctly rounded at any position (stateless rotation from the
//    absolute index; L138/L173: cos/sin loaded from a table).
//  * cache_write    : un-rotated K/V rows -> pages, 16-byte vectorised.
//  * rowwise_attn   : one CTA per (query row, q head), keys strided over 4 warps, K rotated by its absolute
//    angle from the table, online softmax.  It follows PAPER.md Eq. 4 (L94-106) directly and is kept as the
//    LAZY_FLAG_ROWWISE_KERNELS debugging path; the production kernels are decode_splitkv.cu / prefill_umma.cu.
#include <cmath>

#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {

struct FreqTable { double f[64]; };   // rotation frequency of pair j (head_dim / 2 <= 64 entries), by value

__global__ void build_cs_table_kernel(float2* __restrict__ cs, int max_position, int half, FreqTable freq, int D) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)max_position * half;
  if (idx >= total) return;
  int j = (int)(idx % half);
  long long pos = idx / half;
  double s, c;
  sincos((double)pos * freq.f[j], &s, &c);
  float* row = reinterpret_cast<float*>(cs + pos * half);
  const int k = cs_cos_index(j, D);
  row[k] = (float)c;
  row[k + 2] = (float)s;
}

// inv_freq_host == nullptr: theta_j = rope_theta^(-2j/D) (RoPE), computed here in fp64
int launch_build_tables(lazy_handle* h, const double* inv_freq_host, cudaStream_t stream) {
  int half = h->cfg.head_dim / 2;
  FreqTable ft;
  for (int j = 0; j < 64; ++j)
    ft.f[j] = j >= half ? 0.0
              : inv_freq_host ? inv_freq_host[j]
                              : pow(h->cfg.rope_theta, -2.0 * (double)j / (double)h->cfg.head_dim);
  long long total = (long long)h->cfg.max_position * half;
  int threads = 256;
  long long blocks = (total + threads - 1) / threads;
  build_cs_table_kernel<<<(unsigned)blocks, threads, 0, stream>>>(h->ws.cs, h->cfg.max_position, half, ft,
                                                                 h->cfg.head_dim);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------
// cache write: one thread moves one 16-byte chunk of K and the matching chunk of V.
// chunk index c in [0, T*Hkv*D/8): token = c / (Hkv*D/8), head = (c / (D/8)) % Hkv, part = c % (D/8).
__global__ void cache_write_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                   const long long* __restrict__ slot_mapping, long long num_chunks,
                                   int Hkv, int chunks_per_row, int deinterleave, uint4* __restrict__ k_cache,
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
  if (!deinterleave) {
    k_cache[dst] = k_new[c];
  } else {
    // LAZY_ROPE_INTERLEAVED: stored dim d' < D/2 is model dim 2d', stored dim D/2 + d' is model dim 2d' + 1
    // (still position-free; only the order of the dimensions changes, include/lazy_attn.h)
    const int half_chunks = chunks_per_row / 2;
    const int hi = part >= half_chunks;                          // this chunk holds the odd (x2) elements
    const uint4* src = k_new + (c - part) + 2 * (part - hi * half_chunks);   // 16 model dims = two chunks
    const uint4 s0 = src[0], s1 = src[1];
    const uint32_t sel = hi ? 0x7632u : 0x5410u;
    uint4 o;
    o.x = __byte_perm(s0.x, s0.y, sel); o.y = __byte_perm(s0.z, s0.w, sel);
    o.z = __byte_perm(s1.x, s1.y, sel); o.w = __byte_perm(s1.z, s1.w, sel);
    k_cache[dst] = o;
  }
  v_cache[dst] = v_new[c];
}

int launch_cache_write(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                       int num_tokens, void* k_cache, void* v_cache, cudaStream_t stream) {
  if (h->cfg.dtype == LAZY_KV_FP8_E4M3)
    return launch_cache_write_fp8(h, k_new, v_new, slot_mapping, num_tokens, k_cache, v_cache, stream);
  int chunks_per_row = h->cfg.head_dim / 8;
  long long num_chunks = (long long)num_tokens * h->cfg.num_kv_heads * chunks_per_row;
  int threads = 256;
  long long blocks = (num_chunks + threads - 1) / threads;
  cache_write_kernel<<<(unsigned)blocks, threads, 0, stream>>>(
      static_cast<const uint4*>(k_new), static_cast<const uint4*>(v_new),
      reinterpret_cast<const long long*>(slot_mapping), num_chunks, h->cfg.num_kv_heads, chunks_per_row,
      h->cfg.rope_style == LAZY_ROPE_INTERLEAVED, static_cast<uint4*>(k_cache), static_cast<uint4*>(v_cache));
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------
// lazy_debug_validate: one CTA per request counts table entries the attention kernels would misuse.
__global__ void validate_tables_kernel(const int* __restrict__ block_table, const int* __restrict__ page_pos,
                                       const int* __restrict__ seq_lens, int table_stride, int num_pages,
                                       int max_position, int* __restrict__ counter) {
  const int r = blockIdx.x;
  const int L = seq_lens[r];
  int bad = 0;
  if (threadIdx.x == 0 && (L < 0 || L > table_stride * kPageSize)) bad++;
  const int np = L < 0 ? 0 : min((L + kPageSize - 1) / kPageSize, table_stride);
  for (int s = threadIdx.x; s < np; s += blockDim.x) {
    const int pg = block_table[(size_t)r * table_stride + s], pos = page_pos[(size_t)r * table_stride + s];
    if (pg < 0 || pg >= num_pages) bad++;
    if (pos < 0 || pos > max_position - kPageSize) bad++;
  }
  if (bad) atomicAdd(counter, bad);
}

int launch_validate(lazy_handle* h, const int32_t* block_table, const int32_t* page_logical_pos,
                    const int32_t* seq_lens, int num_reqs, int* counter, cudaStream_t stream) {
  validate_tables_kernel<<<num_reqs, 128, 0, stream>>>(block_table, page_logical_pos, seq_lens,
                                                       h->cfg.max_pages_per_req, h->cfg.num_pages, h->cfg.max_position,
                                                       counter);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------
// Materialising re-encoding ("allocate + copy + rotate", L447).  HBM-bound:
// per page it reads Hkv*16*D*2 B of K (and of V) and writes the same.  One thread owns one 8-pair chunk of one
// row: two 16-byte loads (dims 8c.. and D/2+8c..), fp32 rotation from the fp64-built table, two 16-byte stores.
template <int D>
__global__ void __launch_bounds__(256)
materialize_pages_kernel(const uint4* __restrict__ k_src, const uint4* __restrict__ v_src,
                         const int* __restrict__ src_pages, const int* __restrict__ rot_pos, int per_token,
                         uint4* __restrict__ k_dst, uint4* __restrict__ v_dst, const int* __restrict__ dst_pages,
                         long long num_items, int Hkv, const float2* __restrict__ cs) {
  constexpr int CPR = D / 16;                       // chunk pairs per row
  constexpr int CH = D / 8;                         // 16-byte chunks per row
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= num_items) return;
  const int c = (int)(idx % CPR);
  long long row = idx / CPR;                        // (i, hk, t)
  const int t = (int)(row % kPageSize);
  const int hk = (int)((row / kPageSize) % Hkv);
  const int i = (int)(row / ((long long)kPageSize * Hkv));
  const int sp = src_pages[i], dp = dst_pages[i];
  int pos = rot_pos[i] + (per_token ? t : 0);
  const float sgn = pos < 0 ? -1.f : 1.f;
  pos = pos < 0 ? -pos : pos;
  const long long srow = (((long long)sp * Hkv + hk) * kPageSize + t) * CH;
  const long long drow = (((long long)dp * Hkv + hk) * kPageSize + t) * CH;
  uint4 va = k_src[srow + c], vb = k_src[srow + c + CPR];
  uint32_t* aw = reinterpret_cast<uint32_t*>(&va);
  uint32_t* bw = reinterpret_cast<uint32_t*>(&vb);
  const float2* row_cs = cs + (size_t)pos * (D / 2);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const float2 c0 = cs_load(row_cs, 8 * c + 2 * w, D);
    const float2 c1 = cs_load(row_cs, 8 * c + 2 * w + 1, D);
    const float a0 = ptx::bf16_lo(aw[w]), a1 = ptx::bf16_hi(aw[w]);
    const float b0 = ptx::bf16_lo(bw[w]), b1 = ptx::bf16_hi(bw[w]);
    const float s0 = c0.y * sgn, s1 = c1.y * sgn;
    aw[w] = ptx::pack_bf16(a0 * c0.x - b0 * s0, a1 * c1.x - b1 * s1);
    bw[w] = ptx::pack_bf16(a0 * s0 + b0 * c0.x, a1 * s1 + b1 * c1.x);
  }
  k_dst[drow + c] = va;
  k_dst[drow + c + CPR] = vb;
  if (v_src != nullptr && v_dst != nullptr) {
    v_dst[drow + c] = v_src[srow + c];
    v_dst[drow + c + CPR] = v_src[srow + c + CPR];
  }
}

int launch_materialize(lazy_handle* h, const void* k_src, const void* v_src, const int32_t* src_pages,
                       const int32_t* rot_pos, int per_token, void* k_dst, void* v_dst, const int32_t* dst_pages,
                       int num, cudaStream_t stream) {
  const int D = h->cfg.head_dim;
  const long long items = (long long)num * h->cfg.num_kv_heads * kPageSize * (D / 16);
  const int threads = 256;
  const long long blocks = (items + threads - 1) / threads;
  auto ks = static_cast<const uint4*>(k_src);
  auto vs = static_cast<const uint4*>(v_src);
  auto kd = static_cast<uint4*>(k_dst);
  auto vd = static_cast<uint4*>(v_dst);
  if (D == 128)
    materialize_pages_kernel<128><<<(unsigned)blocks, threads, 0, stream>>>(
        ks, vs, src_pages, rot_pos, per_token, kd, vd, dst_pages, items, h->cfg.num_kv_heads, h->ws.cs);
  else
    materialize_pages_kernel<64><<<(unsigned)blocks, threads, 0, stream>>>(
        ks, vs, src_pages, rot_pos, per_token, kd, vd, dst_pages, items, h->cfg.num_kv_heads, h->ws.cs);
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
                    int k_storage, const int* __restrict__ stored_pos, int q_interleaved,
                    const float* __restrict__ alibi, __nv_bfloat16* __restrict__ out) {
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
      float a = __bfloat162float(qp[q_interleaved ? 2 * j : j]);
      float b = __bfloat162float(qp[q_interleaved ? 2 * j + 1 : j + HALF]);
      float2 t = cs_load(cs + (size_t)(alibi ? 0 : pos_q) * HALF, j, D);   // table row 0 is the identity
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
    // rotation still owed to this key: its logical position (un-rotated pages), one relative offset per page
    // (stored-position pages), nothing (absolute pages; table row 0 is the identity)
    int pos = alibi ? 0
              : k_storage == LAZY_K_UNROTATED ? pp[slot] + t
              : k_storage == LAZY_K_STORED_POS ? pp[slot] - stored_pos[page] : 0;
    const float sgn = pos < 0 ? -1.f : 1.f;
    pos = pos < 0 ? -pos : pos;
    size_t base = (((size_t)page * sh.Hkv + hk) * kPageSize + t) * D;
    float dot = 0.f, v1[PER], v2[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) {
      int j = lane * PER + e;
      float a = __bfloat162float(k_cache[base + j]), b = __bfloat162float(k_cache[base + j + HALF]);
      float2 tcs = cs_load(cs + (size_t)pos * HALF, j, D);
      tcs.y *= sgn;
      dot += q1[e] * (a * tcs.x - b * tcs.y) + q2[e] * (a * tcs.y + b * tcs.x);
      v1[e] = __bfloat162float(v_cache[base + j]);
      v2[e] = __bfloat162float(v_cache[base + j + HALF]);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
    if (alibi) dot += alibi[hq] * (float)(pp[slot] + t - pos_q);          // ALiBi bias (log2 units)
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
  if (h->cfg.dtype == LAZY_KV_FP8_E4M3)
    return launch_rowwise_fp8(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, cu_q_lens, num_reqs,
                              total_q, out, stream);
  dim3 grid(total_q, h->cfg.num_q_heads);
  auto qp = static_cast<const __nv_bfloat16*>(q);
  auto kp = static_cast<const __nv_bfloat16*>(k_cache);
  auto vp = static_cast<const __nv_bfloat16*>(v_cache);
  auto op = static_cast<__nv_bfloat16*>(out);
  if (h->cfg.head_dim == 128)
    rowwise_attn_kernel<128><<<grid, 128, 0, stream>>>(qp, kp, vp, block_table, page_logical_pos, seq_lens,
                                                       cu_q_lens, num_reqs, h->shape, h->ws.cs, h->cfg.k_storage,
                                                       h->page_stored_pos,
                                                       h->cfg.rope_style == LAZY_ROPE_INTERLEAVED,
                                                       h->cfg.rope_style == LAZY_POS_ALIBI ? h->ws.alibi : nullptr, op);
  else
    rowwise_attn_kernel<64><<<grid, 128, 0, stream>>>(qp, kp, vp, block_table, page_logical_pos, seq_lens,
                                                      cu_q_lens, num_reqs, h->shape, h->ws.cs, h->cfg.k_storage,
                                                      h->page_stored_pos,
                                                      h->cfg.rope_style == LAZY_ROPE_INTERLEAVED,
                                                      h->cfg.rope_style == LAZY_POS_ALIBI ? h->ws.alibi : nullptr, op);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

}  // namespace lazy
