// mixed_fused.cu -- lazy_attn_mixed in ONE launch (Fig. 5 phases 1-3, L273: with a
// 2,048-token chunk budget every engine step is a mix of prefill chunks and decodes).
//
// One grid, two kinds of CTA.  CTAs 0 .. n_dec-1 run the split-KV decode body (decode_kernel.cuh: persistent, they
// share the decode requests' units and combine in-kernel); every later pair of CTAs runs one prefill work item
// (prefill_pair_kernel.cuh: a thread-block cluster of 2 on tcgen05 cta_group::2).  The hardware's CTA scheduler places
// the decode CTAs first and keeps filling the other SMs with prefill pairs as they retire, so the HBM-bound decode
// stream and the tensor-bound prefill tiles overlap without streams, events or a second launch, and the split of the
// machine is one number (n_dec).  The grid is launched with cluster size 2 throughout (the decode CTAs ignore their
// cluster), 512 threads (the decode body uses 384: its fourth warpgroup gives its registers back and leaves) and the
// larger of the two shared-memory footprints.  head_dim 128, un-rotated K, at most 8 kv heads: the product
// configuration; everything else takes the two-stream path of lazy_api.cu.
#include <climits>

#include "decode_kernel.cuh"
#include "decode_fp8_kernel.cuh"
#include "prefill_pair_kernel.cuh"

namespace lazy {
namespace {

template <int HKV_CTA>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPrefillThreads, 1)
mixed_step_kernel(const __grid_constant__ CUtensorMap tmap_dk, const __grid_constant__ CUtensorMap tmap_dv,
                  const __grid_constant__ CUtensorMap tmap_pq, const __grid_constant__ CUtensorMap tmap_pk,
                  const __grid_constant__ CUtensorMap tmap_pv, const DecodeArgs da, const PrefillArgs pa,
                  const int n_dec) {
  extern __shared__ unsigned char smem_raw[];
  if ((int)blockIdx.x < n_dec) {
    if (threadIdx.x >= kDecodeThreads) {            // registers back to the pool the decode consumers draw from
      ptx::setmaxnreg_dec<24>();
      return;
    }
    decode_cta<128, HKV_CTA, LAZY_K_UNROTATED>(tmap_dk, tmap_dv, da, (int)blockIdx.x, n_dec, 0, 1, smem_raw);
  } else {
    prefill_pair_cta<LAZY_K_UNROTATED>(tmap_pq, tmap_pk, tmap_pv, pa, ((int)blockIdx.x - n_dec) >> 1, smem_raw);
  }
}

// The same step on LAZY_KV_FP8_E4M3 pages: the 12-warp FP8 decode body (it uses all 512 threads; 4 kv heads per CTA, so 8
// kv heads make two head groups that alternate over the decode CTAs) and the FP8 arm of the pair prefill body.
template <int HG>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPrefillThreads, 1)
mixed_step_fp8_kernel(const __grid_constant__ CUtensorMap tmap_dk, const __grid_constant__ CUtensorMap tmap_dv,
                      const __grid_constant__ CUtensorMap tmap_pq, const __grid_constant__ CUtensorMap tmap_pk,
                      const __grid_constant__ CUtensorMap tmap_pv, const DecodeFp8Args da, const PrefillArgs pa,
                      const int n_dec) {
  extern __shared__ unsigned char smem_raw[];
  if ((int)blockIdx.x < n_dec)
    decode_fp8_cta<4, 12>(tmap_dk, tmap_dv, da, (int)blockIdx.x / HG, n_dec / HG, (int)blockIdx.x % HG, HG, smem_raw);
  else
    prefill_pair_cta<LAZY_K_UNROTATED, true>(tmap_pq, tmap_pk, tmap_pv, pa, ((int)blockIdx.x - n_dec) >> 1, smem_raw);
}

template <int HG>
int launch_mixed_fp8_t(const lazy_handle* h, const DecodeFp8Args& da, const PrefillArgs& pa, int n_dec, long long grid,
                       cudaStream_t stream) {
  constexpr int smem = DecodeFp8Cfg<4, 12>::SMEM_BYTES > PairCfg::SMEM_BYTES ? DecodeFp8Cfg<4, 12>::SMEM_BYTES
                                                                             : PairCfg::SMEM_BYTES;
  static_assert(DecodeFp8Cfg<4, 12>::THREADS == kPrefillThreads, "one block size for both bodies");
  auto kern = mixed_step_fp8_kernel<HG>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return LAZY_ERR_CUDA;
  kern<<<(unsigned)grid, kPrefillThreads, smem, stream>>>(
      *reinterpret_cast<const CUtensorMap*>(h->tmap_k), *reinterpret_cast<const CUtensorMap*>(h->tmap_v),
      *reinterpret_cast<const CUtensorMap*>(h->tmap_pq), *reinterpret_cast<const CUtensorMap*>(h->tmap_pk),
      *reinterpret_cast<const CUtensorMap*>(h->tmap_pv), da, pa, n_dec);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

template <int HKV_CTA>
int launch_mixed_t(const lazy_handle* h, const DecodeArgs& da, const PrefillArgs& pa, int n_dec, long long grid,
                   cudaStream_t stream) {
  constexpr int smem = DecodeCfg<128, HKV_CTA>::SMEM_BYTES > PairCfg::SMEM_BYTES ? DecodeCfg<128, HKV_CTA>::SMEM_BYTES
                                                                                  : PairCfg::SMEM_BYTES;
  auto kern = mixed_step_kernel<HKV_CTA>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return LAZY_ERR_CUDA;
  kern<<<(unsigned)grid, kPrefillThreads, smem, stream>>>(
      *reinterpret_cast<const CUtensorMap*>(h->tmap_k), *reinterpret_cast<const CUtensorMap*>(h->tmap_v),
      *reinterpret_cast<const CUtensorMap*>(h->tmap_pq), *reinterpret_cast<const CUtensorMap*>(h->tmap_pk),
      *reinterpret_cast<const CUtensorMap*>(h->tmap_pv), da, pa, n_dec);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

}  // namespace

bool mixed_fused_supported(const lazy_handle* h, int num_reqs_decode) {
  const lazy_config& c = h->cfg;
  return c.head_dim == 128 && c.k_storage == LAZY_K_UNROTATED && c.rope_style != LAZY_POS_ALIBI &&
         (c.num_kv_heads == 4 || c.num_kv_heads == 8) && num_reqs_decode <= kMaxReqsSmem &&
         !(c.flags & (LAZY_FLAG_ROWWISE_KERNELS | LAZY_FLAG_PREFILL_ONE_CTA | LAZY_FLAG_FP8_DECODE_8_WARPS));
}

// Returns the number of kernels launched (1), or LAZY_ERR_*.
int launch_mixed_fused(lazy_handle* h, const lazy_mixed_args* m, const void* k_cache, const void* v_cache, int decode_ctas,
                       cudaStream_t stream) {
  const lazy_config& c = h->cfg;
  const bool fp8 = c.dtype == LAZY_KV_FP8_E4M3;
  const int hkv_cta = fp8 ? 4 : c.num_kv_heads;     // bf16: 4 or 8, one kv-head group; FP8: 4 heads per decode CTA
  const int group = c.num_q_heads / c.num_kv_heads;
  const int tpt = kTileRows / group;
  const long long rows = (long long)c.num_pages * c.num_kv_heads * kPageSize;
  if (h->tmap_k_ptr != k_cache) {
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_k, k_cache, rows, c.head_dim, 16 * hkv_cta, true, c.head_dim)
              : encode_pool_tmap(h->tmap_k, k_cache, rows, c.head_dim, 16 * hkv_cta)))
      return LAZY_ERR_CUDA;
    h->tmap_k_ptr = k_cache;
  }
  if (h->tmap_v_ptr != v_cache) {
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_v, v_cache, rows, c.head_dim, 16 * hkv_cta, true, c.head_dim)
              : encode_pool_tmap(h->tmap_v, v_cache, rows, c.head_dim, 16 * hkv_cta)))
      return LAZY_ERR_CUDA;
    h->tmap_v_ptr = v_cache;
  }
  if (h->tmap_pk_ptr != k_cache) {
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_pk, k_cache, rows, c.head_dim, kPageSize, false, c.head_dim)
              : encode_pool_tmap(h->tmap_pk, k_cache, rows, c.head_dim, kPageSize)))
      return LAZY_ERR_CUDA;
    h->tmap_pk_ptr = k_cache;
  }
  if (h->tmap_pv_ptr != v_cache) {
    if (!(fp8 ? encode_pool_tmap_u8(h->tmap_pv, v_cache, rows, c.head_dim, kPageSize, false, 64)
              : encode_pool_tmap(h->tmap_pv, v_cache, rows, c.head_dim, kPageSize)))
      return LAZY_ERR_CUDA;
    h->tmap_pv_ptr = v_cache;
  }
  if (h->tmap_pq_ptr != m->q_prefill || h->tmap_pq_rows != m->total_q) {
    if (!encode_q_tmap(h->tmap_pq, m->q_prefill, m->total_q, c.num_q_heads, c.num_kv_heads, c.head_dim, tpt))
      return LAZY_ERR_CUDA;
    h->tmap_pq_ptr = m->q_prefill;
    h->tmap_pq_rows = m->total_q;
  }
  DecodeArgs da;
  da.q = static_cast<const __nv_bfloat16*>(m->q_decode);
  da.out = static_cast<__nv_bfloat16*>(m->out_decode);
  da.block_table = m->block_table_decode;
  da.page_pos = m->page_logical_pos_decode;
  da.seq_lens = m->seq_lens_decode;
  da.cs = h->ws.cs;
  da.stored_pos = h->page_stored_pos;
  da.alibi = h->ws.alibi;
  da.part_o = h->ws.part_o;
  da.part_ml = h->ws.part_ml;
  da.req_counter = h->ws.req_counter;
  da.num_reqs = m->num_reqs_decode;
  da.q_interleaved = c.rope_style == LAZY_ROPE_INTERLEAVED;
  da.sh = h->shape;
  PrefillArgs pa;
  pa.block_table = m->block_table_prefill;
  pa.page_pos = m->page_logical_pos_prefill;
  pa.seq_lens = m->seq_lens_prefill;
  pa.cu_q_lens = m->cu_q_lens;
  pa.out = static_cast<__nv_bfloat16*>(m->out_prefill);
  pa.cs = h->ws.cs;
  pa.stored_pos = h->page_stored_pos;
  pa.alibi = h->ws.alibi;
  pa.k_scale = h->k_scale;
  pa.v_scale = h->v_scale;
  pa.num_reqs = m->num_reqs_prefill;
  pa.q_interleaved = c.rope_style == LAZY_ROPE_INTERLEAVED;
  pa.mblocks = (m->max_q_len + 4 * tpt - 1) / (4 * tpt);
  pa.tokens_per_tile = tpt;
  pa.sh = h->shape;
  int n_dec = decode_ctas & ~1;                     // clusters of 2: the decode CTAs fill whole clusters
  if (n_dec < 2) n_dec = 2;
  if (n_dec > kMaxDecodeCtas) n_dec = kMaxDecodeCtas;
  const long long grid = n_dec + 2LL * pa.mblocks * c.num_kv_heads * m->num_reqs_prefill;
  if (grid > INT_MAX) return LAZY_ERR_INVALID;
  if (fp8) {
    DecodeFp8Args fa;
    fa.d = da;
    fa.k_scale = h->k_scale;
    fa.v_scale = h->v_scale;
    return c.num_kv_heads == 8 ? launch_mixed_fp8_t<2>(h, fa, pa, n_dec, grid, stream)
                               : launch_mixed_fp8_t<1>(h, fa, pa, n_dec, grid, stream);
  }
  return hkv_cta == 8 ? launch_mixed_t<8>(h, da, pa, n_dec, grid, stream) : launch_mixed_t<4>(h, da, pa, n_dec, grid, stream);
}

}  // namespace lazy
