// decode_splitkv.cu -- lazy_attn_decode: split-KV flash-decoding over position-free paged K (sm_100a).
//
// Path rows: a1 metadata fetch, a2 page gather (TMA, 128B-swizzled boxes), a3/a4 rotation in
// fp32 registers, a5 QK^T, a6 online softmax (warp-shuffle max), a7 PV, a8 split-KV combine, a9 epilogue.
//
// Rotation identity used (PAPER.md Fact 3.2, L154-158; "rotate Q when the document changes", L175):
//     score(query at m, key t of a page starting at p0) = (R_{m-p0} q)^T (R_t k)
// so K is rotated only by its in-page offset t in [0,16) -- 16 x D/2 angles that live in shared memory for
// the whole kernel (rows 0..15 of the cos/sin table) -- and q is re-rotated once per page by m - p0 with one
// D/2-entry cos/sin row fetched by the same bulk-copy pipeline that brings the page.  No per-token table
// traffic, no writes to the cache.
//
// Work decomposition: the (request, page-group) units of the whole batch are cut into gridDim.x equal
// contiguous ranges (stream-K style), so every SM streams the same number of bytes whatever the length mix.
// A CTA owns HKV_CTA kv heads of a page (8 / HKV_CTA pages per pipeline stage); each of its 8 consumer warps
// owns one (page-lane, kv head) tile per stage and all q heads of that kv head's GQA group.  A 9th warp
// produces: block-table prefetch, TMA issue, mbarrier bookkeeping.  Per tile a warp does
//   S[16 tok x 8 heads] = Khat[16 x D] Qhat^T   (mma.sync m16n8k16, tokens as M so a page is exactly one tile)
//   online softmax over tokens, P -> bf16, transposed in registers with movmatrix
//   O^T[D x 8 heads]  += V^T[D x 16] P          (V^T fragments via ldmatrix.trans from the swizzled tile)
// The legacy mma.sync path is deliberate: this kernel is HBM-bound (512 B per (token, kv head)); the tensor
// work per page is 32 small MMAs and tcgen05's 128-row tiles would be >90% padding at 4-8 query rows.
// Partials (o, m, l) go to the workspace; the last CTA to finish a request combines them (no second launch).
#include <climits>

#include "decode_kernel.cuh"
#include "decode_fp8_kernel.cuh"

namespace lazy {
namespace {

template <int D, int HKV_CTA, int KM>
__global__ void __launch_bounds__(kDecodeThreads, 1)
decode_splitkv_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
                      const DecodeArgs a) {
  extern __shared__ unsigned char smem_raw[];
  decode_cta<D, HKV_CTA, KM>(tmap_k, tmap_v, a, (int)blockIdx.x, (int)gridDim.x, (int)blockIdx.y, (int)gridDim.y, smem_raw);
}

// LAZY_KV_FP8_E4M3 pages (decode_fp8_kernel.cuh), head_dim 128
template <int HKV_CTA, int NCW, int D>
__global__ void __launch_bounds__(NCW * 32 + 128, 1)
decode_fp8_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
                  const DecodeFp8Args a) {
  extern __shared__ unsigned char smem_raw[];
  decode_fp8_cta<HKV_CTA, NCW, D>(tmap_k, tmap_v, a, (int)blockIdx.x, (int)gridDim.x, (int)blockIdx.y, (int)gridDim.y, smem_raw);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

}  // namespace

// 2-D view of a pool: rows = num_pages*Hkv*16 tokens-of-a-head, cols = D; box = [box_rows][64 cols], 128B swizzle.
bool encode_pool_tmap(void* out_map, const void* pool, long long rows, int D, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t gdim[2] = {(cuuint64_t)D, (cuuint64_t)rows};
  cuuint64_t gstride[1] = {(cuuint64_t)D * 2};
  cuuint32_t box[2] = {64u, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult rc = fn(reinterpret_cast<CUtensorMap*>(out_map), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                   const_cast<void*>(pool), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return rc == CUDA_SUCCESS;
}

// FP8 code pool: rows of D bytes; box = [box_rows][D bytes] (swizzled for the decode kernel -- D = 128: one 128-byte
// swizzle span per row -- plain rows for the prefill kernel, which re-writes the tile as bf16)
bool encode_pool_tmap_u8(void* out_map, const void* pool, long long rows, int D, int box_rows, bool swizzle,
                         int box_cols) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t gdim[2] = {(cuuint64_t)D, (cuuint64_t)rows};
  cuuint64_t gstride[1] = {(cuuint64_t)D};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult rc = fn(reinterpret_cast<CUtensorMap*>(out_map), CU_TENSOR_MAP_DATA_TYPE_UINT8, 2,
                   const_cast<void*>(pool), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   !swizzle ? CU_TENSOR_MAP_SWIZZLE_NONE : D == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return rc == CUDA_SUCCESS;
}

bool encode_q_tmap(void* out_map, const void* q, int total_q, int Hq, int Hkv, int D, int tokens_per_tile) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  const int group = Hq / Hkv;
  cuuint64_t gdim[4] = {(cuuint64_t)D, (cuuint64_t)group, (cuuint64_t)Hkv, (cuuint64_t)total_q};
  cuuint64_t gstride[3] = {(cuuint64_t)D * 2, (cuuint64_t)group * D * 2, (cuuint64_t)Hq * D * 2};
  cuuint32_t box[4] = {64u, (cuuint32_t)group, 1u, (cuuint32_t)tokens_per_tile};
  cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  CUresult rc = fn(reinterpret_cast<CUtensorMap*>(out_map), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4,
                   const_cast<void*>(q), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return rc == CUDA_SUCCESS;
}

template <int D, int HKV_CTA, int KM>
static int launch_decode_km(lazy_handle* h, const DecodeArgs& args, int grid_x, int grid_y, cudaStream_t stream) {
  using C = DecodeCfg<D, HKV_CTA>;
  auto kern = decode_splitkv_kernel<D, HKV_CTA, KM>;
  // per launch: the attribute is per device, and a process may hold handles on several devices
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess)
    return LAZY_ERR_CUDA;
  const CUtensorMap* mk = reinterpret_cast<const CUtensorMap*>(h->tmap_k);
  const CUtensorMap* mv = reinterpret_cast<const CUtensorMap*>(h->tmap_v);
  kern<<<dim3(grid_x, grid_y), kDecodeThreads, C::SMEM_BYTES, stream>>>(*mk, *mv, args);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

template <int D, int HKV_CTA>
static int launch_decode_t(lazy_handle* h, const DecodeArgs& args, int grid_x, int grid_y, cudaStream_t stream) {
  if (h->cfg.rope_style == LAZY_POS_ALIBI) return launch_decode_km<D, HKV_CTA, kKmAlibi>(h, args, grid_x, grid_y, stream);
  switch (h->cfg.k_storage) {
    case LAZY_K_STORED_POS: return launch_decode_km<D, HKV_CTA, LAZY_K_STORED_POS>(h, args, grid_x, grid_y, stream);
    case LAZY_K_ABSOLUTE:   return launch_decode_km<D, HKV_CTA, LAZY_K_ABSOLUTE>(h, args, grid_x, grid_y, stream);
    default:                return launch_decode_km<D, HKV_CTA, LAZY_K_UNROTATED>(h, args, grid_x, grid_y, stream);
  }
}

template <int HKV_CTA, int NCW, int D>
static int launch_decode_fp8_d(lazy_handle* h, const DecodeFp8Args& args, int grid_x, int grid_y, cudaStream_t stream) {
  using C = DecodeFp8Cfg<HKV_CTA, NCW, D>;
  auto kern = decode_fp8_kernel<HKV_CTA, NCW, D>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess)
    return LAZY_ERR_CUDA;
  const CUtensorMap* mk = reinterpret_cast<const CUtensorMap*>(h->tmap_k);
  const CUtensorMap* mv = reinterpret_cast<const CUtensorMap*>(h->tmap_v);
  kern<<<dim3(grid_x, grid_y), C::THREADS, C::SMEM_BYTES, stream>>>(*mk, *mv, args);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

template <int HKV_CTA, int NCW>
static int launch_decode_fp8_t(lazy_handle* h, const DecodeFp8Args& args, int grid_x, int grid_y, cudaStream_t stream) {
  return h->cfg.head_dim == 128 ? launch_decode_fp8_d<HKV_CTA, NCW, 128>(h, args, grid_x, grid_y, stream)
                                : launch_decode_fp8_d<HKV_CTA, NCW, 64>(h, args, grid_x, grid_y, stream);
}

int launch_decode(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                  const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                  int num_reqs, void* out, cudaStream_t stream) {
  const lazy_config& c = h->cfg;
  const bool fp8 = c.dtype == LAZY_KV_FP8_E4M3;
  // FP8 pages: 12 consumer warps = 4 kv heads x 3 pages (or fewer heads x more pages) per stage, unless the A/B flag
  // asks for the bf16 kernel's 8-warp cut
  const bool w12 = fp8 && !(c.flags & LAZY_FLAG_FP8_DECODE_8_WARPS);
  const int hkv_cta = w12 ? (c.num_kv_heads >= 4 ? 4 : c.num_kv_heads) : (c.num_kv_heads >= 8 ? 8 : c.num_kv_heads);
  const int HG = c.num_kv_heads / hkv_cta;
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
  int launches = 0;
  const int max_reqs = kMaxReqsSmem;                                // requests per launch (smem prefix sums)
  for (int r0 = 0; r0 < num_reqs; r0 += max_reqs) {
    const int n = (num_reqs - r0 < max_reqs) ? num_reqs - r0 : max_reqs;
    DecodeArgs a;
    a.q = static_cast<const __nv_bfloat16*>(q) + (size_t)r0 * c.num_q_heads * c.head_dim;
    a.out = static_cast<__nv_bfloat16*>(out) + (size_t)r0 * c.num_q_heads * c.head_dim;
    a.block_table = block_table + (size_t)r0 * c.max_pages_per_req;
    a.page_pos = page_logical_pos + (size_t)r0 * c.max_pages_per_req;
    a.seq_lens = seq_lens + r0;
    a.cs = h->ws.cs;
    a.stored_pos = h->page_stored_pos;
    a.alibi = h->ws.alibi;
    a.part_o = h->ws.part_o;
    a.part_ml = h->ws.part_ml;
    a.req_counter = h->ws.req_counter;
    a.num_reqs = n;
    a.q_interleaved = c.rope_style == LAZY_ROPE_INTERLEAVED;
    a.sh = h->shape;
    int gx = (h->decode_cta_limit > 0 ? h->decode_cta_limit : h->num_sms) / HG;
    if (gx < 1) gx = 1;
    if (gx > kMaxDecodeCtas) gx = kMaxDecodeCtas;
    int rc;
    if (fp8) {
      DecodeFp8Args fa;
      fa.d = a;
      fa.k_scale = h->k_scale;
      fa.v_scale = h->v_scale;
      if (w12) {
        if (hkv_cta == 4) rc = launch_decode_fp8_t<4, 12>(h, fa, gx, HG, stream);
        else if (hkv_cta == 2) rc = launch_decode_fp8_t<2, 12>(h, fa, gx, HG, stream);
        else rc = launch_decode_fp8_t<1, 12>(h, fa, gx, HG, stream);
      } else if (hkv_cta == 8) rc = launch_decode_fp8_t<8, 8>(h, fa, gx, HG, stream);
      else if (hkv_cta == 4) rc = launch_decode_fp8_t<4, 8>(h, fa, gx, HG, stream);
      else if (hkv_cta == 2) rc = launch_decode_fp8_t<2, 8>(h, fa, gx, HG, stream);
      else rc = launch_decode_fp8_t<1, 8>(h, fa, gx, HG, stream);
    } else if (c.head_dim == 128) {
      if (hkv_cta == 8) rc = launch_decode_t<128, 8>(h, a, gx, HG, stream);
      else if (hkv_cta == 4) rc = launch_decode_t<128, 4>(h, a, gx, HG, stream);
      else if (hkv_cta == 2) rc = launch_decode_t<128, 2>(h, a, gx, HG, stream);
      else rc = launch_decode_t<128, 1>(h, a, gx, HG, stream);
    } else {
      if (hkv_cta == 8) rc = launch_decode_t<64, 8>(h, a, gx, HG, stream);
      else if (hkv_cta == 4) rc = launch_decode_t<64, 4>(h, a, gx, HG, stream);
      else if (hkv_cta == 2) rc = launch_decode_t<64, 2>(h, a, gx, HG, stream);
      else rc = launch_decode_t<64, 1>(h, a, gx, HG, stream);
    }
    if (rc < 0) return rc;
    launches += rc;
  }
  return launches;
}

}  // namespace lazy
