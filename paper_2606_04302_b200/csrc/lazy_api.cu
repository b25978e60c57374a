// lazy_api.cu -- host side of the C ABI (include/lazy_attn.h): argument checks, workspace carving,
// handle management and dispatch to the kernel launchers.  No torch types, no allocation per call.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <new>

#include "lazy_internal.h"

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool config_supported(const lazy_config* c) {
  if (c->head_dim != 64 && c->head_dim != 128) return false;
  if (c->page_size != lazy::kPageSize) return false;
  if (c->num_q_heads <= 0 || c->num_kv_heads <= 0) return false;
  if (c->num_q_heads % c->num_kv_heads != 0) return false;
  if (c->num_q_heads / c->num_kv_heads > 8) return false;
  int hkv = c->num_kv_heads;
  if (!(hkv == 1 || hkv == 2 || hkv == 4 || hkv % 8 == 0)) return false;
  if (c->dtype != LAZY_KV_BF16 && c->dtype != LAZY_KV_FP8_E4M3) return false;
  if (c->dtype == LAZY_KV_FP8_E4M3 && (c->rope_style == LAZY_POS_ALIBI || c->k_storage != LAZY_K_UNROTATED))
    return false;
  if (c->rope_style < LAZY_ROPE_HALF_SPLIT || c->rope_style > LAZY_POS_ALIBI) return false;
  if (c->rope_style == LAZY_POS_ALIBI && (c->k_storage != LAZY_K_UNROTATED || c->num_q_heads > lazy::kMaxAlibiHeads))
    return false;
  if (c->k_storage < LAZY_K_UNROTATED || c->k_storage > LAZY_K_ABSOLUTE) return false;
  return true;
}

bool config_valid(const lazy_config* c) {
  return c->num_pages > 0 && c->max_position > 0 && c->max_reqs > 0 && c->max_pages_per_req > 0 &&
         c->rope_theta > 0.0;
}

struct Layout {
  size_t cs, part_o, part_ml, req_counter, sched, alibi, total;
};

Layout workspace_layout(const lazy_config* c) {
  Layout l{};
  size_t off = 0;
  // decode partials: one slot per (request, CTA) intersection and page lane (8 / kv-heads-per-CTA lanes)
  int hkv_cta = c->num_kv_heads >= 8 ? 8 : c->num_kv_heads;
  size_t lanes = 8 / hkv_cta;
  size_t head_groups = (size_t)c->num_kv_heads / hkv_cta;
  if (c->dtype == LAZY_KV_FP8_E4M3) {               // 12 consumer warps: at most 4 kv heads per CTA
    int h12 = c->num_kv_heads >= 4 ? 4 : c->num_kv_heads;
    if ((size_t)(12 / h12) > lanes) lanes = 12 / h12;
    if ((size_t)c->num_kv_heads / h12 > head_groups) head_groups = (size_t)c->num_kv_heads / h12;
  }
  size_t parts = ((size_t)c->max_reqs + lazy::kMaxDecodeCtas) * lanes;
  l.cs = off;          off = align_up(off + (size_t)c->max_position * (c->head_dim / 2) * sizeof(float2), 256);
  l.part_o = off;      off = align_up(off + parts * c->num_q_heads * c->head_dim * sizeof(float), 256);
  l.part_ml = off;     off = align_up(off + parts * c->num_q_heads * sizeof(float2), 256);
  l.req_counter = off; off = align_up(off + (size_t)c->max_reqs * head_groups * sizeof(int), 256);
  l.sched = off;       off = align_up(off + 1024 * sizeof(int), 256);
  l.alibi = off;       off = align_up(off + lazy::kMaxAlibiHeads * sizeof(float), 256);
  l.total = off;
  return l;
}

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

}  // namespace

extern "C" {

size_t lazy_workspace_bytes(const lazy_config* cfg) {
  if (!cfg || !config_valid(cfg) || !config_supported(cfg)) return 0;
  return workspace_layout(cfg).total;
}

int lazy_create(const lazy_config* cfg, void* workspace, size_t workspace_bytes, void* stream,
                lazy_handle** out) {
  if (!cfg || !out) return LAZY_ERR_INVALID;
  *out = nullptr;
  if (!config_valid(cfg)) return LAZY_ERR_INVALID;
  if (!config_supported(cfg)) return LAZY_ERR_UNSUPPORTED;
  Layout l = workspace_layout(cfg);
  if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) != 0 || workspace_bytes < l.total)
    return LAZY_ERR_WORKSPACE;

  lazy_handle* h = new (std::nothrow) lazy_handle();
  if (!h) return LAZY_ERR_INVALID;
  std::memset(h, 0, sizeof(*h));
  h->cfg = *cfg;
  h->shape.Hq = cfg->num_q_heads;
  h->shape.Hkv = cfg->num_kv_heads;
  h->shape.D = cfg->head_dim;
  h->shape.group = cfg->num_q_heads / cfg->num_kv_heads;
  h->shape.table_stride = cfg->max_pages_per_req;
  h->shape.max_position = cfg->max_position;
  h->shape.scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)cfg->head_dim));
  char* base = static_cast<char*>(workspace);
  h->ws.cs = reinterpret_cast<float2*>(base + l.cs);
  h->ws.part_o = reinterpret_cast<float*>(base + l.part_o);
  h->ws.part_ml = reinterpret_cast<float2*>(base + l.part_ml);
  h->ws.req_counter = reinterpret_cast<int*>(base + l.req_counter);
  h->ws.sched = reinterpret_cast<int*>(base + l.sched);
  h->ws.alibi = reinterpret_cast<float*>(base + l.alibi);

  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    delete h;
    return LAZY_ERR_CUDA;
  }
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (cudaMemsetAsync(h->ws.req_counter, 0, l.sched - l.req_counter, s) != cudaSuccess ||
      cudaMemsetAsync(h->ws.sched, 0, 1024 * sizeof(int), s) != cudaSuccess ||
      cudaMemsetAsync(h->ws.alibi, 0, lazy::kMaxAlibiHeads * sizeof(float), s) != cudaSuccess) {
    delete h;
    return LAZY_ERR_CUDA;
  }
  int n = lazy::launch_build_tables(h, nullptr, s);
  if (n < 0) { delete h; return n; }
  h->launches += n;
  *out = h;
  return LAZY_OK;
}

void lazy_destroy(lazy_handle* h) {
  if (!h) return;
  if (h->side_stream) {
    cudaStreamDestroy(h->side_stream);
    cudaEventDestroy(h->ev_fork);
    cudaEventDestroy(h->ev_join);
  }
  delete h;
}

int lazy_cache_write(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                     int32_t num_tokens, void* k_cache, void* v_cache, void* stream) {
  if (!h || num_tokens < 0) return LAZY_ERR_INVALID;
  if (num_tokens == 0) return LAZY_OK;
  if (!k_new || !v_new || !slot_mapping || !k_cache || !v_cache) return LAZY_ERR_INVALID;
  if (h->cfg.dtype == LAZY_KV_FP8_E4M3 && !h->k_scale) return LAZY_ERR_INVALID;
  if (misaligned(k_new) || misaligned(v_new) || misaligned(k_cache) || misaligned(v_cache) ||
      (reinterpret_cast<uintptr_t>(slot_mapping) & 7u))
    return LAZY_ERR_INVALID;
  int n = lazy::launch_cache_write(h, k_new, v_new, slot_mapping, num_tokens, k_cache, v_cache,
                                   static_cast<cudaStream_t>(stream));
  if (n < 0) return n;
  h->launches += n;
  return LAZY_OK;
}

int lazy_set_rope_frequencies(lazy_handle* h, const double* inv_freq, double softmax_scale, void* stream) {
  if (!h || softmax_scale < 0.0) return LAZY_ERR_INVALID;
  if (inv_freq)
    for (int j = 0; j < h->cfg.head_dim / 2; ++j)
      if (!(inv_freq[j] >= 0.0) || !std::isfinite(inv_freq[j])) return LAZY_ERR_INVALID;
  int n = lazy::launch_build_tables(h, inv_freq, static_cast<cudaStream_t>(stream));
  if (n < 0) return n;
  h->launches += n;
  if (softmax_scale > 0.0) h->shape.scale_log2 = (float)(1.4426950408889634 * softmax_scale);
  return LAZY_OK;
}

int lazy_set_alibi_slopes(lazy_handle* h, const float* slopes, void* stream) {
  if (!h || !slopes) return LAZY_ERR_INVALID;
  if (h->cfg.rope_style != LAZY_POS_ALIBI) return LAZY_ERR_UNSUPPORTED;
  for (int i = 0; i < h->cfg.num_q_heads; ++i) {
    if (!std::isfinite(slopes[i])) return LAZY_ERR_INVALID;
    h->alibi_host[i] = slopes[i] * 1.4426950408889634f;       // the kernels work in log2 units
  }
  // pageable source: the runtime stages it before returning, so later changes of alibi_host are harmless
  if (cudaMemcpyAsync(h->ws.alibi, h->alibi_host, h->cfg.num_q_heads * sizeof(float), cudaMemcpyHostToDevice,
                      static_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LAZY_ERR_CUDA;
  return LAZY_OK;
}

int lazy_set_page_stored_pos(lazy_handle* h, const int32_t* page_stored_pos) {
  if (!h || !page_stored_pos || (reinterpret_cast<uintptr_t>(page_stored_pos) & 3u)) return LAZY_ERR_INVALID;
  if (h->cfg.k_storage != LAZY_K_STORED_POS) return LAZY_ERR_UNSUPPORTED;
  h->page_stored_pos = page_stored_pos;
  return LAZY_OK;
}

int lazy_set_kv_scales(lazy_handle* h, float* k_scale, float* v_scale) {
  if (!h || !k_scale || !v_scale || misaligned(k_scale) || misaligned(v_scale)) return LAZY_ERR_INVALID;
  if (h->cfg.dtype != LAZY_KV_FP8_E4M3) return LAZY_ERR_UNSUPPORTED;
  h->k_scale = k_scale;
  h->v_scale = v_scale;
  return LAZY_OK;
}

int lazy_materialize_pages(lazy_handle* h, const void* k_src, const void* v_src, const int32_t* src_pages,
                           const int32_t* rot_pos, int32_t per_token, void* k_dst, void* v_dst,
                           const int32_t* dst_pages, int32_t num, void* stream) {
  if (!h || num < 0) return LAZY_ERR_INVALID;
  if (h->cfg.dtype != LAZY_KV_BF16) return LAZY_ERR_UNSUPPORTED;
  if (num == 0) return LAZY_OK;
  if (!k_src || !k_dst || !src_pages || !rot_pos || !dst_pages) return LAZY_ERR_INVALID;
  if (misaligned(k_src) || misaligned(k_dst) || misaligned(v_src) || misaligned(v_dst) ||
      (reinterpret_cast<uintptr_t>(src_pages) & 3u) || (reinterpret_cast<uintptr_t>(rot_pos) & 3u) ||
      (reinterpret_cast<uintptr_t>(dst_pages) & 3u))
    return LAZY_ERR_INVALID;
  int n = lazy::launch_materialize(h, k_src, v_src, src_pages, rot_pos, per_token != 0, k_dst, v_dst, dst_pages,
                                   num, static_cast<cudaStream_t>(stream));
  if (n < 0) return n;
  h->launches += n;
  return LAZY_OK;
}

static int check_attn_args(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                           const int32_t* block_table, const int32_t* page_logical_pos,
                           const int32_t* seq_lens, int32_t num_reqs, void* out) {
  if (!h || num_reqs < 0) return LAZY_ERR_INVALID;
  if (h->cfg.k_storage == LAZY_K_STORED_POS && !h->page_stored_pos) return LAZY_ERR_INVALID;
  if (h->cfg.dtype == LAZY_KV_FP8_E4M3 && !h->k_scale) return LAZY_ERR_INVALID;
  if (num_reqs > h->cfg.max_reqs) return LAZY_ERR_INVALID;
  if (num_reqs == 0) return LAZY_OK;
  if (!q || !k_cache || !v_cache || !block_table || !page_logical_pos || !seq_lens || !out)
    return LAZY_ERR_INVALID;
  if (misaligned(q) || misaligned(k_cache) || misaligned(v_cache) || misaligned(out) ||
      (reinterpret_cast<uintptr_t>(block_table) & 3u) || (reinterpret_cast<uintptr_t>(page_logical_pos) & 3u) ||
      (reinterpret_cast<uintptr_t>(seq_lens) & 3u))
    return LAZY_ERR_INVALID;
  return LAZY_OK;
}

int lazy_attn_prefill(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                      const int32_t* block_table, const int32_t* page_logical_pos,
                      const int32_t* seq_lens, const int32_t* cu_q_lens,
                      int32_t num_reqs, int32_t total_q, int32_t max_q_len, void* out, void* stream) {
  int rc = check_attn_args(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, num_reqs, out);
  if (rc != LAZY_OK) return rc;
  if (total_q < 0 || max_q_len < 0) return LAZY_ERR_INVALID;
  if (num_reqs == 0 || total_q == 0) return LAZY_OK;
  if (!cu_q_lens || (reinterpret_cast<uintptr_t>(cu_q_lens) & 3u) || max_q_len == 0) return LAZY_ERR_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int n;
  if (h->cfg.flags & LAZY_FLAG_ROWWISE_KERNELS)
    n = lazy::launch_rowwise(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, cu_q_lens,
                             num_reqs, total_q, max_q_len, out, s);
  else
    n = lazy::launch_prefill(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, cu_q_lens,
                             num_reqs, total_q, max_q_len, out, s);
  if (n < 0) return n;
  h->launches += n;
  return LAZY_OK;
}

int lazy_attn_decode(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                     const int32_t* block_table, const int32_t* page_logical_pos,
                     const int32_t* seq_lens, int32_t num_reqs, void* out, void* stream) {
  int rc = check_attn_args(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, num_reqs, out);
  if (rc != LAZY_OK) return rc;
  if (num_reqs == 0) return LAZY_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int n;
  if (h->cfg.flags & LAZY_FLAG_ROWWISE_KERNELS)
    n = lazy::launch_rowwise(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, nullptr,
                             num_reqs, num_reqs, 1, out, s);
  else
    n = lazy::launch_decode(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, num_reqs, out, s);
  if (n < 0) return n;
  h->launches += n;
  return LAZY_OK;
}

int lazy_attn_mixed(lazy_handle* h, const lazy_mixed_args* a, const void* k_cache, const void* v_cache, void* stream) {
  if (!h || !a) return LAZY_ERR_INVALID;
  if (a->num_reqs_prefill < 0 || a->num_reqs_decode < 0 || a->decode_sms < 0) return LAZY_ERR_INVALID;
  if (h->cfg.flags & LAZY_FLAG_ROWWISE_KERNELS) return LAZY_ERR_UNSUPPORTED;
  const bool has_p = a->num_reqs_prefill > 0 && a->total_q > 0, has_d = a->num_reqs_decode > 0;
  if (!has_p || !has_d) {                       // nothing to overlap: plain calls
    int rc = LAZY_OK;
    if (has_p)
      rc = lazy_attn_prefill(h, a->q_prefill, k_cache, v_cache, a->block_table_prefill, a->page_logical_pos_prefill,
                             a->seq_lens_prefill, a->cu_q_lens, a->num_reqs_prefill, a->total_q, a->max_q_len,
                             a->out_prefill, stream);
    if (rc == LAZY_OK && has_d)
      rc = lazy_attn_decode(h, a->q_decode, k_cache, v_cache, a->block_table_decode, a->page_logical_pos_decode,
                            a->seq_lens_decode, a->num_reqs_decode, a->out_decode, stream);
    return rc;
  }
  if (lazy::mixed_fused_supported(h, a->num_reqs_decode) && !(a->reserved0 & 1)) {
    // one launch: decode CTAs first, prefill CTA pairs behind them (mixed_fused.cu).  Same argument checks as the
    // separate calls.
    int rc = check_attn_args(h, a->q_prefill, k_cache, v_cache, a->block_table_prefill, a->page_logical_pos_prefill,
                             a->seq_lens_prefill, a->num_reqs_prefill, a->out_prefill);
    if (rc == LAZY_OK)
      rc = check_attn_args(h, a->q_decode, k_cache, v_cache, a->block_table_decode, a->page_logical_pos_decode,
                           a->seq_lens_decode, a->num_reqs_decode, a->out_decode);
    if (rc != LAZY_OK) return rc;
    if (a->total_q < 0 || a->max_q_len <= 0 || !a->cu_q_lens || (reinterpret_cast<uintptr_t>(a->cu_q_lens) & 3u))
      return LAZY_ERR_INVALID;
    // decode is HBM-bound and saturates the memory system from a fraction of the SMs; the prefill pairs get the rest
    // (cfg 5 on B200: 142.5 us at 64 decode CTAs, 143.5 at 56, 145.5 at 96, 148 at 128; 177 us as two separate calls)
    const int n_dec = a->decode_sms > 0 ? (a->decode_sms < h->num_sms ? a->decode_sms : h->num_sms) : h->num_sms * 7 / 16;
    const int n = lazy::launch_mixed_fused(h, a, k_cache, v_cache, n_dec, static_cast<cudaStream_t>(stream));
    if (n < 0) return n;
    h->launches += n;
    return LAZY_OK;
  }
  if (!h->side_stream) {
    // all three host resources or none: a half-built set would be used (null events) by the next call
    cudaStream_t st = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const bool ok = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaEventCreateWithFlags(&e0, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&e1, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
      if (e1) cudaEventDestroy(e1);
      if (e0) cudaEventDestroy(e0);
      if (st) cudaStreamDestroy(st);
      return LAZY_ERR_CUDA;
    }
    h->side_stream = st; h->ev_fork = e0; h->ev_join = e1;
  }
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (cudaEventRecord(h->ev_fork, s) != cudaSuccess || cudaStreamWaitEvent(h->side_stream, h->ev_fork, 0) != cudaSuccess)
    return LAZY_ERR_CUDA;
  // decode first, on the side stream, confined to a subset of the SMs (one persistent CTA per SM)
  h->decode_cta_limit = a->decode_sms > 0 ? (a->decode_sms < h->num_sms ? a->decode_sms : h->num_sms) : h->num_sms * 3 / 4;
  int rc = lazy_attn_decode(h, a->q_decode, k_cache, v_cache, a->block_table_decode, a->page_logical_pos_decode,
                            a->seq_lens_decode, a->num_reqs_decode, a->out_decode, h->side_stream);
  h->decode_cta_limit = 0;
  if (rc == LAZY_OK)
    rc = lazy_attn_prefill(h, a->q_prefill, k_cache, v_cache, a->block_table_prefill, a->page_logical_pos_prefill,
                           a->seq_lens_prefill, a->cu_q_lens, a->num_reqs_prefill, a->total_q, a->max_q_len,
                           a->out_prefill, stream);
  // join even on error so the caller's stream never outruns the side stream
  if (cudaEventRecord(h->ev_join, h->side_stream) != cudaSuccess || cudaStreamWaitEvent(s, h->ev_join, 0) != cudaSuccess)
    return LAZY_ERR_CUDA;
  return rc;
}

int64_t lazy_debug_validate(lazy_handle* h, const int32_t* block_table, const int32_t* page_logical_pos,
                            const int32_t* seq_lens, int32_t num_reqs, void* stream) {
  if (!h || num_reqs < 0 || num_reqs > h->cfg.max_reqs) return LAZY_ERR_INVALID;
  if (num_reqs == 0) return 0;
  if (!block_table || !page_logical_pos || !seq_lens) return LAZY_ERR_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int* counter = h->ws.sched + 512;               // a word of the scheduling scratch no kernel uses
  if (cudaMemsetAsync(counter, 0, sizeof(int), s) != cudaSuccess) return LAZY_ERR_CUDA;
  int n = lazy::launch_validate(h, block_table, page_logical_pos, seq_lens, num_reqs, counter, s);
  if (n < 0) return n;
  h->launches += n;
  int host = 0;
  if (cudaMemcpyAsync(&host, counter, sizeof(int), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaStreamSynchronize(s) != cudaSuccess)
    return LAZY_ERR_CUDA;
  return host;
}

const char* lazy_status_string(int status) {
  switch (status) {
    case LAZY_OK: return "ok";
    case LAZY_ERR_INVALID: return "invalid argument";
    case LAZY_ERR_UNSUPPORTED: return "unsupported configuration";
    case LAZY_ERR_WORKSPACE: return "workspace too small or misaligned";
    case LAZY_ERR_CUDA: return "CUDA error at launch";
    case LAZY_ERR_STATIC_LIMIT: return "configuration needs more scratch than LAZY_STATIC_SCRATCH_BYTES";
    default: return "unknown status";
  }
}

int64_t lazy_launch_count(const lazy_handle* h) { return h ? h->launches : 0; }

}  // extern "C"

namespace {
struct StagePlan {
  size_t q, k_new, v_new, slots, bt, pp, sl, cu, out, total;
  size_t q_bytes, kv_bytes, slots_bytes, table_bytes, sl_bytes, cu_bytes;
};
StagePlan stage_plan(const lazy_handle* h, int num_reqs, int total_q, int num_new) {
  StagePlan p{};
  const lazy_config& c = h->cfg;
  p.q_bytes = (size_t)total_q * c.num_q_heads * c.head_dim * 2;
  p.kv_bytes = (size_t)num_new * c.num_kv_heads * c.head_dim * 2;
  p.slots_bytes = (size_t)num_new * sizeof(int64_t);
  p.table_bytes = (size_t)num_reqs * c.max_pages_per_req * sizeof(int32_t);
  p.sl_bytes = (size_t)num_reqs * sizeof(int32_t);
  p.cu_bytes = (size_t)(num_reqs + 1) * sizeof(int32_t);
  size_t off = 0;
  p.q = off;     off = align_up(off + p.q_bytes, 256);
  p.k_new = off; off = align_up(off + p.kv_bytes, 256);
  p.v_new = off; off = align_up(off + p.kv_bytes, 256);
  p.slots = off; off = align_up(off + p.slots_bytes, 256);
  p.bt = off;    off = align_up(off + p.table_bytes, 256);
  p.pp = off;    off = align_up(off + p.table_bytes, 256);
  p.sl = off;    off = align_up(off + p.sl_bytes, 256);
  p.cu = off;    off = align_up(off + p.cu_bytes, 256);
  p.out = off;   off = align_up(off + p.q_bytes, 256);
  p.total = off;
  return p;
}
}  // namespace

extern "C" size_t lazy_host_step_staging_bytes(const lazy_handle* h, int32_t num_reqs, int32_t total_q,
                                               int32_t num_new_tokens) {
  if (!h || num_reqs < 0 || total_q < 0 || num_new_tokens < 0) return 0;
  return stage_plan(h, num_reqs, total_q, num_new_tokens).total;
}

extern "C" int lazy_host_step(lazy_handle* h, const lazy_host_step_args* a, void* stream) {
  if (!h || !a) return LAZY_ERR_INVALID;
  if (a->num_reqs < 0 || a->total_q < 0 || a->num_new_tokens < 0) return LAZY_ERR_INVALID;
  if (a->num_reqs == 0 || a->total_q == 0) return LAZY_OK;
  if (!a->h_q || !a->h_block_table || !a->h_page_logical_pos || !a->h_seq_lens || !a->h_out ||
      !a->d_k_cache || !a->d_v_cache || !a->d_staging)
    return LAZY_ERR_INVALID;
  if (a->kind == 1 && !a->h_cu_q_lens) return LAZY_ERR_INVALID;
  if (a->num_new_tokens > 0 && (!a->h_k_new || !a->h_v_new || !a->h_slot_mapping)) return LAZY_ERR_INVALID;
  StagePlan p = stage_plan(h, a->num_reqs, a->total_q, a->num_new_tokens);
  if ((reinterpret_cast<uintptr_t>(a->d_staging) & 255u) || a->staging_bytes < p.total) return LAZY_ERR_WORKSPACE;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  char* d = static_cast<char*>(a->d_staging);
  bool ok = true;
  auto h2d = [&](size_t off, const void* src, size_t n) {
    if (n) ok = ok && cudaMemcpyAsync(d + off, src, n, cudaMemcpyHostToDevice, s) == cudaSuccess;
  };
  h2d(p.q, a->h_q, p.q_bytes);
  if (a->num_new_tokens > 0) {
    h2d(p.k_new, a->h_k_new, p.kv_bytes);
    h2d(p.v_new, a->h_v_new, p.kv_bytes);
    h2d(p.slots, a->h_slot_mapping, p.slots_bytes);
  }
  h2d(p.bt, a->h_block_table, p.table_bytes);
  h2d(p.pp, a->h_page_logical_pos, p.table_bytes);
  h2d(p.sl, a->h_seq_lens, p.sl_bytes);
  if (a->kind == 1) h2d(p.cu, a->h_cu_q_lens, p.cu_bytes);
  if (!ok) return LAZY_ERR_CUDA;
  int rc = LAZY_OK;
  if (a->num_new_tokens > 0)
    rc = lazy_cache_write(h, d + p.k_new, d + p.v_new, reinterpret_cast<const int64_t*>(d + p.slots),
                          a->num_new_tokens, a->d_k_cache, a->d_v_cache, stream);
  if (rc != LAZY_OK) return rc;
  if (a->kind == 1)
    rc = lazy_attn_prefill(h, d + p.q, a->d_k_cache, a->d_v_cache, reinterpret_cast<const int32_t*>(d + p.bt),
                           reinterpret_cast<const int32_t*>(d + p.pp), reinterpret_cast<const int32_t*>(d + p.sl),
                           reinterpret_cast<const int32_t*>(d + p.cu), a->num_reqs, a->total_q, a->max_q_len,
                           d + p.out, stream);
  else
    rc = lazy_attn_decode(h, d + p.q, a->d_k_cache, a->d_v_cache, reinterpret_cast<const int32_t*>(d + p.bt),
                          reinterpret_cast<const int32_t*>(d + p.pp), reinterpret_cast<const int32_t*>(d + p.sl),
                          a->num_reqs, d + p.out, stream);
  if (rc != LAZY_OK) return rc;
  if (cudaMemcpyAsync(a->h_out, d + p.out, p.q_bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess)
    return LAZY_ERR_CUDA;
  return LAZY_OK;
}


extern "C" int lazy_host_step_layout(const lazy_handle* h, int32_t num_reqs, int32_t total_q, int32_t num_new_tokens,
                                     lazy_host_step_layout_t* out) {
  if (!h || !out || num_reqs < 0 || total_q < 0 || num_new_tokens < 0) return LAZY_ERR_INVALID;
  const StagePlan p = stage_plan(h, num_reqs, total_q, num_new_tokens);
  out->q = p.q; out->k_new = p.k_new; out->v_new = p.v_new; out->slot_mapping = p.slots;
  out->block_table = p.bt; out->page_logical_pos = p.pp; out->seq_lens = p.sl; out->cu_q_lens = p.cu;
  out->out = p.out; out->in_bytes = p.out; out->staging_bytes = p.total;
  return LAZY_OK;
}

extern "C" int lazy_host_step_packed(lazy_handle* h, const lazy_host_step_packed_args* a, void* stream) {
  if (!h || !a) return LAZY_ERR_INVALID;
  if (a->num_reqs < 0 || a->total_q < 0 || a->num_new_tokens < 0) return LAZY_ERR_INVALID;
  if (a->num_reqs == 0 || a->total_q == 0) return LAZY_OK;
  if (!a->h_packed || !a->h_out || !a->d_k_cache || !a->d_v_cache || !a->d_staging) return LAZY_ERR_INVALID;
  const StagePlan p = stage_plan(h, a->num_reqs, a->total_q, a->num_new_tokens);
  if ((reinterpret_cast<uintptr_t>(a->d_staging) & 255u) || a->staging_bytes < p.total) return LAZY_ERR_WORKSPACE;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  char* d = static_cast<char*>(a->d_staging);
  if (cudaMemcpyAsync(d, a->h_packed, p.out, cudaMemcpyHostToDevice, s) != cudaSuccess) return LAZY_ERR_CUDA;
  int rc = LAZY_OK;
  if (a->num_new_tokens > 0)
    rc = lazy_cache_write(h, d + p.k_new, d + p.v_new, reinterpret_cast<const int64_t*>(d + p.slots),
                          a->num_new_tokens, a->d_k_cache, a->d_v_cache, stream);
  if (rc != LAZY_OK) return rc;
  if (a->kind == 1)
    rc = lazy_attn_prefill(h, d + p.q, a->d_k_cache, a->d_v_cache, reinterpret_cast<const int32_t*>(d + p.bt),
                           reinterpret_cast<const int32_t*>(d + p.pp), reinterpret_cast<const int32_t*>(d + p.sl),
                           reinterpret_cast<const int32_t*>(d + p.cu), a->num_reqs, a->total_q, a->max_q_len,
                           d + p.out, stream);
  else
    rc = lazy_attn_decode(h, d + p.q, a->d_k_cache, a->d_v_cache, reinterpret_cast<const int32_t*>(d + p.bt),
                          reinterpret_cast<const int32_t*>(d + p.pp), reinterpret_cast<const int32_t*>(d + p.sl),
                          a->num_reqs, d + p.out, stream);
  if (rc != LAZY_OK) return rc;
  if (cudaMemcpyAsync(a->h_out, d + p.out, p.q_bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess) return LAZY_ERR_CUDA;
  return LAZY_OK;
}
