// lazy_internal.h -- shared by the translation units of liblazyattn.so (never by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>

#include "lazy_attn.h"

namespace lazy {

constexpr int kPageSize = 16;
constexpr int kMaxDecodeCtas = 1024;   // upper bound on the decode grid (sizes the partial buffers)
constexpr int kKmAlibi = 3;            // kernel template value next to LAZY_K_*: no rotation, ALiBi score bias
constexpr int kMaxAlibiHeads = 256;

// Device-side views the kernels take by value.
struct Shape {
  int Hq, Hkv, D, group;
  int table_stride;      // max_pages_per_req
  int max_position;
  float scale_log2;      // log2(e) / sqrt(D)
};

struct Workspace {
  float2* cs;            // [max_position][D/2] (cos, sin) of pos * theta_j, built from fp64 angles
  float*  part_o;        // [max_reqs + kMaxDecodeCtas][Hq][D] fp32 un-normalised partial outputs
  float2* part_ml;       // [max_reqs + kMaxDecodeCtas][Hq] (running max in log2 units, sum)
  int*    req_counter;   // [max_reqs] arrival counters for the in-kernel combine (self-resetting)
  int*    sched;         // small scratch for device-side scheduling
  float*  alibi;         // [kMaxAlibiHeads] slopes * log2(e) (LAZY_POS_ALIBI)
};

}  // namespace lazy

struct lazy_handle {
  lazy_config cfg;
  lazy::Shape shape;
  lazy::Workspace ws;
  int num_sms;
  int64_t launches;
  const int32_t* page_stored_pos;   // LAZY_K_STORED_POS: device [num_pages], caller-owned
  float* k_scale;                   // LAZY_KV_FP8_E4M3: device [num_pages][Hkv][16] per-row scales, caller-owned
  float* v_scale;
  int decode_cta_limit;             // > 0: lazy_attn_mixed confines the decode kernel to this many CTAs (= SMs)
  cudaStream_t side_stream;         // lazy_attn_mixed: library-owned fork stream and its two events (host resources)
  cudaEvent_t ev_fork, ev_join;
  float alibi_host[lazy::kMaxAlibiHeads];   // staging copy of the slopes (source of the async H2D copy)
  // cached TMA descriptors (128 bytes each), keyed by the pool pointer they were encoded for
  alignas(64) unsigned char tmap_k[128];
  alignas(64) unsigned char tmap_v[128];
  const void* tmap_k_ptr;
  const void* tmap_v_ptr;
  alignas(64) unsigned char tmap_pk[128];
  alignas(64) unsigned char tmap_pv[128];
  alignas(64) unsigned char tmap_pq[128];
  const void* tmap_pk_ptr;
  const void* tmap_pv_ptr;
  const void* tmap_pq_ptr;
  int tmap_pq_rows;
};

namespace lazy {

// TMA descriptors (cuTensorMapEncodeTiled through the runtime's driver entry point; 128-byte swizzle).
//   pool : 2-D view [num_pages*Hkv*16 rows][D], box = [box_rows][64 columns]
//   q    : 4-D view (D, group, Hkv, total_q) of q [total_q][Hq][D], box = (64, group, 1, tokens_per_tile):
//          lands as rows token*group + head-in-group of one kv head's GQA group.
bool encode_pool_tmap(void* out_map, const void* pool, long long rows, int D, int box_rows);
bool encode_pool_tmap_u8(void* out_map, const void* pool, long long rows, int D, int box_rows, bool swizzle,
                         int box_cols);
bool encode_q_tmap(void* out_map, const void* q, int total_q, int Hq, int Hkv, int D, int tokens_per_tile);

// Each launcher enqueues on `stream` and returns the number of kernels launched (<0: LAZY_ERR_*).
int launch_build_tables(lazy_handle* h, const double* inv_freq_host, cudaStream_t stream);
int launch_cache_write(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                       int num_tokens, void* k_cache, void* v_cache, cudaStream_t stream);
// LAZY_KV_FP8_E4M3 (fp8_kernels.cu): quantising cache write, row-wise debug attention over FP8 pages
int launch_cache_write_fp8(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                           int num_tokens, void* k_cache, void* v_cache, cudaStream_t stream);
int launch_rowwise_fp8(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                       const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                       const int32_t* cu_q_lens, int num_reqs, int total_q, void* out, cudaStream_t stream);
int launch_materialize(lazy_handle* h, const void* k_src, const void* v_src, const int32_t* src_pages,
                       const int32_t* rot_pos, int per_token, void* k_dst, void* v_dst, const int32_t* dst_pages,
                       int num, cudaStream_t stream);
int launch_validate(lazy_handle* h, const int32_t* block_table, const int32_t* page_logical_pos,
                    const int32_t* seq_lens, int num_reqs, int* counter, cudaStream_t stream);
int launch_rowwise(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                   const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                   const int32_t* cu_q_lens, int num_reqs, int total_q, int max_q_len, void* out,
                   cudaStream_t stream);
int launch_decode(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                  const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                  int num_reqs, void* out, cudaStream_t stream);
// one launch for a mixed prefill + decode step (mixed_fused.cu); supported for the product configuration only
bool mixed_fused_supported(const lazy_handle* h, int num_reqs_decode);
int launch_mixed_fused(lazy_handle* h, const lazy_mixed_args* m, const void* k_cache, const void* v_cache, int decode_ctas,
                       cudaStream_t stream);
int launch_prefill(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                   const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                   const int32_t* cu_q_lens, int num_reqs, int total_q, int max_q_len, void* out,
                   cudaStream_t stream);

}  // namespace lazy
