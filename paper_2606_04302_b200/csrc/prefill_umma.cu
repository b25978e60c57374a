// prefill_umma.cu -- placeholder: routes to the row-wise kernel until the tcgen05 kernel lands.
#include "lazy_internal.h"
namespace lazy {
int launch_prefill(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                   const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                   const int32_t* cu_q_lens, int num_reqs, int total_q, int max_q_len, void* out,
                   cudaStream_t stream) {
  return launch_rowwise(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, cu_q_lens, num_reqs,
                        total_q, max_q_len, out, stream);
}
}  // namespace lazy
