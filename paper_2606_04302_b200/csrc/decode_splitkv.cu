// decode_splitkv.cu -- placeholder: routes to the row-wise kernel until the split-KV kernel lands.
#include "lazy_internal.h"
namespace lazy {
int launch_decode(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                  const int32_t* block_table, const int32_t* page_logical_pos, const int32_t* seq_lens,
                  int num_reqs, void* out, cudaStream_t stream) {
  return launch_rowwise(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, nullptr, num_reqs,
                        num_reqs, 1, out, stream);
}
}  // namespace lazy
