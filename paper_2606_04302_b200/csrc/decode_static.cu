// decode_static.cu -- lazy_attn_decode_static: the split-KV decode for callers that have no device memory to give.
//
// Every other call of this library works inside a `workspace` the caller allocated on the device (lazy_create).
// Some callers cannot do that: a plugin or custom op running inside a host framework that has already handed all
// device memory to its own pool and forbids raw cudaMalloc; a latency-critical serving loop in which cudaMalloc is
// banned because it synchronises the whole device; a component that is only ever given the input and output
// buffers of one call.  For them the decode kernel's scratch -- split-KV partial outputs, the per-request arrival
// counters of the in-kernel combine and the cos/sin table -- lives in the file-scope array below, which the CUDA
// driver places in device memory when it loads this module.  Nothing in this file (or below it) calls cudaMalloc,
// cudaFree, a stream-ordered allocator or a library routine that allocates device memory; the only allocation at all
// is the few-hundred-byte HOST description of the scratch carving made at set-up.
//
// The array is LAZY_STATIC_SCRATCH_BYTES (48 MiB) long.  Each GPU on which this module gets loaded holds its own copy
// until the process exits; that is the price of the entry point, paid whether or not it is ever called again.
#include <mutex>

#include "lazy_internal.h"

// Device memory.  In HOST code this name is only a handle for the runtime's symbol calls -- it is not a device
// address and must never be handed to a kernel; the address is asked for once per device (device_slot_ready below).
static __device__ __align__(256) unsigned char lazy_static_scratch[LAZY_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;

struct DeviceSlot {
  void* scratch;         // device address of lazy_static_scratch ON THIS DEVICE; null until resolved
  lazy_handle* handle;   // host-side carving of the scratch for `cfg` (lazy_create over `scratch`)
  lazy_config cfg;       // configuration `handle` was made for
};

DeviceSlot g_slots[kMaxDevices];
std::mutex g_mutex;      // protects g_slots: the entry point may be called from several host threads

bool same_config(const lazy_config& a, const lazy_config& b) {
  return a.num_q_heads == b.num_q_heads && a.num_kv_heads == b.num_kv_heads && a.head_dim == b.head_dim &&
         a.page_size == b.page_size && a.num_pages == b.num_pages && a.max_position == b.max_position &&
         a.max_reqs == b.max_reqs && a.max_pages_per_req == b.max_pages_per_req && a.rope_theta == b.rope_theta &&
         a.rope_style == b.rope_style && a.dtype == b.dtype && a.flags == b.flags && a.k_storage == b.k_storage;
}

// Set-up, with the caller's device current.  Resolves the array's address on this device the first time, and
// (re)carves the array whenever the configuration differs from the previous call's: lazy_create zeroes the arrival
// counters and enqueues the cos/sin table build on `stream`, so a layout left behind by another configuration is
// never read.
int device_slot_ready(DeviceSlot& slot, const lazy_config* cfg, cudaStream_t stream) {
  if (!slot.scratch) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, lazy_static_scratch) != cudaSuccess || !ptr) {
      (void)cudaGetLastError();
      return LAZY_ERR_CUDA;
    }
    slot.scratch = ptr;
  }
  if (slot.handle && same_config(slot.cfg, *cfg)) return LAZY_OK;
  if (slot.handle) {
    lazy_destroy(slot.handle);
    slot.handle = nullptr;
  }
  const int rc = lazy_create(cfg, slot.scratch, LAZY_STATIC_SCRATCH_BYTES, stream, &slot.handle);
  if (rc != LAZY_OK) {
    slot.handle = nullptr;
    return rc;
  }
  slot.cfg = *cfg;
  return LAZY_OK;
}

}  // namespace

extern "C" int lazy_attn_decode_static(const lazy_config* cfg, const void* q, const void* k_cache, const void* v_cache,
                                       const int32_t* block_table, const int32_t* page_logical_pos,
                                       const int32_t* seq_lens, int32_t num_reqs, void* out, void* stream) {
  if (!cfg) return LAZY_ERR_INVALID;
  // the product configuration only: the other layouts need per-handle side arrays (scales, stored positions, slopes)
  if (cfg->dtype != LAZY_KV_BF16 || cfg->k_storage != LAZY_K_UNROTATED || cfg->rope_style == LAZY_POS_ALIBI ||
      cfg->flags != 0)
    return LAZY_ERR_UNSUPPORTED;
  const size_t need = lazy_workspace_bytes(cfg);          // 0: invalid or unsupported shape
  if (need == 0) return LAZY_ERR_UNSUPPORTED;
  if (need > (size_t)LAZY_STATIC_SCRATCH_BYTES) return LAZY_ERR_STATIC_LIMIT;
  if (num_reqs < 0 || num_reqs > cfg->max_reqs) return LAZY_ERR_INVALID;

  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return LAZY_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return LAZY_ERR_UNSUPPORTED;

  std::lock_guard<std::mutex> lock(g_mutex);
  DeviceSlot& slot = g_slots[dev];
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = device_slot_ready(slot, cfg, s);
  if (rc != LAZY_OK) return rc;
  if (num_reqs == 0) return LAZY_OK;

  // The array keeps whatever the previous call left.  The combine counts arrivals from zero; a completed call puts
  // its counters back to zero itself, but a call that was cut short (a launch error further down the stream, a
  // reset pool) would not have, so they are cleared every time.  Partials and the table need no clearing: every
  // partial slot is written before it is read, and the table depends on `cfg` only.
  lazy_handle* h = slot.handle;
  const size_t counter_bytes = reinterpret_cast<char*>(h->ws.sched) - reinterpret_cast<char*>(h->ws.req_counter);
  if (cudaMemsetAsync(h->ws.req_counter, 0, counter_bytes, s) != cudaSuccess) return LAZY_ERR_CUDA;
  return lazy_attn_decode(h, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, num_reqs, out, stream);
}
