/*
 * lazy_attn.h -- C ABI of liblazyattn.so: the LazyAttention hot path on B200 (sm_100a).
 *
 * Paged attention over a KV cache that stores keys UN-ROTATED (pre-RoPE).  Every page of a request
 * carries, next to its physical page id, the logical position of its first token; the kernels apply
 * RoPE on chip, so one physical copy of a document's KV serves many requests at different positions
 * with no materialised re-encoding and no writes on the read path.
 *
 * What the calls compute is defined by the paper (arxiv/paper_2606_04302, /root/reference/PAPER.md):
 *   - deferred positional encoding: Q/K/V are produced without positions, RoPE is applied during
 *     attention after fetching from the cache (section 3.1; Fig. 1b L29-31);
 *   - attention with RoPE  softmax(f(Q,m) f(K,n)^T / sqrt(d_k)) V  (Eq. 4);
 *   - half-split rotation  k1' = k1 cos - k2 sin, k2' = k1 sin + k2 cos  (Fig. 3b);
 *   - one cached copy reused by several requests at different global offsets inside one batch
 *     (PAPER.md L83-88 problem statement; L173/L182 offsets carried as metadata);
 *   - the result is exactly what duplicating + re-encoding the KV would give.
 * Readings taken where the paper is silent are listed in DESIGN.md ("Readings of the paper").
 *
 * Conventions common to all calls
 *   - All tensor pointers are DEVICE pointers owned by the caller, 16-byte aligned, bf16 unless stated.
 *     `cfg`, `out` handle pointers and the returned strings are HOST pointers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Every call only
 *     enqueues work on it: no host synchronisation, no device allocation, no host<->device copies.
 *   - The library owns nothing on the device except what it places inside the caller's `workspace`.
 *   - lazy_attn_* never write k_cache / v_cache (read path is read-only).
 *   - Return value: 0 = OK, <0 = error (lazy_status_string).  Errors are detected on the host from the
 *     scalar arguments only; the CONTENTS of device tables are trusted (page id >= num_pages or a
 *     position >= max_position is undefined behaviour).
 *   - Pool layout (frozen):  k_cache, v_cache : [num_pages][num_kv_heads][page_size][head_dim] bf16.
 *     K holds the projection output with NO rotary applied; token t of a page sits at logical position
 *     page_logical_pos + t.
 *   - Sequence model: request r has seq_lens[r] tokens; token s lives in table slot s / page_size at
 *     in-page offset s % page_size.  The query tokens of a call are the LAST tokens of the sequence and
 *     are already in the cache (lazy_cache_write first, same stream).  Causal mask is by sequence index
 *     (key s visible to the query with index sq iff s <= sq); positions feed RoPE only.
 *   - GQA: q head hq reads kv head hq / (num_q_heads / num_kv_heads).
 *   - Scale 1/sqrt(head_dim); theta_j = rope_theta^(-2j/head_dim), j < head_dim/2; pair (j, j+head_dim/2).
 */
#ifndef LAZY_ATTN_H_
#define LAZY_ATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lazy_handle lazy_handle;

typedef struct lazy_config {
  int32_t num_q_heads;       /* Hq                                                              */
  int32_t num_kv_heads;      /* Hkv; Hq % Hkv == 0, group = Hq/Hkv <= 8; Hkv in {1,2,4} or a multiple of 8 */
  int32_t head_dim;          /* D in {64, 128}                                                  */
  int32_t page_size;         /* 16                                                              */
  int32_t num_pages;         /* physical pool size (pages)                                      */
  int32_t max_position;      /* logical positions lie in [0, max_position)                      */
  int32_t max_reqs;          /* upper bound on num_reqs of any call                             */
  int32_t max_pages_per_req; /* row stride (in entries) of block_table and page_logical_pos     */
  double  rope_theta;        /* 1e4, 5e5, 1e6 ...                                               */
  int32_t rope_style;        /* LAZY_ROPE_* : pairing of the rotated dimensions (0 = half-split)  */
  int32_t dtype;             /* LAZY_KV_* : what the KV pages hold (0 = bf16; q, k_new, v_new, out are always bf16) */
  int32_t flags;             /* LAZY_FLAG_* (0 for production)                                  */
  int32_t k_storage;         /* LAZY_K_* : how the pages hold K (0 = un-rotated, the product)    */
} lazy_config;

/* rope_style (section 3.5).
 *   LAZY_ROPE_HALF_SPLIT  pair (j, j + D/2)  (the product path).
 *   LAZY_ROPE_INTERLEAVED pair (2j, 2j + 1)  (L215).  q and k_new arrive in the model's own dimension order;
 *                         lazy_cache_write stores K rows DE-INTERLEAVED (dims 0,2,4,... then 1,3,5,...), which is
 *                         still position-free, and the attention kernels de-interleave q on load: interleaved RoPE
 *                         on x equals half-split RoPE on de-interleaved x, and a dot product does not care about a
 *                         permutation applied to both operands.  k_cache's last axis is therefore in that order
 *                         (V and every output are untouched).
 *   LAZY_POS_ALIBI        no rotation at all: ALiBi.  K and q are used as they are and the score of
 *                         the query at logical position m with the key at logical position n gets the bias
 *                         slope[hq] * (n - m) added after scaling (lazy_set_alibi_slopes; slopes start as 0).
 *                         The positions are the same per-page logical positions RoPE would use, so a cached page
 *                         is reusable at any offset exactly as with RoPE.  k_storage must be LAZY_K_UNROTATED. */
#define LAZY_ROPE_HALF_SPLIT  0
#define LAZY_ROPE_INTERLEAVED 1
#define LAZY_POS_ALIBI        2

/* k_storage: what a physical page's K rows carry (V is position-free in every mode).
 *   LAZY_K_UNROTATED  the product path (north_star): K is the projection output, the kernels
 *                     rotate token t of a page by page_logical_pos + t.
 *   LAZY_K_STORED_POS the paper's own layout ("local position ... indexing from 0", L409): token
 *                     t of physical page g was stored rotated by page_stored_pos[g] + t
 *                     (lazy_set_page_stored_pos); the kernels apply ONE relative rotation per page by
 *                     D = page_logical_pos - page_stored_pos[g] -- to the K tile in prefill (Eq. 5),
 *                     to q in decode (Eq. 6).  |D| and every position must be < max_position.
 *   LAZY_K_ABSOLUTE   position-dependent cache (standard attention, the "without deferred rotation" arm of
 *                     PAPER.md Fig. 5 / L271-297): K is stored rotated at its final position, nothing is
 *                     rotated but q (by the position of its own token).  Pages cannot be shared across
 *                     positions in this mode; it exists to measure what the rotation costs. */
#define LAZY_K_UNROTATED  0
#define LAZY_K_STORED_POS 1
#define LAZY_K_ABSOLUTE   2

/* dtype: storage format of the KV pages (SURVEY.md 8.0 row f4 "FP8 KV pages").  The paper's cache holds "purely
 * content-based keys and values" -- a page carries no position, so a QUANTISED page is as shareable
 * at any logical offset as a bf16 one -- and decode moves 2LD bytes (L204-209), which this halves.  The paper defines
 * no quantised format; this one is the repository's:
 *   LAZY_KV_BF16      the pool layout above.
 *   LAZY_KV_FP8_E4M3  k_cache, v_cache : [num_pages][num_kv_heads][page_size][head_dim] bytes, OCP FP8 E4M3 codes of
 *                     the un-rotated K row / of the V row divided by a per-row scale; the scales are two more device
 *                     arrays [num_pages][num_kv_heads][page_size] fp32 registered with lazy_set_kv_scales (per token,
 *                     because lazy_cache_write appends single tokens to half-filled pages).  lazy_cache_write
 *                     quantises: scale = max|row| / 448 in fp32 (1 for an all-zero row), code = nearest E4M3 (ties
 *                     to even, saturating) of the fp32 quotient row[d] / scale.  k_new / v_new must be FINITE: a row
 *                     with an Inf or NaN element is not rejected (there is no device-side error channel) but stored so
 *                     that it reads back as NaN -- Inf makes the row's scale inf (code x inf = NaN for every element),
 *                     a NaN element becomes the E4M3 NaN code -- and every query that sees the token returns NaN, as
 *                     it would on bf16 pages.  q may have any finite bf16 magnitude (the FP8 decode kernel, which
 *                     multiplies in f16, normalises q by a power of two first).  The attention calls compute what the
 *                     bf16 calls would compute on the exactly dequantised pages (code value x scale).  Supported
 *                     with both RoPE pairings (not ALiBi) and LAZY_K_UNROTATED; lazy_materialize_pages is bf16-only.  Every call
 *                     runs on the product kernels at either head_dim (split-KV decode; tcgen05 prefill, on CTA pairs
 *                     at head_dim 128; the one-launch mixed step at head_dim 128). */
#define LAZY_KV_BF16      0
#define LAZY_KV_FP8_E4M3  1

/* flags: debugging aids, never set by bench.py */
#define LAZY_FLAG_ROWWISE_KERNELS 1  /* run the simple one-row-per-CTA CUDA kernels for prefill and decode */
#define LAZY_FLAG_PREFILL_ONE_CTA 2  /* head_dim 128: run prefill on single CTAs (prefill_umma.cu) instead of CTA
                                      pairs (prefill_umma2.cu); the A/B arm of DESIGN.md 6.2 */

#define LAZY_FLAG_FP8_DECODE_8_WARPS 4  /* LAZY_KV_FP8_E4M3 decode with the bf16 kernel's 8 consumer warps instead of 12
                                        (the A/B arm of DESIGN.md 6.7) */

#define LAZY_OK               0
#define LAZY_ERR_INVALID     -1  /* null / misaligned pointer, negative count, num_reqs > max_reqs ...     */
#define LAZY_ERR_UNSUPPORTED -2  /* head_dim, page_size, head grouping, dtype or rope_style not supported  */
#define LAZY_ERR_WORKSPACE   -3  /* workspace too small or misaligned                                      */
#define LAZY_ERR_CUDA        -4  /* CUDA error at launch (cudaGetLastError)                                */
#define LAZY_ERR_STATIC_LIMIT -5 /* lazy_attn_decode_static: cfg needs more scratch than LAZY_STATIC_SCRATCH_BYTES */

/* Bytes of device workspace lazy_create needs for `cfg` (RoPE cos/sin table built from fp64 angles --
 * PAPER.md L138/L173 "loaded from a table", L455 stateless absolute-index rotation -- plus split-KV
 * partials, PAPER-external: north_star "split-KV flash-decoding ... and a combine pass").
 * Returns 0 if cfg is NULL or unsupported. */
size_t lazy_workspace_bytes(const lazy_config* cfg);

/* Creates a handle (host memory) over caller-owned device `workspace` (256-byte aligned, at least
 * lazy_workspace_bytes(cfg)); enqueues the table build on `stream`.  The workspace must stay alive and
 * untouched by the caller until lazy_destroy.  One host thread at a time per handle. */
int lazy_create(const lazy_config* cfg, void* workspace, size_t workspace_bytes, void* stream,
                lazy_handle** out);
void lazy_destroy(lazy_handle* h);

/* a0. Store un-rotated K and V rows of new tokens into physical pages ("purely
 * content-based keys and values"; L188).  Pure data movement, bit exact.
 *   k_new, v_new : [num_tokens][Hkv][D] bf16     slot_mapping : [num_tokens] int64,
 *   slot = page*page_size + offset, slot < 0 skips the token.  num_tokens == 0 -> no launch. */
int lazy_cache_write(lazy_handle* h, const void* k_new, const void* v_new, const int64_t* slot_mapping,
                     int32_t num_tokens, void* k_cache, void* v_cache, void* stream);

/* Prefill: a chunk of n_q[r] = cu_q_lens[r+1]-cu_q_lens[r] query tokens per request (the last n_q[r]
 * tokens of its sequence) attends to all earlier tokens (shared document pages, at the logical
 * positions this request gives them) and causally to itself (Fig. 5 phase 2; K rotated
 * once per tile, L164-173).  Block-local document prefill is the case n_q == seq_len.
 *   q, out           : [total_q][Hq][D] bf16 (q un-rotated)
 *   block_table      : [num_reqs][max_pages_per_req] int32 physical page per slot
 *   page_logical_pos : same shape, logical position of token 0 of that page
 *   seq_lens         : [num_reqs] int32 KV length INCLUDING the chunk;  cu_q_lens : [num_reqs+1] int32
 *   max_q_len        : host upper bound on n_q[r] (sizes the grid)
 * Rows of a request with seq_len == 0 are written as zeros.  num_reqs == 0 or total_q == 0 -> no launch. */
int lazy_attn_prefill(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                      const int32_t* block_table, const int32_t* page_logical_pos,
                      const int32_t* seq_lens, const int32_t* cu_q_lens,
                      int32_t num_reqs, int32_t total_q, int32_t max_q_len, void* out, void* stream);

/* Decode: one query per request (its last token) over the whole sequence (Fig. 3c;
 * T_decode ~ 2LD/B, L204-209).  Split-KV flash-decoding with an in-kernel combine.
 *   q, out : [num_reqs][Hq][D] bf16.  Other arguments as for prefill.
 * ONE decode call in flight per handle: the split-KV partials, the per-request arrival counters and the scheduling
 * words live in the handle's workspace, so a second lazy_attn_decode (or lazy_attn_mixed / lazy_host_step*) on the
 * same handle may only be enqueued on the SAME stream, behind the first.  Use one handle per concurrent stream. */
int lazy_attn_decode(lazy_handle* h, const void* q, const void* k_cache, const void* v_cache,
                     const int32_t* block_table, const int32_t* page_logical_pos,
                     const int32_t* seq_lens, int32_t num_reqs, void* out, void* stream);

/* Decode WITHOUT a caller-provided workspace, for callers that cannot allocate device memory: code that runs inside
 * a host framework which owns all device memory and forbids raw cudaMalloc, serving loops where cudaMalloc is banned
 * because it synchronises the device, components that only ever see the input and output buffers of one call.  Same
 * computation, same kernel and same results as lazy_create + lazy_attn_decode with `cfg`; the scratch that call keeps
 * in the workspace (cos/sin table, split-KV partials, arrival counters) lives in a device array that is part of the
 * library image: LAZY_STATIC_SCRATCH_BYTES per GPU that loads it, held until the process exits.  The call and
 * everything under it use no cudaMalloc / cudaFree / allocating library routine.
 *   cfg   : HOST pointer.  bf16 pages, LAZY_K_UNROTATED, a RoPE pairing (not ALiBi), flags == 0, otherwise
 *           LAZY_ERR_UNSUPPORTED.  lazy_workspace_bytes(cfg) must be <= LAZY_STATIC_SCRATCH_BYTES, otherwise
 *           LAZY_ERR_STATIC_LIMIT and nothing is enqueued (at Hq 32 / Hkv 8 / D 128 / 64 requests the limit is reached
 *           near max_position = 60000; lower max_position or max_reqs to fit).
 *   other arguments: as lazy_attn_decode.  num_reqs <= cfg->max_reqs.
 * Set-up: the FIRST call on a device, and any call whose cfg differs from the previous call's on that device, also
 * looks up the array's device address, clears the counters and enqueues the table build (one extra launch) on
 * `stream` ahead of the decode kernel; later calls with the same cfg enqueue one small memset and the kernel.  Make
 * that first call during start-up, before any stream capture is begun.
 * Sharing: there is ONE array per GPU and every call on that GPU uses it.  Two calls whose GPU work may overlap
 * (different streams without an event between them, or different host threads racing to enqueue) corrupt each other's
 * partials -- keep all calls on one stream or order them yourself.  Host-side the call is thread-safe. */
#define LAZY_STATIC_SCRATCH_BYTES (48u << 20)
int lazy_attn_decode_static(const lazy_config* cfg, const void* q, const void* k_cache, const void* v_cache,
                            const int32_t* block_table, const int32_t* page_logical_pos,
                            const int32_t* seq_lens, int32_t num_reqs, void* out, void* stream);

/* f3. Frequency-scaled RoPE families (Llama-3.1 / NTK / YaRN scaling only change "variant-specific
 * scaling metadata").  Replaces the rotation frequency of pair j, theta_j = rope_theta^(-2j/D), by inv_freq[j]
 * (HOST array of head_dim/2 doubles; NULL restores the default) and rebuilds the fp64-built cos/sin table on `stream`
 * (one launch; attention calls enqueued later on the same stream see the new table).  A pair with frequency 0 is
 * not rotated (partial rotary).  softmax_scale > 0 replaces 1/sqrt(head_dim) (YaRN's attention temperature);
 * 0 keeps the current one. */
int lazy_set_rope_frequencies(lazy_handle* h, const double* inv_freq, double softmax_scale, void* stream);

/* LAZY_POS_ALIBI only: per-q-head slopes (HOST array of num_q_heads floats, natural-log domain as in the ALiBi
 * definition: bias = slope * (n - m)).  Copied into the workspace on `stream`. */
int lazy_set_alibi_slopes(lazy_handle* h, const float* slopes, void* stream);

/* LAZY_K_STORED_POS only: device array [num_pages] int32, position at which token 0 of each physical page
 * was rotated when it was stored.  The pointer is kept (not copied) and read by every later attention call;
 * it must stay valid until lazy_destroy or the next lazy_set_page_stored_pos.  Host-side, no launch. */
int lazy_set_page_stored_pos(lazy_handle* h, const int32_t* page_stored_pos);

/* LAZY_KV_FP8_E4M3 only: device arrays [num_pages][num_kv_heads][page_size] fp32 holding the per-row scales of the
 * K and V code pools.  lazy_cache_write fills them, the attention calls read them.  The pointers are kept (not
 * copied) and must stay valid until lazy_destroy or the next lazy_set_kv_scales; 16-byte aligned.  Host-side, no
 * launch. */
int lazy_set_kv_scales(lazy_handle* h, float* k_scale, float* v_scale);

/* f2. Materialising re-encoding of whole pages: what a position-dependent cache does on a position mismatch
 * ("allocate + copy + rotate", App. B; "read-modify-write ... doubling HBM traffic", L447) and
 * what the lazy path avoids.  It is also the writer for the LAZY_K_STORED_POS / LAZY_K_ABSOLUTE layouts.
 * For i < num, every kv head, token t < page_size:
 *     k_dst[dst_pages[i]][hk][t][:] = bf16( RoPE(k_src[src_pages[i]][hk][t][:], rot_pos[i] + (per_token ? t : 0)) )
 *     v_dst[dst_pages[i]][hk][t][:] = v_src[src_pages[i]][hk][t][:]          (skipped if v_src or v_dst is NULL)
 * per_token = 1 encodes an un-rotated page at logical start rot_pos[i] >= 0; per_token = 0 applies one
 * relative rotation rot_pos[i] (may be negative) to a page that already carries positions.
 *   src_pages, dst_pages, rot_pos : device int32 [num];  |rot_pos[i]| + page_size <= max_position.
 * Source and destination pools have the pool layout; they may be the same pool (dst_pages[i] == src_pages[i]
 * re-encodes in place: the in-place update that races under sharing).  Destination pages must be
 * distinct.  fp32 rotation from the fp64-built table, one rounding to bf16.  num == 0 -> no launch. */
int lazy_materialize_pages(lazy_handle* h, const void* k_src, const void* v_src, const int32_t* src_pages,
                           const int32_t* rot_pos, int32_t per_token, void* k_dst, void* v_dst,
                           const int32_t* dst_pages, int32_t num, void* stream);

/* Static description of a status code (host string, never NULL). */
const char* lazy_status_string(int status);

/* Debug aid (the ONLY synchronising call; never on the serving path): checks the CONTENTS of the device tables
 * that the attention calls trust -- for every request r < num_reqs and every slot below ceil(seq_len / page_size):
 * 0 <= block_table < num_pages, 0 <= page_logical_pos and page_logical_pos + page_size <= max_position; and
 * 0 <= seq_len <= max_pages_per_req * page_size.  Returns the number of violations (>= 0) after synchronising
 * `stream`, or a negative status.  Uses 4 bytes of the workspace. */
int64_t lazy_debug_validate(lazy_handle* h, const int32_t* block_table, const int32_t* page_logical_pos,
                            const int32_t* seq_lens, int32_t num_reqs, void* stream);

/* Introspection for tests and bench.py: number of kernel launches this handle has enqueued so far. */
int64_t lazy_launch_count(const lazy_handle* h);

/* End-to-end convenience call over HOST buffers (the e2e leg of bench.py): one serving step =
 * optional lazy_cache_write of the step's new tokens + one attention call, with every per-step input
 * (q, k_new, v_new, slot_mapping, block_table, page_logical_pos, seq_lens, cu_q_lens) copied host->device
 * into the caller's device staging area and `out` copied device->host, all enqueued on `stream`
 * (cudaMemcpyAsync; host buffers should be pinned).  The KV pool stays resident on the device -- that is
 * the point of the method (cached documents are served from GPU memory).
 * Pointers named h_* are HOST, d_* DEVICE.  The tables are [num_reqs][max_pages_per_req] int32.
 * The call returns after enqueueing; synchronise the stream before reading h_out. */
typedef struct lazy_host_step_args {
  int32_t kind;              /* 0 = decode, 1 = prefill                                   */
  int32_t num_reqs;
  int32_t total_q;           /* decode: == num_reqs                                       */
  int32_t max_q_len;         /* decode: 1                                                 */
  int32_t num_new_tokens;    /* rows of h_k_new/h_v_new/h_slot_mapping; 0 = no cache write */
  int32_t reserved;
  const void* h_q;           /* [total_q][Hq][D] bf16                                     */
  const void* h_k_new;       /* [num_new_tokens][Hkv][D] bf16 or NULL                     */
  const void* h_v_new;
  const int64_t* h_slot_mapping;
  const int32_t* h_block_table;
  const int32_t* h_page_logical_pos;
  const int32_t* h_seq_lens;
  const int32_t* h_cu_q_lens; /* prefill only                                             */
  void* h_out;               /* [total_q][Hq][D] bf16                                     */
  void* d_k_cache;
  void* d_v_cache;
  void* d_staging;           /* device scratch, 256-byte aligned                          */
  size_t staging_bytes;      /* >= lazy_host_step_staging_bytes(...)                      */
} lazy_host_step_args;

size_t lazy_host_step_staging_bytes(const lazy_handle* h, int32_t num_reqs, int32_t total_q,
                                    int32_t num_new_tokens);
int lazy_host_step(lazy_handle* h, const lazy_host_step_args* a, void* stream);

/* d'. The same step with the inputs PACKED by the caller into one pinned host block laid out like the device staging
 * area, so that the whole step costs ONE host-to-device copy, the kernels and ONE device-to-host copy (with seven
 * separate copies of a few KB to 1 MB each, copy issue latency -- not bandwidth -- was half of cfg 2's end-to-end
 * time).  lazy_host_step_layout fills the byte offsets of each section inside the block (all 256-byte aligned; a
 * section the step does not use keeps its slot) and `in_bytes`, the length of the single H2D copy; the output section
 * starts at `out` in the DEVICE staging area only (h_out is a separate host buffer).  Sections hold exactly what the
 * h_* pointers of lazy_host_step_args hold.  Returns LAZY_ERR_INVALID on bad counts. */
typedef struct lazy_host_step_layout_t {
  size_t q, k_new, v_new, slot_mapping, block_table, page_logical_pos, seq_lens, cu_q_lens, out;
  size_t in_bytes;           /* bytes of the packed host block == offset of `out`            */
  size_t staging_bytes;      /* == lazy_host_step_staging_bytes(...)                        */
} lazy_host_step_layout_t;
int lazy_host_step_layout(const lazy_handle* h, int32_t num_reqs, int32_t total_q, int32_t num_new_tokens,
                          lazy_host_step_layout_t* out);
typedef struct lazy_host_step_packed_args {
  int32_t kind;              /* 0 = decode, 1 = prefill                                   */
  int32_t num_reqs;
  int32_t total_q;
  int32_t max_q_len;
  int32_t num_new_tokens;
  int32_t reserved;
  const void* h_packed;      /* HOST (pinned), in_bytes long, laid out per lazy_host_step_layout */
  void* h_out;               /* HOST, [total_q][Hq][D] bf16                                */
  void* d_k_cache;
  void* d_v_cache;
  void* d_staging;           /* DEVICE scratch, 256-byte aligned, >= staging_bytes          */
  size_t staging_bytes;
} lazy_host_step_packed_args;
int lazy_host_step_packed(lazy_handle* h, const lazy_host_step_packed_args* a, void* stream);

/* f4. One serving step's attention for a MIXED batch: the block-local prefill of cache-miss documents (or any
 * prefill chunk) and the decode of the running requests, issued together (Fig. 5 phases 1-3 happen in one
 * engine step).  Same results as lazy_attn_prefill followed by lazy_attn_decode; the two
 * kernels run CONCURRENTLY: the decode kernel (HBM-bound) is confined to `decode_sms` SMs on a library-owned side
 * stream forked from and joined back into `stream` with events, the prefill kernel (tensor-bound) takes the other
 * SMs and, as decode CTAs retire, theirs too.  No host synchronisation; capturable in a CUDA graph.  The side stream
 * and two events are host-side resources created at the first call and released by lazy_destroy.
 * Field meanings are those of the two calls above; the two request sets use separate tables.
 * For the product configuration (head_dim 128, un-rotated K, RoPE, 4 or 8 kv heads) the step is ONE launch: the first
 * `decode_sms` CTAs of the grid run the decode body, CTA pairs behind them the prefill work items (mixed_fused.cu);
 * decode_sms = 0 picks 7/16 of the SMs (64 of 148).  Bit 0 of `reserved0` forces the two-stream path described above
 * (the A/B arm); other configurations always take it.  LAZY_KV_FP8_E4M3 pages have their own one-launch kernel under the
 * same conditions (head_dim 128, 4 or 8 kv heads, no LAZY_FLAG_*). */
typedef struct lazy_mixed_args {
  const void* q_prefill;  const int32_t* block_table_prefill;  const int32_t* page_logical_pos_prefill;
  const int32_t* seq_lens_prefill;  const int32_t* cu_q_lens;
  int32_t num_reqs_prefill, total_q, max_q_len, reserved0;
  void* out_prefill;
  const void* q_decode;  const int32_t* block_table_decode;  const int32_t* page_logical_pos_decode;
  const int32_t* seq_lens_decode;
  int32_t num_reqs_decode;
  int32_t decode_sms;     /* SMs (= CTAs) given to the decode half; 0 = the default: 7/16 of the device on the one-launch
                             path (64 of 148), three quarters on the two-stream path (reserved0 bit 0, other configurations) */
  void* out_decode;
} lazy_mixed_args;
int lazy_attn_mixed(lazy_handle* h, const lazy_mixed_args* a, const void* k_cache, const void* v_cache, void* stream);

/* ---- f4 (host side): document-granular page pool with reference counts and LRU eviction ----------------------
 * Pure host code, no CUDA call: it hands out PHYSICAL PAGE IDS of the caller's k_cache / v_cache.  One physical copy
 * per document, reusable at any logical position with LAZY_POOL_AGNOSTIC; with
 * LAZY_POOL_POSITION_AWARE the key is (document, logical position), i.e. the position-coupled behaviour the paper
 * compares against (L56-58).  Not thread-safe. */
typedef struct lazy_pool lazy_pool;
#define LAZY_POOL_AGNOSTIC        0
#define LAZY_POOL_POSITION_AWARE  1
lazy_pool* lazy_pool_create(int32_t num_pages, int32_t page_size, int32_t keying);   /* NULL on bad arguments */
void lazy_pool_destroy(lazy_pool* p);
/* Looks a document up for a request that places it at logical_pos and pins it (refcount + 1).
 * Returns 1 = hit (pages_out filled, KV is valid), 0 = miss (pages_out filled with freshly allocated pages: the
 * caller prefills the document block-locally and lazy_cache_write's it), LAZY_ERR_WORKSPACE = does not fit even after
 * evicting every unpinned document, LAZY_ERR_INVALID = bad arguments or a length different from the cached one.
 * pages_out has room for ceil(doc_tokens / page_size) entries (HOST). Eviction is LRU over unpinned documents. */
int lazy_pool_acquire(lazy_pool* p, int64_t doc_id, int32_t doc_tokens, int32_t logical_pos, int32_t* pages_out);
/* Unpins (refcount - 1); at 0 the document becomes evictable (most recently used). */
int lazy_pool_release(lazy_pool* p, int64_t doc_id, int32_t logical_pos);
void lazy_pool_stats(const lazy_pool* p, int64_t* lookups, int64_t* hits, int64_t* evictions, int32_t* pages_in_use);
/* PAPER.md Eq. 1 / Eq. 2 (L60-70): hit ratio of a cache of `capacity_entries` entries over `num_docs` documents with
 * Zipf(alpha) popularity when every document needs `positions` position-specific copies (1 = position-agnostic).
 * Eq. 3 is the ratio of two calls.  Returns -1 on bad arguments. */
double lazy_hit_ratio_model(double alpha, int64_t num_docs, int64_t capacity_entries, int32_t positions);

#ifdef __cplusplus
}
#endif
#endif /* LAZY_ATTN_H_ */
