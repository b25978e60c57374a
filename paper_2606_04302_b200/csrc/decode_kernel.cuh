// decode_kernel.cuh -- the split-KV decode CTA (lazy_attn_decode) as a device function, shared by decode_splitkv.cu
// (its own kernel) and mixed_fused.cu (one launch for a mixed prefill + decode step).  See decode_splitkv.cu for the
// design notes.
#pragma once
#include "lazy_internal.h"
#include "ptx_util.cuh"

namespace lazy {
namespace {

constexpr int kConsumerWarps = 8;
// 3 warpgroups: two of consumers, one holding the producer warp (+ 3 idle warps) so that setmaxnreg can move the
// registers the producer does not need to the consumers (a 9-warp CTA is allocated registers as if it had 12 warps)
constexpr int kDecodeThreads = 384;
constexpr int kRegsConsumer = 224, kRegsProducer = 40;       // 2*128*224 + 128*40 = 62464 <= 65536
constexpr int kMaxReqsSmem = 2048;
#ifndef LAZY_CTAB_REGS
#define LAZY_CTAB_REGS 1
#endif

template <int D, int HKV_CTA>
struct DecodeCfg {
  static constexpr int NH = D / 64;                     // 128-byte column blocks per row
  static constexpr int PPS = kConsumerWarps / HKV_CTA;  // pages per pipeline stage
  static constexpr int BOX_ROWS = 16 * HKV_CTA;
  static constexpr int BOX_BYTES = BOX_ROWS * 128;
  static constexpr int PAGE_BYTES = NH * BOX_BYTES;     // K (or V) of one page, HKV_CTA heads
  static constexpr int CS_ROW_BYTES = D / 2 * 8;
  static constexpr int OFF_V = PPS * PAGE_BYTES;
  static constexpr int OFF_CS = 2 * PPS * PAGE_BYTES;
  static constexpr int OFF_META = OFF_CS + PPS * CS_ROW_BYTES;
  static constexpr int STAGE_BYTES = (OFF_META + PPS * 4 + 1023) / 1024 * 1024;
  static constexpr int NSTAGES = (STAGE_BYTES > 40000) ? 3 : 4;
  static constexpr int JT = D / 8;                      // rotation pairs (j values) per thread
  static constexpr int NL = JT / 2;                     // 16-byte cos/sin loads per thread per token row
  static constexpr int NLK = JT / 8;                    // 16-byte K loads per thread per row per half
  static constexpr int NC = D / 16;                     // MMA k-chunks (QK^T) == dim tiles (PV)
  static constexpr int CTAB_BYTES = 2 * NL * 32 * 16;
  static constexpr int OFF_CTAB = NSTAGES * STAGE_BYTES;
  static constexpr int OFF_CUM = OFF_CTAB + CTAB_BYTES;
  static constexpr int OFF_LEN = OFF_CUM + (kMaxReqsSmem + 4) * 4;   // keeps the mbarriers 16-byte aligned
  static constexpr int OFF_BAR = OFF_LEN + kMaxReqsSmem * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 2 * NSTAGES * 8 + 16 + 1024;  // + alignment slack
};

struct DecodeArgs {
  const __nv_bfloat16* q;
  const int* block_table;
  const int* page_pos;
  const int* seq_lens;
  __nv_bfloat16* out;
  const float2* cs;
  const int* stored_pos;   // LAZY_K_STORED_POS: [num_pages] position each physical page was stored at
  const float* alibi;      // kKmAlibi: [Hq] slopes * log2(e)
  float* part_o;
  float2* part_ml;
  int* req_counter;
  int num_reqs;
  int q_interleaved;       // LAZY_ROPE_INTERLEAVED: q arrives with pairs (2j, 2j+1); de-interleaved on load
  Shape sh;
};

// Split-KV combine (a8) + epilogue (a9) of request r by the LAST CTA to finish a piece of it: warp w takes q heads
// w, w+8, ... of the CTA's head group (heads_cta of them) and merges the n_slots partials (o, m, l) that start at slot0.
//
// Two paths.  When the combining CTA has finished its whole range (the usual case: a request's last arriver is a CTA
// whose piece of it ENDS its range) the pipeline ring is idle, and the partial outputs are pulled into it with bulk
// async copies -- one per slot, all heads of the CTA's head group are contiguous there -- so that every byte of the
// request's partials is in flight at once; the warps then merge out of shared memory.  (Round 1 / early round 2: the
// warps loaded four slots at a time from L2 / HBM, ~0.9 us per dependent batch: 16 us for the 20 slots x 28 heads of a
// cfg-5 request, which held that decode under 70 % of the HBM roofline.)  Otherwise (the ring still holds pages of the
// CTA's next request) the register path below runs.
template <int D, int NCW = kConsumerWarps>
__device__ __forceinline__ void combine_request(const DecodeArgs& a, const int r, const int hg, const int heads_cta,
                                                const int n_slots, const int slot0, const int warp, const int lane,
                                                const bool ring_free, const uint32_t ring_u32, const int ring_bytes,
                                                const uint32_t cbar, uint32_t& cphase) {
  const Shape& sh = a.sh;
  const int slot_bytes = heads_cta * D * 4;
  if (ring_free && slot_bytes <= ring_bytes) {
    const int cap = min(32, ring_bytes / slot_bytes);
    const int hpw = (heads_cta + NCW - 1) / NCW;      // heads per warp (<= 8)
    float mstar[8], lsum[8], acc[8][D / 32];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      mstar[k] = -INFINITY; lsum[k] = 0.f;
#pragma unroll
      for (int x = 0; x < D / 32; ++x) acc[k][x] = 0.f;
    }
    for (int base = 0; base < n_slots; base += cap) {
      const int n = min(cap, n_slots - base);
      if (warp == 0) {
        // the partials were written through the generic proxy: EVERY lane that issues a bulk copy (an async-proxy
        // read) fences first -- a proxy fence orders the executing thread's accesses only, and __syncwarp does not
        // carry it to the other lanes
        if (lane < n) ptx::fence_proxy_async_all();
        if (lane == 0) ptx::mbar_arrive_expect_tx(cbar, (uint32_t)(n * slot_bytes));
        __syncwarp();
        if (lane < n)
          ptx::bulk_load_1d(ring_u32 + lane * slot_bytes,
                            a.part_o + ((size_t)(slot0 + base + lane) * sh.Hq + hg * heads_cta) * D, slot_bytes, cbar);
      }
      // (m, l) of slot base + lane for each of this warp's heads, issued before the wait
      float2 ml[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int hh = warp + k * NCW;
        ml[k] = make_float2(-INFINITY, 0.f);
        if (k < hpw && hh < heads_cta && lane < n)
          ml[k] = __ldcg(&a.part_ml[(size_t)(slot0 + base + lane) * sh.Hq + hg * heads_cta + hh]);
      }
      ptx::mbar_wait(cbar, cphase);
      cphase ^= 1;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int hh = warp + k * NCW;
        if (k < hpw && hh < heads_cta) {
          float mx = ml[k].x;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
          const float mnew = fmaxf(mstar[k], mx);
          if (mnew > -INFINITY) {                   // warp-uniform
            const float f = exp2f(mstar[k] - mnew);                       // mstar = -inf on the first round: 0
            const float w = ml[k].x == -INFINITY ? 0.f : exp2f(ml[k].x - mnew);
            float wl = w * ml[k].y;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) wl += __shfl_xor_sync(0xffffffffu, wl, o);
            mstar[k] = mnew;
            lsum[k] = lsum[k] * f + wl;
#pragma unroll
            for (int x = 0; x < D / 32; ++x) acc[k][x] *= f;
            const uint32_t src = ring_u32 + hh * (D * 4) + lane * (D / 32) * 4;
            for (int i = 0; i < n; ++i) {
              const float wi = __shfl_sync(0xffffffffu, w, i);
              if (D == 128) {
                const float4 v = ptx::lds128f(src + i * slot_bytes);
                acc[k][0] += wi * v.x; acc[k][1] += wi * v.y; acc[k][D / 32 - 2] += wi * v.z; acc[k][D / 32 - 1] += wi * v.w;
              } else {
                const float4 v = ptx::lds128f((src + i * slot_bytes) & ~15u);   // 8-byte pieces: pick the lane's half
                const bool hi = lane & 1;
                acc[k][0] += wi * (hi ? v.z : v.x); acc[k][1] += wi * (hi ? v.w : v.y);
              }
            }
          }
        }
      }
      if (base + cap < n_slots) ptx::named_bar_sync(1, NCW * 32);   // the next round overwrites the ring
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int hh = warp + k * NCW;
      if (k < hpw && hh < heads_cta) {
        const float inv = lsum[k] > 0.f ? 1.f / lsum[k] : 0.f;
        __nv_bfloat16* op = a.out + ((size_t)r * sh.Hq + hg * heads_cta + hh) * D + lane * (D / 32);
#pragma unroll
        for (int x = 0; x < D / 32; x += 2)
          *reinterpret_cast<uint32_t*>(op + x) = ptx::pack_bf16(acc[k][x] * inv, acc[k][x + 1] * inv);
      }
    }
    return;
  }
  for (int hh = warp; hh < heads_cta; hh += NCW) {
    const int hq = hg * heads_cta + hh;
    // single pass with a running max; the loads of four partials are issued together so that their L2
    // latencies overlap (the partials were written by other SMs)
    float mstar = -INFINITY, lsum = 0.f;
    float acc[D / 32];
#pragma unroll
    for (int x = 0; x < D / 32; ++x) acc[x] = 0.f;
    for (int base = 0; base < n_slots; base += 4) {
      float2 ml[4];
      float2 pv[4][D / 64];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int sidx = min(base + i, n_slots - 1);
        ml[i] = __ldcg(&a.part_ml[(size_t)(slot0 + sidx) * sh.Hq + hq]);
        const float2* po = reinterpret_cast<const float2*>(a.part_o + ((size_t)(slot0 + sidx) * sh.Hq + hq) * D +
                                                           lane * (D / 32));
#pragma unroll
        for (int x = 0; x < D / 64; ++x) pv[i][x] = __ldcg(po + x);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (base + i >= n_slots || ml[i].x == -INFINITY) continue;
        const float mnew = fmaxf(mstar, ml[i].x);
        const float f = exp2f(mstar - mnew), w = exp2f(ml[i].x - mnew);   // mstar = -inf on the first: f = 0
        mstar = mnew;
        lsum = lsum * f + w * ml[i].y;
#pragma unroll
        for (int x = 0; x < D / 64; ++x) {
          acc[2 * x] = acc[2 * x] * f + w * pv[i][x].x;
          acc[2 * x + 1] = acc[2 * x + 1] * f + w * pv[i][x].y;
        }
      }
    }
    const float inv = lsum > 0.f ? 1.f / lsum : 0.f;
    __nv_bfloat16* op = a.out + ((size_t)r * sh.Hq + hq) * D + lane * (D / 32);
#pragma unroll
    for (int x = 0; x < D / 32; x += 2)
      *reinterpret_cast<uint32_t*>(op + x) = ptx::pack_bf16(acc[x] * inv, acc[x + 1] * inv);
  }
}

// KM = lazy_config.k_storage.  LAZY_K_UNROTATED: the identity above.  LAZY_K_STORED_POS (Eq. 6,
// L175-182: "rotate Q" by the page's relative offset): K is consumed as stored, q is re-rotated once per page
// by m - (p0 - stored[page]).  LAZY_K_ABSOLUTE: K as stored, q rotated once per request by m (no table rows
// travel with the pages): the "rotation compiled out" arm of the overhead ablation (Fig. 5).
// kKmAlibi: nothing is rotated; the score of token t of a page starting at p0 gets the bias
// slope[head] * (p0 + t - m) -- the same per-page relative offset m - p0 the rotation would use.
// The body of one decode CTA.  `bid` / `G_in`: this CTA's index among, and the number of, the CTAs that share the
// batch's units; `hg` / `HG`: kv-head group and number of groups.  decode_splitkv_kernel maps them to blockIdx /
// gridDim; the fused mixed-step kernel (mixed_fused.cu) runs the same body on the first CTAs of its grid.
template <int D, int HKV_CTA, int KM>
__device__ __forceinline__ void decode_cta(const CUtensorMap& tmap_k, const CUtensorMap& tmap_v, const DecodeArgs& a,
                                           const int bid, const int G_in, const int hg, const int HG,
                                           unsigned char* smem_raw) {
  using C = DecodeCfg<D, HKV_CTA>;
  constexpr bool kNoRows = KM == LAZY_K_ABSOLUTE || KM == kKmAlibi;   // no cos/sin row travels with a page
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t smem_base = ptx::smem_u32(smem);
  int* s_cum = reinterpret_cast<int*>(smem + C::OFF_CUM);
  int* s_len = reinterpret_cast<int*>(smem + C::OFF_LEN);
  const uint32_t bar_full = smem_base + C::OFF_BAR;
  const uint32_t bar_empty = bar_full + C::NSTAGES * 8;
  int* s_flag = reinterpret_cast<int*>(smem + C::OFF_BAR + 2 * C::NSTAGES * 8);
  const uint32_t bar_comb = bar_empty + C::NSTAGES * 8 + 8;     // bulk-copy combine (combine_request)
  uint32_t comb_phase = 0;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int R = a.num_reqs;
  int G = G_in;                                    // clamped to the unit count below: no CTA range is empty
  const Shape sh = a.sh;

  // ---- prologue: barriers, unit prefix sums, in-page rotation constants -------------------------------
  if (tid == 0) {
    for (int s = 0; s < C::NSTAGES; ++s) {
      ptx::mbar_init(bar_full + 8 * s, 1);
      ptx::mbar_init(bar_empty + 8 * s, kConsumerWarps);
    }
    ptx::mbar_init(bar_empty + C::NSTAGES * 8 + 8, 1);
    ptx::fence_mbar_init();
  }
  if (warp == kConsumerWarps && lane == 0) {
    ptx::prefetch_tmap(&tmap_k);
    ptx::prefetch_tmap(&tmap_v);
  }
  if (warp == 0) {
    // units per request (a unit = PPS consecutive pages; empty requests get one empty unit), inclusive scan
    int carry = 0;
    if (lane == 0) s_cum[0] = 0;
    for (int base = 0; base < R; base += 32) {
      int r = base + lane;
      int L = (r < R) ? a.seq_lens[r] : 0;
      if (L < 0) L = 0;
      int np = (L + kPageSize - 1) / kPageSize;
      int nu = (r < R) ? max(1, (np + C::PPS - 1) / C::PPS) : 0;
      int x = nu;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
      }
      if (r < R) { s_cum[r + 1] = carry + x; s_len[r] = L; }
      carry += __shfl_sync(0xffffffffu, x, 31);
    }
  }
  {
    // ctab[k'][lane] (16 B each): (cos, cos, sin, sin) of two rotation pairs of the in-page offsets, pre-multiplied by log2(e)/sqrt(D),
    // in the order thread (g,tq) consumes them: row t = g + 8*(k'/NL), pairs j = JT*tq + 2*(k'%NL), +1.
    float4* ctab = reinterpret_cast<float4*>(smem + C::OFF_CTAB);
    const float4* cs4 = reinterpret_cast<const float4*>(a.cs);
    for (int i = tid; i < 2 * C::NL * 32; i += kDecodeThreads) {
      int kk = i >> 5, ln = i & 31;
      int g = ln >> 2, tq = ln & 3;
      int t = g + 8 * (kk / C::NL);
      float4 v = cs4[(size_t)t * (D / 4) + (kk % C::NL) * 4 + tq];
      v.x *= sh.scale_log2; v.y *= sh.scale_log2; v.z *= sh.scale_log2; v.w *= sh.scale_log2;
      ctab[i] = v;
    }
  }
  __syncthreads();

  const long long U = s_cum[R];
  if (U < G) G = (int)U;
  if (bid >= G) return;
  const int u_begin = (int)(((long long)bid * U) / G);
  const int u_end = (int)(((long long)(bid + 1) * U) / G);
  if (u_begin >= u_end) return;
  int r0;
  {
    int lo = 0, hi = R;                             // smallest r with cum[r+1] > u_begin
    while (lo < hi) { int mid = (lo + hi) >> 1; if (s_cum[mid + 1] > u_begin) hi = mid; else lo = mid + 1; }
    r0 = lo;
  }

  if (warp >= kConsumerWarps) {
    ptx::setmaxnreg_dec<kRegsProducer>();
    if (warp > kConsumerWarps) return;              // idle warps of the producer's warpgroup
    // ================================= producer warp =====================================================
    const int pl = lane;                            // page lane within a stage (lanes < PPS are active)
    int r = r0, u = u_begin;
    int it = 0;
    // state of the unit about to be issued
    auto load_unit = [&](int rr, int uu, int& pg, int& delta, int& nvalid) {
      int L = s_len[rr];
      int np = (L + kPageSize - 1) / kPageSize;
      int ul = uu - s_cum[rr];
      int p = ul * C::PPS + pl;
      nvalid = min(C::PPS, max(0, np - ul * C::PPS));
      pg = 0; delta = 0;
      if (pl < C::PPS && p < np) {
        const int* bt = a.block_table + (size_t)rr * sh.table_stride;
        const int* pp = a.page_pos + (size_t)rr * sh.table_stride;
        int mq = pp[(L - 1) / kPageSize] + (L - 1) % kPageSize;    // position of the query token
        pg = bt[p];
        delta = mq - pp[p];
        if (KM == LAZY_K_STORED_POS) delta += a.stored_pos[pg];
      }
    };
    int pg, delta, nvalid;
    load_unit(r, u, pg, delta, nvalid);
    while (u < u_end) {
      // prefetch the table entries of the next unit before blocking on the ring
      int rn = r, un = u + 1;
      if (un >= s_cum[rn + 1]) rn++;
      int pg_n = 0, delta_n = 0, nvalid_n = 0;
      if (un < u_end) load_unit(rn, un, pg_n, delta_n, nvalid_n);

      const int stage = it % C::NSTAGES;
      const uint32_t parity = (it / C::NSTAGES) & 1;
      ptx::mbar_wait(bar_empty + 8 * stage, parity ^ 1);
      unsigned char* st = smem + stage * C::STAGE_BYTES;
      const uint32_t st_u32 = smem_base + stage * C::STAGE_BYTES;
      const uint32_t full = bar_full + 8 * stage;
      const bool active = pl < nvalid;
      if (pl < C::PPS) reinterpret_cast<int*>(st + C::OFF_META)[pl] = delta;
      __syncwarp();
      if (lane == 0)
        ptx::mbar_arrive_expect_tx(full, nvalid * (2 * C::PAGE_BYTES + (kNoRows ? 0 : C::CS_ROW_BYTES)));
      __syncwarp();
      if (active) {
        const int row0 = (pg * sh.Hkv + hg * HKV_CTA) * kPageSize;
#pragma unroll
        for (int h = 0; h < C::NH; ++h) {
          ptx::tma_load_2d(st_u32 + pl * C::PAGE_BYTES + h * C::BOX_BYTES, &tmap_k, full, h * 64, row0);
          ptx::tma_load_2d(st_u32 + C::OFF_V + pl * C::PAGE_BYTES + h * C::BOX_BYTES, &tmap_v, full, h * 64, row0);
        }
        if (!kNoRows) {
          int ad = delta < 0 ? -delta : delta;
          ptx::bulk_load_1d(st_u32 + C::OFF_CS + pl * C::CS_ROW_BYTES, a.cs + (size_t)ad * (D / 2),
                            C::CS_ROW_BYTES, full);
        }
      }
      pg = pg_n; delta = delta_n; nvalid = nvalid_n;
      r = rn; u = un; ++it;
    }
    return;
  }

  // =================================== consumer warps ====================================================
  ptx::setmaxnreg_inc<kRegsConsumer>();
  const int g = lane >> 2, tq = lane & 3;
  const int pl = warp / HKV_CTA;                    // page lane within a stage
  const int hl = warp % HKV_CTA;                    // kv head within the CTA's head group
  const int hk = hg * HKV_CTA + hl;
  const int group = sh.group;
  const uint32_t ctab_u32 = smem_base + C::OFF_CTAB + lane * 16;   // explicit ld.shared: generic LD costs a long scoreboard

  // in-page rotation constants held in registers for the whole kernel (LAZY_CTAB_REGS token rows of the two a thread
  // owns; the rest is re-read from shared memory for every page)
  float4 ctab_r[LAZY_CTAB_REGS > 0 ? LAZY_CTAB_REGS : 1][C::NL];
  if (KM == LAZY_K_UNROTATED) {
#pragma unroll
    for (int rw = 0; rw < LAZY_CTAB_REGS; ++rw)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) ctab_r[rw][w] = ptx::lds128f(ctab_u32 + (rw * C::NL + w) * 512);
  }

  int r = r0, u = u_begin, it = 0;
  while (u < u_end) {
    const int L = s_len[r];
    const int seg_lo = u - s_cum[r];
    const int seg_hi = min(u_end, s_cum[r + 1]) - s_cum[r];

    // un-rotated q of head g of this kv head's group, as packed bf16 in this thread's k-slot order
    uint32_t qraw[2][C::NL];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) qraw[h][w] = 0u;
    if (g < group) {
      const uint4* qp = reinterpret_cast<const uint4*>(a.q + ((size_t)r * sh.Hq + hk * group + g) * D);
      if (!a.q_interleaved) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int x = 0; x < C::NLK; ++x) {
            uint4 v = qp[(h * (D / 2) + C::JT * tq) / 8 + x];
            qraw[h][4 * x + 0] = v.x; qraw[h][4 * x + 1] = v.y; qraw[h][4 * x + 2] = v.z; qraw[h][4 * x + 3] = v.w;
          }
      } else {
        // model order (x1_j, x2_j) per word -> this thread's x1 words and x2 words (same pairs j as above)
#pragma unroll
        for (int x = 0; x < C::NLK; ++x) {
          const int j0 = C::JT * tq + 8 * x;
          const uint4 s0 = qp[j0 / 4], s1 = qp[j0 / 4 + 1];
          const uint32_t sw[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
#pragma unroll
          for (int wi = 0; wi < 4; ++wi) {
            qraw[0][4 * x + wi] = __byte_perm(sw[2 * wi], sw[2 * wi + 1], 0x5410u);
            qraw[1][4 * x + wi] = __byte_perm(sw[2 * wi], sw[2 * wi + 1], 0x7632u);
          }
        }
      }
    }

    // Qhat = scale * R_angle q from one cos/sin row (a3/a4); `scale` is 1 when the K side carries the scale
    uint32_t qhat[2][C::NL];
    float qf[2][C::NL][2];                          // q widened once per segment (it is re-rotated for every page)
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) { qf[h][w][0] = ptx::bf16_lo(qraw[h][w]); qf[h][w][1] = ptx::bf16_hi(qraw[h][w]); }
    auto rotate_q = [&](auto&& load_cs, float sgn, float scale) {
#pragma unroll
      for (int w = 0; w < C::NL; ++w) {
        const float4 c = load_cs(w);                // (cos lo, cos hi, sin lo, sin hi) of the word's two pairs
        const float2 cc = KM == LAZY_K_UNROTATED ? make_float2(c.x, c.y)      // the K side carries the scale
                                                 : __fmul2_rn(make_float2(c.x, c.y), make_float2(scale, scale));
        const float2 ss = __fmul2_rn(make_float2(c.z, c.w), make_float2(sgn * scale, sgn * scale));
        const float2 x1 = make_float2(qf[0][w][0], qf[0][w][1]), x2 = make_float2(qf[1][w][0], qf[1][w][1]);
        const float2 y1 = __ffma2_rn(make_float2(-x2.x, -x2.y), ss, __fmul2_rn(x1, cc));
        const float2 y2 = __ffma2_rn(x2, cc, __fmul2_rn(x1, ss));
        qhat[0][w] = ptx::pack_bf16(y1.x, y1.y);
        qhat[1][w] = ptx::pack_bf16(y2.x, y2.y);
      }
    };
    float slope0 = 0.f, slope1 = 0.f;               // kKmAlibi: slopes (log2 units) of heads 2tq, 2tq+1
    if (KM == kKmAlibi) {
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int w = 0; w < C::NL; ++w)
          qhat[h][w] = ptx::pack_bf16(ptx::bf16_lo(qraw[h][w]) * sh.scale_log2, ptx::bf16_hi(qraw[h][w]) * sh.scale_log2);
      if (2 * tq < group) slope0 = a.alibi[hk * group + 2 * tq];
      if (2 * tq + 1 < group) slope1 = a.alibi[hk * group + 2 * tq + 1];
    }
    if (KM == LAZY_K_ABSOLUTE && L > 0) {           // once per request: rotate q by the query token's position
      const int* pp = a.page_pos + (size_t)r * sh.table_stride;
      const int mq = pp[(L - 1) / kPageSize] + (L - 1) % kPageSize;
      const float4* row = reinterpret_cast<const float4*>(a.cs + (size_t)mq * (D / 2)) + tq;
      rotate_q([&](int w) { return __ldg(row + w * 4); }, 1.f, sh.scale_log2);
    }

    float oacc[C::NC][4];
#pragma unroll
    for (int i = 0; i < C::NC; ++i) { oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f; }
    float m_run[2] = {-INFINITY, -INFINITY};        // heads 2tq, 2tq+1 (log2 units)
    float l_run[2] = {0.f, 0.f};                    // this thread's share (rows g, g+8) of the softmax sums

    for (int ul = seg_lo; ul < seg_hi; ++ul, ++it) {
      const int stage = it % C::NSTAGES;
      const uint32_t parity = (it / C::NSTAGES) & 1;
      ptx::mbar_wait(bar_full + 8 * stage, parity);
      const int p = ul * C::PPS + pl;
      const int nv = min(kPageSize, L - p * kPageSize);      // valid tokens of this page (<= 0: no page)
      if (nv > 0) {
        const uint32_t st = smem_base + stage * C::STAGE_BYTES;
        const int delta = ptx::lds32(st + C::OFF_META + pl * 4);
        // ---- K tile -> registers (rows g, g+8 of head hl; this thread's JT dims of each half)
        uint32_t kreg[2][2][C::NL];                 // [half][row][word]
        const int R0 = hl * 16 + g;
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int rw = 0; rw < 2; ++rw)
#pragma unroll
            for (int x = 0; x < C::NLK; ++x) {
              int d = h * (D / 2) + C::JT * tq + 8 * x;
              int Rr = R0 + 8 * rw;
              const uint4 v = ptx::lds128(st + pl * C::PAGE_BYTES + (d / 64) * C::BOX_BYTES + Rr * 128 +
                                          ((((d % 64) / 8) ^ (Rr & 7)) * 16));
              kreg[h][rw][4 * x + 0] = v.x; kreg[h][rw][4 * x + 1] = v.y;
              kreg[h][rw][4 * x + 2] = v.z; kreg[h][rw][4 * x + 3] = v.w;
            }
        // ---- q re-rotated for this page: Qhat = R_{m - p0} q   (a3/a4; one cos/sin row per page)
        if (!kNoRows) {
          const uint32_t qcs = st + C::OFF_CS + pl * C::CS_ROW_BYTES + tq * 16;
          rotate_q([&](int w) { return ptx::lds128f(qcs + w * 64); }, delta < 0 ? -1.f : 1.f,
                   KM == LAZY_K_UNROTATED ? 1.f : sh.scale_log2);
        }
        // ---- Khat = scale * R_t k in fp32 registers, rounded to bf16 for the MMA (un-rotated pages only)
        if (KM == LAZY_K_UNROTATED) {
#pragma unroll
          for (int rw = 0; rw < 2; ++rw)
#pragma unroll
            for (int w = 0; w < C::NL; ++w) {
              const float4 c = rw < LAZY_CTAB_REGS ? ctab_r[rw < LAZY_CTAB_REGS ? rw : 0][w]
                                                   : ptx::lds128f(ctab_u32 + (rw * C::NL + w) * 512);
              const float2 cc = make_float2(c.x, c.y), ss = make_float2(c.z, c.w);
              const float2 x1 = make_float2(ptx::bf16_lo(kreg[0][rw][w]), ptx::bf16_hi(kreg[0][rw][w]));
              const float2 x2 = make_float2(ptx::bf16_lo(kreg[1][rw][w]), ptx::bf16_hi(kreg[1][rw][w]));
              const float2 y1 = __ffma2_rn(make_float2(-x2.x, -x2.y), ss, __fmul2_rn(x1, cc));
              const float2 y2 = __ffma2_rn(x2, cc, __fmul2_rn(x1, ss));
              kreg[0][rw][w] = ptx::pack_bf16(y1.x, y1.y);
              kreg[1][rw][w] = ptx::pack_bf16(y2.x, y2.y);
            }
        }
        // ---- S = Khat Qhat^T : rows = tokens (g, g+8), cols = heads (2tq, 2tq+1)
        float s[4] = {0.f, 0.f, 0.f, 0.f}, s_b[4] = {0.f, 0.f, 0.f, 0.f};   // two chains: halves the MMA latency chain
#pragma unroll
        for (int cc = 0; cc < C::NC / 2; ++cc) {
          ptx::mma_bf16_16816(s, kreg[0][0][2 * cc], kreg[0][1][2 * cc], kreg[0][0][2 * cc + 1],
                              kreg[0][1][2 * cc + 1], qhat[0][2 * cc], qhat[0][2 * cc + 1]);
          ptx::mma_bf16_16816(s_b, kreg[1][0][2 * cc], kreg[1][1][2 * cc], kreg[1][0][2 * cc + 1],
                              kreg[1][1][2 * cc + 1], qhat[1][2 * cc], qhat[1][2 * cc + 1]);
        }
#pragma unroll
        for (int x = 0; x < 4; ++x) s[x] += s_b[x];
        if (KM == kKmAlibi) {                        // bias slope * (n - m), n - m = t - delta
          const float rel0 = (float)(g - delta), rel1 = (float)(g + 8 - delta);
          s[0] += slope0 * rel0; s[1] += slope1 * rel0;
          s[2] += slope0 * rel1; s[3] += slope1 * rel1;
        }
        if (g >= nv) { s[0] = -INFINITY; s[1] = -INFINITY; }
        if (g + 8 >= nv) { s[2] = -INFINITY; s[3] = -INFINITY; }
        // ---- online softmax over the 16 tokens (a6): max across the 8 row-lanes with shuffles
        float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
          mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, o));
          mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, o));
        }
        const float mn0 = fmaxf(m_run[0], mx0), mn1 = fmaxf(m_run[1], mx1);   // finite: token 0 is valid
        if (__any_sync(0xffffffffu, mn0 > m_run[0] || mn1 > m_run[1])) {      // rare after the first pages
          const float corr0 = exp2f(m_run[0] - mn0), corr1 = exp2f(m_run[1] - mn1);
          m_run[0] = mn0; m_run[1] = mn1;
          l_run[0] *= corr0; l_run[1] *= corr1;
#pragma unroll
          for (int i = 0; i < C::NC; ++i) {
            oacc[i][0] *= corr0; oacc[i][1] *= corr1; oacc[i][2] *= corr0; oacc[i][3] *= corr1;
          }
        }
        const float p0 = exp2f(s[0] - mn0), p1 = exp2f(s[1] - mn1);
        const float p2 = exp2f(s[2] - mn0), p3 = exp2f(s[3] - mn1);
        l_run[0] += p0 + p2;
        l_run[1] += p1 + p3;
        // ---- P (bf16) transposed into the B-fragment layout: k = tokens, n = heads
        const uint32_t pb0 = ptx::movmatrix_trans(ptx::pack_bf16(p0, p1));
        const uint32_t pb1 = ptx::movmatrix_trans(ptx::pack_bf16(p2, p3));
        // ---- O^T += V^T P  (a7): V^T fragments straight from the swizzled tile
        uint32_t vmask_lo = 0xffffffffu, vmask_hi = 0xffffffffu;   // tail: never let bytes past seq_len in
        if (nv < kPageSize) {
          int t0 = 2 * tq, t1 = 2 * tq + 8;
          vmask_lo = (t0 < nv ? 0x0000ffffu : 0u) | (t0 + 1 < nv ? 0xffff0000u : 0u);
          vmask_hi = (t1 < nv ? 0x0000ffffu : 0u) | (t1 + 1 < nv ? 0xffff0000u : 0u);
        }
        const int mi = lane >> 3;
        const int vrow = hl * 16 + (lane & 7) + 8 * (mi >> 1);
        const uint32_t vbase = smem_base + stage * C::STAGE_BYTES + C::OFF_V + pl * C::PAGE_BYTES + vrow * 128;
#pragma unroll
        for (int i = 0; i < C::NC; ++i) {
          const int chunk = 2 * i + (mi & 1);       // 16-byte chunk (8 dims) along the row
          const uint32_t addr = vbase + (chunk / 8) * C::BOX_BYTES + (((chunk % 8) ^ (vrow & 7)) * 16);
          uint32_t a0, a1, a2, a3;
          ptx::ldmatrix_x4_trans(a0, a1, a2, a3, addr);
          if (nv < kPageSize) { a0 &= vmask_lo; a1 &= vmask_lo; a2 &= vmask_hi; a3 &= vmask_hi; }
          ptx::mma_bf16_16816(oacc[i], a0, a1, a2, a3, pb0, pb1);
        }
      }
      __syncwarp();
      // PPS > 1: the segment's LAST stage stays held -- its K / V tiles are the staging area of the page-lane merge below
      if (lane == 0 && !(C::PPS > 1 && ul == seg_hi - 1)) ptx::mbar_arrive(bar_empty + 8 * stage);
    }

    // ---- segment done.  PPS > 1 (fewer than 8 kv heads per CTA): the PPS page lanes of one kv head are merged inside
    // the CTA first, so that a CTA writes ONE partial per (request, kv head) instead of PPS -- half (a quarter, an
    // eighth) of the partial traffic and of the last arriver's combine work.  Both warps of a kv head hold the same
    // (head column, dim) elements in the same lanes, so the hand-over is lane to lane: warp (pl > 0, hl) parks its
    // accumulators in its OWN K tile of the held stage (NC float4 per lane, [i][lane] order: conflict-free) and
    // (m, m, l, l) in its own V tile; warp (0, hl) folds them in with the usual running-max rescale.
    if (C::PPS > 1) {
      const uint32_t stl = smem_base + ((it - 1) % C::NSTAGES) * C::STAGE_BYTES;
      if (pl > 0) {
#pragma unroll
        for (int i = 0; i < C::NC; ++i)
          ptx::sts128(stl + pl * C::PAGE_BYTES + (i / 4) * C::BOX_BYTES + hl * 2048 + ((i % 4) * 32 + lane) * 16,
                      make_uint4(__float_as_uint(oacc[i][0]), __float_as_uint(oacc[i][1]), __float_as_uint(oacc[i][2]),
                                 __float_as_uint(oacc[i][3])));
        ptx::sts128(stl + C::OFF_V + pl * C::PAGE_BYTES + hl * 2048 + lane * 16,
                    make_uint4(__float_as_uint(m_run[0]), __float_as_uint(m_run[1]), __float_as_uint(l_run[0]),
                               __float_as_uint(l_run[1])));
        ptx::fence_proxy_async();                   // the next fill of this stage is a TMA (async-proxy) write
      }
      ptx::named_bar_sync(1, kConsumerWarps * 32);
      if (pl == 0) {
#pragma unroll 1
        for (int q = 1; q < C::PPS; ++q) {
          const float4 ml = ptx::lds128f(stl + C::OFF_V + q * C::PAGE_BYTES + hl * 2048 + lane * 16);
          const float mn0 = fmaxf(m_run[0], ml.x), mn1 = fmaxf(m_run[1], ml.y);
          const float fa0 = m_run[0] == -INFINITY ? 0.f : exp2f(m_run[0] - mn0);
          const float fa1 = m_run[1] == -INFINITY ? 0.f : exp2f(m_run[1] - mn1);
          const float fb0 = ml.x == -INFINITY ? 0.f : exp2f(ml.x - mn0);
          const float fb1 = ml.y == -INFINITY ? 0.f : exp2f(ml.y - mn1);
          m_run[0] = mn0; m_run[1] = mn1;
          l_run[0] = l_run[0] * fa0 + ml.z * fb0;
          l_run[1] = l_run[1] * fa1 + ml.w * fb1;
#pragma unroll
          for (int i = 0; i < C::NC; ++i) {
            const float4 v = ptx::lds128f(stl + q * C::PAGE_BYTES + (i / 4) * C::BOX_BYTES + hl * 2048 +
                                          ((i % 4) * 32 + lane) * 16);
            oacc[i][0] = oacc[i][0] * fa0 + v.x * fb0; oacc[i][1] = oacc[i][1] * fa1 + v.y * fb1;
            oacc[i][2] = oacc[i][2] * fa0 + v.z * fb0; oacc[i][3] = oacc[i][3] * fa1 + v.w * fb1;
          }
        }
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar_empty + 8 * ((it - 1) % C::NSTAGES));
    }

    // ---- this kv head's partial (o, m, l) -> workspace (a8); written by the page-lane-0 warp
#pragma unroll
    for (int o = 4; o < 32; o <<= 1) {
      l_run[0] += __shfl_xor_sync(0xffffffffu, l_run[0], o);
      l_run[1] += __shfl_xor_sync(0xffffffffu, l_run[1], o);
    }
    const int slot = r + bid;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int n = 2 * tq + e;
      if (n < group && pl == 0) {
        const int hq = hk * group + n;
        float* po = a.part_o + ((size_t)slot * sh.Hq + hq) * D;
#pragma unroll
        for (int i = 0; i < C::NC; ++i) {
          po[16 * i + g] = oacc[i][e];
          po[16 * i + g + 8] = oacc[i][2 + e];
        }
        if (g == 0) a.part_ml[(size_t)slot * sh.Hq + hq] = make_float2(m_run[e], l_run[e]);
      }
    }
    ptx::named_bar_sync(1, kConsumerWarps * 32);    // all partials of this CTA are written (CTA-scope order) ...
    // number of CTAs that hold a piece of request r: those containing units cum[r] .. cum[r+1]-1
    const long long c0 = s_cum[r], c1 = s_cum[r + 1];
    const int b_first = (int)(((c0 + 1) * G + U - 1) / U) - 1;
    const int b_last = (int)((c1 * G + U - 1) / U) - 1;
    const int n_parts = b_last - b_first + 1;
    if (tid == 0) {
      __threadfence();                              // ... and one cumulative gpu-scope release publishes them
      int old = atomicAdd(&a.req_counter[r * HG + hg], 1);
      int last = (old == n_parts - 1);
      if (last) a.req_counter[r * HG + hg] = 0;     // self-resetting: ready for the next call
      *s_flag = last;
    }
    ptx::named_bar_sync(1, kConsumerWarps * 32);
    if (*s_flag) {
      __threadfence();
      // the ring is idle iff this segment ends the CTA's range (every issued stage has been consumed)
      combine_request<D>(a, r, hg, HKV_CTA * group, n_parts, r + b_first, warp, lane,
                         s_cum[r] + seg_hi == u_end, smem_base, C::NSTAGES * C::STAGE_BYTES, bar_comb, comb_phase);
    }
    ptx::named_bar_sync(1, kConsumerWarps * 32);    // s_flag is reused by the next segment
    u = s_cum[r] + seg_hi;
    ++r;
  }
}

}  // namespace
}  // namespace lazy
