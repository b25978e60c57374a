// decode_fp8_kernel.cuh -- the split-KV decode CTA over LAZY_KV_FP8_E4M3 pages (head_dim 128 or 64, un-rotated K).
//
// Same decomposition, pipeline, rotation identity and in-kernel combine as decode_kernel.cuh (see decode_splitkv.cu);
// what changes is the arithmetic type of a tile, chosen so that a tile of HALF the bytes does not cost MORE
// instructions than a bf16 tile (the bf16 kernel's streaming rate is set by its consumer warps):
//   * K codes are widened e4m3x2 -> f16x2 (exact, one instruction per two elements) and rotated by the in-page offset
//     IN F16 on packed halves (HMUL2 / HFMA2: |code| <= 448, cos/sin rounded to f16 -- relative 2^-11, finer than the
//     bf16 rounding the bf16 kernel applies to the rotated K) -- no unpack to fp32, no repack;
//   * q is re-rotated per page in fp32 as before and rounded to f16; QK^T and PV are mma.sync m16n8k16 f16 -> fp32;
//   * the K scale of a token (a row of S) multiplies the fp32 score together with log2(e)/sqrt(D);
//   * V codes come out of shared memory already transposed AND still 8-bit with the 8-bit transposing ldmatrix
//     (m16n16.b8: thread (g, tq) gets tokens 4tq..4tq+3 of dims g, g+8), are widened to f16x2 and used as the A
//     operand; that fixes which MMA k-slot holds which token, and the token -> MMA-row order of the QK^T product is
//     chosen to match, with the ldmatrix row addresses permuted so that both the K loads and the V loads are
//     bank-conflict-free (token order tau in the kernel);
//   * the V scale of a token multiplies P (fp32, then f16) relative to a running reference scale c_run carried like
//     the softmax maximum: P' = p * sv / c_run, O accumulates in units of c_run and is rescaled only when a page's
//     largest V scale leaves [c_run/64, 64 c_run] (f16 has the range: P' <= 64).
#pragma once
#include <cuda_fp16.h>

#include "decode_kernel.cuh"

namespace lazy {
namespace {

// NCW consumer warps: 8 (the bf16 kernel's cut: 224 registers per consumer thread) or 12 (160 registers, which this
// kernel fits: three dependent-chain warps per scheduler instead of two).  A CTA then holds NCW * 32 + 128 threads.
template <int HKV_CTA, int NCW, int D_ = 128>
struct DecodeFp8Cfg {
  static constexpr int D = D_;                          // a row of codes is D bytes: 128-byte (D = 128) or 64-byte swizzle
  static constexpr int THREADS = NCW * 32 + 128;
  static constexpr int REGS_CONSUMER = NCW == 8 ? kRegsConsumer : 160;   // 384 * 160 + 128 * 32 = 65536
  static constexpr int REGS_PRODUCER = NCW == 8 ? kRegsProducer : 32;
  static constexpr int PPS = NCW / HKV_CTA;             // pages per pipeline stage
  static constexpr int BOX_ROWS = 16 * HKV_CTA;
  static constexpr int PAGE_BYTES = BOX_ROWS * D;       // K (or V) codes of one page, HKV_CTA heads: rows of D bytes
  static constexpr int CS_ROW_BYTES = D / 2 * 8;
  static constexpr int SC_BYTES = HKV_CTA * 64;         // K (or V) scales of one page, HKV_CTA heads
  static constexpr int OFF_V = PPS * PAGE_BYTES;
  static constexpr int OFF_CS = 2 * PPS * PAGE_BYTES;
  static constexpr int OFF_SK = OFF_CS + PPS * CS_ROW_BYTES;
  static constexpr int OFF_SV = OFF_SK + PPS * SC_BYTES;
  static constexpr int OFF_META = OFF_SV + PPS * SC_BYTES;
  static constexpr int STAGE_BYTES = (OFF_META + PPS * 4 + 1023) / 1024 * 1024;
  // 37 KB stages x 5 (8 warps) / 52-56 KB stages x 3 (12 warps); a 4th stage was measured: no gain (84.1 -> 85.4 us)
  static constexpr int NSTAGES = NCW == 8 ? 5 : 3;
  static constexpr int MAX_REQS = kMaxReqsSmem;         // requests per launch (smem prefix sums)
  static constexpr int NL = D / 16;                     // words of 2 rotation pairs per thread per half
  static constexpr int NC = D / 16;
  static constexpr int OFF_CUM = NSTAGES * STAGE_BYTES;
  static constexpr int OFF_LEN = OFF_CUM + (MAX_REQS + 4) * 4;
  static constexpr int OFF_BAR = OFF_LEN + MAX_REQS * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 2 * NSTAGES * 8 + 16 + 1024;
  static_assert(SMEM_BYTES <= 232448, "decode_fp8: shared memory");
};

struct DecodeFp8Args {
  DecodeArgs d;            // q, tables, out, cs, partials (stored_pos / alibi unused)
  const float* k_scale;    // [num_pages][Hkv][16]
  const float* v_scale;
};

__device__ __forceinline__ uint32_t h2mul(uint32_t a, uint32_t b) {
  const __half2 r = __hmul2(*reinterpret_cast<const __half2*>(&a), *reinterpret_cast<const __half2*>(&b));
  return *reinterpret_cast<const uint32_t*>(&r);
}
__device__ __forceinline__ uint32_t h2fma(uint32_t a, uint32_t b, uint32_t c) {
  const __half2 r = __hfma2(*reinterpret_cast<const __half2*>(&a), *reinterpret_cast<const __half2*>(&b),
                            *reinterpret_cast<const __half2*>(&c));
  return *reinterpret_cast<const uint32_t*>(&r);
}
// a * b - c * d on packed halves (the negation folds into an operand modifier)
__device__ __forceinline__ uint32_t h2mulsub(uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  const __half2 r = __hfma2(__hneg2(*reinterpret_cast<const __half2*>(&c)), *reinterpret_cast<const __half2*>(&d),
                            __hmul2(*reinterpret_cast<const __half2*>(&a), *reinterpret_cast<const __half2*>(&b)));
  return *reinterpret_cast<const uint32_t*>(&r);
}

template <int HKV_CTA, int NCW, int D_ = 128>
__device__ __forceinline__ void decode_fp8_cta(const CUtensorMap& tmap_k, const CUtensorMap& tmap_v,
                                               const DecodeFp8Args& fa, const int bid, const int G_in, const int hg,
                                               const int HG, unsigned char* smem_raw) {
  using C = DecodeFp8Cfg<HKV_CTA, NCW, D_>;
  constexpr int D = C::D;
  const DecodeArgs& a = fa.d;
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
  int G = G_in;
  const Shape sh = a.sh;

  // ---- prologue: barriers, unit prefix sums ---------------------------------------------------------------
  if (tid == 0) {
    for (int s = 0; s < C::NSTAGES; ++s) {
      ptx::mbar_init(bar_full + 8 * s, 1);
      ptx::mbar_init(bar_empty + 8 * s, NCW);
    }
    ptx::mbar_init(bar_empty + C::NSTAGES * 8 + 8, 1);
    ptx::fence_mbar_init();
  }
  if (warp == NCW && lane == 0) {
    ptx::prefetch_tmap(&tmap_k);
    ptx::prefetch_tmap(&tmap_v);
  }
  if (warp == 0) {
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
  __syncthreads();

  const long long U = s_cum[R];
  if (U < G) G = (int)U;
  if (bid >= G) return;
  const int u_begin = (int)(((long long)bid * U) / G);
  const int u_end = (int)(((long long)(bid + 1) * U) / G);
  if (u_begin >= u_end) return;
  int r0;
  {
    int lo = 0, hi = R;
    while (lo < hi) { int mid = (lo + hi) >> 1; if (s_cum[mid + 1] > u_begin) hi = mid; else lo = mid + 1; }
    r0 = lo;
  }

  if (warp >= NCW) {
    ptx::setmaxnreg_dec<C::REGS_PRODUCER>();
    if (warp > NCW) return;
    // ================================= producer warp =====================================================
    const int pl = lane;
    int r = r0, u = u_begin;
    int it = 0;
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
        int mq = pp[(L - 1) / kPageSize] + (L - 1) % kPageSize;
        pg = bt[p];
        delta = mq - pp[p];
      }
    };
    int pg, delta, nvalid;
    load_unit(r, u, pg, delta, nvalid);
    while (u < u_end) {
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
        ptx::mbar_arrive_expect_tx(full, nvalid * (2 * C::PAGE_BYTES + C::CS_ROW_BYTES + 2 * C::SC_BYTES));
      __syncwarp();
      if (active) {
        const int row0 = (pg * sh.Hkv + hg * HKV_CTA) * kPageSize;
        ptx::tma_load_2d(st_u32 + pl * C::PAGE_BYTES, &tmap_k, full, 0, row0);
        ptx::tma_load_2d(st_u32 + C::OFF_V + pl * C::PAGE_BYTES, &tmap_v, full, 0, row0);
        const int ad = delta < 0 ? -delta : delta;
        ptx::bulk_load_1d(st_u32 + C::OFF_CS + pl * C::CS_ROW_BYTES, a.cs + (size_t)ad * (D / 2), C::CS_ROW_BYTES, full);
        ptx::bulk_load_1d(st_u32 + C::OFF_SK + pl * C::SC_BYTES, fa.k_scale + row0, C::SC_BYTES, full);
        ptx::bulk_load_1d(st_u32 + C::OFF_SV + pl * C::SC_BYTES, fa.v_scale + row0, C::SC_BYTES, full);
      }
      pg = pg_n; delta = delta_n; nvalid = nvalid_n;
      r = rn; u = un; ++it;
    }
    return;
  }

  // =================================== consumer warps ====================================================
  ptx::setmaxnreg_inc<C::REGS_CONSUMER>();
  const int g = lane >> 2, tq = lane & 3;
  const int pl = warp / HKV_CTA;
  const int hl = warp % HKV_CTA;
  const int hk = hg * HKV_CTA + hl;
  const int group = sh.group;
  // MMA row g of the QK^T tile is token t0, row g + 8 token t0 + 2 (see the header: the order the V fragments fix)
  const int t0 = 8 * (g >> 2) + 4 * (g & 1) + ((g >> 1) & 1);

  // in-page rotation constants of this thread's two tokens and 16 pairs, as f16x2 (cos j, cos j+1) / (sin j, sin j+1)
  uint32_t ctc[2][C::NL], cts[2][C::NL];
  {
    const float4* cs4 = reinterpret_cast<const float4*>(a.cs);
#pragma unroll
    for (int rw = 0; rw < 2; ++rw)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) {
        const float4 v = __ldg(cs4 + (size_t)(t0 + 2 * rw) * (D / 4) + w * 4 + tq);
        ctc[rw][w] = ptx::pack_f16(v.x, v.y);
        cts[rw][w] = ptx::pack_f16(v.z, v.w);
      }
  }
  // ldmatrix row address of this lane inside a (page, head) V tile: matrix row i = 4a + b (lane & 15) is token
  // tau(i) = 8(a>>1) + 4(b&1) + 2(b>>1) + (a&1): any 8 consecutive lanes address 8 different 16-byte columns of the
  // swizzled tile (no bank conflicts), and the K rows of a quarter warp differ in bit 2 (ditto)
  const int vtok = 8 * ((lane >> 3) & 1) + 4 * (lane & 1) + 2 * ((lane >> 1) & 1) + ((lane >> 2) & 1);
  const int vrow = hl * 16 + vtok;
  const int vmat = lane >> 4;                       // which of the two 16-dim tiles of an x2 load this lane addresses
  // Per-thread byte offsets inside a stage, fixed for the whole kernel.  They are laundered through an empty asm so
  // that the compiler keeps them in registers: at 160 registers per thread it otherwise re-derives them from the lane
  // id for every tile (~60 integer instructions of the ~390 a tile costs).
  uint32_t kofs[2][2], vofs[C::NC / 2], scofs;
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int rw = 0; rw < 2; ++rw) {
      const int Rr = hl * 16 + t0 + 2 * rw;
      if (D == 128) kofs[h][rw] = pl * C::PAGE_BYTES + Rr * 128 + (((4 * h + tq) ^ (Rr & 7)) * 16);
      else {
        const int off = h * 32 + 8 * tq;
        kofs[h][rw] = pl * C::PAGE_BYTES + Rr * 64 + (((off >> 4) ^ ((Rr >> 1) & 3)) * 16) + (off & 15);
      }
      asm volatile("" : "+r"(kofs[h][rw]));
    }
#pragma unroll
  for (int i = 0; i < C::NC; i += 2) {
    vofs[i / 2] = C::OFF_V + pl * C::PAGE_BYTES + vrow * D + (((i + vmat) ^ (D == 128 ? (vrow & 7) : ((vrow >> 1) & 3))) * 16);
    asm volatile("" : "+r"(vofs[i / 2]));
  }
  scofs = pl * C::SC_BYTES + (hl * 16 + t0) * 4;
  asm volatile("" : "+r"(scofs));

  int r = r0, u = u_begin, it = 0;
  while (u < u_end) {
    const int L = s_len[r];
    const int seg_lo = u - s_cum[r];
    const int seg_hi = min(u_end, s_cum[r + 1]) - s_cum[r];

    // un-rotated q of head g of this kv head's group, widened to fp32 once per segment
    float qf[2][C::NL][2];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) { qf[h][w][0] = 0.f; qf[h][w][1] = 0.f; }
    if (g < group) {
      const uint4* qp = reinterpret_cast<const uint4*>(a.q + ((size_t)r * sh.Hq + hk * group + g) * D);
      if (!a.q_interleaved) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int x = 0; x < D / 64; ++x) {
            const uint4 v = qp[(h * (D / 2) + (D / 8) * tq) / 8 + x];
            const uint32_t ww[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int y = 0; y < 4; ++y) {
              qf[h][4 * x + y][0] = ptx::bf16_lo(ww[y]);
              qf[h][4 * x + y][1] = ptx::bf16_hi(ww[y]);
            }
          }
      } else {
        // LAZY_ROPE_INTERLEAVED: model order (x1_j, x2_j) per word -> this thread's x1 and x2 values of pairs
        // j = (D/8) tq + 8x .. + 7 (two 16-byte loads hold 8 pairs)
#pragma unroll
        for (int x = 0; x < D / 64; ++x) {
          const int j0 = (D / 8) * tq + 8 * x;
          const uint4 s0 = qp[j0 / 4], s1 = qp[j0 / 4 + 1];
          const uint32_t sw[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
#pragma unroll
          for (int wi = 0; wi < 4; ++wi) {
            qf[0][4 * x + wi][0] = ptx::bf16_lo(sw[2 * wi]);     qf[1][4 * x + wi][0] = ptx::bf16_hi(sw[2 * wi]);
            qf[0][4 * x + wi][1] = ptx::bf16_lo(sw[2 * wi + 1]); qf[1][4 * x + wi][1] = ptx::bf16_hi(sw[2 * wi + 1]);
          }
        }
      }
    }
    // One power-of-two normaliser per (request, kv head): the largest |q| of the GQA group goes to [1, 2) before the
    // f16 pack (|R q| <= sqrt(2) max|q| < 2.83), its inverse into the score scale.  Exact (powers of two), once per
    // segment, nothing per page: f16's range (65504, 6e-5) puts no restriction on q.
    float qmax = 0.f;
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) qmax = fmaxf(qmax, fmaxf(fabsf(qf[h][w][0]), fabsf(qf[h][w][1])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o));
    int qexp = 0;
    if (qmax > 0.f && qmax < INFINITY) qexp = max(-126, min(126, ((__float_as_int(qmax) >> 23) & 0xff) - 127));
    const float q_down = __int_as_float((127 - qexp) << 23);
    const float scale_log2 = sh.scale_log2 * __int_as_float((127 + qexp) << 23);
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int w = 0; w < C::NL; ++w) { qf[h][w][0] *= q_down; qf[h][w][1] *= q_down; }
    uint32_t qhat[2][C::NL];

    float oacc[C::NC][4];
#pragma unroll
    for (int i = 0; i < C::NC; ++i) { oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f; }
    float m_run[2] = {-INFINITY, -INFINITY};
    float l_run[2] = {0.f, 0.f};
    // reference V scale: O is accumulated in units of c_run; (c_lo, c_hi) = the band a page's largest scale may
    // move in before O is re-referenced (empty at first: the first page sets it)
    float c_run = 1.f, inv_c = 1.f, c_lo = 0.f, c_hi = 0.f;
    for (int ul = seg_lo; ul < seg_hi; ++ul, ++it) {
      const int stage = it % C::NSTAGES;
      const uint32_t parity = (it / C::NSTAGES) & 1;
      ptx::mbar_wait(bar_full + 8 * stage, parity);
      const int p = ul * C::PPS + pl;
      const int nv = min(kPageSize, L - p * kPageSize);      // valid tokens of this page (<= 0: no page)
      if (nv > 0) {
        const uint32_t st = smem_base + stage * C::STAGE_BYTES;
        const int delta = ptx::lds32(st + C::OFF_META + pl * 4);
        // ---- K codes -> registers: D/8 bytes per (half, token row): dims (D/2)h + (D/8)tq .. (one 16-byte chunk of
        // the 128B-swizzled row at D = 128, half a chunk of the 64B-swizzled row at D = 64)
        uint32_t kc[2][2][C::NL / 2];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int rw = 0; rw < 2; ++rw) {
            if (D == 128) {
              const uint4 v = ptx::lds128(st + kofs[h][rw]);
              kc[h][rw][0] = v.x; kc[h][rw][1] = v.y; kc[h][rw][C::NL / 2 - 2] = v.z; kc[h][rw][C::NL / 2 - 1] = v.w;
            } else {
              const uint2 v = ptx::lds64(st + kofs[h][rw]);
              kc[h][rw][0] = v.x; kc[h][rw][1] = v.y;
            }
          }
        // scales of this thread's two tokens: K (times log2(e)/sqrt(D)) and V
        const uint32_t sc_off = scofs;
        const float sk0 = __int_as_float(ptx::lds32(st + C::OFF_SK + sc_off)) * scale_log2;
        const float sk1 = __int_as_float(ptx::lds32(st + C::OFF_SK + sc_off + 8)) * scale_log2;
        float sv0 = __int_as_float(ptx::lds32(st + C::OFF_SV + sc_off));
        float sv1 = __int_as_float(ptx::lds32(st + C::OFF_SV + sc_off + 8));
        // ---- q re-rotated for this page: Qhat = R_{m - p0} q in fp32, rounded to f16 (a3/a4)
        {
          const uint32_t qcs = st + C::OFF_CS + pl * C::CS_ROW_BYTES + tq * 16;
          const float sgn = delta < 0 ? -1.f : 1.f;
#pragma unroll
          for (int w = 0; w < C::NL; ++w) {
            const float4 c = ptx::lds128f(qcs + w * 64);
            const float2 cc = make_float2(c.x, c.y);
            const float2 ss = __fmul2_rn(make_float2(c.z, c.w), make_float2(sgn, sgn));
            const float2 x1 = make_float2(qf[0][w][0], qf[0][w][1]), x2 = make_float2(qf[1][w][0], qf[1][w][1]);
            const float2 y1 = __ffma2_rn(make_float2(-x2.x, -x2.y), ss, __fmul2_rn(x1, cc));
            const float2 y2 = __ffma2_rn(x2, cc, __fmul2_rn(x1, ss));
            qhat[0][w] = ptx::pack_f16(y1.x, y1.y);
            qhat[1][w] = ptx::pack_f16(y2.x, y2.y);
          }
        }
        // ---- Khat = R_t k on packed f16 lanes (codes, un-scaled: the token's scale goes to the score)
        uint32_t kreg[2][2][C::NL];
#pragma unroll
        for (int rw = 0; rw < 2; ++rw) {
          const uint32_t* a1 = kc[0][rw];
          const uint32_t* a2 = kc[1][rw];
#pragma unroll
          for (int w = 0; w < C::NL; ++w) {
            const uint32_t x1 = (w & 1) ? ptx::e4m3x2_hi_to_f16x2(a1[w >> 1]) : ptx::e4m3x2_lo_to_f16x2(a1[w >> 1]);
            const uint32_t x2 = (w & 1) ? ptx::e4m3x2_hi_to_f16x2(a2[w >> 1]) : ptx::e4m3x2_lo_to_f16x2(a2[w >> 1]);
            kreg[0][rw][w] = h2mulsub(x1, ctc[rw][w], x2, cts[rw][w]);
            kreg[1][rw][w] = h2fma(x2, ctc[rw][w], h2mul(x1, cts[rw][w]));
          }
        }
        // ---- S = Khat Qhat^T : rows = tokens (t0, t0 + 8), cols = heads (2tq, 2tq+1)
        // (four accumulator chains of 4 MMAs: with two warps per scheduler the MMA latency chain is exposed)
        float s[4] = {0.f, 0.f, 0.f, 0.f}, s_b[4] = {0.f, 0.f, 0.f, 0.f};
        float s_c[4] = {0.f, 0.f, 0.f, 0.f}, s_d[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int cc = 0; cc < C::NC / 2; ++cc) {
          ptx::mma_f16_16816((cc & 1) ? s_c : s, kreg[0][0][2 * cc], kreg[0][1][2 * cc], kreg[0][0][2 * cc + 1],
                             kreg[0][1][2 * cc + 1], qhat[0][2 * cc], qhat[0][2 * cc + 1]);
          ptx::mma_f16_16816((cc & 1) ? s_d : s_b, kreg[1][0][2 * cc], kreg[1][1][2 * cc], kreg[1][0][2 * cc + 1],
                             kreg[1][1][2 * cc + 1], qhat[1][2 * cc], qhat[1][2 * cc + 1]);
        }
        s[0] = ((s[0] + s_b[0]) + (s_c[0] + s_d[0])) * sk0; s[1] = ((s[1] + s_b[1]) + (s_c[1] + s_d[1])) * sk0;
        s[2] = ((s[2] + s_b[2]) + (s_c[2] + s_d[2])) * sk1; s[3] = ((s[3] + s_b[3]) + (s_c[3] + s_d[3])) * sk1;
        if (t0 >= nv) { s[0] = -INFINITY; s[1] = -INFINITY; sv0 = 0.f; }
        if (t0 + 2 >= nv) { s[2] = -INFINITY; s[3] = -INFINITY; sv1 = 0.f; }
        // ---- online softmax over the 16 tokens (a6)
        float mx0 = fmaxf(s[0], s[2]), mx1 = fmaxf(s[1], s[3]);
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
          mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, o));
          mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, o));
        }
        const float mn0 = fmaxf(m_run[0], mx0), mn1 = fmaxf(m_run[1], mx1);
        if (__any_sync(0xffffffffu, mn0 > m_run[0] || mn1 > m_run[1])) {
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
        // ---- V scales: P' = p * sv / c_run; re-reference O when the page's largest scale leaves the band
        const float svmax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(sv0, sv1))));
        if (svmax > c_hi || svmax < c_lo) {          // warp-uniform; the first page, then rare
          const float f = c_run / svmax;
          c_run = svmax; inv_c = 1.f / svmax; c_lo = svmax * (1.f / 64.f); c_hi = svmax * 64.f;
#pragma unroll
          for (int i = 0; i < C::NC; ++i) { oacc[i][0] *= f; oacc[i][1] *= f; oacc[i][2] *= f; oacc[i][3] *= f; }
        }
        const float w0 = sv0 * inv_c, w1 = sv1 * inv_c;
        // ---- P' (f16) transposed into the B-fragment layout: k = tokens, n = heads
        const uint32_t pb0 = ptx::movmatrix_trans(ptx::pack_f16(p0 * w0, p1 * w0));
        const uint32_t pb1 = ptx::movmatrix_trans(ptx::pack_f16(p2 * w1, p3 * w1));
        // ---- O^T += V^T P'  (a7): 8-bit transposing ldmatrix, two 16-dim tiles per load; byte b of a register is
        // token tau(4tq + b) = vt + 4(b&1) + 2(b>>1) -- bytes past the tail are cleared (their codes may be NaN)
        uint32_t vmask = 0xffffffffu;
        if (nv < kPageSize) {                       // the last page of a request only
          const int vt = 8 * (tq >> 1) + (tq & 1);
          vmask = (vt < nv ? 0xffu : 0u) | (vt + 4 < nv ? 0xff00u : 0u) | (vt + 2 < nv ? 0xff0000u : 0u) |
                  (vt + 6 < nv ? 0xff000000u : 0u);
        }
#pragma unroll
        for (int i = 0; i < C::NC; i += 2) {
          uint32_t r0, r1, r2, r3;
          ptx::ldmatrix_b8_x2_trans(r0, r1, r2, r3, st + vofs[i / 2]);
          if (nv < kPageSize) { r0 &= vmask; r1 &= vmask; r2 &= vmask; r3 &= vmask; }
          ptx::mma_f16_16816(oacc[i], ptx::e4m3x2_lo_to_f16x2(r0), ptx::e4m3x2_lo_to_f16x2(r1),
                             ptx::e4m3x2_hi_to_f16x2(r0), ptx::e4m3x2_hi_to_f16x2(r1), pb0, pb1);
          ptx::mma_f16_16816(oacc[i + 1], ptx::e4m3x2_lo_to_f16x2(r2), ptx::e4m3x2_lo_to_f16x2(r3),
                             ptx::e4m3x2_hi_to_f16x2(r2), ptx::e4m3x2_hi_to_f16x2(r3), pb0, pb1);
        }
      }
      __syncwarp();
      // PPS > 1: the segment's LAST stage stays held -- its tiles are the staging area of the page-lane merge below
      if (lane == 0 && !(C::PPS > 1 && ul == seg_hi - 1)) ptx::mbar_arrive(bar_empty + 8 * stage);
    }

    // ---- segment done: O back to true units, softmax sums reduced over the token lanes
#pragma unroll
    for (int i = 0; i < C::NC; ++i) { oacc[i][0] *= c_run; oacc[i][1] *= c_run; oacc[i][2] *= c_run; oacc[i][3] *= c_run; }
#pragma unroll
    for (int o = 4; o < 32; o <<= 1) {
      l_run[0] += __shfl_xor_sync(0xffffffffu, l_run[0], o);
      l_run[1] += __shfl_xor_sync(0xffffffffu, l_run[1], o);
    }
    // PPS > 1: the page lanes of one kv head are merged inside the CTA (as in decode_kernel.cuh): warp (pl > 0, hl)
    // parks its accumulators lane to lane in its OWN K and V code tiles of the held stage (NC float4 per lane, half in
    // each tile) and (m, m, l, l) of its four head-column pairs in its own K-scale slot (64 bytes); warp (0, hl) folds
    // them in.  One partial per (request, kv head, CTA) instead of PPS.
    if (C::PPS > 1) {
      const uint32_t stl = smem_base + ((it - 1) % C::NSTAGES) * C::STAGE_BYTES;
      const uint32_t tile = (uint32_t)(hl * 16 * D);
      if (pl > 0) {
#pragma unroll
        for (int i = 0; i < C::NC; ++i)
          ptx::sts128(stl + (i < C::NC / 2 ? 0 : C::OFF_V) + pl * C::PAGE_BYTES + tile + ((i % (C::NC / 2)) * 32 + lane) * 16,
                      make_uint4(__float_as_uint(oacc[i][0]), __float_as_uint(oacc[i][1]), __float_as_uint(oacc[i][2]),
                                 __float_as_uint(oacc[i][3])));
        if (g == 0)
          ptx::sts128(stl + C::OFF_SK + pl * C::SC_BYTES + hl * 64 + tq * 16,
                      make_uint4(__float_as_uint(m_run[0]), __float_as_uint(m_run[1]), __float_as_uint(l_run[0]),
                                 __float_as_uint(l_run[1])));
        ptx::fence_proxy_async();                   // the next fill of this stage is an async-proxy write
      }
      ptx::named_bar_sync(1, NCW * 32);
      if (pl == 0) {
#pragma unroll 1
        for (int q = 1; q < C::PPS; ++q) {
          const float4 ml = ptx::lds128f(stl + C::OFF_SK + q * C::SC_BYTES + hl * 64 + tq * 16);
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
            const float4 v = ptx::lds128f(stl + (i < C::NC / 2 ? 0 : C::OFF_V) + q * C::PAGE_BYTES + tile +
                                          ((i % (C::NC / 2)) * 32 + lane) * 16);
            oacc[i][0] = oacc[i][0] * fa0 + v.x * fb0; oacc[i][1] = oacc[i][1] * fa1 + v.y * fb1;
            oacc[i][2] = oacc[i][2] * fa0 + v.z * fb0; oacc[i][3] = oacc[i][3] * fa1 + v.w * fb1;
          }
        }
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar_empty + 8 * ((it - 1) % C::NSTAGES));
    }
    // ---- this kv head's partial (o, m, l) -> workspace (a8); written by the page-lane-0 warp
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
    ptx::named_bar_sync(1, NCW * 32);
    const long long c0 = s_cum[r], c1 = s_cum[r + 1];
    const int b_first = (int)(((c0 + 1) * G + U - 1) / U) - 1;
    const int b_last = (int)((c1 * G + U - 1) / U) - 1;
    const int n_parts = b_last - b_first + 1;
    if (tid == 0) {
      __threadfence();
      int old = atomicAdd(&a.req_counter[r * HG + hg], 1);
      int last = (old == n_parts - 1);
      if (last) a.req_counter[r * HG + hg] = 0;
      *s_flag = last;
    }
    ptx::named_bar_sync(1, NCW * 32);
    if (*s_flag) {
      __threadfence();
      // the ring is idle iff this segment ends the CTA's range (every issued stage has been consumed)
      combine_request<D, NCW>(a, r, hg, HKV_CTA * group, n_parts, r + b_first, warp, lane,
                         s_cum[r] + seg_hi == u_end, smem_base, C::NSTAGES * C::STAGE_BYTES, bar_comb, comb_phase);
    }
    ptx::named_bar_sync(1, NCW * 32);
    u = s_cum[r] + seg_hi;
    ++r;
  }
}

}  // namespace
}  // namespace lazy
