// prefill_umma2.cu -- lazy_attn_prefill for head_dim 128 on CTA PAIRS (thread-block cluster of 2, tcgen05 cta_group::2).
//
// Same computation and the same roles as prefill_umma.cu (Eq. 4 with deferred RoPE, L94-108; one rotation per
// K tile, L164-173), re-cut so that the two SMs of a pair share every K and V tile:
//
//   * one tcgen05.mma covers M = 256 query rows (128 per CTA) x N = 128 keys.  Each CTA supplies its own Q rows and
//     HALF of the B operand: 64 of the 128 keys for S = Q Khat^T, 64 of the 128 head dims for O += P V.  The tensor
//     cores of the pair exchange the halves themselves, so per SM the K/V bytes landing in shared memory, the K
//     rotation work and the B-operand fetches are all halved;
//   * a CTA therefore loads 4 of a tile's 8 pages of K (both 64-column slabs) and one 64-column slab of all 8 pages
//     of V: 16 KB + 16 KB per tile instead of 32 + 32, which buys FOUR pipeline stages in the same shared memory.
//     With two stages the TMA latency plus the rotation latency of a tile did not fit into the 1.5 iterations a
//     stage is free, and the tensor pipe idled half of the time;
//   * the leader CTA (rank 0) issues every MMA.  Arrivals it waits for (Q rotated, K rotated, P written) come from
//     the warps of both CTAs (remote mbarrier arrive, release.cluster); its tcgen05.commit multicasts to the barrier
//     copies of both CTAs.  V boxes of both CTAs count their bytes on the leader's barrier (TMA .cta_group::2).
//
// CTA = 2 Q tiles of 128 rows (GQA group packed into M); pair = 4 Q tiles.  16 warps per CTA as in prefill_umma.cu.
// TMEM per CTA (512 columns): S0 | S1 | O0 | O1; S_t is two key halves of 64 columns, P_h aliases the first 32 of S_h.
#include <climits>

#include "prefill_pair_kernel.cuh"

namespace lazy {
namespace {

template <int KM, bool F8>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPrefillThreads, 1)
prefill_pair_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v, const PrefillArgs a) {
  extern __shared__ unsigned char smem_raw[];
  prefill_pair_cta<KM, F8>(tmap_q, tmap_k, tmap_v, a, (int)(blockIdx.x >> 1), smem_raw);
}

template <int KM, bool F8 = false>
int launch_pair_t(const lazy_handle* h, const PrefillArgs& args, int grid, cudaStream_t stream) {
  auto kern = prefill_pair_kernel<KM, F8>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, PairCfg::SMEM_BYTES) != cudaSuccess)
    return LAZY_ERR_CUDA;
  const CUtensorMap* mq = reinterpret_cast<const CUtensorMap*>(h->tmap_pq);
  const CUtensorMap* mk = reinterpret_cast<const CUtensorMap*>(h->tmap_pk);
  const CUtensorMap* mv = reinterpret_cast<const CUtensorMap*>(h->tmap_pv);
  kern<<<grid, kPrefillThreads, PairCfg::SMEM_BYTES, stream>>>(*mq, *mk, *mv, args);
  return cudaGetLastError() == cudaSuccess ? 1 : LAZY_ERR_CUDA;
}

}  // namespace

// head_dim 128 only; `a.mblocks` counts CTA PAIRS per (request, kv head); the grid is 2 CTAs per pair.
int launch_prefill_pair(const lazy_handle* h, const PrefillArgs& a, int km, int grid, cudaStream_t stream) {
  if (h->cfg.dtype == LAZY_KV_FP8_E4M3) return launch_pair_t<LAZY_K_UNROTATED, true>(h, a, grid, stream);
  switch (km) {
    case LAZY_K_STORED_POS: return launch_pair_t<LAZY_K_STORED_POS>(h, a, grid, stream);
    case LAZY_K_ABSOLUTE:   return launch_pair_t<LAZY_K_ABSOLUTE>(h, a, grid, stream);
    case kKmAlibi:          return launch_pair_t<kKmAlibi>(h, a, grid, stream);
    default:                return launch_pair_t<LAZY_K_UNROTATED>(h, a, grid, stream);
  }
}

}  // namespace lazy
