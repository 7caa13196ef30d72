// gm_tiles.cu -- instantiates the tile kernels for one PSF side, -DGM_K=<odd>.
// Compiled once per supported K (see build.py) so the builds run in parallel.
#include "gm_fused.cuh"

#ifndef GM_K
#error "compile with -DGM_K=<PSF side>"
#endif
#define GM_CAT_(a, b) a##b
#define GM_CAT(a, b) GM_CAT_(a, b)

namespace gm {

#define GM_TRY(expr)                                   \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) { *err = e__; return GM_ECUDA; } \
  } while (0)

template <typename Kern>
static cudaError_t set_smem(Kern kern, size_t bytes) {
  return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// Threads of a tile CTA.  When the tile is so large that only one CTA fits an SM (K = 41 with
// 128 x 128 tiles) the CTA gets 512 threads: the upper 256 own no output pixels and only
// help with the render, the tile load and the epilogue, which run with the
// convolution warps idle and need the extra warps to hide the SFU / memory latency.
template <int K>
static int tile_threads(const TileGeom& tg, int nthr) {
  const size_t one = smem_bytes<K>(tg, 16, kNSum) + 1024;
  return (2 * one > 233472) ? 512 : nthr;
}

template <int K, int RP, int TC>
static int launch_forward_v(const FwdArgs& a, int mode, int nthr, size_t sm, unsigned grid, cudaStream_t st, cudaError_t* err) {
  if (mode == FWD_RENDER) {
    GM_TRY(set_smem(k_forward<K, FWD_RENDER, RP, TC>, sm));
    k_forward<K, FWD_RENDER, RP, TC><<<grid, nthr, sm, st>>>(a);
  } else if (mode == FWD_DERIV) {
    GM_TRY(set_smem(k_forward<K, FWD_DERIV, RP, TC>, sm));
    k_forward<K, FWD_DERIV, RP, TC><<<grid, nthr, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_forward<K, FWD_LOSS, RP, TC>, sm));
    k_forward<K, FWD_LOSS, RP, TC><<<grid, nthr, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

int GM_CAT(launch_forward_, GM_K)(const FwdArgs& a, int mode, int B, cudaStream_t st, cudaError_t* err) {
  constexpr int K = GM_K;
  int nthr = (a.tg.ntx * a.tg.nty + 31) / 32 * 32;
  if (nthr > 256) return GM_ENOTSUP;
  nthr = tile_threads<K>(a.tg, nthr);
  const size_t sm = smem_bytes<K>(a.tg, nthr / 32, 1);
  const unsigned grid = (unsigned)((size_t)B * a.tg.tiles_x * a.tg.tiles_y);
  return a.tg.variant == 1 ? launch_forward_v<K, 3, 12>(a, mode, nthr, sm, grid, st, err)
                           : launch_forward_v<K, 4, 8>(a, mode, nthr, sm, grid, st, err);
}

int GM_CAT(launch_backward_, GM_K)(const BwdArgs& a, int B, cudaStream_t st, cudaError_t* err) {
  constexpr int K = GM_K;
  int nthr = (a.tg.ntx * a.tg.nty + 31) / 32 * 32;
  if (nthr > 256) return GM_ENOTSUP;
  nthr = tile_threads<K>(a.tg, nthr);
  const size_t sm = smem_bytes<K>(a.tg, nthr / 32, kNSum);
  const unsigned grid = (unsigned)((size_t)B * a.tg.tiles_x * a.tg.tiles_y);
  if (a.tg.variant == 1) {
    GM_TRY(set_smem(k_backward<K, 3, 12>, sm));
    k_backward<K, 3, 12><<<grid, nthr, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_backward<K, 4, 8>, sm));
    k_backward<K, 4, 8><<<grid, nthr, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

// fused loss + gradient (whole cutouts per CTA); variant 0: 8x8 thread tiles, 1: 6x12
int GM_CAT(launch_fused_, GM_K)(const FusedArgs& a, int variant, int n_sm, size_t smem_limit, cudaStream_t st,
                                cudaError_t* err) {
  constexpr int K = GM_K;
  if (a.fg.tpg * a.fg.G > kConvThreads) return GM_ENOTSUP;
  const size_t sm = fused_smem_bytes(K, a.fg);
  if (sm > smem_limit) return GM_ENOTSUP;
  const unsigned grid = (unsigned)(a.B < n_sm ? a.B : n_sm);
  if (variant == 0) {
    GM_TRY(set_smem(k_fused<K, 4, 8>, sm));
    k_fused<K, 4, 8><<<grid, kFusedThreads, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_fused<K, 3, 12>, sm));
    k_fused<K, 3, 12><<<grid, kFusedThreads, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

}  // namespace gm
