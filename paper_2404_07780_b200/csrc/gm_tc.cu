// gm_tc.cu -- launchers of the tensor-core engine (gm_tc.cuh, gm_tc_fused.cuh) for ONE padded PSF
// side, -DGM_TC_K=<9|17|25|33|41> (half width a multiple of 4).  Compiled once per side (build.py).
#include "gm_tc_fused.cuh"

#include <mutex>
#include <utility>
#include <vector>

#include "gm.h"

#ifndef GM_TC_K
#error "compile with -DGM_TC_K=<padded PSF side>"
#endif
#define GM_CAT_(a, b) a##b
#define GM_CAT(a, b) GM_CAT_(a, b)

namespace gm {
namespace tc {

#define GM_TRY(expr)                                   \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) { *err = e__; return GM_ECUDA; } \
  } while (0)

constexpr int KP = GM_TC_K;

static cudaError_t set_smem_once(const void* kern, int bytes) {
  static std::mutex mu;
  static std::vector<std::pair<const void*, int>> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(mu);
  for (const auto& d : done)
    if (d.first == kern && d.second == dev) return cudaSuccess;
  if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
  done.emplace_back(kern, dev);
  return cudaSuccess;
}

size_t GM_CAT(table_bytes_, GM_TC_K)() { return (size_t)KP * Cfg<KP>::kTapBytes; }

// the E_a table of every PSF (flip = 1: flipped taps, the forward convolution; 0: the adjoint) and the PSF scales
int GM_CAT(build_table_, GM_TC_K)(const float* psf, long long psf_stride, int n_psf, int K, int flip, uint8_t* tab, float* bscale,
                                 cudaStream_t st, cudaError_t* err) {
  k_tc_btab<KP><<<n_psf * KP, 256, 0, st>>>(psf, psf_stride, K, flip, tab, bscale);
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

// gm_conv, tensor engine: B cutouts of 128 x 128
int GM_CAT(launch_conv_tc_, GM_TC_K)(const ConvArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  GM_TRY(set_smem_once((const void*)k_tc_conv<KP>, (int)Cfg<KP>::kSmem));
  const int grid = a.B < n_sm ? a.B : n_sm;
  k_tc_conv<KP><<<grid, kThreads, Cfg<KP>::kSmem, st>>>(a);
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

// a1 .. a5 of square cutouts of 64, 96 or 128 pixels in one launch
template <int SIDE, bool UNCONV>
static int launch_fused_u(const FusedTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  using Gm = FusedGeomTc<KP, SIDE>;
  GM_TRY(set_smem_once((const void*)k_tc_fused<KP, SIDE, UNCONV>, (int)Gm::kSmem));
  const int passes = (a.B + Gm::G - 1) / Gm::G;
  const int grid = passes < n_sm ? passes : n_sm;
  k_tc_fused<KP, SIDE, UNCONV><<<grid, Roles<kFusedHW>::kThreads, Gm::kSmem, st>>>(a);
  GM_TRY(cudaGetLastError());
  return GM_OK;
}
template <int SIDE>
static int launch_fused_t(const FusedTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  return a.any_unconv ? launch_fused_u<SIDE, true>(a, n_sm, st, err) : launch_fused_u<SIDE, false>(a, n_sm, st, err);
}

int GM_CAT(launch_fused_tc_, GM_TC_K)(const FusedTcArgs& a, int side, int n_sm, cudaStream_t st, cudaError_t* err) {
  switch (side) {
    case 64: return launch_fused_t<64>(a, n_sm, st, err);
    case 96: return launch_fused_t<96>(a, n_sm, st, err);
    case 128: return launch_fused_t<128>(a, n_sm, st, err);
    default: return GM_ENOTSUP;
  }
}

// larger cutouts, super-tiles of trb x (128 / trb) tiles; bwd = 0: forward kernel, 1: backward kernel
template <int TRB, bool BWD, bool UNCONV>
static int launch_tile_u(const TileTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  GM_TRY(set_smem_once((const void*)k_tc_tile<KP, TRB, BWD, UNCONV>, (int)TileCfg<KP, TRB>::kSmem));
  const long long items = (long long)a.B * a.tiles_x * a.tiles_y;
  int grid = items < n_sm ? (int)items : n_sm;
  if (grid > kTileMaxCtas) grid = kTileMaxCtas;            // the forward kernel's scratch is sized for that many
  k_tc_tile<KP, TRB, BWD, UNCONV><<<grid, Roles<kTileHW>::kThreads, TileCfg<KP, TRB>::kSmem, st>>>(a);
  GM_TRY(cudaGetLastError());
  return GM_OK;
}
template <int TRB, bool BWD>
static int launch_tile_t(const TileTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  return a.any_unconv ? launch_tile_u<TRB, BWD, true>(a, n_sm, st, err) : launch_tile_u<TRB, BWD, false>(a, n_sm, st, err);
}

int GM_CAT(launch_tile_tc_, GM_TC_K)(const TileTcArgs& a, int trb, int bwd, int n_sm, cudaStream_t st, cudaError_t* err) {
  switch (trb) {
    case 128 / kTileR: return bwd ? launch_tile_t<128 / kTileR, true>(a, n_sm, st, err) : launch_tile_t<128 / kTileR, false>(a, n_sm, st, err);   // 128 x 128
    case 64 / kTileR: return bwd ? launch_tile_t<64 / kTileR, true>(a, n_sm, st, err) : launch_tile_t<64 / kTileR, false>(a, n_sm, st, err);      // 64 x 256
    default: return GM_ENOTSUP;
  }
}

}  // namespace tc
}  // namespace gm
