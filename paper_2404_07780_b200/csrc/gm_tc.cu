// gm_tc.cu -- launchers of the tensor-core convolution engine (gm_tc.cuh), one
// instantiation per padded PSF side whose half width is a multiple of 4.
#include "gm_tc_fused.cuh"

#include <mutex>
#include <utility>
#include <vector>

#include "gm.h"

namespace gm {
namespace tc {

#define GM_TRY(expr)                                   \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) { *err = e__; return GM_ECUDA; } \
  } while (0)

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

int g_tc_dbg = 0;   // PROBE ONLY

int padded_side(int K) {
  static const int sides[] = {9, 17, 25, 33, 41};
  for (int s : sides)
    if (K <= s) return s;
  return -1;
}

size_t table_bytes(int KP) {
  switch (KP) {
    case 9: return (size_t)9 * Cfg<9>::kTapBytes;
    case 17: return (size_t)17 * Cfg<17>::kTapBytes;
    case 25: return (size_t)25 * Cfg<25>::kTapBytes;
    case 33: return (size_t)33 * Cfg<33>::kTapBytes;
    case 41: return (size_t)41 * Cfg<41>::kTapBytes;
    default: return 0;
  }
}

template <int KP>
static int launch(const ConvArgs& a, const float* psf, long long psf_stride, int n_psf, int K, int flip, uint8_t* tab,
                  float* bscale, int n_sm, cudaStream_t st, cudaError_t* err, int* launches) {
  k_tc_btab<KP><<<n_psf * KP, 256, 0, st>>>(psf, psf_stride, K, flip, tab, bscale);
  GM_TRY(cudaGetLastError());
  GM_TRY(set_smem_once((const void*)k_tc_conv<KP>, (int)Cfg<KP>::kSmem));
  const int grid = a.B < n_sm ? a.B : n_sm;
  k_tc_conv<KP><<<grid, kThreads, Cfg<KP>::kSmem, st>>>(a);
  GM_TRY(cudaGetLastError());
  *launches += 2;
  return GM_OK;
}

// out = PSF (*) in (flip = 1) or the adjoint (flip = 0) for B cutouts of 128 x 128; tab / bscale: device scratch of
// n_psf * table_bytes(KP) bytes and n_psf floats
int conv(int KP, int B, const float* in, float* out, const float* psf, long long psf_stride, int K, int flip, uint8_t* tab,
         float* bscale, int n_sm, cudaStream_t st, cudaError_t* err, int* launches) {
  ConvArgs a;
  a.dbg = g_tc_dbg;
  a.B = B; a.in = in; a.out = out; a.btab = tab; a.bscale = bscale;
  a.btab_stride = psf_stride ? (long long)table_bytes(KP) : 0;
  const int n_psf = psf_stride ? B : 1;
  switch (KP) {
    case 9: return launch<9>(a, psf, psf_stride, n_psf, K, flip, tab, bscale, n_sm, st, err, launches);
    case 17: return launch<17>(a, psf, psf_stride, n_psf, K, flip, tab, bscale, n_sm, st, err, launches);
    case 25: return launch<25>(a, psf, psf_stride, n_psf, K, flip, tab, bscale, n_sm, st, err, launches);
    case 33: return launch<33>(a, psf, psf_stride, n_psf, K, flip, tab, bscale, n_sm, st, err, launches);
    case 41: return launch<41>(a, psf, psf_stride, n_psf, K, flip, tab, bscale, n_sm, st, err, launches);
    default: return GM_ENOTSUP;
  }
}

// both E_a tables of every PSF (forward: flipped taps, adjoint: taps as given) and the PSF scales
int build_tables(int KP, const float* psf, long long psf_stride, int n_psf, int K, uint8_t* tab_fwd, uint8_t* tab_adj,
                 float* bscale, cudaStream_t st, cudaError_t* err, int* launches) {
  switch (KP) {
#define GM_TC_CASE(S)                                                                     \
    case S:                                                                                 \
      k_tc_btab<S><<<n_psf * S, 256, 0, st>>>(psf, psf_stride, K, 1, tab_fwd, bscale);      \
      k_tc_btab<S><<<n_psf * S, 256, 0, st>>>(psf, psf_stride, K, 0, tab_adj, bscale);      \
      break;
    GM_TC_CASE(9) GM_TC_CASE(17) GM_TC_CASE(25) GM_TC_CASE(33) GM_TC_CASE(41)
#undef GM_TC_CASE
    default: return GM_ENOTSUP;
  }
  GM_TRY(cudaGetLastError());
  *launches += 2;
  return GM_OK;
}

template <int KP>
static int launch_fused_t(const FusedTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  GM_TRY(set_smem_once((const void*)k_tc_fused<KP>, (int)FusedCfg<KP>::kSmem));
  const int grid = a.B < n_sm ? a.B : n_sm;
  k_tc_fused<KP><<<grid, kFusedThreadsTc, FusedCfg<KP>::kSmem, st>>>(a);
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

int launch_fused(int KP, const FusedTcArgs& a, int n_sm, cudaStream_t st, cudaError_t* err) {
  switch (KP) {
    case 9: return launch_fused_t<9>(a, n_sm, st, err);
    case 17: return launch_fused_t<17>(a, n_sm, st, err);
    case 25: return launch_fused_t<25>(a, n_sm, st, err);
    case 33: return launch_fused_t<33>(a, n_sm, st, err);
    case 41: return launch_fused_t<41>(a, n_sm, st, err);
    default: return GM_ENOTSUP;
  }
}

}  // namespace tc
}  // namespace gm
