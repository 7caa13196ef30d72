// gm_tiles.cu -- instantiates the tile kernels for one PSF side, -DGM_K=<odd>.
// Compiled once per supported K (see build.py) so the builds run in parallel.
#include "gm_fused.cuh"

#include <mutex>
#include <utility>
#include <vector>

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

// cudaFuncAttributeMaxDynamicSharedMemorySize is raised once per (kernel, device), to the
// device's opt-in maximum, not on every launch
static cudaError_t set_smem_once(const void* kern) {
  static std::mutex mu;
  static std::vector<std::pair<const void*, int>> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(mu);
  for (const auto& d : done)
    if (d.first == kern && d.second == dev) return cudaSuccess;
  int optin = 0;
  if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess) return e;
  done.emplace_back(kern, dev);
  return cudaSuccess;
}
template <typename Kern>
static cudaError_t set_smem(Kern kern, size_t /*bytes*/) { return set_smem_once((const void*)kern); }

// Threads of a tile CTA.  When the tile is so large that only one CTA fits an SM (K = 41 with
// 128 x 128 tiles and the taps in shared memory; with the taps in the constant bank two fit) the CTA gets 512 threads: the upper 256 own no output pixels and only
// help with the render, the tile load and the epilogue, which run with the
// convolution warps idle and need the extra warps to hide the SFU / memory latency.
template <int K>
static int tile_threads(const TileGeom& tg, int nthr, bool ct) {
  const size_t one = smem_bytes<K>(tg, 8, kNSum, ct) + 1024;   // + the 1 KB the driver reserves per CTA
  return (2 * one > 233472) ? 512 : nthr;
}

// ---------------------------------------------------------------------------
// Host-side allocator of c_tap_pool (one pool per PSF side: each gm_tiles object is its own
// module with its own constant bank).  A region holds the forward + adjoint tap sets of one
// call; it is filled on the call's stream and handed back by an event recorded on that
// stream after the call's last launch, so concurrent calls (gm_fit_multi runs one stream per
// size bucket) never share a region that is still being read; a later call on the SAME stream
// takes the region over at once.  "Same stream" is decided by cudaStreamGetId, never by the
// handle: equal handles do not imply stream order (cudaStreamPerThread is a different stream
// in every host thread, and a destroyed stream's handle can be handed out again), equal ids
// do.  No region free: the caller runs the shared-memory taps instead.  Nothing here blocks
// or synchronises.
// ---------------------------------------------------------------------------
namespace {
struct TapRegion { int dev, off, n; cudaEvent_t ev; bool recorded; unsigned long long sid; };
std::mutex g_pool_mu;
std::vector<TapRegion> g_pool_used;
}  // namespace

int GM_CAT(tap_pool_acquire_, GM_K)(const float2* taps_dev, int n, cudaStream_t st, int* off, cudaError_t* err) {
  *off = -1;
  if (n <= 0 || n > kTapPoolN || (n & 1)) return GM_OK;
  int dev = 0;
  GM_TRY(cudaGetDevice(&dev));
  unsigned long long sid = 0;
  GM_TRY(cudaStreamGetId(st, &sid));
  std::lock_guard<std::mutex> lk(g_pool_mu);
  // A region whose call was enqueued on this very stream can be refilled at once: stream order
  // puts the copy behind that call's last kernel.  This is what keeps a loop of asynchronous
  // calls on one stream (or on a few, round robin) in the constant bank however far the host
  // runs ahead of the device.
  for (TapRegion& r : g_pool_used) {
    if (r.dev != dev || !r.recorded || r.sid != sid || r.n != n) continue;
    GM_TRY(cudaMemcpyToSymbolAsync(c_tap_pool, taps_dev, (size_t)n * sizeof(float2), (size_t)r.off * sizeof(float2),
                                   cudaMemcpyDeviceToDevice, st));
    cudaEventDestroy(r.ev);
    r.ev = nullptr; r.recorded = false;
    *off = r.off;
    return GM_OK;
  }
  for (size_t i = 0; i < g_pool_used.size();) {           // hand back the regions whose call has finished
    TapRegion& r = g_pool_used[i];
    if (r.recorded && cudaEventQuery(r.ev) == cudaSuccess) {
      cudaEventDestroy(r.ev);
      g_pool_used.erase(g_pool_used.begin() + i);
    } else {
      ++i;
    }
  }
  (void)cudaGetLastError();                                // cudaErrorNotReady of the queries above
  int start = 0;
  bool moved = true;
  while (moved) {                                          // first fit among this device's regions
    moved = false;
    for (const TapRegion& r : g_pool_used)
      if (r.dev == dev && start < r.off + r.n && r.off < start + n) { start = r.off + r.n; moved = true; }
  }
  if (start + n > kTapPoolN) return GM_OK;
  GM_TRY(cudaMemcpyToSymbolAsync(c_tap_pool, taps_dev, (size_t)n * sizeof(float2), (size_t)start * sizeof(float2),
                                 cudaMemcpyDeviceToDevice, st));
  g_pool_used.push_back({dev, start, n, nullptr, false, sid});
  *off = start;
  return GM_OK;
}

void GM_CAT(tap_pool_release_, GM_K)(int off, cudaStream_t st) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return;
  std::lock_guard<std::mutex> lk(g_pool_mu);
  for (size_t i = 0; i < g_pool_used.size(); ++i) {
    TapRegion& r = g_pool_used[i];
    if (r.dev != dev || r.off != off || r.recorded) continue;
    unsigned long long sid = 0;
    if (cudaStreamGetId(st, &sid) == cudaSuccess &&
        cudaEventCreateWithFlags(&r.ev, cudaEventDisableTiming) == cudaSuccess && cudaEventRecord(r.ev, st) == cudaSuccess) {
      r.recorded = true;
      r.sid = sid;
    } else {                                               // cannot track it: wait once, then free
      cudaStreamSynchronize(st);
      g_pool_used.erase(g_pool_used.begin() + i);
    }
    return;
  }
}

template <int K, int RP, int TC, bool CT>
static int launch_forward_v(const FwdArgs& a, int mode, int nthr, size_t sm, unsigned grid, cudaStream_t st, cudaError_t* err) {
  if (mode == FWD_RENDER) {
    GM_TRY(set_smem(k_forward<K, FWD_RENDER, RP, TC, CT>, sm));
    k_forward<K, FWD_RENDER, RP, TC, CT><<<grid, nthr, sm, st>>>(a);
  } else if (mode == FWD_DERIV) {
    GM_TRY(set_smem(k_forward<K, FWD_DERIV, RP, TC, CT>, sm));
    k_forward<K, FWD_DERIV, RP, TC, CT><<<grid, nthr, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_forward<K, FWD_LOSS, RP, TC, CT>, sm));
    k_forward<K, FWD_LOSS, RP, TC, CT><<<grid, nthr, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

int GM_CAT(launch_forward_, GM_K)(const FwdArgs& a, int mode, int B, cudaStream_t st, cudaError_t* err) {
  constexpr int K = GM_K;
  int nthr = (a.tg.ntx * a.tg.nty + 31) / 32 * 32;
  if (nthr > 256) return GM_ENOTSUP;
  nthr = tile_threads<K>(a.tg, nthr, a.ct_off >= 0);
  const size_t sm = smem_bytes<K>(a.tg, nthr / 32, 1, a.ct_off >= 0);
  const unsigned grid = (unsigned)((size_t)B * a.tg.tiles_x * a.tg.tiles_y);
  if (a.ct_off >= 0)
    return a.tg.variant == 1 ? launch_forward_v<K, 3, 12, true>(a, mode, nthr, sm, grid, st, err)
                             : launch_forward_v<K, 4, 8, true>(a, mode, nthr, sm, grid, st, err);
  return a.tg.variant == 1 ? launch_forward_v<K, 3, 12, false>(a, mode, nthr, sm, grid, st, err)
                           : launch_forward_v<K, 4, 8, false>(a, mode, nthr, sm, grid, st, err);
}

int GM_CAT(launch_backward_, GM_K)(const BwdArgs& a, int B, cudaStream_t st, cudaError_t* err) {
  constexpr int K = GM_K;
  int nthr = (a.tg.ntx * a.tg.nty + 31) / 32 * 32;
  if (nthr > 256) return GM_ENOTSUP;
  nthr = tile_threads<K>(a.tg, nthr, a.ct_off >= 0);
  const size_t sm = smem_bytes<K>(a.tg, nthr / 32, kNSum, a.ct_off >= 0);
  const unsigned grid = (unsigned)((size_t)B * a.tg.tiles_x * a.tg.tiles_y);
  const bool ct = a.ct_off >= 0;
  if (a.tg.variant == 1 && ct) {
    GM_TRY(set_smem(k_backward<K, 3, 12, true>, sm));
    k_backward<K, 3, 12, true><<<grid, nthr, sm, st>>>(a);
  } else if (a.tg.variant == 1) {
    GM_TRY(set_smem(k_backward<K, 3, 12, false>, sm));
    k_backward<K, 3, 12, false><<<grid, nthr, sm, st>>>(a);
  } else if (ct) {
    GM_TRY(set_smem(k_backward<K, 4, 8, true>, sm));
    k_backward<K, 4, 8, true><<<grid, nthr, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_backward<K, 4, 8, false>, sm));
    k_backward<K, 4, 8, false><<<grid, nthr, sm, st>>>(a);
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
  const bool ct = a.ct_off >= 0;
  if (variant == 0 && ct) {
    GM_TRY(set_smem(k_fused<K, 4, 8, true>, sm));
    k_fused<K, 4, 8, true><<<grid, kFusedThreads, sm, st>>>(a);
  } else if (variant == 0) {
    GM_TRY(set_smem(k_fused<K, 4, 8, false>, sm));
    k_fused<K, 4, 8, false><<<grid, kFusedThreads, sm, st>>>(a);
  } else if (ct) {
    GM_TRY(set_smem(k_fused<K, 3, 12, true>, sm));
    k_fused<K, 3, 12, true><<<grid, kFusedThreads, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_fused<K, 3, 12, false>, sm));
    k_fused<K, 3, 12, false><<<grid, kFusedThreads, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

// gm_conv, FFMA2 engine
int GM_CAT(launch_conv_, GM_K)(const ConvTileArgs& a, int B, cudaStream_t st, cudaError_t* err) {
  constexpr int K = GM_K;
  int nthr = (a.tg.ntx * a.tg.nty + 31) / 32 * 32;
  if (nthr > 256) return GM_ENOTSUP;
  const bool ct = a.ct_off >= 0;
  const size_t sm = smem_bytes<K>(a.tg, 8, 1, ct);
  const unsigned grid = (unsigned)((size_t)B * a.tg.tiles_x * a.tg.tiles_y);
  if (a.tg.variant == 1 && ct) {
    GM_TRY(set_smem(k_conv_ffma2<K, 3, 12, true>, sm));
    k_conv_ffma2<K, 3, 12, true><<<grid, nthr, sm, st>>>(a);
  } else if (a.tg.variant == 1) {
    GM_TRY(set_smem(k_conv_ffma2<K, 3, 12, false>, sm));
    k_conv_ffma2<K, 3, 12, false><<<grid, nthr, sm, st>>>(a);
  } else if (ct) {
    GM_TRY(set_smem(k_conv_ffma2<K, 4, 8, true>, sm));
    k_conv_ffma2<K, 4, 8, true><<<grid, nthr, sm, st>>>(a);
  } else {
    GM_TRY(set_smem(k_conv_ffma2<K, 4, 8, false>, sm));
    k_conv_ffma2<K, 4, 8, false><<<grid, nthr, sm, st>>>(a);
  }
  GM_TRY(cudaGetLastError());
  return GM_OK;
}

}  // namespace gm
