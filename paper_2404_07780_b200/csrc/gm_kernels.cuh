// gm_kernels.cuh -- the per-tile kernels of the hot path (steps a1-a5 of
// SURVEY.md section 8(a)), templated on the PSF side K.
//
// One CTA owns a TH x TW tile of one galaxy's cutout.  Each thread owns an
// 8 x 8 or 6 x 12 block of output pixels (RP row pairs x TC columns) and runs the direct
// PSF convolution as packed FP32 FMAs (FFMA2 on sm_100a): an accumulator pair holds two
// vertically adjacent output pixels, the multiplicand pair holds two vertically adjacent
// PSF taps, and the input sample is the scalar-broadcast operand, so one instruction
// does two of the 2 K^2 multiply-adds per pixel.  FFMA2 holds the issue port for both of
// its cycles, so every other instruction of the loop is overhead;
// with a batch-wide PSF the tap pair is a uniform-register operand filled from the
// constant bank (CT), which removes the tap loads from the loop.
//
//   k_forward<K, MODE, RP, TC, CT>  a1 render S on tile + halo (shared memory)
//                         a2 M = PSF (*) S          (R:C1, flipped-tap correlation)
//                         a3 rho, chi2 partial, G = -2 w rho -> workspace
//                         (FWD_RENDER: write M instead, gm_render; FWD_DERIV: one
//                         column of the Jacobian, gm_uncertainty)
//   k_backward<K, RP, TC, CT>       a4 A = PSF (star) G   (R:C2) from the G tile + halo
//                         a5 per-tile partial sums of A dS/dp (kNSum per component)
//
// Reductions are fixed-order (thread -> warp shuffle tree -> warps in order ->
// tiles in order in k_finalize); no floating-point atomics anywhere.
#pragma once
#include "gm_device.cuh"

namespace gm {

constexpr int kTR = 8, kTC = 8;            // thread tile (rows x cols)
// SFU forms (lg2.approx / ex2.approx, 2^-22) in the forward render as well: the pixel error
// stays below 1e-5 relative wherever the profile has not underflowed
// and the helper warps of k_fused issue a third fewer instructions.  -DGM_PRECISE_FORWARD
// selects log2f / exp2f instead.
#ifdef GM_PRECISE_FORWARD
constexpr bool kFastForward = false;
#else
constexpr bool kFastForward = true;
#endif

struct TileGeom {
  int H, W;                // cutout
  int TH, TW;              // CTA tile (multiples of 8)
  int tiles_x, tiles_y;    // tiles per cutout
  int ntx, nty;            // thread tiles per CTA tile
  int variant;             // thread tile: 0 = 8 x 8 (RP 4, TC 8), 1 = 6 x 12 (RP 3, TC 12)
  int pitch;               // shared row pitch (floats), multiple of 4
  int rows;                // TH + K - 1
  int vec;                 // 1: W % 4 == 0 and data/sigma/mask/out aligned for 128-bit access
};

struct FwdArgs {
  ModelDesc md;
  TileGeom tg;
  const CompConst* cc;     // [B, n_comp]
  const float2* taps; long long taps_stride;   // paired flipped taps, float2 per galaxy (0 = shared)
  int ct_off;              // >= 0: the taps of the shared PSF sit at c_tap_pool[ct_off ..] (constant bank)
  int ct_zero;             // 0 (see conv_tile_ct)
  const float* data; const float* sigma; const uint8_t* mask;
  float* G;                // [B,H,W] workspace (or model_out when RENDER)
  float* chi2_part;        // [B, tiles]
  const int* frozen;       // [B] or nullptr: skip galaxies that stopped
  const int* live; const int* n_live;   // compacted list of galaxies still iterating, or nullptr
  int b0;                  // first galaxy of this launch (FWD_DERIV chunks; 0 otherwise)
  int dpar;                // FWD_DERIV: index of the parameter to differentiate with respect to
};

// what k_forward produces: G = -2 w rho and chi^2 partials (a3), the model image M
// (gm_render), or one column of the Jacobian dM/dp_dpar (covariance row)
enum { FWD_LOSS = 0, FWD_RENDER = 1, FWD_DERIV = 2 };

struct BwdArgs {
  ModelDesc md;
  TileGeom tg;
  const CompConst* cc;
  const float2* taps; long long taps_stride;   // paired unflipped taps
  int ct_off;              // >= 0: taps at c_tap_pool[ct_off ..]
  int ct_zero;             // 0 (see conv_tile_ct)
  const float* G;          // [B,H,W]
  float* grad_part;        // [B, tiles, n_comp, kNSum]
  const int* frozen;
  const int* live; const int* n_live;
};

template <int K> struct ConvCfg {
  static constexpr int kWin = ((kTC + K - 1) + 3) / 4;   // float4 chunks per input row window
  static constexpr int kTapPitch = K + 1;                // float2 per tap-pair row (even)
  static constexpr int kTapRows = K + 1;
  static constexpr int kInRows = kTR + K - 1;
};

// paired taps: T2[a][t] = (P[a][t], P[a-1][t]), a = 0..K, t = 0..K (column K is a zero
// pad), P[-1] = P[K] = 0.  FLIP selects the flipped PSF (true convolution, R:C1) or the
// PSF itself (adjoint, R:C2).  Built once per call by k_make_taps (gm_api.cu).
template <bool FLIP>
__device__ __forceinline__ float2 tap_pair(const float* __restrict__ psf, int K, int a, int t) {
  float lo = 0.0f, hi = 0.0f;
  if (t < K) {
    const int tt = FLIP ? (K - 1 - t) : t;
    if (a < K) lo = psf[(FLIP ? (K - 1 - a) : a) * K + tt];
    if (a >= 1) hi = psf[(FLIP ? (K - a) : (a - 1)) * K + tt];
  }
  return make_float2(lo, hi);
}

// (2 RP) x TC outputs per thread (8 x 8 or 6 x 12).  win points at the thread's window
// origin in the shared tile (row 0 of its 2 RP + K - 1 input rows, first of its TC + K - 1
// input columns).  acc[rp][c] = (out[2rp][c], out[2rp+1][c]).  With TC = 12 the windows
// of the 8 lanes of a shared-memory wavefront start 12 words apart and touch all 32
// banks once; with TC = 8 they collide two by two.
template <int K, int RP, int TC>
__device__ __forceinline__ void conv_tile(const float* __restrict__ win, int pitch,
                                          const float2* __restrict__ taps, float2 (&acc)[RP][TC]) {
  constexpr int NW = ((TC + K - 1) + 3) / 4;
  constexpr int TP = ConvCfg<K>::kTapPitch;
#pragma unroll 1
  for (int y = 0; y < 2 * RP + K - 1; ++y) {
    float in[NW * 4];
    const float4* row = reinterpret_cast<const float4*>(win + y * pitch);
#pragma unroll
    for (int j = 0; j < NW; ++j) {
      const float4 v = row[j];
      in[4 * j + 0] = v.x; in[4 * j + 1] = v.y; in[4 * j + 2] = v.z; in[4 * j + 3] = v.w;
    }
#pragma unroll
    for (int rp = 0; rp < RP; ++rp) {
      const int a = y - 2 * rp;
      if (a >= 0 && a <= K) {
        const float4* tp = reinterpret_cast<const float4*>(taps + a * TP);
#pragma unroll
        for (int t2 = 0; t2 < (K + 1) / 2; ++t2) {
          const float4 w = tp[t2];                      // two tap pairs
#pragma unroll
          for (int c = 0; c < TC; ++c)
            acc[rp][c] = __ffma2_rn(make_float2(in[c + 2 * t2], in[c + 2 * t2]),
                                    make_float2(w.x, w.y), acc[rp][c]);
          if (2 * t2 + 1 < K) {
#pragma unroll
            for (int c = 0; c < TC; ++c)
              acc[rp][c] = __ffma2_rn(make_float2(in[c + 2 * t2 + 1], in[c + 2 * t2 + 1]),
                                      make_float2(w.z, w.w), acc[rp][c]);
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------
// Taps in the constant bank.  FFMA2 takes its tap pair straight from a UNIFORM register
// (FFMA2 R, R.F32, UR.F32x2, R) that LDCU fills from constant memory: no shared-memory
// load, no vector register and no register-bank conflict per tap.  That needs a tap
// address that is uniform over the warp and a constant-bank home for the taps, so the
// paired taps of a batch-wide PSF are copied (device to device, on the call's stream)
// into a region of this pool for the duration of the call; the region is handed out by
// the host-side allocator in gm_tiles.cu, and when none is free, or the PSF is per
// galaxy, the shared-memory form above runs instead.  The loop runs tap row a outermost
// (so the row's taps are loop constants) and reloads the input row for each row pair;
// every accumulator still sees its K^2 products in the same (a, t) order as conv_tile.
// Stand-alone (148 CTAs, 128 x 128, K = 25): 0.935 of the FP32 peak against 0.823.
// ---------------------------------------------------------------------------
constexpr int kTapPoolN = 7424;                           // float2: 59,392 bytes of the 64 KB bank
__constant__ float2 c_tap_pool[kTapPoolN];

template <int K, int RP, int TC>
__device__ __forceinline__ void conv_tile_ct(const float* __restrict__ win, int pitch, int ct_off, int ct_zero,
                                             float2 (&acc)[RP][TC]) {
  constexpr int NW = ((TC + K - 1) + 3) / 4;
  constexpr int TP = ConvCfg<K>::kTapPitch;
#pragma unroll 2
  for (int a = 0; a <= K; ++a) {
#pragma unroll
    for (int rp = 0; rp < RP; ++rp) {
      // ct_zero is 0 at run time.  Without it the compiler keeps the K tap pairs of row a live
      // across the RP row pairs; beyond K = 33 that exceeds the 63 uniform registers and it
      // falls back to vector registers and shared-memory-speed code.  An address it cannot
      // prove equal makes every row pair reload its taps (LDCU is nearly free).
      const float2* tp = c_tap_pool + ct_off + a * TP + rp * ct_zero;
      float in[NW * 4];
      const float4* row = reinterpret_cast<const float4*>(win + (a + 2 * rp) * pitch);
#pragma unroll
      for (int j = 0; j < NW; ++j) {
        const float4 v = row[j];
        in[4 * j + 0] = v.x; in[4 * j + 1] = v.y; in[4 * j + 2] = v.z; in[4 * j + 3] = v.w;
      }
#pragma unroll
      for (int t = 0; t < K; ++t) {
        const float2 w = tp[t];
#pragma unroll
        for (int c = 0; c < TC; ++c)
          acc[rp][c] = __ffma2_rn(make_float2(in[c + t], in[c + t]), w, acc[rp][c]);
      }
    }
  }
}

// cp.async with zero fill: copies `bytes` (4 or 16) when valid, writes zeros otherwise
__device__ __forceinline__ void cp_async_zfill4(float* dst, const float* src, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(dst);
  const int n = valid ? 4 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(sa), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_zfill16(float* dst, const float* src, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(dst);
  const int n = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// (K+1) x (K+1) float2 of paired taps, global -> shared, 16 bytes per cp.async
template <int K>
__device__ __forceinline__ void copy_taps(float2* dst, const float2* __restrict__ src, int tid, int nthr) {
  constexpr int n16 = (K + 1) * ConvCfg<K>::kTapPitch / 2;
  for (int i = tid; i < n16; i += nthr)
    cp_async_zfill16(reinterpret_cast<float*>(dst) + 4 * i, reinterpret_cast<const float*>(src) + 4 * i, true);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// acc -> the thread's block of the shared tile (rows 2rp, 2rp+1), TC / 4 float4 per row
template <int RP, int TC>
__device__ __forceinline__ void store_acc(float* dst, int pitch, const float2 (&acc)[RP][TC]) {
#pragma unroll
  for (int rp = 0; rp < RP; ++rp) {
    float4* r0 = reinterpret_cast<float4*>(dst + (size_t)(2 * rp) * pitch);
    float4* r1 = reinterpret_cast<float4*>(dst + (size_t)(2 * rp + 1) * pitch);
#pragma unroll
    for (int c = 0; c < TC; c += 4) {
      r0[c >> 2] = make_float4(acc[rp][c].x, acc[rp][c + 1].x, acc[rp][c + 2].x, acc[rp][c + 3].x);
      r1[c >> 2] = make_float4(acc[rp][c].y, acc[rp][c + 1].y, acc[rp][c + 2].y, acc[rp][c + 3].y);
    }
  }
}

// dynamic shared memory: [ tile: rows x pitch floats | taps: (K+1) x (K+1) float2 | red ];
// no tap area when the taps are in the constant bank (ct)
template <int K>
__host__ __device__ inline size_t smem_bytes(const TileGeom& tg, int nwarps, int n_red, bool ct) {
  return (size_t)tg.rows * tg.pitch * 4 + (ct ? 0 : (size_t)(K + 1) * ConvCfg<K>::kTapPitch * 8) +
         (size_t)nwarps * n_red * 4 + 64;
}

// ---------------------------------------------------------------------------
// forward: render + convolve + residual
// ---------------------------------------------------------------------------
template <int K, int MODE, int RP, int TC, bool CT>
__global__ void __launch_bounds__(512) k_forward(const FwdArgs a) {
  constexpr bool RENDER = (MODE != FWD_LOSS);            // an image is written, no residual
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileGeom& tg = a.tg;
  const int tiles = tg.tiles_x * tg.tiles_y;
  int b = a.b0 + blockIdx.x / tiles;
  const int tile = blockIdx.x % tiles;
  if (a.live) {
    if (b >= *a.n_live) return;
    b = a.live[b];
  }
  if (a.frozen && a.frozen[b]) return;
  const int tile_y = tile / tg.tiles_x, tile_x = tile - tile_y * tg.tiles_x;
  const int i0 = tile_y * tg.TH, j0 = tile_x * tg.TW;     // tile origin in the cutout
  constexpr int h = (K - 1) / 2;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int lane = tid & 31, wid = tid >> 5, nwarps = nthr >> 5;

  float* tilebuf = reinterpret_cast<float*>(smem_raw);
  float2* taps = reinterpret_cast<float2*>(tilebuf + (size_t)tg.rows * tg.pitch);
  float* red = reinterpret_cast<float*>(taps + (CT ? 0 : (K + 1) * ConvCfg<K>::kTapPitch));

  if (!CT) copy_taps<K>(taps, a.taps + (long long)b * a.taps_stride, tid, nthr);

  // a1: S on the tile plus its halo; zero outside the cutout (R:C1) and in the pad.
  // One pass per convolved component, its radial law selected outside the pixel loops.
  // FWD_DERIV: one pass per (component, slot) that names parameter dpar, filling
  // dS/dp_dpar instead (tied parameters add).
  const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
  const int cols = tg.TW + K - 1;
  bool first = true;
  // groups of four consecutive columns, one group per lane (row4 / value4, gm_device.cuh)
  const int P4 = tg.pitch >> 2;
  const int ngrp = tg.rows * P4;
  const float inv_p4 = 1.0f / (float)P4;
  auto fill = [&](int kind, const CompConst cc, bool box, bool mag, int slot) {
    dispatch_kind(kind, [&]<int KIND>() {
      for (int idx = tid; idx < ngrp; idx += nthr) {
        const int yy = (int)(((float)idx + 0.5f) * inv_p4), xx = (idx - yy * P4) << 2;
        const int i = i0 - h + yy, j = j0 - h + xx;
        float4* dst = reinterpret_cast<float4*>(tilebuf + (size_t)yy * tg.pitch + xx);
        const bool any = KIND != GM_SKY && i >= 0 && i < tg.H && xx < cols && j + 3 >= 0 && j < tg.W;
        if (!any) {
          if (first) *dst = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
          continue;
        }
        const float y = (float)tg.H - 0.5f - (float)i;   // R:G1
        float v[4];
        if (MODE == FWD_DERIV) {
#pragma unroll
          for (int k = 0; k < 4; ++k) v[k] = component_deriv_t<KIND>(cc, box, mag, slot, (float)(j + k) + 0.5f, y);
        } else {
          value4<KIND, kFastForward>(cc, box, (float)j + 0.5f, y, v);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (!(xx + k < cols && j + k >= 0 && j + k < tg.W)) v[k] = 0.0f;
        float4 o = make_float4(v[0], v[1], v[2], v[3]);
        if (!first) {
          const float4 q = *dst;
          o.x += q.x; o.y += q.y; o.z += q.z; o.w += q.w;
        }
        *dst = o;
      }
    });
    first = false;
  };
  for (int c = 0; c < a.md.n_comp; ++c) {
    if (!a.md.conv[c]) continue;
    const bool box = a.md.box[c] != 0, mag = a.md.mag[c] != 0;
    if (MODE == FWD_DERIV) {
      for (int k = 0; k < GM_NSLOT; ++k)
        if (a.md.slot[c][k] == a.dpar) fill(a.md.kind[c], ccb[c], box, mag, k);
    } else {
      fill(a.md.kind[c], ccb[c], box, mag, -1);
    }
  }
  if (first) fill((int)GM_SKY, ccb[0], false, false, -1);   // nothing convolved: a zero tile
  cp_async_wait_all();
  __syncthreads();

  // a2: M = PSF (*) S on this thread's 8x8 block
  const int ty = tid / tg.ntx, tx = tid - ty * tg.ntx;
  const bool active = ty < tg.nty;
  float2 acc[RP][TC];
#pragma unroll
  for (int rp = 0; rp < RP; ++rp)
#pragma unroll
    for (int c = 0; c < TC; ++c) acc[rp][c] = make_float2(0.0f, 0.0f);
  if (active) {
    const float* win = tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC;
    if (CT) conv_tile_ct<K, RP, TC>(win, tg.pitch, a.ct_off, a.ct_zero, acc);
    else conv_tile<K, RP, TC>(win, tg.pitch, taps, acc);
  }

  // park M in the (now dead) tile buffer so that the epilogue can walk the tile
  // row-major with coalesced global accesses
  __syncthreads();
  if (active) store_acc<RP, TC>(tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC, tg.pitch, acc);
  __syncthreads();

  // a3: unconvolved components, residual, chi2, back-seed G
  float chi2 = 0.0f;
  const size_t img = (size_t)(MODE == FWD_DERIV ? b - a.b0 : b) * tg.H * tg.W;
  bool any_unconv = false;
  for (int c = 0; c < a.md.n_comp; ++c) any_unconv |= (a.md.conv[c] == 0);
  auto add_unconv = [&](float m, float x, float y) {
    for (int c = 0; c < a.md.n_comp; ++c) {
      if (a.md.conv[c]) continue;
      const CompConst cc = ccb[c];
      const int kind = a.md.kind[c];
      const bool box = a.md.box[c] != 0;
      if (MODE == FWD_DERIV) {
        for (int k = 0; k < GM_NSLOT; ++k)
          if (a.md.slot[c][k] == a.dpar) m += component_deriv(kind, cc, box, a.md.mag[c] != 0, k, x, y);
      } else {
        const float U = (kind == GM_SKY) ? 1.0f : profile_value(kind, cc, geometry<false>(cc, box, x, y).r);
        m = fmaf(cc.amp, U, m);
      }
    }
    return m;
  };
  // branch free; weight and residual are SELECTED for unused pixels, never multiplied by 0 (R:X1)
  auto residual = [&](float m, float d, float sg, bool used, float& g) {
    float w = rcp_fast(sg * sg), rho = d - m;
    w = used ? w : 0.0f;
    rho = used ? rho : 0.0f;
    const float t = w * rho;
    chi2 = fmaf(t, rho, chi2);
    g = -2.0f * t;
  };
  if (tg.vec) {
    // 128-bit path: one lane = 4 consecutive pixels, two groups per thread in flight
    const int T4 = tg.TW >> 2, ng = tg.TH * T4;
    const float inv_t4 = 1.0f / (float)T4;
#pragma unroll 1
    for (int idx = tid; idx < ng; idx += 2 * nthr) {
      float4 m4[2], d4[2], s4[2];
      uchar4 k4[2];
      bool ok[2];
      size_t off[2];
      int yr[2], xc[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int id = idx + u * nthr;
        yr[u] = (int)(((float)id + 0.5f) * inv_t4); xc[u] = (id - yr[u] * T4) << 2;
        const int i = i0 + yr[u], j = j0 + xc[u];
        ok[u] = (id < ng) && (i < tg.H) && (j < tg.W);
        off[u] = img + (size_t)i * tg.W + j;
        k4[u] = make_uchar4(1, 1, 1, 1);
        if (ok[u]) {
          m4[u] = *reinterpret_cast<const float4*>(tilebuf + (size_t)yr[u] * tg.pitch + xc[u]);
          if (!RENDER) {
            d4[u] = *reinterpret_cast<const float4*>(a.data + off[u]);
            s4[u] = *reinterpret_cast<const float4*>(a.sigma + off[u]);
            if (a.mask) k4[u] = *reinterpret_cast<const uchar4*>(a.mask + off[u]);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        if (!ok[u]) continue;
        if (any_unconv) {
          const float y = (float)tg.H - 0.5f - (float)(i0 + yr[u]);
          const float x = (float)(j0 + xc[u]) + 0.5f;
          m4[u].x = add_unconv(m4[u].x, x, y);
          m4[u].y = add_unconv(m4[u].y, x + 1.0f, y);
          m4[u].z = add_unconv(m4[u].z, x + 2.0f, y);
          m4[u].w = add_unconv(m4[u].w, x + 3.0f, y);
        }
        if (RENDER) {
          *reinterpret_cast<float4*>(a.G + off[u]) = m4[u];
        } else {
          float4 g;
          residual(m4[u].x, d4[u].x, s4[u].x, k4[u].x != 0, g.x);
          residual(m4[u].y, d4[u].y, s4[u].y, k4[u].y != 0, g.y);
          residual(m4[u].z, d4[u].z, s4[u].z, k4[u].z != 0, g.z);
          residual(m4[u].w, d4[u].w, s4[u].w, k4[u].w != 0, g.w);
          *reinterpret_cast<float4*>(a.G + off[u]) = g;
        }
      }
    }
  } else {
    for (int yy = wid; yy < tg.TH; yy += nwarps) {
      const int i = i0 + yy;
      if (i >= tg.H) break;
      const float y = (float)tg.H - 0.5f - (float)i;
      for (int xx = lane; xx < tg.TW; xx += 32) {
        const int j = j0 + xx;
        if (j >= tg.W) break;
        float m = tilebuf[(size_t)yy * tg.pitch + xx];
        if (any_unconv) m = add_unconv(m, (float)j + 0.5f, y);
        const size_t o = img + (size_t)i * tg.W + j;
        if (RENDER) {
          a.G[o] = m;
        } else {
          float g;
          residual(m, a.data[o], a.sigma[o], a.mask ? (a.mask[o] != 0) : true, g);
          a.G[o] = g;
        }
      }
    }
  }
  if (!RENDER) {
    chi2 = warp_sum(chi2);
    if (lane == 0) red[wid] = chi2;
    __syncthreads();
    if (tid == 0) {
      float s = 0.0f;
      for (int w = 0; w < nwarps; ++w) s += red[w];
      a.chi2_part[(size_t)b * tiles + tile] = s;
    }
  }
}

// ---------------------------------------------------------------------------
// backward: adjoint convolution + parameter-gradient partial sums
// (10 per component, see grad_accumulate in gm_device.cuh)
// ---------------------------------------------------------------------------
template <int K, int RP, int TC, bool CT>
__global__ void __launch_bounds__(512) k_backward(const BwdArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileGeom& tg = a.tg;
  const int tiles = tg.tiles_x * tg.tiles_y;
  int b = blockIdx.x / tiles;
  const int tile = blockIdx.x - b * tiles;
  if (a.live) {
    if (b >= *a.n_live) return;
    b = a.live[b];
  }
  if (a.frozen && a.frozen[b]) return;
  const int tile_y = tile / tg.tiles_x, tile_x = tile - tile_y * tg.tiles_x;
  const int i0 = tile_y * tg.TH, j0 = tile_x * tg.TW;
  constexpr int h = (K - 1) / 2;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int lane = tid & 31, wid = tid >> 5, nwarps = nthr >> 5;

  float* tilebuf = reinterpret_cast<float*>(smem_raw);
  float2* taps = reinterpret_cast<float2*>(tilebuf + (size_t)tg.rows * tg.pitch);
  float* red = reinterpret_cast<float*>(taps + (CT ? 0 : (K + 1) * ConvCfg<K>::kTapPitch));

  if (!CT) copy_taps<K>(taps, a.taps + (long long)b * a.taps_stride, tid, nthr);

  // G tile + halo through cp.async (no register staging, all copies in flight at
  // once); zero outside the cutout (R:C2) and in the pad columns
  const float* Gb = a.G + (size_t)b * tg.H * tg.W;
  const bool vec16 = ((tg.W & 3) == 0) && ((h & 3) == 0);
  if (vec16) {
    const int chunks = tg.pitch >> 2;
    for (int yy = wid; yy < tg.rows; yy += nwarps) {
      const int i = i0 - h + yy;
      float* rowp = tilebuf + (size_t)yy * tg.pitch;
      const bool row_in = (i >= 0 && i < tg.H);
      const float* src_row = Gb + (size_t)(row_in ? i : 0) * tg.W;
      for (int ch = lane; ch < chunks; ch += 32) {
        const int j = j0 - h + 4 * ch;
        const bool ok = row_in && j >= 0 && j < tg.W;
        cp_async_zfill16(rowp + 4 * ch, src_row + (ok ? j : 0), ok);
      }
    }
  } else {
    for (int yy = wid; yy < tg.rows; yy += nwarps) {
      const int i = i0 - h + yy;
      float* rowp = tilebuf + (size_t)yy * tg.pitch;
      const bool row_in = (i >= 0 && i < tg.H);
      const float* src_row = Gb + (size_t)(row_in ? i : 0) * tg.W;
      for (int xx = lane; xx < tg.pitch; xx += 32) {
        const int j = j0 - h + xx;
        const bool ok = row_in && j >= 0 && j < tg.W;
        cp_async_zfill4(rowp + xx, src_row + (ok ? j : 0), ok);
      }
    }
  }
  cp_async_wait_all();
  __syncthreads();

  const int ty = tid / tg.ntx, tx = tid - ty * tg.ntx;
  const bool active = ty < tg.nty;
  float2 acc[RP][TC];
#pragma unroll
  for (int rp = 0; rp < RP; ++rp)
#pragma unroll
    for (int c = 0; c < TC; ++c) acc[rp][c] = make_float2(0.0f, 0.0f);
  if (active) {
    const float* win = tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC;
    if (CT) conv_tile_ct<K, RP, TC>(win, tg.pitch, a.ct_off, a.ct_zero, acc);
    else conv_tile<K, RP, TC>(win, tg.pitch, taps, acc);
  }

  // park A in the tile buffer (G itself stays in global memory for the
  // unconvolved components), then walk the tile row-major
  __syncthreads();
  if (active) store_acc<RP, TC>(tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC, tg.pitch, acc);
  __syncthreads();

  // a5: partial sums per component
  const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
  float* outp = a.grad_part + ((size_t)b * tiles + tile) * a.md.n_comp * kNSum;
  for (int c = 0; c < a.md.n_comp; ++c) {
    float s[kNSum];
#pragma unroll
    for (int k = 0; k < kNSum; ++k) s[k] = 0.0f;
    const CompConst cc = ccb[c];
    const bool conv = a.md.conv[c] != 0, box = a.md.box[c] != 0;
    dispatch_kind(a.md.kind[c], [&]<int KIND>() {
      if (box) {                                           // Eq. 2 with B != 0: per-pixel geometry
        for (int yy = wid; yy < tg.TH; yy += nwarps) {
          const int i = i0 + yy;
          if (i >= tg.H) break;
          const float y = (float)tg.H - 0.5f - (float)i;
          for (int xx = lane; xx < tg.TW; xx += 32) {
            const int j = j0 + xx;
            if (j >= tg.W) break;
            const float seed = conv ? tilebuf[(size_t)yy * tg.pitch + xx] : Gb[(size_t)i * tg.W + j];
            grad_accumulate<KIND>(cc, true, seed, (float)j + 0.5f, y, s);
          }
        }
      } else {                                             // groups of four pixels of a row per lane
        GradAcc<KIND> acc;
        acc.init();
        const int T4 = (tg.TW + 3) >> 2, ng = tg.TH * T4;
        const float inv_t4 = 1.0f / (float)T4;
        for (int idx = tid; idx < ng; idx += nthr) {
          const int yy = (int)(((float)idx + 0.5f) * inv_t4), xx = (idx - yy * T4) << 2;
          const int i = i0 + yy, j = j0 + xx;
          if (i >= tg.H || j >= tg.W) continue;
          float seed[4];
          if (conv) {
            const float4 q = *reinterpret_cast<const float4*>(tilebuf + (size_t)yy * tg.pitch + xx);
            seed[0] = q.x; seed[1] = q.y; seed[2] = q.z; seed[3] = q.w;
          }
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const bool in = xx + k < tg.TW && j + k < tg.W;
            if (!conv) seed[k] = in ? Gb[(size_t)i * tg.W + j + k] : 0.0f;
            else if (!in) seed[k] = 0.0f;
          }
          grad_add4<KIND>(acc, cc, seed, (float)j + 0.5f, (float)tg.H - 0.5f - (float)i);
        }
        acc.finish(cc, s);
      }
    });
    if (!box) s[8] = s[2];
#pragma unroll
    for (int k = 0; k < kNSum; ++k) {
      const float v = warp_sum(s[k]);
      if (lane == 0) red[wid * kNSum + k] = v;
    }
    __syncthreads();
    if (tid < kNSum) {
      float t = 0.0f;
      for (int w = 0; w < nwarps; ++w) t += red[w * kNSum + tid];
      outp[c * kNSum + tid] = t;
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------
// gm_conv, engine GM_CONV_FFMA2: the convolution loop above on its own (out = PSF (*) in
// with the flipped taps, or the adjoint with the taps as given), one tile per CTA.  It is
// the FP32 side of the comparison with the tensor-core engine (gm_tc.cuh).
// ---------------------------------------------------------------------------
struct ConvTileArgs {
  TileGeom tg;
  const float2* taps; long long taps_stride;
  int ct_off, ct_zero;
  const float* in;         // [B,H,W]
  float* out;              // [B,H,W]
};

template <int K, int RP, int TC, bool CT>
__global__ void __launch_bounds__(512) k_conv_ffma2(const ConvTileArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileGeom& tg = a.tg;
  const int tiles = tg.tiles_x * tg.tiles_y;
  const int b = blockIdx.x / tiles, tile = blockIdx.x - b * tiles;
  const int tile_y = tile / tg.tiles_x, tile_x = tile - tile_y * tg.tiles_x;
  const int i0 = tile_y * tg.TH, j0 = tile_x * tg.TW;
  constexpr int h = (K - 1) / 2;
  const int tid = threadIdx.x, nthr = blockDim.x;
  float* tilebuf = reinterpret_cast<float*>(smem_raw);
  float2* taps = reinterpret_cast<float2*>(tilebuf + (size_t)tg.rows * tg.pitch);
  if (!CT) copy_taps<K>(taps, a.taps + (long long)b * a.taps_stride, tid, nthr);
  const float* src = a.in + (size_t)b * tg.H * tg.W;
  for (int idx = tid; idx < tg.rows * tg.pitch; idx += nthr) {       // tile + halo, zero outside the cutout
    const int yy = idx / tg.pitch, xx = idx - yy * tg.pitch;
    const int i = i0 - h + yy, j = j0 - h + xx;
    const bool ok = i >= 0 && i < tg.H && j >= 0 && j < tg.W;
    cp_async_zfill4(tilebuf + idx, src + (ok ? (size_t)i * tg.W + j : 0), ok);
  }
  cp_async_wait_all();
  __syncthreads();
  const int ty = tid / tg.ntx, tx = tid - ty * tg.ntx;
  const bool active = ty < tg.nty;
  float2 acc[RP][TC];
#pragma unroll
  for (int rp = 0; rp < RP; ++rp)
#pragma unroll
    for (int c = 0; c < TC; ++c) acc[rp][c] = make_float2(0.0f, 0.0f);
  if (active) {
    const float* win = tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC;
    if (CT) conv_tile_ct<K, RP, TC>(win, tg.pitch, a.ct_off, a.ct_zero, acc);
    else conv_tile<K, RP, TC>(win, tg.pitch, taps, acc);
  }
  __syncthreads();
  if (active) store_acc<RP, TC>(tilebuf + (size_t)(ty * 2 * RP) * tg.pitch + tx * TC, tg.pitch, acc);
  __syncthreads();
  float* dst = a.out + (size_t)b * tg.H * tg.W;
  for (int idx = tid; idx < tg.TH * tg.TW; idx += nthr) {
    const int yy = idx / tg.TW, xx = idx - yy * tg.TW;
    const int i = i0 + yy, j = j0 + xx;
    if (i < tg.H && j < tg.W) dst[(size_t)i * tg.W + j] = tilebuf[(size_t)yy * tg.pitch + xx];
  }
}

}  // namespace gm
