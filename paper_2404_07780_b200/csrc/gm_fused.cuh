// gm_fused.cuh -- the fused loss + gradient kernel for cutouts that fit one CTA
// (H, W <= 128): steps a1..a5 of SURVEY.md section 8(a) in ONE launch, with nothing but
// chi^2 and the kNSum partial sums per component leaving the SM.
//
// One persistent CTA per SM, 512 threads, two roles that run concurrently:
//
//   conv warps   (0..7)   only the FFMA2 convolution loop: forward M = PSF (*) S, then
//                         adjoint A = PSF (star) G, in place in a shared-memory slot
//   helper warps (8..15)  everything else: a1 render S into a slot, a3 residual
//                         (M -> G in place, chi^2), a5 gradient sums from A
//
// A SLOT holds G whole cutouts (G = 1, 2, 4 or 8, chosen on the host so that the 256 conv
// threads are all busy: four 64x64 cutouts, two 96x96, one 128x128).  Each thread owns a
// (2 RP) x TC block of output pixels of one cutout; the helper warps split into G groups,
// one per cutout of the slot.  Two slots are in flight; the conv warps run
// C1(a) C1(b) C2(a) C2(b) back to back while the helpers prepare the other slot:
//
//   conv   : C1(a)   | C1(b)   | C2(a)   | C2(b)          | C1(c) ...
//   helper : P1(b)   | E1(a)   | E1(b)   | E2(a) P1(c)    | E2(b) P1(d) ...
//
// so the FP32 pipe never waits for the memory and SFU latency of render, residual and
// gradient.  That work is NOT free, though: FFMA2 holds the issue port for both of its
// cycles, so every helper instruction takes a cycle from the convolution (measured,
// DESIGN.md section 5) and the helper loops are written to issue as little as possible.
// Hand-off is by named barriers (bar.arrive / bar.sync): full[s] helper -> conv,
// done[s] conv -> helper.  The taps of a batch-wide PSF are read from the constant bank
// through uniform registers (CT, conv_rows_ct); per-galaxy taps from shared memory.
//
// Slot layout.  Outside the cutout both convolution inputs are zero (R:C1, R:C2), so a
// cutout is stored as its H rows of `pitch` floats ([h zeros | W pixels | zeros]) plus ONE
// shared zero row; the convolution loop redirects every input row outside [0, H) to that
// row.  That is 24 (K = 25) or 40 (K = 41) rows less per cutout than a full halo, which
// is what lets two 128x128 slots with a 41x41 PSF (the paper's SDSS set-up) or
// eight 64x64 cutouts fit the 227 KB of shared memory.
#pragma once
#include "gm_kernels.cuh"

namespace gm {

constexpr int kConvWarps = 8, kHelpWarps = 8;
constexpr int kConvThreads = 32 * kConvWarps;
constexpr int kFusedThreads = 32 * (kConvWarps + kHelpWarps);

struct FusedGeom {
  int H, W;
  int ntx, nty, tpg;         // thread tiles per cutout: across, down, total
  int G;                     // cutouts per slot (1, 2, 4, 8)
  int pitch;                 // floats per slot row, multiple of 4
  int gal_elems;             // (H + 1) * pitch: H rows + the zero row
  int vec;                   // 128-bit global access is possible (W % 4 == 0, pointers aligned)
  int shared_taps;           // one PSF for the batch: taps are loaded once per CTA
};

struct FusedArgs {
  ModelDesc md;
  FusedGeom fg;
  int B;
  int mode;                  // 0 render (write M), 1 chi^2 only, 2 chi^2 + gradient
  int any_unconv;            // model has unconvolved components (G also goes to global)
  const CompConst* cc;
  const float2* taps_fwd; const float2* taps_adj; long long taps_stride;
  int ct_off;                // >= 0: both tap sets of the shared PSF at c_tap_pool[ct_off ..] (forward, then adjoint)
  int ct_zero;               // 0 (see conv_tile_ct)
  const float* data; const float* sigma; const uint8_t* mask;
  float* G;                  // [B,H,W]: model_out (mode 0) or back-seed spill (any_unconv)
  float* chi2_part;          // [B]
  float* grad_part;          // [B, n_comp, kNSum]
  const int* frozen;
  const int* live; const int* n_live;   // compacted list of galaxies still iterating (gm_fit) or nullptr
};

enum { BAR_FULL0 = 1, BAR_FULL1 = 2, BAR_DONE0 = 3, BAR_DONE1 = 4, BAR_CONV = 5, BAR_HELP = 6 };

__device__ __forceinline__ void bar_sync(int id, int n) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int n) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}

template <int K>
__host__ __device__ constexpr int fused_tapn() { return (K + 1) * ConvCfg<K>::kTapPitch; }

// shared memory of one CTA: [2 slots][G cutouts][gal_elems] floats | tap sets | reduction scratch
__host__ __device__ inline size_t fused_smem_bytes(int KP, const FusedGeom& fg) {
  const size_t tapn = (size_t)(KP + 1) * (KP + 1);
  const size_t sets = fg.shared_taps ? 2 : (size_t)4 * fg.G;
  return 2 * (size_t)fg.G * fg.gal_elems * 4 + sets * tapn * 8 + (size_t)kHelpWarps * kNSum * 4 + 64;
}

// (2 RP) x TC outputs per thread, accumulator pairs = vertically adjacent pixels (see
// conv_tile in gm_kernels.cuh for the FFMA2 scheme).  `gal` is the cutout's slot, i0 the
// image row of the thread's first input row (may be negative), c0 its first slot column.
template <int K, int RP, int TC>
__device__ __forceinline__ void conv_rows(const float* __restrict__ gal, int pitch, int H, int i0, int c0,
                                          const float2* __restrict__ taps, float2 (&acc)[RP][TC]) {
  constexpr int NW = ((TC + K - 1) + 3) / 4;
  constexpr int TP = ConvCfg<K>::kTapPitch;
#pragma unroll 1
  for (int y = 0; y < 2 * RP + K - 1; ++y) {
    const int i = i0 + y;
    const int r = ((unsigned)i < (unsigned)H) ? i : H;          // outside the cutout: the zero row
    float in[NW * 4];
    const float4* row = reinterpret_cast<const float4*>(gal + r * pitch + c0);
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
            acc[rp][c] = __ffma2_rn(make_float2(in[c + 2 * t2], in[c + 2 * t2]), make_float2(w.x, w.y), acc[rp][c]);
          if (2 * t2 + 1 < K) {
#pragma unroll
            for (int c = 0; c < TC; ++c)
              acc[rp][c] = __ffma2_rn(make_float2(in[c + 2 * t2 + 1], in[c + 2 * t2 + 1]), make_float2(w.z, w.w),
                                      acc[rp][c]);
          }
        }
      }
    }
  }
}

// the same with the taps in the constant bank (conv_tile_ct, gm_kernels.cuh): tap row a
// outermost, the input row (or the zero row) reloaded for every row pair
template <int K, int RP, int TC>
__device__ __forceinline__ void conv_rows_ct(const float* __restrict__ gal, int pitch, int H, int i0, int c0,
                                             int ct_off, int ct_zero, float2 (&acc)[RP][TC]) {
  constexpr int NW = ((TC + K - 1) + 3) / 4;
  constexpr int TP = ConvCfg<K>::kTapPitch;
#pragma unroll 2
  for (int a = 0; a <= K; ++a) {
#pragma unroll
    for (int rp = 0; rp < RP; ++rp) {
      const float2* tp = c_tap_pool + ct_off + a * TP + rp * ct_zero;   // ct_zero = 0: see conv_tile_ct
      const int i = i0 + a + 2 * rp;
      const int r = ((unsigned)i < (unsigned)H) ? i : H;          // outside the cutout: the zero row
      float in[NW * 4];
      const float4* row = reinterpret_cast<const float4*>(gal + r * pitch + c0);
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

// acc -> interior of the cutout's slot (row r, column c + h); 128-bit stores when aligned.
// Outputs that fall outside the H x W cutout (ragged thread tile) are not stored: the slot
// is the input of the adjoint convolution next, whose zero fill starts at the cutout edge.
template <int K, int RP, int TC>
__device__ __forceinline__ void store_acc_slot(float* gal, int pitch, int r0, int c0, int H, int W,
                                               const float2 (&acc)[RP][TC]) {
  constexpr int h = (K - 1) / 2;
  float* dst = gal + (size_t)r0 * pitch + c0 + h;
  if ((h & 3) == 0 && (TC & 3) == 0 && r0 + 2 * RP <= H && c0 + TC <= W) {
#pragma unroll
    for (int rp = 0; rp < RP; ++rp) {
      float4* q0 = reinterpret_cast<float4*>(dst + (size_t)(2 * rp) * pitch);
      float4* q1 = reinterpret_cast<float4*>(dst + (size_t)(2 * rp + 1) * pitch);
#pragma unroll
      for (int c = 0; c < TC; c += 4) {
        q0[c >> 2] = make_float4(acc[rp][c].x, acc[rp][c + 1].x, acc[rp][c + 2].x, acc[rp][c + 3].x);
        q1[c >> 2] = make_float4(acc[rp][c].y, acc[rp][c + 1].y, acc[rp][c + 2].y, acc[rp][c + 3].y);
      }
    }
  } else {
#pragma unroll
    for (int rp = 0; rp < RP; ++rp)
#pragma unroll
      for (int c = 0; c < TC; ++c) {
        if (c0 + c < W) {
          if (r0 + 2 * rp < H) dst[(size_t)(2 * rp) * pitch + c] = acc[rp][c].x;
          if (r0 + 2 * rp + 1 < H) dst[(size_t)(2 * rp + 1) * pitch + c] = acc[rp][c].y;
        }
      }
  }
}

template <int K, int RP, int TC, bool CT>
__global__ void __launch_bounds__(kFusedThreads, 1) k_fused(const FusedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const FusedGeom& fg = a.fg;
  constexpr int h = (K - 1) / 2;
  constexpr int TAPN = fused_tapn<K>();                           // float2 per tap set
  const int G = fg.G;
  const size_t slot_elems = (size_t)G * fg.gal_elems;
  float* buf0 = reinterpret_cast<float*>(smem_raw);
  float2* taps0 = reinterpret_cast<float2*>(buf0 + 2 * slot_elems);
  float* red = reinterpret_cast<float*>(taps0 + (fg.shared_taps ? 2 : 4 * G) * TAPN);

  const int tid = threadIdx.x;
  const int wid = tid >> 5, lane = tid & 31;
  const bool with_grad = a.mode == 2;
  const int n_gal = a.live ? *a.n_live : a.B;
  // the galaxies of this CTA: entries blockIdx.x, blockIdx.x + gridDim.x, ... of the list,
  // taken G at a time (one item = one slot load)
  const int n_k = (n_gal - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int n_items = (n_k + G - 1) / G;
  auto galaxy = [&](int item, int g) -> int {                     // -1: no galaxy in this place
    const int k = item * G + g;
    if (k >= n_k) return -1;
    const int i = (int)blockIdx.x + k * (int)gridDim.x;
    const int b = a.live ? a.live[i] : i;
    return (a.frozen && a.frozen[b]) ? -1 : b;
  };
  auto taps_of = [&](int s, int g, int phase) -> float2* {
    return fg.shared_taps ? taps0 + phase * TAPN : taps0 + ((s * G + g) * 2 + phase) * TAPN;
  };

  if (wid < kConvWarps) {
    // ------------------------------ conv warps ------------------------------------
    const int g = tid / fg.tpg, rem = tid - g * fg.tpg;
    const int ty = rem / fg.ntx, tx = rem - ty * fg.ntx;
    const bool mine = g < G;
    for (int m = 0; 2 * m < n_items; ++m) {
      for (int phase = 0; phase < (with_grad ? 2 : 1); ++phase) {
        for (int s = 0; s < 2; ++s) {
          const int item = 2 * m + s;
          if (item >= n_items) continue;
          const bool active = mine && galaxy(item, g) >= 0;
          float* gal = buf0 + s * slot_elems + (size_t)(mine ? g : 0) * fg.gal_elems;
          bar_sync(BAR_FULL0 + s, kFusedThreads);               // input (S or G) is ready
          float2 acc[RP][TC];
#pragma unroll
          for (int rp = 0; rp < RP; ++rp)
#pragma unroll
            for (int c = 0; c < TC; ++c) acc[rp][c] = make_float2(0.0f, 0.0f);
          if (active) {
            if (CT) conv_rows_ct<K, RP, TC>(gal, fg.pitch, fg.H, ty * 2 * RP - h, tx * TC, a.ct_off + phase * TAPN, a.ct_zero, acc);
            else conv_rows<K, RP, TC>(gal, fg.pitch, fg.H, ty * 2 * RP - h, tx * TC, taps_of(s, g, phase), acc);
          }
          bar_sync(BAR_CONV, kConvThreads);                     // every conv thread is done reading
          if (active) store_acc_slot<K, RP, TC>(gal, fg.pitch, ty * 2 * RP, tx * TC, fg.H, fg.W, acc);
          bar_arrive(BAR_DONE0 + s, kFusedThreads);             // M (or A) is parked in the slot
        }
      }
    }
    return;
  }

  // -------------------------------- helper warps ------------------------------------
  const int hw = wid - kConvWarps;                 // 0..7
  const int htid = tid - kConvThreads;             // 0..255
  constexpr int HN = 32 * kHelpWarps;
  const int hpg = kHelpWarps / G;                  // helper warps per cutout of a slot
  const int hg = hw / hpg, lw = hw - hg * hpg;     // this warp's cutout and its rank there

  // Every slot is zeroed once per CTA: the zero row and the left / right margins of the
  // rows stay zero from then on (render, convolution output and residual only ever write
  // the H x W interior).  The taps of a shared PSF are loaded once per CTA as well.
  {
    float4* z = reinterpret_cast<float4*>(buf0);
    const int n4 = (int)((2 * slot_elems) >> 2);            // gal_elems is a multiple of 4
    for (int i = htid; i < n4; i += HN) z[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  if (!CT && fg.shared_taps) {
    for (int i = htid; i < TAPN / 2; i += HN) {
      cp_async_zfill16(reinterpret_cast<float*>(taps0) + 4 * i, reinterpret_cast<const float*>(a.taps_fwd) + 4 * i, true);
      cp_async_zfill16(reinterpret_cast<float*>(taps0 + TAPN) + 4 * i,
                       reinterpret_cast<const float*>(a.taps_adj) + 4 * i, true);
    }
    cp_async_wait_all();
  }

  // The helper loops walk a cutout in groups of four consecutive pixels of a row, one group
  // per lane: group idx -> (row, first column).  The warps of a cutout interleave by 32 groups.
  const int W4 = (fg.W + 3) >> 2;
  const int ngrp = fg.H * W4;
  const float inv_w4 = 1.0f / (float)W4;
  const int gstart = lw * 32 + lane, gstep = hpg * 32;
  auto group_row = [&](int idx) -> int { return (int)(((float)idx + 0.5f) * inv_w4); };   // exact: idx < 2^16
  constexpr bool kAligned = (h & 3) == 0;                  // slot interior is 16-byte aligned

  // a1: S of this group's cutout, and its taps when they are per galaxy
  auto produce = [&](int item, int s) {
    const int b = galaxy(item, hg);
    if (b < 0) return;
    float* gal = buf0 + s * slot_elems + (size_t)hg * fg.gal_elems;
    if (!fg.shared_taps) {
      float2* tp = taps_of(s, hg, 0);
      const float2* src = a.taps_fwd + (long long)b * a.taps_stride;
      const float2* srca = a.taps_adj + (long long)b * a.taps_stride;
      for (int i = lw * 32 + lane; i < TAPN / 2; i += hpg * 32) {
        cp_async_zfill16(reinterpret_cast<float*>(tp) + 4 * i, reinterpret_cast<const float*>(src) + 4 * i, true);
        cp_async_zfill16(reinterpret_cast<float*>(tp + TAPN) + 4 * i, reinterpret_cast<const float*>(srca) + 4 * i, true);
      }
    }
    const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
    bool first = true;
    for (int c = 0; c <= a.md.n_comp; ++c) {
      const bool zero_pass = (c == a.md.n_comp);           // nothing convolved: S = 0
      if (zero_pass && !first) break;
      if (!zero_pass && (!a.md.conv[c] || a.md.kind[c] == GM_SKY)) continue;
      const CompConst cc = ccb[zero_pass ? 0 : c];
      const bool box = !zero_pass && a.md.box[c] != 0;
      dispatch_kind(zero_pass ? (int)GM_SKY : a.md.kind[c], [&]<int KIND>() {
        for (int idx = gstart; idx < ngrp; idx += gstep) {
          const int i = group_row(idx), x = (idx - i * W4) << 2;
          float v[4] = {0.0f, 0.0f, 0.0f, 0.0f};
          if (KIND != GM_SKY) value4<KIND, kFastForward>(cc, box, (float)x + 0.5f, (float)fg.H - 0.5f - (float)i, v);   // R:G1
          float* p = gal + (size_t)i * fg.pitch + h + x;
          if (kAligned && x + 4 <= fg.W) {
            float4 o = make_float4(v[0], v[1], v[2], v[3]);
            if (!first) {
              const float4 q = *reinterpret_cast<const float4*>(p);
              o.x += q.x; o.y += q.y; o.z += q.z; o.w += q.w;
            }
            *reinterpret_cast<float4*>(p) = o;
          } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
              if (x + k < fg.W) p[k] = first ? v[k] : p[k] + v[k];
          }
        }
      });
      first = false;
    }
    if (!fg.shared_taps) cp_async_wait_all();
  };

  // a3: M (slot interior) -> chi^2 and G in place; mode 0 writes M out instead
  auto residual = [&](int item, int s) {
    const int b = galaxy(item, hg);
    float chi2 = 0.0f;
    if (b >= 0) {
      float* gal = buf0 + s * slot_elems + (size_t)hg * fg.gal_elems;
      const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
      const size_t img = (size_t)b * fg.H * fg.W;
      auto add_unconv = [&](float m, float x, float y) {
        for (int c = 0; c < a.md.n_comp; ++c) {
          if (a.md.conv[c]) continue;
          const CompConst cc = ccb[c];
          const int kind = a.md.kind[c];
          const float U = (kind == GM_SKY) ? 1.0f : profile_value(kind, cc, geometry<false>(cc, a.md.box[c] != 0, x, y).r);
          m = fmaf(cc.amp, U, m);
        }
        return m;
      };
      // branch free; the weight and the residual are SELECTED for unused pixels, never
      // multiplied by 0, so NaN / sigma = 0 under the mask cannot propagate (R:X1)
      auto one = [&](float m, float d, float sg, bool used, float& gv) {
        float w = rcp_fast(sg * sg), rho = d - m;
        w = used ? w : 0.0f;
        rho = used ? rho : 0.0f;
        const float t = w * rho;
        chi2 = fmaf(t, rho, chi2);
        gv = -2.0f * t;
      };
      if (fg.vec && kAligned && a.mode != 0 && !a.any_unconv) {
        // the hot form: chi^2 (+ gradient) of a model without unconvolved components.
        // 128-bit accesses, one lane = 4 pixels, two groups per lane in flight, 32-bit offsets
        const float* dptr = a.data + img;
        const float* sptr = a.sigma + img;
        auto hot = [&]<bool MASKED>() {
          const uint8_t* kptr = MASKED ? a.mask + img : nullptr;
#pragma unroll 1
          for (int idx = gstart; idx < ngrp; idx += 2 * gstep) {
            const int id1 = idx + gstep;
            const bool ok1 = id1 < ngrp;
            const int r0 = group_row(idx), r1 = group_row(ok1 ? id1 : idx);
            const int c0 = (idx - r0 * W4) << 2, c1 = ((ok1 ? id1 : idx) - r1 * W4) << 2;
            const int o0 = r0 * fg.W + c0, o1 = r1 * fg.W + c1;
            float* mp0 = gal + r0 * fg.pitch + c0 + h;
            float* mp1 = gal + r1 * fg.pitch + c1 + h;
            const float4 d0 = *reinterpret_cast<const float4*>(dptr + o0), d1 = *reinterpret_cast<const float4*>(dptr + o1);
            const float4 s0 = *reinterpret_cast<const float4*>(sptr + o0), s1 = *reinterpret_cast<const float4*>(sptr + o1);
            uchar4 k0 = make_uchar4(1, 1, 1, 1), k1 = k0;
            if (MASKED) { k0 = *reinterpret_cast<const uchar4*>(kptr + o0); k1 = *reinterpret_cast<const uchar4*>(kptr + o1); }
            const float4 m0 = *reinterpret_cast<const float4*>(mp0), m1 = *reinterpret_cast<const float4*>(mp1);
            float4 g0, g1;
            one(m0.x, d0.x, s0.x, !MASKED || k0.x != 0, g0.x);
            one(m0.y, d0.y, s0.y, !MASKED || k0.y != 0, g0.y);
            one(m0.z, d0.z, s0.z, !MASKED || k0.z != 0, g0.z);
            one(m0.w, d0.w, s0.w, !MASKED || k0.w != 0, g0.w);
            *reinterpret_cast<float4*>(mp0) = g0;
            if (ok1) {                                     // the pair of a last, odd group is the group itself
              one(m1.x, d1.x, s1.x, !MASKED || k1.x != 0, g1.x);
              one(m1.y, d1.y, s1.y, !MASKED || k1.y != 0, g1.y);
              one(m1.z, d1.z, s1.z, !MASKED || k1.z != 0, g1.z);
              one(m1.w, d1.w, s1.w, !MASKED || k1.w != 0, g1.w);
              *reinterpret_cast<float4*>(mp1) = g1;
            }
          }
        };
        if (a.mask) hot.template operator()<true>();
        else hot.template operator()<false>();
      } else if (fg.vec && kAligned) {
        // general 128-bit path (render output, unconvolved components)
        auto pass = [&]<bool MASKED>() {
#pragma unroll 1
          for (int idx = gstart; idx < ngrp; idx += 2 * gstep) {
            float4 m4[2], d4[2], s4[2];
            uchar4 k4[2];
            bool ok[2];
            size_t off[2];
            float* mp[2];
            int row[2], col[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              const int id = idx + u * gstep;
              ok[u] = id < ngrp;
              row[u] = group_row(id); col[u] = (id - row[u] * W4) << 2;
              off[u] = img + (size_t)row[u] * fg.W + col[u];
              mp[u] = gal + (size_t)row[u] * fg.pitch + col[u] + h;
              k4[u] = make_uchar4(1, 1, 1, 1);
              if (ok[u]) {
                m4[u] = *reinterpret_cast<const float4*>(mp[u]);
                if (a.mode != 0) {
                  d4[u] = *reinterpret_cast<const float4*>(a.data + off[u]);
                  s4[u] = *reinterpret_cast<const float4*>(a.sigma + off[u]);
                  if (MASKED) k4[u] = *reinterpret_cast<const uchar4*>(a.mask + off[u]);
                }
              }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              if (!ok[u]) continue;
              if (a.any_unconv) {
                const float y = (float)fg.H - 0.5f - (float)row[u];
                const float x = (float)col[u] + 0.5f;
                m4[u].x = add_unconv(m4[u].x, x, y);
                m4[u].y = add_unconv(m4[u].y, x + 1.0f, y);
                m4[u].z = add_unconv(m4[u].z, x + 2.0f, y);
                m4[u].w = add_unconv(m4[u].w, x + 3.0f, y);
              }
              if (a.mode == 0) {
                *reinterpret_cast<float4*>(a.G + off[u]) = m4[u];
              } else {
                float4 gv;
                one(m4[u].x, d4[u].x, s4[u].x, !MASKED || k4[u].x != 0, gv.x);
                one(m4[u].y, d4[u].y, s4[u].y, !MASKED || k4[u].y != 0, gv.y);
                one(m4[u].z, d4[u].z, s4[u].z, !MASKED || k4[u].z != 0, gv.z);
                one(m4[u].w, d4[u].w, s4[u].w, !MASKED || k4[u].w != 0, gv.w);
                *reinterpret_cast<float4*>(mp[u]) = gv;
                if (a.any_unconv && with_grad) *reinterpret_cast<float4*>(a.G + off[u]) = gv;
              }
            }
          }
        };
        if (a.mask) pass.template operator()<true>();
        else pass.template operator()<false>();
      } else {
        for (int i = lw; i < fg.H; i += hpg) {
          const float y = (float)fg.H - 0.5f - (float)i;
          for (int j = lane; j < fg.W; j += 32) {
            float* mp = gal + (size_t)i * fg.pitch + j + h;
            float m = *mp;
            if (a.any_unconv) m = add_unconv(m, (float)j + 0.5f, y);
            const size_t o = img + (size_t)i * fg.W + j;
            if (a.mode == 0) {
              a.G[o] = m;
            } else {
              float gv;
              one(m, a.data[o], a.sigma[o], a.mask ? (a.mask[o] != 0) : true, gv);
              *mp = gv;
              if (a.any_unconv && with_grad) a.G[o] = gv;
            }
          }
        }
      }
    }
    if (a.mode != 0) {                                   // every helper thread takes the barriers
      chi2 = warp_sum(chi2);
      if (lane == 0) red[hw] = chi2;
      bar_sync(BAR_HELP, HN);
      if (htid < G) {
        const int bb = galaxy(item, htid);
        if (bb >= 0) {
          float t = 0.0f;
          for (int w = 0; w < hpg; ++w) t += red[htid * hpg + w];
          a.chi2_part[bb] = t;
        }
      }
      bar_sync(BAR_HELP, HN);
    }
  };

  // a5: the partial sums of every component from A (slot interior)
  auto gradient = [&](int item, int s) {
    const int b = galaxy(item, hg);
    const float* gal = buf0 + s * slot_elems + (size_t)hg * fg.gal_elems;
    for (int c = 0; c < a.md.n_comp; ++c) {
      float sm[kNSum];
#pragma unroll
      for (int k = 0; k < kNSum; ++k) sm[k] = 0.0f;
      if (b >= 0) {
        const CompConst cc = a.cc[(size_t)b * a.md.n_comp + c];
        const float* Gb = a.G + (size_t)b * fg.H * fg.W;
        const bool conv = a.md.conv[c] != 0, box = a.md.box[c] != 0;
        dispatch_kind(a.md.kind[c], [&]<int KIND>() {
          if (box) {                                       // Eq. 2 with B != 0: per-pixel geometry
            for (int i = lw; i < fg.H; i += hpg) {
              const float y = (float)fg.H - 0.5f - (float)i;
              for (int j = lane; j < fg.W; j += 32) {
                const float seed = conv ? gal[(size_t)i * fg.pitch + j + h] : Gb[(size_t)i * fg.W + j];
                grad_accumulate<KIND>(cc, true, seed, (float)j + 0.5f, y, sm);
              }
            }
          } else {
            GradAcc<KIND> acc;
            acc.init();
            for (int idx = gstart; idx < ngrp; idx += gstep) {
              const int i = group_row(idx), x = (idx - i * W4) << 2;
              float seed[4];
              if (conv && kAligned && x + 4 <= fg.W) {
                const float4 q = *reinterpret_cast<const float4*>(gal + (size_t)i * fg.pitch + h + x);
                seed[0] = q.x; seed[1] = q.y; seed[2] = q.z; seed[3] = q.w;
              } else {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                  seed[k] = (x + k < fg.W) ? (conv ? gal[(size_t)i * fg.pitch + h + x + k] : Gb[(size_t)i * fg.W + x + k]) : 0.0f;
              }
              grad_add4<KIND>(acc, cc, seed, (float)x + 0.5f, (float)fg.H - 0.5f - (float)i);
            }
            acc.finish(cc, sm);
          }
        });
        if (!box) sm[8] = sm[2];
      }
#pragma unroll
      for (int k = 0; k < kNSum; ++k) {
        const float v = warp_sum(sm[k]);
        if (lane == 0) red[hw * kNSum + k] = v;
      }
      bar_sync(BAR_HELP, HN);
      if (htid < G * kNSum) {
        const int gg = htid / kNSum, k = htid - gg * kNSum;
        const int bb = galaxy(item, gg);
        if (bb >= 0) {
          float t = 0.0f;
          for (int w = 0; w < hpg; ++w) t += red[(gg * hpg + w) * kNSum + k];
          a.grad_part[((size_t)bb * a.md.n_comp + c) * kNSum + k] = t;
        }
      }
      bar_sync(BAR_HELP, HN);
    }
  };

  auto feed = [&](int item, int s) {                    // next item of slot s, if any
    if (item < n_items) { produce(item, s); bar_arrive(BAR_FULL0 + s, kFusedThreads); }
  };
  bar_sync(BAR_HELP, HN);                               // zero rows and shared taps are in place
  feed(0, 0);
  feed(1, 1);
  for (int m = 0; 2 * m < n_items; ++m) {
    for (int s = 0; s < 2; ++s) {                       // after C1: residual
      const int item = 2 * m + s;
      if (item >= n_items) continue;
      bar_sync(BAR_DONE0 + s, kFusedThreads);
      residual(item, s);
      if (with_grad) bar_arrive(BAR_FULL0 + s, kFusedThreads);   // G in place: adjoint may start
      else feed(item + 2, s);
    }
    if (with_grad) {
      for (int s = 0; s < 2; ++s) {                     // after C2: gradient, then the next item
        const int item = 2 * m + s;
        if (item >= n_items) continue;
        bar_sync(BAR_DONE0 + s, kFusedThreads);
        gradient(item, s);
        feed(item + 2, s);
      }
    }
  }
}

}  // namespace gm
