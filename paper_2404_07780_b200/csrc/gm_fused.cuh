// gm_fused.cuh -- the fused loss + gradient kernel for cutouts that fit one CTA tile
// (H, W <= 128): steps a1..a5 of SURVEY.md section 8(a) in ONE launch, with nothing but
// chi^2 and the kNSum partial sums per component leaving the SM.
//
// One persistent CTA per SM, 512 threads, two roles that run concurrently:
//
//   conv warps   (0..7)   only the FFMA2 convolution loop (conv8x8): forward
//                         M = PSF (*) S, then adjoint A = PSF (star) G, in place in a
//                         shared-memory buffer that holds one whole cutout + zero halo
//   helper warps (8..15)  everything else: a1 render S into a buffer, a3 residual
//                         (M -> G in place, chi^2), a5 gradient sums from A
//
// Two buffers hold two galaxies (a, b) in flight; the conv warps run
// C1(a) C1(b) C2(a) C2(b) back to back while the helpers prepare the other buffer:
//
//   conv   : C1(a)   | C1(b)   | C2(a)   | C2(b)          | C1(c) ...
//   helper : P1(b)   | E1(a)   | E1(b)   | E2(a) P1(c)    | E2(b) P1(d) ...
//
// so the FP32 pipe never waits for the SFU/ALU work of render, residual and gradient
// (that work fills the issue slots FFMA2 leaves free).  Hand-off is by named barriers
// (bar.arrive / bar.sync): full[s] helper -> conv, done[s] conv -> helper.
#pragma once
#include "gm_kernels.cuh"

namespace gm {

constexpr int kConvWarps = 8, kHelpWarps = 8;
constexpr int kFusedThreads = 32 * (kConvWarps + kHelpWarps);

struct FusedArgs {
  ModelDesc md;
  TileGeom tg;               // tiles_x = tiles_y = 1, TH x TW covers the cutout
  int B;
  int mode;                  // 0 render (write M), 1 chi^2 only, 2 chi^2 + gradient
  int any_unconv;            // model has unconvolved components (G also goes to global)
  const CompConst* cc;
  const float2* taps_fwd; const float2* taps_adj; long long taps_stride;
  const float* data; const float* sigma; const uint8_t* mask;
  float* G;                  // [B,H,W]: model_out (mode 0) or back-seed spill (any_unconv)
  float* chi2_part;          // [B]      (tiles = 1)
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
__host__ __device__ inline size_t fused_smem_bytes(const TileGeom& tg) {
  return 2 * (size_t)tg.rows * tg.pitch * 4 + 4 * (size_t)(K + 1) * ConvCfg<K>::kTapPitch * 8 +
         (size_t)kHelpWarps * kNSum * 4 + 64;
}

// acc -> interior of the buffer (row + h, col + h); 128-bit stores when h % 4 == 0.
// Outputs of the 8x8 block that fall outside the H x W cutout (ragged tile) are stored
// as zero: the buffer is the input of the adjoint convolution next, whose zero fill
// (R:C2) starts at the cutout edge, not at the tile edge.
template <int K>
__device__ __forceinline__ void store_acc_interior(float* buf, int pitch, int ty, int tx, int H, int W,
                                                   const float2 (&acc)[4][kTC]) {
  constexpr int h = (K - 1) / 2;
  const int r0 = ty * kTR, c0 = tx * kTC;
  float* dst = buf + (size_t)(r0 + h) * pitch + c0 + h;
  if ((h & 3) == 0 && r0 + kTR <= H && c0 + kTC <= W) {
    store_acc(dst, pitch, acc);
  } else {
#pragma unroll
    for (int rp = 0; rp < 4; ++rp)
#pragma unroll
      for (int c = 0; c < kTC; ++c) {
        const bool cin = c0 + c < W;
        dst[(size_t)(2 * rp) * pitch + c] = (cin && r0 + 2 * rp < H) ? acc[rp][c].x : 0.0f;
        dst[(size_t)(2 * rp + 1) * pitch + c] = (cin && r0 + 2 * rp + 1 < H) ? acc[rp][c].y : 0.0f;
      }
  }
}

template <int K>
__global__ void __launch_bounds__(kFusedThreads, 1) k_fused(const FusedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileGeom& tg = a.tg;
  constexpr int h = (K - 1) / 2;
  constexpr int TAPN = (K + 1) * ConvCfg<K>::kTapPitch;          // float2 per tap set
  const size_t buf_elems = (size_t)tg.rows * tg.pitch;
  float* buf0 = reinterpret_cast<float*>(smem_raw);
  float2* taps0 = reinterpret_cast<float2*>(buf0 + 2 * buf_elems);   // [buffer][fwd|adj][TAPN]
  float* red = reinterpret_cast<float*>(taps0 + 4 * TAPN);

  const int tid = threadIdx.x;
  const int wid = tid >> 5, lane = tid & 31;
  const bool with_grad = a.mode == 2;
  const int n_gal = a.live ? *a.n_live : a.B;
  const int n_k = (n_gal - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // galaxies of this CTA
  auto galaxy = [&](int k) {
    const int i = (int)blockIdx.x + k * (int)gridDim.x;
    return a.live ? a.live[i] : i;
  };
  auto live = [&](int k) { return k < n_k && !(a.frozen && a.frozen[galaxy(k)]); };

  if (wid < kConvWarps) {
    // ------------------------------ conv warps ------------------------------------
    const int ty = tid / tg.ntx, tx = tid - ty * tg.ntx;
    const bool active = ty < tg.nty;
    for (int m = 0; 2 * m < n_k; ++m) {
      for (int phase = 0; phase < (with_grad ? 2 : 1); ++phase) {
        for (int s = 0; s < 2; ++s) {
          if (!live(2 * m + s)) continue;
          float* buf = buf0 + s * buf_elems;
          const float2* taps = taps0 + (2 * s + phase) * TAPN;
          bar_sync(BAR_FULL0 + s, kFusedThreads);               // input tile (S or G) is ready
          float2 acc[4][kTC];
#pragma unroll
          for (int rp = 0; rp < 4; ++rp)
#pragma unroll
            for (int c = 0; c < kTC; ++c) acc[rp][c] = make_float2(0.0f, 0.0f);
          if (active) conv8x8<K>(buf + (size_t)(ty * kTR) * tg.pitch + tx * kTC, tg.pitch, taps, acc);
          bar_sync(BAR_CONV, 32 * kConvWarps);                  // every conv thread is done reading
          if (active) store_acc_interior<K>(buf, tg.pitch, ty, tx, tg.H, tg.W, acc);
          bar_arrive(BAR_DONE0 + s, kFusedThreads);             // M (or A) is parked in the buffer
        }
      }
    }
    return;
  }

  // -------------------------------- helper warps ------------------------------------
  const int hw = wid - kConvWarps;                 // 0..7
  const int htid = tid - 32 * kConvWarps;          // 0..255
  constexpr int HN = 32 * kHelpWarps;
  const int cols = tg.TW + K - 1;

  // a1: taps of galaxy g and S on the whole buffer (zero halo, zero pad)
  auto produce = [&](int g, int s) {
    float* buf = buf0 + s * buf_elems;
    float2* tp = taps0 + 2 * s * TAPN;
    const float2* src = a.taps_fwd + (long long)g * a.taps_stride;
    const float2* srca = a.taps_adj + (long long)g * a.taps_stride;
    for (int i = htid; i < TAPN / 2; i += HN) {
      cp_async_zfill16(reinterpret_cast<float*>(tp) + 4 * i, reinterpret_cast<const float*>(src) + 4 * i, true);
      cp_async_zfill16(reinterpret_cast<float*>(tp + TAPN) + 4 * i, reinterpret_cast<const float*>(srca) + 4 * i, true);
    }
    const CompConst* ccb = a.cc + (size_t)g * a.md.n_comp;
    bool first = true;
    for (int c = 0; c <= a.md.n_comp; ++c) {
      const bool zero_pass = (c == a.md.n_comp);
      if (zero_pass && !first) break;
      if (!zero_pass && !a.md.conv[c]) continue;
      const CompConst cc = ccb[zero_pass ? 0 : c];
      const bool box = !zero_pass && a.md.box[c] != 0;
      dispatch_kind(zero_pass ? (int)GM_SKY : a.md.kind[c], [&]<int KIND>() {
        for (int yy = hw; yy < tg.rows; yy += kHelpWarps) {
          const int i = yy - h;
          float* rowp = buf + (size_t)yy * tg.pitch;
          const bool row_in = (i >= 0 && i < tg.H);
          const float y = (float)tg.H - 0.5f - (float)i;        // R:G1
          for (int xx = lane; xx < tg.pitch; xx += 32) {
            const int j = xx - h;
            const bool in = row_in && xx < cols && j >= 0 && j < tg.W;
            float sv = 0.0f;
            if (KIND != GM_SKY && in)
              sv = cc.amp * profile_value_t<KIND, kFastForward>(cc, geometry<kFastForward>(cc, box, (float)j + 0.5f, y).r);
            if (first) rowp[xx] = sv;
            else if (in) rowp[xx] += sv;
          }
        }
      });
      first = false;
    }
    cp_async_wait_all();
  };

  // a3: M (buffer interior) -> chi^2 and G in place; mode 0 writes M out instead
  auto residual = [&](int g, int s) {
    float* buf = buf0 + s * buf_elems;
    const CompConst* ccb = a.cc + (size_t)g * a.md.n_comp;
    const size_t img = (size_t)g * tg.H * tg.W;
    float chi2 = 0.0f;
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
    auto one = [&](float m, float d, float sg, bool used, float& gv) {
      gv = 0.0f;
      if (used) {                                       // select, never multiply by 0 (R:X1)
        const float w = __fdividef(1.0f, sg * sg);
        const float rho = d - m;
        chi2 = fmaf(w * rho, rho, chi2);
        gv = -2.0f * w * rho;
      }
    };
    if (tg.vec && (h & 3) == 0) {
      // 128-bit path: one lane = 4 pixels, two rows per warp in flight
      for (int yy = hw; yy < tg.H; yy += 2 * kHelpWarps) {
        float4 m4[2], d4[2], s4[2];
        uchar4 k4[2];
        bool ok[2];
        size_t off[2];
        float* mp[2];
        const int xx = lane * 4;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int i = yy + u * kHelpWarps;
          ok[u] = (i < tg.H) && (xx < tg.W);
          off[u] = img + (size_t)i * tg.W + xx;
          mp[u] = buf + (size_t)(i + h) * tg.pitch + xx + h;
          if (ok[u]) {
            m4[u] = *reinterpret_cast<const float4*>(mp[u]);
            if (a.mode != 0) {
              d4[u] = *reinterpret_cast<const float4*>(a.data + off[u]);
              s4[u] = *reinterpret_cast<const float4*>(a.sigma + off[u]);
              k4[u] = a.mask ? *reinterpret_cast<const uchar4*>(a.mask + off[u]) : make_uchar4(1, 1, 1, 1);
            }
          }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          if (!ok[u]) continue;
          if (a.any_unconv) {
            const float y = (float)tg.H - 0.5f - (float)(yy + u * kHelpWarps);
            const float x = (float)xx + 0.5f;
            m4[u].x = add_unconv(m4[u].x, x, y);
            m4[u].y = add_unconv(m4[u].y, x + 1.0f, y);
            m4[u].z = add_unconv(m4[u].z, x + 2.0f, y);
            m4[u].w = add_unconv(m4[u].w, x + 3.0f, y);
          }
          if (a.mode == 0) {
            *reinterpret_cast<float4*>(a.G + off[u]) = m4[u];
          } else {
            float4 gv;
            one(m4[u].x, d4[u].x, s4[u].x, k4[u].x != 0, gv.x);
            one(m4[u].y, d4[u].y, s4[u].y, k4[u].y != 0, gv.y);
            one(m4[u].z, d4[u].z, s4[u].z, k4[u].z != 0, gv.z);
            one(m4[u].w, d4[u].w, s4[u].w, k4[u].w != 0, gv.w);
            *reinterpret_cast<float4*>(mp[u]) = gv;
            if (a.any_unconv && with_grad) *reinterpret_cast<float4*>(a.G + off[u]) = gv;
          }
        }
      }
    } else {
      for (int i = hw; i < tg.H; i += kHelpWarps) {
        const float y = (float)tg.H - 0.5f - (float)i;
        for (int j = lane; j < tg.W; j += 32) {
          float* mp = buf + (size_t)(i + h) * tg.pitch + j + h;
          float m = *mp;
          if (a.any_unconv) m = add_unconv(m, (float)j + 0.5f, y);
          const size_t o = img + (size_t)i * tg.W + j;
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
    if (a.mode != 0) {
      chi2 = warp_sum(chi2);
      if (lane == 0) red[hw] = chi2;
      bar_sync(BAR_HELP, HN);
      if (htid == 0) {
        float t = 0.0f;
        for (int w = 0; w < kHelpWarps; ++w) t += red[w];
        a.chi2_part[g] = t;
      }
      bar_sync(BAR_HELP, HN);
    }
  };

  // a5: the partial sums of every component from A (buffer interior)
  auto gradient = [&](int g, int s) {
    const float* buf = buf0 + s * buf_elems;
    const CompConst* ccb = a.cc + (size_t)g * a.md.n_comp;
    const float* Gb = a.G + (size_t)g * tg.H * tg.W;
    float* outp = a.grad_part + (size_t)g * a.md.n_comp * kNSum;
    for (int c = 0; c < a.md.n_comp; ++c) {
      float sm[kNSum];
#pragma unroll
      for (int k = 0; k < kNSum; ++k) sm[k] = 0.0f;
      const CompConst cc = ccb[c];
      const bool conv = a.md.conv[c] != 0, box = a.md.box[c] != 0;
      dispatch_kind(a.md.kind[c], [&]<int KIND>() {
        for (int i = hw; i < tg.H; i += kHelpWarps) {
          const float y = (float)tg.H - 0.5f - (float)i;
          for (int j = lane; j < tg.W; j += 32) {
            const float seed = conv ? buf[(size_t)(i + h) * tg.pitch + j + h] : Gb[(size_t)i * tg.W + j];
            grad_accumulate<KIND>(cc, box, seed, (float)j + 0.5f, y, sm);
          }
        }
      });
      if (!box) sm[8] = sm[2];
#pragma unroll
      for (int k = 0; k < kNSum; ++k) {
        const float v = warp_sum(sm[k]);
        if (lane == 0) red[hw * kNSum + k] = v;
      }
      bar_sync(BAR_HELP, HN);
      if (htid < kNSum) {
        float t = 0.0f;
        for (int w = 0; w < kHelpWarps; ++w) t += red[w * kNSum + htid];
        outp[c * kNSum + htid] = t;
      }
      bar_sync(BAR_HELP, HN);
    }
  };

  auto feed = [&](int k, int s) {                       // next galaxy of buffer s, if any
    if (live(k)) { produce(galaxy(k), s); bar_arrive(BAR_FULL0 + s, kFusedThreads); }
  };
  feed(0, 0);
  feed(1, 1);
  for (int m = 0; 2 * m < n_k; ++m) {
    for (int s = 0; s < 2; ++s) {                       // after C1: residual
      const int k = 2 * m + s;
      if (live(k)) {
        bar_sync(BAR_DONE0 + s, kFusedThreads);
        residual(galaxy(k), s);
        if (with_grad) { bar_arrive(BAR_FULL0 + s, kFusedThreads); continue; }   // G in place: adjoint may start
      }
      if (!with_grad || !live(k)) feed(k + 2, s);
    }
    if (with_grad) {
      for (int s = 0; s < 2; ++s) {                     // after C2: gradient, then the next galaxy
        const int k = 2 * m + s;
        if (!live(k)) continue;                         // its successor was fed above
        bar_sync(BAR_DONE0 + s, kFusedThreads);
        gradient(galaxy(k), s);
        feed(k + 2, s);
      }
    }
  }
}

}  // namespace gm
