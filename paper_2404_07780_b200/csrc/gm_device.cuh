// gm_device.cuh -- device-side arithmetic of the forward model (steps a0, a1, a5
// of SURVEY.md section 8(a)): per-galaxy prologue constants in fp64, the radial
// laws of the paper (Eq. 1, 7, 9, 11, 12, 13, 16) and their derivatives in fp32.
//
// Written from the paper (PAPER.md "P:<line>") and DESIGN.md's readings; shares
// nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/gm.h"

namespace gm {

constexpr float kRGuard = 1e-6f;               // R:S4
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// model descriptor passed by value to kernels
struct ModelDesc {
  int32_t n_comp, n_par;
  int32_t kind[GM_MAX_COMP];
  int32_t conv[GM_MAX_COMP];                   // 1: through the PSF
  int8_t slot[GM_MAX_COMP][GM_NSLOT];          // -1 unused
  int8_t box[GM_MAX_COMP];                     // 1: boxiness slot used (Eq. 2 with B != 0)
  int8_t mag[GM_MAX_COMP];                     // 1: amplitude slot holds a magnitude (Eq. 5/8/10/15)
};

// per (galaxy, component) constants produced by the prologue (step a0), 96 bytes
struct __align__(16) CompConst {
  float xc, yc, ct, st;      // centre, cos/sin(theta)
  float iq, q, amp, a0;      // 1/q, q, amplitude (intensity), kind specific ...
  float a1, a2, a3, a4;
  float a5, a6, a7, a8;
  float c, ic, cm1, dl_box;  // Eq. 2 exponent c = B + 2, 1/c, c - 1; d ln(amp) / dB
  float dl_m, dl_q, dl_s0, dl_s1;   // magnitude mode: d ln(amp) / d (m, q, s0, s1, s2);
  float dl_s2, b0, b1, b2;          //   d/d m0 = -dl_m; b0, b1: Sersic 1/re^2 and 1/(2n) for the
                                    //   sqrt-free forms of value_uv / GradAcc
};

// ---------------------------------------------------------------------------
// step a1: elliptical radius, Eq. 2-4 (R:G2): rotate, then scale v by 1/q;
// r = sqrt(u^2 + (v/q)^2) for B = 0, else r = (|u|^c + |v/q|^c)^(1/c), c = B + 2
// ---------------------------------------------------------------------------
struct Geo { float u, vq, r; };

// SFU forms.  FAST = MUFU.LG2 / MUFU.EX2 approximations (absolute error 2^-22 in the logarithm,
// 2 ulp in the exponential): used by the gradient pass and, with kFastForward (the default,
// gm_kernels.cuh), by every pass that produces a pixel of M as well -- gm_render included.
// Accuracy contract of a rendered, UNCONVOLVED pixel: relative error below 2e-5 wherever the profile
// has not underflowed (nu t < 30; worst measured 1.3e-5 at that edge for n = 0.5, where the fp32
// rounding of the exponent adds to the lg2 term), derived in DESIGN.md section 6 and checked by
// tests/test_gpu_parity.py::test_render_accuracy_high_n_wings.  (After the tensor-core convolution the
// error is absolute, relative to the cutout's maximum: include/gm.h, GM_OPT_TENSOR.)  !FAST = log2f / exp2f of the CUDA math library
// (<= 2 ulp), selected for all pixel values by -DGM_PRECISE_FORWARD.
template <bool FAST> __device__ __forceinline__ float lg2(float x) {
  if (FAST) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  return log2f(x);
}
template <bool FAST> __device__ __forceinline__ float ex2(float x) {
  if (FAST) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  return exp2f(x);
}

template <bool FAST>
__device__ __forceinline__ Geo geometry(const CompConst& cc, bool box, float x, float y) {
  const float dx = x - cc.xc, dy = y - cc.yc;
  Geo g;
  g.u = fmaf(cc.ct, dx, cc.st * dy);
  g.vq = fmaf(cc.ct, dy, -cc.st * dx) * cc.iq;
  if (box) {                                   // warp-uniform: a property of the component
    const float uc = ex2<FAST>(cc.c * lg2<FAST>(fabsf(g.u)));      // 0 at u = 0 (c > 0)
    const float vc = ex2<FAST>(cc.c * lg2<FAST>(fabsf(g.vq)));
    g.r = ex2<FAST>(cc.ic * lg2<FAST>(uc + vc));
  } else {
    const float r2 = fmaf(g.u, g.u, g.vq * g.vq);
    if (FAST) asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(g.r) : "f"(r2));   // MUFU.SQRT, <= 1 ulp
    else g.r = sqrtf(r2);
  }
  return g;
}

// d r / d u, d r / d (v/q) and d r / d B at rg = max(r, 1e-6) (R:S4), Eq. 2:
//   dr/du = sgn(u) |u|^(c-1) / rg^(c-1)                      (u / rg when B = 0)
//   dr/dB = (rg / c) [(|u|^c ln|u| + |v/q|^c ln|v/q|) / (|u|^c + |v/q|^c) - ln rg]
struct GeoGrad { float gu, gv, db; };
template <bool FAST>
__device__ __forceinline__ GeoGrad geometry_grad(const CompConst& cc, bool box, const Geo& g, float rg) {
  GeoGrad d;
  if (box) {
    const float au = fabsf(g.u), av = fabsf(g.vq);
    const float lu = lg2<FAST>(au), lv = lg2<FAST>(av), lr = lg2<FAST>(rg);
    const float uc = ex2<FAST>(cc.c * lu), vc = ex2<FAST>(cc.c * lv);
    d.gu = au > 0.0f ? copysignf(ex2<FAST>(cc.cm1 * (lu - lr)), g.u) : 0.0f;
    d.gv = av > 0.0f ? copysignf(ex2<FAST>(cc.cm1 * (lv - lr)), g.vq) : 0.0f;
    const float tu = au > 0.0f ? uc * lu : 0.0f, tv = av > 0.0f ? vc * lv : 0.0f;
    const float sum = uc + vc;
    d.db = sum > 0.0f ? rg * cc.ic * kLn2 * (__fdividef(tu + tv, sum) - lr) : 0.0f;
  } else {
    const float ir = __fdividef(1.0f, rg);
    d.gu = g.u * ir; d.gv = g.vq * ir; d.db = 0.0f;
  }
  return d;
}

// radial law with unit amplitude at radius r (value only); KIND is a gm_kind
template <int KIND, bool FAST>
__device__ __forceinline__ float profile_value_t(const CompConst& cc, float r) {
  if (KIND == GM_SERSIC) {
    const float t = ex2<FAST>(lg2<FAST>(r * cc.a0) * cc.a1);       // (r/re)^(1/n); 0 at r = 0
    return ex2<FAST>(-cc.a2 * (t - 1.0f));
  } else if (KIND == GM_EXPDISK) {
    return ex2<FAST>(-r * cc.a0);
  } else if (KIND == GM_GAUSSIAN) {
    return ex2<FAST>(-r * r * cc.a0);
  } else if (KIND == GM_MOFFAT) {
    return ex2<FAST>(-cc.a1 * lg2<FAST>(fmaf(r * r, cc.a0, 1.0f)));
  } else if (KIND == GM_FERRER) {
    if (!(r < cc.a3)) return 0.0f;
    const float w = ex2<FAST>(cc.a2 * lg2<FAST>(r * cc.a0));
    return ex2<FAST>(cc.a1 * lg2<FAST>(1.0f - w));
  } else if (KIND == GM_KING) {
    if (!(r < cc.a8)) return 0.0f;
    const float ra = r * cc.a0;
    const float R = ex2<FAST>(cc.a1 * lg2<FAST>(fmaf(ra, ra, 1.0f)));
    const float X = (R - cc.a2) * cc.a3;
    return X > 0.0f ? ex2<FAST>(cc.a4 * lg2<FAST>(X)) : 0.0f;
  }
  return 1.0f;                                                     // sky
}

// run f.template operator()<KIND>() for the runtime kind (warp-uniform branch)
template <typename F>
__device__ __forceinline__ void dispatch_kind(int kind, F&& f) {
  switch (kind) {
    case GM_SERSIC: f.template operator()<GM_SERSIC>(); break;
    case GM_EXPDISK: f.template operator()<GM_EXPDISK>(); break;
    case GM_FERRER: f.template operator()<GM_FERRER>(); break;
    case GM_KING: f.template operator()<GM_KING>(); break;
    case GM_GAUSSIAN: f.template operator()<GM_GAUSSIAN>(); break;
    case GM_MOFFAT: f.template operator()<GM_MOFFAT>(); break;
    default: f.template operator()<GM_SKY>(); break;
  }
}

__device__ __forceinline__ float profile_value(int kind, const CompConst& cc, float r) {
  float v = 1.0f;
  dispatch_kind(kind, [&]<int KIND>() { v = profile_value_t<KIND, false>(cc, r); });
  return v;
}

// radial law and its derivatives, evaluated at rg (the caller passes rg = max(r, 1e-6))
// U value, dUdr, d0..d2 = d/d(s0, s1, s2), unit amplitude
template <int KIND, bool FAST>
__device__ __forceinline__ void profile_grad_t(const CompConst& cc, float rg, float& U, float& dUdr,
                                               float& d0, float& d1, float& d2) {
  U = 0.0f; dUdr = 0.0f; d0 = 0.0f; d1 = 0.0f; d2 = 0.0f;
  if (KIND == GM_SERSIC) {
    const float L = lg2<FAST>(rg * cc.a0);
    const float t = ex2<FAST>(L * cc.a1);
    U = ex2<FAST>(-cc.a2 * (t - 1.0f));
    const float k = U * cc.a3 * t * cc.a1;                        // U nu t / n
    dUdr = -__fdividef(k, rg);
    d0 = k * cc.a0;                                               // d/d re
    d1 = U * (-cc.a4 * (t - 1.0f) + cc.a3 * t * (L * kLn2) * cc.a1 * cc.a1);   // d/d n
  } else if (KIND == GM_EXPDISK) {
    U = ex2<FAST>(-rg * cc.a0);
    dUdr = -U * cc.a1;
    d0 = U * rg * cc.a1 * cc.a1;
  } else if (KIND == GM_GAUSSIAN) {
    U = ex2<FAST>(-rg * rg * cc.a0);
    dUdr = -U * rg * cc.a1;
    d0 = U * rg * rg * cc.a2;
  } else if (KIND == GM_MOFFAT) {
    const float A = fmaf(rg * rg, cc.a0, 1.0f);
    const float lA = lg2<FAST>(A);
    U = ex2<FAST>(-cc.a1 * lA);
    const float UA = __fdividef(U, A);
    dUdr = -cc.a2 * UA * rg;
    d0 = cc.a3 * UA * rg * rg;                                    // d/d FWHM
    d1 = -U * (lA * kLn2) + UA * rg * rg * cc.a4;                 // d/d n
  } else if (KIND == GM_FERRER) {
    if (!(rg < cc.a3)) return;
    const float Lr = lg2<FAST>(rg * cc.a0);
    const float w = ex2<FAST>(cc.a2 * Lr);
    const float omw = 1.0f - w;
    if (!(omw > 0.0f)) return;
    const float lo = lg2<FAST>(omw);
    U = ex2<FAST>(cc.a1 * lo);
    const float core = cc.a1 * __fdividef(U, omw);                // a (1-w)^(a-1)
    dUdr = -__fdividef(core * cc.a2 * w, rg);
    d0 = core * cc.a2 * w * cc.a0;                                // d/d r_out
    d1 = U * (lo * kLn2);                                         // d/d a
    d2 = core * w * (Lr * kLn2);                                  // d/d b
  } else if (KIND == GM_KING) {
    if (!(rg < cc.a8)) return;
    const float ra = rg * cc.a0;
    const float z = fmaf(ra, ra, 1.0f);
    const float lz = lg2<FAST>(z);
    const float R = ex2<FAST>(cc.a1 * lz);
    const float X = (R - cc.a2) * cc.a3;
    if (!(X > 0.0f)) return;
    const float lX = lg2<FAST>(X);
    U = ex2<FAST>(cc.a4 * lX);
    const float UR = cc.a4 * __fdividef(U, X) * cc.a3;            // alpha X^(alpha-1) / (1-T)
    const float UT = UR * (R - 1.0f) * cc.a3;
    const float m2a = -2.0f * cc.a1;                              // 2/alpha
    const float Rr = -m2a * __fdividef(R * (rg * cc.a0 * cc.a0), z);
    const float Rrc = m2a * __fdividef(R * (ra * ra * cc.a0), z);
    const float Ral = R * (lz * kLn2) * cc.a1 * cc.a1;
    dUdr = UR * Rr;
    d0 = UR * Rrc + UT * cc.a5;                                   // d/d rc
    d1 = UT * cc.a6;                                              // d/d rt
    d2 = U * (lX * kLn2) + UR * Ral + UT * cc.a7;                 // d/d alpha
  }
}

// d I / d (slot k) of one component at pixel centre (x, y): the forward-mode column of
// the Jacobian J = dM/dp used by the covariance row.  Same guards as the
// gradient pass (R:S4): derivative factors at rg = max(r, 1e-6), d/d amp at r itself.
// mag: the amplitude slot is a magnitude; every slot the amplitude depends on gains
// I * d ln(amp) / d slot (Eq. 5, 8, 10, 15).
template <int KIND>
__device__ __forceinline__ float component_deriv_t(const CompConst& cc, bool box, bool mag, int k, float x, float y) {
  if (KIND == GM_SKY) return k == GM_SLOT_AMP ? 1.0f : 0.0f;
  const Geo g = geometry<false>(cc, box, x, y);
  const float rg = fmaxf(g.r, kRGuard);
  float U, dUdr, d0, d1, d2;
  profile_grad_t<KIND, false>(cc, rg, U, dUdr, d0, d1, d2);
  const GeoGrad d = geometry_grad<false>(cc, box, g, rg);
  const float A = cc.amp * dUdr;
  const float Uv = (g.r < kRGuard) ? profile_value_t<KIND, true>(cc, g.r) : U;
  const float I = cc.amp * Uv;
  switch (k) {
    case GM_SLOT_XC: return A * (-cc.ct * d.gu + cc.st * cc.iq * d.gv);
    case GM_SLOT_YC: return A * (-cc.st * d.gu - cc.ct * cc.iq * d.gv);
    case GM_SLOT_THETA:                        // B = 0: u (v/q) (q - 1/q) / r, exactly 0 at q = 1
      return box ? A * (cc.q * d.gu * g.vq - cc.iq * d.gv * g.u) : A * d.gu * g.vq * (cc.q - cc.iq);
    case GM_SLOT_Q: return -cc.iq * A * d.gv * g.vq + (mag ? I * cc.dl_q : 0.0f);
    case GM_SLOT_AMP: return mag ? I * cc.dl_m : Uv;
    case GM_SLOT_S0: return cc.amp * d0 + (mag ? I * cc.dl_s0 : 0.0f);
    case GM_SLOT_S1: return cc.amp * d1 + (mag ? I * cc.dl_s1 : 0.0f);
    case GM_SLOT_S2: return cc.amp * d2 + (mag ? I * cc.dl_s2 : 0.0f);
    case GM_SLOT_BOX: return A * d.db + (mag ? I * cc.dl_box : 0.0f);
    case GM_SLOT_M0: return mag ? -I * cc.dl_m : 0.0f;
    default: return 0.0f;
  }
}

__device__ __forceinline__ float component_deriv(int kind, const CompConst& cc, bool box, bool mag, int k,
                                                 float x, float y) {
  float v = 0.0f;
  dispatch_kind(kind, [&]<int KIND>() { v = component_deriv_t<KIND>(cc, box, mag, k, x, y); });
  return v;
}

// ---------------------------------------------------------------------------
// step a5: one pixel's contribution to the partial sums of a component.  With
// seed = A (convolved) or G (unconvolved), X = seed * amp * dU/dr:
//   s0 = sum X dr/du        s1 = sum X dr/d(v/q)     s2 = sum X dr/du (v/q)
//   s3 = sum X dr/d(v/q) (v/q)                       s4 = sum seed U
//   s5..s7 = sum seed amp dU/d(s0, s1, s2)
//   s8 = sum X dr/d(v/q) u  (= s2 when B = 0)        s9 = sum X dr/dB
// from which (assemble, gm_api.cu)
//   d/dxc = -ct s0 + st s1 / q      d/dyc = -st s0 - ct s1 / q
//   d/dtheta = q s2 - s8 / q        d/dq = -s3 / q        d/dB = s9
// ---------------------------------------------------------------------------
constexpr int kNSum = 10;

template <int KIND>
__device__ __forceinline__ void grad_accumulate(const CompConst& cc, bool box, float seed, float x, float y,
                                                float (&s)[kNSum]) {
  if (KIND == GM_SKY) { s[4] += seed; return; }
  const Geo g = geometry<true>(cc, box, x, y);
  const float rg = fmaxf(g.r, kRGuard);
  float U, dUdr, d0, d1, d2;
  profile_grad_t<KIND, true>(cc, rg, U, dUdr, d0, d1, d2);
  // d/d amp uses the value at r itself (differs from rg only below 1e-6 px)
  const float Uv = (g.r < kRGuard) ? profile_value_t<KIND, true>(cc, g.r) : U;
  const float sa = seed * cc.amp;
  if (box) {
    const GeoGrad d = geometry_grad<true>(cc, true, g, rg);
    const float X = sa * dUdr;
    s[0] = fmaf(X, d.gu, s[0]);
    s[1] = fmaf(X, d.gv, s[1]);
    s[2] = fmaf(X * d.gu, g.vq, s[2]);
    s[3] = fmaf(X * d.gv, g.vq, s[3]);
    s[8] = fmaf(X * d.gv, g.u, s[8]);
    s[9] = fmaf(X, d.db, s[9]);
  } else {
    const float cgeo = __fdividef(sa * dUdr, rg);
    s[0] = fmaf(cgeo, g.u, s[0]);
    s[1] = fmaf(cgeo, g.vq, s[1]);
    s[2] = fmaf(cgeo * g.u, g.vq, s[2]);
    s[3] = fmaf(cgeo * g.vq, g.vq, s[3]);
  }
  s[4] = fmaf(seed, Uv, s[4]);
  s[5] = fmaf(sa, d0, s[5]);
  s[6] = fmaf(sa, d1, s[6]);
  s[7] = fmaf(sa, d2, s[7]);
}


// ---------------------------------------------------------------------------
// Row forms of a1 and a5 (B = 0).  Every instruction of the helper warps costs an issue
// cycle that the FFMA2 convolution loop wants (FFMA2 holds the issue port for both of
// its cycles: DESIGN.md section 5), so the per-pixel arithmetic is kept minimal:
//   * u and v/q are linear in the column: four consecutive pixels of a row share one
//     evaluation of the rotation (row4),
//   * laws that are functions of r^2 skip the square root (Sersic: (r/re)^(1/n) =
//     2^(lg2(r^2/re^2) / 2n)),
//   * the gradient sums of the Sersic and exponential laws accumulate seed-weighted
//     monomials and apply the per-galaxy constant factors once per thread (GradAcc).
// ---------------------------------------------------------------------------
__device__ __forceinline__ float rcp_fast(float x) {
  float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}
__device__ __forceinline__ float rsqrt_fast(float x) {
  float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}
__device__ __forceinline__ float sqrt_fast(float x) {
  float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}

// rotated coordinates (u, v/q) of the pixels (x0 + k, y), k = 0..3 (x0, y: pixel centres)
__device__ __forceinline__ void row4(const CompConst& cc, float x0, float y, float (&u)[4], float (&vq)[4]) {
  const float dx = x0 - cc.xc, dy = y - cc.yc;
  const float u0 = fmaf(cc.ct, dx, cc.st * dy);
  const float v0 = fmaf(cc.ct, dy, -cc.st * dx) * cc.iq;
  const float dv = -cc.st * cc.iq;
  u[0] = u0; vq[0] = v0;
#pragma unroll
  for (int k = 1; k < 4; ++k) { u[k] = fmaf((float)k, cc.ct, u0); vq[k] = fmaf((float)k, dv, v0); }
}

// radial law with unit amplitude from (u, v/q), B = 0
template <int KIND, bool FAST>
__device__ __forceinline__ float value_uv(const CompConst& cc, float u, float vq) {
  const float r2 = fmaf(u, u, vq * vq);
  if (KIND == GM_SERSIC) {
    const float t = ex2<FAST>(lg2<FAST>(r2 * cc.b0) * cc.b1);      // (r/re)^(1/n); 0 at r = 0
    return ex2<FAST>(fmaf(-cc.a2, t, cc.a2));
  } else if (KIND == GM_GAUSSIAN) {
    return ex2<FAST>(-r2 * cc.a0);
  } else if (KIND == GM_MOFFAT) {
    return ex2<FAST>(-cc.a1 * lg2<FAST>(fmaf(r2, cc.a0, 1.0f)));
  } else if (KIND == GM_SKY) {
    return 1.0f;
  }
  return profile_value_t<KIND, FAST>(cc, FAST ? sqrt_fast(r2) : sqrtf(r2));
}

// amp * U at the four pixels (x0 + k, y); box: Eq. 2 with B != 0 (per-pixel geometry)
template <int KIND, bool FAST>
__device__ __forceinline__ void value4(const CompConst& cc, bool box, float x0, float y, float (&v)[4]) {
  if (box) {
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = cc.amp * profile_value_t<KIND, FAST>(cc, geometry<FAST>(cc, true, x0 + (float)k, y).r);
  } else {
    float u[4], vq[4];
    row4(cc, x0, y, u, vq);
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = cc.amp * value_uv<KIND, FAST>(cc, u[k], vq[k]);
  }
}

// a5 accumulators of one component, B = 0.  add() takes one pixel (seed, u, v/q);
// finish() returns the kNSum sums defined above grad_accumulate.
template <int KIND> struct GradAcc {                       // generic: the sums themselves
  float s[kNSum];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int k = 0; k < kNSum; ++k) s[k] = 0.0f;
  }
  __device__ __forceinline__ void add(const CompConst& cc, float seed, float u, float vq) {
    if (KIND == GM_SKY) { s[4] += seed; return; }
    const float r = sqrt_fast(fmaf(u, u, vq * vq));
    const float rg = fmaxf(r, kRGuard);
    float U, dUdr, d0, d1, d2;
    profile_grad_t<KIND, true>(cc, rg, U, dUdr, d0, d1, d2);
    const float Uv = (r < kRGuard) ? profile_value_t<KIND, true>(cc, r) : U;
    const float sa = seed * cc.amp;
    const float cgeo = sa * dUdr * rcp_fast(rg);
    s[0] = fmaf(cgeo, u, s[0]);
    s[1] = fmaf(cgeo, vq, s[1]);
    s[2] = fmaf(cgeo * u, vq, s[2]);
    s[3] = fmaf(cgeo * vq, vq, s[3]);
    s[4] = fmaf(seed, Uv, s[4]);
    s[5] = fmaf(sa, d0, s[5]);
    s[6] = fmaf(sa, d1, s[6]);
    s[7] = fmaf(sa, d2, s[7]);
  }
  __device__ __forceinline__ void fix(const CompConst&, float, float) {}   // add() already did
  __device__ __forceinline__ void finish(const CompConst&, float (&out)[kNSum]) const {
#pragma unroll
    for (int k = 0; k < kNSum; ++k) out[k] = s[k];
    out[8] = s[2];
  }
};

constexpr float kRGuard2 = 1e-12f;                         // kRGuard^2

// Sersic (Eq. 1): with L2 = lg2(rg^2 / re^2), t = 2^(L2 / 2n), U = 2^(nu lg2e (1 - t)):
//   dU/dr = -U nu t / (n rg)         dU/dre = U nu t / (n re)
//   dU/dn = -nu' U (t - 1) + (nu ln2 / 2 n^2) U t L2
// so with sU = seed U and W = sU t the sums are multiples of
//   q0..q3 = sum (W / rg^2) (u, v/q, u v/q, (v/q)^2),  q4 = sum sU,  q5 = sum W,
//   q6 = sum sU (t - 1),  q7 = sum W L2
template <> struct GradAcc<GM_SERSIC> {
  float q[8];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int k = 0; k < 8; ++k) q[k] = 0.0f;
  }
  __device__ __forceinline__ void add(const CompConst& cc, float seed, float u, float vq) {
    const float r2 = fmaf(u, u, vq * vq);
    const float r2g = fmaxf(r2, kRGuard2);
    const float L2 = lg2<true>(r2g * cc.b0);
    const float t = ex2<true>(L2 * cc.b1);
    const float U = ex2<true>(fmaf(-cc.a2, t, cc.a2));
    const float sU = seed * U, W = sU * t;
    const float cg = W * rcp_fast(r2g);
    q[0] = fmaf(cg, u, q[0]);
    q[1] = fmaf(cg, vq, q[1]);
    q[2] = fmaf(cg * u, vq, q[2]);
    q[3] = fmaf(cg * vq, vq, q[3]);
    q[4] += sU;
    q[5] += W;
    q[6] = fmaf(sU, t - 1.0f, q[6]);
    q[7] = fmaf(W, L2, q[7]);
  }
  // R:S4: d/d amp takes the value at r itself; called only for a pixel with r^2 < kRGuard2
  __device__ __forceinline__ void fix(const CompConst& cc, float seed, float r2) {
    const float Ug = ex2<true>(fmaf(-cc.a2, ex2<true>(lg2<true>(kRGuard2 * cc.b0) * cc.b1), cc.a2));
    q[4] += seed * (profile_value_t<GM_SERSIC, true>(cc, sqrt_fast(r2)) - Ug);
  }
  __device__ __forceinline__ void finish(const CompConst& cc, float (&out)[kNSum]) const {
    const float kf = cc.amp * cc.a3 * cc.a1;               // amp nu / n
    out[0] = -kf * q[0]; out[1] = -kf * q[1]; out[2] = -kf * q[2]; out[3] = -kf * q[3];
    out[4] = q[4];
    out[5] = kf * cc.a0 * q[5];
    out[6] = cc.amp * (-cc.a4 * q[6] + cc.a3 * cc.a1 * cc.a1 * (0.5f * kLn2) * q[7]);
    out[7] = 0.0f; out[8] = out[2]; out[9] = 0.0f;
  }
};

// exponential disk (Eq. 7): U = exp(-rg / rs), dU/dr = -U / rs, dU/drs = U rg / rs^2
template <> struct GradAcc<GM_EXPDISK> {
  float q[6];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int k = 0; k < 6; ++k) q[k] = 0.0f;
  }
  __device__ __forceinline__ void add(const CompConst& cc, float seed, float u, float vq) {
    const float r2 = fmaf(u, u, vq * vq);
    const float r2g = fmaxf(r2, kRGuard2);
    const float ir = rsqrt_fast(r2g), rg = r2g * ir;
    const float U = ex2<true>(-rg * cc.a0);
    const float sU = seed * U, cg = sU * ir;
    q[0] = fmaf(cg, u, q[0]);
    q[1] = fmaf(cg, vq, q[1]);
    q[2] = fmaf(cg * u, vq, q[2]);
    q[3] = fmaf(cg * vq, vq, q[3]);
    q[4] += sU;
    q[5] = fmaf(sU, rg, q[5]);
  }
  __device__ __forceinline__ void fix(const CompConst& cc, float seed, float r2) {
    const float Ug = ex2<true>(-(kRGuard2 * rsqrt_fast(kRGuard2)) * cc.a0);
    q[4] += seed * (ex2<true>(-sqrt_fast(r2) * cc.a0) - Ug);
  }
  __device__ __forceinline__ void finish(const CompConst& cc, float (&out)[kNSum]) const {
    const float kf = cc.amp * cc.a1;
    out[0] = -kf * q[0]; out[1] = -kf * q[1]; out[2] = -kf * q[2]; out[3] = -kf * q[3];
    out[4] = q[4];
    out[5] = kf * cc.a1 * q[5];
    out[6] = 0.0f; out[7] = 0.0f; out[8] = out[2]; out[9] = 0.0f;
  }
};

// the sums of four consecutive pixels of a row: seed[k] at (x0 + k, y)
template <int KIND>
__device__ __forceinline__ void grad_add4(GradAcc<KIND>& acc, const CompConst& cc, const float (&seed)[4], float x0, float y) {
  if (KIND == GM_SKY) {
#pragma unroll
    for (int k = 0; k < 4; ++k) acc.add(cc, seed[k], 0.0f, 0.0f);
    return;
  }
  float u[4], vq[4], r2[4];
  row4(cc, x0, y, u, vq);
#pragma unroll
  for (int k = 0; k < 4; ++k) { acc.add(cc, seed[k], u[k], vq[k]); r2[k] = fmaf(u[k], u[k], vq[k] * vq[k]); }
  if (KIND == GM_SERSIC || KIND == GM_EXPDISK) {           // one test per group for the rare r < 1e-6 pixel
    if (fminf(fminf(r2[0], r2[1]), fminf(r2[2], r2[3])) < kRGuard2) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (r2[k] < kRGuard2) acc.fix(cc, seed[k], r2[k]);
    }
  }
}

}  // namespace gm
