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
};

// per (galaxy, component) constants produced by the prologue (step a0), 64 bytes
struct __align__(16) CompConst {
  float xc, yc, ct, st;      // centre, cos/sin(theta)
  float iq, q, amp, a0;      // 1/q, q, amplitude, kind specific ...
  float a1, a2, a3, a4;
  float a5, a6, a7, a8;
};

// ---------------------------------------------------------------------------
// step a0: Sersic nu_n, the root of P(2n, nu) = 1/2, and d nu / d n by
// implicit differentiation, in fp64.  Near the root x ~ a - 1/3 < a + 1, where
// the power series of the incomplete gamma function converges quickly.
// ---------------------------------------------------------------------------
__device__ inline double digamma_pos(double z) {
  double acc = 0.0;
  while (z < 10.0) { acc -= 1.0 / z; z += 1.0; }
  const double i2 = 1.0 / (z * z);
  return acc + log(z) - 0.5 / z -
         i2 * (1.0 / 12.0 - i2 * (1.0 / 120.0 - i2 * (1.0 / 252.0 - i2 * (1.0 / 240.0 - i2 * (1.0 / 132.0)))));
}

// returns P(a,x) by series; also d P / d a when dPda != nullptr
__device__ inline double gamma_P_series(double a, double x, double* dPda) {
  const double lx = log(x);
  double T = exp(a * lx - x - lgamma(a + 1.0));    // T_0 = x^a e^-x / Gamma(a+1)
  double psi = dPda ? digamma_pos(a + 1.0) : 0.0;
  double P = 0.0, dA = 0.0;
  for (int k = 0; k < 600; ++k) {
    P += T;
    dA += T * (lx - psi);
    if (T < 1e-17 * P && k > 2) break;
    psi += 1.0 / (a + k + 1.0);
    T *= x / (a + k + 1.0);
  }
  if (dPda) *dPda = dA;
  return P;
}

__device__ inline void sersic_nu(double n, double* nu, double* dnu) {
  const double a = 2.0 * n;
  if (!(n > 0.02) || !(n < 100.0)) { *nu = NAN; *dnu = NAN; return; }
  double x = a - 1.0 / 3.0 + 4.0 / (405.0 * n) + 46.0 / (25515.0 * n * n);
  double lo = 0.0, hi = a + 1.0;                   // P(a, a+1) > 1/2 for every a > 0
  if (!(x > 0.0 && x < hi)) x = 0.5 * a;
  const double lga = lgamma(a);
  for (int it = 0; it < 60; ++it) {
    const double f = gamma_P_series(a, x, nullptr) - 0.5;
    if (f > 0.0) hi = x; else lo = x;
    const double dpdx = exp((a - 1.0) * log(x) - x - lga);
    double xn = x - f / dpdx;
    if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
    const bool done = fabs(xn - x) <= 4e-16 * xn;
    x = xn;
    if (done) break;
  }
  double dPda;
  gamma_P_series(a, x, &dPda);
  const double dPdx = exp((a - 1.0) * log(x) - x - lga);
  *nu = x;
  *dnu = -2.0 * dPda / dPdx;
}

// One thread per (galaxy, component): physical parameters -> CompConst.
__device__ inline void make_comp_const(const ModelDesc& md, int c, const float* __restrict__ par,
                                       CompConst* out) {
  auto get = [&](int s, double dflt) -> double {
    const int idx = md.slot[c][s];
    return idx >= 0 ? (double)par[idx] : dflt;
  };
  CompConst cc;
  const double th = get(GM_SLOT_THETA, 0.0), q = get(GM_SLOT_Q, 1.0);
  cc.xc = (float)get(GM_SLOT_XC, 0.0);
  cc.yc = (float)get(GM_SLOT_YC, 0.0);
  cc.ct = (float)cos(th);
  cc.st = (float)sin(th);
  cc.iq = (float)(1.0 / q);
  cc.q = (float)q;
  cc.amp = (float)get(GM_SLOT_AMP, 0.0);
  double a[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  const double s0 = get(GM_SLOT_S0, 1.0), s1 = get(GM_SLOT_S1, 1.0), s2 = get(GM_SLOT_S2, 1.0);
  const double log2e = 1.4426950408889634074;
  switch (md.kind[c]) {
    case GM_SERSIC: {                       // Eq. 1
      double nu, dnu;
      sersic_nu(s1, &nu, &dnu);
      a[0] = 1.0 / s0;                      // 1/re
      a[1] = 1.0 / s1;                      // 1/n
      a[2] = nu * log2e;
      a[3] = nu;
      a[4] = dnu;
      break;
    }
    case GM_EXPDISK:                        // Eq. 7
      a[0] = log2e / s0;
      a[1] = 1.0 / s0;
      break;
    case GM_GAUSSIAN: {                     // Eq. 12, FWHM = 2 sqrt(2 ln 2) sigma
      const double cF = 2.0 * sqrt(2.0 * log(2.0));
      const double sg = s0 / cF;
      a[0] = log2e / (2.0 * sg * sg);
      a[1] = 1.0 / (sg * sg);
      a[2] = 1.0 / (sg * sg * sg * cF);
      break;
    }
    case GM_MOFFAT: {                       // Eq. 13-14
      const double p2 = pow(2.0, 1.0 / s1);
      const double rd = s0 / (2.0 * sqrt(p2 - 1.0));
      a[0] = 1.0 / (rd * rd);
      a[1] = s1;                            // n
      a[2] = 2.0 * s1 / (rd * rd);
      a[3] = 2.0 * s1 / (rd * rd * s0);
      a[4] = p2 * log(2.0) / (rd * rd * s1 * (p2 - 1.0));
      break;
    }
    case GM_FERRER:                         // Eq. 9
      a[0] = 1.0 / s0;                      // 1/r_out
      a[1] = s1;                            // a
      a[2] = 2.0 - s2;                      // 2 - b
      a[3] = s0;                            // r_out
      break;
    case GM_KING: {                         // Eq. 11 (R:K1)
      const double rc = s0, rt = s1, al = s2;
      const double zt = 1.0 + (rt / rc) * (rt / rc);
      const double T = pow(zt, -1.0 / al);
      a[0] = 1.0 / rc;
      a[1] = -1.0 / al;
      a[2] = T;
      a[3] = 1.0 / (1.0 - T);
      a[4] = al;
      a[5] = (2.0 / al) * T * (rt * rt / (rc * rc * rc)) / zt;     // dT/drc
      a[6] = -(2.0 / al) * T * (rt / (rc * rc)) / zt;              // dT/drt
      a[7] = T * log(zt) / (al * al);                              // dT/dalpha
      a[8] = rt;
      break;
    }
    default: break;                         // sky: amplitude only
  }
  cc.a0 = (float)a[0]; cc.a1 = (float)a[1]; cc.a2 = (float)a[2]; cc.a3 = (float)a[3];
  cc.a4 = (float)a[4]; cc.a5 = (float)a[5]; cc.a6 = (float)a[6]; cc.a7 = (float)a[7];
  cc.a8 = (float)a[8];
  *out = cc;
}

// ---------------------------------------------------------------------------
// step a1: elliptical radius, Eq. 2-4 with B = 0 (R:G2): rotate, then scale v by 1/q
// ---------------------------------------------------------------------------
struct Geo { float u, vq, r; };

__device__ __forceinline__ Geo geometry(const CompConst& cc, float x, float y) {
  const float dx = x - cc.xc, dy = y - cc.yc;
  Geo g;
  g.u = fmaf(cc.ct, dx, cc.st * dy);
  g.vq = fmaf(cc.ct, dy, -cc.st * dx) * cc.iq;
  g.r = sqrtf(fmaf(g.u, g.u, g.vq * g.vq));
  return g;
}

// radial law with unit amplitude at radius r (value only)
__device__ __forceinline__ float profile_value(int kind, const CompConst& cc, float r) {
  switch (kind) {
    case GM_SERSIC: {
      const float t = exp2f(log2f(r * cc.a0) * cc.a1);           // (r/re)^(1/n); 0 at r = 0
      return exp2f(-cc.a2 * (t - 1.0f));
    }
    case GM_EXPDISK:
      return exp2f(-r * cc.a0);
    case GM_GAUSSIAN:
      return exp2f(-r * r * cc.a0);
    case GM_MOFFAT:
      return exp2f(-cc.a1 * log2f(fmaf(r * r, cc.a0, 1.0f)));
    case GM_FERRER: {
      if (!(r < cc.a3)) return 0.0f;
      const float w = exp2f(cc.a2 * log2f(r * cc.a0));
      return exp2f(cc.a1 * log2f(1.0f - w));
    }
    case GM_KING: {
      if (!(r < cc.a8)) return 0.0f;
      const float ra = r * cc.a0;
      const float R = exp2f(cc.a1 * log2f(fmaf(ra, ra, 1.0f)));
      const float X = (R - cc.a2) * cc.a3;
      return X > 0.0f ? exp2f(cc.a4 * log2f(X)) : 0.0f;
    }
    default:
      return 1.0f;                                                // sky
  }
}

// radial law and its derivatives, evaluated at rg (the caller passes rg = max(r, 1e-6))
// U value, dUdr, dUds[0..2] = d/d(s0, s1, s2), unit amplitude
__device__ __forceinline__ void profile_grad(int kind, const CompConst& cc, float rg, float& U,
                                             float& dUdr, float& d0, float& d1, float& d2) {
  U = 0.0f; dUdr = 0.0f; d0 = 0.0f; d1 = 0.0f; d2 = 0.0f;
  switch (kind) {
    case GM_SERSIC: {
      const float L = log2f(rg * cc.a0);
      const float t = exp2f(L * cc.a1);
      U = exp2f(-cc.a2 * (t - 1.0f));
      const float k = U * cc.a3 * t * cc.a1;                      // U nu t / n
      dUdr = -__fdividef(k, rg);
      d0 = k * cc.a0;                                             // d/d re
      d1 = U * (-cc.a4 * (t - 1.0f) + cc.a3 * t * (L * kLn2) * cc.a1 * cc.a1);   // d/d n
      break;
    }
    case GM_EXPDISK:
      U = exp2f(-rg * cc.a0);
      dUdr = -U * cc.a1;
      d0 = U * rg * cc.a1 * cc.a1;
      break;
    case GM_GAUSSIAN:
      U = exp2f(-rg * rg * cc.a0);
      dUdr = -U * rg * cc.a1;
      d0 = U * rg * rg * cc.a2;
      break;
    case GM_MOFFAT: {
      const float A = fmaf(rg * rg, cc.a0, 1.0f);
      const float lA = log2f(A);
      U = exp2f(-cc.a1 * lA);
      const float UA = __fdividef(U, A);
      dUdr = -cc.a2 * UA * rg;
      d0 = cc.a3 * UA * rg * rg;                                  // d/d FWHM
      d1 = -U * (lA * kLn2) + UA * rg * rg * cc.a4;               // d/d n
      break;
    }
    case GM_FERRER: {
      if (!(rg < cc.a3)) break;
      const float Lr = log2f(rg * cc.a0);
      const float w = exp2f(cc.a2 * Lr);
      const float omw = 1.0f - w;
      if (!(omw > 0.0f)) break;
      const float lo = log2f(omw);
      U = exp2f(cc.a1 * lo);
      const float core = cc.a1 * __fdividef(U, omw);                       // a (1-w)^(a-1)
      dUdr = -__fdividef(core * cc.a2 * w, rg);
      d0 = core * cc.a2 * w * cc.a0;                              // d/d r_out
      d1 = U * (lo * kLn2);                                       // d/d a
      d2 = core * w * (Lr * kLn2);                                // d/d b
      break;
    }
    case GM_KING: {
      if (!(rg < cc.a8)) break;
      const float ra = rg * cc.a0;
      const float z = fmaf(ra, ra, 1.0f);
      const float lz = log2f(z);
      const float R = exp2f(cc.a1 * lz);
      const float X = (R - cc.a2) * cc.a3;
      if (!(X > 0.0f)) break;
      const float lX = log2f(X);
      U = exp2f(cc.a4 * lX);
      const float UR = cc.a4 * __fdividef(U, X) * cc.a3;                   // alpha X^(alpha-1) / (1-T)
      const float UT = UR * (R - 1.0f) * cc.a3;
      const float m2a = -2.0f * cc.a1;                            // 2/alpha
      const float Rr = -m2a * __fdividef(R * (rg * cc.a0 * cc.a0), z);
      const float Rrc = m2a * __fdividef(R * (ra * ra * cc.a0), z);
      const float Ral = R * (lz * kLn2) * cc.a1 * cc.a1;
      dUdr = UR * Rr;
      d0 = UR * Rrc + UT * cc.a5;                                 // d/d rc
      d1 = UT * cc.a6;                                            // d/d rt
      d2 = U * (lX * kLn2) + UR * Ral + UT * cc.a7;               // d/d alpha
      break;
    }
    default: break;
  }
}

}  // namespace gm
