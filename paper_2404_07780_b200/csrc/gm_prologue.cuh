// gm_prologue.cuh -- step a0 of the hot path: per-galaxy, per-component constants
// in fp64 (nu_n and d nu_n / d n for the Sersic law, FWHM -> sigma / r_d, King's T
// and its derivatives).  Included by gm_api.cu only (it owns the nu table symbol).
#pragma once
#include "gm_device.cuh"

namespace gm {

// ---------------------------------------------------------------------------
// step a0: Sersic nu_n, the root of P(2n, nu) = 1/2, and d nu / d n by
// implicit differentiation, in fp64.  Near the root x ~ a - 1/3 < a + 1, where
// the power series of the incomplete gamma function converges quickly.
// ---------------------------------------------------------------------------
__host__ __device__ inline double digamma_pos(double z) {
  double acc = 0.0;
  while (z < 10.0) { acc -= 1.0 / z; z += 1.0; }
  const double i2 = 1.0 / (z * z);
  return acc + log(z) - 0.5 / z -
         i2 * (1.0 / 12.0 - i2 * (1.0 / 120.0 - i2 * (1.0 / 252.0 - i2 * (1.0 / 240.0 - i2 * (1.0 / 132.0)))));
}

// returns P(a,x) by series; also d P / d a when dPda != nullptr
__host__ __device__ inline double gamma_P_series(double a, double x, double* dPda) {
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

__host__ __device__ inline void sersic_nu_exact(double n, double* nu, double* dnu) {
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

// Fast path for the prologue: cubic Hermite interpolation of nu(s), s = ln n, from a
// table of (nu, d nu / d s) that the host builds once with sersic_nu_exact (gm_api.cu)
// and uploads to this symbol.  Grid spacing h = ln(1024) / 4096 gives an interpolation
// error below 1e-11 in nu over n in [1/16, 64]; outside it the exact solver runs.
constexpr int kNuTableN = 4096;
constexpr double kNuTableS0 = -2.772588722239781;       // ln(1/16)
constexpr double kNuTableS1 = 4.1588830833596715;       // ln(64)
__device__ double2 g_nu_table[kNuTableN + 1];

__device__ inline void sersic_nu(double n, double* nu, double* dnu) {
  const double s = log(n);
  if (!(s >= kNuTableS0 && s < kNuTableS1)) { sersic_nu_exact(n, nu, dnu); return; }
  const double h = (kNuTableS1 - kNuTableS0) / kNuTableN;
  const double pos = (s - kNuTableS0) / h;
  int i = (int)pos;
  if (i > kNuTableN - 1) i = kNuTableN - 1;
  const double t = pos - i;
  const double2 e0 = g_nu_table[i], e1 = g_nu_table[i + 1];
  const double t2 = t * t, t3 = t2 * t;
  const double h00 = 2 * t3 - 3 * t2 + 1, h10 = t3 - 2 * t2 + t, h01 = -2 * t3 + 3 * t2, h11 = t3 - t2;
  *nu = h00 * e0.x + h10 * h * e0.y + h01 * e1.x + h11 * h * e1.y;
  const double d00 = 6 * t2 - 6 * t, d10 = 3 * t2 - 4 * t + 1, d01 = -d00, d11 = 3 * t2 - 2 * t;
  const double dnuds = (d00 * e0.x + d01 * e1.x) / h + d10 * e0.y + d11 * e1.y;
  *dnu = dnuds / n;
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
  cc.b0 = cc.b1 = cc.b2 = 0.0f;
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
      cc.b0 = (float)(1.0 / (s0 * s0));     // value_uv, GradAcc: lg2(r^2 / re^2) / (2n)
      cc.b1 = (float)(0.5 / s1);
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
  // Eq. 2 exponent and, in magnitude mode, the amplitude of Eq. 5 / 8 / 10 / 15 with the
  // logarithmic derivatives the gradient needs (all fp64, once per galaxy and component)
  const double Bx = get(GM_SLOT_BOX, 0.0), cexp = 2.0 + Bx;
  cc.c = (float)cexp; cc.ic = (float)(1.0 / cexp); cc.cm1 = (float)(cexp - 1.0);
  cc.dl_box = 0.0f; cc.dl_m = 0.0f; cc.dl_q = 0.0f; cc.dl_s0 = 0.0f; cc.dl_s1 = 0.0f; cc.dl_s2 = 0.0f;
  if (md.mag[c]) {
    const double ln10 = 2.302585092994045684, pi = 3.14159265358979323846;
    const double m = get(GM_SLOT_AMP, 0.0), m0 = get(GM_SLOT_M0, 0.0);
    // Eq. 6: ln r_box = ln(pi c / 2) - 2 lnGamma(1/c) + lnGamma(2/c)
    double lamp = log(pi * cexp / 2.0) - 2.0 * lgamma(1.0 / cexp) + lgamma(2.0 / cexp)
                  - 0.4 * ln10 * (m - m0) - log(q);
    cc.dl_box = (float)(1.0 / cexp + 2.0 * (digamma_pos(1.0 / cexp) - digamma_pos(2.0 / cexp)) / (cexp * cexp));
    cc.dl_m = (float)(-0.4 * ln10);
    cc.dl_q = (float)(-1.0 / q);
    cc.dl_s0 = (float)(-2.0 / s0);
    switch (md.kind[c]) {
      case GM_SERSIC: {                     // Eq. 5
        const double nu = a[3], dnu = a[4], n = s1;
        lamp += 2.0 * n * log(nu) - log(2.0 * pi * s0 * s0 * n) - lgamma(2.0 * n) - nu;
        cc.dl_s1 = (float)(2.0 * log(nu) + 2.0 * n * dnu / nu - 1.0 / n - 2.0 * digamma_pos(2.0 * n) - dnu);
        break;
      }
      case GM_EXPDISK:                      // Eq. 8
        lamp -= log(2.0 * pi * s0 * s0);
        break;
      case GM_FERRER: {                     // Eq. 10
        const double fa = s1, z = 1.0 + 2.0 / (2.0 - s2);
        lamp -= log(pi * s0 * s0 * fa) + lgamma(fa) + lgamma(z) - lgamma(fa + z);
        cc.dl_s1 = (float)(-1.0 / fa - digamma_pos(fa) + digamma_pos(fa + z));
        cc.dl_s2 = (float)((digamma_pos(fa + z) - digamma_pos(z)) * 2.0 / ((2.0 - s2) * (2.0 - s2)));
        break;
      }
      case GM_MOFFAT: {                     // Eq. 15 with rd of Eq. 14
        const double p2 = pow(2.0, 1.0 / s1);
        const double rd = s0 / (2.0 * sqrt(p2 - 1.0));
        lamp += log(s1 - 1.0) - log(pi * rd * rd);
        cc.dl_s1 = (float)(1.0 / (s1 - 1.0) - p2 * log(2.0) / (s1 * s1 * (p2 - 1.0)));
        break;
      }
      default: lamp = NAN; break;           // rejected by validate()
    }
    cc.amp = (float)exp(lamp);
  }
  cc.a0 = (float)a[0]; cc.a1 = (float)a[1]; cc.a2 = (float)a[2]; cc.a3 = (float)a[3];
  cc.a4 = (float)a[4]; cc.a5 = (float)a[5]; cc.a6 = (float)a[6]; cc.a7 = (float)a[7];
  cc.a8 = (float)a[8];
  *out = cc;
}

}  // namespace gm
