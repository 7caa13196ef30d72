/* gm_oracle.c -- ORACLE for the batched galaxy-profile chi^2 + gradient + update
 * hot path of arxiv 2404.07780 (Galmoss).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, double
 * precision CPU restatement of the paper's forward model, PSF convolution,
 * chi^2, analytic gradient and gradient-descent (Adam) update, written from
 * /root/reference/PAPER.md ("P:<line>") so a reader can check it against the
 * paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with the CUDA path under
 * paper_2404_07780_b200/csrc/ and neither includes the other.
 *
 * No blocking, fusion or reordering beyond the definitions: every convolution
 * is the four-deep loop of its definition, every sum runs in index order.
 * OpenMP is used over galaxies only (galaxies are independent).
 *
 * Readings of the paper where it is silent / garbled:
 *   G1 grid  x = j + 0.5, y = H - 0.5 - i           (App. C)
 *   G2 r_maj = |u|, r_min = |v| (abs of the rotated sum, not per term)
 *   K1 King bracket is R(r) - T (P:146-150 prints the opposite sign)
 *   F1 FWHM = 2 sqrt(2 ln 2) sigma exactly (P:160 prints 2.354)
 *   S1 nu_n is the exact root of P(2n, nu) = 1/2
 *   S4 derivative factors are evaluated at r_g = max(r, 1e-6 px)
 *   S5 point sampling at pixel centres, no oversampling
 *   C1 true convolution, PSF centre (K-1)/2, zero fill, same size
 *   X1 mask = Omega: 1 used, 0 ignored; weight chosen by select
 *   O1 optimiser = Adam (bias corrected), per galaxy -- PARITY UNPINNED against
 *      the real galmoss package (P:39, P:206, P:635 do not name the optimiser);
 *      the update rule itself is pinned against torch.optim.Adam in tests.
 *   O3 bounds by projection of the optimiser variable after each step
 *   O4 log=True means u = log10(p)
 *
 * Pins (tests/test_oracle_*.py): closed-form total fluxes (Eq. 5, 8, 10, 15),
 * scipy.special.gammaincinv, scipy.signal.convolve2d, central finite
 * differences, brute-force chi^2, torch.optim.Adam, identities n=0.5/n=1;
 * covariance sigma_p: numpy.linalg.inv, the closed form of a linear model, and the
 * scatter of refits over noise realisations; bootstrap: splitmix64 test vectors, count
 * invariants, chi^2 over the explicit list of drawn pixels, numpy.std, the closed form
 * sigma/sqrt(N) of a resampled mean.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GMO_SERSIC   0
#define GMO_EXPDISK  1
#define GMO_FERRER   2
#define GMO_KING     3
#define GMO_GAUSSIAN 4
#define GMO_MOFFAT   5
#define GMO_SKY      6

/* component descriptor: 12 int32 per component
 *   [0] kind  [1] convolve flag  [2..11] parameter-vector index ("slot") for
 *   xc, yc, theta[rad], q, amplitude, s0, s1, s2, boxiness B, zero point m0 ;
 *   -1 = unused.  When the m0 slot is used the amplitude slot holds a MAGNITUDE m
 *   and the intensity follows from Eq. 5 / 8 / 10 / 15 (P:84-93, P:115, P:129,
 *   P:178) with the zero point m0 = par[slot m0] (the paper's gm.p(m, M0=...),
 *   P:279-281; m0 is normally held fixed by the caller's free_mask).
 *   Sersic: amp=Ie s0=re s1=n | Exp: amp=I0 s0=rs | Ferrer: amp=I0 s0=r_out
 *   s1=a s2=b | King: amp=I0 s0=rc s1=rt s2=alpha | Gaussian: amp=I0 s0=FWHM |
 *   Moffat: amp=I0 s0=FWHM s1=n | Sky: amp=I_sky.
 *   Two components naming the same index share ("tie") that parameter. */
#define GMO_DESC 12
enum { S_XC = 0, S_YC, S_TH, S_Q, S_AMP, S_S0, S_S1, S_S2, S_BOX, S_M0, N_SLOT };

#define GMO_RGUARD 1e-6 /* reading S4 */

/* ------------------------------------------------------------------------- */
/* nu_n: "computed numerically from the inverse cumulative distribution  */
/* function of the gamma distribution": root of P(2n, nu) = 1/2.              */
/* ------------------------------------------------------------------------- */

/* regularised lower incomplete gamma P(a,x), a>0, x>=0.
 * series   P = e^{-x} x^a sum_k x^k / Gamma(a+k+1)          for x < a+1
 * fraction Q = 1-P by the modified Lentz continued fraction  otherwise      */
double gmo_gammainc_P(double a, double x)
{
    if (x <= 0.0) return 0.0;
    if (x < a + 1.0) {
        double term = 1.0 / a, sum = term, ak = a;
        for (int k = 0; k < 10000; ++k) {
            ak += 1.0;
            term *= x / ak;
            sum += term;
            if (fabs(term) < fabs(sum) * 1e-17) break;
        }
        return sum * exp(-x + a * log(x) - lgamma(a));
    } else {
        const double tiny = 1e-300;
        double b = x + 1.0 - a, c = 1.0 / tiny, d = 1.0 / b, h = d;
        for (int i = 1; i < 10000; ++i) {
            double an = -i * (i - a);
            b += 2.0;
            d = an * d + b; if (fabs(d) < tiny) d = tiny;
            c = b + an / c; if (fabs(c) < tiny) c = tiny;
            d = 1.0 / d;
            double del = d * c;
            h *= del;
            if (fabs(del - 1.0) < 1e-16) break;
        }
        return 1.0 - exp(-x + a * log(x) - lgamma(a)) * h;
    }
}

/* digamma psi(z), z>0: upward shift to z>=12, then the asymptotic series */
static double digamma_pos(double z)
{
    double acc = 0.0;
    while (z < 12.0) { acc -= 1.0 / z; z += 1.0; }
    double i2 = 1.0 / (z * z);
    double s = log(z) - 0.5 / z
             - i2 * (1.0 / 12.0 - i2 * (1.0 / 120.0 - i2 * (1.0 / 252.0 - i2 * (1.0 / 240.0
             - i2 * (1.0 / 132.0 - i2 * (691.0 / 32760.0 - i2 * (1.0 / 12.0)))))));
    return acc + s;
}

/* nu_n: safeguarded Newton on f(nu) = P(2n,nu) - 1/2, seed 2n - 1/3 */
double gmo_sersic_nu(double n)
{
    const double a = 2.0 * n;
    double lo = 0.0, hi = a + 10.0 * sqrt(a) + 10.0; /* P(a,hi) ~ 1 */
    double x = a - 1.0 / 3.0;
    if (x <= 0.0) x = 0.5 * a;
    for (int it = 0; it < 200; ++it) {
        double f = gmo_gammainc_P(a, x) - 0.5;
        if (f > 0.0) hi = x; else lo = x;
        double dpdx = exp((a - 1.0) * log(x) - x - lgamma(a));
        double xn = x - f / dpdx;
        if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
        if (fabs(xn - x) <= 1e-15 * fabs(xn)) { x = xn; break; }
        x = xn;
    }
    return x;
}

/* d nu_n / d n by implicit differentiation of P(a, x) = 1/2 at a = 2n, x = nu:
 *   dnu/dn = -2 (dP/da) / (dP/dx),  dP/dx = x^{a-1} e^{-x} / Gamma(a),
 *   P(a,x) = sum_k T_k,  T_k = x^{a+k} e^{-x} / Gamma(a+k+1),
 *   dP/da  = sum_k T_k (ln x - psi(a+k+1)).                                   */
double gmo_sersic_dnu_dn(double n)
{
    const double a = 2.0 * n;
    const double x = gmo_sersic_nu(n);
    const double lx = log(x);
    double T = exp(a * lx - x - lgamma(a + 1.0));
    double psi = digamma_pos(a + 1.0);
    double dPda = 0.0;
    for (int k = 0; k < 10000; ++k) {
        double c = T * (lx - psi);
        dPda += c;
        if (k > 4 && fabs(T) * (1.0 + fabs(lx - psi)) < 1e-18) break;
        psi += 1.0 / (a + k + 1.0);  /* psi(z+1) = psi(z) + 1/z */
        T *= x / (a + k + 1.0);      /* T_{k+1} = T_k x / (a+k+1) */
    }
    double dPdx = exp((a - 1.0) * lx - x - lgamma(a));
    return -2.0 * dPda / dPdx;
}

/* ------------------------------------------------------------------------- */
/* magnitude <-> intensity helpers, Eq. 5, 6, 8, 10, 15 */
/* "flux" below is 10^{-0.4 (m - m0)}                                         */
/* ------------------------------------------------------------------------- */
static double beta_fn(double a, double b) { return exp(lgamma(a) + lgamma(b) - lgamma(a + b)); }

double gmo_r_box(double B) /* Eq. 6 */
{
    const double pi = 3.14159265358979323846;
    double c = 2.0 + B;
    return pi * c / (2.0 * beta_fn(1.0 / c, 1.0 / c));
}
double gmo_sersic_Ie_from_flux(double flux, double re, double n, double q, double B) /* Eq. 5 */
{
    const double pi = 3.14159265358979323846;
    double nu = gmo_sersic_nu(n);
    return gmo_r_box(B) * pow(nu, 2.0 * n) * flux / (2.0 * pi * q * re * re * n * tgamma(2.0 * n) * exp(nu));
}
double gmo_expdisk_I0_from_flux(double flux, double rs, double q, double B) /* Eq. 8 */
{
    const double pi = 3.14159265358979323846;
    return gmo_r_box(B) * flux / (2.0 * pi * q * rs * rs);
}
double gmo_ferrer_I0_from_flux(double flux, double rout, double a, double b, double q, double B) /* Eq. 10 */
{
    const double pi = 3.14159265358979323846;
    return gmo_r_box(B) * flux / (pi * q * rout * rout * a * beta_fn(a, 1.0 + 2.0 / (2.0 - b)));
}
double gmo_moffat_rd(double fwhm, double n) /* Eq. 14 */
{
    return fwhm / (2.0 * sqrt(pow(2.0, 1.0 / n) - 1.0));
}
double gmo_moffat_I0_from_flux(double flux, double fwhm, double n, double q, double B) /* Eq. 15 */
{
    const double pi = 3.14159265358979323846;
    double rd = gmo_moffat_rd(fwhm, n);
    return gmo_r_box(B) * (n - 1.0) * flux / (pi * q * rd * rd);
}
/* Eq. 17: ln L of the chi^2 distribution with k degrees of freedom */
double gmo_loglike(double chi2, double k)
{
    return -0.5 * k * log(2.0) - lgamma(0.5 * k) + (0.5 * k - 1.0) * log(chi2) - 0.5 * chi2;
}

/* Amplitude (I_e or I_0) from the magnitude parameterisation, and the derivatives
 * of its logarithm with respect to every slot it depends on:
 *   flux = 10^{-0.4 (m - m0)};  amp = Eq. 5 (Sersic), 8 (ExpDisk), 10 (Ferrer),
 *   15 (Moffat) exactly as printed (the helpers above).
 * dla[k] = d ln(amp) / d slot_k.  With c = 2 + B, from Eq. 6:
 *   ln r_box = ln(pi c / 2) - 2 lnGamma(1/c) + lnGamma(2/c)
 *   d ln r_box / dB = 1/c + 2 [psi(1/c) - psi(2/c)] / c^2.
 * Returns 0, or -1 for a kind the paper gives no magnitude relation for.        */
static int amplitude_from_mag(int kind, const double p[/*N_SLOT*/], double nu, double dnu,
                              double *amp, double dla[/*N_SLOT*/])
{
    const double ln10 = log(10.0);
    const double m = p[S_AMP], m0 = p[S_M0], q = p[S_Q], B = p[S_BOX];
    const double s0 = p[S_S0], s1 = p[S_S1], s2 = p[S_S2];
    const double flux = pow(10.0, -0.4 * (m - m0));
    const double c = 2.0 + B;
    for (int k = 0; k < N_SLOT; ++k) dla[k] = 0.0;
    dla[S_AMP] = -0.4 * ln10;                 /* d/dm  */
    dla[S_M0] = +0.4 * ln10;                 /* d/dm0 */
    dla[S_Q] = -1.0 / q;                    /* every relation carries 1/q */
    dla[S_BOX] = 1.0 / c + 2.0 * (digamma_pos(1.0 / c) - digamma_pos(2.0 / c)) / (c * c);
    switch (kind) {
    case GMO_SERSIC: {  /* Eq. 5: r_box nu^{2n} F / (2 pi q re^2 n Gamma(2n) e^{nu}) */
        const double re = s0, n = s1;
        *amp = gmo_sersic_Ie_from_flux(flux, re, n, q, B);
        dla[S_S0] = -2.0 / re;
        dla[S_S1] = 2.0 * log(nu) + 2.0 * n * dnu / nu - 1.0 / n - 2.0 * digamma_pos(2.0 * n) - dnu;
        return 0; }
    case GMO_EXPDISK:   /* Eq. 8: r_box F / (2 pi q rs^2) */
        *amp = gmo_expdisk_I0_from_flux(flux, s0, q, B);
        dla[S_S0] = -2.0 / s0;
        return 0;
    case GMO_FERRER: {  /* Eq. 10: r_box F / (pi q rout^2 a beta(a, 1 + 2/(2-b))) */
        const double rout = s0, a = s1, b = s2;
        const double z = 1.0 + 2.0 / (2.0 - b);
        *amp = gmo_ferrer_I0_from_flux(flux, rout, a, b, q, B);
        dla[S_S0] = -2.0 / rout;
        dla[S_S1] = -1.0 / a - (digamma_pos(a) - digamma_pos(a + z));
        dla[S_S2] = -(digamma_pos(z) - digamma_pos(a + z)) * 2.0 / ((2.0 - b) * (2.0 - b));
        return 0; }
    case GMO_MOFFAT: {  /* Eq. 15 with rd of Eq. 14: r_box (n-1) F / (pi q rd^2) */
        const double fwhm = s0, n = s1;
        const double p2 = pow(2.0, 1.0 / n);
        *amp = gmo_moffat_I0_from_flux(flux, fwhm, n, q, B);
        dla[S_S0] = -2.0 / fwhm;
        dla[S_S1] = 1.0 / (n - 1.0) - p2 * log(2.0) / (n * n * (p2 - 1.0));
        return 0; }
    default:
        *amp = NAN;
        return -1;
    }
}

/* ------------------------------------------------------------------------- */
/* radial profiles, Eq. 1, 7, 9, 11, 12, 13, 16, with their derivatives.      */
/* value at r; derivative factors at rg = max(r, GMO_RGUARD) (reading S4).    */
/* out: *I value, *dIdr, dIds[3] = d/d(s0,s1,s2); d/d(amp) = I/amp is done by  */
/* the caller as "unit", the profile evaluated with amplitude 1.               */
/* ------------------------------------------------------------------------- */
typedef struct {
    double nu, dnu; /* Sersic nu_n, d nu / d n (computed once per galaxy) */
} gmo_aux;

static void profile_unit(int kind, double r, const double s[3], const gmo_aux *aux,
                         double *U, double *dUdr, double dUds[3])
{
    const double rg = r > GMO_RGUARD ? r : GMO_RGUARD;
    dUds[0] = dUds[1] = dUds[2] = 0.0;
    *U = 0.0; *dUdr = 0.0;
    switch (kind) {
    case GMO_SERSIC: { /* Eq. 1 */
        const double re = s[0], n = s[1], nu = aux->nu;
        const double t = pow(r / re, 1.0 / n);
        *U = exp(-nu * (t - 1.0));
        const double tg = pow(rg / re, 1.0 / n);
        const double Ug = exp(-nu * (tg - 1.0));
        *dUdr = -Ug * nu * tg / (n * rg);
        dUds[0] = Ug * nu * tg / (n * re);
        dUds[1] = Ug * (-aux->dnu * (tg - 1.0) + nu * tg * log(rg / re) / (n * n));
        break; }
    case GMO_EXPDISK: { /* Eq. 7 */
        const double rs = s[0];
        *U = exp(-r / rs);
        const double Ug = exp(-rg / rs);
        *dUdr = -Ug / rs;
        dUds[0] = Ug * rg / (rs * rs);
        break; }
    case GMO_FERRER: { /* Eq. 9: [1 - (r/r_out)^{2-b}]^a inside r_out, 0 outside */
        const double rout = s[0], a = s[1], b = s[2];
        if (r >= rout) break;
        const double w = pow(r / rout, 2.0 - b);
        *U = pow(1.0 - w, a);
        const double wg = pow(rg / rout, 2.0 - b);
        const double omw = 1.0 - wg;
        if (omw <= 0.0) break;
        const double Ug = pow(omw, a);
        const double core = a * pow(omw, a - 1.0);      /* a (1-w)^{a-1} */
        *dUdr = -core * (2.0 - b) * wg / rg;
        dUds[0] = core * (2.0 - b) * wg / rout;
        dUds[1] = Ug * log(omw);
        dUds[2] = core * wg * log(rg / rout);
        break; }
    case GMO_KING: { /* Eq. 11 with the bracket read as R(r) - T (reading K1) */
        const double rc = s[0], rt = s[1], al = s[2];
        if (r >= rt) break;
        const double zt = 1.0 + (rt / rc) * (rt / rc);
        const double T = pow(zt, -1.0 / al);
        const double z = 1.0 + (r / rc) * (r / rc);
        const double R = pow(z, -1.0 / al);
        *U = pow((R - T) / (1.0 - T), al);
        const double zg = 1.0 + (rg / rc) * (rg / rc);
        const double Rg = pow(zg, -1.0 / al);
        const double X = (Rg - T) / (1.0 - T);
        if (X <= 0.0) break;
        const double Ug = pow(X, al);
        const double U_R = al * pow(X, al - 1.0) / (1.0 - T);
        const double U_T = al * pow(X, al - 1.0) * (Rg - 1.0) / ((1.0 - T) * (1.0 - T));
        const double R_r  = -(2.0 / al) * Rg * (rg / (rc * rc)) / zg;
        const double R_rc =  (2.0 / al) * Rg * (rg * rg / (rc * rc * rc)) / zg;
        const double T_rt = -(2.0 / al) * T * (rt / (rc * rc)) / zt;
        const double T_rc =  (2.0 / al) * T * (rt * rt / (rc * rc * rc)) / zt;
        const double R_al = Rg * log(zg) / (al * al);
        const double T_al = T * log(zt) / (al * al);
        *dUdr = U_R * R_r;
        dUds[0] = U_R * R_rc + U_T * T_rc;
        dUds[1] = U_T * T_rt;
        dUds[2] = Ug * log(X) + U_R * R_al + U_T * T_al;
        break; }
    case GMO_GAUSSIAN: { /* Eq. 12, sigma = FWHM / (2 sqrt(2 ln 2)) (reading F1) */
        const double cF = 2.0 * sqrt(2.0 * log(2.0));
        const double sg = s[0] / cF;
        *U = exp(-r * r / (2.0 * sg * sg));
        const double Ug = exp(-rg * rg / (2.0 * sg * sg));
        *dUdr = -Ug * rg / (sg * sg);
        dUds[0] = Ug * rg * rg / (sg * sg * sg) / cF;
        break; }
    case GMO_MOFFAT: { /* Eq. 13-14 */
        const double fwhm = s[0], n = s[1];
        const double p2 = pow(2.0, 1.0 / n);
        const double rd = fwhm / (2.0 * sqrt(p2 - 1.0));
        const double A = 1.0 + (r / rd) * (r / rd);
        *U = pow(A, -n);
        const double Ag = 1.0 + (rg / rd) * (rg / rd);
        const double Ug = pow(Ag, -n);
        const double dUdrd = 2.0 * n * Ug * rg * rg / (rd * rd * rd * Ag);
        *dUdr = -2.0 * n * Ug * rg / (rd * rd * Ag);
        dUds[0] = dUdrd * rd / fwhm;
        dUds[1] = -Ug * log(Ag) + dUdrd * rd * p2 * log(2.0) / (2.0 * n * n * (p2 - 1.0));
        break; }
    default: break;
    }
}

/* one component at pixel centre (x,y): value I and dI/d(slot) for the 10 slots.
 * mag != 0: the amplitude slot holds a magnitude (amplitude_from_mag above); then
 * dI/d(slot) gains I * d ln(amp)/d(slot) for every slot the amplitude depends on. */
static void component_eval(int kind, int mag, const double p[N_SLOT], const gmo_aux *aux,
                           double x, double y, double *I, double dI[N_SLOT], int want_grad)
{
    for (int k = 0; k < N_SLOT; ++k) dI[k] = 0.0;
    if (kind == GMO_SKY) { /* Eq. 16 */
        *I = p[S_AMP];
        dI[S_AMP] = 1.0;
        return;
    }
    const double xc = p[S_XC], yc = p[S_YC], th = p[S_TH], q = p[S_Q];
    const double B = p[S_BOX];
    double amp = p[S_AMP], dla[N_SLOT];
    if (mag) amplitude_from_mag(kind, p, aux->nu, aux->dnu, &amp, dla);
    const double c = B + 2.0;
    const double ct = cos(th), st = sin(th);
    const double dx = x - xc, dy = y - yc;
    /* Eq. 3-4 (reading G2): rotate, then absolute value */
    const double u = ct * dx + st * dy;
    const double v = -st * dx + ct * dy;
    const double au = fabs(u), av = fabs(v) / q;
    /* Eq. 2 */
    const double uc = (au > 0.0) ? pow(au, c) : 0.0;
    const double vc = (av > 0.0) ? pow(av, c) : 0.0;
    const double r = pow(uc + vc, 1.0 / c);
    double U, dUdr, dUds[3];
    const double s[3] = { p[S_S0], p[S_S1], p[S_S2] };
    profile_unit(kind, r, s, aux, &U, &dUdr, dUds);
    *I = amp * U;
    if (!want_grad) return;
    dI[S_AMP] = U;
    dI[S_S0] = amp * dUds[0];
    dI[S_S1] = amp * dUds[1];
    dI[S_S2] = amp * dUds[2];
    /* geometry chain rule, general exponent c = B + 2, at rg */
    const double rg = r > GMO_RGUARD ? r : GMO_RGUARD;
    const double rcm1 = pow(rg, c - 1.0);
    const double su = (u > 0.0) - (u < 0.0), sv = (v > 0.0) - (v < 0.0);
    const double dr_du = (au > 0.0) ? su * pow(au, c - 1.0) / rcm1 : 0.0;
    const double dr_dv = (av > 0.0) ? sv * pow(fabs(v), c - 1.0) / (pow(q, c) * rcm1) : 0.0;
    const double dr_dq = (av > 0.0) ? -pow(fabs(v), c) / (pow(q, c + 1.0) * rcm1) : 0.0;
    const double lu = (au > 0.0) ? uc * log(au) : 0.0;
    const double lv = (av > 0.0) ? vc * log(av) : 0.0;
    const double dr_dB = (uc + vc > 0.0) ? (rg / c) * ((lu + lv) / (uc + vc) - log(rg)) : 0.0;
    /* du/dxc=-cos dv/dxc=sin | du/dyc=-sin dv/dyc=-cos | du/dth=v dv/dth=-u */
    const double A = amp * dUdr;
    dI[S_XC] = A * (dr_du * (-ct) + dr_dv * st);
    dI[S_YC] = A * (dr_du * (-st) + dr_dv * (-ct));
    dI[S_TH] = A * (dr_du * v + dr_dv * (-u));
    dI[S_Q]  = A * dr_dq;
    dI[S_BOX] = A * dr_dB;
    if (mag) {
        dI[S_AMP] = 0.0;
        for (int k = 0; k < N_SLOT; ++k) dI[k] += (*I) * dla[k];
    }
}

static void gather_params(const int32_t *d, const double *par, double p[N_SLOT])
{
    for (int k = 0; k < N_SLOT; ++k) {
        int s = d[2 + k];
        p[k] = (s >= 0) ? par[s] : 0.0;
    }
    if (d[2 + S_Q] < 0) p[S_Q] = 1.0;   /* unused q: circular */
}

static void make_aux(int kind, const double p[N_SLOT], gmo_aux *aux)
{
    aux->nu = aux->dnu = 0.0;
    if (kind == GMO_SERSIC) {
        aux->nu = gmo_sersic_nu(p[S_S1]);
        aux->dnu = gmo_sersic_dnu_dn(p[S_S1]);
    }
}

static int is_convolved(const int32_t *d) { return d[0] != GMO_SKY && d[1] != 0; }

/* pixel-centre coordinates, reading G1 */
static double pix_x(int j) { return j + 0.5; }
static double pix_y(int i, int H) { return H - 0.5 - i; }

/* exported for unit pins: one component, amplitude and all, at one point */
void gmo_component_at(int kind, int mag, const double p[N_SLOT], double x, double y, double *I, double *dI /*[10]*/)
{
    gmo_aux aux; make_aux(kind, p, &aux);
    component_eval(kind, mag, p, &aux, x, y, I, dI, 1);
}

/* exported for unit pins: amplitude of the magnitude parameterisation and d ln(amp)/d slot */
int gmo_amplitude_from_mag(int kind, const double p[N_SLOT], double *amp, double *dla /*[10]*/)
{
    gmo_aux aux; make_aux(kind, p, &aux);
    return amplitude_from_mag(kind, p, aux.nu, aux.dnu, amp, dla);
}

static int uses_mag(const int32_t *d) { return d[2 + S_M0] >= 0; }

/* descriptor check shared by the batched entry points: the paper gives a magnitude
 * relation for Sersic, ExpDisk, Ferrer and Moffat only */
static int desc_ok(int n_comp, const int32_t *desc)
{
    for (int c = 0; c < n_comp; ++c) {
        const int32_t *d = desc + c * GMO_DESC;
        if (uses_mag(d) && !(d[0] == GMO_SERSIC || d[0] == GMO_EXPDISK || d[0] == GMO_FERRER || d[0] == GMO_MOFFAT))
            return 0;
    }
    return 1;
}

/* ------------------------------------------------------------------------- */
/* convolution (reading C1) and its adjoint (C2), written as their definitions */
/*   M[i,j] = sum_{a,b} PSF[a,b] S[i-(a-h), j-(b-h)],  h=(K-1)/2, zero fill   */
/*   A[i,j] = sum_{a,b} PSF[a,b] G[i+(a-h), j+(b-h)]                          */
/* ------------------------------------------------------------------------- */
void gmo_conv2d_same(const double *S, int H, int W, const double *psf, int K, double *M)
{
    const int h = (K - 1) / 2;
    for (int i = 0; i < H; ++i)
        for (int j = 0; j < W; ++j) {
            double acc = 0.0;
            for (int a = 0; a < K; ++a) {
                int ii = i - (a - h);
                if (ii < 0 || ii >= H) continue;
                for (int b = 0; b < K; ++b) {
                    int jj = j - (b - h);
                    if (jj < 0 || jj >= W) continue;
                    acc += psf[a * K + b] * S[ii * W + jj];
                }
            }
            M[i * W + j] = acc;
        }
}

void gmo_corr2d_same(const double *G, int H, int W, const double *psf, int K, double *A)
{
    const int h = (K - 1) / 2;
    for (int i = 0; i < H; ++i)
        for (int j = 0; j < W; ++j) {
            double acc = 0.0;
            for (int a = 0; a < K; ++a) {
                int ii = i + (a - h);
                if (ii < 0 || ii >= H) continue;
                for (int b = 0; b < K; ++b) {
                    int jj = j + (b - h);
                    if (jj < 0 || jj >= W) continue;
                    acc += psf[a * K + b] * G[ii * W + jj];
                }
            }
            A[i * W + j] = acc;
        }
}

/* ------------------------------------------------------------------------- */
/* forward model of one galaxy: S (sum of convolved components), U (sum of    */
/* unconvolved components incl. sky), M = PSF (*) S + U  */
/* ------------------------------------------------------------------------- */
static void model_one(int n_comp, const int32_t *desc, int H, int W, int K, const double *psf,
                      const double *par, double *S, double *U, double *M)
{
    const int N = H * W;
    for (int k = 0; k < N; ++k) { S[k] = 0.0; U[k] = 0.0; }
    for (int c = 0; c < n_comp; ++c) {
        const int32_t *d = desc + c * GMO_DESC;
        double p[N_SLOT], dI[N_SLOT], I;
        gmo_aux aux;
        gather_params(d, par, p);
        make_aux(d[0], p, &aux);
        double *dst = is_convolved(d) ? S : U;
        for (int i = 0; i < H; ++i)
            for (int j = 0; j < W; ++j) {
                component_eval(d[0], uses_mag(d), p, &aux, pix_x(j), pix_y(i, H), &I, dI, 0);
                dst[i * W + j] += I;
            }
    }
    gmo_conv2d_same(S, H, W, psf, K, M);
    for (int k = 0; k < N; ++k) M[k] += U[k];
}

int gmo_render(int n_comp, const int32_t *desc, int n_par, int B, int H, int W, int K,
               const double *psf, int64_t psf_stride, const double *params, double *model)
{
    if (K < 1 || (K & 1) == 0) return -1;
    if (!desc_ok(n_comp, desc)) return -3;
    const int64_t N = (int64_t)H * W;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int g = 0; g < B; ++g) {
        double *S = (double *)malloc(sizeof(double) * N * 2);
        if (!S) { err = -2; continue; }
        model_one(n_comp, desc, H, W, K, psf + g * psf_stride, params + (int64_t)g * n_par,
                  S, S + N, model + g * N);
        free(S);
    }
    return err;
}

/* ------------------------------------------------------------------------- */
/* chi^2 (Eq. 18) and its analytic gradient for one galaxy             */
/*   w = mask ? 1/sigma^2 : 0  (select),  rho = D - M,  chi2 = sum w rho^2    */
/*   G = -2 w rho,  A = PSF (star) G,                                          */
/*   dchi2/dp = sum A dS/dp (convolved) + sum G dI/dp (unconvolved)            */
/* optional Gauss-Newton blocks: J = dM/dp,                            */
/*   jtj = sum w J_k J_l,  jtr = sum w J_k rho                                 */
/* ------------------------------------------------------------------------- */
static double loss_grad_one(int n_comp, const int32_t *desc, int n_par, int H, int W, int K,
                            const double *psf, const double *data, const double *sigma,
                            const uint8_t *mask, const double *par, double *grad /*[P] or NULL*/,
                            double *jtj /*[P*P] or NULL*/, double *jtr /*[P] or NULL*/)
{
    const int N = H * W;
    double *buf = (double *)malloc(sizeof(double) * (size_t)N * 6);
    double *S = buf, *U = buf + N, *M = buf + 2 * N, *G = buf + 3 * N, *A = buf + 4 * N, *wgt = buf + 5 * N;
    model_one(n_comp, desc, H, W, K, psf, par, S, U, M);
    double chi2 = 0.0;
    for (int k = 0; k < N; ++k) {
        const int used = mask ? (mask[k] != 0) : 1;
        const double w = used ? 1.0 / (sigma[k] * sigma[k]) : 0.0;
        const double rho = used ? data[k] - M[k] : 0.0;
        wgt[k] = w;
        chi2 += w * rho * rho;
        G[k] = -2.0 * w * rho;
    }
    if (grad) {
        for (int k = 0; k < n_par; ++k) grad[k] = 0.0;
        gmo_corr2d_same(G, H, W, psf, K, A);
        for (int c = 0; c < n_comp; ++c) {
            const int32_t *d = desc + c * GMO_DESC;
            double p[N_SLOT], dI[N_SLOT], I;
            gmo_aux aux;
            gather_params(d, par, p);
            make_aux(d[0], p, &aux);
            const double *seed = is_convolved(d) ? A : G;
            double acc[N_SLOT] = { 0 };
            for (int i = 0; i < H; ++i)
                for (int j = 0; j < W; ++j) {
                    component_eval(d[0], uses_mag(d), p, &aux, pix_x(j), pix_y(i, H), &I, dI, 1);
                    const double sd = seed[i * W + j];
                    for (int k = 0; k < N_SLOT; ++k) acc[k] += sd * dI[k];
                }
            for (int k = 0; k < N_SLOT; ++k)
                if (d[2 + k] >= 0) grad[d[2 + k]] += acc[k];
        }
    }
    if (jtj || jtr) {
        /* forward mode: one derivative image per parameter */
        double *J = (double *)calloc((size_t)N * n_par, sizeof(double));
        double *dS = (double *)malloc(sizeof(double) * (size_t)N * 2);
        double *dM = dS + N;
        for (int c = 0; c < n_comp; ++c) {
            const int32_t *d = desc + c * GMO_DESC;
            double p[N_SLOT], dI[N_SLOT], I;
            gmo_aux aux;
            gather_params(d, par, p);
            make_aux(d[0], p, &aux);
            for (int k = 0; k < N_SLOT; ++k) {
                const int slot = d[2 + k];
                if (slot < 0) continue;
                for (int i = 0; i < H; ++i)
                    for (int j = 0; j < W; ++j) {
                        component_eval(d[0], uses_mag(d), p, &aux, pix_x(j), pix_y(i, H), &I, dI, 1);
                        dS[i * W + j] = dI[k];
                    }
                if (is_convolved(d)) gmo_conv2d_same(dS, H, W, psf, K, dM);
                else memcpy(dM, dS, sizeof(double) * N);
                for (int px = 0; px < N; ++px) J[(size_t)slot * N + px] += dM[px];
            }
        }
        for (int k = 0; k < n_par; ++k) {
            if (jtr) {
                double s = 0.0;
                for (int px = 0; px < N; ++px) {
                    const int used = mask ? (mask[px] != 0) : 1;
                    if (used) s += wgt[px] * J[(size_t)k * N + px] * (data[px] - M[px]);
                }
                jtr[k] = s;
            }
            if (jtj)
                for (int l = 0; l < n_par; ++l) {
                    double s = 0.0;
                    for (int px = 0; px < N; ++px)
                        s += wgt[px] * J[(size_t)k * N + px] * J[(size_t)l * N + px];
                    jtj[k * n_par + l] = s;
                }
        }
        free(J); free(dS);
    }
    free(buf);
    return chi2;
}

int gmo_loss_grad(int n_comp, const int32_t *desc, int n_par, int B, int H, int W, int K,
                  const double *psf, int64_t psf_stride, const double *data, const double *sigma,
                  const uint8_t *mask, const double *params, double *chi2, double *grad,
                  double *jtj, double *jtr)
{
    if (K < 1 || (K & 1) == 0) return -1;
    if (!desc_ok(n_comp, desc)) return -3;
    const int64_t N = (int64_t)H * W;
#pragma omp parallel for schedule(dynamic, 1)
    for (int g = 0; g < B; ++g) {
        chi2[g] = loss_grad_one(n_comp, desc, n_par, H, W, K, psf + g * psf_stride,
                                data + g * N, sigma + g * N, mask ? mask + g * N : NULL,
                                params + (int64_t)g * n_par,
                                grad ? grad + (int64_t)g * n_par : NULL,
                                jtj ? jtj + (int64_t)g * n_par * n_par : NULL,
                                jtr ? jtr + (int64_t)g * n_par : NULL);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* covariance-matrix uncertainties (Sec. 5.2):                          */
/*   sigma_p = sqrt(diag[(J^T W J)^-1]) over the free parameters.              */
/* The inverse is the textbook Gauss-Jordan elimination with partial pivoting  */
/* on [A | I]; fixed parameters are left out of A and get sigma_p = 0.         */
/* returns 0, or 1 when A is singular / not finite / has a non-positive        */
/* diagonal in its inverse (sigma_p then NaN).                                 */
/* ------------------------------------------------------------------------- */
int gmo_covariance_sigma(int P, const double *jtj /*[P*P]*/, const uint8_t *free_mask, double *sigma_p /*[P]*/)
{
    int idx[64], nf = 0;
    for (int k = 0; k < P; ++k) { sigma_p[k] = 0.0; if (!free_mask || free_mask[k]) idx[nf++] = k; }
    if (nf == 0) return 0;
    long double *M = (long double *)malloc(sizeof(long double) * (size_t)nf * 2 * nf);
    const int Wd = 2 * nf;
    for (int i = 0; i < nf; ++i)
        for (int j = 0; j < nf; ++j) {
            M[i * Wd + j] = jtj[idx[i] * P + idx[j]];
            M[i * Wd + nf + j] = (i == j) ? 1.0L : 0.0L;
        }
    int bad = 0;
    for (int c = 0; c < nf && !bad; ++c) {
        int piv = c;
        for (int r = c + 1; r < nf; ++r)
            if (fabsl(M[r * Wd + c]) > fabsl(M[piv * Wd + c])) piv = r;
        if (!(fabsl(M[piv * Wd + c]) > 0.0L) || !isfinite((double)M[piv * Wd + c])) { bad = 1; break; }
        if (piv != c)
            for (int j = 0; j < Wd; ++j) { long double t = M[c * Wd + j]; M[c * Wd + j] = M[piv * Wd + j]; M[piv * Wd + j] = t; }
        const long double d = M[c * Wd + c];
        for (int j = 0; j < Wd; ++j) M[c * Wd + j] /= d;
        for (int r = 0; r < nf; ++r) {
            if (r == c) continue;
            const long double f = M[r * Wd + c];
            if (f == 0.0L) continue;
            for (int j = 0; j < Wd; ++j) M[r * Wd + j] -= f * M[c * Wd + j];
        }
    }
    for (int i = 0; i < nf; ++i) {
        const long double v = bad ? -1.0L : M[i * Wd + nf + i];
        if (!(v > 0.0L)) bad = 1;
    }
    for (int i = 0; i < nf; ++i) sigma_p[idx[i]] = bad ? NAN : (double)sqrtl(M[i * Wd + nf + i]);
    free(M);
    return bad;
}

/* ------------------------------------------------------------------------- */
/* update rule (readings O1-O5): Adam on the optimiser variable u, u = p or   */
/* log10 p, projection onto [T(lo), T(hi)] after each step.                    */
/*   g_u = dchi2/dp * dp/du   (dp/du = p ln 10 in log space)                   */
/*   m <- b1 m + (1-b1) g ; s <- b2 s + (1-b2) g^2                             */
/*   u <- u - lr decay^{t-1} [m/(1-b1^t)] / (sqrt(s/(1-b2^t)) + eps)           */
/* ------------------------------------------------------------------------- */
void gmo_adam_step(int P, double *u, const double *g_u, double *m, double *s, int t,
                   const double *lr, double lr_decay, double b1, double b2, double eps,
                   const double *ulo, const double *uhi, const uint8_t *free_mask)
{
    const double c1 = 1.0 - pow(b1, (double)t), c2 = 1.0 - pow(b2, (double)t);
    const double dec = pow(lr_decay, (double)(t - 1));
    for (int k = 0; k < P; ++k) {
        if (free_mask && !free_mask[k]) continue;
        m[k] = b1 * m[k] + (1.0 - b1) * g_u[k];
        s[k] = b2 * s[k] + (1.0 - b2) * g_u[k] * g_u[k];
        double step = lr[k] * dec * (m[k] / c1) / (sqrt(s[k] / c2) + eps);
        double un = u[k] - step;
        if (un < ulo[k]) un = ulo[k];
        if (un > uhi[k]) un = uhi[k];
        u[k] = un;
    }
}

/* fixed-iteration fit of one galaxy.  Sequence:
 *   for t = 1..n_iter: evaluate chi2_t, grad at p; stop checks; Adam update.
 *   then one last evaluation so chi2_out is chi^2 at the returned parameters.
 * status: 0 ran all iterations, 1 stopped early (|chi2_t - chi2_{t-1}| <=
 * tol chi2_t for `patience` consecutive iterations), 2 non-finite chi^2
 * (parameters put back to the last point with a finite chi^2).               */
static void fit_one(int n_comp, const int32_t *desc, int P, int H, int W, int K, const double *psf,
                    const double *data, const double *sigma, const uint8_t *mask, double *par,
                    int n_iter, double b1, double b2, double eps, double lr_decay, const double *lr,
                    const double *lo, const double *hi, const uint8_t *log10_space,
                    const uint8_t *free_mask, double tol, int patience,
                    double *chi2_out, int32_t *iters_used, int32_t *status, double *trace)
{
    double *w = (double *)calloc((size_t)P * 8, sizeof(double));
    double *u = w, *m = w + P, *s = w + 2 * P, *g = w + 3 * P, *gu = w + 4 * P,
           *ulo = w + 5 * P, *uhi = w + 6 * P, *pprev = w + 7 * P;
    const double ln10 = log(10.0);
    for (int k = 0; k < P; ++k) {
        const int lg = log10_space && log10_space[k];
        u[k] = lg ? log10(par[k]) : par[k];
        ulo[k] = lg ? (lo[k] > 0.0 ? log10(lo[k]) : -INFINITY) : lo[k];
        uhi[k] = lg ? log10(hi[k]) : hi[k];
        pprev[k] = par[k];
    }
    double chi2_prev = NAN;
    int st = 0, used = 0, calm = 0;
    for (int t = 1; t <= n_iter + 1; ++t) {
        const int last = (t == n_iter + 1);
        double chi2 = loss_grad_one(n_comp, desc, P, H, W, K, psf, data, sigma, mask, par,
                                    last ? NULL : g, NULL, NULL);
        if (trace && !last) trace[t - 1] = chi2;
        if (!isfinite(chi2)) {
            st = 2;
            if (t > 1) { for (int k = 0; k < P; ++k) par[k] = pprev[k]; }
            else chi2_prev = chi2;
            break;
        }
        if (last) { chi2_prev = chi2; break; }
        if (tol > 0.0 && t > 1) {
            if (fabs(chi2 - chi2_prev) <= tol * chi2) ++calm; else calm = 0;
            if (calm >= patience) { st = 1; chi2_prev = chi2; break; }
        }
        chi2_prev = chi2;
        for (int k = 0; k < P; ++k) {
            pprev[k] = par[k];
            const int lg = log10_space && log10_space[k];
            gu[k] = lg ? g[k] * par[k] * ln10 : g[k];
        }
        gmo_adam_step(P, u, gu, m, s, t, lr, lr_decay, b1, b2, eps, ulo, uhi, free_mask);
        for (int k = 0; k < P; ++k) {
            if (free_mask && !free_mask[k]) continue;
            const int lg = log10_space && log10_space[k];
            par[k] = lg ? pow(10.0, u[k]) : u[k];
        }
        used = t;
    }
    *chi2_out = chi2_prev;
    if (iters_used) *iters_used = used;
    if (status) *status = st;
    free(w);
}

int gmo_fit(int n_comp, const int32_t *desc, int n_par, int B, int H, int W, int K,
            const double *psf, int64_t psf_stride, const double *data, const double *sigma,
            const uint8_t *mask, double *params, int n_iter, double beta1, double beta2,
            double eps, double lr_decay, const double *lr, const double *lo, const double *hi,
            const uint8_t *log10_space, const uint8_t *free_mask, double tol, int patience,
            double *chi2_out, int32_t *iters_used, int32_t *status, double *trace /*[B,n_iter] or NULL*/)
{
    if (K < 1 || (K & 1) == 0) return -1;
    if (!desc_ok(n_comp, desc)) return -3;
    const int64_t N = (int64_t)H * W;
#pragma omp parallel for schedule(dynamic, 1)
    for (int g = 0; g < B; ++g) {
        fit_one(n_comp, desc, n_par, H, W, K, psf + g * psf_stride, data + g * N, sigma + g * N,
                mask ? mask + g * N : NULL, params + (int64_t)g * n_par, n_iter, beta1, beta2, eps,
                lr_decay, lr, lo, hi, log10_space, free_mask, tol, patience, chi2_out + g,
                iters_used ? iters_used + g : NULL, status ? status + g : NULL,
                trace ? trace + (int64_t)g * n_iter : NULL);
    }
    return 0;
}

/* ---------------------------------------------------------------------------
 * Bootstrap resampling (Sec. 5.2): "resampling with replacement each galaxy
 * image multiple times (typically 100 iterations) and refitting", then
 * sigma^2 = (1/M) sum_i (m_i - mean)^2.
 *
 * Reading B1: one resample draws n_used pixel positions, independently
 * and uniformly WITH replacement, from the n_used pixels of the galaxy that have
 * mask = 1 (row-major order); c_ij = how often pixel (i,j) was drawn, so
 * sum c = n_used and the resampled loss is chi2 = sum c_ij (D-M)^2 / sigma^2
 * (a pixel drawn twice counts twice, a pixel never drawn is ignored).
 *
 * The draws come from a counter-based generator that each side implements itself
 * from this definition (nothing is shared with the CUDA path):
 *   mix(z): z = (z ^ z>>30) * 0xBF58476D1CE4E5B9; z = (z ^ z>>27) * 0x94D049BB133111EB;
 *           return z ^ z>>31                        (the splitmix64 finaliser)
 *   z(d)  = mix(mix(mix(seed ^ (id * 0x9E3779B97F4A7C15)) + r) + d),  64-bit wrap-around
 *   k(d)  = ((z >> 32) * n_used) >> 32             (k-th used pixel), d = 0 .. n_used-1
 * with id the galaxy's identifier and r the resample index.  Pins: the published
 * splitmix64 test vectors, sum c = n_used, zero on masked pixels, P(c = 0) ~ 1/e.
 * ------------------------------------------------------------------------- */
uint64_t gmo_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* counts [N] of one galaxy and one resample; returns n_used */
int64_t gmo_bootstrap_counts(uint64_t seed, uint64_t id, uint64_t r, const uint8_t *mask /*[N] or NULL*/,
                             int64_t N, int32_t *counts /*[N]*/)
{
    int64_t n_used = 0;
    int64_t *used = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    for (int64_t i = 0; i < N; ++i) {
        counts[i] = 0;
        if (!mask || mask[i]) used[n_used++] = i;
    }
    const uint64_t base = gmo_mix64(gmo_mix64(seed ^ (id * 0x9E3779B97F4A7C15ull)) + r);
    for (int64_t d = 0; d < n_used; ++d) {
        const uint64_t z = gmo_mix64(base + (uint64_t)d);
        const uint64_t k = ((z >> 32) * (uint64_t)n_used) >> 32;
        counts[used[k]] += 1;
    }
    free(used);
    return n_used;
}

/* number of OpenMP threads the parallel loops above use */
#ifdef _OPENMP
#include <omp.h>
int gmo_num_threads(void) { return omp_get_max_threads(); }
void gmo_set_num_threads(int n) { omp_set_num_threads(n); }
#else
int gmo_num_threads(void) { return 1; }
void gmo_set_num_threads(int n) { (void)n; }
#endif
