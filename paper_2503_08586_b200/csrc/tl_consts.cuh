// tl_consts.cuh -- per-parameter-row derived constants (step a0 of DESIGN.md) and the FP64
// prologue kernel that fills them.
//
// One thread per (row, slot): slot 0 = SIE + shear, slots 1.. = Sersic components.  All of it
// is FP64 and runs once per row; the pixel loop receives the sensitive constants as
// hi + lo float pairs so that their FP32 rounding (a *coherent* error over the whole image)
// never reaches logL.
//
// Units: positions are carried in "u-units", u = pix_scale / (2 S) arcsec, in which every
// sub-sample coordinate is an odd integer (exact in FP32).  The SIE deflection is homogeneous
// of degree 0 in position and the shear is linear, so only the constants change.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace tl {

constexpr int MAX_COMP = 3;          // n_lens_light (<= 1) + n_source (<= 2)

struct LensC {                       // SIE + external shear
    float cXh, cXl, cYh, cYl;        // centre, u-units
    float ch, cl, sh, sl;            // cos(phi), sin(phi)
    float q2h, q2l, qph, qpl;        // q^2, q' = sqrt(1 - q^2)
    float fh, fl;                    // theta_E sqrt(q) / q', u-units
    float g1, g2;                    // shear
    double dcX, dcY, dc, ds, dq2, dqp, df;   // FP64 copies for the selective refinement
    int32_t valid, pad;
};

struct SersicC {                     // one elliptical Sersic component
    float cXh, cXl, cYh, cYl;        // centre, u-units
    float c, s;                      // cos, sin of the position angle
    float A, B;                      // q u^2 / r_e^2,  u^2 / (q r_e^2):  t = A x1^2 + B x2^2 = (R_p/r_e)^2
    float ph, pl;                    // 1 / (2 n)
    float kh, kl;                    // b_n log2(e)
    float amp;                       // I_e / S^2
    float cflag;                     // refinement criterion constant (sources only, else 0)
    int32_t valid, pad;
    double dcX, dcY;                 // FP64 centre for the refinement
};

struct RowC {
    LensC lens;
    SersicC comp[MAX_COMP];
};
static_assert(sizeof(RowC) % 16 == 0, "RowC is copied as 16-byte words");

struct PrologueArgs {
    const float *params;             // [B][P]
    RowC *rows;                      // [B]
    const float *sigma_min;          // [n_lens]
    int64_t B;                       // rows in this chunk
    int64_t row0;                    // global index of the chunk's first row
    int64_t rows_per_lens;
    int P, n_lens_light, n_source, S;
    double inv_u;                    // 2 S / pix_scale   (u-units per arcsec)
    double fov_half;                 // arcsec, half the extended field of view
    double refine_tau;               // refinement threshold in units of sigma_min
};

// ---- b_n of PAPER.md:139 Eq. 9:  P(2n, b_n) = 1/2 ---------------------------------------
// Safeguarded Newton on the regularised lower incomplete gamma function, evaluated with its
// power series (the root lies below a = 2n, where the series converges geometrically).
__device__ inline double gamma_p_series(double a, double x, double *prefactor)
{
    // P(a,x) = x^a e^-x / Gamma(a+1) * sum_{k>=0} x^k / ((a+1)...(a+k))
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 4000; ++k) {
        term *= x / (a + (double)k);
        sum += term;
        if (term < sum * 1e-17) break;
    }
    double pf = exp(a * log(x) - x - lgamma(a + 1.0));
    *prefactor = pf;
    return pf * sum;
}

__device__ inline double sersic_bn(double n)
{
    const double a = 2.0 * n;
    double lo = 0.0, hi = fmax(a, 1.0);
    double pf;
    for (int it = 0; it < 64 && gamma_p_series(a, hi, &pf) < 0.5; ++it) hi *= 2.0;
    // asymptotic start (Ciotti & Bertin 1999) where it is inside the bracket
    double b = a - 1.0 / 3.0 + 4.0 / (405.0 * n);
    if (!(b > lo && b < hi)) b = 0.5 * (lo + hi);
    for (int it = 0; it < 100; ++it) {
        double P = gamma_p_series(a, b, &pf);
        if (P < 0.5) lo = b; else hi = b;
        double dPdb = pf * a / b;                 // x^(a-1) e^-x / Gamma(a)
        double nb = b - (P - 0.5) / dPdb;
        if (!(nb > lo && nb < hi)) nb = 0.5 * (lo + hi);
        double step = fabs(nb - b);
        b = nb;
        if (step <= 4e-16 * b) break;
    }
    return b;
}

__device__ inline void split2(double v, float *h, float *l)
{
    float hh = (float)v;
    *h = hh;
    *l = (float)(v - (double)hh);
}

// Inverse of PAPER.md:152 Eq. 11 (G3): e = hypot(e1,e2), q = (1-e)/(1+e), phi = atan2(e2,e1)/2.
__device__ inline bool shape_from_e(double e1, double e2, double *q, double *c, double *s)
{
    double e = hypot(e1, e2);
    if (!(e < 1.0)) return false;
    *q = (1.0 - e) / (1.0 + e);
    double phi = 0.5 * atan2(e2, e1);
    sincos(phi, s, c);
    return true;
}

__global__ void __launch_bounds__(128) prologue_kernel(PrologueArgs a)
{
    const int nslot = 1 + a.n_lens_light + a.n_source;
    int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= a.B * nslot) return;
    int64_t row = gid / nslot;
    int slot = (int)(gid - row * nslot);
    const float *p = a.params + row * a.P;
    RowC *rc = a.rows + row;

    if (slot == 0) {
        LensC L;
        bool ok = true;
        for (int i = 0; i < 7; ++i) ok = ok && isfinite(p[i]);
        double thE = p[0], q = 1.0, c = 1.0, s = 0.0;
        ok = ok && (thE >= 0.0);
        ok = ok && shape_from_e(p[1], p[2], &q, &c, &s);
        if (!ok) { thE = 0.0; q = 1.0; c = 1.0; s = 0.0; }
        // q' = sqrt((1-q)(1+q)); clamped away from 0 so that f = theta_E sqrt(q)/q' stays
        // finite: for q' <= 1e-6 the exact deflection differs from the clamped one by a
        // relative O(q'^2) < 1e-12 (A(z), H(z) -> 1).
        double qp = fmax(sqrt((1.0 - q) * (1.0 + q)), 1e-6);
        double f = thE * sqrt(q) / qp * a.inv_u;
        double cX = (double)p[3] * a.inv_u, cY = (double)p[4] * a.inv_u;
        split2(cX, &L.cXh, &L.cXl); split2(cY, &L.cYh, &L.cYl);
        split2(c, &L.ch, &L.cl);    split2(s, &L.sh, &L.sl);
        split2(q * q, &L.q2h, &L.q2l); split2(qp, &L.qph, &L.qpl);
        split2(f, &L.fh, &L.fl);
        L.g1 = ok ? p[5] : 0.f; L.g2 = ok ? p[6] : 0.f;
        L.dcX = cX; L.dcY = cY; L.dc = c; L.ds = s; L.dq2 = q * q; L.dqp = qp; L.df = f;
        L.valid = ok ? 1 : 0; L.pad = 0;
        rc->lens = L;
        return;
    }

    const int k = slot - 1;
    const float *sp = p + 7 + 7 * k;
    SersicC C;
    bool ok = true;
    for (int i = 0; i < 7; ++i) ok = ok && isfinite(sp[i]);
    double Ie = sp[0], re = sp[1], n = sp[2], q = 1.0, c = 1.0, s = 0.0;
    ok = ok && (re > 0.0) && (n > 0.0);
    ok = ok && shape_from_e(sp[3], sp[4], &q, &c, &s);
    if (!ok) { Ie = 0.0; re = 1.0; n = 1.0; q = 1.0; c = 1.0; s = 0.0; }
    double bn = sersic_bn(n);
    double u_arc = 1.0 / a.inv_u;                     // arcsec per u-unit
    double cX = (ok ? (double)sp[5] : 0.0) * a.inv_u, cY = (ok ? (double)sp[6] : 0.0) * a.inv_u;
    split2(cX, &C.cXh, &C.cXl); split2(cY, &C.cYh, &C.cYl);
    C.c = (float)c; C.s = (float)s;
    C.A = (float)(q * u_arc * u_arc / (re * re));
    C.B = (float)(u_arc * u_arc / (q * re * re));
    split2(0.5 / n, &C.ph, &C.pl);
    split2(bn * 1.4426950408889634074, &C.kh, &C.kl);
    double amp = Ie / (double)(a.S * a.S);
    C.amp = (float)amp;
    // Selective FP64 refinement of beta:
    // the FP32 ray-trace carries an absolute error delta_beta ~ 2^-22 (theta_E + |theta|);
    // the induced brightness error of a sample is  I (b_n/n) u delta_beta / R.  It is refined
    // when that exceeds tau * sigma_min:   (cflag * e * u)^2 > t,  t = (R/r_e)^2.
    C.cflag = 0.f;
    if (k >= a.n_lens_light && ok) {
        double thE = fmax((double)p[0], 0.0);
        double dbeta = 2.4e-7 * (thE + a.fov_half);               // arcsec
        double smin = a.sigma_min[(a.row0 + row) / a.rows_per_lens];
        double thr = a.refine_tau * smin;
        double cf = fabs(amp) * (bn / n) * dbeta / (re * thr);
        C.cflag = (float)fmin(cf, 1e30);
    }
    C.valid = ok ? 1 : 0; C.pad = 0;
    C.dcX = cX; C.dcY = cY;
    rc->comp[k] = C;
}

}  // namespace tl
