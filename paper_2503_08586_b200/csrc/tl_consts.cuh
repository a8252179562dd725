// tl_consts.cuh -- per-parameter-row derived constants (step a0 of DESIGN.md) and the FP64
// prologue kernel that fills them.
//
// One thread per (row, slot): slot 0 = SIE + shear, slots 1.. = Sersic components.  All of it
// is FP64 and runs once per row; the pixel loop receives the sensitive constants as
// hi + lo float pairs so that their FP32 rounding (a *coherent* error over the whole image)
// never reaches logL.  A pair is always applied as
//     fmaf(x, c_hi, x * c_lo [+ small constant])
// -- the small term first, the large product inside the FMA -- so that the sum is rounded
// once and without bias; the other order, fmaf(x, c_lo, x * c_hi), rounds the large product
// first and then always loses the low term (it is below half an ulp).
//
// Units: positions are carried in "u-units", u = pix_scale / (2 S) arcsec, in which every
// sub-sample coordinate is an odd integer (exact in FP32).  The SIE deflection is homogeneous
// of degree 0 in position and the shear is linear, so only the constants change.
//
// Frames: the ray-trace works in the LENS frame (rotated by phi about the lens centre),
//     (x', y') = R^T (theta - c),   R = [[cos phi, -sin phi], [sin phi, cos phi]],
// and never rotates back: with Gamma = [[g1, g2], [g2, -g1]] (alpha_shear = -Gamma theta),
//     R^T beta = N (theta - c) + D0 - alpha',   N = R^T (I + Gamma),  D0 = N c,
// where alpha' = (alpha_x', alpha_y') is the SIE deflection in its own frame.  Every source
// Sersic is expressed as a quadratic form in the lens-frame offset R^T (beta - s).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "tl_bn_table.h"

namespace tl {

constexpr int MAX_COMP = 4;          // n_lens_light (<= 1; MGE mode: <= 2 sets) + n_source (<= 2)
constexpr int MASS_SIE = 0, MASS_EPL = 1;          // tl_config.mass_model
constexpr int EPL_TERMS = 24;        // angular-series terms of the FP32 EPL path (rows needing more: FP64)
constexpr int EPL_TERMS64 = 64;      // terms kept in FP64 for the selective refinement (remainder < 1e-16)

struct LensC {                       // SIE + external shear
    float cXa, cYa;                  // centre rounded to 2^-8 u-units: X - cXa is exact
    float pcC, psC, qcC, qsC;        // -(c - cXa) * cos/sin: the sub-grid remainder of the centre
    float uC, u2C, vL, v2L;          //   ... and its image under N, plus the low part of D0
    float ch, cl, sh, sl;            // cos(phi), sin(phi)
    float n11h, n11l, n12h, n12l;    // N = R^T (I + Gamma)
    float n21h, n21l, n22h, n22l;
    float d1h, d2h;                  // high part of D0 = N c - R^T s_1
    float q2h, q2l;                  // q^2
    float qph, qpl;                  // q' = sqrt(1 - q^2)  (clamped at 1e-6)
    float c0, s0;                    // ~cos/sin(atan(q'/q)/2) as floats; theta0 := atan2(s0, c0) exactly
    float z0;                        // ~tanh(atanh(q')/2) as a float;    T0 := atanh(z0) exactly
    float pad0;
    float fh, fl;                    // f = theta_E sqrt(q) / q', u-units
    float ft0h, ft0l;                // f theta0
    float fT2h, fT2l;                // f T0
    int32_t mode;                    // SIE  0: polynomial path (q >= 0.5), 1: libdevice path
                                     // EPL  2: FP32 series (<= EPL_TERMS terms), 3: FP64 series
    int32_t valid;
    double dcX, dcY, dc, ds, dq2, dqp, df, dg1, dg2;   // FP64 copies for the selective refinement
    // ---- elliptical power law (mass_model = MASS_EPL only; tl_sample.cuh "EPL") ----
    double dt, dA, dq, dfe;          // t = gamma - 1;  alpha_u = A R_u^(1-t) Omega;  q;  f = (1-q)/(1+q)
    float eqh, eql;                  // q
    float ekh, ekl;                  // kappa = (1 - t) / 2
    float ea0h, ea0l;                // alpha at R = b:  2 b_u / (1 + q)
    float einvb2;                    // 1 / b_u^2,  b = theta_E sqrt(q)
    int32_t enterm;                  // N (even): Omega = e^{i phi} (1 + sum_{n=1..N} a_n e^{2 i n phi})
    double edcoef[EPL_TERMS64];      // a_n in FP64, continued until |a_n| < 1e-16 (selective refinement)
    int32_t ednterm, epad[3];        // number of FP64 terms (even)
    alignas(8) float ecoef[EPL_TERMS];          // a_n = prod_{k<=n} -f (2k - (2-t)) / (2k + (2-t)),  ecoef[n-1] = a_n
};

struct SersicC {                     // one elliptical Sersic component
    // lens light: centre in the image frame (u-units); source: R^T (s - s_first) in the lens frame
    float cXh, cXl, cYh, cYl;
    // quadratic form t = (R_p / r_e)^2 = a x^2 + b2 x y + cc y^2 in the frame of the offsets
    float ah, al, b2h, b2l, cch, ccl;
    float ph, pl;                    // 1 / (2 n)
    float kh, kl;                    // b_n log2(e)
    float amp;                       // I_e / S^2
    float nlcf;                      // -log2 of the refinement criterion constant (sources), else +1e30
    float pm;                        // 1/(2n) - 1/2
    int32_t valid;
    double dcX, dcY;                 // image-frame centre (u-units), FP64, for the refinement
};

struct alignas(16) RowC {
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
    int mass_model, lens_np;         // MASS_SIE / MASS_EPL; floats of the lens block (7, or 8 with the slope)
    double inv_u;                    // 2 S / pix_scale   (u-units per arcsec)
    double fov_half;                 // arcsec, half the extended field of view
    double refine_tau;               // refinement threshold in units of sigma_min
    // small-batch path: what a cudaMemsetAsync used to do, folded into this launch (one API call less on
    // a path whose cost is host-side latency): work-queue / band counters, and the pitch padding of the
    // binned images (read by zero-padded taps only, but it must be finite)
    int *zero_words; int n_zero_words;
    float *pad_ext; int pad_rows, pad_pitch, pad_We;     // pad_rows = B * He image rows of pad_pitch floats
    int unit_amp;                    // linear-amplitude mode: every I_e is taken as 1
    int mge;                         // MGE mode (tl_loglike_mge_batch): of the lens-light block only e1, e2, cx, cy are
                                     // read; its quadratic form becomes t = R_p^2 in arcsec^2 (r_e := 1, n := 1);
                                     // component order in RowC: sources first, then the Gaussian set's shape
};

// ---- b_n of PAPER.md:139 Eq. 9:  P(2n, b_n) = 1/2 ---------------------------------------
// Safeguarded Newton on the regularised lower incomplete gamma function, evaluated with its
// power series (the root lies below a = 2n, where the series converges geometrically).
__device__ inline double gamma_p_series(double a, double x, double *prefactor)
{
    // P(a,x) = x^a e^-x / Gamma(a+1) * sum_{k>=0} x^k / ((a+1)...(a+k))
    // eight terms per trip: the eight divisions are independent of the running product and
    // pipeline, only the multiply-add chain is serial (the prologue is one thread per component
    // and sits on the critical path of every call)
    double term = 1.0, sum = 1.0;
    for (int k0 = 1; k0 < 4000; k0 += 8) {
        double r[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) r[j] = x / (a + (double)(k0 + j));
#pragma unroll
        for (int j = 0; j < 8; ++j) { term *= r[j]; sum += term; }
        if (term < sum * 1e-17) break;
    }
    double pf = exp(a * log(x) - x - lgamma(a + 1.0));
    *prefactor = pf;
    return pf * sum;
}

// b_n from the Chebyshev table of tl_bn_table.h (n in [0.3, 15]: 2e-15 relative; Clenshaw recurrence),
// else by the iteration below.  The iterative solve drags in lgamma / exp / log and ~60 divisions --
// most of the prologue kernel's code, whose instruction-cache misses were most of a one-row call.
static __device__ __noinline__ double sersic_bn_solve(double n);
__device__ inline double sersic_bn(double n)
{
    if (!(n >= BN_N_LO && n <= BN_N_HI)) return sersic_bn_solve(n);
    const double *T = n >= BN_N_MID ? BN_PIECE0 : BN_PIECE1;
    const double x = 1.0 / n, xa = T[0], xb = T[1];
    const double y = (2.0 * x - (xa + xb)) / (xb - xa), y2 = 2.0 * y;
    double b1 = 0.0, b2 = 0.0;
    for (int k = BN_NCOEF - 1; k >= 1; --k) { const double b0 = fma(y2, b1, T[2 + k] - b2); b2 = b1; b1 = b0; }
    return (2.0 * n - 1.0 / 3.0) + (fma(y, b1, T[2]) - b2);
}

static __device__ __noinline__ double sersic_bn_solve(double n)
{
    const double a = 2.0 * n;
    double lo = 0.0, hi = INFINITY, pf;
    // start: asymptotic series (Ciotti & Bertin 1999, relative error < 1e-5 for n >= 0.36);
    // for smaller n the small-x limit P(a,x) ~ x^a / Gamma(a+1)
    double b;
    if (n >= 0.36) {
        const double r = 1.0 / n;
        b = a - 1.0 / 3.0 + r * (4.0 / 405.0 + r * (46.0 / 25515.0 + r * (131.0 / 1148175.0 - r * (2194697.0 / 30690717750.0))));
    } else {
        b = exp((lgamma(a + 1.0) + log(0.5)) / a);
    }
    for (int it = 0; it < 60; ++it) {
        const double P = gamma_p_series(a, b, &pf);
        if (P < 0.5) lo = b; else hi = b;
        const double f = P - 0.5;
        const double d1 = pf * a / b;             // dP/db   = b^(a-1) e^-b / Gamma(a)
        const double d2 = d1 * ((a - 1.0) / b - 1.0);   // d2P/db2
        // Halley step (cubic convergence: from the 1e-5 start one evaluation reaches 1e-15)
        const double newton = f / d1;
        double nb = b - newton / (1.0 - 0.5 * newton * d2 / d1);
        if (!(nb > lo && nb < hi)) nb = isinf(hi) ? 2.0 * b : 0.5 * (lo + hi);
        const double step = fabs(nb - b);
        b = nb;
        // a step below 2e-5 b leaves an error of order step^3: below 1e-14 b
        if (step <= 2e-5 * b) break;
    }
    return b;
}

__device__ inline void split2(double v, float *h, float *l)
{
    float hh = (float)v;
    *h = hh;
    *l = (float)(v - (double)hh);
}

// v > 0 as hi + lo with lo > 0 strictly: used for 1/(2n), which multiplies lg2(t) = -inf at the
// centre of a profile (t = 0): -inf * lo must be -inf, not NaN (lo = 0) or +inf (lo < 0), so that
// u = ex2(-inf) = 0 and the sample is I_e e^{b_n} (Eq. 8 at R = 0).
__device__ inline void split2_poslo(double v, float *h, float *l)
{
    float hh = (float)v;
    if (!(v - (double)hh > 0.0)) hh = __int_as_float(__float_as_int(hh) - 1);     // next float towards zero (v > 0)
    *h = hh;
    *l = (float)(v - (double)hh);
}

// Inverse of PAPER.md:152 Eq. 11 (G3): e = hypot(e1,e2), q = (1-e)/(1+e), phi = atan2(e2,e1)/2.
// cos / sin of phi in (-pi/2, pi/2] by the half-angle formulas from (cos 2phi, sin 2phi) = (e1, e2)/e,
// taking the square root of whichever of (1 +- cos 2phi)/2 does not cancel (no atan2 / sincos: their
// code was a large part of the prologue's instruction footprint).
__device__ inline bool shape_from_e(double e1, double e2, double *q, double *c, double *s)
{
    const double e = sqrt(e1 * e1 + e2 * e2);
    if (!(e < 1.0)) return false;
    *q = (1.0 - e) / (1.0 + e);
    if (!(e > 0.0)) { *c = 1.0; *s = 0.0; return true; }          // atan2(0, 0) = 0
    const double c2 = e1 / e, s2 = e2 / e;
    if (c2 >= 0.0) {
        const double cc = sqrt(0.5 * (1.0 + c2));
        *c = cc; *s = s2 / (2.0 * cc);
    } else {
        const double sa = sqrt(0.5 * (1.0 - c2));                 // |sin phi| >= 0.707
        const double ss = e2 < 0.0 ? -sa : sa;                    // phi = +pi/2 for e2 = +0 (atan2(+0, -1) = pi)
        *s = ss; *c = s2 / (2.0 * ss);
    }
    return true;
}

// the constants of one slot of one row: slot 0 = lens, slot 1 + k = Sersic component k
__device__ __forceinline__ void prologue_slot(const PrologueArgs &a, int64_t row, int slot)
{
    const float *p = a.params + row * a.P;
    RowC *rc = a.rows + row;

    // lens shape is needed by every slot (sources live in the lens frame)
    const int LP = a.lens_np;
    bool lens_ok = true;
    for (int i = 0; i < LP; ++i) lens_ok = lens_ok && isfinite(p[i]);
    double thE = p[0], q = 1.0, c = 1.0, s = 0.0;
    lens_ok = lens_ok && (thE >= 0.0);
    lens_ok = lens_ok && shape_from_e(p[1], p[2], &q, &c, &s);
    // EPL: Eq. 12 has a deflection for 1 < gamma < 3 only
    if (a.mass_model == MASS_EPL) lens_ok = lens_ok && (p[7] > 1.f) && (p[7] < 3.f);
    if (!lens_ok) { thE = 0.0; q = 1.0; c = 1.0; s = 0.0; }

    if (slot == 0) {
        LensC &L = rc->lens;             // written in place: the SIE fills only the first 232 bytes
        // q' = sqrt((1-q)(1+q)); clamped away from 0 so that f = theta_E sqrt(q)/q' stays
        // finite: for q' <= 1e-6 the exact deflection differs from the clamped one by a
        // relative O(q'^2) < 1e-12 (atan(z)/z, atanh(z)/z -> 1).
        double qp = fmax(sqrt((1.0 - q) * (1.0 + q)), 1e-6);
        double f = thE * sqrt(q) / qp * a.inv_u;
        double g1 = lens_ok ? (double)p[5] : 0.0, g2 = lens_ok ? (double)p[6] : 0.0;
        double cX = (lens_ok ? (double)p[3] : 0.0) * a.inv_u, cY = (lens_ok ? (double)p[4] : 0.0) * a.inv_u;
        double n11 = c * (1.0 + g1) + s * g2, n12 = c * g2 + s * (1.0 - g1);
        double n21 = -s * (1.0 + g1) + c * g2, n22 = -s * g2 + c * (1.0 - g1);
        // D0 = N c - R^T s_1: the first source's centre is folded into the linear map, so
        // (U + V, U2 + V2) - alpha' is directly the lens-frame offset R^T (beta - s_1)
        const float *s1 = p + LP + 7 * a.n_lens_light;
        const bool s1ok = isfinite(s1[5]) && isfinite(s1[6]);
        double s1X = (s1ok ? (double)s1[5] : 0.0) * a.inv_u, s1Y = (s1ok ? (double)s1[6] : 0.0) * a.inv_u;
        double d1 = n11 * cX + n12 * cY - (c * s1X + s * s1Y), d2 = n21 * cX + n22 * cY - (-s * s1X + c * s1Y);
        // theta0 = atan(q'/q)/2 with (cos, sin)(2 theta0) = (q, q'): half-angle formulas; z0 = tanh(atanh(q')/2)
        // = q'/(1 + q).  (Only their float roundings are used: the angles added back come from those.)
        double c0 = sqrt(0.5 * (1.0 + q)), s0 = qp / (2.0 * c0);
        double z0 = qp / (1.0 + q);
        // centre = (multiple of 2^-8) + remainder: sub-sample coordinates are odd integers, so
        // X - cXa is exact in FP32 and the remainder enters through small additive constants
        L.cXa = (float)(rint(cX * 256.0) / 256.0); L.cYa = (float)(rint(cY * 256.0) / 256.0);
        const double cXb = cX - (double)L.cXa, cYb = cY - (double)L.cYa;
        L.pcC = (float)(-cXb * c); L.psC = (float)(-cXb * s); L.qcC = (float)(-cYb * c); L.qsC = (float)(-cYb * s);
        split2(c, &L.ch, &L.cl);    split2(s, &L.sh, &L.sl);
        split2(n11, &L.n11h, &L.n11l); split2(n12, &L.n12h, &L.n12l);
        split2(n21, &L.n21h, &L.n21l); split2(n22, &L.n22h, &L.n22l);
        L.d1h = (float)d1; L.d2h = (float)d2;
        L.uC = (float)(-cXb * n11); L.u2C = (float)(-cXb * n21);
        L.vL = (float)((d1 - (double)L.d1h) - cYb * n12); L.v2L = (float)((d2 - (double)L.d2h) - cYb * n22);
        split2(q * q, &L.q2h, &L.q2l); split2(qp, &L.qph, &L.qpl);
        // The rotation / hyperbolic shift are applied with single-float constants; the angle
        // added back is the one those floats really encode, so their rounding never appears
        // as a coherent deflection error.
        L.c0 = (float)c0; L.s0 = (float)s0; L.z0 = (float)z0;
        L.pad0 = 0.f;
        const double th0_eff = atan2((double)L.s0, (double)L.c0);
        const double T0_eff = atanh((double)L.z0);
        split2(f, &L.fh, &L.fl);
        split2(f * th0_eff, &L.ft0h, &L.ft0l);
        split2(f * T0_eff, &L.fT2h, &L.fT2l);
        L.mode = (q >= 0.5) ? 0 : 1;
        L.valid = lens_ok ? 1 : 0;
        L.dcX = cX; L.dcY = cY; L.dc = c; L.ds = s; L.dq2 = q * q; L.dqp = qp; L.df = f;
        L.dg1 = g1; L.dg2 = g2;
        // ---- EPL (Eq. 12; Tessore & Metcalf 2015 angular series, G22)
        // (the EPL block of LensC is left unwritten for the SIE: nothing reads it)
        if (a.mass_model == MASS_EPL) {
            L.dq = q; L.dfe = (1.0 - q) / (1.0 + q);
            for (int n = 0; n < EPL_TERMS; ++n) L.ecoef[n] = 0.f;
            for (int n = 0; n < EPL_TERMS64; ++n) L.edcoef[n] = 0.0;
            L.ednterm = 2; L.epad[0] = L.epad[1] = L.epad[2] = 0;
            const double t = lens_ok ? (double)p[7] - 1.0 : 1.0;
            const double bu = thE * sqrt(q) * a.inv_u;                   // b = theta_E sqrt(q), u-units
            L.dt = t;
            L.dA = bu > 0.0 ? 2.0 * pow(bu, t) / (1.0 + q) : 0.0;
            split2(q, &L.eqh, &L.eql);
            split2(0.5 * (1.0 - t), &L.ekh, &L.ekl);
            split2(bu > 1e-18 ? 2.0 * bu / (1.0 + q) : 0.0, &L.ea0h, &L.ea0l);
            L.einvb2 = bu > 1e-18 ? (float)(1.0 / (bu * bu)) : 1.f;
            // a_n and the number of terms that leaves a remainder below 2e-8 (|Omega| ~ 1)
            const double fe = L.dfe, s2t = 2.0 - t;
            double an = 1.0;
            int N = 0;
            for (int n = 1; n <= EPL_TERMS + 1; ++n) {
                an *= -fe * (2.0 * n - s2t) / (2.0 * n + s2t);
                if (fabs(an) < 2e-8 * (1.0 - fe)) { N = n - 1; break; }
                if (n <= EPL_TERMS) L.ecoef[n - 1] = (float)an;
                N = n;
            }
            L.mode = (N <= EPL_TERMS) ? 2 : 3;
            if (L.mode == 2) {                                           // FP64 continuation of the same table
                double ad = 1.0;
                int N64 = 0;
                for (int n = 1; n <= EPL_TERMS64; ++n) {
                    ad *= -fe * (2.0 * n - s2t) / (2.0 * n + s2t);
                    if (fabs(ad) < 1e-16) break;
                    L.edcoef[n - 1] = ad;
                    N64 = n;
                }
                N64 = (N64 + 1) & ~1;
                L.ednterm = N64 < 2 ? 2 : N64;
            }
            N = (N + 1) & ~1;                                            // even: the recurrence takes two terms per trip
            L.enterm = N < 2 ? 2 : (N > EPL_TERMS ? EPL_TERMS : N);
        }
        return;
    }

    const int k = slot - 1;
    const bool is_lens_light = k < a.n_lens_light;
    const float *sp = p + LP + 7 * k;
    SersicC C;
    bool ok = true;
    const bool mge_shape = a.mge && is_lens_light;
    for (int i = mge_shape ? 3 : (a.unit_amp ? 1 : 0); i < 7; ++i) ok = ok && isfinite(sp[i]);
    // linear mode: unit amplitude; the row's own I_e (when usable) only scales the refinement
    // criterion, as a hint of the magnitude the solved amplitude will have
    const double Ie_hint = (isfinite(sp[0]) && fabsf(sp[0]) > 1.f) ? fabs((double)sp[0]) : 1.0;
    double Ie = a.unit_amp ? 1.0 : (double)sp[0], re = sp[1], n = sp[2], qs = 1.0, cs = 1.0, ss = 0.0;
    if (mge_shape) { Ie = 1.0; re = 1.0; n = 1.0; }
    ok = ok && (re > 0.0) && (n > 0.0);
    ok = ok && shape_from_e(sp[3], sp[4], &qs, &cs, &ss);
    if (!ok) { Ie = 0.0; re = 1.0; n = 1.0; qs = 1.0; cs = 1.0; ss = 0.0; }
    const double bn = sersic_bn(n);
    const double u_arc = 1.0 / a.inv_u;                     // arcsec per u-unit
    const double cX = (ok ? (double)sp[5] : 0.0) * a.inv_u, cY = (ok ? (double)sp[6] : 0.0) * a.inv_u;
    C.dcX = cX; C.dcY = cY;
    // Eq. 10: t = (R_p/r_e)^2 = A x1^2 + B x2^2 in the component's own frame
    const double A = qs * u_arc * u_arc / (re * re), Bq = u_arc * u_arc / (qs * re * re);
    // rotation from the frame the offsets are given in to the component frame
    double cd, sd, oX, oY;
    if (is_lens_light) { cd = cs; sd = ss; oX = cX; oY = cY; }                 // image frame
    else {                                                                      // lens frame
        cd = cs * c + ss * s; sd = ss * c - cs * s;                             // cos, sin(phi_s - phi)
        // R^T (s_k - s_1): offsets are measured from the first source (folded into D0)
        const float *s1 = p + LP + 7 * a.n_lens_light;
        const bool s1ok = isfinite(s1[5]) && isfinite(s1[6]);
        const double rX = cX - (s1ok ? (double)s1[5] : 0.0) * a.inv_u, rY = cY - (s1ok ? (double)s1[6] : 0.0) * a.inv_u;
        oX = c * rX + s * rY; oY = -s * rX + c * rY;
    }
    if (is_lens_light) {     // (multiple of 2^-8) + remainder, as for the lens centre
        C.cXh = (float)(rint(oX * 256.0) / 256.0); C.cXl = (float)(oX - (double)C.cXh);
        C.cYh = (float)(rint(oY * 256.0) / 256.0); C.cYl = (float)(oY - (double)C.cYh);
    } else {
        split2(oX, &C.cXh, &C.cXl); split2(oY, &C.cYh, &C.cYl);
    }
    split2(A * cd * cd + Bq * sd * sd, &C.ah, &C.al);
    split2(2.0 * (A - Bq) * cd * sd, &C.b2h, &C.b2l);
    split2(A * sd * sd + Bq * cd * cd, &C.cch, &C.ccl);
    split2_poslo(0.5 / n, &C.ph, &C.pl);
    split2(bn * 1.4426950408889634074, &C.kh, &C.kl);
    const double amp = Ie / (double)(a.S * a.S);
    C.amp = (float)amp;
    // Selective FP64 refinement of beta:
    // the FP32 ray-trace carries an absolute error delta_beta ~ 2^-22 (theta_E + |theta|);
    // the induced brightness error of a sample is  I (b_n/n) u delta_beta / R.  It is refined
    // when that exceeds tau * sigma_min:  (cf e u)^2 > t, i.e. in log2 (v = lg2 t, vp = v/2n,
    // arg = lg2 e):  arg + v (1/2n - 1/2) > -lg2 cf.
    C.nlcf = 1e30f;
    C.pm = (float)(0.5 / n - 0.5);
    if (!is_lens_light && ok && amp != 0.0) {
        double dbeta = 2.4e-7 * (fmax((double)p[0], 0.0) + a.fov_half);               // arcsec
        double smin = a.sigma_min[(a.row0 + row) / a.rows_per_lens];
        double cf = fabs(amp) * (a.unit_amp ? Ie_hint : 1.0) * (bn / n) * dbeta / (re * a.refine_tau * smin);
        C.nlcf = fminf(fmaxf(-__log2f((float)cf), -1e30f), 1e30f);      // a threshold: MUFU accuracy is plenty
    }
    C.valid = ok ? 1 : 0;
    // MGE mode: the sources come first (comp[0 .. n_source-1], what the NLL = 0 ray-trace kernels read)
    // and the shape of the Gaussian set after them (comp[n_source])
    rc->comp[a.mge ? (is_lens_light ? a.n_source + k : k - a.n_lens_light) : k] = C;
}

#ifdef TL_MAIN_TU
// One block = 32 rows; warp w takes slot w, w + 4, ... of them, so that the lens branch and the Sersic
// branch never share a warp (they are long FP64 chains: side by side in a warp they run one after the
// other, which was half of a one-row call's prologue).  Grid: prologue_blocks(B).
__global__ void __launch_bounds__(128) prologue_kernel(PrologueArgs a)
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // (small-batch path: see tl_kernels.cuh pdl_*)
    const int nslot = 1 + a.n_lens_light + a.n_source;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int64_t row = (int64_t)blockIdx.x * 32 + lane;
    if (a.zero_words || a.pad_ext) {
        // the idle warps of the last block first: on a one-row call the lens / Sersic warps do not wait for this
        const int64_t nthr = (int64_t)gridDim.x * blockDim.x;
        const int64_t gid = nthr - 1 - ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
        for (int64_t i = gid; i < a.n_zero_words; i += nthr) a.zero_words[i] = 0;
        const int pw = a.pad_pitch - a.pad_We;
        if (a.pad_ext && pw > 0)
            for (int64_t i = gid; i < (int64_t)a.pad_rows * pw; i += nthr)
                a.pad_ext[(i / pw) * a.pad_pitch + a.pad_We + (i % pw)] = 0.f;
    }
    if (row >= a.B) return;
    for (int slot = warp; slot < nslot; slot += nwarp) prologue_slot(a, row, slot);
}
inline unsigned prologue_blocks(int64_t B) { return (unsigned)((B + 31) / 32); }

#endif  // TL_MAIN_TU

}  // namespace tl
