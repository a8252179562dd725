// tl_sample.cuh -- per-sub-sample arithmetic: steps a2 (deflection), a3 (source light),
// a4 (lens light) of DESIGN.md.  FP32 with hi/lo constants; FP64 only in refine_offsets().
//
// SIE deflection (Eq. 12 with gamma = 2 made elliptical through R_p of
// PAPER.md:143-148 Eq. 10; Kormann et al. 1994 closed form, G1), in the lens frame:
//     psi = sqrt(q^2 x'^2 + y'^2),  f = theta_E sqrt(q) / q',
//     alpha_x' = f atan(q' x' / psi),   alpha_y' = f atanh(q' y' / psi).
// Both inverse functions are evaluated without range tests:
//   atan:  the angle of (psi, q'|x'|) lies in [0, thmax], thmax = atan(q'/q); rotating the
//          vector by -theta0 = -thmax/2 leaves an angle in [-theta0, theta0], |tan| <= 0.58 for
//          q >= 0.5, where a degree-5 odd minimax polynomial is exact to 5e-9;
//   atanh: z = q'|y'|/psi lies in [0, q']; the hyperbolic shift by T/2, T = atanh(q'),
//          r = (z - z0)/(1 - z z0), z0 = tanh(T/2), leaves |r| <= z0 <= 0.58 (degree-6, 4e-9).
// One MUFU.RSQ and two MUFU.RCP per sample; rows with q < 0.5 take the libdevice path.
// External shear (PAPER.md:162 Eq. 13, :187-190 Eq. 14; G4, G5) and the identity are the
// linear map N of tl_consts.cuh.  Ray-trace (Eq. 1): beta = theta - alpha.
// Sersic (Eq. 8): I = I_e exp(-b_n (u - 1)),  u = (R_p/r_e)^(1/n) = t^(1/2n),
// evaluated as amp * ex2(k (1 - ex2(p lg2 t))) with three MUFU ops.
#pragma once
#include "tl_consts.cuh"

namespace tl {

__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// atan(r) for |r| <= 0.58 (max relative error 4.6e-9 before rounding)
__device__ __forceinline__ float atan_small(float r)
{
    const float s = r * r;
    float p = 3.199305013e-02f;
    p = fmaf(p, s, -7.467620820e-02f);
    p = fmaf(p, s, 1.079487726e-01f);
    p = fmaf(p, s, -1.425360143e-01f);
    p = fmaf(p, s, 1.999849826e-01f);
    p = fmaf(p, s, -3.333331048e-01f);
    return fmaf(r * s, p, r);
}

// atanh(r) for |r| <= 0.58 (max relative error 4.3e-9 before rounding)
__device__ __forceinline__ float atanh_small(float r)
{
    const float s = r * r;
    float p = 2.593644857e-01f;
    p = fmaf(p, s, -5.470913649e-02f);
    p = fmaf(p, s, 1.322188675e-01f);
    p = fmaf(p, s, 1.043291166e-01f);
    p = fmaf(p, s, 1.434355527e-01f);
    p = fmaf(p, s, 1.999771595e-01f);
    p = fmaf(p, s, 3.333336413e-01f);
    return fmaf(r * s, p, r);
}

// Per-row constants of the pixel loop, copied from shared memory into registers once per row
// (a by-value copy also tells the compiler they cannot alias the image stores).
struct SieHot {
    float q2h, q2l, c0, s0, z0, qph, qpl, fh, fl, ft0h, ft0l, fT2h, fT2l;
    __device__ __forceinline__ explicit SieHot(const LensC &L)
        : q2h(L.q2h), q2l(L.q2l), c0(L.c0), s0(L.s0), z0(L.z0),
          qph(L.qph), qpl(L.qpl), fh(L.fh), fl(L.fl), ft0h(L.ft0h), ft0l(L.ft0l), fT2h(L.fT2h), fT2l(L.fT2l) {}
};
struct SersicHot {
    float ph, pl, kh, kl, amp, pm, nlcf;
    __device__ __forceinline__ SersicHot() {}
    __device__ __forceinline__ explicit SersicHot(const SersicC &C)
        : ph(C.ph), pl(C.pl), kh(C.kh), kl(C.kl), amp(C.amp), pm(C.pm), nlcf(C.nlcf) {}
};
struct QuadHot {
    float ah, al, b2h, b2l, cch, ccl, oxh, oxl, oyh, oyl;
    __device__ __forceinline__ QuadHot() {}
    __device__ __forceinline__ explicit QuadHot(const SersicC &C)
        : ah(C.ah), al(C.al), b2h(C.b2h), b2l(C.b2l), cch(C.cch), ccl(C.ccl),
          oxh(C.cXh), oxl(C.cXl), oyh(C.cYh), oyl(C.cYl) {}
};

// ---- step a2: SIE deflection in the lens frame (q >= 0.5) ------------------------------------
__device__ __forceinline__ void sie_alpha(const SieHot &L, float xp, float yp, float &axp, float &ayp)
{
    const float xx = xp * xp;
    // the 1e-30 keeps psi > 0: at the lens centre both angles come out as 0 +- rounding (G6)
    const float psi2 = fmaf(L.q2h, xx, fmaf(L.q2l, xx, fmaf(yp, yp, 1e-30f)));
    const float psi = psi2 * mufu_rsq(psi2);
    // q'|x'|, q'|y'| with the hi/lo q'
    const float ax = fabsf(xp), ay = fabsf(yp);
    const float Ax = fmaf(ax, L.qph, ax * L.qpl), Ay = fmaf(ay, L.qph, ay * L.qpl);
    // atan: rotate (psi, q'|x'|) by -theta0 (c0, s0 need not be normalised: only n2/d2 matters)
    const float d2 = fmaf(Ax, L.s0, psi * L.c0);
    const float n2 = fmaf(Ax, L.c0, -psi * L.s0);
    const float pa = atan_small(n2 * mufu_rcp(d2));
    const float a1 = fmaf(L.fh, pa, fmaf(L.fl, pa, L.ft0l)) + L.ft0h;       // low terms first: unbiased
    // atanh: hyperbolic shift of z = q'|y'|/psi by z0:  r = (z - z0) / (1 - z z0)
    const float num = fmaf(-L.z0, psi, Ay);
    const float den = fmaf(-L.z0, Ay, psi);
    const float ph = atanh_small(num * mufu_rcp(den));
    const float a2 = fmaf(L.fh, ph, fmaf(L.fl, ph, L.fT2l)) + L.fT2h;
    axp = copysignf(a1, xp);
    ayp = copysignf(a2, yp);
}

// strongly flattened lenses (q < 0.5): libdevice inverse functions, out of line
static __device__ __noinline__ void sie_alpha_slow(const LensC &L, float xp, float yp, float &axp, float &ayp)
{
    const float xx = xp * xp;
    const float psi2 = fmaf(L.q2h, xx, fmaf(L.q2l, xx, yp * yp));
    const float psi = sqrtf(psi2);
    const float nx = fmaf(L.qph, xp, L.qpl * xp), ny = fmaf(L.qph, yp, L.qpl * yp);
    const float at = atan2f(nx, psi);
    const float ah = atanhf(psi2 > 0.f ? ny / psi : 0.f);
    axp = fmaf(L.fh, at, L.fl * at);
    ayp = fmaf(L.fh, ah, L.fl * ah);
}

// ---- step a2, EPL (mass_model = MASS_EPL): elliptical power law with free slope ---------------
// PAPER.md:158 Eq. 12, kappa = (3-gamma)/2 (theta_E/R)^(gamma-1) on the ellipses of Eq. 10
// (G22), deflection by the angular series of Tessore & Metcalf (2015): with
// t = gamma - 1, R = sqrt(q^2 x'^2 + y'^2), e^{i phi} = (q x' + i y')/R, b = theta_E sqrt(q),
// f = (1-q)/(1+q),
//     alpha_x' + i alpha_y' = 2b/(1+q) (R/b)^(1-t) e^{i phi} sum_{n>=0} a_n e^{2 i n phi},
//     a_0 = 1,  a_n = a_{n-1} (-f) (2n - (2-t)) / (2n + (2-t)).
// The a_n come from the prologue (FP64, rounded once).  They are real, so the complex sum is a
// cosine and a sine series in theta = 2 phi, and ONE Clenshaw recurrence serves both:
//     b_k = a_k + 2 cos(theta) b_{k+1} - b_{k+2}   (k = N .. 0,  b_{N+1} = b_{N+2} = 0),
//     sum a_n cos(n theta) = b_0 - b_1 cos(theta),   sum a_n sin(n theta) = b_1 sin(theta),
// two instructions per term (a complex Horner step takes four).  The radial factor is
//     (R^2/b^2)^kappa = 2^(kappa lg2 v),  kappa = (1-t)/2,  v = R^2/b^2 = m 2^e:
// lg2 v = e + lg2 m with MUFU.LG2 on the mantissa only (absolute error 2^-22, then scaled by
// |kappa| <= 1/2), and 2^x by splitting off the integer part and a degree-6 polynomial on
// [-1/2, 1/2] (9e-9) -- MUFU.EX2 alone would carry a 3e-8 bias into every deflection.
struct EplHot {
    float q2h, q2l, qh, ql, kh, kl, a0h, a0l, invb2;
    int nterm;
    __device__ __forceinline__ explicit EplHot(const LensC &L)
        : q2h(L.q2h), q2l(L.q2l), qh(L.eqh), ql(L.eql), kh(L.ekh), kl(L.ekl), a0h(L.ea0h), a0l(L.ea0l),
          invb2(L.einvb2), nterm(L.enterm) {}
};

__device__ __forceinline__ float exp2_poly(float x)      // 2^x, |x| <= 100
{
    // round to nearest integer with the 1.5 * 2^23 trick: no conversion instructions (F2I / I2F /
    // FRND issue at a quarter of the FMA rate), and the integer sits in the low mantissa bits
    const float big = x + 12582912.f;
    const float r = x - (big - 12582912.f);               // exact, |r| <= 1/2
    float p = 1.545316336e-04f;
    p = fmaf(p, r, 1.339086331e-03f);
    p = fmaf(p, r, 9.618083015e-03f);
    p = fmaf(p, r, 5.550356954e-02f);
    p = fmaf(p, r, 2.402265072e-01f);
    p = fmaf(p, r, 6.931471825e-01f);
    p = fmaf(p, r, 1.0f);                                 // in [0.707, 1.415]
    return __int_as_float(__float_as_int(p) + (__float_as_int(big) << 23));
}

// NS sub-samples at once: the coefficient loads and the loop control of the Horner recurrence are
// shared by the NS independent chains.
template <int NS>
__device__ __forceinline__ void epl_alpha_vec(const EplHot &L, const float *coef, const float (&xp)[NS], const float (&yp)[NS],
                                              float (&axp)[NS], float (&ayp)[NS])
{
    float c2[NS], s2[NS], pc[NS], ps[NS], tc[NS], b1[NS], b2[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const float xx = xp[s] * xp[s];
        const float psi2 = fmaf(L.q2h, xx, fmaf(L.q2l, xx, fmaf(yp[s], yp[s], 1e-30f)));   // R^2 (> 0, G6)
        const float rinv = mufu_rsq(psi2);
        const float cph = fmaf(xp[s], L.qh, xp[s] * L.ql) * rinv, sph = yp[s] * rinv;       // e^{i phi}
        c2[s] = (cph - sph) * (cph + sph); s2[s] = 2.f * cph * sph;                         // w = e^{2 i phi}
        // radial factor 2 b/(1+q) (R^2/b^2)^kappa; exponent and mantissa of v taken apart with
        // integer ops (e = biased exponent - 127 through the 2^23 trick, again no conversion)
        const int vb = __float_as_int(psi2 * L.invb2);
        const float ef = __int_as_float((vb >> 23) | 0x4b000000) - 8388735.f;
        const float lm = mufu_lg2(__int_as_float((vb & 0x007fffff) | 0x3f800000));          // mantissa in [1, 2)
        float arg = fmaf(ef, L.kh, fmaf(lm, L.kh, (ef + lm) * L.kl));
        arg = fminf(fmaxf(arg, -100.f), 100.f);
        const float pw = exp2_poly(arg);
        const float P = fmaf(pw, L.a0h, pw * L.a0l);
        pc[s] = P * cph; ps[s] = P * sph;
        tc[s] = 2.f * c2[s]; b1[s] = 0.f; b2[s] = 0.f;
    }
    // Clenshaw, two terms per trip (nterm is even): no register moves, one LDS.64 of coefficients
    for (int n = L.nterm; n >= 2; n -= 2) {
        const float2 cf = *reinterpret_cast<const float2 *>(coef + n - 2);                  // a_{n-1}, a_n
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            b2[s] = fmaf(tc[s], b1[s], cf.y) - b2[s];                                       // b_n
            b1[s] = fmaf(tc[s], b2[s], cf.x) - b1[s];                                       // b_{n-1}
        }
    }
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const float b0 = fmaf(tc[s], b1[s], 1.f) - b2[s];                                   // a_0 = 1
        const float sr = fmaf(-c2[s], b1[s], b0), si = s2[s] * b1[s];
        axp[s] = fmaf(pc[s], sr, -ps[s] * si);
        ayp[s] = fmaf(pc[s], si, ps[s] * sr);
    }
}

__device__ __forceinline__ void epl_alpha(const EplHot &L, const float *coef, float xp, float yp, float &axp, float &ayp)
{
    const float x1[1] = {xp}, y1[1] = {yp};
    float a1[1], b1[1];
    epl_alpha_vec<1>(L, coef, x1, y1, a1, b1);
    axp = a1[0]; ayp = b1[0];
}

// The same in FP64 (series summed forward until it has converged): selective refinement, rows
// whose series needs more than EPL_TERMS terms (q < 0.35), and the FP64 validation mode.
__device__ inline void epl_alpha_f64(double t, double A, double q, double fe, double xp, double yp,
                                     double &axp, double &ayp)
{
    const double R2 = q * q * xp * xp + yp * yp;
    axp = 0.0; ayp = 0.0;
    if (!(R2 > 0.0) || A == 0.0) return;
    const double rinv = 1.0 / sqrt(R2);
    const double cph = q * xp * rinv, sph = yp * rinv;
    const double c2 = (cph - sph) * (cph + sph), s2 = 2.0 * cph * sph;
    const double s2t = 2.0 - t;
    double tr = cph, ti = sph, sr = cph, si = sph;
    for (int n = 1; n < 20000; ++n) {
        const double fac = -fe * (2.0 * n - s2t) / (2.0 * n + s2t);
        const double nr = fac * (tr * c2 - ti * s2), ni = fac * (tr * s2 + ti * c2);
        tr = nr; ti = ni;
        sr += tr; si += ti;
        if (fabs(tr) + fabs(ti) < 1e-17) break;
    }
    const double P = A * exp(0.5 * (1.0 - t) * log(R2));
    axp = P * sr; ayp = P * si;
}

// FP64 with the prologue's coefficient table (rows on the FP32 series path, mode 2): the same
// Clenshaw recurrence as epl_alpha_vec over the table continued to 1e-16, no divisions.
__device__ inline void epl_alpha_f64_tab(const LensC &L, double xp, double yp, double &axp, double &ayp)
{
    const double q = L.dq;
    const double R2 = q * q * xp * xp + yp * yp;
    axp = 0.0; ayp = 0.0;
    if (!(R2 > 0.0) || L.dA == 0.0) return;
    const double rinv = 1.0 / sqrt(R2);
    const double cph = q * xp * rinv, sph = yp * rinv;
    const double c2 = (cph - sph) * (cph + sph), s2 = 2.0 * cph * sph, tc = 2.0 * c2;
    double b1 = 0.0, b2 = 0.0;
    for (int n = L.ednterm; n >= 2; n -= 2) {
        b2 = fma(tc, b1, L.edcoef[n - 1]) - b2;
        b1 = fma(tc, b2, L.edcoef[n - 2]) - b1;
    }
    const double b0 = fma(tc, b1, 1.0) - b2;
    const double sr = b0 - c2 * b1, si = s2 * b1;
    const double P = L.dA * exp(0.5 * (1.0 - L.dt) * log(R2));
    axp = P * (cph * sr - sph * si);
    ayp = P * (cph * si + sph * sr);
}

static __device__ __noinline__ void epl_alpha_slow(const LensC &L, float xp, float yp, float &axp, float &ayp)
{
    double ax, ay;
    epl_alpha_f64(L.dt, L.dA, L.dq, L.dfe, (double)xp, (double)yp, ax, ay);
    axp = (float)ax; ayp = (float)ay;
}

// ---- steps a3 / a4: Sersic value from t = (R_p/r_e)^2 -----------------------------------------
// Returns 2^(k (1 - u)), u = t^(1/2n) (the caller multiplies by amp).  `flag` is set when the
// sample needs the FP64 refinement (meaningful for sources only; see tl_consts.cuh).
__device__ __forceinline__ float sersic_from_t(const SersicHot &C, float t, bool &flag)
{
    const float v = mufu_lg2(t);                     // t = 0 -> -inf -> u = 0 -> I_e e^{b_n}
    const float vp = fmaf(v, C.ph, v * C.pl);
    const float u = mufu_ex2(vp);
    const float arg = fmaf(-C.kh, u, fmaf(-C.kl, u, C.kl)) + C.kh;          // K (1 - u), low terms first
    flag = fmaf(v, C.pm, arg) > C.nlcf;
    return mufu_ex2(arg);
}

__device__ __forceinline__ float quad_form(const QuadHot &C, float x, float y)
{
    const float w = fmaf(C.ah, x, fmaf(C.b2h, y, fmaf(C.al, x, C.b2l * y)));
    return fmaf(x, w, fmaf(C.cch * y, y, (C.ccl * y) * y));
}

// ---- step a2 in FP64 (selective refinement only): lens-frame offset R^T (beta - s) ----------
template <int MASS>
__device__ __forceinline__ void refine_offsets(const LensC &L, const SersicC &C, float Xf, float Yf,
                                               float &xi, float &eta)
{
    const double X = Xf, Y = Yf;
    const double dx = X - L.dcX, dy = Y - L.dcY;
    const double xp = dx * L.dc + dy * L.ds;
    const double yp = dy * L.dc - dx * L.ds;
    const double psi = sqrt(L.dq2 * xp * xp + yp * yp);
    double axp = 0.0, ayp = 0.0;
    if (MASS == MASS_EPL) {
        if (L.mode == 2) epl_alpha_f64_tab(L, xp, yp, axp, ayp);
        else epl_alpha_f64(L.dt, L.dA, L.dq, L.dfe, xp, yp, axp, ayp);
    } else if (psi > 0.0) {
        axp = L.df * atan(L.dqp * xp / psi);
        ayp = L.df * atanh(L.dqp * yp / psi);
    }
    const double ax = axp * L.dc - ayp * L.ds;
    const double ay = axp * L.ds + ayp * L.dc;
    const double bx = X - ax + (L.dg1 * X + L.dg2 * Y) - C.dcX;      // beta - s, image frame
    const double by = Y - ay + (L.dg2 * X - L.dg1 * Y) - C.dcY;
    xi = (float)(bx * L.dc + by * L.ds);
    eta = (float)(by * L.dc - bx * L.ds);
}

// Source light of one sub-sample with the ray-trace redone in FP64 (rare, out of line).
template <int MASS>
static __device__ __noinline__ float refined_source_light(const RowC &rc, int k0, int k1, float X, float Y)
{
    float src = 0.f;
    for (int k = k0; k < k1; ++k) {
        const SersicC &C = rc.comp[k];
        float xi, eta;
        refine_offsets<MASS>(rc.lens, C, X, Y, xi, eta);
        QuadHot Q(C);
        Q.oxh = Q.oxl = Q.oyh = Q.oyl = 0.f;
        bool fl;
        src = fmaf(C.amp, sersic_from_t(SersicHot(C), quad_form(Q, xi, eta), fl), src);
    }
    return src;
}

// Same for one source component k only (linear-amplitude mode keeps the components apart).
template <int MASS>
static __device__ __noinline__ float refined_source_light_k(const RowC &rc, int k, float X, float Y)
{
    return refined_source_light<MASS>(rc, k, k + 1, X, Y);
}

}  // namespace tl
