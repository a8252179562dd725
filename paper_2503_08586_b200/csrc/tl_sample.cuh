// tl_sample.cuh -- per-sub-sample arithmetic: steps a2 (deflection), a3 (source light),
// a4 (lens light) of DESIGN.md.  FP32 with hi/lo constants; FP64 only in refine_beta().
//
// SIE deflection (Eq. 12 with gamma = 2 made elliptical through R_p of
// PAPER.md:143-148 Eq. 10; Kormann et al. 1994 closed form, G1), in the frame
// rotated by phi about the lens centre:
//     psi = sqrt(q^2 x'^2 + y'^2),  f = theta_E sqrt(q) / q',
//     alpha_x' = f atan(q' x' / psi),   alpha_y' = f atanh(q' y' / psi).
// External shear (PAPER.md:162 Eq. 13, :187-190 Eq. 14; G4, G5):
//     alpha_shear = -(g1 x + g2 y, g2 x - g1 y)   about the image origin.
// Ray-trace (Eq. 1): beta = theta - alpha.
// Sersic (Eq. 8): I = I_e exp(-b_n (u - 1)),  u = (R_p/r_e)^(1/n) = t^(1/2n).
#pragma once
#include "tl_consts.cuh"

namespace tl {

// ---- step a2, FP32 ---------------------------------------------------------------------
__device__ __forceinline__ void deflect_f32(const LensC &L, float X, float Y, float &bx, float &by)
{
    float dx = (X - L.cXh) - L.cXl;
    float dy = (Y - L.cYh) - L.cYl;
    // rotate into the lens frame with hi/lo cos, sin
    float xp = fmaf(dx, L.ch, fmaf(dy, L.sh, fmaf(dx, L.cl, dy * L.sl)));
    float yp = fmaf(dy, L.ch, fmaf(-dx, L.sh, fmaf(dy, L.cl, -dx * L.sl)));
    float xx = xp * xp;
    float psi2 = fmaf(L.q2h, xx, fmaf(L.q2l, xx, yp * yp));
    float psi = sqrtf(psi2);
    float nx = fmaf(L.qpl, xp, L.qph * xp);         // q' x'
    float ny = fmaf(L.qpl, yp, L.qph * yp);         // q' y'
    float at = atan2f(nx, psi);                     // psi >= 0: angle in [-pi/2, pi/2]
    float zy = psi2 > 0.f ? ny / psi : 0.f;         // |zy| <= q' < 1; alpha = 0 at psi = 0 (G6)
    float ah = atanhf(zy);
    float axp = fmaf(L.fl, at, L.fh * at);
    float ayp = fmaf(L.fl, ah, L.fh * ah);
    // rotate back
    float ax = fmaf(axp, L.ch, fmaf(-ayp, L.sh, fmaf(axp, L.cl, -ayp * L.sl)));
    float ay = fmaf(axp, L.sh, fmaf(ayp, L.ch, fmaf(axp, L.sl, ayp * L.cl)));
    // beta = theta - alpha_SIE - alpha_shear
    bx = fmaf(L.g1, X, fmaf(L.g2, Y, X - ax));
    by = fmaf(L.g2, X, fmaf(-L.g1, Y, Y - ay));
}

// ---- step a2, FP64 (selective refinement only) --------------------------------------------
__device__ __noinline__ void refine_beta(const LensC &L, float Xf, float Yf, double &bx, double &by)
{
    double X = Xf, Y = Yf;
    double dx = X - L.dcX, dy = Y - L.dcY;
    double xp = dx * L.dc + dy * L.ds;
    double yp = dy * L.dc - dx * L.ds;
    double psi = sqrt(L.dq2 * xp * xp + yp * yp);
    double axp = 0.0, ayp = 0.0;
    if (psi > 0.0) {
        axp = L.df * atan(L.dqp * xp / psi);
        ayp = L.df * atanh(L.dqp * yp / psi);
    }
    double ax = axp * L.dc - ayp * L.ds;
    double ay = axp * L.ds + ayp * L.dc;
    double g1 = L.g1, g2 = L.g2;
    bx = X - ax + (g1 * X + g2 * Y);
    by = Y - ay + (g2 * X - g1 * Y);
}

// ---- steps a3 / a4: one elliptical Sersic at offset (dx, dy) from its centre ----------------
// Returns amp * exp2(k (1 - u)); `u_out`, `t_out`, `e_out` feed the refinement test.
__device__ __forceinline__ float sersic_eval(const SersicC &C, float dx, float dy,
                                             float &t_out, float &u_out, float &e_out)
{
    float x1 = fmaf(dx, C.c, dy * C.s);
    float x2 = fmaf(dy, C.c, -dx * C.s);
    float t = fmaf(C.A * x1, x1, (C.B * x2) * x2);   // (R_p / r_e)^2
    float v = log2f(t);                              // t = 0 -> -inf -> u = 0 -> I_e e^{b_n}
    float vp = fmaf(v, C.pl, v * C.ph);
    float u = exp2f(vp);
    float arg = fmaf(-C.kh, u, C.kh) + fmaf(-C.kl, u, C.kl);
    float e = exp2f(arg);
    t_out = t; u_out = u; e_out = e;
    return C.amp * e;
}

// One sub-sample: lens light at theta, sources at beta (Eq. 2).  Already scaled
// by 1/S^2, so the caller only adds (step a5, bin = mean).
template <bool REFINE>
__device__ __forceinline__ float sample_value(const RowC &rc, int n_lens_light, int n_comp,
                                              float X, float Y)
{
    float acc = 0.f, t, u, e;
    for (int k = 0; k < n_lens_light; ++k) {
        const SersicC &C = rc.comp[k];
        acc += sersic_eval(C, (X - C.cXh) - C.cXl, (Y - C.cYh) - C.cYl, t, u, e);
    }
    float bx, by;
    deflect_f32(rc.lens, X, Y, bx, by);
    float src = 0.f;
    bool flag = false;
    for (int k = n_lens_light; k < n_comp; ++k) {
        const SersicC &C = rc.comp[k];
        src += sersic_eval(C, (bx - C.cXh) - C.cXl, (by - C.cYh) - C.cYl, t, u, e);
        float w = C.cflag * e * u;
        flag = flag || (w * w > t);
    }
    if (REFINE && flag) {
        double dbx, dby;
        refine_beta(rc.lens, X, Y, dbx, dby);
        src = 0.f;
        for (int k = n_lens_light; k < n_comp; ++k) {
            const SersicC &C = rc.comp[k];
            src += sersic_eval(C, (float)(dbx - C.dcX), (float)(dby - C.dcY), t, u, e);
        }
    }
    return acc + src;
}

}  // namespace tl
