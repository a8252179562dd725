// tl_precise.cuh -- FP64 validation mode (tl_set_precision(ctx, TL_PRECISION_FP64)).
//
// The same forward model (DESIGN.md steps a0-a8) evaluated in double precision on the device:
// plain formulas, CUDA's double math library, no MUFU, no hi/lo tricks.  About an order of
// magnitude slower than the FP32 path; it exists so that a caller can check the fast path -- or
// obtain logL to 1e-3 absolute where FP32 arithmetic cannot (rows near the best fit, DESIGN.md
// "Tolerances") -- without leaving the GPU.  Included by tinylens.cu only.
//
// Formulas and their citations are those of tl_sample.cuh / tl_consts.cuh: SIE of PAPER.md:158-160
// Eq. 12 (gamma = 2, elliptical through Eq. 10), shear of Eq. 13-14, ray-trace Eq. 1, Sersic Eq. 8-10
// with b_n from Eq. 9, bin = mean, true convolution Eq. 3, likelihood Eq. 5.
#pragma once
#include "tl_kernels.cuh"

namespace tl {

struct PreciseComp { double amp, inv_re, inv_n, bn, q, c, s, cx, cy; };
struct PreciseRow {
    double thE_sq, q, qp, c, s, cx, cy, g1, g2;        // thE_sq = theta_E sqrt(q)
    double t, A, fe;                                   // EPL: t = gamma - 1, alpha = A R^(1-t) Omega, f = (1-q)/(1+q)
    PreciseComp comp[MAX_COMP];
    int valid, epl;
};

// per row: shapes, b_n (arcsec units throughout)
__device__ inline void precise_row_setup(const float *p, int n_lens_light, int n_source, int mass_model, PreciseRow *R)
{
    const int nc = n_lens_light + n_source;
    const int LP = 7 + (mass_model == MASS_EPL ? 1 : 0);
    bool ok = true;
    for (int i = 0; i < LP + 7 * nc; ++i) ok = ok && isfinite(p[i]);
    double q = 1.0, c = 1.0, s = 0.0;
    ok = ok && (p[0] >= 0.f) && shape_from_e(p[1], p[2], &q, &c, &s);
    R->q = q; R->qp = sqrt((1.0 - q) * (1.0 + q)); R->c = c; R->s = s;
    R->thE_sq = (double)p[0] * sqrt(q);
    R->cx = p[3]; R->cy = p[4]; R->g1 = p[5]; R->g2 = p[6];
    R->epl = mass_model == MASS_EPL; R->t = 1.0; R->A = 0.0; R->fe = (1.0 - q) / (1.0 + q);
    if (R->epl) {
        ok = ok && (p[7] > 1.f) && (p[7] < 3.f);
        if (ok) {
            R->t = (double)p[7] - 1.0;
            R->A = R->thE_sq > 0.0 ? 2.0 * pow(R->thE_sq, R->t) / (1.0 + q) : 0.0;
        }
    }
    for (int k = 0; k < nc; ++k) {
        const float *sp = p + LP + 7 * k;
        PreciseComp &C = R->comp[k];
        double qs = 1.0, cs = 1.0, ss = 0.0;
        bool okc = (sp[1] > 0.f) && (sp[2] > 0.f) && shape_from_e(sp[3], sp[4], &qs, &cs, &ss);
        ok = ok && okc;
        C.amp = sp[0]; C.inv_re = okc ? 1.0 / (double)sp[1] : 1.0; C.inv_n = okc ? 1.0 / (double)sp[2] : 1.0;
        C.bn = (ok && okc) ? sersic_bn((double)sp[2]) : 1.0;
        C.q = qs; C.c = cs; C.s = ss; C.cx = sp[5]; C.cy = sp[6];
    }
    R->valid = ok ? 1 : 0;
}

__device__ inline double precise_sersic(const PreciseComp &C, double x, double y)
{
    const double dx = x - C.cx, dy = y - C.cy;
    const double x1 = dx * C.c + dy * C.s, x2 = dy * C.c - dx * C.s;
    const double rp = sqrt(C.q * x1 * x1 + x2 * x2 / C.q);
    return C.amp * exp(-C.bn * (pow(rp * C.inv_re, C.inv_n) - 1.0));
}

__device__ inline double precise_sample(const PreciseRow &R, int n_lens_light, int nc, double x, double y)
{
    double v = 0.0;
    for (int k = 0; k < n_lens_light; ++k) v += precise_sersic(R.comp[k], x, y);
    const double dx = x - R.cx, dy = y - R.cy;
    const double xp = dx * R.c + dy * R.s, yp = dy * R.c - dx * R.s;
    const double psi = sqrt(R.q * R.q * xp * xp + yp * yp);
    double axp = 0.0, ayp = 0.0;
    if (R.epl) {
        epl_alpha_f64(R.t, R.A, R.q, R.fe, xp, yp, axp, ayp);
    } else if (psi > 0.0) {
        // A(z) = atan(z)/z, H(z) = atanh(z)/z -> 1 as z -> 0 keeps q = 1 exact (G6)
        const double zx = R.qp * xp / psi, zy = R.qp * yp / psi;
        const double A = fabs(zx) < 1e-4 ? 1.0 - zx * zx / 3.0 : atan(zx) / zx;
        const double H = fabs(zy) < 1e-4 ? 1.0 + zy * zy / 3.0 : atanh(zy) / zy;
        axp = R.thE_sq * (xp / psi) * A;
        ayp = R.thE_sq * (yp / psi) * H;
    }
    const double ax = axp * R.c - ayp * R.s - (R.g1 * x + R.g2 * y);
    const double ay = axp * R.s + ayp * R.c - (R.g2 * x - R.g1 * y);
    const double bx = x - ax, by = y - ay;
    for (int k = n_lens_light; k < nc; ++k) v += precise_sersic(R.comp[k], bx, by);
    return v;
}

struct PreciseArgs {
    const float *params;      // [B][P] (chunk start)
    const float *psf;         // [n_lens][K][Kp] flipped, padded
    const float *data, *noise;
    const double *lconst;
    double *ext;              // [chunk][He][We] binned extended image, FP64
    float *logL, *images;
    int64_t row0, rows_per_lens;
    int P, ny, nx, K, Kp, h, He, We, S, n_lens_light, n_comp, edge_zero, mass_model;
    double pix_scale;
};

// one CTA per (row, slab): steps a1-a5 in FP64
__global__ void __launch_bounds__(256) precise_trace_kernel(const PreciseArgs a)
{
    __shared__ PreciseRow R;
    const int r = blockIdx.x;
    if (threadIdx.x == 0) precise_row_setup(a.params + (size_t)r * a.P, a.n_lens_light, a.n_comp - a.n_lens_light, a.mass_model, &R);
    __syncthreads();
    if (!R.valid) return;
    double *dst = a.ext + (size_t)r * a.He * a.We;
    const double s = a.pix_scale, inv_S = 1.0 / a.S;
    const int g = a.h;                                  // the extended grid always carries the halo
    for (int pix = blockIdx.y * blockDim.x + threadIdx.x; pix < a.He * a.We; pix += gridDim.y * blockDim.x) {
        const int i = pix / a.We, j = pix - i * a.We;
        double acc = 0.0;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        if (!edge) {
            const double yi = (i - g - 0.5 * (a.ny - 1)) * s, xj = (j - g - 0.5 * (a.nx - 1)) * s;
            for (int sa = 0; sa < a.S; ++sa)
                for (int sb = 0; sb < a.S; ++sb)
                    acc += precise_sample(R, a.n_lens_light, a.n_comp,
                                          xj + ((sb + 0.5) * inv_S - 0.5) * s, yi + ((sa + 0.5) * inv_S - 0.5) * s);
            acc *= inv_S * inv_S;
        }
        dst[pix] = acc;
    }
}

// one CTA per row: steps a6-a8 in FP64, fixed-shape reduction
__global__ void __launch_bounds__(256) precise_conv_kernel(const PreciseArgs a)
{
    __shared__ double red[32];
    __shared__ int valid_s;
    const int r = blockIdx.x;
    const int64_t row = a.row0 + r, lens = row / a.rows_per_lens;
    const size_t npix = (size_t)a.ny * a.nx;
    if (threadIdx.x == 0) {
        // validity only: cheap re-check (no b_n solve needed for the decision)
        const float *p = a.params + (size_t)r * a.P;
        bool ok = true;
        for (int i = 0; i < a.P; ++i) ok = ok && isfinite(p[i]);
        ok = ok && (p[0] >= 0.f) && (hypot((double)p[1], (double)p[2]) < 1.0);
        const int LP = 7 + (a.mass_model == MASS_EPL ? 1 : 0);
        if (a.mass_model == MASS_EPL) ok = ok && (p[7] > 1.f) && (p[7] < 3.f);
        for (int k = 0; k < a.n_comp; ++k) {
            const float *sp = p + LP + 7 * k;
            ok = ok && (sp[1] > 0.f) && (sp[2] > 0.f) && (hypot((double)sp[3], (double)sp[4]) < 1.0);
        }
        valid_s = ok ? 1 : 0;
    }
    __syncthreads();
    if (!valid_s) {
        if (a.logL && threadIdx.x == 0) a.logL[row] = -INFINITY;
        if (a.images) for (size_t i = threadIdx.x; i < npix; i += blockDim.x) a.images[row * npix + i] = NAN;
        return;
    }
    const double *img = a.ext + (size_t)r * a.He * a.We;
    const float *taps = a.psf + lens * a.K * a.Kp;
    double part = 0.0;
    for (int o = threadIdx.x; o < (int)npix; o += blockDim.x) {
        const int i = o / a.nx, x = o - i * a.nx;
        double m = 0.0;
        for (int ka = 0; ka < a.K; ++ka)
            for (int kb = 0; kb < a.K; ++kb)
                m += (double)taps[ka * a.Kp + kb] * img[(size_t)(i + ka) * a.We + x + kb];
        if (a.images) a.images[row * npix + o] = (float)m;
        if (a.logL) {
            const double d = (double)a.data[lens * npix + o] - m;
            const double sg = (double)a.noise[lens * npix + o];
            part += d * d / (sg * sg);
        }
    }
    if (a.logL) {
        const double chi2 = block_sum(part, red);
        if (threadIdx.x == 0) a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[lens]));
    }
}

}  // namespace tl
