// tl_dp.cuh -- the double-precision path (tl_set_precision: TL_PRECISION_FP64, and the re-evaluation
// pass of TL_PRECISION_AUTO).
//
// Why it exists (DESIGN.md 6 "Tolerances"): near the best fit  delta logL = sum_i z_i SNR_i eps_i
// with sum SNR^2 ~ 1e8, so |delta logL| <= 1e-3 needs every bright pixel to ~1e-8 relative -- below
// the resolution of an FP32 pixel value.  B200 runs FP64 FMAs at half the FP32 rate (measured: a DFMA
// costs two issue slots, `bench.py --peaks`), so the cure is the same forward model with every
// per-sample quantity in FP64 and the transcendental functions as short hand-ordered polynomials
// (accurate to ~1e-12, not to 1 ulp: that is what logL needs), instead of CUDA's double libm
// (tl_precise.cuh, ~4x slower):
//   log2 t   exponent / mantissa taken apart with integer instructions, a 129-entry table of
//            {1/c_i, log2 c_i} in shared memory, r = m/c_i - 1 by one FMA, degree-4 polynomial
//   2^x      magic-number rounding to 1/32, 32-entry table of 2^(j/32), degree-4 polynomial, the
//            integer part added to the exponent field
//   1/x, 1/sqrt(x)   MUFU.RCP64H / MUFU.RSQ64H seed (1e-6) + one Newton step (1e-12)
//   atan     after the per-row rotation of tl_sample.cuh (|tan| <= 0.58 for q >= 0.5), degree-10
//            polynomial in r^2
//   atanh    (1/2) ln((psi + A)/(psi - A)) through log2 (no range restriction)
// No float <-> double conversions in the sample loop (F2F issues at 1/8 rate).  Same formulas and
// citations as tl_sample.cuh / tl_consts.cuh: SIE of PAPER.md:158-160 Eq. 12 (gamma = 2, elliptical
// through Eq. 10; G1), shear Eq. 13-14, ray-trace Eq. 1, Sersic Eq. 8-10 with b_n of Eq. 9, bin =
// mean, true convolution Eq. 3, likelihood Eq. 5.
//
// Kernels (one stream, no host sync):
//   prologue_dp_kernel   per row: RowD (FP64 constants; b_n by the Halley solve of tl_consts.cuh)
//   trace_dp_kernel      one warp per (row, tile of 32 extended pixels): steps a1-a5 -> binned
//                        extended image, FP64, in global memory (0.23 MB per row on configs[1]:
//                        1 GB per 4096-row call against 12 ms of arithmetic)
//   conv_dp_kernel       one CTA per (row, band of output rows): FP64 direct convolution of 1 x 8
//                        strips from shared memory, chi^2 of the band -> partial[row][band]
//   finalize_dp_kernel   fixed-order sum of the band partials -> logL
// Rows can be addressed through an index list whose length lives in device memory (AUTO mode).
#pragma once
#include "tl_kernels.cuh"
#include "tl_dp_tables.h"

namespace tl {

struct CompD {
    double a, b2, cc;            // t = (R_p/r_e)^2 = a x^2 + b2 x y + cc y^2 in the frame of the offsets (arcsec)
    double ox, oy;               // lens light: centre (image frame); source k: R^T (s_k - s_first) (lens frame;
                                 // rows without any deflection: s_k itself, the lens frame being the identity)
    double p, K, amp;            // 1/(2n), b_n log2(e), I_e / S^2
    int valid, pad;
};
struct RowD {
    double cx, cy, c, s;         // lens centre (arcsec), cos / sin phi
    double n11, n12, n21, n22;   // N = R^T (I + Gamma)
    double d1, d2;               // N c - R^T s_first, folded so that N (theta - c) + d - alpha' = R^T (beta - s_first)
    double q2, qp, f;            // q^2, q' = sqrt(1 - q^2) (clamped at 1e-9), f = theta_E sqrt(q) / q'
    double c0, s0, fth0;         // rotation by theta0 = atan(q'/q)/2; f theta0
    double fl2;                  // f ln(2) / 2:  f atanh(z) = fl2 log2((1+z)/(1-z))
    double g1, g2, thE_sq, q;    // slow path (q < 0.5) and EPL
    double t, A, fe;             // EPL: t = gamma - 1, alpha = A R^(1-t) Omega, f = (1-q)/(1+q)
    int mode;                    // 0: polynomial SIE, 1: libm SIE (q < 0.5), 2: EPL (FP64 series)
    int valid;
    CompD comp[MAX_COMP];
};

struct DpArgs {
    const float *params;         // [B][P] of the whole call
    RowD *rows;                  // [chunk]
    const int *row_index;        // [chunk] global row of chunk row r, or null (global row = row0 + r)
    const int *n_rows_dev;       // length of the whole index list, in device memory, or null (then n_rows)
    int n_rows;                  // rows of this chunk (with n_rows_dev: the most it can hold)
    int list_offset;             // first entry of row_index this chunk serves
    int64_t row0, rows_per_lens;
    const float *psf;            // [n_lens][K][Kp] flipped, padded (FP32 as given)
    const float *data;           // [n_lens][ny][nx]
    const double *wgt64;         // [n_lens][ny][nx]  1 / sigma^2 in FP64
    const double *lconst;
    double *ext;                 // [chunk][He][Wp] binned extended images
    double *partial;             // [chunk][n_bands]
    float *logL, *images;
    // linear-amplitude mode (tl_loglike_linear_batch in FP64): the components are kept apart
    int lin;                     // 1: ext is [chunk][n_comp][He][Wp], unit amplitudes; conv writes m64
    double *m64;                 // [chunk][n_comp][ny][nx] blurred unit-amplitude component images (columns of M)
    float *amps;                 // [B][n_comp] or null
    // MGE mode in FP64 (tl_loglike_mge_batch under TL_PRECISION_FP64): RowD holds the sources first, then the
    // shapes of the Gaussian sets (r_e := 1: t = R_p^2 in arcsec^2); ext / m64 have ext_nc = n_gauss + n_source
    // components per row, the ray-traced sources from slot ext_k0 = n_gauss on
    int mge, ext_nc, ext_k0, n_gauss, n_source;
    const double *mge_c;         // [n_gauss] log2(e) / (2 sigma_k^2), FP64
    const int *mge_set;          // [n_gauss] set of Gaussian k
    int P, ny, nx, K, Kp, h, He, We, Wp, S, n_lens_light, n_comp, edge_zero, mass_model, lens_np;
    int band_rows, n_bands;
    int CW, CH, tiles_x, tiles_y;
    double u;                    // arcsec per u-unit: pix_scale / (2 S)
};

__device__ __forceinline__ int dp_n_rows(const DpArgs &a)
{
    if (!a.n_rows_dev) return a.n_rows;
    const int left = *a.n_rows_dev - a.list_offset;
    return left < 0 ? 0 : (left < a.n_rows ? left : a.n_rows);
}
__device__ __forceinline__ int64_t dp_row(const DpArgs &a, int r)
{
    return a.row_index ? (int64_t)a.row_index[a.list_offset + r] : a.row0 + r;
}

__device__ __forceinline__ double dp_rcp(double x)       // 1/x to 1e-12 (x normal, finite)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return fma(r, fma(-x, r, 1.0), r);
}
__device__ __forceinline__ double dp_rsqrt(double x)     // 1/sqrt(x) to 1.3e-12
{
    double q;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(q) : "d"(x));
    return fma(0.5 * q, fma(-x * q, q, 1.0), q);
}
// num / den to ~1e-16 (seed, one Newton step, one residual correction)
__device__ __forceinline__ double dp_div(double num, double den)
{
    const double rc = dp_rcp(den);
    const double q0 = num * rc;
    return fma(rc, fma(-den, q0, num), q0);
}

// The tables live in shared memory and are read through 32-bit shared-window addresses computed
// once per kernel (a generic pointer makes the compiler rebuild the window base -- S2R, LEA --
// next to every table load).
struct DpTabs { unsigned ltab, etab; };
__device__ __forceinline__ double2 lds_f64x2(unsigned addr)
{
    double2 v;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds_f64(unsigned addr)
{
    double v;
    asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// log2 t for t >= 0 (t = 0 gives -1023; denormals are not distinguished from 0)
__device__ __forceinline__ double dp_log2(double t, const DpTabs &tb_)
{
    const int hi = __double2hiint(t), lo = __double2loint(t);
    const int e = (hi >> 20) - 1023;
    const int i16 = (((hi >> 9) & 0x7f8) + 8) & 0xff0;              // 16 round((m - 1) 128), entries 0 .. 128
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
    const double2 tb = lds_f64x2(tb_.ltab + i16);                  // {1/c_i, log2 c_i}
    const double r = fma(m, tb.x, -1.0);
    double p = DP_LOGP3;
    p = fma(p, r, DP_LOGP2); p = fma(p, r, DP_LOGP1); p = fma(p, r, DP_LOGP0);
    const double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - 4503601774854144.0;   // (double)e: 2^52 + 2^31
    return fma(r, p, ed + tb.y);
}

// 2^x for -6e7 < x <= 1000; below -1022 the result is ~1e-308, i.e. 0 for every use here
__device__ __forceinline__ double dp_exp2(double x, const DpTabs &tb_)
{
    const double xs = x + 211106232532992.0;                       // 1.5 * 2^47: ulp = 1/32
    const double r = x - (xs - 211106232532992.0);                 // |r| <= 1/64
    const int n = __double2loint(xs);                              // round(32 x)
    const double T = lds_f64(tb_.etab + ((n & 31) << 3));
    double q = DP_EXPP3;
    q = fma(q, r, DP_EXPP2); q = fma(q, r, DP_EXPP1); q = fma(q, r, DP_EXPP0);
    const double y = fma(T * r, q, T);                             // in [0.98, 2.03)
    return __hiloint2double(__double2hiint(y) + (max(n >> 5, -1022) << 20), __double2loint(y));
}

__device__ __forceinline__ double dp_atan_small(double r)         // |r| <= 0.6
{
    const double s = r * r;
    double p = DP_ATANP9;
    p = fma(p, s, DP_ATANP8); p = fma(p, s, DP_ATANP7); p = fma(p, s, DP_ATANP6); p = fma(p, s, DP_ATANP5);
    p = fma(p, s, DP_ATANP4); p = fma(p, s, DP_ATANP3); p = fma(p, s, DP_ATANP2); p = fma(p, s, DP_ATANP1);
    p = fma(p, s, DP_ATANP0);
    return fma(r * s, p, r);
}

// Sersic value 2^(K (1 - u)), u = t^(1/2n) (the caller multiplies by amp)
__device__ __forceinline__ double dp_sersic(double p, double K, double t, const DpTabs &tb)
{
    const double u = dp_exp2(p * dp_log2(t, tb), tb);              // |p log2 t| <= 1023 p
    double x = fma(-K, u, K);
    x = x < -1100.0 ? -1100.0 : x;                                 // u can be huge (small n, far out): 2^x = 0
    return dp_exp2(x, tb);
}

// SIE deflection in the lens frame (arcsec)
__device__ __forceinline__ void dp_sie(const RowD &R, double xp, double yp, const DpTabs &tb, double &axp, double &ayp)
{
    const double psi2 = fma(R.q2 * xp, xp, fma(yp, yp, 1e-280));  // > 0: at the lens centre both angles come out as 0 (G6)
    const double psi = psi2 * dp_rsqrt(psi2);
    const double Ax = R.qp * fabs(xp), Ay = R.qp * fabs(yp);
    // atan: rotate (psi, q'|x'|) by -theta0
    const double d2 = fma(Ax, R.s0, psi * R.c0), n2 = fma(Ax, R.c0, -psi * R.s0);
    const double pa = dp_atan_small(n2 * dp_rcp(d2));
    const double a1 = fma(R.f, pa, R.fth0);
    // atanh(z) = ln((1 + z)/(1 - z))/2, z = q'|y'|/psi
    const double a2 = R.fl2 * dp_log2(dp_div(psi + Ay, psi - Ay), tb);
    axp = copysign(a1, xp);
    ayp = copysign(a2, yp);
}

// strongly flattened lenses (q < 0.5) and the EPL: CUDA's double math library, out of line
static __device__ __noinline__ void dp_alpha_slow(const RowD &R, double xp, double yp, double &axp, double &ayp)
{
    axp = 0.0; ayp = 0.0;
    if (R.mode == 2) { epl_alpha_f64(R.t, R.A, R.q, R.fe, xp, yp, axp, ayp); return; }
    const double psi = sqrt(R.q2 * xp * xp + yp * yp);
    if (!(psi > 0.0)) return;
    axp = R.f * atan(R.qp * xp / psi);
    ayp = R.f * atanh(R.qp * yp / psi);
}

#ifdef TL_MAIN_TU
// ---- step a0 in FP64: one thread per row ----------------------------------------------------------
__global__ void __launch_bounds__(64) prologue_dp_kernel(const DpArgs a)
{
    const int n_rows = dp_n_rows(a);
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const int64_t row = dp_row(a, r);
    const float *p = a.params + row * a.P;
    RowD &R = a.rows[r];
    const int LP = a.lens_np;
    bool ok = true;
    for (int i = 0; i < LP; ++i) ok = ok && isfinite(p[i]);
    double q = 1.0, c = 1.0, s = 0.0;
    ok = ok && (p[0] >= 0.f) && shape_from_e(p[1], p[2], &q, &c, &s);
    if (a.mass_model == MASS_EPL) ok = ok && (p[7] > 1.f) && (p[7] < 3.f);
    const double thE = ok ? (double)p[0] : 0.0;
    if (!ok) { q = 1.0; c = 1.0; s = 0.0; }
    const double g1 = ok ? (double)p[5] : 0.0, g2 = ok ? (double)p[6] : 0.0;
    // No deflection at all (theta_E = 0 and no shear): beta = theta EXACTLY, and a Sersic of large n
    // is not Lipschitz at its centre (I ~ I_0 (1 - b_n (R/r_e)^(1/n))), so a source centre that
    // coincides with a sample must give R = 0 exactly, not the 1e-16 residual of the lens-frame
    // constants.  Such rows use the identity as "lens frame" and plain source centres.
    const bool nolens = thE == 0.0 && g1 == 0.0 && g2 == 0.0;
    if (nolens) { q = 1.0; c = 1.0; s = 0.0; }
    R.cx = (ok && !nolens) ? (double)p[3] : 0.0; R.cy = (ok && !nolens) ? (double)p[4] : 0.0; R.c = c; R.s = s;
    R.n11 = c * (1.0 + g1) + s * g2; R.n12 = c * g2 + s * (1.0 - g1);
    R.n21 = -s * (1.0 + g1) + c * g2; R.n22 = -s * g2 + c * (1.0 - g1);
    const float *s1 = p + LP + 7 * a.n_lens_light;
    const bool s1ok = isfinite(s1[5]) && isfinite(s1[6]);
    const double s1x = (s1ok && !nolens) ? (double)s1[5] : 0.0, s1y = (s1ok && !nolens) ? (double)s1[6] : 0.0;
    R.d1 = R.n11 * R.cx + R.n12 * R.cy - (c * s1x + s * s1y);
    R.d2 = R.n21 * R.cx + R.n22 * R.cy - (-s * s1x + c * s1y);
    // q' clamped away from 0 (relative change of alpha < 1e-18; atan(z)/z, atanh(z)/z -> 1, G6)
    const double qp = fmax(sqrt((1.0 - q) * (1.0 + q)), 1e-9);
    R.q2 = q * q; R.qp = qp; R.q = q; R.thE_sq = thE * sqrt(q);
    R.f = R.thE_sq / qp;
    R.c0 = sqrt(0.5 * (1.0 + q)); R.s0 = qp / (2.0 * R.c0);   // ~ (cos, sin)(atan(q'/q)/2): half-angle formulas
    R.fth0 = R.f * atan2(R.s0, R.c0);                 // the angle the stored pair really encodes
    R.fl2 = R.f * 0.34657359027997265471;             // ln(2)/2
    R.g1 = g1; R.g2 = g2;
    R.t = 1.0; R.A = 0.0; R.fe = (1.0 - q) / (1.0 + q);
    R.mode = (q >= 0.5) ? 0 : 1;
    if (a.mass_model == MASS_EPL) {
        R.mode = 2;
        if (ok) { R.t = (double)p[7] - 1.0; R.A = R.thE_sq > 0.0 ? 2.0 * pow(R.thE_sq, R.t) / (1.0 + q) : 0.0; }
    }
    bool all_ok = ok;
    for (int k = 0; k < a.n_comp; ++k) {
        const float *sp = p + LP + 7 * k;
        // MGE order: sources first (what the NLL = 0 trace kernel reads), then the sets' shapes
        CompD &C = R.comp[a.mge ? (k < a.n_lens_light ? a.n_comp - a.n_lens_light + k : k - a.n_lens_light) : k];
        bool okc = true;
        for (int i = 0; i < 7; ++i) okc = okc && isfinite(sp[i]);
        double qs = 1.0, cs = 1.0, ss = 0.0;
        if (a.lin) { okc = true; for (int i = 1; i < 7; ++i) okc = okc && isfinite(sp[i]); }
        const bool set_shape = a.mge && k < a.n_lens_light;       // MGE: only e1, e2, cx, cy of a lens-light block are read
        if (set_shape) {
            okc = true;
            for (int i = 3; i < 7; ++i) okc = okc && isfinite(sp[i]);
            okc = okc && shape_from_e(sp[3], sp[4], &qs, &cs, &ss);
        } else {
            okc = okc && (sp[1] > 0.f) && (sp[2] > 0.f) && shape_from_e(sp[3], sp[4], &qs, &cs, &ss);
        }
        const double Ie = a.lin ? 1.0 : (okc ? (double)sp[0] : 0.0);
        const double re = (okc && !set_shape) ? (double)sp[1] : 1.0, n = (okc && !set_shape) ? (double)sp[2] : 1.0;
        if (!okc) { qs = 1.0; cs = 1.0; ss = 0.0; }
        const double bn = sersic_bn(n);
        const double A = qs / (re * re), Bq = 1.0 / (qs * re * re);     // Eq. 10: t = A x1^2 + B x2^2
        const double kx = okc ? (double)sp[5] : 0.0, ky = okc ? (double)sp[6] : 0.0;
        double cd, sd;
        if (k < a.n_lens_light) { cd = cs; sd = ss; C.ox = kx; C.oy = ky; }
        else {
            cd = cs * c + ss * s; sd = ss * c - cs * s;                 // cos, sin(phi_s - phi)
            const double rx = kx - s1x, ry = ky - s1y;
            C.ox = c * rx + s * ry; C.oy = -s * rx + c * ry;
        }
        C.a = A * cd * cd + Bq * sd * sd;
        C.b2 = 2.0 * (A - Bq) * cd * sd;
        C.cc = A * sd * sd + Bq * cd * cd;
        C.p = 0.5 / n; C.K = bn * 1.4426950408889634074;
        C.amp = Ie / (double)(a.S * a.S);
        C.valid = okc ? 1 : 0; C.pad = 0;
        all_ok = all_ok && okc;
    }
    R.valid = all_ok ? 1 : 0;
}

// ---- steps a1-a5 in FP64: one warp per (row, tile of CW x CH = 32 extended pixels) -----------------
// Two passes over the S x S sub-samples of a pixel -- lens light, then ray-trace + sources -- so that
// each loop keeps few row constants live and the compiler can interleave the dependency chains of
// several sub-samples (the FP64 pipe needs ~4 independent DFMAs in flight per scheduler, and 128
// registers hold only one full sample's worth of FP64 state).  S_T > 0: compile-time supersampling.
template <int S_T, int NLL, int NSRC>
__global__ void __launch_bounds__(256, 2) trace_dp_kernel(const DpArgs a)
{
    __shared__ double2 ltab[DP_LOG_N + 1];
    __shared__ double etab[DP_EXP_N];
    __shared__ RowD rsh[8];
    for (int i = threadIdx.x; i <= DP_LOG_N; i += blockDim.x) ltab[i] = make_double2(DP_LOG_TABLE[i][0], DP_LOG_TABLE[i][1]);
    for (int i = threadIdx.x; i < DP_EXP_N; i += blockDim.x) etab[i] = DP_EXP_TABLE[i];
    __syncthreads();
    DpTabs tb;
    tb.ltab = (unsigned)__cvta_generic_to_shared(ltab);
    tb.etab = (unsigned)__cvta_generic_to_shared(etab);
    const int n_rows = dp_n_rows(a);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int lj = lane % a.CW, li = lane / a.CW;
    const int n_tiles = a.tiles_x * a.tiles_y;
    const long long n_items = (long long)n_rows * n_tiles;
    const long long n_warps = (long long)gridDim.x * (blockDim.x >> 5);
    RowD &R = rsh[wid];
    int cur = -1;
    const int S = S_T > 0 ? S_T : a.S;
    const double u = a.u, du = 2.0 * u;
    constexpr int UA = S_T >= 4 ? 4 : (S_T > 0 ? S_T : 1);          // sub-samples interleaved: lens-light pass
    constexpr int UB = S_T >= 2 ? 2 : 1;                            //                          ray-trace pass
    for (long long item = (long long)blockIdx.x * (blockDim.x >> 5) + wid; item < n_items; item += n_warps) {
        const int r = (int)(item / n_tiles), tile = (int)(item - (long long)r * n_tiles);
        if (r != cur) {                                            // this warp's copy of the row constants
            __syncwarp();
            const double *src = reinterpret_cast<const double *>(a.rows + r);
            double *dst = reinterpret_cast<double *>(&R);
            for (int k = lane; k < (int)(sizeof(RowD) / 8); k += 32) dst[k] = src[k];
            __syncwarp();
            cur = r;
        }
        if (!R.valid) continue;
        const int tc = tile / a.tiles_y, tr = tile - tc * a.tiles_y;
        const int j = tc * a.CW + lj, i = tr * a.CH + li;
        if (i >= a.He || j >= a.We) continue;
        double acc = 0.0;
        double comp_out[NLL + NSRC];                               // linear mode: the components, each on its own
#pragma unroll
        for (int k = 0; k < NLL + NSRC; ++k) comp_out[k] = 0.0;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        if (!edge) {
            const double x0 = (double)(2 * j * S + 1 - S * a.We) * u, y0 = (double)(2 * i * S + 1 - S * a.He) * u;
            if (NLL) {                                             // ---- pass A: lens light at theta (step a4)
                const CompD &C = R.comp[0];
                const double la = C.a, lb2 = C.b2, lcc = C.cc, lp = C.p, lK = C.K;
                const double dxl0 = x0 - C.ox;
                double dyl = y0 - C.oy;
                double accl = 0.0;
#pragma unroll 1
                for (int sa = 0; sa < S; ++sa, dyl += du) {
                    const double LC = lcc * dyl * dyl, LBy = lb2 * dyl;
#pragma unroll 1
                    for (int sb = 0; sb < S; sb += UA) {
                        double t[UA], v[UA];
#pragma unroll
                        for (int q = 0; q < UA; ++q) {
                            const double dxl = dxl0 + (double)(sb + q) * du;
                            t[q] = fma(dxl, fma(la, dxl, LBy), LC);
                        }
#pragma unroll
                        for (int q = 0; q < UA; ++q) v[q] = dp_sersic(lp, lK, t[q], tb);
#pragma unroll
                        for (int q = 0; q < UA; ++q) accl += v[q];
                    }
                }
                acc = C.amp * accl;
                comp_out[0] = acc;
            }
            {                                                      // ---- pass B: ray-trace + sources (a2, a3)
                const double dx0 = x0 - R.cx;
                double dy = y0 - R.cy;
                double accs[NSRC];
#pragma unroll
                for (int k = 0; k < NSRC; ++k) accs[k] = 0.0;
#pragma unroll 1
                for (int sa = 0; sa < S; ++sa, dy += du) {
                    const double Qc = dy * R.c, Qs = dy * R.s;
                    const double V = fma(dy, R.n12, R.d1), V2 = fma(dy, R.n22, R.d2);
#pragma unroll 1
                    for (int sb = 0; sb < S; sb += UB) {
                        double bx[UB], by[UB];
#pragma unroll
                        for (int q = 0; q < UB; ++q) {
                            const double dx = dx0 + (double)(sb + q) * du;
                            const double xp = fma(dx, R.c, Qs), yp = fma(-dx, R.s, Qc);
                            double axp, ayp;
                            if (R.mode == 0) dp_sie(R, xp, yp, tb, axp, ayp);
                            else dp_alpha_slow(R, xp, yp, axp, ayp);
                            bx[q] = fma(dx, R.n11, V) - axp; by[q] = fma(dx, R.n21, V2) - ayp;   // R^T (beta - s_first)
                        }
#pragma unroll
                        for (int k = 0; k < NSRC; ++k) {
                            const CompD &C = R.comp[NLL + k];
#pragma unroll
                            for (int q = 0; q < UB; ++q) {
                                const double ex = bx[q] - C.ox, ey = by[q] - C.oy;      // (0, 0) for the first source unless nolens
                                const double t = fma(ex, fma(C.a, ex, C.b2 * ey), C.cc * ey * ey);
                                accs[k] += dp_sersic(C.p, C.K, t, tb);
                            }
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < NSRC; ++k) { comp_out[NLL + k] = R.comp[NLL + k].amp * accs[k]; acc += comp_out[NLL + k]; }
            }
        }
        if (a.lin) {
#pragma unroll
            for (int k = 0; k < NLL + NSRC; ++k)
                a.ext[(((size_t)r * (a.ext_nc ? a.ext_nc : NLL + NSRC) + a.ext_k0 + k) * a.He + i) * a.Wp + j] = comp_out[k];
        } else {
            a.ext[((size_t)r * a.He + i) * a.Wp + j] = acc;
        }
    }
}

// ---- MGE in FP64: the binned unit-amplitude Gaussians (reading G23) --------------
// one thread per (row, extended pixel, Gaussian): exp(-R_p^2 / 2 sigma_k^2) = 2^(-t c_k) at every sub-sample
__global__ void __launch_bounds__(256) gauss_dp_kernel(const DpArgs a)
{
    __shared__ double etab[DP_EXP_N];
    for (int i = threadIdx.x; i < DP_EXP_N; i += blockDim.x) etab[i] = DP_EXP_TABLE[i];
    __syncthreads();
    DpTabs tb;
    tb.ltab = 0; tb.etab = (unsigned)__cvta_generic_to_shared(etab);
    const int n_rows = dp_n_rows(a);
    const int r = blockIdx.x;
    if (r >= n_rows || !a.rows[r].valid) return;
    const RowD &R = a.rows[r];
    const int S = a.S, npx = a.He * a.We;
    const double u = a.u, du = 2.0 * u, inv_s2 = 1.0 / (double)(S * S);
    for (int w = blockIdx.y * blockDim.x + threadIdx.x; w < npx * a.n_gauss; w += gridDim.y * blockDim.x) {
        const int k = w / npx, pix = w - k * npx, i = pix / a.We, j = pix - i * a.We;
        const CompD &C = R.comp[a.n_source + a.mge_set[k]];
        const double ck = -a.mge_c[k];
        double acc = 0.0;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        if (!edge) {
            const double dx0 = (double)(2 * j * S + 1 - S * a.We) * u - C.ox;
            double dy = (double)(2 * i * S + 1 - S * a.He) * u - C.oy;
            for (int sa = 0; sa < S; ++sa, dy += du) {
                const double LC = C.cc * dy * dy, LBy = C.b2 * dy;
                double dx = dx0;
                for (int sb = 0; sb < S; ++sb, dx += du) {
                    double x = fma(dx, fma(C.a, dx, LBy), LC) * ck;
                    x = x < -1100.0 ? -1100.0 : x;
                    acc += dp_exp2(x, tb);
                }
            }
        }
        a.ext[(((size_t)r * a.ext_nc + k) * a.He + i) * a.Wp + j] = acc * inv_s2;
    }
}

// ---- steps a6-a7 in FP64: one CTA per (row, band of output rows) -----------------------------------
// 1 x 8 output strips: per kernel row a thread reads its window of K + 7 doubles with LDS.128 and
// the K taps as broadcast LDS.128 for 8 K DFMAs (1 x 4 strips would be bound by shared-memory
// bandwidth).  The common PSF sizes are compiled with the window in registers; other odd sizes
// take the generic loop (window re-read from shared memory per tap pair).
template <int K>
__device__ __forceinline__ void dp_conv_strip(const double *win, int Wp, const double *taps, double (&acc)[8])
{
    constexpr int Kd = (K + 1) & ~1, NW = (K + 7 + 1) / 2;          // taps per row (even), double2 per window
#pragma unroll 1
    for (int ka = 0; ka < K; ++ka) {
        double w[2 * NW];
#pragma unroll
        for (int g = 0; g < NW; ++g) { const double2 v = *reinterpret_cast<const double2 *>(win + ka * Wp + 2 * g); w[2 * g] = v.x; w[2 * g + 1] = v.y; }
        const double *tp = taps + ka * Kd;
#pragma unroll
        for (int kb = 0; kb < Kd; kb += 2) {
            const double2 tv = *reinterpret_cast<const double2 *>(tp + kb);
#pragma unroll
            for (int o = 0; o < 8; ++o) acc[o] = fma(tv.x, w[kb + o], acc[o]);
            if (kb + 1 < K) {
#pragma unroll
                for (int o = 0; o < 8; ++o) acc[o] = fma(tv.y, w[kb + 1 + o], acc[o]);
            }
        }
    }
}

__device__ __forceinline__ void dp_conv_strip_any(const double *win, int Wp, const double *taps, int K, double (&acc)[8])
{
    const int Kd = (K + 1) & ~1;
    for (int ka = 0; ka < K; ++ka)
        for (int kb = 0; kb < K; ++kb) {
            const double t = taps[ka * Kd + kb];
            const double *wp = win + ka * Wp + kb;
#pragma unroll
            for (int o = 0; o < 8; ++o) acc[o] = fma(t, wp[o], acc[o]);
        }
}

__global__ void __launch_bounds__(256) conv_dp_kernel(const DpArgs a)
{
    extern __shared__ __align__(16) unsigned char dp_dyn[];
    __shared__ double red[32];
    const int n_rows = dp_n_rows(a);
    const int r = blockIdx.x, band = blockIdx.y, comp = blockIdx.z, ncmp = gridDim.z;   // (linear mode: one component per z)
    if (r >= n_rows) return;
    const int64_t row = dp_row(a, r);
    const int64_t lens = row / a.rows_per_lens;
    const size_t npix = (size_t)a.ny * a.nx;
    const int i0 = band * a.band_rows, i1 = min(a.ny, i0 + a.band_rows);
    if (!a.rows[r].valid) {
        if (a.lin) return;                                         // solve_dp_kernel reports the row
        if (a.images)
            for (size_t i = (size_t)i0 * a.nx + threadIdx.x; i < (size_t)i1 * a.nx; i += blockDim.x) a.images[row * npix + i] = NAN;
        if (a.partial && threadIdx.x == 0) a.partial[(size_t)r * a.n_bands + band] = INFINITY;
        return;
    }
    const int Kd = (a.K + 1) & ~1;                                   // taps per kernel row, padded to even
    double *taps = reinterpret_cast<double *>(dp_dyn);               // [K][Kd]
    double *img = taps + a.K * Kd;                                   // [erows][Wp] + slack
    const float *tsrc = a.psf + lens * a.K * a.Kp;
    for (int t = threadIdx.x; t < a.K * Kd; t += blockDim.x) {
        const int ka = t / Kd, kb = t - ka * Kd;
        taps[t] = kb < a.K ? (double)tsrc[ka * a.Kp + kb] : 0.0;
    }
    const int erows = (i1 - i0) + a.K - 1;
    const double2 *src = reinterpret_cast<const double2 *>(a.ext + (((size_t)r * ncmp + comp) * a.He + i0) * a.Wp);
    double2 *dst = reinterpret_cast<double2 *>(img);
    const int n2 = erows * a.Wp / 2;
    for (int t = threadIdx.x; t < n2; t += blockDim.x) dst[t] = src[t];
    for (int t = threadIdx.x; t < Kd + 16; t += blockDim.x) img[erows * a.Wp + t] = 0.0;     // read by discarded lanes only
    __syncthreads();
    // strips are numbered with the ROW fastest: the lanes of a warp then read window addresses one row
    // pitch apart, and the pitch is 2 (mod 16) doubles = 16 bytes (mod 128), so the 8 lanes of a
    // quarter-warp cover 8 different 16-byte bank groups: every LDS.128 is conflict-free.  (With the
    // column fastest the lanes sit 64 bytes apart -- a 4-way conflict that made the kernel
    // shared-memory bound at a third of the FP64 peak.)
    const int nsx = (a.nx + 7) / 8, nrow = i1 - i0, total = nrow * nsx;
    const float *data = a.data + lens * npix;
    const double *wgt = a.wgt64 + lens * npix;
    double part = 0.0;
    for (int sIdx = threadIdx.x; sIdx < total; sIdx += blockDim.x) {
        const int xs = sIdx / nrow, ir = sIdx - xs * nrow, x0 = xs * 8, i = i0 + ir;
        double acc[8];
#pragma unroll
        for (int o = 0; o < 8; ++o) acc[o] = 0.0;
        const double *win = img + (size_t)ir * a.Wp + x0;
        switch (a.K) {
        case 5: dp_conv_strip<5>(win, a.Wp, taps, acc); break;
        case 15: dp_conv_strip<15>(win, a.Wp, taps, acc); break;
        case 21: dp_conv_strip<21>(win, a.Wp, taps, acc); break;
        case 31: dp_conv_strip<31>(win, a.Wp, taps, acc); break;
        case 41: dp_conv_strip<41>(win, a.Wp, taps, acc); break;
        default: dp_conv_strip_any(win, a.Wp, taps, a.K, acc); break;
        }
#pragma unroll
        for (int o = 0; o < 8; ++o) {
            const int x = x0 + o;
            if (x < a.nx) {
                const size_t off = (size_t)i * a.nx + x;
                if (a.lin) { a.m64[((size_t)r * ncmp + comp) * npix + off] = acc[o]; continue; }
                if (a.images) a.images[row * npix + off] = (float)acc[o];
                if (a.partial) { const double d = (double)data[off] - acc[o]; part = fma(d * d, wgt[off], part); }
            }
        }
    }
    if (a.partial && !a.lin) {
        const double sum = block_sum(part, red);
        if (threadIdx.x == 0) a.partial[(size_t)r * a.n_bands + band] = sum;
    }
}

// linear-amplitude mode in FP64 (PAPER.md:86-93 Eq. 6, :97-129 Eq. 7): one CTA per row.  G = M'WM,
// b = M'Wd, d'Wd by fixed-shape block sums over the FP64 columns, the paper's NNLS (tl_nnls.cuh),
// then chi^2 of the residual d - M s -> logL, amplitudes.
__global__ void __launch_bounds__(256) solve_dp_kernel(const DpArgs a)
{
    __shared__ double red[32];
    __shared__ double s_sh[3];
    const int n_rows = dp_n_rows(a);
    const int r = blockIdx.x;
    if (r >= n_rows) return;
    const int64_t row = dp_row(a, r);
    const int NC = a.n_comp, npix = a.ny * a.nx;
    if (!a.rows[r].valid) {
        if (threadIdx.x == 0) {
            a.logL[row] = -INFINITY;
            if (a.amps) for (int k = 0; k < NC; ++k) a.amps[row * NC + k] = NAN;
        }
        return;
    }
    const int64_t lens = row / a.rows_per_lens;
    const double *M = a.m64 + (size_t)r * NC * npix;
    const float *d = a.data + lens * (size_t)npix;
    const double *w = a.wgt64 + lens * (size_t)npix;
    double g[6] = {0, 0, 0, 0, 0, 0}, bb[3] = {0, 0, 0}, dd = 0.0;
    for (int i = threadIdx.x; i < npix; i += blockDim.x) {
        const double wi = w[i], di = d[i];
        double m[3] = {0.0, 0.0, 0.0};
        for (int k = 0; k < NC; ++k) m[k] = M[(size_t)k * npix + i];
        g[0] += wi * m[0] * m[0]; g[1] += wi * m[0] * m[1]; g[2] += wi * m[0] * m[2];
        g[3] += wi * m[1] * m[1]; g[4] += wi * m[1] * m[2]; g[5] += wi * m[2] * m[2];
        bb[0] += wi * m[0] * di; bb[1] += wi * m[1] * di; bb[2] += wi * m[2] * di;
        dd += wi * di * di;
    }
    double G[3][3], b[3];
    const double g0 = block_sum(g[0], red), g1 = block_sum(g[1], red), g2 = block_sum(g[2], red),
                 g3 = block_sum(g[3], red), g4 = block_sum(g[4], red), g5 = block_sum(g[5], red);
    b[0] = block_sum(bb[0], red); b[1] = block_sum(bb[1], red); b[2] = block_sum(bb[2], red);
    const double dwd = block_sum(dd, red);
    if (threadIdx.x == 0) {
        G[0][0] = g0; G[0][1] = G[1][0] = g1; G[0][2] = G[2][0] = g2; G[1][1] = g3; G[1][2] = G[2][1] = g4; G[2][2] = g5;
        double s[3] = {0.0, 0.0, 0.0}, Lc[9], z[3];
        nnls_gram<3>(NC, &G[0][0], 3, b, dwd, s, Lc, z);
        s_sh[0] = s[0]; s_sh[1] = s[1]; s_sh[2] = s[2];
    }
    __syncthreads();
    const double s0 = s_sh[0], s1 = s_sh[1], s2 = s_sh[2];
    double part = 0.0;
    for (int i = threadIdx.x; i < npix; i += blockDim.x) {
        double m = s0 * M[i];
        if (NC > 1) m += s1 * M[(size_t)npix + i];
        if (NC > 2) m += s2 * M[2 * (size_t)npix + i];
        const double res = (double)d[i] - m;
        part += res * res * w[i];
    }
    const double chi2 = block_sum(part, red);
    if (threadIdx.x == 0) {
        a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[lens]));
        if (a.amps) { a.amps[row * NC] = (float)s0; if (NC > 1) a.amps[row * NC + 1] = (float)s1; if (NC > 2) a.amps[row * NC + 2] = (float)s2; }
    }
}

__global__ void finalize_dp_kernel(const DpArgs a)
{
    const int n_rows = dp_n_rows(a);
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const int64_t row = dp_row(a, r);
    double s = 0.0;
    for (int t = 0; t < a.n_bands; ++t) s += a.partial[(size_t)r * a.n_bands + t];
    const double ll = -0.5 * (s + a.lconst[row / a.rows_per_lens]);
    a.logL[row] = isfinite(s) ? (float)ll : -INFINITY;
}
#endif  // TL_MAIN_TU

}  // namespace tl
