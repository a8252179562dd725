// tl_mge.cuh -- NEXT-3: MGE lens light with linear amplitudes (tl_loglike_mge_batch).
//
// PAPER.md:291-293 (section 4.3) names the Multiple Gaussian Expansion; reading G23:
//     I_l(theta) = sum_k a_k exp(-R_p(theta)^2 / (2 sigma_k^2)),   R_p of PAPER.md:143-148 Eq. 10,
// one centre and one (q, phi) for the set, fixed sigma_k, and the a_k >= 0 solved together with
// the source amplitudes as the NNLS minimiser of PAPER.md:86-93 Eq. 6 / :97-129 Eq. 7.
//
// Pipeline per chunk of rows (all on one stream; included by tinylens.cu only):
//   prologue_kernel (mge = 1)  lens-light quadratic form becomes t = R_p^2 in arcsec^2; the row's
//                              components are stored sources first, then the Gaussian set's shape
//   trace_kernel<S,0,1> / trace_lin_kernel<S,0,2>   ray-traced unit-amplitude source images (the NLL = 0
//                              instantiations: no lens-light stand-in is evaluated; one source
//                              takes the packed pair loop of tl_pair.cuh) -> ext, one slot per source
//   gauss_conv_kernel          one CTA per (row, Gaussian): the binned unit-amplitude Gaussian is
//                              evaluated straight into shared memory and blurred from there -- the
//                              unblurred Gaussians never touch global memory.  (Images too large
//                              for that: mge_gauss_kernel -> ext, then conv_lin_kernel.)
//   conv_lin_kernel            the source images blurred with the PSF
//   gram_reg_kernel / gram_mge_kernel   G = M'WM, b = M'Wd, d'Wd in FP64 (fixed summation order) -> global
//                              (up to 11 columns: every entry in registers; more: staged through shared memory)
//   nnls_mge_kernel            NNLS by the Gram-matrix active-set iteration of Bro & De Jong (the
//                              paper's solver), one warp per row -> amplitudes,
//                              and chi^2 = d'Wd - 2 s'b + s'Gs -> logL.  All of it FP64 on exact
//                              products of the FP32 columns: the three terms are ~1e9 and chi^2
//                              ~1e4, a loss of 5 of 16 digits (1e-7 absolute), so the second pass
//                              over M that round 1 made for the residual is not needed.
#pragma once
#include "tl_kernels.cuh"

namespace tl {

constexpr int MGE_MAX_GAUSS = 30;                    // over all sets ("several dozen amplitudes")
constexpr int MGE_MAX_COL = MGE_MAX_GAUSS + 2;       // + n_source: 32, the width of the solver's bit masks
constexpr int MGE_MAX_SETS = 2;                      // Gaussian sets with their own (e1, e2, centre) = n_lens_light
constexpr int MGE_SOLVE_THREADS = 128;               // gram_mge_kernel: 128 threads up to 20 columns + data, else 512
constexpr int MGE_GRAM_STRIDE = MGE_MAX_COL * (MGE_MAX_COL + 1) + MGE_MAX_COL + 2;   // doubles per row: G [n][NCP] | b [n] | d'Wd
constexpr int MGE_NNLS_WARPS = 4;                    // rows per CTA of nnls_mge_kernel (one warp each)
constexpr int MGE_TILE = 64;                         // pixels staged per step of the Gram reduction

// One thread per extended native pixel (grid.x = row in chunk, grid.y = slabs of the image).
// t = R_p^2 is evaluated exactly like the lens-light term of col_values / row_values (hi/lo
// constants, exact first differences), each Gaussian is one FMUL + MUFU.EX2 per sub-sample: the
// kernel is bound by the MUFU pipe (NG ex2 per sample), so NG is a template parameter (no
// predicated-off MUFU issue) and the sub-sample offsets advance by exact FP32 additions (no I2F,
// which shares that pipe).
template <int NG>
__global__ void __launch_bounds__(256) mge_gauss_kernel(const KArgs a, int chunk_rows)
{
    const int r = blockIdx.x;
    if (r >= chunk_rows) return;
    const RowC &rc = a.rows[r];
    if (!row_is_valid(rc, a.n_comp)) return;
    const SersicC &C = rc.comp[a.n_comp - a.n_lens_light + a.mge_shape];   // MGE order: the sets' shapes follow the sources
    const float cXh = C.cXh, cXl = C.cXl, cYh = C.cYh, cYl = C.cYl;
    const float ah = C.ah, al = C.al, b2h = C.b2h, b2l = C.b2l, cch = C.cch, ccl = C.ccl;
    const int S = a.S;
    float ck[NG];
#pragma unroll
    for (int k = 0; k < NG; ++k) ck[k] = -a.mge_c[a.mge_k0 + k];
    const float inv_s2 = 1.f / (float)(S * S);
    const size_t comp_stride = (size_t)a.He * a.pitch;
    float *dst = a.ext + ((size_t)r * a.ext_nc + a.mge_k0) * comp_stride;     // this set's slots
    const int npx = a.He * a.pitch;
    for (int p = blockIdx.y * blockDim.x + threadIdx.x; p < npx; p += gridDim.y * blockDim.x) {
        const int i = p / a.pitch, j = p - i * a.pitch;
        if (j >= a.We) {                               // pitch padding of every component reads as zero
            for (int k = -a.mge_k0; k < a.ext_nc - a.mge_k0; ++k) dst[k * (long long)comp_stride + (size_t)i * a.pitch + j] = 0.f;
            continue;
        }
        float acc[NG];
#pragma unroll
        for (int k = 0; k < NG; ++k) acc[k] = 0.f;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        if (!edge) {
            const float X0 = (float)(2 * j * S + 1 - S * a.We);
            float Y = (float)(2 * i * S + 1 - S * a.He);          // small integers: the additions below are exact
#pragma unroll 1
            for (int sa = 0; sa < S; ++sa, Y += 2.f) {
                const float dyl = (Y - cYh) - cYl;
                const float y2 = dyl * dyl;
                const float LC = fmaf(cch, y2, ccl * y2);
                float X = X0;
#pragma unroll 2
                for (int sb = 0; sb < S; ++sb, X += 2.f) {
                    const float dxl = (X - cXh) - cXl;
                    const float x2 = dxl * dxl;
                    const float LA = fmaf(ah, x2, al * x2);
                    const float LB = fmaf(dxl, b2h, dxl * b2l);
                    const float t = fmaf(LB, dyl, LA + LC);
#pragma unroll
                    for (int k = 0; k < NG; ++k) acc[k] += mufu_ex2(t * ck[k]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NG; ++k) dst[k * comp_stride + (size_t)i * a.pitch + j] = acc[k] * inv_s2;
    }
}

// The 2 x 4 blocks of output row pairs ip0 .. ip1 x strips xb0 .. xb1 (inclusive) of one blurred image
// -> image_out; every other pixel of the row pairs zp0 .. zp1 of image_out is written as 0.  (gauss_conv_kernel: outside that
// rectangle every window holds nothing but exact zeros, and ConvBlock's sums of +-0 products are +0.)
template <int K>
__device__ __forceinline__ void conv_blocks_rect(const KArgs &a, const float *img, const float *taps,
                                                 int ip0, int ip1, int xb0, int xb1, float *image_out, int zp0, int zp1)
{
    const int nsx = (a.nx + 3) / 4;
    const int nbx = xb1 - xb0 + 1, nby = ip1 - ip0 + 1;
    const float zero[4] = {0.f, 0.f, 0.f, 0.f};
    if (nbx > 0 && nby > 0) {
        for (int s = threadIdx.x; s < nby * nbx; s += blockDim.x) {
            const int iy = s / nbx, i = 2 * (ip0 + iy), x0 = 4 * (xb0 + s - iy * nbx);
            float a0[4], a1[4];
            ConvBlock<K>::run(img + i * a.pitch + x0, a.pitch, taps, a0, a1);
            chi2_strip(a, a0, i, x0, nullptr, nullptr, image_out);
            if (i + 1 < a.ny) chi2_strip(a, a1, i + 1, x0, nullptr, nullptr, image_out);
        }
    }
    for (int s = threadIdx.x; s < (zp1 - zp0 + 1) * nsx; s += blockDim.x) {           // the pairs zp0 .. zp1 are this CTA's
        const int ip = zp0 + s / nsx, xb = s - (ip - zp0) * nsx;
        if (ip >= ip0 && ip <= ip1 && xb >= xb0 && xb <= xb1) continue;
        chi2_strip(a, zero, 2 * ip, 4 * xb, nullptr, nullptr, image_out);
        if (2 * ip + 1 < a.ny) chi2_strip(a, zero, 2 * ip + 1, 4 * xb, nullptr, nullptr, image_out);
    }
}

// One CTA per (row, Gaussian k): steps a4-a6 for one column of M without a round trip through global
// memory.  t = R_p^2 of a sub-sample is LA(x) + LC(y) + LB(x) dyl(y) (tl_kernels.cuh col_values /
// row_values): the column parts of a pixel's S sub-columns are computed once per pixel and kept in
// registers as pairs (tl_pair.cuh), the row parts once per sub-row, so a pair of samples costs
// FADD2 + FFMA2 + FMUL2 + 2 MUFU.EX2 + FADD2.  The evaluation is MUFU-bound, the convolution
// FMA-bound; with two or three CTAs per SM the two phases of different CTAs overlap.
// Support box: 2^(-c_k t) is flushed to an exact 0 once c_k t > 126 (ex2.approx.ftz), and
// t >= lambda_min rho^2, lambda_min the smaller eigenvalue of the set's quadratic form and rho the
// distance from the centre; so outside a box of half-width rho_k = sqrt(130 / (0.98 lambda_min c_k))
// round the centre every sub-sample is exactly 0.  Only the pixels of the box are evaluated and only
// the outputs whose window meets the box are convolved; the rest of the column is written as 0 --
// the same bits as evaluating everything (a 0.6-pixel Gaussian covers 1/30 of a 120 x 120 image).
// S_T = 0: any S (scalar loop).
// K_T: the PSF size when it has a register-blocked convolution (a kernel of its own per size, so that the
// small sizes are not held to the registers of the 41 x 41 blocks: up to 21 x 21 three CTAs share an SM),
// 0 = any other size.
template <int S_T, int K_T>
__global__ void __launch_bounds__(256, (K_T > 0 && K_T <= 21) ? 3 : 2) gauss_conv_kernel(const KArgs a, int chunk_rows)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *taps = reinterpret_cast<float *>(smem_raw);
    float *img = taps + a.K * a.Kp;
    const int r = blockIdx.x, k = blockIdx.y;
    if (r >= chunk_rows) return;
    const RowC &rc = a.rows[r];
    if (!row_is_valid(rc, a.n_comp)) return;
    const int64_t lens = (a.row0 + r) / a.rows_per_lens;
    load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp);
    const SersicC &C = rc.comp[a.n_comp - a.n_lens_light + a.mge_set[k]];     // the shape of this Gaussian's set
    const float cXh = C.cXh, cXl = C.cXl, cYh = C.cYh, cYl = C.cYl;
    const float ah = C.ah, al = C.al, b2h = C.b2h, b2l = C.b2l, cch = C.cch, ccl = C.ccl;
    const float ck = -a.mge_c[k];
    const int S = S_T > 0 ? S_T : a.S;
    const float inv_s2 = 1.f / (float)(S * S);
    const int npx = a.He * a.pitch;
    // the support box in extended pixels [i_lo, i_hi] x [j_lo, j_hi] (one pixel of slack on every side)
    int i_lo = 0, i_hi = a.He - 1, j_lo = 0, j_hi = a.We - 1;
    {
        const float hd = 0.5f * (ah - cch), hb = 0.5f * b2h;
        const float lmax = 0.5f * (ah + cch) + sqrtf(fmaf(hd, hd, hb * hb));
        const float lmin = fmaf(ah, cch, -hb * hb) / lmax;
        const float rho = sqrtf(130.f / (0.98f * lmin * -ck));              // u-units
        if (lmin > 0.f && ck < 0.f && rho < 1e7f) {
            const float inv2s = 0.5f / (float)S, cX = cXh + cXl, cY = cYh + cYl;
            // pixel j spans X0 .. X0 + 2 (S - 1), X0 = 2 j S + 1 - S We
            j_lo = max(j_lo, (int)floorf((cX - rho - (float)(2 * S - 1) + (float)(S * a.We)) * inv2s) - 1);
            j_hi = min(j_hi, (int)ceilf((cX + rho - 1.f + (float)(S * a.We)) * inv2s) + 1);
            i_lo = max(i_lo, (int)floorf((cY - rho - (float)(2 * S - 1) + (float)(S * a.He)) * inv2s) - 1);
            i_hi = min(i_hi, (int)ceilf((cY + rho - 1.f + (float)(S * a.He)) * inv2s) + 1);
        }
    }
    // calls with a few rows: the output row pairs are shared out over gridDim.z CTAs (bands), each evaluating only the
    // extended rows its outputs read
    const int npair = (a.ny + 1) / 2, per_band = (npair + gridDim.z - 1) / gridDim.z;
    const int pb0 = blockIdx.z * per_band, pb1 = min(npair, pb0 + per_band) - 1;       // this CTA's pairs (inclusive)
    if (pb0 > pb1) return;
    const int e_lo = 2 * pb0, e_hi = min(a.He - 1, 2 * pb1 + 1 + a.K - 1);            // the extended rows they read
    i_lo = max(i_lo, e_lo); i_hi = min(i_hi, e_hi);
    const int bw = j_hi - j_lo + 1, bh = i_hi - i_lo + 1;
    {   // everything outside the box, the pitch padding and the slack read as zero
        float4 *z = reinterpret_cast<float4 *>(img) + (e_lo * a.pitch) / 4;           // (pitch is a multiple of 4)
        const int n4 = (((gridDim.z == 1 ? npx : (e_hi + 1) * a.pitch) - e_lo * a.pitch) + a.pitch + a.Kp + 8 + 3) / 4;
        for (int p = threadIdx.x; p < n4; p += blockDim.x) z[p] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
    for (int p = threadIdx.x; p < bw * bh; p += blockDim.x) {
        const int ib = p / bw, i = i_lo + ib, j = j_lo + (p - ib * bw);
        float acc = 0.f;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        if (!edge) {
            const float X0 = (float)(2 * j * S + 1 - S * a.We);
            float Y = (float)(2 * i * S + 1 - S * a.He);
            if constexpr (S_T > 0 && S_T % 2 == 0) {
                constexpr int NP = S_T / 2;
                f2 LA[NP], LB[NP];
#pragma unroll
                for (int q = 0; q < NP; ++q) {
                    float la[2], lb[2];
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const float dxl = ((X0 + (float)(4 * q + 2 * e)) - cXh) - cXl;
                        const float x2 = dxl * dxl;
                        la[e] = fmaf(ah, x2, al * x2);
                        lb[e] = fmaf(dxl, b2h, dxl * b2l);
                    }
                    LA[q] = mk2(la[0], la[1]); LB[q] = mk2(lb[0], lb[1]);
                }
                f2 acc2 = bc2(0.f);
#pragma unroll
                for (int sa = 0; sa < S_T; ++sa, Y += 2.f) {
                    const float dyl = (Y - cYh) - cYl;
                    const float y2 = dyl * dyl;
                    const float LC = fmaf(cch, y2, ccl * y2);
#pragma unroll
                    for (int q = 0; q < NP; ++q)
                        acc2 = add2(acc2, ex2_2(mul2(fma2(LB[q], bc2(dyl), add2(LA[q], bc2(LC))), bc2(ck))));
                }
                float a0, a1;
                un2(acc2, a0, a1);
                acc = a0 + a1;
            } else {
#pragma unroll 1
                for (int sa = 0; sa < S; ++sa, Y += 2.f) {
                    const float dyl = (Y - cYh) - cYl;
                    const float y2 = dyl * dyl;
                    const float LC = fmaf(cch, y2, ccl * y2);
                    float X = X0;
                    for (int sb = 0; sb < S; ++sb, X += 2.f) {
                        const float dxl = (X - cXh) - cXl;
                        const float x2 = dxl * dxl;
                        const float LA = fmaf(ah, x2, al * x2);
                        const float LB = fmaf(dxl, b2h, dxl * b2l);
                        acc += mufu_ex2(fmaf(LB, dyl, LA + LC) * ck);
                    }
                }
            }
            acc *= inv_s2;
        }
        img[i * a.pitch + j] = acc;
    }
    __syncthreads();
    const size_t npix = (size_t)a.ny * a.nx;
    float *out = a.mimg + ((size_t)r * a.ext_nc + k) * npix;
    // output (i, x) reads extended rows i .. i + K - 1 and columns x .. x + K - 1
    const int oi0 = max(0, i_lo - a.K + 1), oi1 = min(a.ny - 1, i_hi), ox0 = max(0, j_lo - a.K + 1), ox1 = min(a.nx - 1, j_hi);
    const bool none = bw <= 0 || bh <= 0 || oi0 > oi1 || ox0 > ox1;
    const int ip0 = none ? 1 : max(pb0, oi0 / 2), ip1 = none ? 0 : min(pb1, oi1 / 2), xb0 = none ? 1 : ox0 / 4, xb1 = none ? 0 : ox1 / 4;
    if constexpr (K_T > 0) { conv_blocks_rect<K_T>(a, img, taps, ip0, ip1, xb0, xb1, out, pb0, pb1); return; }
    if (gridDim.z != 1) return;                                               // (other PSF sizes are launched without bands)
    // other PSF sizes: the generic 1 x 4 strips over the whole image
    const int nsx = (a.nx + CONV_R - 1) / CONV_R;
    for (int s = threadIdx.x; s < a.ny * nsx; s += blockDim.x) {
        const int i = s / nsx, x0 = (s - i * nsx) * CONV_R;
        float acc[CONV_R];
        conv_strip(img + i * a.pitch + x0, a.pitch, taps, a.K, a.Kp, acc);
        chi2_strip(a, acc, i, x0, nullptr, nullptr, out);
    }
}

typedef void (*gauss_conv_fn)(const KArgs, int);
template <int S_T>
inline gauss_conv_fn gauss_conv_for_k(int K)
{
    switch (K) {
    case 5: return gauss_conv_kernel<S_T, 5>;
    case 15: return gauss_conv_kernel<S_T, 15>;
    case 21: return gauss_conv_kernel<S_T, 21>;
    case 31: return gauss_conv_kernel<S_T, 31>;
    case 41: return gauss_conv_kernel<S_T, 41>;
    default: return gauss_conv_kernel<S_T, 0>;
    }
}
inline gauss_conv_fn gauss_conv_for(int S, int K)
{
    switch (S) {
    case 2: return gauss_conv_for_k<2>(K);
    case 4: return gauss_conv_for_k<4>(K);
    case 8: return gauss_conv_for_k<8>(K);
    default: return gauss_conv_for_k<0>(K);
    }
}

typedef void (*mge_gauss_fn)(const KArgs, int);
inline mge_gauss_fn mge_gauss_for(int ng)
{
    switch (ng) {
    case 1: return mge_gauss_kernel<1>;   case 2: return mge_gauss_kernel<2>;   case 3: return mge_gauss_kernel<3>;
    case 4: return mge_gauss_kernel<4>;   case 5: return mge_gauss_kernel<5>;   case 6: return mge_gauss_kernel<6>;
    case 7: return mge_gauss_kernel<7>;   case 8: return mge_gauss_kernel<8>;   case 9: return mge_gauss_kernel<9>;
    case 10: return mge_gauss_kernel<10>; case 11: return mge_gauss_kernel<11>; case 12: return mge_gauss_kernel<12>;
    case 13: return mge_gauss_kernel<13>; case 14: return mge_gauss_kernel<14>; case 15: return mge_gauss_kernel<15>;
    case 16: return mge_gauss_kernel<16>;
    case 17: return mge_gauss_kernel<17>; case 18: return mge_gauss_kernel<18>; case 19: return mge_gauss_kernel<19>;
    case 20: return mge_gauss_kernel<20>; case 21: return mge_gauss_kernel<21>; case 22: return mge_gauss_kernel<22>;
    case 23: return mge_gauss_kernel<23>; case 24: return mge_gauss_kernel<24>; case 25: return mge_gauss_kernel<25>;
    case 26: return mge_gauss_kernel<26>; case 27: return mge_gauss_kernel<27>; case 28: return mge_gauss_kernel<28>;
    case 29: return mge_gauss_kernel<29>; case 30: return mge_gauss_kernel<30>;
    default: return nullptr;
    }
}

// G = M'WM, b = M'Wd, d'Wd: one CTA of 128 threads per row.  The pixels are staged through shared
// memory MGE_TILE at a time (w m_k and m_k, d as doubles, the next tile prefetched into registers);
// every sum has a fixed order, so the result is bitwise reproducible.
// Output: a.mge_gram[r][MGE_GRAM_STRIDE].
// T = float: the FP32 pipeline's columns and weights; T = double: the FP64 pipeline's (a.mimg64, a.wgt64).
template <int THREADS, typename T = float>
__global__ void __launch_bounds__(THREADS) gram_mge_kernel(const KArgs a, int chunk_rows)
{
    constexpr int NCP = MGE_MAX_COL + 2;               // columns + data, rounded up to even
    // column-major tiles with an odd pitch: the staging stores of a warp (consecutive pixels of one
    // column) and the loads of the sums (one pixel, different columns) are both free of bank conflicts
    // (pixel-major rows of 20 doubles made every staging store an 8-way conflict)
    constexpr int TP = MGE_TILE + 1;
    __shared__ double As[NCP][TP];                     // w_i m_ki   (column n: w_i d_i)
    __shared__ double Bs[NCP][TP];                     // m_ki       (column n: d_i)
    const int r = blockIdx.x;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    const int n = a.ext_nc;
    if (!row_is_valid(a.rows[r], a.n_comp)) return;   // nnls_mge_kernel reports the row
    const int64_t lens = row / a.rows_per_lens;
    const int npix = a.ny * a.nx;
    const T *M = (sizeof(T) == 8 ? reinterpret_cast<const T *>(a.mimg64) : reinterpret_cast<const T *>(a.mimg)) + (size_t)r * n * npix;
    const float *d = a.data + lens * (size_t)npix;
    const T *w = (sizeof(T) == 8 ? reinterpret_cast<const T *>(a.wgt64) : reinterpret_cast<const T *>(a.wgt)) + lens * (size_t)npix;
    double *gout = a.mge_gram + (size_t)r * MGE_GRAM_STRIDE;
    // [G | b | d'Wd] = A'B with A = [w m_k | w d], B = [m_k | d]  (n1 = n + 1 columns, the data last).
    // Register blocking: a thread owns a 2 x 2 block of entries (columns 2bi, 2bi+1 of A against
    // 2bj, 2bj+1 of B, bi <= bj) and every Q-th pixel of a tile, so two loads of A and two of B
    // feed four DFMAs (one entry per thread is bound by the shared-memory pipe); the Q pixel
    // slices of an entry are then added in slice order -- a fixed summation order.
    const int n1 = n + 1, NB = (n1 + 1) >> 1, nblk = NB * (NB + 1) / 2;
    const int Q = THREADS / nblk;                                 // >= 2 (nblk <= 55 at 128 threads, <= 153 at 512)
    const int slice = threadIdx.x / nblk;
    int bi = 0, bj = 0;
    {
        int p = threadIdx.x - slice * nblk;
        while (p >= NB - bi) { p -= NB - bi; ++bi; }
        bj = bi + p;
    }
    const bool gram_thread = slice < Q;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    // the next tile's values are fetched into registers while the current one is consumed, so the
    // global-memory latency (M does not fit in L2 for a whole batch) overlaps the FP64 sums.
    // Thread t stages pixel t % MGE_TILE of the tile for the columns t / MGE_TILE, + 2, + 4, ...
    constexpr int EPT = (MGE_TILE * NCP + THREADS - 1) / THREADS;
    static_assert(THREADS % MGE_TILE == 0, "a thread stages one pixel of the tile");
    const int ncol = 2 * NB;                                      // n1 rounded up to even: a zero column
    const int sii = threadIdx.x % MGE_TILE, sk0 = threadIdx.x / MGE_TILE;
    T fv[EPT], fwv = (T)0;
    auto fetch = [&](int t0) {
        const int i = t0 + sii;
        fwv = i < npix ? w[i] : (T)0;
#pragma unroll
        for (int u = 0; u < EPT; ++u) {
            const int k = sk0 + u * (THREADS / MGE_TILE);
            fv[u] = (T)0;
            if (k < n1 && i < npix) fv[u] = k < n ? M[(size_t)k * npix + i] : (T)d[i];
        }
    };
    fetch(0);
    for (int t0 = 0; t0 < npix; t0 += MGE_TILE) {
        __syncthreads();
        {
            const double wd = (double)fwv;
#pragma unroll
            for (int u = 0; u < EPT; ++u) {
                const int k = sk0 + u * (THREADS / MGE_TILE);
                if (k < ncol) { const double v = (double)fv[u]; As[k][sii] = wd * v; Bs[k][sii] = v; }
            }
        }
        __syncthreads();
        if (t0 + MGE_TILE < npix) fetch(t0 + MGE_TILE);
        if (gram_thread) {
#pragma unroll 4
            for (int ii = slice; ii < MGE_TILE; ii += Q) {
                const double ax = As[2 * bi][ii], ay = As[2 * bi + 1][ii];
                const double bx = Bs[2 * bj][ii], by = Bs[2 * bj + 1][ii];
                acc[0] = fma(ax, bx, acc[0]); acc[1] = fma(ax, by, acc[1]);
                acc[2] = fma(ay, bx, acc[2]); acc[3] = fma(ay, by, acc[3]);
            }
        }
    }
    __syncthreads();
    double *Ps = &As[0][0];                                       // [Q * nblk][4] partial blocks (As is free now)
    if (gram_thread) {
#pragma unroll
        for (int e = 0; e < 4; ++e) Ps[(size_t)threadIdx.x * 4 + e] = acc[e];
    }
    __syncthreads();
    constexpr int NCG = MGE_MAX_COL + 1;                          // row pitch of G in a.mge_gram
    for (int t = threadIdx.x; t < nblk * 4; t += blockDim.x) {
        const int blk = t >> 2, e = t & 3;
        double v = 0.0;
        for (int q = 0; q < Q; ++q) v += Ps[(size_t)(q * nblk + blk) * 4 + e];
        int ci = 0, p = blk;
        while (p >= NB - ci) { p -= NB - ci; ++ci; }
        const int k = 2 * ci + (e >> 1), l = 2 * (ci + p) + (e & 1);
        if (k < n && l < n) { gout[k * NCG + l] = v; gout[l * NCG + k] = v; }
        else if (k < n && l == n) gout[MGE_MAX_COL * NCG + k] = v;
        else if (k == n && l == n) gout[MGE_MAX_COL * NCG + MGE_MAX_COL] = v;
    }
}

// The same sums for up to MGE_GRAM_REG_COLS columns + data (the FP32 pipeline), every entry in a REGISTER
// of every thread: gram_mge_kernel reads one operand from shared memory per DFMA and is bound by that
// pipe at a quarter of the FP64 rate; here a thread takes two neighbouring pixels per step (one
// 8-byte load per column, the next step's loads in flight meanwhile), forms w m_k once and feeds the
// N1 (N1 + 1) / 2 entries from registers.  Fixed order: a thread's pixels in sequence, then a butterfly
// over the warp and the four warps in order.  Needs an even pixel count.
constexpr int MGE_GRAM_REG_COLS = 11;          // (13 columns + data would spill)
// W = 4: four neighbouring pixels per step (16-byte loads, no explicit prefetch: 13 x 16 bytes per thread in flight);
// needs a pixel count that is a multiple of 4.  W = 2: two pixels per step, the next step's loads in flight meanwhile.
template <int N1, int W>
__global__ void __launch_bounds__(128) gram_reg_kernel(const KArgs a, int chunk_rows)
{
    constexpr int NE = N1 * (N1 + 1) / 2;
    __shared__ double red[4][NE];
    const int r = blockIdx.x;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    constexpr int n = N1 - 1;
    if (!row_is_valid(a.rows[r], a.n_comp)) return;   // nnls_mge_kernel reports the row
    const int64_t lens = row / a.rows_per_lens;
    const int npix = a.ny * a.nx;
    double acc[NE];
#pragma unroll
    for (int e = 0; e < NE; ++e) acc[e] = 0.0;
    auto pixel = [&](const double (&v)[N1], double wd) {
        int e = 0;
#pragma unroll
        for (int k = 0; k < N1; ++k) {
            const double wk = wd * v[k];
#pragma unroll
            for (int l = k; l < N1; ++l, ++e) acc[e] = fma(wk, v[l], acc[e]);
        }
    };
    if constexpr (W == 4) {
        const int np4 = npix >> 2;
        const float4 *M4 = reinterpret_cast<const float4 *>(a.mimg + (size_t)r * n * npix);
        const float4 *d4 = reinterpret_cast<const float4 *>(a.data + lens * (size_t)npix);
        const float4 *w4 = reinterpret_cast<const float4 *>(a.wgt + lens * (size_t)npix);
#pragma unroll 1
        for (int p = threadIdx.x; p < np4; p += 128) {
            float4 c[N1];
#pragma unroll
            for (int k = 0; k < n; ++k) c[k] = __ldg(M4 + (size_t)k * np4 + p);
            c[n] = __ldg(d4 + p);
            const float4 wv = __ldg(w4 + p);
            double v[N1];
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)c[k].x;
            pixel(v, (double)wv.x);
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)c[k].y;
            pixel(v, (double)wv.y);
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)c[k].z;
            pixel(v, (double)wv.z);
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)c[k].w;
            pixel(v, (double)wv.w);
        }
    } else {
        const int np2 = npix >> 1;
        const float2 *M2 = reinterpret_cast<const float2 *>(a.mimg + (size_t)r * n * npix);
        const float2 *d2 = reinterpret_cast<const float2 *>(a.data + lens * (size_t)npix);
        const float2 *w2 = reinterpret_cast<const float2 *>(a.wgt + lens * (size_t)npix);
        float2 cur[N1], nxt[N1], wc, wn;
        auto fetch = [&](int p, float2 (&v)[N1], float2 &wv) {
            if (p < np2) {
#pragma unroll
                for (int k = 0; k < n; ++k) v[k] = __ldg(M2 + (size_t)k * np2 + p);
                v[n] = __ldg(d2 + p);
                wv = __ldg(w2 + p);
            } else {
#pragma unroll
                for (int k = 0; k < N1; ++k) v[k] = make_float2(0.f, 0.f);
                wv = make_float2(0.f, 0.f);
            }
        };
        fetch(threadIdx.x, cur, wc);
#pragma unroll 1
        for (int p = threadIdx.x; p < np2; p += 128) {
            fetch(p + 128, nxt, wn);
            double v[N1];
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)cur[k].x;
            pixel(v, (double)wc.x);
#pragma unroll
            for (int k = 0; k < N1; ++k) v[k] = (double)cur[k].y;
            pixel(v, (double)wc.y);
#pragma unroll
            for (int k = 0; k < N1; ++k) cur[k] = nxt[k];
            wc = wn;
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int e = 0; e < NE; ++e) {
        double v = acc[e];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][e] = v;
    }
    __syncthreads();
    constexpr int NCG = MGE_MAX_COL + 1;                          // row pitch of G in a.mge_gram
    double *gout = a.mge_gram + (size_t)r * MGE_GRAM_STRIDE;
    for (int e = threadIdx.x; e < NE; e += 128) {
        const double v = ((red[0][e] + red[1][e]) + red[2][e]) + red[3][e];
        int k = 0, q = e;
        while (q >= N1 - k) { q -= N1 - k; ++k; }
        const int l = k + q;
        if (l < n) { gout[k * NCG + l] = v; gout[l * NCG + k] = v; }
        else if (k < n) gout[MGE_MAX_COL * NCG + k] = v;
        else gout[MGE_MAX_COL * NCG + MGE_MAX_COL] = v;
    }
}

typedef void (*gram_reg_fn)(const KArgs, int);
template <int W>
inline gram_reg_fn gram_reg_for_w(int n1)
{
    switch (n1) {
    case 2: return gram_reg_kernel<2, W>;   case 3: return gram_reg_kernel<3, W>;   case 4: return gram_reg_kernel<4, W>;
    case 5: return gram_reg_kernel<5, W>;   case 6: return gram_reg_kernel<6, W>;   case 7: return gram_reg_kernel<7, W>;
    case 8: return gram_reg_kernel<8, W>;   case 9: return gram_reg_kernel<9, W>;   case 10: return gram_reg_kernel<10, W>;
    case 11: return gram_reg_kernel<11, W>; case 12: return gram_reg_kernel<12, W>;
    default: return nullptr;
    }
}
// npix: a multiple of 4 takes the 16-byte loads, else (even) the 8-byte ones
inline gram_reg_fn gram_reg_for(int n1, int npix) { return (npix & 3) == 0 ? gram_reg_for_w<4>(n1) : gram_reg_for_w<2>(n1); }

// NNLS: one warp per row, the iteration run by the whole warp (nnls_gram_warp, tl_nnls.cuh); four warps per
// CTA, a compact copy of G in dynamic shared memory (2 n^2 + 3 n doubles per row).  Writes the amplitudes and
// logL from the Gram quantities, and reports invalid rows.
__global__ void __launch_bounds__(32 * MGE_NNLS_WARPS) nnls_mge_kernel(const KArgs a, int chunk_rows)
{
    // per warp (dynamic shared memory, sized by the actual column count n): G [n][n] | b [n] | L [n][n] | z [n] | s [n]
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NCG = MGE_MAX_COL + 1;                          // row pitch of G in a.mge_gram
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * MGE_NNLS_WARPS + wid;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    const int n = a.ext_nc;
    double *Gs = reinterpret_cast<double *>(smem_raw) + (size_t)wid * (2 * n * n + 3 * n);
    double *bs = Gs + n * n, *Ls = bs + n, *zs = Ls + n * n, *ss = zs + n;
    if (!row_is_valid(a.rows[r], a.n_comp)) {
        if (lane == 0) a.logL[row] = -INFINITY;
        if (a.amps && lane < n) a.amps[row * n + lane] = NAN;
        return;
    }
    const double *gin = a.mge_gram + (size_t)r * MGE_GRAM_STRIDE;
    for (int e = lane; e < n * n; e += 32) Gs[e] = gin[(e / n) * NCG + (e % n)];
    if (lane < n) bs[lane] = gin[MGE_MAX_COL * NCG + lane];
    const double dwd = gin[MGE_MAX_COL * NCG + MGE_MAX_COL];
    __syncwarp();
    nnls_gram_warp<MGE_MAX_COL>(n, Gs, n, bs, dwd, ss, Ls, n);
    if (lane < n && a.amps) a.amps[row * n + lane] = (float)ss[lane];
    // chi^2 = d'Wd - 2 s'b + s'G s at the solved amplitudes (Eq. 5): lane i forms its terms,
    // lane 0 adds them in column order
    if (lane < n) {
        const double si = ss[lane];
        double gi = 0.0;
        for (int k = 0; k < n; ++k) gi += Gs[lane * n + k] * ss[k];
        zs[lane] = si * bs[lane];
        Ls[lane] = si * gi;
    }
    __syncwarp();
    if (lane == 0) {
        double sb = 0.0, sGs = 0.0;
        for (int i = 0; i < n; ++i) {
            if (ss[i] == 0.0) continue;
            sb += zs[i];
            sGs += Ls[i];
        }
        const double chi2 = (dwd - 2.0 * sb) + sGs;
        a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[row / a.rows_per_lens]));
    }
}

}  // namespace tl
