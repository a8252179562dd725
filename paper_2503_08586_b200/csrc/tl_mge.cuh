// tl_mge.cuh -- NEXT-3: MGE lens light with linear amplitudes (tl_loglike_mge_batch).
//
// PAPER.md:291-293 (section 4.3) names the Multiple Gaussian Expansion; reading G23:
//     I_l(theta) = sum_k a_k exp(-R_p(theta)^2 / (2 sigma_k^2)),   R_p of PAPER.md:143-148 Eq. 10,
// one centre and one (q, phi) for the set, fixed sigma_k, and the a_k >= 0 solved together with
// the source amplitudes as the NNLS minimiser of PAPER.md:86-93 Eq. 6 / :97-129 Eq. 7.
//
// Pipeline per chunk of rows (all on one stream; included by tinylens.cu only):
//   prologue_kernel (mge = 1)  lens-light quadratic form becomes t = R_p^2 in arcsec^2
//   trace_lin_kernel           ray-traced unit-amplitude source images -> component slots n_gauss..
//   mge_gauss_kernel           the n_gauss binned Gaussians -> component slots 0..n_gauss-1
//   conv_lin_kernel            every component blurred with the PSF (columns of M)
//   gram_mge_kernel            G = M'WM, b = M'Wd, d'Wd in FP64 (fixed summation order) -> global
//   nnls_mge_kernel            NNLS by the Gram-matrix active-set iteration of Bro & De Jong (the
//                              paper's solver), one warp per row -> amplitudes
//   resid_mge_kernel           chi^2 of the residual d - M s in FP64 -> logL
#pragma once
#include "tl_kernels.cuh"

namespace tl {

constexpr int MGE_MAX_GAUSS = 16;
constexpr int MGE_MAX_COL = MGE_MAX_GAUSS + 2;       // + n_source
constexpr int MGE_SOLVE_THREADS = 128;
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
    const SersicC &C = rc.comp[0];
    const float cXh = C.cXh, cXl = C.cXl, cYh = C.cYh, cYl = C.cYl;
    const float ah = C.ah, al = C.al, b2h = C.b2h, b2l = C.b2l, cch = C.cch, ccl = C.ccl;
    const int S = a.S;
    float ck[NG];
#pragma unroll
    for (int k = 0; k < NG; ++k) ck[k] = -a.mge_c[k];
    const float inv_s2 = 1.f / (float)(S * S);
    const size_t comp_stride = (size_t)a.He * a.pitch;
    float *dst = a.ext + (size_t)r * a.ext_nc * comp_stride;
    const int npx = a.He * a.pitch;
    for (int p = blockIdx.y * blockDim.x + threadIdx.x; p < npx; p += gridDim.y * blockDim.x) {
        const int i = p / a.pitch, j = p - i * a.pitch;
        if (j >= a.We) {                               // pitch padding of every component reads as zero
            for (int k = 0; k < a.ext_nc; ++k) dst[k * comp_stride + (size_t)i * a.pitch + j] = 0.f;
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
    default: return nullptr;
    }
}

// G = M'WM, b = M'Wd, d'Wd: one CTA of 128 threads per row.  The pixels are staged through shared
// memory MGE_TILE at a time (w m_k and m_k, d as doubles, the next tile prefetched into registers);
// every sum has a fixed order, so the result is bitwise reproducible.
// Output: a.mge_gram[r][MGE_GRAM_STRIDE].
__global__ void __launch_bounds__(MGE_SOLVE_THREADS) gram_mge_kernel(const KArgs a, int chunk_rows)
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
    const float *M = a.mimg + (size_t)r * n * npix;
    const float *d = a.data + lens * (size_t)npix, *w = a.wgt + lens * (size_t)npix;
    double *gout = a.mge_gram + (size_t)r * MGE_GRAM_STRIDE;
    // [G | b | d'Wd] = A'B with A = [w m_k | w d], B = [m_k | d]  (n1 = n + 1 columns, the data last).
    // Register blocking: a thread owns a 2 x 2 block of entries (columns 2bi, 2bi+1 of A against
    // 2bj, 2bj+1 of B, bi <= bj) and every Q-th pixel of a tile, so two loads of A and two of B
    // feed four DFMAs (one entry per thread is bound by the shared-memory pipe); the Q pixel
    // slices of an entry are then added in slice order -- a fixed summation order.
    const int n1 = n + 1, NB = (n1 + 1) >> 1, nblk = NB * (NB + 1) / 2;
    const int Q = MGE_SOLVE_THREADS / nblk;                       // >= 2 (nblk <= 55)
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
    constexpr int EPT = (MGE_TILE * NCP + MGE_SOLVE_THREADS - 1) / MGE_SOLVE_THREADS;
    static_assert(MGE_SOLVE_THREADS % MGE_TILE == 0, "a thread stages one pixel of the tile");
    const int ncol = 2 * NB;                                      // n1 rounded up to even: a zero column
    const int sii = threadIdx.x % MGE_TILE, sk0 = threadIdx.x / MGE_TILE;
    float fv[EPT], fwv = 0.f;
    auto fetch = [&](int t0) {
        const int i = t0 + sii;
        fwv = i < npix ? w[i] : 0.f;
#pragma unroll
        for (int u = 0; u < EPT; ++u) {
            const int k = sk0 + u * (MGE_SOLVE_THREADS / MGE_TILE);
            fv[u] = 0.f;
            if (k < n1 && i < npix) fv[u] = k < n ? M[(size_t)k * npix + i] : d[i];
        }
    };
    fetch(0);
    for (int t0 = 0; t0 < npix; t0 += MGE_TILE) {
        __syncthreads();
        {
            const double wd = (double)fwv;
#pragma unroll
            for (int u = 0; u < EPT; ++u) {
                const int k = sk0 + u * (MGE_SOLVE_THREADS / MGE_TILE);
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

// NNLS: one warp per row (lane 0 iterates; the iteration is a chain of dependent FP64 operations
// through shared memory, so what matters is how many rows are in flight per SM: 4 warps per CTA,
// ~6 KB of shared memory each).  Writes the amplitudes (FP64, for resid_mge_kernel; float for the
// caller) and reports invalid rows.
__global__ void __launch_bounds__(32 * MGE_NNLS_WARPS) nnls_mge_kernel(const KArgs a, int chunk_rows)
{
    constexpr int NCP = MGE_MAX_COL + 1;
    __shared__ double Gw[MGE_NNLS_WARPS][MGE_GRAM_STRIDE];
    __shared__ double Lw[MGE_NNLS_WARPS][MGE_MAX_COL * MGE_MAX_COL];
    __shared__ double zw[MGE_NNLS_WARPS][MGE_MAX_COL], sw[MGE_NNLS_WARPS][MGE_MAX_COL];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * MGE_NNLS_WARPS + wid;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    const int n = a.ext_nc;
    if (!row_is_valid(a.rows[r], a.n_comp)) {
        if (lane == 0) a.logL[row] = -INFINITY;
        if (a.amps && lane < n) a.amps[row * n + lane] = NAN;
        return;
    }
    const double *gin = a.mge_gram + (size_t)r * MGE_GRAM_STRIDE;
    for (int e = lane; e < MGE_GRAM_STRIDE; e += 32) Gw[wid][e] = gin[e];
    __syncwarp();
    if (lane == 0)
        nnls_gram<MGE_MAX_COL>(n, Gw[wid], NCP, Gw[wid] + MGE_MAX_COL * NCP, Gw[wid][MGE_MAX_COL * NCP + MGE_MAX_COL], sw[wid], Lw[wid], zw[wid]);
    __syncwarp();
    if (lane < n) {
        a.mge_sol[(size_t)r * MGE_MAX_COL + lane] = sw[wid][lane];
        if (a.amps) a.amps[row * n + lane] = (float)sw[wid][lane];
    }
}

// chi^2 of the residual d - M s in FP64 (never via d'Wd - 2 s'b + s'Gs, which cancels) -> logL.
// One CTA per row; the loads of a pixel's n columns are independent.
__global__ void __launch_bounds__(256) resid_mge_kernel(const KArgs a, int chunk_rows)
{
    __shared__ double red[32];
    __shared__ double ss[MGE_MAX_COL];
    const int r = blockIdx.x;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    const int n = a.ext_nc;
    if (!row_is_valid(a.rows[r], a.n_comp)) return;
    const int64_t lens = row / a.rows_per_lens;
    const int npix = a.ny * a.nx;
    const float *M = a.mimg + (size_t)r * n * npix;
    const float *d = a.data + lens * (size_t)npix, *w = a.wgt + lens * (size_t)npix;
    if (threadIdx.x < MGE_MAX_COL) ss[threadIdx.x] = threadIdx.x < n ? a.mge_sol[(size_t)r * MGE_MAX_COL + threadIdx.x] : 0.0;
    __syncthreads();
    double part = 0.0;
    for (int i = threadIdx.x; i < npix; i += blockDim.x) {
        float mv[MGE_MAX_COL];
#pragma unroll
        for (int k = 0; k < MGE_MAX_COL; ++k) mv[k] = k < n ? M[(size_t)k * npix + i] : 0.f;
        double m = 0.0;
#pragma unroll
        for (int k = 0; k < MGE_MAX_COL; ++k) if (k < n) m += ss[k] * (double)mv[k];
        const double res = (double)d[i] - m;
        part += res * res * (double)w[i];
    }
    const double chi2 = block_sum(part, red);
    if (threadIdx.x == 0) a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[lens]));
}

}  // namespace tl
