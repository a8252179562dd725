// tl_nnls.cuh -- the non-negative least-squares solver of the linear-amplitude modes.
//
// PAPER.md:123-129 (Eq. 7 and the sentence after it): the amplitudes minimise ||(M s - d)/n||^2
// subject to s >= 0, "solved with the fast non-negative least-squares (fnnls) algorithm of Bro &
// De Jong (1997)" -- the Lawson-Hanson active-set iteration run on the cross products G = M'WM,
// b = M'Wd instead of on M.  Used by tl_loglike_linear_batch (<= 3 columns) and
// tl_loglike_mge_batch (<= MGE_MAX_COL columns).  Written from the mathematics; the oracle reaches
// the same optimum by a different route (enumeration of supports / its own FP64 active set).
#pragma once

namespace tl {

// minimise s'G s - 2 b's over s >= 0 (n <= MAXC <= 32 columns) -- one thread.  Active-set iteration on
// the Gram matrix (Lawson & Hanson; in this cross-product form Bro & De Jong's "fast NNLS"):
// the passive set P grows by the column with the largest positive gradient w = b - G s, the
// unconstrained problem on P is solved by Cholesky, and a step towards it that would leave the
// feasible region is cut at the boundary, the columns that reach 0 leaving P.
// G is [n][ldg]; L (scratch) [n][ldl]; z (scratch) [n]; dwd = d'Wd sets the scale of "zero".
template <int MAXC>
__device__ inline void nnls_gram(int n, const double *G, int ldg, const double *b, double dwd, double *s,
                                 double *L, double *z, int ldl = MAXC)
{
    int idx[MAXC];
    int m = 0;
    unsigned passive = 0u, banned = 0u;
    for (int i = 0; i < n; ++i) s[i] = 0.0;
    const double eps = 1e-10;
    for (int outer = 0; outer < 3 * n + 3; ++outer) {
        int j = -1;
        double wbest = 0.0;
        for (int i = 0; i < n; ++i) {
            if ((passive | banned) & (1u << i)) continue;
            double w = b[i];
            for (int k = 0; k < n; ++k) w -= G[i * ldg + k] * s[k];
            const double thr = eps * sqrt(fmax(G[i * ldg + i] * dwd, 0.0));
            if (w > thr && w > wbest) { wbest = w; j = i; }
        }
        if (j < 0) break;
        passive |= 1u << j;
        bool first = true, added = true;
        for (int inner = 0; inner <= n; ++inner) {
            m = 0;
            for (int i = 0; i < n; ++i) if (passive & (1u << i)) idx[m++] = i;
            // Cholesky G_PP = L L'
            bool pd = true;
            for (int r = 0; r < m && pd; ++r) {
                for (int c = 0; c <= r; ++c) {
                    double v = G[idx[r] * ldg + idx[c]];
                    for (int k = 0; k < c; ++k) v -= L[r * ldl + k] * L[c * ldl + k];
                    if (c == r) {
                        if (!(v > 1e-13 * G[idx[r] * ldg + idx[r]])) { pd = false; break; }
                        L[r * ldl + r] = rsqrt(v);             // the diagonal is kept as 1 / l_rr
                    } else L[r * ldl + c] = v * L[c * ldl + c];
                }
            }
            if (pd) {
                for (int r = 0; r < m; ++r) {
                    double v = b[idx[r]];
                    for (int k = 0; k < r; ++k) v -= L[r * ldl + k] * z[k];
                    z[r] = v * L[r * ldl + r];
                }
                for (int r = m - 1; r >= 0; --r) {
                    double v = z[r];
                    for (int k = r + 1; k < m; ++k) v -= L[k * ldl + r] * z[k];
                    z[r] = v * L[r * ldl + r];
                }
            }
            if (first) {
                // the entering column must come out positive; if it is numerically dependent on P
                // (or rounding makes it non-positive) it is set aside until P changes
                int pj = 0;
                for (int r = 0; r < m; ++r) if (idx[r] == j) pj = r;
                if (!pd || !(z[pj] > 0.0)) { passive &= ~(1u << j); banned |= 1u << j; added = false; break; }
                first = false;
            } else if (!pd) break;                       // cannot happen for a subset of a PD set; keep s
            double alpha = 2.0;
            int rmin = -1;
            for (int r = 0; r < m; ++r)
                if (!(z[r] > 0.0)) {
                    const double si = s[idx[r]];
                    const double al = si / (si - z[r]);
                    if (al < alpha) { alpha = al; rmin = r; }
                }
            if (rmin < 0) {                               // all positive: accept
                for (int r = 0; r < m; ++r) s[idx[r]] = z[r];
                break;
            }
            for (int r = 0; r < m; ++r) {
                const int i = idx[r];
                s[i] += alpha * (z[r] - s[i]);
                if (r == rmin || !(s[i] > 0.0)) { s[i] = 0.0; passive &= ~(1u << i); }
            }
        }
        if (added) banned = 0u;
    }
}

// The same iteration run by a whole warp (tl_loglike_mge_batch: up to 32 columns; one lane spent ~0.3 ms on
// a row of 11 columns, every step a shared-memory load feeding one dependent DFMA).  Lane i owns gradient
// entry i; lane r owns row r of the Cholesky factor and entry r of the triangular solves, which run as
// column sweeps; maxima / minima and the sets are warp votes, so every lane follows the same path.
// Each sum runs over k in nnls_gram's order except the back-substitution, which subtracts its terms from the
// last column down; ties are broken as there (lowest index).  G, b, s, L in shared memory; all 32 lanes call.
template <int MAXC>
__device__ inline void nnls_gram_warp(int n, const double *G, int ldg, const double *b, double dwd, double *s,
                                      double *L, int ldl)
{
    static_assert(MAXC <= 32, "one lane per column");
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    unsigned passive = 0u, banned = 0u;
    if (lane < n) s[lane] = 0.0;
    __syncwarp();
    const double eps = 1e-10;
    for (int outer = 0; outer < 3 * n + 3; ++outer) {
        double w = 0.0;
        bool cand = false;
        if (lane < n && !(((passive | banned) >> lane) & 1u)) {
            w = b[lane];
            for (int k = 0; k < n; ++k) w -= G[lane * ldg + k] * s[k];
            cand = w > eps * sqrt(fmax(G[lane * ldg + lane] * dwd, 0.0));
        }
        double wmax = cand ? w : -1.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) wmax = fmax(wmax, __shfl_xor_sync(FULL, wmax, o));
        const unsigned hit = __ballot_sync(FULL, cand && w == wmax);
        if (!hit) break;
        const int j = __ffs(hit) - 1;
        passive |= 1u << j;
        bool first = true, added = true;
        for (int inner = 0; inner <= n; ++inner) {
            const int m = __popc(passive);
            const int my_i = lane < m ? (int)__fns(passive, 0, lane + 1) : 0;     // column of passive position `lane`
            // Cholesky G_PP = L L', column by column (the diagonal is kept as 1 / l_cc)
            bool pd = true;
            for (int c = 0; c < m; ++c) {
                const int ic = __shfl_sync(FULL, my_i, c);
                double v = 0.0;
                if (lane >= c && lane < m) {
                    v = G[my_i * ldg + ic];
                    for (int k = 0; k < c; ++k) v -= L[lane * ldl + k] * L[c * ldl + k];
                }
                const double vcc = __shfl_sync(FULL, v, c);
                if (!(vcc > 1e-13 * G[ic * ldg + ic])) { pd = false; break; }
                const double inv = rsqrt(vcc);
                if (lane == c) L[c * ldl + c] = inv;
                else if (lane > c && lane < m) L[lane * ldl + c] = v * inv;
                __syncwarp();
            }
            double zr = 0.0;                                     // entry `lane` of the unconstrained solution on P
            if (pd) {
                double v = lane < m ? b[my_i] : 0.0;
                for (int k = 0; k < m; ++k) {
                    const double zk = __shfl_sync(FULL, v * L[k * ldl + k], k);
                    if (lane == k) v = zk;
                    else if (lane > k && lane < m) v -= L[lane * ldl + k] * zk;
                }
                for (int k = m - 1; k >= 0; --k) {
                    const double zk = __shfl_sync(FULL, v * L[k * ldl + k], k);
                    if (lane == k) v = zk;
                    else if (lane < k) v -= L[k * ldl + lane] * zk;
                }
                zr = v;
            }
            if (first) {
                // the entering column must come out positive; if it is numerically dependent on P
                // (or rounding makes it non-positive) it is set aside until P changes
                const double zj = __shfl_sync(FULL, zr, __popc(passive & ((1u << j) - 1u)));
                if (!pd || !(zj > 0.0)) { passive &= ~(1u << j); banned |= 1u << j; added = false; break; }
                first = false;
            } else if (!pd) break;                       // cannot happen for a subset of a PD set; keep s
            const double si = lane < m ? s[my_i] : 0.0;
            double al = 2.0;
            if (lane < m && !(zr > 0.0)) al = si / (si - zr);
            double amin = al < 2.0 ? al : 2.0;                   // (a NaN does not take part)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) amin = fmin(amin, __shfl_xor_sync(FULL, amin, o));
            const unsigned hitr = __ballot_sync(FULL, lane < m && al < 2.0 && al == amin);
            if (!hitr) {                                         // all positive: accept
                if (lane < m) s[my_i] = zr;
                __syncwarp();
                break;
            }
            const int rmin = __ffs(hitr) - 1;
            bool drop = false;
            if (lane < m) {
                double sn = si + amin * (zr - si);
                if (lane == rmin || !(sn > 0.0)) { sn = 0.0; drop = true; }
                s[my_i] = sn;
            }
            passive &= ~__reduce_or_sync(FULL, drop ? (1u << my_i) : 0u);
            __syncwarp();
        }
        if (added) banned = 0u;
    }
    __syncwarp();
}

}  // namespace tl
