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

}  // namespace tl
