// tl_kernels.cuh -- the hot-path kernels (steps a1..a8 of DESIGN.md).
//
// fused_kernel: persistent CTAs, one parameter row at a time per CTA.
//   phase 1  every thread ray-traces whole native pixels (S*S sub-samples accumulated in a
//            register = step a5) and stores the binned value into the extended image held
//            in shared memory;
//   phase 2  register-blocked direct PSF convolution (1 x 4 output strip per thread, LDS.128
//            for both the image window and the taps) straight from shared memory, followed
//            by the chi^2 terms against data / inverse-variance read through L2;
//   phase 3  deterministic FP64 reduction: per-thread partial -> warp shuffle tree -> fixed
//            order over warps.  No atomics, so logL is bitwise reproducible.
// The split path (large images) runs phase 1 into global memory (trace_kernel) and phases
// 2-3 from shared-memory tiles of it (conv_kernel + finalize_kernel).
#pragma once
#include <type_traits>
#include "tl_sample.cuh"
#include "tl_pair.cuh"
#include "tl_nnls.cuh"

namespace tl {

constexpr int CONV_R = 4;            // outputs per thread strip (along x)

// Programmatic dependent launch (the small-batch path, whose cost is launch latency): a kernel launched
// with cudaLaunchAttributeProgrammaticStreamSerialization may start while its predecessor still runs;
// pdl_wait() blocks until the predecessor has completed and its writes are visible, pdl_launch() lets
// the successor's CTAs be scheduled early.  Both are no-ops for ordinary launches.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

struct KArgs {
    const RowC *rows;        // [B] derived constants
    const float *psf;        // [n_lens][K][Kp]  flipped, rows zero-padded to Kp (multiple of 4)
    const float *data;       // [n_lens][ny][nx]
    const float *wgt;        // [n_lens][ny][nx]  1 / sigma^2
    const double *lconst;    // [n_lens]          sum ln(2 pi sigma^2)
    float *logL;             // [B] or null
    float *images;           // [B][ny][nx] or null
    float *ext;              // split path: [chunk][He][pitch] binned extended images
    double *partial;         // split path: [chunk][n_tiles] chi^2 partials
    float *mimg;             // linear mode: [chunk][C][ny][nx] blurred unit-amplitude component images
    float *amps;             // linear mode: [B][C] solved amplitudes or null
    int64_t B, rows_per_lens, row0;
    int ny, nx, K, Kp, h, He, We, pitch, S, n_lens_light, n_comp, edge_zero;
    int tile_rows, n_tiles;  // split path
    int CW, CH, tiles_x, tiles_y;   // phase-1 warp tiles (see trace_tiles)
    int rowtab;              // 1: the kernel's shared memory holds a RowV table (He * S entries)
    int *tile_counters;      // small-batch path: [chunk] zeroed work-queue heads (one per row), else null
    // MGE mode (tl_mge.cuh): ext / mimg hold ext_nc = n_gauss + n_source components per row;
    // trace_lin_kernel writes its components from slot ext_k0 on (0, 0 = the linear-mode layout)
    int ext_nc, ext_k0, n_gauss;
    // AUTO precision (fused path): rows whose first-order FP32 error bound exceeds the tolerance are
    // appended to flag_list (their count in *flag_count) for re-evaluation by the FP64 path
    int *flag_count, *flag_list;
    float err_coh, err_rnd;  // bound = err_coh |sum e_i| + err_rnd sqrt(sum e_i^2),  e_i = (d_i - m_i) m_i / sigma_i^2
    const float *mge_c;      // [n_gauss] log2(e) / (2 sigma_k^2), arcsec^-2
    const int *mge_set;      // [n_gauss] the set (0 .. n_lens_light-1) Gaussian k belongs to: its shape is comp[n_source + set]
    int mge_k0, mge_shape;   // mge_gauss_kernel (unfused path, one launch per set): first Gaussian and set of this launch
    double *mge_gram;        // [chunk][MGE_GRAM_STRIDE]  G | b | d'Wd
    const double *mimg64;    // FP64 MGE pipeline: [chunk][C][ny][nx] blurred columns in double, and
    const double *wgt64;     //                    [n_lens][ny][nx] 1 / sigma^2 in double
    // conv_lin_kernel: component strides of ext and of mimg, first mimg slot (0, 0, 0 = gridDim.z, gridDim.z, 0)
    int conv_ext_nc, conv_m_nc, conv_m_k0;
};

__device__ __forceinline__ bool row_is_valid(const RowC &rc, int n_comp)
{
    bool ok = rc.lens.valid != 0;
    for (int k = 0; k < n_comp; ++k) ok = ok && (rc.comp[k].valid != 0);
    return ok;
}

// Values that depend only on the sub-sample column (abscissa X) / only on the sub-sample row
// (ordinate Y).  x' = Pc + Qs, y' = Qc - Ps, N (theta - c) + D0 = (U + V, U2 + V2); the
// lens-light quadratic form is  t = LA + LC + LB * dyl.
struct ColV { float Pc, Ps, U, U2, LA, LB; };
struct alignas(16) RowV { float Qc, Qs, V, V2, LC, dyl, pad0, pad1; };      // 32 bytes: two LDS.128

template <int NLL>
__device__ __forceinline__ ColV col_values(const RowC &rc, float X)
{
    const LensC &L = rc.lens;
    ColV c;
    const float dx = X - L.cXa;                                  // exact
    c.Pc = fmaf(dx, L.ch, fmaf(dx, L.cl, L.pcC));
    c.Ps = fmaf(dx, L.sh, fmaf(dx, L.sl, L.psC));
    c.U = fmaf(dx, L.n11h, fmaf(dx, L.n11l, L.uC));
    c.U2 = fmaf(dx, L.n21h, fmaf(dx, L.n21l, L.u2C));
    if (NLL) {
        const SersicC &C = rc.comp[0];
        const float dxl = (X - C.cXh) - C.cXl;                    // first difference exact
        const float x2 = dxl * dxl;
        c.LA = fmaf(C.ah, x2, C.al * x2);
        c.LB = fmaf(dxl, C.b2h, dxl * C.b2l);
    } else { c.LA = 0.f; c.LB = 0.f; }
    return c;
}

// Column values of two horizontally adjacent sub-samples as register pairs (tl_pair.cuh)
struct ColV2 { f2 Pc, Ps, U, U2, LA, LB; };
template <int NLL>
__device__ __forceinline__ ColV2 col_values2(const RowC &rc, float Xa, float Xb)
{
    const ColV a = col_values<NLL>(rc, Xa), b = col_values<NLL>(rc, Xb);
    ColV2 c;
    c.Pc = mk2(a.Pc, b.Pc); c.Ps = mk2(a.Ps, b.Ps); c.U = mk2(a.U, b.U); c.U2 = mk2(a.U2, b.U2);
    c.LA = mk2(a.LA, b.LA); c.LB = mk2(a.LB, b.LB);
    return c;
}

template <int NLL>
__device__ __forceinline__ RowV row_values(const RowC &rc, float Y)
{
    const LensC &L = rc.lens;
    RowV r;
    const float dy = Y - L.cYa;                                  // exact
    r.Qc = fmaf(dy, L.ch, fmaf(dy, L.cl, L.qcC));
    r.Qs = fmaf(dy, L.sh, fmaf(dy, L.sl, L.qsC));
    r.V = fmaf(dy, L.n12h, fmaf(dy, L.n12l, L.vL)) + L.d1h;
    r.V2 = fmaf(dy, L.n22h, fmaf(dy, L.n22l, L.v2L)) + L.d2h;
    if (NLL) {
        const SersicC &C = rc.comp[0];
        r.dyl = (Y - C.cYh) - C.cYl;
        const float y2 = r.dyl * r.dyl;
        r.LC = fmaf(C.cch, y2, C.ccl * y2);
    } else { r.dyl = 0.f; r.LC = 0.f; }
    r.pad0 = r.pad1 = 0.f;
    return r;
}

// Register-resident constants of one row for the sample loop.
template <int NLL, int NSRC, int MASS = MASS_SIE>
struct HotC {
    typename std::conditional<MASS == MASS_EPL, EplHot, SieHot>::type sie;
    SersicHot ll;                 // lens light (NLL = 1)
    SersicHot src[NSRC];
    QuadHot q[NSRC];
    __device__ __forceinline__ explicit HotC(const RowC &rc) : sie(rc.lens)
    {
        if (NLL) ll = SersicHot(rc.comp[0]);
#pragma unroll
        for (int k = 0; k < NSRC; ++k) { src[k] = SersicHot(rc.comp[NLL + k]); q[k] = QuadHot(rc.comp[NLL + k]); }
    }
};

// One sub-sample (steps a2-a4, Eq. 2): lens light at theta (added to `acc`) and
// sources at beta (returned), both already scaled by 1/S^2 so that the caller only adds
// (step a5, bin = mean).  FAST = polynomial SIE path (q >= 0.5) / FP32 EPL series.
template <int NLL, int NSRC, bool FAST, int MASS>
__device__ __forceinline__ void sample_value(const RowC &rc, const HotC<NLL, NSRC, MASS> &h, const ColV &c, const RowV &r,
                                             float &acc, float (&src)[NSRC], bool &flag)
{
    bool fl;
    if (NLL) acc = fmaf(h.ll.amp, sersic_from_t(h.ll, fmaf(c.LB, r.dyl, c.LA + r.LC), fl), acc);
    const float xp = c.Pc + r.Qs, yp = r.Qc - c.Ps;
    float axp, ayp;
    if constexpr (MASS == MASS_EPL) {
        if (FAST) epl_alpha(h.sie, rc.lens.ecoef, xp, yp, axp, ayp);
        else epl_alpha_slow(rc.lens, xp, yp, axp, ayp);
    } else {
        if (FAST) sie_alpha(h.sie, xp, yp, axp, ayp);
        else sie_alpha_slow(rc.lens, xp, yp, axp, ayp);
    }
    const float bx = (c.U + r.V) - axp, by = (c.U2 + r.V2) - ayp;      // R^T (beta - s_1)
    src[0] = h.src[0].amp * sersic_from_t(h.src[0], quad_form(h.q[0], bx, by), fl);
    flag = fl;
    if (NSRC > 1) {
        const float t2 = quad_form(h.q[1], (bx - h.q[1].oxh) - h.q[1].oxl, (by - h.q[1].oyh) - h.q[1].oyl);
        src[NSRC - 1] = h.src[1].amp * sersic_from_t(h.src[1], t2, fl);
        flag = flag || fl;
    }
}

// Two horizontally adjacent sub-samples at once with packed FP32 arithmetic (tl_pair.cuh): the
// lens-light profile values go to `llv` (not yet scaled by the amplitude), the sources are returned
// (a half is NaN when that sample wants the FP64 ray-trace).
// MASS_EPL: (axp, ayp) come from the caller, which deflects the pairs of a sub-row together (epl_alpha_pairs).
template <int NLL, int NSRC, int MASS = MASS_SIE>
__device__ __forceinline__ f2 sample_pair_parts(const HotC<NLL, NSRC, MASS> &h, const ColV2 &c, const RowV &r, f2 &llv, bool &any,
                                                f2 axp = f2{0ull}, f2 ayp = f2{0ull})
{
    if (NLL) llv = sersic_from_t2(h.ll, fma2(c.LB, bc2(r.dyl), add2(c.LA, bc2(r.LC))));
    if constexpr (MASS == MASS_SIE) {
        const f2 xp = add2(c.Pc, bc2(r.Qs)), yp = fma2(c.Ps, bc2(-1.f), bc2(r.Qc));
        sie_alpha2(h.sie, xp, yp, axp, ayp);
    }
    const f2 bx = fma2(axp, bc2(-1.f), add2(c.U, bc2(r.V))), by = fma2(ayp, bc2(-1.f), add2(c.U2, bc2(r.V2)));   // R^T (beta - s_1)
    bool f0, f1;
    f2 s = mul2(bc2(h.src[0].amp), sersic_from_t2(h.src[0], quad_form2(h.q[0], bx, by), f0, f1));
    if (NSRC > 1) {
        const f2 ex = add2(add2(bx, bc2(-h.q[1].oxh)), bc2(-h.q[1].oxl)), ey = add2(add2(by, bc2(-h.q[1].oyh)), bc2(-h.q[1].oyl));
        bool g0, g1;
        s = fma2(bc2(h.src[1].amp), sersic_from_t2(h.src[1], quad_form2(h.q[1], ex, ey), g0, g1), s);
        f0 = f0 || g0; f1 = f1 || g1;
    }
    float s0, s1;
    un2(s, s0, s1);
    if (f0) s0 = __int_as_float(0x7fc00000);           // NaN marks "refine me"
    if (f1) s1 = __int_as_float(0x7fc00000);
    any = any || f0 || f1;
    return mk2(s0, s1);
}
// Linear-amplitude mode: the sources stay apart (s[k], each at its unit amplitude); a half of s[0] is NaN
// when that sample wants the FP64 ray-trace.
template <int NLL, int NSRC, int MASS = MASS_SIE>
__device__ __forceinline__ void sample_pair_comps(const HotC<NLL, NSRC, MASS> &h, const ColV2 &c, const RowV &r, f2 &llv,
                                                  f2 (&s)[NSRC], bool &any, f2 axp = f2{0ull}, f2 ayp = f2{0ull})
{
    if (NLL) llv = sersic_from_t2(h.ll, fma2(c.LB, bc2(r.dyl), add2(c.LA, bc2(r.LC))));
    if constexpr (MASS == MASS_SIE) {
        const f2 xp = add2(c.Pc, bc2(r.Qs)), yp = fma2(c.Ps, bc2(-1.f), bc2(r.Qc));
        sie_alpha2(h.sie, xp, yp, axp, ayp);
    }
    const f2 bx = fma2(axp, bc2(-1.f), add2(c.U, bc2(r.V))), by = fma2(ayp, bc2(-1.f), add2(c.U2, bc2(r.V2)));   // R^T (beta - s_1)
    bool f0, f1;
    s[0] = mul2(bc2(h.src[0].amp), sersic_from_t2(h.src[0], quad_form2(h.q[0], bx, by), f0, f1));
    if (NSRC > 1) {
        const f2 ex = add2(add2(bx, bc2(-h.q[1].oxh)), bc2(-h.q[1].oxl)), ey = add2(add2(by, bc2(-h.q[1].oyh)), bc2(-h.q[1].oyl));
        bool g0, g1;
        s[NSRC - 1] = mul2(bc2(h.src[1].amp), sersic_from_t2(h.src[1], quad_form2(h.q[1], ex, ey), g0, g1));
        f0 = f0 || g0; f1 = f1 || g1;
    }
    if (f0 || f1) {
        float s0, s1;
        un2(s[0], s0, s1);
        if (f0) s0 = __int_as_float(0x7fc00000);       // NaN marks "refine me"
        if (f1) s1 = __int_as_float(0x7fc00000);
        s[0] = mk2(s0, s1);
        any = true;
    }
}
// ... with the lens light added to `acc2`
template <int NLL, int NSRC, int MASS = MASS_SIE>
__device__ __forceinline__ f2 sample_pair(const HotC<NLL, NSRC, MASS> &h, const ColV2 &c, const RowV &r, f2 &acc2, bool &any,
                                          f2 axp = f2{0ull}, f2 ayp = f2{0ull})
{
    f2 llv;
    llv.v = 0ull;
    const f2 s = sample_pair_parts<NLL, NSRC, MASS>(h, c, r, llv, any, axp, ayp);
    if (NLL) acc2 = fma2(bc2(h.ll.amp), llv, acc2);
    return s;
}

// Steps a3-a4 of one sub-sample once its deflection is known (EPL: the deflections of the S_T
// sub-samples of a pixel row are computed together, see epl_alpha_vec).
template <int NLL, int NSRC, int MASS>
__device__ __forceinline__ void sample_light(const HotC<NLL, NSRC, MASS> &h, const ColV &c, const RowV &r, float axp, float ayp,
                                             float &acc, float (&src)[NSRC], bool &flag)
{
    bool fl;
    if (NLL) acc = fmaf(h.ll.amp, sersic_from_t(h.ll, fmaf(c.LB, r.dyl, c.LA + r.LC), fl), acc);
    const float bx = (c.U + r.V) - axp, by = (c.U2 + r.V2) - ayp;      // R^T (beta - s_1)
    src[0] = h.src[0].amp * sersic_from_t(h.src[0], quad_form(h.q[0], bx, by), fl);
    flag = fl;
    if (NSRC > 1) {
        const float t2 = quad_form(h.q[1], (bx - h.q[1].oxh) - h.q[1].oxl, (by - h.q[1].oyh) - h.q[1].oyl);
        src[NSRC - 1] = h.src[1].amp * sersic_from_t(h.src[1], t2, fl);
        flag = flag || fl;
    }
}

// steps a1-a5 for a run of `count` warp tiles.  A warp tile is CW x CH = 32 extended native
// pixels (lane -> column lane % CW, row lane / CW), so the samples a warp works on are
// neighbours in the image (coherent refinement branches) and all lanes are busy; tiles are
// numbered column-major (t = c * tiles_y + r), so a thread's column -- and the column values it
// keeps in registers -- changes only when the whole warp moves to the next tile column.
// S_T > 0: compile-time supersampling; S_T = 0: any S (column values recomputed per sample).
// `next()` yields the warp's next tile index (uniform over the warp) or -1.
// `rowtab` (optional, shared memory): the RowV of every sub-sample row of the image, filled once
// per parameter row by fill_rowtab(); without it each thread recomputes them (18 instructions
// per sub-row instead of two LDS.128).
// LIN (linear-amplitude mode): the components are kept apart and handed to store(i, j, k, v),
// k = 0 .. NLL + NSRC - 1; otherwise their sum goes to store(i, j, v).
template <int S_T, int NLL, int NSRC, bool FAST, bool LIN, int MASS, class Next, class Store>
__device__ __forceinline__ void trace_tiles(const RowC &rc, const HotC<NLL, NSRC, MASS> &h, const KArgs &a,
                                            const RowV *rowtab, Next next, Store store)
{
    const int S = S_T > 0 ? S_T : a.S;
    const int lane = threadIdx.x & 31;
    const int lj = lane % a.CW, li = lane / a.CW;
    int tile = next();
    if (tile < 0) return;
    int c = tile / a.tiles_y, r = tile - c * a.tiles_y;
    int j = c * a.CW + lj;
    // u-units: X = 2 (j S + b) + 1 - S We is the exact sub-sample abscissa (DESIGN.md a1)
    float X0 = (float)(2 * j * S + 1 - S * a.We);
    // even compile-time S, SIE polynomial path, components summed: pairs of sub-samples (tl_pair.cuh)
    constexpr bool PAIR = S_T > 0 && S_T % 2 == 0 && FAST;     // SIE polynomial path / FP32 EPL series
    constexpr int NP = PAIR ? S_T / 2 : 1;
    ColV cv[(S_T > 0 && !PAIR) ? S_T : 1];
    ColV2 cv2[NP];
    auto load_cols = [&]() {
        if constexpr (PAIR) {
#pragma unroll
            for (int b = 0; b < NP; ++b) cv2[b] = col_values2<NLL>(rc, X0 + (float)(4 * b), X0 + (float)(4 * b + 2));
        } else if (S_T > 0) {
#pragma unroll
            for (int b = 0; b < S_T; ++b) cv[b] = col_values<NLL>(rc, X0 + (float)(2 * b));
        }
    };
    load_cols();
#pragma unroll 1
    for (;;) {
        const int i = r * a.CH + li;
        if (i < a.He && j < a.We) {
            float acc = 0.f;                           // lens light (and, unless LIN, everything)
            float accs[NSRC];                          // LIN: the sources, each on its own
#pragma unroll
            for (int k = 0; k < NSRC; ++k) accs[k] = 0.f;
            const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
            if (!edge) {
                const float Y0 = (float)(2 * i * S + 1 - S * a.He);
                f2 acc2 = bc2(0.f);
                f2 accs2[NSRC];                        // (LIN with pairs)
#pragma unroll
                for (int k = 0; k < NSRC; ++k) accs2[k] = bc2(0.f);
#pragma unroll 1
                for (int sa = 0; sa < S; ++sa) {
                    const float Y = Y0 + (float)(2 * sa);
                    const RowV rv = rowtab ? rowtab[i * S + sa] : row_values<NLL>(rc, Y);
                    f2 dax[NP], day[NP];                            // EPL: the deflections of the sub-row's pairs, together
                    if constexpr (PAIR && MASS == MASS_EPL) {
                        f2 xp[NP], yp[NP];
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp) {
                            xp[sp] = add2(cv2[sp].Pc, bc2(rv.Qs));
                            yp[sp] = fma2(cv2[sp].Ps, bc2(-1.f), bc2(rv.Qc));
                        }
                        epl_alpha_pairs<NP>(h.sie, rc.lens.ecoef, xp, yp, dax, day);
                    } else {
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp) { dax[sp].v = 0ull; day[sp].v = 0ull; }
                    }
                    if constexpr (PAIR && LIN) {
                        f2 sk[NP][NSRC];
                        bool any = false;
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp) {
                            f2 llv;
                            llv.v = 0ull;
                            sample_pair_comps<NLL, NSRC, MASS>(h, cv2[sp], rv, llv, sk[sp], any, dax[sp], day[sp]);
                            if (NLL) acc2 = fma2(bc2(h.ll.amp), llv, acc2);
                        }
                        if (any) {                                  // rare: FP64 ray-trace, out of line
#pragma unroll
                            for (int sp = 0; sp < NP; ++sp) {
                                float m0, m1;
                                un2(sk[sp][0], m0, m1);
                                if (m0 != m0 || m1 != m1) {
#pragma unroll
                                    for (int k = 0; k < NSRC; ++k) {
                                        float s0, s1;
                                        un2(sk[sp][k], s0, s1);
                                        if (m0 != m0) s0 = refined_source_light_k<MASS>(rc, NLL + k, X0 + (float)(4 * sp), Y);
                                        if (m1 != m1) s1 = refined_source_light_k<MASS>(rc, NLL + k, X0 + (float)(4 * sp + 2), Y);
                                        sk[sp][k] = mk2(s0, s1);
                                    }
                                }
                            }
                        }
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp)
#pragma unroll
                            for (int k = 0; k < NSRC; ++k) accs2[k] = add2(accs2[k], sk[sp][k]);
                    } else if constexpr (PAIR) {
                        f2 src2[NP];
                        bool any = false;
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp) src2[sp] = sample_pair<NLL, NSRC, MASS>(h, cv2[sp], rv, acc2, any, dax[sp], day[sp]);
                        if (any) {                                  // rare: FP64 ray-trace, out of line
#pragma unroll
                            for (int sp = 0; sp < NP; ++sp) {
                                float s0, s1;
                                un2(src2[sp], s0, s1);
                                if (s0 != s0) s0 = refined_source_light<MASS>(rc, NLL, NLL + NSRC, X0 + (float)(4 * sp), Y);
                                if (s1 != s1) s1 = refined_source_light<MASS>(rc, NLL, NLL + NSRC, X0 + (float)(4 * sp + 2), Y);
                                src2[sp] = mk2(s0, s1);
                            }
                        }
#pragma unroll
                        for (int sp = 0; sp < NP; ++sp) acc2 = add2(acc2, src2[sp]);
                    } else if constexpr (S_T > 0) {
                        float src[S_T > 0 ? S_T : 1][NSRC];
                        bool any = false;
                        if constexpr (MASS == MASS_EPL && FAST) {
                            float xp[S_T > 0 ? S_T : 1], yp[S_T > 0 ? S_T : 1], axp[S_T > 0 ? S_T : 1], ayp[S_T > 0 ? S_T : 1];
#pragma unroll
                            for (int sb = 0; sb < S_T; ++sb) { xp[sb] = cv[sb].Pc + rv.Qs; yp[sb] = rv.Qc - cv[sb].Ps; }
                            epl_alpha_vec<(S_T > 0 ? S_T : 1)>(h.sie, rc.lens.ecoef, xp, yp, axp, ayp);
#pragma unroll
                            for (int sb = 0; sb < S_T; ++sb) {
                                bool fl;
                                sample_light<NLL, NSRC, MASS>(h, cv[sb], rv, axp[sb], ayp[sb], acc, src[sb], fl);
                                any = any || fl;
                                if (fl) src[sb][0] = __int_as_float(0x7fc00000);
                            }
                        } else {
#pragma unroll
                        for (int sb = 0; sb < S_T; ++sb) {
                            bool fl;
                            sample_value<NLL, NSRC, FAST, MASS>(rc, h, cv[sb], rv, acc, src[sb], fl);
                            any = any || fl;
                            if (fl) src[sb][0] = __int_as_float(0x7fc00000);      // NaN marks "refine me"
                        }
                        }
                        if (any) {                                  // rare: FP64 ray-trace, out of line
#pragma unroll
                            for (int sb = 0; sb < S_T; ++sb)
                                if (src[sb][0] != src[sb][0]) {
                                    if (LIN && NSRC > 1) {
#pragma unroll
                                        for (int k = 0; k < NSRC; ++k)
                                            src[sb][k] = refined_source_light_k<MASS>(rc, NLL + k, X0 + (float)(2 * sb), Y);
                                    } else {
                                        src[sb][0] = refined_source_light<MASS>(rc, NLL, NLL + NSRC, X0 + (float)(2 * sb), Y);
                                        if (NSRC > 1) src[sb][NSRC - 1] = 0.f;
                                    }
                                }
                        }
#pragma unroll
                        for (int sb = 0; sb < S_T; ++sb) {
                            if (LIN) {
#pragma unroll
                                for (int k = 0; k < NSRC; ++k) accs[k] += src[sb][k];
                            } else {
                                acc += src[sb][0];
                                if (NSRC > 1) acc += src[sb][NSRC - 1];
                            }
                        }
                    } else {
                        for (int sb = 0; sb < S; ++sb) {
                            const float X = X0 + (float)(2 * sb);
                            bool fl;
                            float sv[NSRC];
                            sample_value<NLL, NSRC, FAST, MASS>(rc, h, col_values<NLL>(rc, X), rv, acc, sv, fl);
                            if (fl) {
#pragma unroll
                                for (int k = 0; k < NSRC; ++k) sv[k] = refined_source_light_k<MASS>(rc, NLL + k, X, Y);
                            }
                            if (LIN) {
#pragma unroll
                                for (int k = 0; k < NSRC; ++k) accs[k] += sv[k];
                            } else {
#pragma unroll
                                for (int k = 0; k < NSRC; ++k) acc += sv[k];
                            }
                        }
                    }
                }
                if constexpr (PAIR) { float a0, a1; un2(acc2, a0, a1); acc = a0 + a1; }
                if constexpr (PAIR && LIN) {
#pragma unroll
                    for (int k = 0; k < NSRC; ++k) { float a0, a1; un2(accs2[k], a0, a1); accs[k] = a0 + a1; }
                }
            }
            if constexpr (LIN) {
                if (NLL) store(i, j, 0, acc);
#pragma unroll
                for (int k = 0; k < NSRC; ++k) store(i, j, NLL + k, accs[k]);
            } else {
                store(i, j, acc);
            }
        }
        tile = next();
        if (tile < 0) break;
        const int c2 = tile / a.tiles_y;
        r = tile - c2 * a.tiles_y;
        if (c2 != c) {                                 // another tile column (uniform over the warp)
            c = c2;
            j = c * a.CW + lj;
            X0 = (float)(2 * j * S + 1 - S * a.We);
            load_cols();
        }
    }
}

// RowV of all He * S sub-sample rows -> shared memory (all threads of the CTA; caller syncs).
template <int NLL>
__device__ __forceinline__ void fill_rowtab(const RowC &rc, const KArgs &a, RowV *rowtab)
{
    const int S = a.S, n = a.He * S;
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const int i = k / S, sa = k - i * S;
        rowtab[k] = row_values<NLL>(rc, (float)(2 * i * S + 1 - S * a.He + 2 * sa));
    }
}

// Work distribution of phase 1.  Static (split path): warp w of W takes the contiguous tile
// range [w n / W, (w + 1) n / W), n = tiles_x * tiles_y.  Dynamic (fused path): the warps of the
// CTA draw tiles from a shared-memory counter, so they all reach the barrier that ends the
// phase within one tile of each other whatever the refinement branches cost; the value of a
// pixel does not depend on which warp computes it, so logL stays bitwise reproducible.
template <int S_T, int NLL, int NSRC, int MASS, class Store>
__device__ __forceinline__ void trace_image_lin(const RowC &rc, const KArgs &a, const RowV *rowtab, int warp, int n_warps, int *counter, Store store)
{
    const int n = a.tiles_x * a.tiles_y;
    const HotC<NLL, NSRC, MASS> h(rc);
    const bool fast = rc.lens.mode == (MASS == MASS_EPL ? 2 : 0);
    if (counter) {
        auto next = [&]() -> int {
            int t = 0;
            if ((threadIdx.x & 31) == 0) t = atomicAdd(counter, 1);
            t = __shfl_sync(0xffffffffu, t, 0);
            return t < n ? t : -1;
        };
        if (fast) trace_tiles<S_T, NLL, NSRC, true, true, MASS>(rc, h, a, rowtab, next, store);
        else trace_tiles<S_T, NLL, NSRC, false, true, MASS>(rc, h, a, rowtab, next, store);
    } else {
        int t = (int)((long long)n * warp / n_warps);
        const int t_end = (int)((long long)n * (warp + 1) / n_warps);
        auto next = [&]() -> int { return t < t_end ? t++ : -1; };
        if (fast) trace_tiles<S_T, NLL, NSRC, true, true, MASS>(rc, h, a, rowtab, next, store);
        else trace_tiles<S_T, NLL, NSRC, false, true, MASS>(rc, h, a, rowtab, next, store);
    }
}

template <int S_T, int NLL, int NSRC, int MASS, class Store>
__device__ __forceinline__ void trace_image(const RowC &rc, const KArgs &a, const RowV *rowtab, int warp, int n_warps, int *counter, Store store)
{
    const int n = a.tiles_x * a.tiles_y;
    const HotC<NLL, NSRC, MASS> h(rc);
    const bool fast = rc.lens.mode == (MASS == MASS_EPL ? 2 : 0);      // uniform over the CTA
    if (counter) {
        auto next = [&]() -> int {
            int t = 0;
            if ((threadIdx.x & 31) == 0) t = atomicAdd(counter, 1);
            t = __shfl_sync(0xffffffffu, t, 0);
            return t < n ? t : -1;
        };
        if (fast) trace_tiles<S_T, NLL, NSRC, true, false, MASS>(rc, h, a, rowtab, next, store);
        else trace_tiles<S_T, NLL, NSRC, false, false, MASS>(rc, h, a, rowtab, next, store);
    } else {
        int t = (int)((long long)n * warp / n_warps);
        const int t_end = (int)((long long)n * (warp + 1) / n_warps);
        auto next = [&]() -> int { return t < t_end ? t++ : -1; };
        if (fast) trace_tiles<S_T, NLL, NSRC, true, false, MASS>(rc, h, a, rowtab, next, store);
        else trace_tiles<S_T, NLL, NSRC, false, false, MASS>(rc, h, a, rowtab, next, store);
    }
}

// step a6 for a 1 x CONV_R strip whose window starts at `win` (16-byte aligned) in an image of
// row pitch `pitch`; `taps` = flipped PSF [K][Kp] in shared memory.  Taps are consumed four at
// a time (one LDS.128 of taps + one LDS.128 of window per 16 FMAs), the last K % 4 taps of a row
// on their own so that no FMA is spent on padding.  Every kernel row is summed into a fresh
// partial that is then added to the total: the rounding error of the K^2-term sum grows like
// sqrt(K) half-ulps of the total instead of K (1.5e-7 instead of 5e-7 relative at K = 31).
__device__ __forceinline__ void conv_strip(const float *win, int pitch, const float *taps,
                                           int K, int Kp, float acc[CONV_R])
{
#pragma unroll
    for (int r = 0; r < CONV_R; ++r) acc[r] = 0.f;
    const int kfull = K & ~3, rem = K & 3;
    for (int ka = 0; ka < K; ++ka) {
        const float *rp = win + ka * pitch;
        const float *kp = taps + ka * Kp;
        float4 lo = *reinterpret_cast<const float4 *>(rp);
        float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f;
        for (int kb = 0; kb < kfull; kb += 4) {
            const float4 hi = *reinterpret_cast<const float4 *>(rp + kb + 4);
            const float4 t = *reinterpret_cast<const float4 *>(kp + kb);
            p0 = fmaf(t.x, lo.x, fmaf(t.y, lo.y, fmaf(t.z, lo.z, fmaf(t.w, lo.w, p0))));
            p1 = fmaf(t.x, lo.y, fmaf(t.y, lo.z, fmaf(t.z, lo.w, fmaf(t.w, hi.x, p1))));
            p2 = fmaf(t.x, lo.z, fmaf(t.y, lo.w, fmaf(t.z, hi.x, fmaf(t.w, hi.y, p2))));
            p3 = fmaf(t.x, lo.w, fmaf(t.y, hi.x, fmaf(t.z, hi.y, fmaf(t.w, hi.z, p3))));
            lo = hi;
        }
        if (rem) {                                   // uniform: K is a launch constant
            const float4 t = *reinterpret_cast<const float4 *>(kp + kfull);
            p0 = fmaf(t.x, lo.x, p0); p1 = fmaf(t.x, lo.y, p1); p2 = fmaf(t.x, lo.z, p2); p3 = fmaf(t.x, lo.w, p3);
            if (rem > 1) {
                const float4 hi = *reinterpret_cast<const float4 *>(rp + kfull + 4);
                p0 = fmaf(t.y, lo.y, p0); p1 = fmaf(t.y, lo.z, p1); p2 = fmaf(t.y, lo.w, p2); p3 = fmaf(t.y, hi.x, p3);
                if (rem > 2) {
                    p0 = fmaf(t.z, lo.z, p0); p1 = fmaf(t.z, lo.w, p1); p2 = fmaf(t.z, hi.x, p2); p3 = fmaf(t.z, hi.y, p3);
                }
            }
        }
        acc[0] += p0; acc[1] += p1; acc[2] += p2; acc[3] += p3;
    }
}

// step a7 reduction: fixed-shape FP64 tree; result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double *red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < nw; ++w) s += red[w];
    __syncthreads();
    return s;
}

// N sums at once through one pair of barriers: value by value the operations of block_sum in the same order, so
// the same bits; red: N * 32 doubles.
template <int N>
__device__ __forceinline__ void block_sum_n(double (&v)[N], double *red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int n = 0; n < N; ++n) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[n] += __shfl_down_sync(0xffffffffu, v[n], o);
        if (lane == 0) red[n * 32 + wid] = v[n];
    }
    __syncthreads();
    if (threadIdx.x < N) {
        double s = 0.0;
        for (int w = 0; w < nw; ++w) s += red[threadIdx.x * 32 + w];
        red[threadIdx.x * 32] = s;
    }
    __syncthreads();
#pragma unroll
    for (int n = 0; n < N; ++n) v[n] = red[n * 32];
    __syncthreads();
}

__device__ __forceinline__ void load_row_consts(RowC *dst, const RowC *src)
{
    const int n16 = sizeof(RowC) / 16;
    const uint4 *s = reinterpret_cast<const uint4 *>(src);
    uint4 *d = reinterpret_cast<uint4 *>(dst);
    for (int i = threadIdx.x; i < n16; i += blockDim.x) d[i] = s[i];
}

__device__ __forceinline__ void load_psf(float *dst, const float *src, int n)
{
    for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = src[i];
}

// step a6 for a 2 x 4 output block, PSF size known at compile time.  Per kernel row `ka` the
// thread holds the windows of image rows i+ka and i+ka+1 (NW float4 each) in registers: the
// second one is loaded (NW LDS.128) and becomes the first one of the next kernel row, so every
// window float is read from shared memory once and used for up to 2 x 4 FMAs per tap: the
// shared-memory pipe carries NW window loads + KG (broadcast) tap loads per 8 K FMAs, about 70 %
// of its bandwidth at K = 21, instead of being the limiter as with 1 x 4 strips.  (Feeding the
// taps through the constant bank instead was measured: no faster, LDC is the slower path.)
template <int K>
struct ConvBlock {
    static constexpr int KG = (K + 3) / 4;           // tap groups of 4 per kernel row
    static constexpr int Kp = KG * 4;
    static constexpr int NW = (K + 3 + 3) / 4;       // float4 per window: columns 0 .. K + 2

    static __device__ __forceinline__ void load_window(float4 (&w)[NW], const float *rp)
    {
#pragma unroll
        for (int g = 0; g < NW; ++g) w[g] = *reinterpret_cast<const float4 *>(rp + 4 * g);
    }

    // one kernel row applied to one image-row window -> 4 outputs, summed into a fresh partial
    static __device__ __forceinline__ void row(const float4 (&w)[NW], const float *kp, float (&acc)[4])
    {
        float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f;
#pragma unroll
        for (int g = 0; g < KG; ++g) {
            const float4 t = *reinterpret_cast<const float4 *>(kp + 4 * g);
            const float4 lo = w[g];
            const float4 hi = (g + 1 < NW) ? w[g + 1] : make_float4(0.f, 0.f, 0.f, 0.f);
            const int nt = (K - 4 * g) >= 4 ? 4 : (K - 4 * g);     // real taps in this group
            p0 = fmaf(t.x, lo.x, p0); p1 = fmaf(t.x, lo.y, p1); p2 = fmaf(t.x, lo.z, p2); p3 = fmaf(t.x, lo.w, p3);
            if (nt > 1) { p0 = fmaf(t.y, lo.y, p0); p1 = fmaf(t.y, lo.z, p1); p2 = fmaf(t.y, lo.w, p2); p3 = fmaf(t.y, hi.x, p3); }
            if (nt > 2) { p0 = fmaf(t.z, lo.z, p0); p1 = fmaf(t.z, lo.w, p1); p2 = fmaf(t.z, hi.x, p2); p3 = fmaf(t.z, hi.y, p3); }
            if (nt > 3) { p0 = fmaf(t.w, lo.w, p0); p1 = fmaf(t.w, hi.x, p1); p2 = fmaf(t.w, hi.y, p2); p3 = fmaf(t.w, hi.z, p3); }
        }
        acc[0] += p0; acc[1] += p1; acc[2] += p2; acc[3] += p3;
    }

    // `win` = image row i, column x0 (16-byte aligned); taps = flipped PSF [K][Kp]
    static __device__ __forceinline__ void run(const float *win, int pitch, const float *taps,
                                               float (&a0)[4], float (&a1)[4])
    {
#pragma unroll
        for (int r = 0; r < 4; ++r) { a0[r] = 0.f; a1[r] = 0.f; }
        float4 wa[NW], wb[NW];
        load_window(wa, win);
        // kernel rows two at a time so that the windows ping-pong without register moves
#pragma unroll 1
        for (int ka = 0; ka + 1 < K; ka += 2) {
            load_window(wb, win + (ka + 1) * pitch);
            row(wa, taps + ka * Kp, a0);
            row(wb, taps + ka * Kp, a1);
            load_window(wa, win + (ka + 2) * pitch);
            row(wb, taps + (ka + 1) * Kp, a0);
            row(wa, taps + (ka + 1) * Kp, a1);
        }
        if (K & 1) {                                  // K is odd: last kernel row
            load_window(wb, win + K * pitch);
            row(wa, taps + (K - 1) * Kp, a0);
            row(wb, taps + (K - 1) * Kp, a1);
        }
    }
};

// chi^2 terms of up to 4 outputs of row i starting at column x0 (and the optional image store).
// x0 is a multiple of 4, so when nx is too the four data / weight values are one aligned 16-byte
// load each (north_star (3): "vectorised coalesced loads"); the sum order is the same either way.
// `err` (optional, AUTO precision): accumulates e = (d - m) m w and e^2, the first-order sensitivity
// of logL to a relative error of the model pixel (delta logL = sum_i e_i eps_i).
struct ErrAcc { float s1, s2; };
__device__ __forceinline__ float chi2_strip(const KArgs &a, const float acc[4], int i, int x0,
                                            const float *data, const float *wgt, float *image_out, ErrAcc *err = nullptr)
{
    float c = 0.f;
    if ((a.nx & 3) == 0) {                           // uniform over the grid
        if (x0 >= a.nx) return 0.f;
        const int o = i * a.nx + x0;
        if (image_out) *reinterpret_cast<float4 *>(image_out + o) = make_float4(acc[0], acc[1], acc[2], acc[3]);
        if (data) {
            const float4 dv = __ldg(reinterpret_cast<const float4 *>(data + o));
            const float4 wv = __ldg(reinterpret_cast<const float4 *>(wgt + o));
            const float d0 = dv.x - acc[0], d1 = dv.y - acc[1], d2 = dv.z - acc[2], d3 = dv.w - acc[3];
            c = fmaf(d0 * d0, wv.x, c); c = fmaf(d1 * d1, wv.y, c); c = fmaf(d2 * d2, wv.z, c); c = fmaf(d3 * d3, wv.w, c);
            if (err) {
                const float e0 = d0 * wv.x * acc[0], e1 = d1 * wv.y * acc[1], e2 = d2 * wv.z * acc[2], e3 = d3 * wv.w * acc[3];
                err->s1 += (e0 + e1) + (e2 + e3);
                err->s2 = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, err->s2))));
            }
        }
        return c;
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int x = x0 + r;
        if (x < a.nx) {
            const int o = i * a.nx + x;
            if (image_out) image_out[o] = acc[r];
            if (data) {
                const float d = __ldg(data + o) - acc[r], wv = __ldg(wgt + o);
                c = fmaf(d * d, wv, c);
                if (err) { const float e = d * wv * acc[r]; err->s1 += e; err->s2 = fmaf(e, e, err->s2); }
            }
        }
    }
    return c;
}

template <int K>
__device__ __forceinline__ double conv_chi2_blocks(const KArgs &a, const float *img, int e0, const float *taps,
                                                   int i0, int i1, const float *data, const float *wgt, float *image_out, ErrAcc *err)
{
    const int nsx = (a.nx + 3) / 4, npair = (i1 - i0 + 1) / 2;
    const int total = npair * nsx;
    double part = 0.0;
    for (int s = threadIdx.x; s < total; s += blockDim.x) {
        const int ip = s / nsx, i = i0 + 2 * ip, x0 = (s - ip * nsx) * 4;
        float a0[4], a1[4];
        ConvBlock<K>::run(img + (i - e0) * a.pitch + x0, a.pitch, taps, a0, a1);
        float c = chi2_strip(a, a0, i, x0, data, wgt, image_out, err);
        if (i + 1 < i1) c += chi2_strip(a, a1, i + 1, x0, data, wgt, image_out, err);
        part += (double)c;
    }
    return part;
}

// convolve + chi^2 over output rows [i0, i1) of one image; `img` is a shared-memory image
// whose row 0 corresponds to extended row `e0` (one spare row after the last one must be
// readable).  Returns this thread's chi^2 partial.  The common PSF sizes get the register-
// blocked 2 x 4 kernel, any other odd size the generic 1 x 4 strip.
// KSMALL: only the blocks up to 21 x 21 are compiled in (a kernel that holds the 41 x 41 blocks is held to
// their ~120 registers whatever PSF it is run with).
template <bool KSMALL = false>
__device__ __forceinline__ double conv_chi2_rows(const KArgs &a, const float *img, int e0,
                                                 const float *taps, int i0, int i1,
                                                 const float *data, const float *wgt, float *image_out, ErrAcc *err = nullptr)
{
#define TL_CONV_CASE(KK) \
    case KK: return conv_chi2_blocks<KK>(a, img, e0, taps, i0, i1, data, wgt, image_out, err);
    if constexpr (KSMALL) {
        switch (a.K) {
            TL_CONV_CASE(5)
            TL_CONV_CASE(15)
            TL_CONV_CASE(21)
        default: break;
        }
    } else {
        switch (a.K) {
            TL_CONV_CASE(5)
            TL_CONV_CASE(15)
            TL_CONV_CASE(21)
            TL_CONV_CASE(31)
            TL_CONV_CASE(41)
        default: break;
        }
    }
#undef TL_CONV_CASE
    const int nsx = (a.nx + CONV_R - 1) / CONV_R;
    const int total = (i1 - i0) * nsx;
    double part = 0.0;
    for (int s = threadIdx.x; s < total; s += blockDim.x) {
        const int ir = s / nsx, i = i0 + ir, x0 = (s - ir * nsx) * CONV_R;
        float acc[CONV_R];
        conv_strip(img + (i - e0) * a.pitch + x0, a.pitch, taps, a.K, a.Kp, acc);
        part += (double)chi2_strip(a, acc, i, x0, data, wgt, image_out, err);
    }
    return part;
}

// ------------------------------------------------------------------------------ fused path
#ifndef TL_LB_T
#define TL_LB_T 512
#define TL_LB_B 1
#endif
// VAR = 1: the variant for small rows (256 threads, PSF up to 21 x 21): three CTAs per SM.
template <int S_T, int NLL, int NSRC, int MASS = MASS_SIE, int VAR = 0>
__global__ void __launch_bounds__(VAR ? 256 : TL_LB_T, VAR ? 3 : TL_LB_B) fused_kernel(const KArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RowC *rc = reinterpret_cast<RowC *>(smem_raw);
    double *red = reinterpret_cast<double *>(smem_raw + sizeof(RowC));            // [0, 16): block_sum
    int *tile_counter = reinterpret_cast<int *>(red + 24);                          // phase-1 work queue
    float *taps = reinterpret_cast<float *>(smem_raw + sizeof(RowC) + 32 * sizeof(double));
    float *img = taps + a.K * a.Kp;
    const int n_img = a.He * a.pitch;
    RowV *rowtab = a.rowtab ? reinterpret_cast<RowV *>(img + ((n_img + a.pitch + a.Kp + 8 + 3) & ~3)) : nullptr;
    // pitch padding and the slack after the image are read by zero-padded taps only (and by
    // discarded strip lanes); phase 1 never writes them, so zero them once
    for (int i = threadIdx.x; i < n_img + a.pitch + a.Kp + 8; i += blockDim.x) img[i] = 0.f;

    int64_t cur_lens = -1;
    for (int64_t r = blockIdx.x; r < a.B; r += gridDim.x) {
        const int64_t row = a.row0 + r;                // global row; a.rows is chunk-local
        const int64_t lens = row / a.rows_per_lens;
        __syncthreads();                               // previous row fully consumed
        load_row_consts(rc, a.rows + r);
        if (threadIdx.x == 0) *tile_counter = 0;
        if (lens != cur_lens) { load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp); cur_lens = lens; }
        __syncthreads();
        const size_t npix = (size_t)a.ny * a.nx;
        if (!row_is_valid(*rc, a.n_comp)) {            // uniform over the CTA
            if (a.logL && threadIdx.x == 0) a.logL[row] = -INFINITY;
            if (a.images)
                for (size_t i = threadIdx.x; i < npix; i += blockDim.x) a.images[row * npix + i] = NAN;
            continue;
        }
        // phase 1: ray-trace + light + bin into shared memory
        if (rowtab) { fill_rowtab<NLL>(*rc, a, rowtab); __syncthreads(); }
        trace_image<S_T, NLL, NSRC, MASS>(*rc, a, rowtab, threadIdx.x >> 5, blockDim.x >> 5, tile_counter,
                                    [&](int i, int j, float v) { img[i * a.pitch + j] = v; });
        __syncthreads();
        // phase 2: PSF convolution from shared memory + chi^2
        ErrAcc err = {0.f, 0.f};
        const bool want_err = a.flag_count != nullptr && a.logL != nullptr;      // AUTO precision (uniform)
        const double part = conv_chi2_rows<VAR != 0>(a, img, 0, taps, 0, a.ny,
                                           a.logL ? a.data + lens * npix : nullptr,
                                           a.wgt + lens * npix,
                                           a.images ? a.images + row * npix : nullptr, want_err ? &err : nullptr);
        // phase 3: deterministic reduction (Eq. 5)
        if (a.logL) {
            const double chi2 = block_sum(part, red);
            const double ll = -0.5 * (chi2 + a.lconst[lens]);
            if (threadIdx.x == 0) a.logL[row] = (float)ll;
            if (want_err) {
                // first-order FP32 error bound of this row (DESIGN.md 6 "AUTO"): delta logL = sum_i e_i eps_i
                const double s1 = block_sum((double)err.s1, red), s2 = block_sum((double)err.s2, red);
                if (threadIdx.x == 0) {
                    const double bound = (double)a.err_coh * fabs(s1) + (double)a.err_rnd * sqrt(s2);
                    const double tol = fmax(1e-3, 1e-6 * fabs(ll));
                    if (!(bound <= tol)) a.flag_list[atomicAdd(a.flag_count, 1)] = (int)row;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------ split path
// trace_kernel: one parameter row per blockIdx.x iteration, the row's items spread over
// gridDim.y CTAs (slabs); binned extended image -> global memory.
template <int S_T, int NLL, int NSRC, int MASS = MASS_SIE>
__global__ void __launch_bounds__(256, 2) trace_kernel(const KArgs a, int chunk_rows)
{
    __shared__ RowC rc_s;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RowV *rowtab = a.rowtab ? reinterpret_cast<RowV *>(smem_raw) : nullptr;
    pdl_launch();
    pdl_wait();                                        // the row constants come from the prologue kernel
    for (int r = blockIdx.x; r < chunk_rows; r += gridDim.x) {
        __syncthreads();
        load_row_consts(&rc_s, a.rows + r);
        __syncthreads();
        if (!row_is_valid(rc_s, a.n_comp)) continue;
        if (rowtab) { fill_rowtab<NLL>(rc_s, a, rowtab); __syncthreads(); }
        // (MGE mode: the source image is component slot ext_k0 of ext_nc per row)
        float *dst = a.ext + ((size_t)r * (a.ext_nc ? a.ext_nc : 1) + a.ext_k0) * a.He * a.pitch;
        // small batches: the row's CTAs draw warp tiles from one global queue, so a tile full of
        // FP64-refined samples does not leave the other warps of the row waiting for its owner
        trace_image<S_T, NLL, NSRC, MASS>(rc_s, a, rowtab, (blockIdx.y * blockDim.x + threadIdx.x) >> 5, (gridDim.y * blockDim.x) >> 5,
                                    a.tile_counters ? a.tile_counters + r : nullptr,
                                    [&](int i, int j, float v) { dst[i * a.pitch + j] = v; });
    }
}

// trace_pairs_kernel: the ray-trace of calls with a handful of rows (run_small_batch), where the time
// of a call is the longest dependent chain, not the arithmetic.  A lane takes ONE pair of horizontally
// adjacent sub-samples, the S^2 / 2 lanes of a native pixel sit side by side in a warp, and the pixel's
// sum is formed from their values in the order of trace_tiles (per sub-sample row: lens light left to
// right, then the sources left to right), so that the pixel is BITWISE what trace_tiles gives.  The
// longest chain of the call -- the FP64 refinement of the samples next to the source centre, which
// trace_tiles runs sixteen deep per lane at S = 4 -- becomes two deep, and one row fills the GPU.
// Rows on the q < 0.5 branch go through trace_tiles.  Grid (rows, CTAs per row): as many as are resident at once.
// (body: warp `warp` of the `n_warps` that share the row whose constants are rc_s; no CTA-wide barrier inside)
template <int S_T, int NLL, int NSRC>
__device__ __forceinline__ void trace_pairs_row(const RowC &rc_s, const KArgs &a, float *dst, int warp, int n_warps)
{
    static_assert(S_T == 2 || S_T == 4 || S_T == 8, "S^2 / 2 lanes per pixel must divide a warp");
    constexpr int NP = S_T / 2, LPP = S_T * NP, PPW = 32 / LPP;
    const int lane = threadIdx.x & 31;
    const HotC<NLL, NSRC, MASS_SIE> h(rc_s);
    if (rc_s.lens.mode != 0) {                         // uniform over the row
        const int n = a.tiles_x * a.tiles_y;
        int t = (int)((long long)n * warp / n_warps);
        const int t_end = (int)((long long)n * (warp + 1) / n_warps);
        trace_tiles<S_T, NLL, NSRC, false, false, MASS_SIE>(rc_s, h, a, nullptr, [&]() -> int { return t < t_end ? t++ : -1; },
                                                            [&](int i, int j, float v) { dst[i * a.pitch + j] = v; });
        return;
    }
    const int sub = lane % LPP, sa = sub / NP, sp = sub - sa * NP, base = lane - sub;
    const int npix = a.He * a.We;
    // warp tiles of PPW pixels, dealt out round-robin: neighbouring tiles (the refined ones cluster
    // round the source centre) go to different warps
    for (int p0 = warp * PPW; p0 < npix; p0 += n_warps * PPW) {
        const int pix = p0 + lane / LPP;
        const bool live = pix < npix;
        const int pc = live ? pix : npix - 1;
        const int i = pc / a.We, j = pc - i * a.We;
        const bool edge = a.edge_zero && (j < a.h || j >= a.We - a.h || i < a.h || i >= a.He - a.h);
        f2 llv, s;
        llv.v = 0ull; s.v = 0ull;
        if (!edge) {
            // u-units, as in trace_tiles: X = 2 (j S + b) + 1 - S We, Y = 2 (i S + sa) + 1 - S He
            const float X = (float)(2 * j * S_T + 1 - S_T * a.We) + (float)(4 * sp);
            const float Y = (float)(2 * i * S_T + 1 - S_T * a.He) + (float)(2 * sa);
            const ColV2 cv = col_values2<NLL>(rc_s, X, X + 2.f);
            const RowV rv = row_values<NLL>(rc_s, Y);
            bool any = false;
            s = sample_pair_parts<NLL, NSRC>(h, cv, rv, llv, any);
            if (any) {                                 // rare: FP64 ray-trace, out of line
                float s0, s1;
                un2(s, s0, s1);
                if (s0 != s0) s0 = refined_source_light<MASS_SIE>(rc_s, NLL, NLL + NSRC, X, Y);
                if (s1 != s1) s1 = refined_source_light<MASS_SIE>(rc_s, NLL, NLL + NSRC, X + 2.f, Y);
                s = mk2(s0, s1);
            }
        }
        __syncwarp();
        f2 acc2 = bc2(0.f);
#pragma unroll
        for (int ra = 0; ra < S_T; ++ra) {
            if (NLL) {
#pragma unroll
                for (int b = 0; b < NP; ++b) {
                    f2 v;
                    v.v = __shfl_sync(0xffffffffu, llv.v, base + ra * NP + b);
                    acc2 = fma2(bc2(h.ll.amp), v, acc2);
                }
            }
#pragma unroll
            for (int b = 0; b < NP; ++b) {
                f2 v;
                v.v = __shfl_sync(0xffffffffu, s.v, base + ra * NP + b);
                acc2 = add2(acc2, v);
            }
        }
        float a0, a1;
        un2(acc2, a0, a1);
        if (live && sub == 0) dst[i * a.pitch + j] = edge ? 0.f : a0 + a1;
    }
}

template <int S_T, int NLL, int NSRC>
__global__ void __launch_bounds__(256, 2) trace_pairs_kernel(const KArgs a, int chunk_rows)
{
    __shared__ RowC rc_s;
    pdl_launch();
    pdl_wait();                                        // the row constants come from the prologue kernel
    const int r = blockIdx.x;
    if (r >= chunk_rows) return;
    load_row_consts(&rc_s, a.rows + r);
    __syncthreads();
    if (!row_is_valid(rc_s, a.n_comp)) return;
    trace_pairs_row<S_T, NLL, NSRC>(rc_s, a, a.ext + (size_t)r * a.He * a.pitch, (blockIdx.y * blockDim.x + threadIdx.x) >> 5,
                                    (gridDim.y * blockDim.x) >> 5);
}

#ifdef TL_MAIN_TU
// conv_kernel: one CTA per (row_in_chunk, tile of `tile_rows` output rows).
__global__ void __launch_bounds__(256) conv_kernel(const KArgs a, int chunk_rows)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *red = reinterpret_cast<double *>(smem_raw);
    float *taps = reinterpret_cast<float *>(smem_raw + 32 * sizeof(double));
    float *img = taps + a.K * a.Kp;
    const int r = blockIdx.x, tile = blockIdx.y;
    const int64_t row = a.row0 + r;
    const int64_t lens = row / a.rows_per_lens;
    const size_t npix = (size_t)a.ny * a.nx;
    const RowC *rcg = a.rows + r;
    bool ok = rcg->lens.valid != 0;
    for (int k = 0; k < a.n_comp; ++k) ok = ok && (rcg->comp[k].valid != 0);
    const int i0 = tile * a.tile_rows, i1 = min(a.ny, i0 + a.tile_rows);
    if (!ok) {
        if (a.images)
            for (size_t i = (size_t)i0 * a.nx + threadIdx.x; i < (size_t)i1 * a.nx; i += blockDim.x)
                a.images[row * npix + i] = NAN;
        if (a.partial && threadIdx.x == 0) a.partial[(size_t)r * a.n_tiles + tile] = INFINITY;
        return;
    }
    load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp);
    // extended rows i0 .. i1 + 2h - 1 of this row's binned image, plus slack
    const int erows = (i1 - i0) + 2 * a.h;
    const float4 *src = reinterpret_cast<const float4 *>(a.ext + ((size_t)r * a.He + i0) * a.pitch);
    float4 *dst = reinterpret_cast<float4 *>(img);
    const int n4 = erows * a.pitch / 4;
    for (int i = threadIdx.x; i < n4; i += blockDim.x) dst[i] = src[i];
    for (int i = threadIdx.x; i < a.pitch + a.Kp + 8; i += blockDim.x) img[erows * a.pitch + i] = 0.f;
    __syncthreads();
    const double part = conv_chi2_rows(a, img, i0, taps, i0, i1,
                                       a.partial ? a.data + lens * npix : nullptr,
                                       a.wgt + lens * npix,
                                       a.images ? a.images + row * npix : nullptr);
    if (a.partial) {
        const double s = block_sum(part, red);
        if (threadIdx.x == 0) a.partial[(size_t)r * a.n_tiles + tile] = s;
    }
}

// finalize_kernel: fixed-order sum of the tile partials -> logL.
__global__ void finalize_kernel(const KArgs a, int chunk_rows)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= chunk_rows) return;
    const int64_t row = a.row0 + r;
    double s = 0.0;
    for (int t = 0; t < a.n_tiles; ++t) s += a.partial[(size_t)r * a.n_tiles + t];
    const double ll = -0.5 * (s + a.lconst[row / a.rows_per_lens]);
    a.logL[row] = isfinite(s) ? (float)ll : -INFINITY;
}

#endif  // TL_MAIN_TU

// ------------------------------------------------------------------------------ small batches
// (NEXT-4: the sampler hands over small proposal batches.)  With fewer rows
// than SMs the fused path leaves most of the GPU idle and a call takes one row's time (0.18 ms on
// configs[1]) whatever B.  Here a row is spread over many CTAs -- trace_kernel with as many slabs
// as fill the GPU, then conv_small_kernel over bands of output row pairs -- and the result is
// BITWISE what the fused kernel gives: the pixel values do not depend on which warp traces them,
// the 2 x 4 convolution blocks are the same code, each block's chi^2 term is stored, and the
// row's last CTA to finish (conv_small_kernel runs with the fused kernel's block size) adds them
// per thread and across the CTA in exactly the fused kernel's order (same block_sum).
template <int K>
__device__ __forceinline__ void conv_blocks_store(const KArgs &a, const float *img, int e0, const float *taps, int p0, int p1,
                                                  const float *data, const float *wgt, float *image_out, float *cblk)
{
    const int nsx = (a.nx + 3) / 4;
    const int total = (p1 - p0) * nsx;
    for (int s = threadIdx.x; s < total; s += blockDim.x) {
        const int ip = s / nsx, xb = s - ip * nsx, i = 2 * (p0 + ip), x0 = xb * 4;
        float a0[4], a1[4];
        ConvBlock<K>::run(img + (i - e0) * a.pitch + x0, a.pitch, taps, a0, a1);
        float c = chi2_strip(a, a0, i, x0, data, wgt, image_out);
        if (i + 1 < a.ny) c += chi2_strip(a, a1, i + 1, x0, data, wgt, image_out);
        if (cblk) cblk[(p0 + ip) * nsx + xb] = c;
    }
}

// The 2 x 4 blocks of output row pairs [p0, p1) x strips [xb0, xb1), with the K kernel rows of a block
// on K different threads: thread (block, ka) forms the two fresh per-kernel-row partials of
// ConvBlock<K>::run (same code: ConvBlock<K>::row), they go to `part` in shared memory, and one
// thread per (block, output row) adds them in the order ka = 0 .. K-1 -- the sums ConvBlock<K>::run
// forms, bit for bit, in 1/K of its time.  `part`: [blockDim.x / K blocks][K][8] floats.
template <int K>
__device__ __forceinline__ void conv_blocks_split(const KArgs &a, const float *img, int e0, const float *taps, float *part,
                                                  int p0, int p1, int xb0, int xb1,
                                                  const float *data, const float *wgt, float *image_out, float *cblk)
{
    using CB = ConvBlock<K>;
    const int nsx = (a.nx + 3) / 4;
    const int nbx = xb1 - xb0, nblk = (p1 - p0) * nbx;
    const int per_pass = blockDim.x / K;               // whole blocks per pass
    for (int b0 = 0; b0 < nblk; b0 += per_pass) {
        const int nb = min(per_pass, nblk - b0);
        if (b0) __syncthreads();                       // the previous pass has read `part`
        if ((int)threadIdx.x < nb * K) {
            const int bl = threadIdx.x / K, ka = threadIdx.x - bl * K, blk = b0 + bl;
            const int ip = blk / nbx, xb = xb0 + (blk - ip * nbx), i = 2 * (p0 + ip), x0 = xb * 4;
            const float *win = img + (i - e0 + ka) * a.pitch + x0;
            float4 wa[CB::NW], wb[CB::NW];
            CB::load_window(wa, win);
            CB::load_window(wb, win + a.pitch);
            float q0[4] = {0.f, 0.f, 0.f, 0.f}, q1[4] = {0.f, 0.f, 0.f, 0.f};
            CB::row(wa, taps + ka * CB::Kp, q0);
            CB::row(wb, taps + ka * CB::Kp, q1);
            float4 *dst = reinterpret_cast<float4 *>(part + (size_t)threadIdx.x * 8);
            dst[0] = make_float4(q0[0], q0[1], q0[2], q0[3]);
            dst[1] = make_float4(q1[0], q1[1], q1[2], q1[3]);
        }
        __syncthreads();
        // (block, output row) on adjacent lanes; whole warps take part in the shuffle
        if ((int)(threadIdx.x & ~31u) < 2 * nb) {
            const int t = threadIdx.x, bl = t >> 1, rs = t & 1, blk = b0 + bl;
            float c = 0.f;
            int ip = 0, xb = 0;
            if (t < 2 * nb) {
                ip = blk / nbx; xb = xb0 + (blk - ip * nbx);
                const int i = 2 * (p0 + ip) + rs, x0 = xb * 4;
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
                const float4 *src = reinterpret_cast<const float4 *>(part + (size_t)bl * K * 8 + rs * 4);
#pragma unroll
                for (int ka = 0; ka < K; ++ka) {
                    const float4 v = src[2 * ka];
                    acc[0] += v.x; acc[1] += v.y; acc[2] += v.z; acc[3] += v.w;
                }
                if (i < a.ny) c = chi2_strip(a, acc, i, x0, data, wgt, image_out);
            }
            const float c1 = __shfl_down_sync(0xffffffffu, c, 1);
            if (t < 2 * nb && rs == 0) {
                if (2 * (p0 + ip) + 1 < a.ny) c += c1;
                if (cblk) cblk[(p0 + ip) * nsx + xb] = c;
            }
        }
    }
}

// one CTA per (row, band of `band_pairs` output row pairs x one of `xseg` runs of strips); cblk:
// [chunk][npair * nsx] or null; a.tile_counters[chunk_rows + r] (zeroed) counts the finished CTAs of row r.
// xseg = 0: whole bands, one thread per block (conv_blocks_store: more rows than the split form pays for)
// (body: row r, virtual block `by` of `n_by` per row; every thread of the CTA calls; `wait`: the rows / images
// come from kernels launched before this one with programmatic dependent launch)
// Returns true (to every thread) when this call wrote the row's logL.
__device__ __forceinline__ bool conv_small_body(const KArgs &a, int chunk_rows, int r, int by, int n_by, int band_pairs, int xseg,
                                                float *cblk, unsigned char *smem_raw, bool wait)
{
    __shared__ double red[32];
    __shared__ int is_last;
    float *taps = reinterpret_cast<float *>(smem_raw);
    float *part = taps + a.K * a.Kp;                                // [blockDim.x / K][K][8]
    float *img = xseg ? part + (blockDim.x / a.K) * a.K * 8 : part;
    const int npair = (a.ny + 1) / 2, nsx = (a.nx + 3) / 4;
    const int nseg = xseg ? xseg : 1;
    const int band = by / nseg, seg = by - band * nseg;
    const int p0 = band * band_pairs, p1 = min(npair, p0 + band_pairs);
    const int xb0 = (int)((long long)nsx * seg / nseg), xb1 = (int)((long long)nsx * (seg + 1) / nseg);
    const int64_t row = a.row0 + r;
    const int64_t lens = row / a.rows_per_lens;
    const size_t npix = (size_t)a.ny * a.nx;
    load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp);          // context data: before the wait
    if (wait) pdl_wait();                                         // rows / ext come from the preceding kernels
    if (!row_is_valid(a.rows[r], a.n_comp)) {
        if (a.images && seg == 0)
            for (size_t i = (size_t)2 * p0 * a.nx + threadIdx.x; i < (size_t)min(a.ny, 2 * p1) * a.nx; i += blockDim.x)
                a.images[row * npix + i] = NAN;
        if (a.logL && by == 0 && threadIdx.x == 0) a.logL[row] = -INFINITY;
        return a.logL && by == 0;
    }
    // extended rows 2 p0 .. 2 (p1 - 1) + K of this row's binned image (the last one may lie past
    // the image when ny is odd: zeros), plus the slack the strips may touch
    const int e0 = 2 * p0, erows = 2 * (p1 - p0) + a.K - 1, have = min(erows, a.He - e0);
    const float4 *src = reinterpret_cast<const float4 *>(a.ext + ((size_t)r * a.He + e0) * a.pitch);
    float4 *dst = reinterpret_cast<float4 *>(img);
    const int n4 = have * a.pitch / 4;
    for (int i = threadIdx.x; i < n4; i += blockDim.x) dst[i] = src[i];
    for (int i = have * a.pitch + threadIdx.x; i < erows * a.pitch + a.pitch + a.Kp + 8; i += blockDim.x) img[i] = 0.f;
    __syncthreads();
    const float *data = a.logL ? a.data + lens * npix : nullptr;
    float *image_out = a.images ? a.images + row * npix : nullptr;
    float *cb = (a.logL && cblk) ? cblk + (size_t)r * npair * nsx : nullptr;
#define TL_CONV_CASE(KK)                                                                                                       \
    case KK:                                                                                                                   \
        if (xseg) conv_blocks_split<KK>(a, img, e0, taps, part, p0, p1, xb0, xb1, data, a.wgt + lens * npix, image_out, cb);   \
        else conv_blocks_store<KK>(a, img, e0, taps, p0, p1, data, a.wgt + lens * npix, image_out, cb);                        \
        break;
    switch (a.K) {
        TL_CONV_CASE(5)
        TL_CONV_CASE(15)
        TL_CONV_CASE(21)
        TL_CONV_CASE(31)
        TL_CONV_CASE(41)
    default: break;
    }
#undef TL_CONV_CASE
    if (!cb) return false;
    // the row's last band to finish reduces the stored terms: per-thread partials over
    // s = tid, tid + blockDim, ... and block_sum, exactly as fused_kernel does
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(a.tile_counters + chunk_rows + r, 1) == n_by - 1;
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    const int total = npair * nsx;
    double psum = 0.0;
    for (int s = threadIdx.x; s < total; s += blockDim.x) psum += (double)__ldcg(cb + s);
    const double chi2 = block_sum(psum, red);
    if (threadIdx.x == 0) a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[lens]));
    return true;
}

#ifdef TL_MAIN_TU
__global__ void __launch_bounds__(512) conv_small_kernel(const KArgs a, int chunk_rows, int band_pairs, int xseg, float *cblk)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    conv_small_body(a, chunk_rows, blockIdx.x, blockIdx.y, gridDim.y, band_pairs, xseg, cblk, smem_raw, true);
}

#endif  // TL_MAIN_TU

// ------------------------------------------------------------------------------ linear mode
// (NEXT-1, Eq. 6-7)  trace_lin_kernel -> conv_lin_kernel -> solve_lin_kernel.
template <int S_T, int NLL, int NSRC, int MASS = MASS_SIE>
__global__ void __launch_bounds__(256, 2) trace_lin_kernel(const KArgs a, int chunk_rows)
{
    __shared__ RowC rc_s;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RowV *rowtab = a.rowtab ? reinterpret_cast<RowV *>(smem_raw) : nullptr;
    constexpr int NC = NLL + NSRC;
    for (int r = blockIdx.x; r < chunk_rows; r += gridDim.x) {
        __syncthreads();
        load_row_consts(&rc_s, a.rows + r);
        __syncthreads();
        if (!row_is_valid(rc_s, a.n_comp)) continue;
        if (rowtab) { fill_rowtab<NLL>(rc_s, a, rowtab); __syncthreads(); }
        float *dst = a.ext + ((size_t)r * (a.ext_nc ? a.ext_nc : NC) + a.ext_k0) * a.He * a.pitch;
        const size_t comp_stride = (size_t)a.He * a.pitch;
        trace_image_lin<S_T, NLL, NSRC, MASS>(rc_s, a, rowtab, (blockIdx.y * blockDim.x + threadIdx.x) >> 5, (gridDim.y * blockDim.x) >> 5,
                                      a.tile_counters ? a.tile_counters + r : nullptr,
                                      [&](int i, int j, int k, float v) { dst[k * comp_stride + i * a.pitch + j] = v; });
    }
}

#ifdef TL_MAIN_TU
// one CTA per (row_in_chunk, tile of output rows, component): M_k = K (*) L_k  (blurring matrix B)
__global__ void __launch_bounds__(256, 2) conv_lin_kernel(const KArgs a, int chunk_rows)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *taps = reinterpret_cast<float *>(smem_raw);
    float *img = taps + a.K * a.Kp;
    const int r = blockIdx.x, tile = blockIdx.y, k = blockIdx.z, NC = gridDim.z;
    const int64_t row = a.row0 + r;
    const int64_t lens = row / a.rows_per_lens;
    const size_t npix = (size_t)a.ny * a.nx;
    if (!row_is_valid(a.rows[r], a.n_comp)) return;
    const int i0 = tile * a.tile_rows, i1 = min(a.ny, i0 + a.tile_rows);
    load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp);
    const int erows = (i1 - i0) + 2 * a.h;
    const int enc = a.conv_ext_nc ? a.conv_ext_nc : NC, mnc = a.conv_m_nc ? a.conv_m_nc : NC;
    const float4 *src = reinterpret_cast<const float4 *>(a.ext + (((size_t)r * enc + k) * a.He + i0) * a.pitch);
    float4 *dst = reinterpret_cast<float4 *>(img);
    const int n4 = erows * a.pitch / 4;
    for (int i = threadIdx.x; i < n4; i += blockDim.x) dst[i] = src[i];
    for (int i = threadIdx.x; i < a.pitch + a.Kp + 8; i += blockDim.x) img[erows * a.pitch + i] = 0.f;
    __syncthreads();
    conv_chi2_rows(a, img, i0, taps, i0, i1, nullptr, nullptr, a.mimg + ((size_t)r * mnc + a.conv_m_k0 + k) * npix);
}

#endif  // TL_MAIN_TU

// G = M'WM, b = M'Wd, d'Wd (fixed-shape FP64 reductions), NNLS, chi^2 = d'Wd - 2 s'b + s'G s -> logL.
// All threads of the CTA; M = the row's blurred unit-amplitude component images [C][npix].
// red: 32 doubles, or -- red_wide -- 10 * 32 (then the ten sums share one pair of barriers: calls with a few rows,
// where the row's one CTA is what the caller waits for).
__device__ __forceinline__ void solve_row(const KArgs &a, const float *M, int64_t row, int64_t lens,
                                          double *red, double *s_sh, bool red_wide = false)
{
    (void)s_sh;
    const int NC = a.n_comp, npix = a.ny * a.nx;
    const float *d = a.data + lens * (size_t)npix, *w = a.wgt + lens * (size_t)npix;
    double g[6] = {0, 0, 0, 0, 0, 0}, bb[3] = {0, 0, 0};             // G00 G01 G02 G11 G12 G22
    double dd = 0.0;                                               // d'Wd: the scale of "zero" for the solver
    const float *M1 = NC > 1 ? M + (size_t)npix : M, *M2 = NC > 2 ? M + 2 * (size_t)npix : M;
    const double k1 = NC > 1 ? 1.0 : 0.0, k2 = NC > 2 ? 1.0 : 0.0;   // (absent components: exact zeros, as before)
#pragma unroll 4
    for (int i = threadIdx.x; i < npix; i += blockDim.x) {
        const double wi = w[i], di = d[i];
        const double m[3] = {(double)M[i], k1 * (double)M1[i], k2 * (double)M2[i]};
        g[0] += wi * m[0] * m[0]; g[1] += wi * m[0] * m[1]; g[2] += wi * m[0] * m[2];
        g[3] += wi * m[1] * m[1]; g[4] += wi * m[1] * m[2]; g[5] += wi * m[2] * m[2];
        bb[0] += wi * m[0] * di; bb[1] += wi * m[1] * di; bb[2] += wi * m[2] * di;
        dd += wi * di * di;
    }
    double G[3][3], b[3];
    double g0, g1, g2, g3, g4, g5, dwd;
    if (red_wide) {
        double v[10] = {g[0], g[1], g[2], g[3], g[4], g[5], bb[0], bb[1], bb[2], dd};
        block_sum_n<10>(v, red);
        g0 = v[0]; g1 = v[1]; g2 = v[2]; g3 = v[3]; g4 = v[4]; g5 = v[5]; b[0] = v[6]; b[1] = v[7]; b[2] = v[8]; dwd = v[9];
    } else {
        g0 = block_sum(g[0], red); g1 = block_sum(g[1], red); g2 = block_sum(g[2], red);
        g3 = block_sum(g[3], red); g4 = block_sum(g[4], red); g5 = block_sum(g[5], red);
        b[0] = block_sum(bb[0], red); b[1] = block_sum(bb[1], red); b[2] = block_sum(bb[2], red);
        dwd = block_sum(dd, red);
    }
    if (threadIdx.x == 0) {
        G[0][0] = g0; G[0][1] = G[1][0] = g1; G[0][2] = G[2][0] = g2; G[1][1] = g3; G[1][2] = G[2][1] = g4; G[2][2] = g5;
        // the paper's solver (Bro & De Jong's Gram-matrix active set), as in the MGE mode
        double s[3] = {0.0, 0.0, 0.0}, Lc[9], z[3];
        nnls_gram<3>(NC, &G[0][0], 3, b, dwd, s, Lc, z);
        // chi^2 = d'Wd - 2 s'b + s'G s at the solved amplitudes (Eq. 5), as in the MGE mode: the three
        // terms are FP64 sums of exact products of the FP32 columns, ~1e9 against chi^2 ~1e4 -- 1e-7 absolute, so
        // the second pass over the pixels that formed the residual is not needed
        double sb = 0.0, sGs = 0.0;
        for (int i = 0; i < NC; ++i) {
            if (s[i] == 0.0) continue;
            sb += s[i] * b[i];
            double gi = 0.0;
            for (int k = 0; k < NC; ++k) gi += G[i][k] * s[k];
            sGs += s[i] * gi;
        }
        const double chi2 = (dwd - 2.0 * sb) + sGs;
        a.logL[row] = (float)(-0.5 * (chi2 + a.lconst[lens]));
        if (a.amps) { a.amps[row * NC] = (float)s[0]; if (NC > 1) a.amps[row * NC + 1] = (float)s[1]; if (NC > 2) a.amps[row * NC + 2] = (float)s[2]; }
    }
}

__device__ __forceinline__ void invalid_row_lin(const KArgs &a, int64_t row)
{
    if (threadIdx.x == 0) {
        a.logL[row] = -INFINITY;
        if (a.amps) for (int k = 0; k < a.n_comp; ++k) a.amps[row * a.n_comp + k] = NAN;
    }
}

#ifdef TL_MAIN_TU
// staged pipeline: one CTA per row
__global__ void __launch_bounds__(256) solve_lin_kernel(const KArgs a, int chunk_rows)
{
    __shared__ double red[10 * 32];
    __shared__ double s_sh[3];
    const int r = blockIdx.x;
    const int64_t row = a.row0 + r;
    if (!row_is_valid(a.rows[r], a.n_comp)) { invalid_row_lin(a, row); return; }
    solve_row(a, a.mimg + (size_t)r * a.n_comp * a.ny * a.nx, row, row / a.rows_per_lens, red, s_sh, true);
}

#endif  // TL_MAIN_TU

// fused pipeline (when the C binned component images fit in shared memory): persistent CTAs,
// per row  trace (components apart, dynamic tile queue) -> C convolutions from shared memory,
// blurred columns of M to a per-CTA global scratch (L2-resident) -> solve_row.
template <int S_T, int NLL, int NSRC, int MASS = MASS_SIE>
__global__ void __launch_bounds__(512, 1) fused_lin_kernel(const KArgs a)
{
    constexpr int NC = NLL + NSRC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RowC *rc = reinterpret_cast<RowC *>(smem_raw);
    double *red = reinterpret_cast<double *>(smem_raw + sizeof(RowC));            // [0, 16): block_sum
    double *s_sh = red + 20;
    int *tile_counter = reinterpret_cast<int *>(red + 24);
    float *taps = reinterpret_cast<float *>(smem_raw + sizeof(RowC) + 32 * sizeof(double));
    float *img = taps + a.K * a.Kp;
    const int img_stride = (a.He * a.pitch + a.pitch + a.Kp + 8 + 3) & ~3;         // floats per component image
    RowV *rowtab = a.rowtab ? reinterpret_cast<RowV *>(img + NC * img_stride) : nullptr;
    for (int i = threadIdx.x; i < NC * img_stride; i += blockDim.x) img[i] = 0.f;
    const size_t npix = (size_t)a.ny * a.nx;
    float *M = a.mimg + (size_t)blockIdx.x * NC * npix;                            // this CTA's scratch

    int64_t cur_lens = -1;
    for (int64_t r = blockIdx.x; r < a.B; r += gridDim.x) {
        const int64_t row = a.row0 + r;
        const int64_t lens = row / a.rows_per_lens;
        __syncthreads();
        load_row_consts(rc, a.rows + r);
        if (threadIdx.x == 0) *tile_counter = 0;
        if (lens != cur_lens) { load_psf(taps, a.psf + lens * a.K * a.Kp, a.K * a.Kp); cur_lens = lens; }
        __syncthreads();
        if (!row_is_valid(*rc, a.n_comp)) { invalid_row_lin(a, row); continue; }
        if (rowtab) { fill_rowtab<NLL>(*rc, a, rowtab); __syncthreads(); }
        trace_image_lin<S_T, NLL, NSRC, MASS>(*rc, a, rowtab, threadIdx.x >> 5, blockDim.x >> 5, tile_counter,
                                        [&](int i, int j, int k, float v) { img[k * img_stride + i * a.pitch + j] = v; });
        __syncthreads();
#pragma unroll 1
        for (int k = 0; k < NC; ++k)
            conv_chi2_rows(a, img + k * img_stride, 0, taps, 0, a.ny, nullptr, nullptr, M + k * npix);
        __syncthreads();                               // M (global) visible to the whole CTA
        solve_row(a, M, row, lens, red, s_sh);
    }
}

}  // namespace tl
