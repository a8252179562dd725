// tl_pair.cuh -- the per-sub-sample arithmetic of tl_sample.cuh on PAIRS of sub-samples, with
// Blackwell's packed FP32 instructions (fma / mul / add .f32x2 -> FFMA2 / FMUL2 / FADD2).
//
// Measured on B200 (`python bench.py --peaks`, profiles/r2_peaks.md): an FFMA2 occupies the FP32
// pipe for two cycles like two FFMAs, but takes ONE issue slot, and the scalar path of the fused
// kernel is bound by the issue port (79 % busy; FMA pipe 61 %, MUFU pipe 49 %).  Two horizontally
// adjacent sub-samples of a pixel share every row value and every per-row constant (these enter as
// broadcast scalar operands, "R.F32"), so all of steps a2-a4 except the MUFU calls and the sign
// handling can be issued once per pair.  A pair lives in an even-aligned register pair; the MUFU
// instructions read and write its halves in place, so packing and unpacking cost no instruction.
// Same formulas, same hi/lo constants applied low-term-first, same polynomials as tl_sample.cuh.
#pragma once
#include "tl_sample.cuh"

namespace tl {

struct f2 { unsigned long long v; };
__device__ __forceinline__ f2 mk2(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void un2(f2 a, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
__device__ __forceinline__ f2 bc2(float c) { return mk2(c, c); }        // ptxas turns this into a scalar broadcast operand
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
// scalar function on both halves (MUFU, sign operations)
#define TL_MAP2(name, fn)                                                                   \
    __device__ __forceinline__ f2 name(f2 a) { float x, y; un2(a, x, y); return mk2(fn(x), fn(y)); }
TL_MAP2(lg2_2, mufu_lg2)
TL_MAP2(ex2_2, mufu_ex2)
TL_MAP2(rsq_2, mufu_rsq)
TL_MAP2(rcp_2, mufu_rcp)
TL_MAP2(abs_2, fabsf)
#undef TL_MAP2
__device__ __forceinline__ f2 copysign_2(f2 mag, f2 sgn)
{
    float m0, m1, s0, s1;
    un2(mag, m0, m1); un2(sgn, s0, s1);
    return mk2(copysignf(m0, s0), copysignf(m1, s1));
}

__device__ __forceinline__ f2 atan_small2(f2 r)                  // tl_sample.cuh atan_small
{
    const f2 s = mul2(r, r);
    f2 p = bc2(3.199305013e-02f);
    p = fma2(p, s, bc2(-7.467620820e-02f));
    p = fma2(p, s, bc2(1.079487726e-01f));
    p = fma2(p, s, bc2(-1.425360143e-01f));
    p = fma2(p, s, bc2(1.999849826e-01f));
    p = fma2(p, s, bc2(-3.333331048e-01f));
    return fma2(mul2(r, s), p, r);
}

__device__ __forceinline__ f2 atanh_small2(f2 r)                 // tl_sample.cuh atanh_small
{
    const f2 s = mul2(r, r);
    f2 p = bc2(2.593644857e-01f);
    p = fma2(p, s, bc2(-5.470913649e-02f));
    p = fma2(p, s, bc2(1.322188675e-01f));
    p = fma2(p, s, bc2(1.043291166e-01f));
    p = fma2(p, s, bc2(1.434355527e-01f));
    p = fma2(p, s, bc2(1.999771595e-01f));
    p = fma2(p, s, bc2(3.333336413e-01f));
    return fma2(mul2(r, s), p, r);
}

// step a2 for two samples (tl_sample.cuh sie_alpha, q >= 0.5)
__device__ __forceinline__ void sie_alpha2(const SieHot &L, f2 xp, f2 yp, f2 &axp, f2 &ayp)
{
    const f2 xx = mul2(xp, xp);
    const f2 psi2 = fma2(bc2(L.q2h), xx, fma2(bc2(L.q2l), xx, fma2(yp, yp, bc2(1e-30f))));
    const f2 psi = mul2(psi2, rsq_2(psi2));
    const f2 ax = abs_2(xp), ay = abs_2(yp);
    const f2 Ax = fma2(ax, bc2(L.qph), mul2(ax, bc2(L.qpl))), Ay = fma2(ay, bc2(L.qph), mul2(ay, bc2(L.qpl)));
    const f2 d2 = fma2(Ax, bc2(L.s0), mul2(psi, bc2(L.c0)));
    const f2 n2 = fma2(Ax, bc2(L.c0), mul2(psi, bc2(-L.s0)));
    const f2 pa = atan_small2(mul2(n2, rcp_2(d2)));
    const f2 a1 = add2(fma2(bc2(L.fh), pa, fma2(bc2(L.fl), pa, bc2(L.ft0l))), bc2(L.ft0h));
    const f2 num = fma2(bc2(-L.z0), psi, Ay);
    const f2 den = fma2(bc2(-L.z0), Ay, psi);
    const f2 ph = atanh_small2(mul2(num, rcp_2(den)));
    const f2 a2 = add2(fma2(bc2(L.fh), ph, fma2(bc2(L.fl), ph, bc2(L.fT2l))), bc2(L.fT2h));
    axp = copysign_2(a1, xp);
    ayp = copysign_2(a2, yp);
}

// steps a3 / a4 for two samples (tl_sample.cuh sersic_from_t); flag0 / flag1: FP64 refinement wanted
__device__ __forceinline__ f2 sersic_from_t2(const SersicHot &C, f2 t, bool &flag0, bool &flag1)
{
    const f2 v = lg2_2(t);
    const f2 vp = fma2(v, bc2(C.ph), mul2(v, bc2(C.pl)));
    const f2 u = ex2_2(vp);
    const f2 arg = add2(fma2(bc2(-C.kh), u, fma2(bc2(-C.kl), u, bc2(C.kl))), bc2(C.kh));
    float c0, c1;
    un2(fma2(v, bc2(C.pm), arg), c0, c1);
    flag0 = c0 > C.nlcf; flag1 = c1 > C.nlcf;
    return ex2_2(arg);
}
__device__ __forceinline__ f2 sersic_from_t2(const SersicHot &C, f2 t)      // lens light: never refined
{
    const f2 v = lg2_2(t);
    const f2 u = ex2_2(fma2(v, bc2(C.ph), mul2(v, bc2(C.pl))));
    return ex2_2(add2(fma2(bc2(-C.kh), u, fma2(bc2(-C.kl), u, bc2(C.kl))), bc2(C.kh)));
}

__device__ __forceinline__ f2 quad_form2(const QuadHot &C, f2 x, f2 y)      // tl_sample.cuh quad_form
{
    const f2 w = fma2(bc2(C.ah), x, fma2(bc2(C.b2h), y, fma2(bc2(C.al), x, mul2(bc2(C.b2l), y))));
    return fma2(x, w, fma2(mul2(bc2(C.cch), y), y, mul2(mul2(bc2(C.ccl), y), y)));
}

// step a2, EPL, for NP pairs of sub-samples at once (tl_sample.cuh epl_alpha_vec: same formulas, same
// operations in the same order on each half, so the deflections are bit for bit the scalar ones; x - y is
// fma(y, -1, x), exact like the subtraction).  The exponent / mantissa split and the clamp stay scalar.
__device__ __forceinline__ f2 exp2_poly2(f2 x)                  // tl_sample.cuh exp2_poly
{
    const f2 big = add2(x, bc2(12582912.f));
    const f2 r = fma2(add2(big, bc2(-12582912.f)), bc2(-1.f), x);
    f2 p = bc2(1.545316336e-04f);
    p = fma2(p, r, bc2(1.339086331e-03f));
    p = fma2(p, r, bc2(9.618083015e-03f));
    p = fma2(p, r, bc2(5.550356954e-02f));
    p = fma2(p, r, bc2(2.402265072e-01f));
    p = fma2(p, r, bc2(6.931471825e-01f));
    p = fma2(p, r, bc2(1.0f));
    float p0, p1, b0, b1;
    un2(p, p0, p1); un2(big, b0, b1);
    return mk2(__int_as_float(__float_as_int(p0) + (__float_as_int(b0) << 23)),
               __int_as_float(__float_as_int(p1) + (__float_as_int(b1) << 23)));
}

template <int NP>
__device__ __forceinline__ void epl_alpha_pairs(const EplHot &L, const float *coef, const f2 (&xp)[NP], const f2 (&yp)[NP],
                                                f2 (&axp)[NP], f2 (&ayp)[NP])
{
    const f2 m1 = bc2(-1.f);
    f2 c2[NP], s2[NP], pc[NP], ps[NP], tc[NP], b1[NP], b2[NP];
#pragma unroll
    for (int s = 0; s < NP; ++s) {
        const f2 xx = mul2(xp[s], xp[s]);
        const f2 psi2 = fma2(bc2(L.q2h), xx, fma2(bc2(L.q2l), xx, fma2(yp[s], yp[s], bc2(1e-30f))));   // R^2 (> 0, G6)
        const f2 rinv = rsq_2(psi2);
        const f2 cph = mul2(fma2(xp[s], bc2(L.qh), mul2(xp[s], bc2(L.ql))), rinv), sph = mul2(yp[s], rinv);   // e^{i phi}
        c2[s] = mul2(fma2(sph, m1, cph), add2(cph, sph));
        s2[s] = mul2(mul2(bc2(2.f), cph), sph);                                                         // w = e^{2 i phi}
        float v0, v1;
        un2(mul2(psi2, bc2(L.invb2)), v0, v1);
        const int vb0 = __float_as_int(v0), vb1 = __float_as_int(v1);
        const f2 ef = add2(mk2(__int_as_float((vb0 >> 23) | 0x4b000000), __int_as_float((vb1 >> 23) | 0x4b000000)), bc2(-8388735.f));
        const f2 lm = mk2(mufu_lg2(__int_as_float((vb0 & 0x007fffff) | 0x3f800000)),
                          mufu_lg2(__int_as_float((vb1 & 0x007fffff) | 0x3f800000)));                    // mantissas in [1, 2)
        float a0, a1;
        un2(fma2(ef, bc2(L.kh), fma2(lm, bc2(L.kh), mul2(add2(ef, lm), bc2(L.kl)))), a0, a1);
        const f2 pw = exp2_poly2(mk2(fminf(fmaxf(a0, -100.f), 100.f), fminf(fmaxf(a1, -100.f), 100.f)));
        const f2 P = fma2(pw, bc2(L.a0h), mul2(pw, bc2(L.a0l)));
        pc[s] = mul2(P, cph); ps[s] = mul2(P, sph);
        tc[s] = mul2(bc2(2.f), c2[s]); b1[s] = bc2(0.f); b2[s] = bc2(0.f);
    }
    // Clenshaw, two terms per trip (nterm is even)
    for (int n = L.nterm; n >= 2; n -= 2) {
        const float2 cf = *reinterpret_cast<const float2 *>(coef + n - 2);                  // a_{n-1}, a_n
#pragma unroll
        for (int s = 0; s < NP; ++s) {
            b2[s] = fma2(b2[s], m1, fma2(tc[s], b1[s], bc2(cf.y)));                         // b_n
            b1[s] = fma2(b1[s], m1, fma2(tc[s], b2[s], bc2(cf.x)));                         // b_{n-1}
        }
    }
#pragma unroll
    for (int s = 0; s < NP; ++s) {
        const f2 b0 = fma2(b2[s], m1, fma2(tc[s], b1[s], bc2(1.f)));                        // a_0 = 1
        const f2 sr = fma2(mul2(c2[s], m1), b1[s], b0), si = mul2(s2[s], b1[s]);
        axp[s] = fma2(pc[s], sr, mul2(mul2(ps[s], m1), si));
        ayp[s] = fma2(pc[s], si, mul2(ps[s], sr));
    }
}

}  // namespace tl
