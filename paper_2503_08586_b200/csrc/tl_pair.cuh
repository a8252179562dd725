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

}  // namespace tl
