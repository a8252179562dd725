// tl_peaks.cu -- tl_measure_peaks: issue-rate micro-benchmarks of the pipes the hot path is bound
// by.  The roofline denominator of
// bench.py (148 SMs x 128 thread-instruction slots per clock) and the choice between scalar FFMA,
// packed FFMA2 and the FP64 pipe for each piece of the kernels are decided by these numbers, so
// they are measured by committed code (`python bench.py --peaks`), not by loose probes.
//
// Every probe runs one persistent CTA of 1024 threads per SM (32 warps: enough to cover the
// dependent-issue latency of every pipe), each thread iterating over 8 independent dependency
// chains; SM cycles are read with clock64() round the loop, the slowest CTA counts.
#include <cstdint>
#include <cstring>
#include <cuda_runtime.h>

#include "../../include/tinylens.h"

namespace {

__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
// p = p * a + b on both halves, in place (a separate destination made ptxas shuffle the register
// pairs with 12 MOVs per loop trip)
__device__ __forceinline__ void ffma2_acc(unsigned long long &p, unsigned long long a, unsigned long long b)
{
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p) : "l"(a), "l"(b));
}
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ double rcp64h(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double rsq64h(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }

enum {
    P_FFMA = 0,        // 8 scalar FFMA per trip
    P_FFMA2,           // 8 packed FFMA2 per trip (16 FMAs)
    P_FFMA_MUFU,       // 7 FFMA + 1 MUFU.EX2
    P_FFMA2_MUFU,      // 6 FFMA2 + 2 MUFU.EX2
    P_MUFU,            // 8 MUFU.EX2
    P_DFMA,            // 8 DFMA
    P_DFMA_FFMA,       // 4 DFMA + 4 FFMA
    P_DFMA_FFMA2,      // 4 DFMA + 4 FFMA2
    P_DFMA_MUFU,       // 6 DFMA + 2 MUFU.EX2
    P_F2F,             // 4 x (F2F.F64.F32 + F2F.F32.F64)
    P_RCP64H,          // 8 MUFU.RCP64H
    P_COUNT
};

template <int KIND>
__global__ void __launch_bounds__(1024, 1) probe_kernel(int trips, float seed, unsigned long long *cycles, float *sink)
{
    float f[8];
    double d[8];
    unsigned long long p[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        f[i] = seed + 0.001f * (float)(threadIdx.x + i);
        d[i] = (double)f[i];
        p[i] = pack2(f[i], f[i] + 0.5f);
    }
    const float a = 0.999f + seed * 1e-6f, b = 1e-3f;
    const double da = (double)a, db = (double)b;
    const unsigned long long pa = pack2(a, a), pb = pack2(b, b);
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
        if (KIND == P_FFMA) {
#pragma unroll
            for (int i = 0; i < 8; ++i) f[i] = fmaf(f[i], a, b);
        } else if (KIND == P_FFMA2) {
            // four rounds per trip: ptxas gives FFMA2 a destination pair different from its source
            // pair and would otherwise copy the 8 pairs back at the end of every trip
#pragma unroll
            for (int rep = 0; rep < 4; ++rep)
#pragma unroll
                for (int i = 0; i < 8; ++i) ffma2_acc(p[i], pa, pb);
        } else if (KIND == P_FFMA_MUFU) {
#pragma unroll
            for (int i = 0; i < 7; ++i) f[i] = fmaf(f[i], a, b);
            f[7] = mufu_ex2(f[7]) - 1.f;
        } else if (KIND == P_FFMA2_MUFU) {
#pragma unroll
            for (int rep = 0; rep < 4; ++rep) {
#pragma unroll
                for (int i = 0; i < 6; ++i) ffma2_acc(p[i], pa, pb);
                f[6] = mufu_ex2(f[6] * b);
                f[7] = mufu_ex2(f[7] * b);
            }
        } else if (KIND == P_MUFU) {
#pragma unroll
            for (int i = 0; i < 8; ++i) f[i] = mufu_ex2(f[i]);
        } else if (KIND == P_DFMA) {
#pragma unroll
            for (int i = 0; i < 8; ++i) d[i] = fma(d[i], da, db);
        } else if (KIND == P_DFMA_FFMA) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { d[i] = fma(d[i], da, db); f[i] = fmaf(f[i], a, b); }
        } else if (KIND == P_DFMA_FFMA2) {
#pragma unroll
            for (int rep = 0; rep < 4; ++rep)
#pragma unroll
                for (int i = 0; i < 4; ++i) { d[i] = fma(d[i], da, db); ffma2_acc(p[i], pa, pb); }
        } else if (KIND == P_DFMA_MUFU) {
#pragma unroll
            for (int i = 0; i < 6; ++i) d[i] = fma(d[i], da, db);
            f[6] = mufu_ex2(f[6] * b);
            f[7] = mufu_ex2(f[7] * b);
        } else if (KIND == P_F2F) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { d[i] = (double)f[i] + db; f[i] = (float)d[i]; }
        } else if (KIND == P_RCP64H) {
#pragma unroll
            for (int i = 0; i < 8; ++i) d[i] = rcp64h(d[i]);
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i] + (float)d[i] + __uint_as_float((unsigned)(p[i] >> 32)) + __uint_as_float((unsigned)p[i]);
    if (s == 123.456f) sink[0] = s;                    // keeps the chains alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

// worst relative error of the FP64 seeds (MUFU.RCP64H / MUFU.RSQ64H) and of one Newton step on
// them, over 2^20 arguments in [1, 4): what the FP64 kernels of tl_dp.cuh rely on
__global__ void seed_accuracy_kernel(double *out)
{
    double e_rcp = 0.0, e_rsq = 0.0, e_rcp1 = 0.0, e_rsq1 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < (1 << 20); i += gridDim.x * blockDim.x) {
        const double x = 1.0 + 3.0 * ((double)i + 0.37) / (double)(1 << 20);
        const double r = rcp64h(x), q = rsq64h(x);
        const double r1 = fma(r, fma(-x, r, 1.0), r);
        const double hq = 0.5 * q, q1 = fma(hq, fma(-x * q, q, 1.0), q);
        e_rcp = fmax(e_rcp, fabs(r * x - 1.0));
        e_rcp1 = fmax(e_rcp1, fabs(r1 * x - 1.0));
        e_rsq = fmax(e_rsq, fabs(q * q * x - 1.0) * 0.5);
        e_rsq1 = fmax(e_rsq1, fabs(q1 * q1 * x - 1.0) * 0.5);
    }
    // max over the grid through ordered integer atomics (all values are >= 0)
    atomicMax(reinterpret_cast<unsigned long long *>(out + 0), (unsigned long long)__double_as_longlong(e_rcp));
    atomicMax(reinterpret_cast<unsigned long long *>(out + 1), (unsigned long long)__double_as_longlong(e_rcp1));
    atomicMax(reinterpret_cast<unsigned long long *>(out + 2), (unsigned long long)__double_as_longlong(e_rsq));
    atomicMax(reinterpret_cast<unsigned long long *>(out + 3), (unsigned long long)__double_as_longlong(e_rsq1));
}

struct ProbeDesc { const char *name; double ops_per_trip; double fma_per_trip; };
const ProbeDesc DESCS[P_COUNT] = {
    {"8 FFMA", 8, 8},
    {"32 FFMA2 (fma.rn.f32x2)", 32, 64},
    {"7 FFMA + 1 MUFU.EX2", 8, 7},
    {"4 x (6 FFMA2 + 2 MUFU.EX2 + 2 FMUL)", 40, 56},
    {"8 MUFU.EX2", 8, 0},
    {"8 DFMA", 8, 8},
    {"4 DFMA + 4 FFMA", 8, 8},
    {"4 x (4 DFMA + 4 FFMA2)", 32, 48},
    {"6 DFMA + 2 MUFU.EX2 (+2 FMUL)", 10, 6},
    {"4 x (F2F.F64.F32 + DADD + F2F.F32.F64)", 12, 0},
    {"8 MUFU.RCP64H", 8, 0},
};

typedef void (*probe_fn)(int, float, unsigned long long *, float *);
const probe_fn FNS[P_COUNT] = {
    probe_kernel<P_FFMA>, probe_kernel<P_FFMA2>, probe_kernel<P_FFMA_MUFU>, probe_kernel<P_FFMA2_MUFU>, probe_kernel<P_MUFU>,
    probe_kernel<P_DFMA>, probe_kernel<P_DFMA_FFMA>, probe_kernel<P_DFMA_FFMA2>, probe_kernel<P_DFMA_MUFU>, probe_kernel<P_F2F>,
    probe_kernel<P_RCP64H>,
};

}  // namespace

extern "C" int tl_measure_peaks(tl_peak *out, int32_t n_max, double *seed_err4)
{
    if (!out || n_max < 1) return TL_EINVAL;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return TL_ECUDA;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm < 1) return TL_ECUDA;
    unsigned long long *cyc = nullptr;
    float *sink = nullptr;
    double *serr = nullptr;
    if (cudaMalloc(&cyc, sizeof(unsigned long long) * n_sm) != cudaSuccess) return TL_ENOMEM;
    if (cudaMalloc(&sink, sizeof(float)) != cudaSuccess) { cudaFree(cyc); return TL_ENOMEM; }
    if (cudaMalloc(&serr, 4 * sizeof(double)) != cudaSuccess) { cudaFree(cyc); cudaFree(sink); return TL_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int trips = 1 << 16;
    int n = 0, rc = TL_OK;
    unsigned long long *h = new unsigned long long[n_sm];
    for (int k = 0; k < P_COUNT && n < n_max; ++k, ++n) {
        FNS[k]<<<n_sm, 1024>>>(1024, 1.f, cyc, sink);                    // warm-up
        cudaEventRecord(e0);
        FNS[k]<<<n_sm, 1024>>>(trips, 1.f, cyc, sink);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = TL_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h, cyc, sizeof(unsigned long long) * n_sm, cudaMemcpyDeviceToHost);
        unsigned long long mx = 0;
        for (int i = 0; i < n_sm; ++i) if (h[i] > mx) mx = h[i];
        tl_peak &o = out[n];
        memset(&o, 0, sizeof(o));
        strncpy(o.name, DESCS[k].name, sizeof(o.name) - 1);
        o.inst_per_clk_sm = DESCS[k].ops_per_trip * trips * 1024.0 / (double)mx;
        o.fma_per_clk_sm = DESCS[k].fma_per_trip * trips * 1024.0 / (double)mx;
        o.sm_mhz = (double)mx / (ms * 1e3);
        o.ms = ms;
    }
    if (rc == TL_OK && seed_err4) {
        cudaMemset(serr, 0, 4 * sizeof(double));
        seed_accuracy_kernel<<<n_sm, 256>>>(serr);
        if (cudaMemcpy(seed_err4, serr, 4 * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) rc = TL_ECUDA;
    }
    delete[] h;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(cyc); cudaFree(sink); cudaFree(serr);
    if (cudaGetLastError() != cudaSuccess) rc = TL_ECUDA;
    return rc == TL_OK ? n : rc;
}
