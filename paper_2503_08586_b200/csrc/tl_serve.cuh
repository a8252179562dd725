// tl_serve.cuh -- NEXT-4 ("the CPU<->GPU round trips" of a sampler that
// proposes a handful of rows at a time): a PERSISTENT kernel that serves such requests without any launch.
//
// tl_serve_start launches serve_kernel once, one CTA per resident slot of every SM; it then polls a request
// block in pinned, mapped host memory.  tl_serve_eval writes the parameter rows and a sequence number there and
// spins on the answer -- no cudaMemcpy, no launch, no stream synchronisation on the way:
//   CTA 0     sees the new sequence number (ld.acquire.sys over PCIe), copies the rows to device memory, derives
//             the per-row constants (prologue_slot, the code of prologue_kernel) and publishes the request to the
//             other CTAs through a flag in device memory
//   all CTAs  ray-trace the rows, one pair of sub-samples per lane (trace_pairs_row, the code of
//             trace_pairs_kernel); one grid-wide barrier (a counter in device memory: every CTA is resident)
//   all CTAs  convolution + chi^2 of (row, band) blocks and the row's final reduction (conv_small_body, the code
//             of conv_small_kernel), logL written straight into the mapped request block; the CTA that finishes
//             the last row posts the sequence number back.
// Same device functions, same sums: logL is bit for bit tl_loglike_batch's.
// Every wait inside the kernel is bounded: the kernel leaves after `idle_ns` without a request and after `life_ns`
// whatever happens (tl_serve_eval then starts it again), so a lost host cannot leave a spinning GPU behind.
#pragma once
#include "tl_kernels.cuh"

namespace tl {

constexpr int SERVE_MAX_ROWS = 16;
constexpr int SERVE_MAX_P = 8 + 7 * MAX_COMP;
constexpr unsigned long long SERVE_EXIT = ~0ull;

struct ServeCtl {                        // pinned + mapped host memory
    unsigned long long seq;              // host -> device: number of the request to serve (0: none yet; SERVE_EXIT: leave)
    unsigned long long done;             // device -> host: number of the last request served
    int alive;                           // device -> host: 1 while the kernel runs
    int error;                           // device -> host: a wait inside the kernel ran out of time
    int B, per_row, bands, band_pairs, xseg, pad;      // the request and its launch geometry (host-computed)
    float params[SERVE_MAX_ROWS * SERVE_MAX_P];
    float logL[SERVE_MAX_ROWS];
};

struct ServeDev {                        // device memory
    unsigned long long seq;              // CTA 0 -> all CTAs
    unsigned long long start;            // the last request served before this launch
    unsigned long long bar;              // grid barrier: arrivals so far
    int B, per_row, bands, band_pairs, xseg, rows_done;
};

__device__ __forceinline__ unsigned long long ld_acquire_sys(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_release_sys(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long global_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// a.rows / a.ext / a.tile_counters: device buffers for SERVE_MAX_ROWS rows (the pitch padding of ext zeroed once
// by the host); a.logL = the mapped ctl->logL; pa.params = device staging for the rows, pa.rows = a.rows.
template <int S_T, int NLL, int NSRC>
__global__ void __launch_bounds__(TL_LB_T, TL_LB_B) serve_kernel(const KArgs a, const PrologueArgs pa, ServeCtl *ctl, ServeDev *dev,
                                                                 float *cblk, unsigned long long idle_ns, unsigned long long life_ns)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ RowC rc_s;
    __shared__ unsigned long long s_seq;
    __shared__ int s_hdr[5];
    const int G = gridDim.x, tid = threadIdx.x;
    const unsigned long long t_start = global_ns();
    unsigned long long last = dev->start, arrivals = 0;
    bool timed_out = false;
    if (blockIdx.x == 0 && tid == 0) { ctl->alive = 1; __threadfence_system(); }
    for (;;) {
        // ---- CTA 0: wait for the host, stage the rows, derive the row constants, publish
        if (blockIdx.x == 0) {
            if (tid == 0) {
                unsigned long long q;
                const unsigned long long t_idle = global_ns();
                for (;;) {
                    q = ld_acquire_sys(&ctl->seq);
                    if (q != last) break;
                    const unsigned long long now = global_ns();
                    if (now - t_idle > idle_ns || now - t_start > life_ns) { q = SERVE_EXIT; break; }
                }
                s_seq = q;
            }
            __syncthreads();
            const unsigned long long q = s_seq;
            if (q != SERVE_EXIT) {
                // header and rows in ONE round trip over PCIe: every word by a thread of its own (the rows are read
                // for the largest request; B is not known yet)
                const volatile int *h = &ctl->B;
                const volatile float *hp = ctl->params;
                float *dp = const_cast<float *>(pa.params);
                if (tid < 5) s_hdr[tid] = h[tid];
                for (int i = tid; i < SERVE_MAX_ROWS * pa.P; i += blockDim.x) dp[i] = hp[i];
                for (int i = tid; i < 2 * SERVE_MAX_ROWS; i += blockDim.x) a.tile_counters[i] = 0;
                __syncthreads();
                const int B = s_hdr[0];
                const int nslot = 1 + pa.n_lens_light + pa.n_source, lane = tid & 31;
                if (lane < B)
                    for (int slot = tid >> 5; slot < nslot; slot += blockDim.x >> 5) prologue_slot(pa, lane, slot);
                __threadfence();
                __syncthreads();
                if (tid == 0) {
                    dev->B = s_hdr[0]; dev->per_row = s_hdr[1]; dev->bands = s_hdr[2]; dev->band_pairs = s_hdr[3]; dev->xseg = s_hdr[4];
                    dev->rows_done = 0;
                    st_release_gpu(&dev->seq, q);
                }
            } else if (tid == 0) st_release_gpu(&dev->seq, SERVE_EXIT);
            __syncthreads();
        }
        // ---- every CTA: pick the request up
        if (tid == 0) {
            unsigned long long q;
            for (;;) {
                q = ld_acquire_gpu(&dev->seq);
                if (q != last) break;
                if (global_ns() - t_start > life_ns + 1000000000ull) { q = SERVE_EXIT; break; }     // (CTA 0 leaves first)
            }
            s_seq = q;
            if (q != SERVE_EXIT) { s_hdr[0] = dev->B; s_hdr[1] = dev->per_row; s_hdr[2] = dev->bands; s_hdr[3] = dev->band_pairs; s_hdr[4] = dev->xseg; }
        }
        __syncthreads();
        const unsigned long long q = s_seq;
        if (q == SERVE_EXIT) break;
        const int B = s_hdr[0], per_row = s_hdr[1], bands = s_hdr[2], band_pairs = s_hdr[3], xseg = s_hdr[4];
        // ---- ray-trace: virtual block (row, slab)
        for (int vb = blockIdx.x; vb < B * per_row; vb += G) {
            const int r = vb % B, y = vb / B;
            __syncthreads();
            load_row_consts(&rc_s, a.rows + r);
            __syncthreads();
            if (row_is_valid(rc_s, a.n_comp))
                trace_pairs_row<S_T, NLL, NSRC>(rc_s, a, a.ext + (size_t)r * a.He * a.pitch, (y * blockDim.x + tid) >> 5, (per_row * blockDim.x) >> 5);
        }
        // ---- grid barrier (all CTAs are resident)
        __syncthreads();
        arrivals += G;
        if (tid == 0) {
            __threadfence();
            atomicAdd(&dev->bar, 1ull);
            while (ld_acquire_gpu(&dev->bar) < arrivals)
                if (global_ns() - t_start > life_ns + 1000000000ull) { timed_out = true; break; }
            s_hdr[0] = timed_out ? -1 : B;
        }
        __syncthreads();
        if (s_hdr[0] < 0) { if (tid == 0) ctl->error = 1; break; }
        // ---- convolution + chi^2 + the rows' final reductions: virtual block (row, band x segment)
        const int n_by = bands * (xseg ? xseg : 1);
        for (int vb = blockIdx.x; vb < B * n_by; vb += G) {
            const int r = vb % B, by = vb / B;
            __syncthreads();
            const bool finished = conv_small_body(a, SERVE_MAX_ROWS, r, by, n_by, band_pairs, xseg, cblk, smem_raw, false);
            if (finished && tid == 0) {
                __threadfence_system();                            // this row's logL is on its way to the host
                if (atomicAdd(&dev->rows_done, 1) == B - 1) {
                    __threadfence_system();
                    st_release_sys(&ctl->done, q);
                }
            }
        }
        last = q;
    }
    if (blockIdx.x == 0 && tid == 0) { __threadfence_system(); ctl->alive = 0; __threadfence_system(); }
}

}  // namespace tl
