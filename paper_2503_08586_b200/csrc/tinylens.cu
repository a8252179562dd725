// tinylens.cu -- C ABI (include/tinylens.h) and host-side launch logic.
//
// No CPU fallback lives here: every compute entry point either enqueues the CUDA kernels of
// tl_kernels.cuh or returns an error code.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <ctime>
#include <mutex>
#include <unordered_map>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/tinylens.h"
#define TL_MAIN_TU            /* this unit owns the non-template kernels */
#include "tl_kernels.cuh"
#include "tl_dispatch.h"
#include "tl_precise.cuh"
#include "tl_dp.cuh"
#include "tl_mge.cuh"
#include "tl_serve.cuh"

#define TL_VERSION_STRING "tinylens-b200 0.2 (sm_100a)"

typedef void (*dp_trace_fn)(const tl::DpArgs);
template <int S_T>
static dp_trace_fn tl_trace_dp_s(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_dp_kernel<S_T, 0, 1> : tl::trace_dp_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::trace_dp_kernel<S_T, 1, 1> : tl::trace_dp_kernel<S_T, 1, 2>;
}
static dp_trace_fn tl_trace_dp_for(int S, int nll, int nsrc)
{
    switch (S) {
    case 1: return tl_trace_dp_s<1>(nll, nsrc);
    case 2: return tl_trace_dp_s<2>(nll, nsrc);
    case 4: return tl_trace_dp_s<4>(nll, nsrc);
    case 8: return tl_trace_dp_s<8>(nll, nsrc);
    default: return tl_trace_dp_s<0>(nll, nsrc);
    }
}

struct tl_ctx {
    tl_config cfg;
    int device = 0;
    int n_sm = 0;
    int P = 0, lens_np = 7, K = 0, Kp = 0, h = 0, He = 0, We = 0, pitch = 0, n_comp = 0;
    // device arrays (library-owned)
    float *psf = nullptr, *data = nullptr, *wgt = nullptr, *sigma_min = nullptr, *noise = nullptr;
    double *wgt64 = nullptr;      // 1 / sigma^2 in FP64 (the double-precision path, tl_dp.cuh)
    int precision = 0;            // TL_PRECISION_*
    // double-precision path: launch geometry
    int dp_Wp = 0, dp_band_rows = 0, dp_n_bands = 0, dp_trace_grid = 0, dp_conv_threads = 256;
    size_t dp_conv_smem = 0;
    int64_t dp_chunk_rows = 0;
    void (*dp_trace)(const tl::DpArgs) = nullptr;
    void (*mge_dp_trace)(const tl::DpArgs) = nullptr;   // FP64 MGE pipeline: the sources only (NLL = 0)
    double *lconst = nullptr;
    double lconst0 = 0.0, sigma_min0 = 0.0;
    // launch geometry
    int path = 0;                 // 0 fused, 1 split
    int threads = 256, ctas_per_sm = 1, grid = 1;
    size_t smem = 0;
    int tile_rows = 0, n_tiles = 0, CW = 32, CH = 1, trace_slabs = 1;
    // linear-amplitude mode (tl_loglike_linear_batch): always the staged pipeline
    void (*trace_lin)(const tl::KArgs, int) = nullptr;
    int lin_tile_rows = 0, lin_n_tiles = 0, lin_rowtab = 0;
    void (*fused_lin)(const tl::KArgs) = nullptr;     // component images in shared memory, when they fit
    size_t lin_fused_smem = 0;
    int lin_fused_rowtab = 0, lin_fused_grid = 0;
    size_t lin_conv_smem = 0, lin_trace_smem = 0;
    int rowtab = 0;               // RowV table in shared memory (fused: after the image; split: trace_kernel)
    size_t trace_smem = 0;
    void (*fused)(const tl::KArgs) = nullptr;
    void (*trace)(const tl::KArgs, int) = nullptr;
    size_t conv_smem = 0;
    int64_t chunk_rows = 0;       // rows per scratch chunk
    // small-batch path of fused contexts (rows spread over many CTAs, bitwise equal to fused)
    void (*sb_trace)(const tl::KArgs, int) = nullptr;
    void (*sb_pairs)(const tl::KArgs, int) = nullptr;      // trace_pairs_kernel: calls of at most sb_pairs_rows rows
    int sb_pairs_rows = 0;
    size_t sb_trace_smem = 0;
    int sb_rowtab = 0, sb_max_rows = 0;
    // MGE mode (tl_set_mge / tl_loglike_mge_batch)
    float *mge_c = nullptr;       // device [n_gauss]: log2(e) / (2 sigma_k^2)
    double *mge_c64 = nullptr;    // the same in FP64, for the FP64 pipeline (a float coefficient is 6e-8 off: 3e-7 in the profile at 3 sigma)
    int *mge_set = nullptr;       // device [n_gauss]: the set each Gaussian belongs to
    int n_gauss = 0, mge_n_sets = 0, mge_per_set[tl::MGE_MAX_SETS] = {0, 0};
    void (*mge_trace)(const tl::KArgs, int) = nullptr;   // sources only: trace_kernel<S,0,1> or trace_lin_kernel<S,0,2>
    size_t mge_trace_smem = 0, mge_gc_smem = 0;
    int mge_rowtab = 0, mge_fused = 0;                   // fused: gauss_conv_kernel (extended image in shared memory)
    double refine_tau = 7.5e-4;   // x S at create: a pixel averages S^2 samples
    // asynchronous host entry (tl_loglike_batch_host_async / tl_wait): two staging slots, each with
    // pinned host and device buffers for one batch, an upload and a download stream of the library's
    // own, so that the upload of batch k + 1 overlaps the kernels of batch k
    struct HostSlot {
        float *h_params = nullptr, *h_logl = nullptr, *d_params = nullptr, *d_logl = nullptr;
        int64_t cap_rows = 0, B = 0;
        float *user_logl = nullptr;
        cudaEvent_t up = nullptr, done = nullptr, fin = nullptr;
        int busy = 0, rc = 0;
    } slots[2];
    int next_slot = 0;
    cudaStream_t s_up = nullptr, s_down = nullptr;
    // serve mode (tl_serve_start: the persistent kernel of tl_serve.cuh)
    struct Serve {
        serve_fn fn = nullptr;
        tl::ServeCtl *ctl = nullptr, *ctl_dev = nullptr;     // pinned + mapped request block: host / device address
        tl::ServeDev *dev = nullptr;
        tl::RowC *rows = nullptr;
        float *ext = nullptr, *cblk = nullptr, *params = nullptr;
        int *counters = nullptr;
        cudaStream_t stream = nullptr;
        int grid = 0, max_rows = 0;
        size_t smem = 0;
        unsigned long long seq = 0, idle_ns = 0;
    } sv;
    tl_options opt;               // create-time options (tl_create_ex); defaults = automatic
    // tl_options.debug_canaries: every scratch allocation carries 256 guard bytes on either side, checked when it is freed
    int *canary_errors = nullptr;                              // device counter of guard words found changed
    mutable std::mutex canary_mu;
    mutable std::unordered_map<void *, size_t> canary_size;    // user pointer -> bytes (rounded up to 256)
    cudaMemPool_t pool = nullptr; // library-owned stream-ordered pool: per-call scratch (never the device's default pool)
    // benchmark facility (tl_set_profiling): events around the dominant kernel of the last call
    int profile = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    int prof_pending = 0;
};

namespace {

// phase-1 warp tile CW x CH = 32 lanes: the shape that wastes the fewest lanes on the ragged
// right / bottom edge of the extended image
void best_warp_tile(int He, int We, int *CW, int *CH)
{
    double best = -1.0;
    for (int cw = 32; cw >= 1; cw >>= 1) {
        const int ch = 32 / cw;
        const double eff = (double)He * We / ((double)((We + cw - 1) / cw * cw) * ((He + ch - 1) / ch * ch));
        if (eff > best + 1e-12) { best = eff; *CW = cw; *CH = ch; }
    }
}

constexpr size_t SMEM_LIMIT = 227 * 1024;
constexpr int64_t CONST_CHUNK = 1 << 17;        // rows of RowC scratch per chunk (fused path)
constexpr size_t EXT_SCRATCH_BYTES = 512u << 20; // split path: binned-image scratch per chunk
constexpr size_t MGE_SCRATCH_BYTES = (size_t)2 << 30;  // MGE: source images + blurred columns of a chunk of rows

inline bool cuda_ok(cudaError_t e) { return e == cudaSuccess; }

// The context is bound to the device that was current at tl_create; calls made with another
// device current switch to it for their duration and restore the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool ok = true, switched = false;
    explicit DeviceGuard(int want)
    {
        ok = cuda_ok(cudaGetDevice(&prev));
        if (ok && prev != want) { ok = cuda_ok(cudaSetDevice(want)); switched = ok; }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// per-call scratch: stream-ordered allocation from the context's own pool
constexpr size_t CANARY_BYTES = 256;
constexpr unsigned CANARY_WORD = 0xA5A5A5A5u;

__global__ void canary_check_kernel(const unsigned *front, const unsigned *back, int *errors)
{
    if (front[threadIdx.x] != CANARY_WORD) atomicAdd(errors, 1);
    if (back[threadIdx.x] != CANARY_WORD) atomicAdd(errors, 1);
}

template <class T>
inline bool pool_alloc(const tl_ctx *c, T **p, size_t bytes, cudaStream_t st)
{
    *p = nullptr;
    void *v = nullptr;
    const bool guard = c->canary_errors != nullptr;
    const size_t body = guard ? ((bytes ? bytes : 1) + CANARY_BYTES - 1) / CANARY_BYTES * CANARY_BYTES : (bytes ? bytes : 1);
    const size_t total = guard ? body + 2 * CANARY_BYTES : body;
    const cudaError_t e = c->pool ? cudaMallocFromPoolAsync(&v, total, c->pool, st) : cudaMallocAsync(&v, total, st);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    if (guard) {
        unsigned char *b = static_cast<unsigned char *>(v);
        cudaMemsetAsync(b, 0xA5, CANARY_BYTES, st);
        cudaMemsetAsync(b + CANARY_BYTES, 0xFF, body, st);           // the body starts as NaNs / -1: a read of scratch nobody wrote shows in the result
        cudaMemsetAsync(b + CANARY_BYTES + body, 0xA5, CANARY_BYTES, st);
        v = b + CANARY_BYTES;
        std::lock_guard<std::mutex> lock(c->canary_mu);
        c->canary_size[v] = body;
    }
    *p = static_cast<T *>(v);
    return true;
}

inline void pool_free(const tl_ctx *c, void *p, cudaStream_t st)
{
    if (!p) return;
    if (c->canary_errors) {
        size_t body = 0;
        {
            std::lock_guard<std::mutex> lock(c->canary_mu);
            auto it = c->canary_size.find(p);
            if (it != c->canary_size.end()) { body = it->second; c->canary_size.erase(it); }
        }
        if (body) {
            unsigned char *b = static_cast<unsigned char *>(p) - CANARY_BYTES;
            canary_check_kernel<<<1, (unsigned)(CANARY_BYTES / sizeof(unsigned)), 0, st>>>(
                reinterpret_cast<const unsigned *>(b), reinterpret_cast<const unsigned *>(b + CANARY_BYTES + body), c->canary_errors);
            p = b;
        }
    }
    cudaFreeAsync(p, st);
}

size_t fused_smem_bytes(const tl_ctx *c)
{
    return sizeof(tl::RowC) + 32 * sizeof(double) + sizeof(float) * ((size_t)c->K * c->Kp + (size_t)(c->He + 1) * c->pitch + c->Kp + 8);
}

size_t conv_smem_bytes(const tl_ctx *c, int tile_rows)
{
    return 32 * sizeof(double) + sizeof(float) * ((size_t)c->K * c->Kp + (size_t)(tile_rows + 2 * c->h + 1) * c->pitch + c->Kp + 8);
}

tl::KArgs base_args(const tl_ctx *c)
{
    tl::KArgs a;
    memset(&a, 0, sizeof(a));
    a.psf = c->psf; a.data = c->data; a.wgt = c->wgt; a.lconst = c->lconst;
    a.ny = c->cfg.ny; a.nx = c->cfg.nx; a.K = c->K; a.Kp = c->Kp; a.h = c->h;
    a.He = c->He; a.We = c->We; a.pitch = c->pitch; a.S = c->cfg.supersample;
    a.n_lens_light = c->cfg.n_lens_light; a.n_comp = c->n_comp;
    a.edge_zero = c->cfg.edge_mode == TL_EDGE_ZERO;
    a.tile_rows = c->tile_rows; a.n_tiles = c->n_tiles;
    a.rowtab = c->rowtab;
    a.CW = c->CW; a.CH = c->CH; a.tiles_x = (c->We + c->CW - 1) / c->CW; a.tiles_y = (c->He + c->CH - 1) / c->CH;
    return a;
}

void fill_prologue_args(const tl_ctx *c, tl::PrologueArgs &pa, const float *params, tl::RowC *rows, int64_t nb, int64_t r0,
                        int64_t rows_per_lens, int unit_amp)
{
    pa.params = params + r0 * c->P; pa.rows = rows; pa.sigma_min = c->sigma_min;
    pa.B = nb; pa.row0 = r0; pa.rows_per_lens = rows_per_lens;
    pa.P = c->P; pa.n_lens_light = c->cfg.n_lens_light; pa.n_source = c->cfg.n_source;
    pa.S = c->cfg.supersample;
    pa.mass_model = c->cfg.mass_model; pa.lens_np = c->lens_np;
    pa.inv_u = 2.0 * c->cfg.supersample / c->cfg.pix_scale;
    pa.fov_half = 0.5 * c->cfg.pix_scale * (c->He > c->We ? c->He : c->We);
    pa.refine_tau = c->refine_tau;
    pa.unit_amp = unit_amp; pa.mge = 0;
    pa.zero_words = nullptr; pa.n_zero_words = 0; pa.pad_ext = nullptr; pa.pad_rows = 0; pa.pad_pitch = 0; pa.pad_We = 0;
}

// B <= n_sm / 2 rows on a fused context: prologue -> trace_kernel (rows x slabs) -> conv_small_kernel
// (rows x bands; the row's last band reduces); bitwise the fused kernel's result (tl_kernels.cuh)
// `params`, `logL`, `images` address the whole call; the B rows served are row0 .. row0 + B - 1 of it, a lens owning
// rows_per_lens consecutive rows of the call (0: B / n_lens, i.e. the B rows are the whole call)
int run_small_batch(tl_ctx *c, const float *params, int64_t B, float *logL, float *images, cudaStream_t st,
                    int64_t row0 = 0, int64_t rows_per_lens = 0)
{
    const int nb = (int)B;
    if (rows_per_lens == 0) rows_per_lens = B / c->cfg.n_lens;
    const int npair = (c->cfg.ny + 1) / 2, nsx = (c->cfg.nx + 3) / 4;
    // binned images, then one work-queue head and one finished-band counter per row; zeroed together
    const size_t img_bytes = sizeof(float) * (size_t)nb * c->He * c->pitch;
    const size_t ext_bytes = img_bytes + 2 * sizeof(int) * (size_t)nb;     // + finished-band counters
    // ONE allocation (rows | images + counters | chi^2 terms) and no memset: on this path the host-side
    // API calls are the cost (a one-row call is ~25 us of GPU work)
    const size_t rows_bytes = (sizeof(tl::RowC) * (size_t)nb + 255) & ~(size_t)255;
    const size_t ext_al = (ext_bytes + 255) & ~(size_t)255;
    const size_t cblk_bytes = logL ? sizeof(float) * (size_t)nb * npair * nsx : 0;
    unsigned char *blob = nullptr;
    if (!pool_alloc(c, &blob, rows_bytes + ext_al + cblk_bytes, st)) return TL_ENOMEM;
    tl::RowC *rows = reinterpret_cast<tl::RowC *>(blob);
    float *ext = reinterpret_cast<float *>(blob + rows_bytes);
    float *cblk = logL ? reinterpret_cast<float *>(blob + rows_bytes + ext_al) : nullptr;
    tl::PrologueArgs pa;
    fill_prologue_args(c, pa, params, rows, nb, row0, rows_per_lens, 0);
    pa.zero_words = reinterpret_cast<int *>(reinterpret_cast<unsigned char *>(ext) + img_bytes); pa.n_zero_words = 2 * nb;
    pa.pad_ext = ext; pa.pad_rows = nb * c->He; pa.pad_pitch = c->pitch; pa.pad_We = c->We;
    tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);
    tl::KArgs a = base_args(c);
    a.rows = rows; a.B = nb; a.rows_per_lens = rows_per_lens; a.row0 = row0;
    a.logL = logL; a.images = images; a.ext = ext; a.rowtab = c->sb_rowtab;
    a.tile_counters = reinterpret_cast<int *>(reinterpret_cast<unsigned char *>(ext) + img_bytes);
    // as many CTAs per row as are resident at once (two per SM; one more would start a second,
    // nearly empty wave), but no more than there are warp tiles / row pairs
    int want = 2 * c->n_sm / nb;
    if (want < 1) want = 1;
    const int n_wtiles = a.tiles_x * a.tiles_y;
    int slabs = want < (n_wtiles + 7) / 8 ? want : (n_wtiles + 7) / 8;
    int bands = want < npair ? want : npair;
    // the whole band (+ K - 1 rows of halo) and the taps must fit in shared memory
    const size_t fixed = sizeof(float) * ((size_t)c->K * c->Kp + c->pitch + c->Kp + 8);
    int band_pairs = (npair + bands - 1) / bands;
    const int max_pairs = (int)(((SMEM_LIMIT - 1024 - fixed) / (sizeof(float) * c->pitch) - (c->K - 1)) / 2);
    if (band_pairs > max_pairs) band_pairs = max_pairs;
    bands = (npair + band_pairs - 1) / band_pairs;
    // few rows: the K kernel rows of a 2 x 4 block on K threads (conv_blocks_split), the CTAs left over
    // splitting the bands along x; it pays while a CTA gets through its blocks in one or two passes
    const int per_pass = c->threads / c->K;
    int xseg = want / bands;
    const int one_pass = (band_pairs * nsx + per_pass - 1) / per_pass;
    if (xseg > one_pass) xseg = one_pass;
    if (xseg > nsx) xseg = nsx;
    if (xseg < 1) xseg = 1;
    if ((band_pairs * ((nsx + xseg - 1) / xseg) + per_pass - 1) / per_pass > 2) xseg = 0;
    const size_t conv_smem = fixed + sizeof(float) * ((size_t)(2 * band_pairs + c->K - 1) * c->pitch + (xseg ? (size_t)per_pass * c->K * 8 : 0));
    // programmatic dependent launch: the next kernel's CTAs are scheduled while the previous one drains
    // (the kernels wait with griddepcontrol.wait before touching what their predecessor wrote)
    cudaLaunchAttribute pdl;
    pdl.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    pdl.val.programmaticStreamSerializationAllowed = c->profile ? 0 : 1;     // (profiling events sit between the kernels)
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof(lc));
    lc.stream = st; lc.attrs = &pdl; lc.numAttrs = 1;
    if (c->profile) cudaEventRecord(c->ev0, st);
    bool okl;
    if (c->sb_pairs && nb <= c->sb_pairs_rows) {
        // one pair of sub-samples per lane, one warp tile per warp (tl_kernels.cuh trace_pairs_kernel)
        const int S = c->cfg.supersample, ppw = 32 / (S * S / 2);
        const int n_wt = (c->He * c->We + ppw - 1) / ppw;
        a.rowtab = 0;
        const int per_row = want < (n_wt + 7) / 8 ? want : (n_wt + 7) / 8;
        lc.gridDim = dim3((unsigned)nb, (unsigned)per_row); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0;
        okl = cuda_ok(cudaLaunchKernelEx(&lc, c->sb_pairs, (const tl::KArgs)a, nb));
    } else {
        lc.gridDim = dim3((unsigned)nb, (unsigned)slabs); lc.blockDim = dim3(256); lc.dynamicSmemBytes = c->sb_trace_smem;
        okl = cuda_ok(cudaLaunchKernelEx(&lc, c->sb_trace, (const tl::KArgs)a, nb));
    }
    if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
    lc.gridDim = dim3((unsigned)nb, (unsigned)(bands * (xseg ? xseg : 1))); lc.blockDim = dim3((unsigned)c->threads); lc.dynamicSmemBytes = conv_smem;
    okl = okl && cuda_ok(cudaLaunchKernelEx(&lc, tl::conv_small_kernel, (const tl::KArgs)a, nb, band_pairs, xseg, cblk));
    const int rc = (okl && cuda_ok(cudaGetLastError())) ? TL_OK : TL_ECUDA;
    pool_free(c, blob, st);
    return rc;
}

// The double-precision path (tl_dp.cuh) over rows [0, B) of `params`, or -- with row_index /
// n_rows_dev -- over the rows listed in device memory (AUTO mode: the count is not known on the
// host, so every chunk is launched and the kernels of an empty chunk return at once).
int run_dp(tl_ctx *c, const float *params, int64_t B, float *logL, float *images, cudaStream_t st,
           const int *row_index, const int *n_rows_dev, int lin = 0, float *amps = nullptr)
{
    const int64_t rows_per_lens = B / c->cfg.n_lens;
    const int NCL = lin ? c->n_comp : 1;                         // component images kept apart (linear mode)
    int64_t chunk = c->dp_chunk_rows / (lin ? 2 * NCL : 1);
    if (chunk < 1) chunk = 1;
    if (chunk > B) chunk = B;
    tl::RowD *rows = nullptr;
    double *ext = nullptr, *partial = nullptr, *m64 = nullptr;
    const size_t ext_row = sizeof(double) * (size_t)NCL * c->He * c->dp_Wp;
    const size_t m_row = sizeof(double) * (size_t)NCL * c->cfg.ny * c->cfg.nx;
    if (!pool_alloc(c, &rows, sizeof(tl::RowD) * (size_t)chunk, st)) return TL_ENOMEM;
    if (!pool_alloc(c, &ext, ext_row * (size_t)chunk, st) ||
        !pool_alloc(c, &partial, sizeof(double) * (size_t)chunk * c->dp_n_bands, st) ||
        (lin && !pool_alloc(c, &m64, m_row * (size_t)chunk, st))) {
        pool_free(c, rows, st);
        if (ext) pool_free(c, ext, st);
        if (partial) pool_free(c, partial, st);
        return TL_ENOMEM;
    }
    // the pitch padding (Wp - We <= 1 column) is read by discarded strip lanes only, but must be finite
    if (c->dp_Wp != c->We) cudaMemsetAsync(ext, 0, ext_row * (size_t)chunk, st);
    int rc = TL_OK;
    for (int64_t r0 = 0; r0 < B && rc == TL_OK; r0 += chunk) {
        const int64_t nb = (B - r0 < chunk) ? (B - r0) : chunk;
        tl::DpArgs a;
        memset(&a, 0, sizeof(a));
        a.params = params; a.rows = rows; a.row_index = row_index; a.n_rows_dev = n_rows_dev;
        a.n_rows = (int)nb; a.list_offset = row_index ? (int)r0 : 0;
        a.row0 = r0; a.rows_per_lens = rows_per_lens;
        a.psf = c->psf; a.data = c->data; a.wgt64 = c->wgt64; a.lconst = c->lconst;
        a.ext = ext; a.partial = logL ? partial : nullptr; a.logL = logL; a.images = images;
        a.lin = lin; a.m64 = m64; a.amps = amps;
        a.P = c->P; a.ny = c->cfg.ny; a.nx = c->cfg.nx; a.K = c->K; a.Kp = c->Kp; a.h = c->h;
        a.He = c->He; a.We = c->We; a.Wp = c->dp_Wp; a.S = c->cfg.supersample;
        a.n_lens_light = c->cfg.n_lens_light; a.n_comp = c->n_comp;
        a.edge_zero = c->cfg.edge_mode == TL_EDGE_ZERO; a.mass_model = c->cfg.mass_model; a.lens_np = c->lens_np;
        a.band_rows = c->dp_band_rows; a.n_bands = c->dp_n_bands;
        a.CW = c->CW; a.CH = c->CH; a.tiles_x = (c->We + c->CW - 1) / c->CW; a.tiles_y = (c->He + c->CH - 1) / c->CH;
        a.u = c->cfg.pix_scale / (2.0 * c->cfg.supersample);
        tl::prologue_dp_kernel<<<(unsigned)((nb + 63) / 64), 64, 0, st>>>(a);
        // one warp per (row, tile): no more CTAs than there is work for
        const int64_t items = nb * a.tiles_x * a.tiles_y;
        int grid = c->dp_trace_grid;
        if ((int64_t)grid * 8 > items) grid = (int)((items + 7) / 8);
        if (c->profile) cudaEventRecord(c->ev0, st);
        c->dp_trace<<<grid, 256, 0, st>>>(a);
        if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
        tl::conv_dp_kernel<<<dim3((unsigned)nb, (unsigned)c->dp_n_bands, (unsigned)NCL), c->dp_conv_threads, c->dp_conv_smem, st>>>(a);
        if (lin) tl::solve_dp_kernel<<<(unsigned)nb, 256, 0, st>>>(a);
        else if (logL) tl::finalize_dp_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(a);
        if (!cuda_ok(cudaGetLastError())) rc = TL_ECUDA;
    }
    pool_free(c, rows, st); pool_free(c, ext, st); pool_free(c, partial, st);
    if (m64) pool_free(c, m64, st);
    return rc;
}

int run_batch(tl_ctx *c, const float *params, int64_t B, float *logL, float *images, cudaStream_t st)
{
    if (!c || B < 0) return TL_EINVAL;
    if (c->cfg.n_lens_light > 1) return TL_EINVAL;               // several lens-light blocks: MGE sets only
    if (B == 0) return TL_OK;
    if (!params || (!logL && !images)) return TL_EINVAL;
    if (B % c->cfg.n_lens) return TL_EINVAL;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;

    const int64_t rows_per_lens = B / c->cfg.n_lens;
    if (c->precision == TL_PRECISION_FP64) return run_dp(c, params, B, logL, images, st, nullptr, nullptr);
    if (c->precision == TL_PRECISION_FP64_LIBM) {
        const size_t ext_row = sizeof(double) * (size_t)c->He * c->We;
        int64_t pch = (int64_t)(EXT_SCRATCH_BYTES / ext_row);
        if (pch < 1) pch = 1;
        if (pch > 65535) pch = 65535;
        if (pch > B) pch = B;
        double *pext = nullptr;
        if (!pool_alloc(c, &pext, ext_row * (size_t)pch, st)) return TL_ENOMEM;
        int prc = TL_OK;
        for (int64_t r0 = 0; r0 < B && prc == TL_OK; r0 += pch) {
            const int64_t nb = (B - r0 < pch) ? (B - r0) : pch;
            tl::PreciseArgs pa;
            pa.params = params + r0 * c->P; pa.psf = c->psf; pa.data = c->data; pa.noise = c->noise;
            pa.lconst = c->lconst; pa.ext = pext; pa.logL = logL; pa.images = images;
            pa.row0 = r0; pa.rows_per_lens = rows_per_lens;
            pa.P = c->P; pa.ny = c->cfg.ny; pa.nx = c->cfg.nx; pa.K = c->K; pa.Kp = c->Kp; pa.h = c->h;
            pa.He = c->He; pa.We = c->We; pa.S = c->cfg.supersample;
            pa.n_lens_light = c->cfg.n_lens_light; pa.n_comp = c->n_comp;
            pa.edge_zero = c->cfg.edge_mode == TL_EDGE_ZERO; pa.pix_scale = c->cfg.pix_scale;
            pa.mass_model = c->cfg.mass_model;
            int slabs = (int)((2 * (int64_t)c->n_sm * 8 + nb - 1) / nb);          // enough CTAs for small batches
            const int max_slabs = (c->He * c->We + 255) / 256;
            if (slabs > max_slabs) slabs = max_slabs;
            if (slabs < 1) slabs = 1;
            if (c->profile) cudaEventRecord(c->ev0, st);
            tl::precise_trace_kernel<<<dim3((unsigned)nb, (unsigned)slabs), 256, 0, st>>>(pa);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
            tl::precise_conv_kernel<<<(unsigned)nb, 256, 0, st>>>(pa);
            if (!cuda_ok(cudaGetLastError())) prc = TL_ECUDA;
        }
        pool_free(c, pext, st);
        return prc;
    }
    const bool autop = c->precision == TL_PRECISION_AUTO && logL != nullptr;
    // AUTO on the split path (large images): the conv tiles do not carry the error sums, so every row
    // is evaluated in FP64; AUTO renders are FP32 renders (the image has no 1e-8 requirement)
    if (autop && c->path == 1) return run_dp(c, params, B, logL, images, st, nullptr, nullptr);
    // AUTO with a few rows: the FP32 pass would give each row to one CTA (a whole row-time of one SM), the FP64 path
    // spreads a row over the GPU and is the faster of the two up to half the SM count of rows (71 against 166 us for one
    // row of configs[1]) -- and meets the tolerance on every row by construction
    if (autop && B <= c->n_sm / 2) return run_dp(c, params, B, logL, nullptr, st, nullptr, nullptr);
    if (c->path == 0 && B <= c->sb_max_rows && !autop) return run_small_batch(c, params, B, logL, images, st);
    int *flags = nullptr;                            // [0] = count, [1 .. B] = flagged rows
    if (autop) {
        if (B > 0x7ffffff0) return TL_ESIZE;
        if (!pool_alloc(c, &flags, sizeof(int) * (size_t)(B + 1), st)) return TL_ENOMEM;
        cudaMemsetAsync(flags, 0, sizeof(int), st);
    }
    // fused path, one chunk: the persistent grid takes the rows in waves of `grid`; the rows of a last, mostly empty wave
    // (up to half the SM count of them) cost a whole row-time all the same -- they go through the small-batch path
    // instead, which spreads them over the GPU and returns the same bits (B = 300 on configs[1]: 0.41 -> 0.31 ms)
    int64_t B_tail = 0;
    if (c->path == 0 && !autop && c->sb_max_rows > 0 && B <= c->chunk_rows && B > c->grid) {
        const int64_t rem = B % c->grid;
        if (rem > 0 && rem <= c->sb_max_rows) B_tail = rem;
    }
    const int64_t B_all = B;
    B -= B_tail;
    const int64_t chunk = c->chunk_rows < B ? c->chunk_rows : B;
    tl::RowC *rows = nullptr;
    float *ext = nullptr;
    double *partial = nullptr;
    // (split path: + one tile-queue head per row for the ray-trace kernel)
    if (!pool_alloc(c, &rows, (sizeof(tl::RowC) + (c->path == 1 ? sizeof(int) : 0)) * (size_t)chunk, st)) return TL_ENOMEM;
    if (c->path == 1) {
        const size_t ext_bytes = sizeof(float) * (size_t)chunk * c->He * c->pitch;
        if (!pool_alloc(c, &ext, ext_bytes, st) ||
            !pool_alloc(c, &partial, sizeof(double) * (size_t)chunk * c->n_tiles, st)) {
            pool_free(c, rows, st);
            if (ext) pool_free(c, ext, st);
            return TL_ENOMEM;
        }
        cudaMemsetAsync(ext, 0, ext_bytes, st);      // pitch padding must read as finite zeros
    }

    int rc = TL_OK;
    for (int64_t r0 = 0; r0 < B && rc == TL_OK; r0 += chunk) {
        const int64_t nb = (B - r0 < chunk) ? (B - r0) : chunk;
        tl::PrologueArgs pa;
        fill_prologue_args(c, pa, params, rows, nb, r0, rows_per_lens, 0);
        tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);

        tl::KArgs a = base_args(c);
        a.rows = rows; a.B = nb; a.rows_per_lens = rows_per_lens; a.row0 = r0;
        a.logL = logL; a.images = images;
        if (autop) {
            a.flag_count = flags; a.flag_list = flags + 1;
            // the FP32 error model of DESIGN.md 6: coherent 2^-22, random 5 sigma of 2^-21 / S + 2^-22 per pixel
            a.err_coh = 2.384185791015625e-07f;
            a.err_rnd = (float)(5.0 * (4.76837158203125e-07 / c->cfg.supersample + 2.384185791015625e-07));
        }
        if (c->path == 0) {
            int grid = c->grid;
            if ((int64_t)grid > nb) grid = (int)nb;
            if (c->profile) cudaEventRecord(c->ev0, st);
            c->fused<<<grid, c->threads, c->smem, st>>>(a);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
        } else {
            a.ext = ext; a.partial = logL ? partial : nullptr;
            // the row's CTAs draw warp tiles from one queue: the tiles next to a source centre, full of FP64-refined
            // samples, cost several times an ordinary one, and a static split leaves their CTA's other warps idle
            if (nb <= 65535) {
                a.tile_counters = reinterpret_cast<int *>(rows + chunk);
                cudaMemsetAsync(a.tile_counters, 0, sizeof(int) * (size_t)nb, st);
            }
            dim3 tg((unsigned)(nb < 65535 ? nb : 65535), (unsigned)c->trace_slabs);
            if (c->profile) cudaEventRecord(c->ev0, st);
            c->trace<<<tg, 256, c->trace_smem, st>>>(a, (int)nb);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
            dim3 cg((unsigned)nb, (unsigned)c->n_tiles);
            tl::conv_kernel<<<cg, 256, c->conv_smem, st>>>(a, (int)nb);
            if (logL) tl::finalize_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(a, (int)nb);
        }
        if (!cuda_ok(cudaGetLastError())) rc = TL_ECUDA;
    }
    pool_free(c, rows, st);
    if (ext) pool_free(c, ext, st);
    if (partial) pool_free(c, partial, st);
    if (B_tail && rc == TL_OK) rc = run_small_batch(c, params, B_tail, logL, images, st, B, rows_per_lens);
    B = B_all;
    if (autop) {
        if (rc == TL_OK) rc = run_dp(c, params, B, logL, nullptr, st, flags + 1, flags);
        pool_free(c, flags, st);
    }
    return rc;
}

}  // namespace

// ------------------------------------------------------------------ serve mode (tl_serve.cuh)
namespace {

// launch geometry of a B-row request on `grid` resident CTAs: run_small_batch's, with the CTAs of the persistent grid
void serve_geometry(const tl_ctx *c, int B, int grid, int *per_row, int *bands_out, int *band_pairs_out, int *xseg_out, size_t *conv_smem)
{
    const int npair = (c->cfg.ny + 1) / 2, nsx = (c->cfg.nx + 3) / 4;
    int want = grid / B;
    if (want < 1) want = 1;
    const int S = c->cfg.supersample, ppw = 32 / (S * S / 2), wpc = c->threads / 32;
    const int n_wt = (c->He * c->We + ppw - 1) / ppw;
    *per_row = want < (n_wt + wpc - 1) / wpc ? want : (n_wt + wpc - 1) / wpc;
    int bands = want < npair ? want : npair;
    const size_t fixed = sizeof(float) * ((size_t)c->K * c->Kp + c->pitch + c->Kp + 8);
    int band_pairs = (npair + bands - 1) / bands;
    const int max_pairs = (int)(((SMEM_LIMIT - 4096 - fixed) / (sizeof(float) * c->pitch) - (c->K - 1)) / 2);
    if (band_pairs > max_pairs) band_pairs = max_pairs;
    bands = (npair + band_pairs - 1) / band_pairs;
    const int per_pass = c->threads / c->K;
    int xseg = want / bands;
    const int one_pass = (band_pairs * nsx + per_pass - 1) / per_pass;
    if (xseg > one_pass) xseg = one_pass;
    if (xseg > nsx) xseg = nsx;
    if (xseg < 1) xseg = 1;
    if ((band_pairs * ((nsx + xseg - 1) / xseg) + per_pass - 1) / per_pass > 2) xseg = 0;
    *bands_out = bands; *band_pairs_out = band_pairs; *xseg_out = xseg;
    *conv_smem = fixed + sizeof(float) * ((size_t)(2 * band_pairs + c->K - 1) * c->pitch + (xseg ? (size_t)per_pass * c->K * 8 : 0));
}

void serve_free(tl_ctx *c)
{
    tl_ctx::Serve &v = c->sv;
    if (v.stream) cudaStreamDestroy(v.stream);
    if (v.ctl) cudaFreeHost(v.ctl);
    cudaFree(v.dev); cudaFree(v.rows); cudaFree(v.ext); cudaFree(v.cblk); cudaFree(v.params); cudaFree(v.counters);
    v = tl_ctx::Serve();
}

// (re)start the persistent kernel; it takes up where the last one left (requests up to ctl->done are served)
bool serve_launch(tl_ctx *c)
{
    tl_ctx::Serve &v = c->sv;
    if (!cuda_ok(cudaStreamSynchronize(v.stream))) return false;               // the previous kernel, if any, has left
    tl::ServeDev d0;
    memset(&d0, 0, sizeof(d0));
    d0.seq = v.ctl->done; d0.start = v.ctl->done;
    if (!cuda_ok(cudaMemcpyAsync(v.dev, &d0, sizeof(d0), cudaMemcpyHostToDevice, v.stream))) return false;
    if (!cuda_ok(cudaStreamSynchronize(v.stream))) return false;               // (d0 is on the stack)
    tl::KArgs a = base_args(c);
    a.rows = v.rows; a.B = tl::SERVE_MAX_ROWS; a.rows_per_lens = (int64_t)1 << 40; a.row0 = 0;
    a.logL = v.ctl_dev->logL; a.ext = v.ext; a.rowtab = 0; a.tile_counters = v.counters;
    tl::PrologueArgs pa;
    fill_prologue_args(c, pa, v.params, v.rows, tl::SERVE_MAX_ROWS, 0, (int64_t)1 << 40, 0);
    v.ctl->alive = 1; v.ctl->error = 0;
    v.fn<<<v.grid, c->threads, v.smem, v.stream>>>(a, pa, v.ctl_dev, v.dev, v.cblk, v.idle_ns, (unsigned long long)120e9);   // (lifetime: 120 s, then restarted on demand)
    return cuda_ok(cudaGetLastError());
}

}  // namespace

extern "C" {

int tl_debug_canary_errors(tl_ctx *c, int64_t *count)
{
    if (!c || !count) return TL_EINVAL;
    *count = 0;
    if (!c->canary_errors) return TL_EINVAL;                   // the context was not created with tl_options.debug_canaries
    DeviceGuard guard(c->device);
    int n = 0;
    if (!guard.ok || !cuda_ok(cudaDeviceSynchronize()) || !cuda_ok(cudaMemcpy(&n, c->canary_errors, sizeof(int), cudaMemcpyDeviceToHost))) return TL_ECUDA;
    *count = n;
    return TL_OK;
}

namespace { __global__ void canary_poke_kernel(unsigned *p) { *p = 0u; } }

int tl_debug_canary_selftest(tl_ctx *c)
{
    if (!c || !c->canary_errors) return TL_EINVAL;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    int64_t before = 0, after = 0;
    if (tl_debug_canary_errors(c, &before) != TL_OK) return TL_ECUDA;
    unsigned *buf = nullptr;
    if (!pool_alloc(c, &buf, 1000, nullptr)) return TL_ENOMEM;        // 1000 bytes: the body is rounded up to 1024
    canary_poke_kernel<<<1, 1>>>(buf + 1024 / sizeof(unsigned));      // the first guard word behind the body
    canary_poke_kernel<<<1, 1>>>(buf - 1);                            // the last guard word in front of it
    pool_free(c, buf, nullptr);
    if (tl_debug_canary_errors(c, &after) != TL_OK) return TL_ECUDA;
    if (!cuda_ok(cudaMemset(c->canary_errors, 0, sizeof(int)))) return TL_ECUDA;   // the two deliberate hits do not count
    return after - before == 2 ? TL_OK : TL_ECUDA;
}

int tl_serve_start(tl_ctx *c, int32_t max_rows, double idle_timeout_s)
{
    if (!c || max_rows < 1 || max_rows > tl::SERVE_MAX_ROWS || !(idle_timeout_s > 0.0) || idle_timeout_s > 300.0) return TL_EINVAL;
    if (c->sv.fn) return TL_EINVAL;                                             // already serving
    if (c->cfg.n_lens != 1 || c->cfg.n_lens_light > 1 || c->cfg.mass_model != TL_MASS_SIE || c->precision != TL_PRECISION_FP32) return TL_EINVAL;
    const bool kblk = c->K == 5 || c->K == 15 || c->K == 21 || c->K == 31 || c->K == 41;
    serve_fn fn = tl_serve_for(c->cfg.supersample, c->cfg.n_lens_light, c->cfg.n_source);
    if (c->path != 0 || !kblk || !fn || c->P > tl::SERVE_MAX_P) return TL_ESIZE;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    tl_ctx::Serve &v = c->sv;
    v.max_rows = max_rows; v.idle_ns = (unsigned long long)(idle_timeout_s * 1e9);
    const size_t npair = (size_t)(c->cfg.ny + 1) / 2, nsx = (size_t)(c->cfg.nx + 3) / 4, ext_row = (size_t)c->He * c->pitch;
    bool ok = cuda_ok(cudaHostAlloc(reinterpret_cast<void **>(&v.ctl), sizeof(tl::ServeCtl), cudaHostAllocMapped));
    if (ok) memset(v.ctl, 0, sizeof(tl::ServeCtl));
    ok = ok && cuda_ok(cudaHostGetDevicePointer(reinterpret_cast<void **>(&v.ctl_dev), v.ctl, 0));
    ok = ok && cuda_ok(cudaMalloc(&v.dev, sizeof(tl::ServeDev))) && cuda_ok(cudaMalloc(&v.rows, sizeof(tl::RowC) * tl::SERVE_MAX_ROWS)) &&
         cuda_ok(cudaMalloc(&v.ext, sizeof(float) * ext_row * tl::SERVE_MAX_ROWS)) &&
         cuda_ok(cudaMalloc(&v.cblk, sizeof(float) * npair * nsx * tl::SERVE_MAX_ROWS)) &&
         cuda_ok(cudaMalloc(&v.params, sizeof(float) * tl::SERVE_MAX_ROWS * tl::SERVE_MAX_P)) &&
         cuda_ok(cudaMalloc(&v.counters, sizeof(int) * 2 * tl::SERVE_MAX_ROWS)) &&
         cuda_ok(cudaMemset(v.ext, 0, sizeof(float) * ext_row * tl::SERVE_MAX_ROWS)) &&       // the pitch padding reads as zeros
         cuda_ok(cudaStreamCreateWithFlags(&v.stream, cudaStreamNonBlocking));
    if (ok) {
        // the grid: every resident slot; shared memory: the largest band any request size needs on that grid
        ok = cuda_ok(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_LIMIT - 4096)));
        int occ = 0;
        size_t smem = 0;
        for (int pass = 0; pass < 2 && ok; ++pass) {                             // the occupancy depends on the size, the size on the grid
            ok = cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, c->threads, smem)) && occ >= 1;
            v.grid = occ * c->n_sm;
            smem = 0;
            for (int B = 1; B <= max_rows && ok; ++B) {
                int pr, bd, bp, xs;
                size_t cs;
                serve_geometry(c, B, v.grid, &pr, &bd, &bp, &xs, &cs);
                if (cs > smem) smem = cs;
            }
        }
        v.smem = smem;
        ok = ok && cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, c->threads, smem)) && occ * c->n_sm >= v.grid;
    }
    if (ok) { v.fn = fn; ok = serve_launch(c); }
    if (!ok) { cudaGetLastError(); serve_free(c); return TL_ECUDA; }
    return TL_OK;
}

int tl_serve_eval(tl_ctx *c, const float *params_host, int32_t B, float *logL_host)
{
    if (!c || !c->sv.fn || !params_host || !logL_host || B < 1 || B > c->sv.max_rows) return TL_EINVAL;
    tl_ctx::Serve &v = c->sv;
    tl::ServeCtl *ctl = v.ctl;
    int pr, bd, bp, xs;
    size_t cs;
    serve_geometry(c, B, v.grid, &pr, &bd, &bp, &xs, &cs);
    ctl->B = B; ctl->per_row = pr; ctl->bands = bd; ctl->band_pairs = bp; ctl->xseg = xs;
    memcpy(ctl->params, params_host, sizeof(float) * (size_t)B * c->P);
    const unsigned long long n = ++v.seq;
    __atomic_store_n(&ctl->seq, n, __ATOMIC_RELEASE);
    struct timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    for (unsigned spin = 0;; ++spin) {
        if (__atomic_load_n(&ctl->done, __ATOMIC_ACQUIRE) == n) break;
        if ((spin & 1023) == 1023) {
            if (__atomic_load_n(&ctl->alive, __ATOMIC_ACQUIRE) == 0 && __atomic_load_n(&ctl->done, __ATOMIC_ACQUIRE) != n) {
                // the kernel left (idle or lifetime limit) before it saw this request: start it again
                DeviceGuard guard(c->device);
                if (!guard.ok || ctl->error || !serve_launch(c)) return TL_ECUDA;
            }
            clock_gettime(CLOCK_MONOTONIC, &t1);
            if ((t1.tv_sec - t0.tv_sec) + 1e-9 * (t1.tv_nsec - t0.tv_nsec) > 20.0) return TL_ECUDA;
        }
    }
    memcpy(logL_host, const_cast<const float *>(ctl->logL), sizeof(float) * (size_t)B);
    return TL_OK;
}

int tl_serve_stop(tl_ctx *c)
{
    if (!c) return TL_EINVAL;
    if (!c->sv.fn) return TL_OK;
    DeviceGuard guard(c->device);
    __atomic_store_n(&c->sv.ctl->seq, tl::SERVE_EXIT, __ATOMIC_RELEASE);
    const bool ok = guard.ok && cuda_ok(cudaStreamSynchronize(c->sv.stream));
    serve_free(c);
    return ok ? TL_OK : TL_ECUDA;
}

}  // extern "C"

// ------------------------------------------------------------------ tl_loglike_batch_noalloc
// The per-row constants of tl_loglike_batch's fused path (RowC[B], written by prologue_kernel, read by
// fused_kernel) in a fixed array of the device image instead of pool memory: see include/tinylens.h.
// Every device that loads the library holds the array (5 MiB) until the process exits; every call on
// a device shares it.
static __device__ __align__(256) unsigned char tl_noalloc_scratch[(size_t)TL_NOALLOC_MAX_ROWS * sizeof(tl::RowC)];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
void *g_noalloc_addr[NOALLOC_MAX_DEVICES];          // device address of the array on device d; null = not resolved yet

// In host code `tl_noalloc_scratch` is a host-side stand-in for the symbol, not a device address: a
// kernel handed &tl_noalloc_scratch faults (or scribbles over host memory where the GPU can reach it).
// The address on `device` -- which must be current -- comes from cudaGetSymbolAddress, once per device.
bool noalloc_rows(int device, tl::RowC **out)
{
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return false;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_addr[device]) {
        void *p = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress(&p, tl_noalloc_scratch)) || !p) return false;
        g_noalloc_addr[device] = p;
    }
    *out = static_cast<tl::RowC *>(g_noalloc_addr[device]);
    return true;
}

}  // namespace

extern "C" {

int tl_loglike_batch_noalloc(tl_ctx *c, const float *params, int64_t B, float *logL, void *cuda_stream)
{
    if (!c || B < 0) return TL_EINVAL;
    if (B > TL_NOALLOC_MAX_ROWS) return TL_ESIZE;                 // the array holds TL_NOALLOC_MAX_ROWS rows
    if (c->path != 0) return TL_ESIZE;                            // split path: needs an image per row in global memory
    if (c->precision != TL_PRECISION_FP32 || c->cfg.n_lens_light > 1) return TL_EINVAL;
    if (B > 0 && (!params || !logL)) return TL_EINVAL;
    if (B % c->cfg.n_lens) return TL_EINVAL;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    tl::RowC *rows = nullptr;
    if (!noalloc_rows(c->device, &rows)) return TL_ECUDA;
    if (B == 0) return TL_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // one chunk: the two launches of run_batch's fused path, `rows` being the fixed array
    tl::PrologueArgs pa;
    fill_prologue_args(c, pa, params, rows, B, 0, B / c->cfg.n_lens, 0);
    tl::prologue_kernel<<<tl::prologue_blocks(B), 128, 0, st>>>(pa);
    tl::KArgs a = base_args(c);
    a.rows = rows; a.B = B; a.rows_per_lens = B / c->cfg.n_lens; a.row0 = 0;
    a.logL = logL; a.images = nullptr;
    int grid = c->grid;
    if ((int64_t)grid > B) grid = (int)B;
    c->fused<<<grid, c->threads, c->smem, st>>>(a);
    return cuda_ok(cudaGetLastError()) ? TL_OK : TL_ECUDA;
}

}  // extern "C"

extern "C" {

const char *tl_version(void) { return TL_VERSION_STRING; }

const char *tl_strerror(int code)
{
    switch (code) {
    case TL_OK: return "success";
    case TL_EINVAL: return "invalid argument (shape, even PSF size, null pointer, or noise not finite and positive)";
    case TL_ENOMEM: return "out of host or device memory";
    case TL_ECUDA: return "no usable CUDA device or a CUDA runtime call failed (there is no CPU fallback)";
    case TL_ESIZE: return "configuration exceeds what the kernels support";
    default: return "unknown tinylens error code";
    }
}

int tl_create(tl_ctx **out, const tl_config *cfg, const float *psf, int32_t psf_ny, int32_t psf_nx,
              const float *data, const float *noise, void *cuda_stream)
{
    return tl_create_ex(out, cfg, psf, psf_ny, psf_nx, data, noise, nullptr, cuda_stream);
}

int tl_create_ex(tl_ctx **out, const tl_config *cfg, const float *psf_in, int32_t psf_ny, int32_t psf_nx,
                 const float *data_in, const float *noise_in, const tl_options *opt, void *cuda_stream)
{
    if (out) *out = nullptr;
    if (!out || !cfg || !psf_in || !data_in || !noise_in) return TL_EINVAL;
    if (opt) {
        if (opt->small_batch_rows < -1 || opt->mge_chunk_rows < 0 || opt->scratch_keep_bytes < 0) return TL_EINVAL;
        if (opt->block_threads && (opt->block_threads < 32 || opt->block_threads > 512 || opt->block_threads % 32)) return TL_EINVAL;
        if (opt->refine_tau < 0.0 || !std::isfinite(opt->refine_tau)) return TL_EINVAL;
        if (opt->debug_canaries < 0 || opt->debug_canaries > 1 || opt->reserved != 0) return TL_EINVAL;
    }
    if (cfg->ny < 1 || cfg->nx < 1 || !(cfg->pix_scale > 0.0) || !std::isfinite(cfg->pix_scale)) return TL_EINVAL;
    if (cfg->supersample < 1 || cfg->supersample > 16) return TL_EINVAL;
    // n_lens_light = 2: two MGE sets with their own shapes; such a context serves tl_loglike_mge_batch only
    if (cfg->n_lens_light < 0 || cfg->n_lens_light > tl::MGE_MAX_SETS || cfg->n_source < 1 || cfg->n_source > 2) return TL_EINVAL;
    if (cfg->edge_mode != TL_EDGE_EXTEND && cfg->edge_mode != TL_EDGE_ZERO) return TL_EINVAL;
    if (cfg->n_lens < 1) return TL_EINVAL;
    if (cfg->mass_model != TL_MASS_SIE && cfg->mass_model != TL_MASS_EPL) return TL_EINVAL;
    if (psf_ny != psf_nx || psf_ny < 1 || (psf_ny & 1) == 0) return TL_EINVAL;
    // exact sub-sample coordinates need 2 S (n + K) < 2^24
    if ((int64_t)2 * cfg->supersample * ((int64_t)(cfg->ny > cfg->nx ? cfg->ny : cfg->nx) + psf_ny) >= (1 << 24)) return TL_ESIZE;

    const size_t npix = (size_t)cfg->ny * cfg->nx, L = (size_t)cfg->n_lens;
    // psf / data / noise may be host or device pointers (SURVEY.md 8(b) "Ownership"); the
    // preparation below runs on the host, so device arrays are staged into host copies first
    std::vector<float> stage_psf, stage_data, stage_noise;
    auto host_view = [](const float *p, size_t n, std::vector<float> &stage, int *err) -> const float * {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return p; }   // no driver: plain host memory
        if (at.type != cudaMemoryTypeDevice) return p;             // unregistered / pinned host, or managed
        stage.resize(n);
        if (cudaMemcpy(stage.data(), p, n * sizeof(float), cudaMemcpyDeviceToHost) != cudaSuccess) *err = TL_ECUDA;
        return stage.data();
    };
    int herr = TL_OK;
    const float *psf = host_view(psf_in, L * (size_t)psf_ny * psf_nx, stage_psf, &herr);
    const float *data = host_view(data_in, npix * L, stage_data, &herr);
    const float *noise = host_view(noise_in, npix * L, stage_noise, &herr);
    if (herr != TL_OK) return herr;
    for (size_t i = 0; i < npix * L; ++i)
        if (!(noise[i] > 0.f) || !std::isfinite(noise[i])) return TL_EINVAL;

    int ndev = 0;
    if (!cuda_ok(cudaGetDeviceCount(&ndev)) || ndev < 1) return TL_ECUDA;

    tl_ctx *c = new (std::nothrow) tl_ctx;
    if (!c) return TL_ENOMEM;
    c->cfg = *cfg;
    memset(&c->opt, 0, sizeof(c->opt));
    c->opt.small_batch_rows = -1;
    if (opt) c->opt = *opt;
    if (!cuda_ok(cudaGetDevice(&c->device))) { delete c; return TL_ECUDA; }
    cudaDeviceProp prop;
    if (!cuda_ok(cudaGetDeviceProperties(&prop, c->device))) { delete c; return TL_ECUDA; }
    c->n_sm = prop.multiProcessorCount;
    {   // per-call scratch comes from a stream-ordered pool owned by the context (the device's
        // default pool, which other libraries share, is left alone): freed blocks stay cached in it
        // across synchronisations up to `scratch_keep_bytes` and are returned by tl_destroy
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = c->device;
        if (cuda_ok(cudaMemPoolCreate(&c->pool, &props))) {
            unsigned long long keep = c->opt.scratch_keep_bytes > 0 ? (unsigned long long)c->opt.scratch_keep_bytes : (2ull << 30);
            cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &keep);
        } else c->pool = nullptr;                     // falls back to the default pool (untouched)
        cudaGetLastError();
    }
    if (c->opt.debug_canaries) {
        if (!cuda_ok(cudaMalloc(&c->canary_errors, sizeof(int))) || !cuda_ok(cudaMemset(c->canary_errors, 0, sizeof(int)))) { tl_destroy(c); return TL_ECUDA; }
    }
    c->n_comp = cfg->n_lens_light + cfg->n_source;
    c->lens_np = 7 + (cfg->mass_model == TL_MASS_EPL ? 1 : 0);
    c->P = c->lens_np + 7 * c->n_comp;
    c->K = psf_ny; c->Kp = (c->K + 3) & ~3; c->h = (c->K - 1) / 2;
    c->He = cfg->ny + 2 * c->h; c->We = cfg->nx + 2 * c->h;
    c->pitch = (c->We + 3) & ~3;

    // host-side preparation in FP64: flipped + padded PSF, inverse variance, Eq. 5 constant
    std::vector<float> psf_f((size_t)L * c->K * c->Kp, 0.f), wgt(npix * L), smin(L);
    std::vector<double> lconst(L), wgt64(npix * L);
    for (size_t l = 0; l < L; ++l) {
        // true convolution (Eq. 3, G11) == correlation with the flipped kernel
        for (int a = 0; a < c->K; ++a)
            for (int b = 0; b < c->K; ++b)
                psf_f[(l * c->K + a) * c->Kp + b] = psf[(l * c->K + (c->K - 1 - a)) * c->K + (c->K - 1 - b)];
        double s = 0.0, comp = 0.0, mn = INFINITY;
        for (size_t i = 0; i < npix; ++i) {
            const double sg = noise[l * npix + i];
            wgt64[l * npix + i] = 1.0 / (sg * sg);
            wgt[l * npix + i] = (float)wgt64[l * npix + i];
            const double t = std::log(2.0 * M_PI * sg * sg) - comp, u = s + t;   // Kahan
            comp = (u - s) - t; s = u;
            if (sg < mn) mn = sg;
        }
        lconst[l] = s; smin[l] = (float)mn;
    }
    c->lconst0 = lconst[0]; c->sigma_min0 = smin[0];
    c->refine_tau *= cfg->supersample;
    if (c->opt.refine_tau > 0.0 && std::isfinite(c->opt.refine_tau)) c->refine_tau = c->opt.refine_tau;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    bool ok = cuda_ok(cudaMalloc(&c->psf, psf_f.size() * sizeof(float))) &&
              cuda_ok(cudaMalloc(&c->data, npix * L * sizeof(float))) &&
              cuda_ok(cudaMalloc(&c->wgt, npix * L * sizeof(float))) &&
              cuda_ok(cudaMalloc(&c->wgt64, npix * L * sizeof(double))) &&
              cuda_ok(cudaMalloc(&c->noise, npix * L * sizeof(float))) &&
              cuda_ok(cudaMalloc(&c->sigma_min, L * sizeof(float))) &&
              cuda_ok(cudaMalloc(&c->lconst, L * sizeof(double)));
    if (!ok) { tl_destroy(c); return TL_ENOMEM; }
    ok = cuda_ok(cudaMemcpyAsync(c->psf, psf_f.data(), psf_f.size() * sizeof(float), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->data, data, npix * L * sizeof(float), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->wgt, wgt.data(), npix * L * sizeof(float), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->wgt64, wgt64.data(), npix * L * sizeof(double), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->noise, noise, npix * L * sizeof(float), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->sigma_min, smin.data(), L * sizeof(float), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaMemcpyAsync(c->lconst, lconst.data(), L * sizeof(double), cudaMemcpyHostToDevice, st)) &&
         cuda_ok(cudaStreamSynchronize(st));
    if (!ok) { tl_destroy(c); return TL_ECUDA; }

    // launch geometry
    best_warp_tile(c->He, c->We, &c->CW, &c->CH);
    size_t fs = fused_smem_bytes(c);
    const size_t rowtab_bytes = sizeof(tl::RowV) * (size_t)c->He * cfg->supersample;
    if (fs <= SMEM_LIMIT && !c->opt.force_split) {
        // the row-value table is worth its shared memory unless it costs a resident CTA
        const size_t fs2 = ((fs + 15) & ~(size_t)15) + rowtab_bytes;
        const int per_sm_1 = (int)(SMEM_LIMIT / (fs + 1024)), per_sm_2 = (int)(SMEM_LIMIT / (fs2 + 1024));
        if (fs2 <= SMEM_LIMIT && (per_sm_2 >= per_sm_1 || per_sm_2 >= 2)) { c->rowtab = 1; fs = fs2; }
        c->path = 0; c->smem = fs;
        // one CTA of 16 warps per SM when the image has enough warp tiles to keep them busy
        // (measured +3 % on configs[1] and lower small-batch latency), else two CTAs of 8 warps
        const int n_tiles_img = ((c->We + c->CW - 1) / c->CW) * ((c->He + c->CH - 1) / c->CH);
        c->threads = (fs > SMEM_LIMIT / 2 || n_tiles_img >= 300) ? 512 : 256;
        if (c->opt.block_threads) c->threads = c->opt.block_threads;
        c->fused = cfg->mass_model == TL_MASS_EPL ? tl_fused_epl_for(cfg->supersample, cfg->n_lens_light, cfg->n_source)
                                                  : tl_fused_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
        // small rows (256-thread CTAs), S = 2, PSF up to 21 x 21: the variant that fits three CTAs per SM
        if (c->threads == 256 && c->K <= 21 && cfg->mass_model != TL_MASS_EPL && 3 * (fs + 1024) <= SMEM_LIMIT) {
            fused_fn small = tl_fused_small_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
            if (small) c->fused = small;
        }
        if (!cuda_ok(cudaFuncSetAttribute(c->fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT))) { tl_destroy(c); return TL_ECUDA; }
        int occ = 0;
        if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->fused, c->threads, fs)) || occ < 1) { tl_destroy(c); return TL_ECUDA; }
        c->ctas_per_sm = occ; c->grid = occ * c->n_sm;
        c->chunk_rows = CONST_CHUNK;
        // small-batch path: needs a register-blocked PSF size and the whole image + taps in one CTA's shared memory
        const bool kblk = c->K == 5 || c->K == 15 || c->K == 21 || c->K == 31 || c->K == 41;
        // ... and a row long enough for three more launches to pay (measured: configs 1-3 gain, Tiny loses)
        const int64_t samples_row = (int64_t)c->He * c->We * cfg->supersample * cfg->supersample;
        if (kblk && (samples_row >= 16384 || c->opt.small_batch_rows > 0) && c->opt.small_batch_rows != 0) {
            c->sb_trace = cfg->mass_model == TL_MASS_EPL ? tl_trace_epl_for(cfg->supersample, cfg->n_lens_light, cfg->n_source)
                                                         : tl_trace_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
            bool oks = cuda_ok(cudaFuncSetAttribute(tl::conv_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_LIMIT - 1024)));   // 1 KB: its static shared memory
            if (rowtab_bytes <= 96 * 1024) {
                c->sb_rowtab = 1; c->sb_trace_smem = rowtab_bytes;
                oks = oks && cuda_ok(cudaFuncSetAttribute(c->sb_trace, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rowtab_bytes));
            }
            c->sb_max_rows = oks ? c->n_sm / 2 : 0;
            if (c->opt.small_batch_rows > 0) c->sb_max_rows = oks ? c->opt.small_batch_rows : 0;
            if (cfg->mass_model != TL_MASS_EPL) {
                c->sb_pairs = tl_trace_pairs_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
                c->sb_pairs_rows = 16;             // measured on configs[1]: faster than trace_kernel up to ~20 rows
            }
            cudaGetLastError();
        }
    } else {
        c->path = 1;
        // tile rows: as many as fit in ~100 KB so two CTAs share an SM
        int tr = (int)((100 * 1024 / sizeof(float) - (size_t)c->K * c->Kp - c->Kp - 8) / c->pitch) - 2 * c->h - 1;
        if (tr < 4) tr = (int)((SMEM_LIMIT / sizeof(float) - 64 - (size_t)c->K * c->Kp - c->Kp - 8) / c->pitch) - 2 * c->h - 1;
        if (tr < 1) { tl_destroy(c); return TL_ESIZE; }
        if (tr > cfg->ny) tr = cfg->ny;
        c->tile_rows = tr; c->n_tiles = (cfg->ny + tr - 1) / tr;
        c->conv_smem = conv_smem_bytes(c, tr);
        if (!cuda_ok(cudaFuncSetAttribute(tl::conv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT))) { tl_destroy(c); return TL_ECUDA; }
        c->threads = 256; c->smem = c->conv_smem;
        c->trace = cfg->mass_model == TL_MASS_EPL ? tl_trace_epl_for(cfg->supersample, cfg->n_lens_light, cfg->n_source)
                                                  : tl_trace_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
        if (rowtab_bytes <= 48 * 1024 && cfg->supersample <= 4) {   // S = 8 amortises row values over 8 samples already
            c->rowtab = 1; c->trace_smem = rowtab_bytes;
            if (!cuda_ok(cudaFuncSetAttribute(c->trace, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rowtab_bytes))) { tl_destroy(c); return TL_ECUDA; }
        }
        // one CTA slab = 256 columns-items; G row groups so that a row of the batch fills >= 8 CTAs
        c->trace_slabs = 8;
        int occ = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->trace, 256, c->trace_smem);
        c->ctas_per_sm = occ > 0 ? occ : 1; c->grid = 0;
        int64_t cr = (int64_t)(EXT_SCRATCH_BYTES / (sizeof(float) * (size_t)c->He * c->pitch));
        if (cr < 1) cr = 1;
        if (cr > 65535) cr = 65535;
        c->chunk_rows = cr;
    }
    {   // linear-amplitude pipeline: conv tiles of ~100 KB, row-value table when small
        int tr = (int)((100 * 1024 / sizeof(float) - (size_t)c->K * c->Kp - c->Kp - 8) / c->pitch) - 2 * c->h - 1;
        if (tr < 4) tr = (int)((SMEM_LIMIT / sizeof(float) - 64 - (size_t)c->K * c->Kp - c->Kp - 8) / c->pitch) - 2 * c->h - 1;
        if (tr >= 1) {
            if (tr > cfg->ny) tr = cfg->ny;
            c->lin_tile_rows = tr; c->lin_n_tiles = (cfg->ny + tr - 1) / tr;
            c->lin_conv_smem = sizeof(float) * ((size_t)c->K * c->Kp + (size_t)(tr + 2 * c->h + 1) * c->pitch + c->Kp + 8);
            c->trace_lin = cfg->mass_model == TL_MASS_EPL ? tl_trace_lin_epl_for(cfg->supersample, cfg->n_lens_light, cfg->n_source)
                                                          : tl_trace_lin_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
            bool okl = cuda_ok(cudaFuncSetAttribute(tl::conv_lin_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT));
            // two or three tiles per SM: ask for the largest shared-memory carveout
            okl = okl && cuda_ok(cudaFuncSetAttribute(tl::conv_lin_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            if (rowtab_bytes <= 48 * 1024) {
                c->lin_rowtab = 1; c->lin_trace_smem = rowtab_bytes;
                okl = okl && cuda_ok(cudaFuncSetAttribute(c->trace_lin, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rowtab_bytes));
            }
            if (!okl) { tl_destroy(c); return TL_ECUDA; }
        }
        // fused variant: C binned component images (+ the row-value table) in shared memory
        const size_t img_floats = ((size_t)c->He * c->pitch + c->pitch + c->Kp + 8 + 3) & ~(size_t)3;
        size_t fl = sizeof(tl::RowC) + 32 * sizeof(double) + sizeof(float) * ((size_t)c->K * c->Kp + (size_t)c->n_comp * img_floats);
        int rt = 0;
        if (fl + rowtab_bytes <= SMEM_LIMIT) { fl += rowtab_bytes; rt = 1; }
        if (fl <= SMEM_LIMIT) {
            fused_fn fn = cfg->mass_model == TL_MASS_EPL ? tl_fused_lin_epl_for(cfg->supersample, cfg->n_lens_light, cfg->n_source)
                                                         : tl_fused_lin_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
            int occ = 0;
            if (cuda_ok(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT)) &&
                cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, 512, fl)) && occ >= 1) {
                c->fused_lin = fn; c->lin_fused_smem = fl; c->lin_fused_rowtab = rt; c->lin_fused_grid = occ * c->n_sm;
            }
            cudaGetLastError();
        }
    }
    {   // double-precision path (tl_dp.cuh).  conv_dp_kernel: one CTA per (row, band of output rows).
        // Bands and CTA size are chosen together: the band's FP64 tile (+ K - 1 halo rows) and the taps
        // must fit in shared memory; several CTAs per SM hide the tile load behind other CTAs'
        // arithmetic; and the band's 1 x 8 strips should fill a whole number of rounds over the CTA's
        // threads.  Score = strip-round efficiency x min(1, warps per SM / 12) / halo re-read factor.
        c->dp_Wp = ((c->We + 13) & ~15) + 2;        // >= We and = 2 (mod 16): see conv_dp_kernel
        const int Kd = (c->K + 1) & ~1;
        const size_t fixed = (size_t)c->K * Kd + Kd + 16;
        const int nsx = (cfg->nx + 7) / 8;
        double best = -1.0;
        for (int nb = 1; nb <= cfg->ny && nb <= 64; ++nb) {
            const int br = (cfg->ny + nb - 1) / nb;
            if ((br - 1) * nb >= cfg->ny && nb > 1) continue;                 // an empty last band
            const size_t smem = sizeof(double) * (fixed + (size_t)(br + c->K - 1) * c->dp_Wp);
            if (smem > SMEM_LIMIT - 1024) continue;
            for (int thr = 64; thr <= 256; thr += 32) {
                int ctas = (int)(SMEM_LIMIT / (smem + 1024));
                const int by_regs = 65536 / (thr * 96), by_thr = 2048 / thr;
                if (ctas > by_regs) ctas = by_regs;
                if (ctas > by_thr) ctas = by_thr;
                if (ctas > 16) ctas = 16;
                if (ctas < 1) continue;
                const int strips = br * nsx, rounds = (strips + thr - 1) / thr;
                const double eff = (double)strips / ((double)rounds * thr);
                const double occ = ctas * thr / 32.0 >= 12.0 ? 1.0 : ctas * thr / 32.0 / 12.0;
                const double halo = 1.0 + 0.1 * (double)(c->K - 1) / br;       // the load is ~10 % of a band's time
                const double score = eff * occ / halo;
                if (score > best + 1e-9) { best = score; c->dp_n_bands = nb; c->dp_band_rows = br; c->dp_conv_threads = thr; c->dp_conv_smem = smem; }
            }
        }
        if (best > 0.0) {
            c->dp_trace = tl_trace_dp_for(cfg->supersample, cfg->n_lens_light, cfg->n_source);
            c->mge_dp_trace = tl_trace_dp_for(cfg->supersample, 0, cfg->n_source);
            int occ = 0;
            bool okd = cuda_ok(cudaFuncSetAttribute(tl::conv_dp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_LIMIT - 1024))) &&
                       cuda_ok(cudaFuncSetAttribute(tl::conv_dp_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) &&
                       cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->dp_trace, 256, 0)) && occ >= 1;
            if (!okd) { tl_destroy(c); return TL_ECUDA; }
            c->dp_trace_grid = occ * c->n_sm;
            int64_t cr = (int64_t)(((size_t)1 << 30) / (sizeof(double) * (size_t)c->He * c->dp_Wp));
            if (cr < 1) cr = 1;
            if (cr > 65535) cr = 65535;
            c->dp_chunk_rows = cr;
        }
    }
    *out = c;
    return TL_OK;
}

int tl_param_count(const tl_ctx *ctx) { return ctx ? ctx->P : TL_EINVAL; }

int tl_get_info(const tl_ctx *c, tl_info *info)
{
    if (!c || !info) return TL_EINVAL;
    info->n_params = c->P; info->path = c->path; info->block_threads = c->threads;
    info->ctas_per_sm = c->ctas_per_sm; info->grid = c->grid; info->smem_bytes = (int32_t)c->smem;
    info->n_sm = c->n_sm; info->launches_per_call = c->path == 0 ? 2 : 4;
    const bool ext = c->cfg.edge_mode == TL_EDGE_EXTEND;
    const int64_t hy = ext ? c->He : c->cfg.ny, wx = ext ? c->We : c->cfg.nx;
    info->samples_per_row = hy * wx * c->cfg.supersample * c->cfg.supersample;
    info->conv_fma_per_row = (int64_t)c->K * c->K * c->cfg.ny * c->cfg.nx;
    info->logl_const = c->lconst0; info->sigma_min = c->sigma_min0;
    info->small_batch_rows = c->path == 0 ? c->sb_max_rows : 0; info->chunk_rows = (int32_t)c->chunk_rows;
    return TL_OK;
}

int tl_loglike_batch(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream)
{
    return run_batch(ctx, params, B, logL, nullptr, (cudaStream_t)cuda_stream);
}

int tl_render_batch(tl_ctx *ctx, const float *params, int64_t B, float *images, void *cuda_stream)
{
    return run_batch(ctx, params, B, nullptr, images, (cudaStream_t)cuda_stream);
}

int tl_loglike_linear_batch(tl_ctx *c, const float *params, int64_t B, float *logL, float *amps, void *cuda_stream)
{
    if (!c || B < 0) return TL_EINVAL;
    if (B == 0) return TL_OK;
    if (!params || !logL || (B % c->cfg.n_lens) || c->cfg.n_lens_light > 1) return TL_EINVAL;
    if (!c->trace_lin) return TL_ESIZE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    const int NC = c->n_comp;
    const size_t npix = (size_t)c->cfg.ny * c->cfg.nx;
    // FP64 (and AUTO: with the amplitudes solved every row is near its best fit, so every row needs it)
    if (c->precision == TL_PRECISION_FP64 || c->precision == TL_PRECISION_AUTO)
        return run_dp(c, params, B, logL, nullptr, st, nullptr, nullptr, 1, amps);
    // few rows (a sampler's small proposal batches): the fused pipeline gives a row to ONE CTA, so such
    // a call costs a whole row-time of one SM (0.21 ms on configs[1]); the staged pipeline spreads a row over many
    // CTAs -- and returns the same bits
    bool few = B <= c->n_sm / 2 && c->opt.small_batch_rows != 0;
    int64_t r_begin = 0;                                       // the staged pipeline serves rows r_begin .. B - 1
    if (c->fused_lin && !c->opt.linear_staged && !few) {
        // the rows of a last, mostly empty wave of the persistent grid go through the staged pipeline (as in run_batch)
        int64_t B_tail = 0;
        if (c->opt.small_batch_rows != 0 && B <= CONST_CHUNK && B > c->lin_fused_grid) {
            const int64_t rem = B % c->lin_fused_grid;
            if (rem > 0 && rem <= c->n_sm / 2) B_tail = rem;
        }
        const int64_t B_all = B;
        B -= B_tail;
        const int64_t chunkf = CONST_CHUNK < B ? CONST_CHUNK : B;
        tl::RowC *rowsf = nullptr;
        float *mscr = nullptr;
        if (!pool_alloc(c, &rowsf, sizeof(tl::RowC) * (size_t)chunkf, st)) return TL_ENOMEM;
        if (!pool_alloc(c, &mscr, sizeof(float) * (size_t)c->lin_fused_grid * NC * npix, st)) { pool_free(c, rowsf, st); return TL_ENOMEM; }
        const int64_t rpl = B_all / c->cfg.n_lens;
        int rcf = TL_OK;
        for (int64_t r0 = 0; r0 < B && rcf == TL_OK; r0 += chunkf) {
            const int64_t nb = (B - r0 < chunkf) ? (B - r0) : chunkf;
            tl::PrologueArgs pa;
            fill_prologue_args(c, pa, params, rowsf, nb, r0, rpl, 1);
            tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);
            tl::KArgs a = base_args(c);
            a.rows = rowsf; a.B = nb; a.rows_per_lens = rpl; a.row0 = r0;
            a.logL = logL; a.amps = amps; a.mimg = mscr; a.rowtab = c->lin_fused_rowtab;
            int grid = c->lin_fused_grid;
            if ((int64_t)grid > nb) grid = (int)nb;
            if (c->profile) cudaEventRecord(c->ev0, st);
            c->fused_lin<<<grid, 512, c->lin_fused_smem, st>>>(a);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
            if (!cuda_ok(cudaGetLastError())) rcf = TL_ECUDA;
        }
        pool_free(c, rowsf, st); pool_free(c, mscr, st);
        r_begin = B;
        B = B_all;
        if (rcf != TL_OK || B_tail == 0) return rcf;
        few = true;
    }
    const size_t ext_row = sizeof(float) * (size_t)NC * c->He * c->pitch, m_row = sizeof(float) * NC * npix;
    int64_t chunk = (int64_t)(EXT_SCRATCH_BYTES / (ext_row + m_row));
    if (chunk < 1) chunk = 1;
    if (chunk > 65535) chunk = 65535;
    if (chunk > B - r_begin) chunk = B - r_begin;
    tl::RowC *rows = nullptr;
    float *ext = nullptr, *mimg = nullptr;
    if (!pool_alloc(c, &rows, (sizeof(tl::RowC) + sizeof(int)) * (size_t)chunk, st)) return TL_ENOMEM;   // + a tile-queue head per row
    if (!pool_alloc(c, &ext, ext_row * (size_t)chunk, st) ||
        !pool_alloc(c, &mimg, m_row * (size_t)chunk, st)) {
        pool_free(c, rows, st);
        if (ext) pool_free(c, ext, st);
        return TL_ENOMEM;
    }
    cudaMemsetAsync(ext, 0, ext_row * (size_t)chunk, st);      // pitch padding must read as finite zeros
    const int64_t rows_per_lens = B / c->cfg.n_lens;
    int rc = TL_OK;
    for (int64_t r0 = r_begin; r0 < B && rc == TL_OK; r0 += chunk) {
        const int64_t nb = (B - r0 < chunk) ? (B - r0) : chunk;
        tl::PrologueArgs pa;
        fill_prologue_args(c, pa, params, rows, nb, r0, rows_per_lens, 1);
        tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);
        tl::KArgs a = base_args(c);
        a.rows = rows; a.B = nb; a.rows_per_lens = rows_per_lens; a.row0 = r0;
        a.logL = logL; a.amps = amps; a.ext = ext; a.mimg = mimg;
        a.tile_rows = c->lin_tile_rows; a.n_tiles = c->lin_n_tiles; a.rowtab = c->lin_rowtab;
        a.tile_counters = reinterpret_cast<int *>(rows + chunk);          // the row's CTAs draw warp tiles from one queue (see run_batch)
        cudaMemsetAsync(a.tile_counters, 0, sizeof(int) * (size_t)nb, st);
        int slabs = 8;
        size_t conv_smem = c->lin_conv_smem;
        if (few) {
            // as many CTAs per row as are resident at once: more ray-trace slabs, thinner convolution tiles (pairs of rows)
            const int want = 2 * c->n_sm / (int)nb, n_wtiles = a.tiles_x * a.tiles_y;
            slabs = want < (n_wtiles + 7) / 8 ? want : (n_wtiles + 7) / 8;
            if (slabs < 1) slabs = 1;
            int nt = want / NC;
            if (nt < 1) nt = 1;
            int tr = (c->cfg.ny + nt - 1) / nt;
            tr = (tr + 1) & ~1;
            if (tr < 2) tr = 2;
            if (tr < c->lin_tile_rows) {
                a.tile_rows = tr; a.n_tiles = (c->cfg.ny + tr - 1) / tr;
                conv_smem = conv_smem_bytes(c, tr);
            }
        }
        dim3 tg((unsigned)nb, (unsigned)slabs);
        if (c->profile) cudaEventRecord(c->ev0, st);
        c->trace_lin<<<tg, 256, c->lin_trace_smem, st>>>(a, (int)nb);
        if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
        dim3 cg((unsigned)nb, (unsigned)a.n_tiles, (unsigned)NC);
        tl::conv_lin_kernel<<<cg, 256, conv_smem, st>>>(a, (int)nb);
        tl::solve_lin_kernel<<<(unsigned)nb, 256, 0, st>>>(a, (int)nb);
        if (!cuda_ok(cudaGetLastError())) rc = TL_ECUDA;
    }
    pool_free(c, rows, st); pool_free(c, ext, st); pool_free(c, mimg, st);
    return rc;
}

namespace { int64_t mge_chunk_rows(const tl_ctx *c); }

int tl_set_mge(tl_ctx *c, const float *sigmas, int32_t n_gauss)
{
    return tl_set_mge_sets(c, sigmas, &n_gauss, 1);
}

int tl_set_mge_sets(tl_ctx *c, const float *sigmas, const int32_t *n_per_set, int32_t n_sets)
{
    if (!c || !sigmas || !n_per_set || n_sets < 1 || n_sets > tl::MGE_MAX_SETS) return TL_EINVAL;
    if (c->cfg.n_lens_light != n_sets) return TL_EINVAL;           // one lens-light block of the row per set
    int n_gauss = 0;
    for (int j = 0; j < n_sets; ++j) { if (n_per_set[j] < 1) return TL_EINVAL; n_gauss += n_per_set[j]; }
    if (n_gauss > tl::MGE_MAX_GAUSS) return TL_EINVAL;
    if (!c->trace_lin) return TL_ESIZE;
    float ck[tl::MGE_MAX_GAUSS];
    double ck64[tl::MGE_MAX_GAUSS];
    int set_of[tl::MGE_MAX_GAUSS];
    for (int k = 0, j = 0, left = n_per_set[0]; k < n_gauss; ++k, --left) {
        while (left == 0) left = n_per_set[++j];
        set_of[k] = j;
        if (!std::isfinite(sigmas[k]) || !(sigmas[k] > 0.f)) return TL_EINVAL;
        ck64[k] = 1.4426950408889634074 / (2.0 * (double)sigmas[k] * (double)sigmas[k]);
        ck[k] = (float)ck64[k];
        if (!std::isfinite(ck[k])) return TL_EINVAL;
    }
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    if (!c->mge_c && (!cuda_ok(cudaMalloc(&c->mge_c, sizeof(float) * tl::MGE_MAX_GAUSS)) ||
                      !cuda_ok(cudaMalloc(&c->mge_c64, sizeof(double) * tl::MGE_MAX_GAUSS)) ||
                      !cuda_ok(cudaMalloc(&c->mge_set, sizeof(int) * tl::MGE_MAX_GAUSS)))) return TL_ENOMEM;
    if (!cuda_ok(cudaMemcpy(c->mge_c, ck, sizeof(float) * n_gauss, cudaMemcpyHostToDevice)) ||
        !cuda_ok(cudaMemcpy(c->mge_c64, ck64, sizeof(double) * n_gauss, cudaMemcpyHostToDevice)) ||
        !cuda_ok(cudaMemcpy(c->mge_set, set_of, sizeof(int) * n_gauss, cudaMemcpyHostToDevice))) return TL_ECUDA;
    c->mge_n_sets = n_sets;
    for (int j = 0; j < tl::MGE_MAX_SETS; ++j) c->mge_per_set[j] = j < n_sets ? n_per_set[j] : 0;
    c->n_gauss = n_gauss;
    if (!c->mge_trace) {
        // sources through the NLL = 0 ray-trace kernels (no lens-light stand-in; one source: packed pair loop)
        const bool epl = c->cfg.mass_model == TL_MASS_EPL;
        const int S = c->cfg.supersample, ns = c->cfg.n_source;
        c->mge_trace = ns == 1 ? (epl ? tl_trace_epl_for(S, 0, 1) : tl_trace_for(S, 0, 1))
                               : (epl ? tl_trace_lin_epl_for(S, 0, 2) : tl_trace_lin_for(S, 0, 2));
        const size_t rowtab_bytes = sizeof(tl::RowV) * (size_t)c->He * S;
        bool okm = true;
        if (rowtab_bytes <= 48 * 1024) {
            c->mge_rowtab = 1; c->mge_trace_smem = rowtab_bytes;
            okm = cuda_ok(cudaFuncSetAttribute(c->mge_trace, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rowtab_bytes));
        }
        // gauss_conv_kernel needs the whole extended image of one Gaussian (+ taps) in shared memory
        c->mge_gc_smem = sizeof(float) * ((size_t)c->K * c->Kp + (size_t)(c->He + 1) * c->pitch + c->Kp + 8);
        c->mge_fused = c->mge_gc_smem <= SMEM_LIMIT - 1024;
        if (c->mge_fused)
            okm = okm && cuda_ok(cudaFuncSetAttribute(tl::gauss_conv_for(S, c->K), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM_LIMIT - 1024))) &&
                  cuda_ok(cudaFuncSetAttribute(tl::gauss_conv_for(S, c->K), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        okm = okm && cuda_ok(cudaFuncSetAttribute(tl::nnls_mge_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)(sizeof(double) * tl::MGE_NNLS_WARPS * (2 * tl::MGE_MAX_COL * tl::MGE_MAX_COL + 3 * tl::MGE_MAX_COL))));
        if (!okm) { c->mge_trace = nullptr; c->n_gauss = 0; cudaGetLastError(); return TL_ECUDA; }
    }
    if (c->pool) {   // the MGE call stages a chunk's component images: let the pool keep that much cached between calls
        const int NC = n_gauss + c->cfg.n_source;
        const size_t per_row = sizeof(float) * ((size_t)(c->mge_fused ? c->cfg.n_source : NC) * c->He * c->pitch + (size_t)NC * c->cfg.ny * c->cfg.nx);
        unsigned long long want = (unsigned long long)per_row * (unsigned long long)mge_chunk_rows(c) + (64ull << 20), cur = 0;
        if (want > MGE_SCRATCH_BYTES + (256ull << 20)) want = MGE_SCRATCH_BYTES + (256ull << 20);
        cudaMemPoolGetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &cur);
        if (want > cur) cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &want);
        cudaGetLastError();
    }
    return TL_OK;
}

namespace {
int64_t mge_chunk_rows(const tl_ctx *c)
{
    const int NC = c->n_gauss + c->cfg.n_source;
    const size_t npix = (size_t)c->cfg.ny * c->cfg.nx;
    const size_t ext_row = sizeof(float) * (size_t)(c->mge_fused ? c->cfg.n_source : NC) * c->He * c->pitch, m_row = sizeof(float) * NC * npix;
    int64_t chunk = (int64_t)(MGE_SCRATCH_BYTES / (ext_row + m_row));
    if (chunk < 1) chunk = 1;
    if (chunk > 65535) chunk = 65535;
    if (c->opt.mge_chunk_rows >= 1 && c->opt.mge_chunk_rows < chunk) chunk = c->opt.mge_chunk_rows;   // tests: the multi-chunk path
    return chunk;
}
}  // namespace

int64_t tl_mge_chunk_rows(const tl_ctx *c) { return (c && c->n_gauss > 0) ? mge_chunk_rows(c) : (int64_t)TL_EINVAL; }

int tl_mge_columns(const tl_ctx *c) { return (c && c->n_gauss > 0) ? c->n_gauss + c->cfg.n_source : TL_EINVAL; }

namespace {
// tl_loglike_mge_batch in FP64 (TL_PRECISION_FP64 / AUTO: with solved amplitudes every row is near its best
// fit): the sources through trace_dp_kernel<S,0,NSRC> with the components apart, the Gaussians by
// gauss_dp_kernel, every column blurred by conv_dp_kernel, then the Gram / NNLS kernels of tl_mge.cuh on
// the FP64 columns.  The FP32 prologue also runs: the solver kernels take the row validity from RowC.
int run_mge_dp(tl_ctx *c, const float *params, int64_t B, float *logL, float *amps, cudaStream_t st)
{
    const int NG = c->n_gauss, NS = c->cfg.n_source, NC = NG + NS;
    const size_t npix = (size_t)c->cfg.ny * c->cfg.nx;
    const size_t ext_row = sizeof(double) * (size_t)NC * c->He * c->dp_Wp, m_row = sizeof(double) * NC * npix;
    int64_t chunk = (int64_t)(MGE_SCRATCH_BYTES / (ext_row + m_row));
    if (chunk < 1) chunk = 1;
    if (chunk > 65535) chunk = 65535;
    if (c->opt.mge_chunk_rows >= 1 && c->opt.mge_chunk_rows < chunk) chunk = c->opt.mge_chunk_rows;
    if (chunk > B) chunk = B;
    tl::RowC *rows = nullptr;
    tl::RowD *rowsd = nullptr;
    double *ext = nullptr, *m64 = nullptr, *gram = nullptr;
    const size_t g_row = sizeof(double) * tl::MGE_GRAM_STRIDE;
    if (!pool_alloc(c, &rows, sizeof(tl::RowC) * (size_t)chunk, st) || !pool_alloc(c, &rowsd, sizeof(tl::RowD) * (size_t)chunk, st) ||
        !pool_alloc(c, &ext, ext_row * (size_t)chunk, st) || !pool_alloc(c, &m64, m_row * (size_t)chunk, st) ||
        !pool_alloc(c, &gram, g_row * (size_t)chunk, st)) {
        if (rows) pool_free(c, rows, st);
        if (rowsd) pool_free(c, rowsd, st);
        if (ext) pool_free(c, ext, st);
        if (m64) pool_free(c, m64, st);
        return TL_ENOMEM;
    }
    if (c->dp_Wp != c->We) cudaMemsetAsync(ext, 0, ext_row * (size_t)chunk, st);     // pitch padding must be finite
    const int64_t rows_per_lens = B / c->cfg.n_lens;
    int rc = TL_OK;
    for (int64_t r0 = 0; r0 < B && rc == TL_OK; r0 += chunk) {
        const int64_t nb = (B - r0 < chunk) ? (B - r0) : chunk;
        tl::PrologueArgs pa;
        fill_prologue_args(c, pa, params, rows, nb, r0, rows_per_lens, 1);
        pa.mge = 1;
        tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);
        tl::DpArgs d;
        memset(&d, 0, sizeof(d));
        d.params = params; d.rows = rowsd; d.n_rows = (int)nb; d.row0 = r0; d.rows_per_lens = rows_per_lens;
        d.psf = c->psf; d.data = c->data; d.wgt64 = c->wgt64; d.lconst = c->lconst;
        d.ext = ext; d.m64 = m64; d.logL = logL; d.amps = amps; d.lin = 1; d.mge = 1;
        d.ext_nc = NC; d.ext_k0 = NG; d.n_gauss = NG; d.n_source = NS; d.mge_c = c->mge_c64; d.mge_set = c->mge_set;
        d.P = c->P; d.ny = c->cfg.ny; d.nx = c->cfg.nx; d.K = c->K; d.Kp = c->Kp; d.h = c->h;
        d.He = c->He; d.We = c->We; d.Wp = c->dp_Wp; d.S = c->cfg.supersample;
        d.n_lens_light = c->cfg.n_lens_light; d.n_comp = c->n_comp;
        d.edge_zero = c->cfg.edge_mode == TL_EDGE_ZERO; d.mass_model = c->cfg.mass_model; d.lens_np = c->lens_np;
        d.band_rows = c->dp_band_rows; d.n_bands = c->dp_n_bands;
        d.CW = c->CW; d.CH = c->CH; d.tiles_x = (c->We + c->CW - 1) / c->CW; d.tiles_y = (c->He + c->CH - 1) / c->CH;
        d.u = c->cfg.pix_scale / (2.0 * c->cfg.supersample);
        tl::prologue_dp_kernel<<<(unsigned)((nb + 63) / 64), 64, 0, st>>>(d);
        const int64_t items = nb * d.tiles_x * d.tiles_y;
        int grid = c->dp_trace_grid;
        if ((int64_t)grid * 8 > items) grid = (int)((items + 7) / 8);
        c->mge_dp_trace<<<grid, 256, 0, st>>>(d);
        int gslabs = (int)(((int64_t)c->He * c->We * NG + 255) / 256);
        if (gslabs > 64) gslabs = 64;
        tl::gauss_dp_kernel<<<dim3((unsigned)nb, (unsigned)gslabs), 256, 0, st>>>(d);
        if (c->profile) cudaEventRecord(c->ev0, st);
        tl::conv_dp_kernel<<<dim3((unsigned)nb, (unsigned)c->dp_n_bands, (unsigned)NC), c->dp_conv_threads, c->dp_conv_smem, st>>>(d);
        if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
        tl::KArgs a = base_args(c);
        a.rows = rows; a.B = nb; a.rows_per_lens = rows_per_lens; a.row0 = r0;
        a.logL = logL; a.amps = amps; a.ext_nc = NC; a.mimg64 = m64; a.wgt64 = c->wgt64; a.mge_gram = gram;
        if (NC + 1 <= 20) tl::gram_mge_kernel<128, double><<<(unsigned)nb, 128, 0, st>>>(a, (int)nb);
        else tl::gram_mge_kernel<512, double><<<(unsigned)nb, 512, 0, st>>>(a, (int)nb);
        const size_t nnls_smem = sizeof(double) * tl::MGE_NNLS_WARPS * (size_t)(2 * NC * NC + 3 * NC);
        tl::nnls_mge_kernel<<<(unsigned)((nb + tl::MGE_NNLS_WARPS - 1) / tl::MGE_NNLS_WARPS), 32 * tl::MGE_NNLS_WARPS, nnls_smem, st>>>(a, (int)nb);
        if (!cuda_ok(cudaGetLastError())) rc = TL_ECUDA;
    }
    pool_free(c, rows, st); pool_free(c, rowsd, st); pool_free(c, ext, st); pool_free(c, m64, st); pool_free(c, gram, st);
    return rc;
}
}  // namespace

int tl_loglike_mge_batch(tl_ctx *c, const float *params, int64_t B, float *logL, float *amps, void *cuda_stream)
{
    if (!c || B < 0) return TL_EINVAL;
    if (c->n_gauss < 1) return TL_EINVAL;
    if (B == 0) return TL_OK;
    if (!params || !logL || (B % c->cfg.n_lens)) return TL_EINVAL;
    if (!c->trace_lin || !c->mge_trace) return TL_ESIZE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(c->device);
    if (!guard.ok) return TL_ECUDA;
    if (c->precision == TL_PRECISION_FP64 || c->precision == TL_PRECISION_AUTO) {
        if (!c->mge_dp_trace) return TL_ESIZE;
        return run_mge_dp(c, params, B, logL, amps, st);
    }
    const int NG = c->n_gauss, NS = c->cfg.n_source, NC = NG + NS;
    const int fused = c->mge_fused;
    const size_t npix = (size_t)c->cfg.ny * c->cfg.nx;
    const int ext_nc = fused ? NS : NC;                        // component images staged in global memory per row
    const size_t ext_row = sizeof(float) * (size_t)ext_nc * c->He * c->pitch, m_row = sizeof(float) * NC * npix;
    int64_t chunk = mge_chunk_rows(c);
    if (chunk > B) chunk = B;
    tl::RowC *rows = nullptr;
    float *ext = nullptr, *mimg = nullptr;
    double *gram = nullptr;                                    // [chunk][MGE_GRAM_STRIDE]
    const size_t g_row = sizeof(double) * tl::MGE_GRAM_STRIDE;
    // the budget is a target, not a promise: when the device cannot give that much, halve the chunk
    for (;;) {
        rows = nullptr; ext = nullptr; mimg = nullptr; gram = nullptr;
        if (pool_alloc(c, &rows, (sizeof(tl::RowC) + sizeof(int)) * (size_t)chunk, st) &&    // + one tile-queue head per row
            pool_alloc(c, &ext, ext_row * (size_t)chunk, st) &&
            pool_alloc(c, &mimg, m_row * (size_t)chunk, st) &&
            pool_alloc(c, &gram, g_row * (size_t)chunk, st)) break;
        cudaGetLastError();                                    // an allocation failure is not sticky
        if (rows) pool_free(c, rows, st);
        if (ext) pool_free(c, ext, st);
        if (mimg) pool_free(c, mimg, st);
        if (gram) pool_free(c, gram, st);
        if (chunk == 1) return TL_ENOMEM;
        chunk = (chunk + 1) / 2;
    }
    // the pitch padding of ext must read as finite zeros: written by mge_gauss_kernel when it runs,
    // else (fused: ext holds the source images only) cleared here
    if (fused) cudaMemsetAsync(ext, 0, ext_row * (size_t)chunk, st);
    const int64_t rows_per_lens = B / c->cfg.n_lens;
    int gslabs = (c->He * c->pitch + 255) / 256;
    if (gslabs > 16) gslabs = 16;
    int rc = TL_OK;
    for (int64_t r0 = 0; r0 < B && rc == TL_OK; r0 += chunk) {
        const int64_t nb = (B - r0 < chunk) ? (B - r0) : chunk;
        tl::PrologueArgs pa;
        fill_prologue_args(c, pa, params, rows, nb, r0, rows_per_lens, 1);
        pa.mge = 1;
        tl::prologue_kernel<<<tl::prologue_blocks(nb), 128, 0, st>>>(pa);
        tl::KArgs a = base_args(c);
        a.rows = rows; a.B = nb; a.rows_per_lens = rows_per_lens; a.row0 = r0;
        a.logL = logL; a.amps = amps; a.ext = ext; a.mimg = mimg;
        a.tile_rows = c->lin_tile_rows; a.n_tiles = c->lin_n_tiles;
        a.n_gauss = NG; a.mge_c = c->mge_c; a.mge_set = c->mge_set; a.mge_gram = gram;
        // 1. the sources, ray-traced at unit amplitude -> ext slots (fused: 0.., else NG..)
        // (the row's CTAs draw warp tiles from one queue per row: the tile next to the source centre, full of
        // FP64-refined samples, costs several times an ordinary one and a static split leaves its CTA's other warps idle)
        tl::KArgs at = a;
        at.rowtab = c->mge_rowtab; at.ext_nc = ext_nc; at.ext_k0 = fused ? 0 : NG;
        at.tile_counters = reinterpret_cast<int *>(rows + chunk);
        cudaMemsetAsync(at.tile_counters, 0, sizeof(int) * (size_t)nb, st);
        // calls with a few rows (a sampler's small proposal batches): as many CTAs per row as are resident at once
        const bool few = nb <= c->n_sm / 2 && c->opt.small_batch_rows != 0;
        const int want = few ? 2 * c->n_sm / (int)nb : 0;
        int tslabs = 2;                                        // (slabs per row: 1 .. 4 measured equal, 8 1 % slower)
        if (few) {
            const int n_wtiles = at.tiles_x * at.tiles_y;
            tslabs = want < (n_wtiles + 7) / 8 ? want : (n_wtiles + 7) / 8;
            if (tslabs < 1) tslabs = 1;
        }
        c->mge_trace<<<dim3((unsigned)nb, (unsigned)tslabs), 256, c->mge_trace_smem, st>>>(at, (int)nb);
        a.ext_nc = NC;                                         // from here on: the width of M
        if (fused) {
            // 2. every Gaussian evaluated into shared memory and blurred from there -> M[0 .. NG)
            if (c->profile) cudaEventRecord(c->ev0, st);
            int gbands = 1;                                    // few rows: the output row pairs of a Gaussian over several CTAs
            const bool kblk = c->K == 5 || c->K == 15 || c->K == 21 || c->K == 31 || c->K == 41;
            if (few && kblk) {
                gbands = want / NG;
                const int npair = (c->cfg.ny + 1) / 2;
                if (gbands > npair) gbands = npair;
                if (gbands < 1) gbands = 1;
            }
            tl::gauss_conv_for(c->cfg.supersample, c->K)<<<dim3((unsigned)nb, (unsigned)NG, (unsigned)gbands), 256, c->mge_gc_smem, st>>>(a, (int)nb);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
            // 3. the sources blurred -> M[NG ..)
            tl::KArgs ac = a;
            ac.conv_ext_nc = NS; ac.conv_m_nc = NC; ac.conv_m_k0 = NG;
            size_t lsmem = c->lin_conv_smem;
            if (few) {                                         // thin tiles (pairs of rows): the source images over many CTAs too
                int nt = want / NS;
                if (nt < 1) nt = 1;
                int tr = ((c->cfg.ny + nt - 1) / nt + 1) & ~1;
                if (tr < 2) tr = 2;
                if (tr < c->lin_tile_rows) { ac.tile_rows = tr; ac.n_tiles = (c->cfg.ny + tr - 1) / tr; lsmem = conv_smem_bytes(c, tr); }
            }
            tl::conv_lin_kernel<<<dim3((unsigned)nb, (unsigned)ac.n_tiles, (unsigned)NS), 256, lsmem, st>>>(ac, (int)nb);
        } else {
            for (int j = 0, k0 = 0; j < c->mge_n_sets; k0 += c->mge_per_set[j], ++j) {          // one launch per set
                tl::KArgs ag = a;
                ag.mge_k0 = k0; ag.mge_shape = j;
                tl::mge_gauss_for(c->mge_per_set[j])<<<dim3((unsigned)nb, (unsigned)gslabs), 256, 0, st>>>(ag, (int)nb);
            }
            if (c->profile) cudaEventRecord(c->ev0, st);
            tl::conv_lin_kernel<<<dim3((unsigned)nb, (unsigned)c->lin_n_tiles, (unsigned)NC), 256, c->lin_conv_smem, st>>>(a, (int)nb);
            if (c->profile) { cudaEventRecord(c->ev1, st); c->prof_pending = 1; }
        }
        // 4. Gram matrix, 5. NNLS + logL
        if (NC <= tl::MGE_GRAM_REG_COLS && ((c->cfg.ny * c->cfg.nx) & 1) == 0) tl::gram_reg_for(NC + 1, c->cfg.ny * c->cfg.nx)<<<(unsigned)nb, 128, 0, st>>>(a, (int)nb);
        else if (NC + 1 <= 20) tl::gram_mge_kernel<128><<<(unsigned)nb, 128, 0, st>>>(a, (int)nb);
        else tl::gram_mge_kernel<512><<<(unsigned)nb, 512, 0, st>>>(a, (int)nb);
        const size_t nnls_smem = sizeof(double) * tl::MGE_NNLS_WARPS * (size_t)(2 * NC * NC + 3 * NC);
        tl::nnls_mge_kernel<<<(unsigned)((nb + tl::MGE_NNLS_WARPS - 1) / tl::MGE_NNLS_WARPS), 32 * tl::MGE_NNLS_WARPS, nnls_smem, st>>>(a, (int)nb);
        if (!cuda_ok(cudaGetLastError())) rc = TL_ECUDA;
    }
    pool_free(c, rows, st); pool_free(c, ext, st); pool_free(c, mimg, st); pool_free(c, gram, st);
    return rc;
}

int tl_loglike_batch_host_async(tl_ctx *c, const float *params, int64_t B, float *logL, void *cuda_stream)
{
    if (!c || B < 1 || !params || !logL || (B % c->cfg.n_lens)) return TL_EINVAL;
    DeviceGuard guard(c->device);                    // before any allocation: the buffers belong to the context's device
    if (!guard.ok) return TL_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int id = c->next_slot;
    tl_ctx::HostSlot &sl = c->slots[id];
    if (sl.busy) {                                   // a third submission waits for the oldest one
        const int wrc = tl_wait(c, id);
        if (wrc != TL_OK) return wrc;
    }
    if (!c->s_up) {
        if (!cuda_ok(cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking)) ||
            !cuda_ok(cudaStreamCreateWithFlags(&c->s_down, cudaStreamNonBlocking))) return TL_ECUDA;
    }
    if (!sl.up) {
        if (!cuda_ok(cudaEventCreateWithFlags(&sl.up, cudaEventDisableTiming)) ||
            !cuda_ok(cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming)) ||
            !cuda_ok(cudaEventCreateWithFlags(&sl.fin, cudaEventDisableTiming))) return TL_ECUDA;
    }
    if (B > sl.cap_rows) {                           // grow the slot (first call, or a larger batch than ever before)
        cudaFreeHost(sl.h_params); cudaFreeHost(sl.h_logl); cudaFree(sl.d_params); cudaFree(sl.d_logl);
        sl.h_params = sl.h_logl = sl.d_params = sl.d_logl = nullptr; sl.cap_rows = 0;
        const int64_t cap = B < 1024 ? 1024 : B;
        if (!cuda_ok(cudaMallocHost(&sl.h_params, sizeof(float) * (size_t)cap * c->P)) ||
            !cuda_ok(cudaMallocHost(&sl.h_logl, sizeof(float) * (size_t)cap)) ||
            !cuda_ok(cudaMalloc(&sl.d_params, sizeof(float) * (size_t)cap * c->P)) ||
            !cuda_ok(cudaMalloc(&sl.d_logl, sizeof(float) * (size_t)cap))) { cudaGetLastError(); return TL_ENOMEM; }
        sl.cap_rows = cap;
    }
    memcpy(sl.h_params, params, sizeof(float) * (size_t)B * c->P);       // the caller's buffer is free again on return
    int rc = TL_OK;
    // up to 8 rows (measured: 56 -> 45 us host to host for one row, no gain from 16): the kernels read the rows from and write logL to the pinned staging buffers themselves (under 1 KB over
    // PCIe inside the prologue / the last reduction) -- two copies, three events and two stream waits less per call
    void *hp_dev = nullptr, *hl_dev = nullptr;
    if (B <= 8 && cuda_ok(cudaHostGetDevicePointer(&hp_dev, sl.h_params, 0)) && cuda_ok(cudaHostGetDevicePointer(&hl_dev, sl.h_logl, 0))) {
        rc = run_batch(c, static_cast<const float *>(hp_dev), B, static_cast<float *>(hl_dev), nullptr, st);
        if (rc == TL_OK && !cuda_ok(cudaEventRecord(sl.fin, st))) rc = TL_ECUDA;
        if (rc != TL_OK) return rc;
        sl.B = B; sl.user_logl = logL; sl.busy = 1; sl.rc = TL_OK;
        c->next_slot = id ^ 1;
        return id;
    }
    cudaGetLastError();
    if (!cuda_ok(cudaMemcpyAsync(sl.d_params, sl.h_params, sizeof(float) * (size_t)B * c->P, cudaMemcpyHostToDevice, c->s_up)) ||
        !cuda_ok(cudaEventRecord(sl.up, c->s_up)) || !cuda_ok(cudaStreamWaitEvent(st, sl.up, 0))) rc = TL_ECUDA;
    if (rc == TL_OK) rc = run_batch(c, sl.d_params, B, sl.d_logl, nullptr, st);
    if (rc == TL_OK &&
        (!cuda_ok(cudaEventRecord(sl.done, st)) || !cuda_ok(cudaStreamWaitEvent(c->s_down, sl.done, 0)) ||
         !cuda_ok(cudaMemcpyAsync(sl.h_logl, sl.d_logl, sizeof(float) * (size_t)B, cudaMemcpyDeviceToHost, c->s_down)) ||
         !cuda_ok(cudaEventRecord(sl.fin, c->s_down)))) rc = TL_ECUDA;
    if (rc != TL_OK) return rc;
    sl.B = B; sl.user_logl = logL; sl.busy = 1; sl.rc = TL_OK;
    c->next_slot = id ^ 1;
    return id;
}

int tl_wait(tl_ctx *c, int slot)
{
    if (!c || slot < 0 || slot > 1 || !c->slots[slot].busy) return TL_EINVAL;
    tl_ctx::HostSlot &sl = c->slots[slot];
    int rc = sl.rc;
    if (!cuda_ok(cudaEventSynchronize(sl.fin))) rc = TL_ECUDA;
    if (rc == TL_OK) memcpy(sl.user_logl, sl.h_logl, sizeof(float) * (size_t)sl.B);
    sl.busy = 0;
    return rc;
}

int tl_loglike_batch_host(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream)
{
    if (!ctx || B < 0 || (B > 0 && (!params || !logL))) return TL_EINVAL;
    if (B == 0) return TL_OK;
    const int slot = tl_loglike_batch_host_async(ctx, params, B, logL, cuda_stream);
    return slot < 0 ? slot : tl_wait(ctx, slot);
}

int tl_set_precision(tl_ctx *c, int precision)
{
    if (!c || precision < TL_PRECISION_FP32 || precision > TL_PRECISION_AUTO) return TL_EINVAL;
    if ((precision == TL_PRECISION_FP64 || precision == TL_PRECISION_AUTO) && !c->dp_trace) return TL_ESIZE;
    c->precision = precision;
    return TL_OK;
}

int tl_set_profiling(tl_ctx *c, int enable)
{
    if (!c) return TL_EINVAL;
    if (enable && !c->ev0) {
        if (!cuda_ok(cudaEventCreate(&c->ev0)) || !cuda_ok(cudaEventCreate(&c->ev1))) return TL_ECUDA;
    }
    c->profile = enable ? 1 : 0;
    c->prof_pending = 0;
    return TL_OK;
}

int tl_last_kernel_ms(tl_ctx *c, float *ms)
{
    if (!c || !ms || !c->profile || !c->prof_pending) return TL_EINVAL;
    if (!cuda_ok(cudaEventSynchronize(c->ev1)) || !cuda_ok(cudaEventElapsedTime(ms, c->ev0, c->ev1))) return TL_ECUDA;
    return TL_OK;
}

void tl_destroy(tl_ctx *c)
{
    if (!c) return;
    tl_serve_stop(c);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    for (auto &sl : c->slots) {
        if (sl.busy && sl.fin) cudaEventSynchronize(sl.fin);
        if (sl.up) cudaEventDestroy(sl.up);
        if (sl.done) cudaEventDestroy(sl.done);
        if (sl.fin) cudaEventDestroy(sl.fin);
        cudaFreeHost(sl.h_params); cudaFreeHost(sl.h_logl); cudaFree(sl.d_params); cudaFree(sl.d_logl);
    }
    if (c->s_up) cudaStreamDestroy(c->s_up);
    if (c->s_down) cudaStreamDestroy(c->s_down);
    cudaFree(c->mge_c); cudaFree(c->mge_c64); cudaFree(c->mge_set); cudaFree(c->canary_errors);
    cudaFree(c->psf); cudaFree(c->data); cudaFree(c->wgt); cudaFree(c->wgt64); cudaFree(c->noise); cudaFree(c->sigma_min); cudaFree(c->lconst);
    if (c->pool) cudaMemPoolDestroy(c->pool);
    delete c;
}

}  // extern "C"
