/*
 * tinylens.h -- C ABI of the B200-native batched lens-model likelihood.
 *
 * The library evaluates, for a batch of B parameter vectors, the forward model of
 * arxiv 2503.08586 (TinyLensGpu) and its Gaussian log-likelihood, entirely in hand-written
 * sm_100a CUDA kernels.  There is NO CPU fallback: every compute entry point returns
 * TL_ECUDA when no CUDA device is usable.
 *
 * Citations are PAPER.md:<line> (+ equation) of the paper text; "G<k>" are the readings of
 * points the paper leaves open, listed in DESIGN.md "Readings of the paper".
 *
 * The operation (per parameter row; PAPER.md:52-71 section 2.1, :80-84 Eq. 5, :133-162 section 2.4):
 *   1. every S x S sub-sample theta of every native pixel ("4x4 supersampling")
 *      is ray-traced, beta = theta - alpha(theta)                       (Eq. 1),
 *      alpha = SIE (EPL with gamma = 2, Eq. 12) + external shear
 *      (PAPER.md:162 Eq. 13, :187-190 Eq. 14);
 *   2. I(theta) = sum_lens-light Sersic(theta) + sum_sources Sersic(beta)  (Eq. 2)
 *      with the elliptical Sersic profile of PAPER.md:135 Eq. 8, :139 Eq. 9 (b_n), :143-148 Eq. 10;
 *   3. the S*S samples of a native pixel are averaged ("binning");
 *   4. the binned image is convolved with the PSF kernel K               (Eq. 3);
 *   5. logL = -1/2 sum_i [ (d_i - Im_i)^2 / sigma_i^2 + ln(2 pi sigma_i^2) ]  (Eq. 5).
 *
 * Conventions (G2, G4, G5, G10, G11, G13): angles in arcsec, origin at the image
 * centre, native pixel (i, j) (i = row) centred at x = (j - (nx-1)/2) s, y = (i - (ny-1)/2) s,
 * row index increases with +y; phi is the major-axis direction counter-clockwise from +x;
 * shear taken about the image origin with the sign of Eq. 13; true convolution with the PSF
 * used as given (not renormalised, odd sizes only).
 *
 * Parameter row layout, P = 7 + 7*n_lens_light + 7*n_source floats:
 *   [0] theta_E  [1] e1  [2] e2  [3] cx  [4] cy          SIE (ellipticities: Eq. 11)
 *   [5] gamma1   [6] gamma2                               external shear
 *   [7] gamma                                             mass_model = TL_MASS_EPL only: the slope
 *                                                         of PAPER.md:158 Eq. 12 (then P is 8 + ...)
 *   then per Sersic component, lens light first, then sources:
 *   [+0] I_e  [+1] r_e  [+2] n  [+3] e1  [+4] e2  [+5] cx  [+6] cy
 *
 * Invalid rows are not errors: hypot(e1,e2) >= 1, theta_E < 0, r_e <= 0, n <= 0, a slope outside
 * 1 < gamma < 3, or any non-finite entry gives logL = -INFINITY and a NaN-filled image for that row.
 *
 * Threading: what tl_create builds (device copies of psf / data / noise, launch geometry, options)
 * never changes afterwards, and batch calls may be issued from several host threads / streams
 * concurrently: per-call scratch comes from a stream-ordered memory pool owned by the context.
 * The following state IS mutable and must only be changed while no call is in flight on the
 * context: the precision mode (tl_set_precision), the MGE Gaussian set (tl_set_mge), the
 * profiling switch and its event pair (tl_set_profiling: a single-thread benchmark facility),
 * and the staging slots of the asynchronous host entry (tl_loglike_batch_host_async / tl_wait:
 * one submitting thread per context).
 * A call made while another CUDA device is current switches to the context's device for its
 * duration and restores the caller's device before returning.
 */
#ifndef TINYLENS_H
#define TINYLENS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TL_OK       0
#define TL_EINVAL  -1   /* bad shape, even PSF size, null pointer, noise not finite/positive  */
#define TL_ENOMEM  -2   /* host or device allocation failed                                   */
#define TL_ECUDA   -3   /* no usable CUDA device, or a CUDA runtime call failed               */
#define TL_ESIZE   -4   /* configuration exceeds what the kernels support (see tl_create)     */

#define TL_PRECISION_FP32      0 /* default: the FP32 / MUFU kernels (DESIGN.md 6 "Precision design")        */
#define TL_PRECISION_FP64      1 /* every per-sample quantity in FP64, functions as hand-ordered            */
                                 /* polynomials (csrc/tl_dp.cuh): meets |dlogL| <= max(1e-3, 1e-6 |logL|)    */
                                 /* on every row, rows near the best fit included                            */
#define TL_PRECISION_FP64_LIBM 2 /* the same model with CUDA's double math library (csrc/tl_precise.cuh):   */
                                 /* slow; an independent check of the polynomial FP64 path                  */
#define TL_PRECISION_AUTO      3 /* FP32 for every row, then the rows whose first-order FP32 error bound    */
                                 /* exceeds the tolerance are re-evaluated in FP64 (rows near the best fit); */
                                 /* calls of at most half the SM count of rows are evaluated in FP64 outright */
                                 /* (faster there than the FP32 pass, which gives a row to one CTA)            */

#define TL_EDGE_EXTEND 0 /* evaluate the analytic model on a border of h = (K-1)/2 pixels so   */
                         /* every output pixel sees its full PSF support (Eq. 3 with only the  */
                         /* kernel truncated; G10)                                   */
#define TL_EDGE_ZERO   1 /* model taken as zero outside the cutout ('same' zero-padded conv)   */

#define TL_MASS_SIE 0 /* singular isothermal ellipsoid: Eq. 12 with gamma = 2        */
#define TL_MASS_EPL 1 /* elliptical power law, Eq. 12 with the slope gamma a parameter  */
                      /* of every row: kappa = (3-gamma)/2 (theta_E/R_p)^(gamma-1) on the ellipses   */
                      /* R_p of Eq. 10, deflection by the angular series of Tessore & Metcalf 2015   */
                      /* (G22).  gamma = 2 reproduces TL_MASS_SIE.                          */

typedef struct tl_ctx tl_ctx;     /* opaque; owned by the library */

typedef struct {
    int32_t ny, nx;          /* native image size (rows, columns)                              */
    double  pix_scale;       /* arcsec per native pixel, > 0                                   */
    int32_t supersample;     /* S >= 1: S x S samples per native pixel, S <= 16  */
    int32_t n_lens_light;    /* 0 or 1 Sersic components evaluated at theta (2: two MGE sets,  */
                             /* tl_set_mge_sets; such a context serves tl_loglike_mge_batch only) */
    int32_t n_source;        /* 1 or 2 Sersic components evaluated at beta                     */
    int32_t edge_mode;       /* TL_EDGE_EXTEND or TL_EDGE_ZERO                                 */
    int32_t n_lens;          /* 1, or L for a heterogeneous batch of L lenses (own psf, data,  */
                             /* noise per lens; row r of a B-row call belongs to lens          */
                             /* r / (B / L), B must be a multiple of L)                        */
    int32_t mass_model;      /* TL_MASS_SIE or TL_MASS_EPL                                     */
} tl_config;

/* What a context will launch; filled by tl_get_info (for benchmarks and reports).             */
typedef struct {
    int32_t n_params;          /* P                                                            */
    int32_t path;              /* 0 = fused (binned image in shared memory), 1 = split (binned  */
                               /*     image staged through global memory, for large images)    */
    int32_t block_threads;     /* threads per CTA of the dominant kernel                       */
    int32_t ctas_per_sm;       /* resident CTAs per SM of the dominant kernel                  */
    int32_t grid;              /* CTAs launched (persistent: n_sm * ctas_per_sm)                */
    int32_t smem_bytes;        /* dynamic shared memory per CTA                                */
    int32_t n_sm;              /* SMs of the device                                            */
    int32_t launches_per_call; /* kernels launched by one tl_loglike_batch                     */
    int64_t samples_per_row;   /* ray-traced sub-samples per likelihood                        */
    int64_t conv_fma_per_row;  /* K*K*ny*nx                                                    */
    double  logl_const;        /* lens 0:  sum_i ln(2 pi sigma_i^2)                            */
    double  sigma_min;         /* lens 0:  min_i sigma_i                                       */
    int32_t small_batch_rows;  /* calls with at most this many rows spread every row over many  */
                               /* CTAs (see tl_loglike_batch); 0 = never                        */
    int32_t chunk_rows;        /* a call with more rows is processed in chunks of this many     */
                               /* (one set of launches each, same stream)                       */
} tl_info;

/*
 * tl_create -- build a context (image d, noise sigma, PSF kernel K are
 * fixed per lens; only the parameter vector varies between evaluations).
 *   out        receives the handle (set to NULL on failure)
 *   cfg        see tl_config
 *   psf        HOST or DEVICE pointer, float [n_lens][psf_ny][psf_nx], psf_ny == psf_nx odd,
 *              row-major, K[a][b] with a the row (y) index.  Used as given.
 *   data       HOST or DEVICE pointer, float [n_lens][ny][nx], row-major (d_i of Eq. 5)
 *   noise      HOST or DEVICE pointer, float [n_lens][ny][nx], every value finite and > 0 (sigma_i)
 *              (device arrays are recognised with cudaPointerGetAttributes and staged through
 *              the host: 1/sigma^2 and the Eq. 5 constant are prepared there in FP64)
 *   cuda_stream  a cudaStream_t (NULL = default stream) on which uploads are enqueued;
 *              the call synchronises that stream before returning, so the host arrays may
 *              be freed immediately.
 * The arrays are copied; the caller keeps ownership of its buffers.  The context is bound to
 * the CUDA device current at the time of the call.
 * Returns TL_OK, TL_EINVAL, TL_ENOMEM, TL_ECUDA or TL_ESIZE (PSF larger than the image plus
 * halo allows, or a tile that cannot fit in 227 KB of shared memory).
 */
int tl_create(tl_ctx **out, const tl_config *cfg,
              const float *psf, int32_t psf_ny, int32_t psf_nx,
              const float *data, const float *noise, void *cuda_stream);

/*
 * tl_create_ex -- tl_create with explicit options (NULL = all automatic, which is tl_create).
 * These replace every environment variable the library once read; nothing in the library calls
 * getenv.  Zero-initialise the struct and set small_batch_rows = -1 for the defaults.
 */
typedef struct {
    int32_t small_batch_rows;   /* -1 automatic (half the SM count when the path supports it),  */
                                /*  0 never spread a row over several CTAs (every call runs the */
                                /*    fused kernel), > 0 calls of at most this many rows do      */
    int32_t force_split;        /* 1: stage the binned image through global memory (the large-  */
                                /*    image path) even when it fits in shared memory            */
    int32_t block_threads;      /* 0 automatic, else threads per CTA of the fused kernel        */
                                /*    (multiple of 32, 32..512)                                  */
    int32_t linear_staged;      /* 1: tl_loglike_linear_batch stages the component images       */
                                /*    through global memory even when the fused pipeline fits   */
    int64_t mge_chunk_rows;     /* 0 automatic, else an upper limit on rows per MGE chunk       */
    int64_t scratch_keep_bytes; /* 0 = 2 GiB: freed per-call scratch the context's memory pool  */
                                /*    keeps cached between calls                                */
    double  refine_tau;         /* 0 default, else the selective-FP64 threshold in units of     */
                                /*    sigma_min                                  */
    int32_t debug_canaries;     /* 1: every per-call scratch allocation carries 256 guard bytes */
                                /*    on either side, checked when it is freed, and starts      */
                                /*    filled with 0xFF (NaN / -1: a read of scratch that nobody */
                                /*    wrote shows in the results)                               */
                                /*    (tl_debug_canary_errors); a debugging aid, a few launches */
                                /*    more per call                                             */
    int32_t reserved;           /* 0                                                            */
} tl_options;
int tl_create_ex(tl_ctx **out, const tl_config *cfg,
                 const float *psf, int32_t psf_ny, int32_t psf_nx,
                 const float *data, const float *noise, const tl_options *opt, void *cuda_stream);

/* Number of floats per parameter row, P = 7 (8 for TL_MASS_EPL) + 7*n_lens_light + 7*n_source;
 * < 0 on NULL.                                                                                */
int tl_param_count(const tl_ctx *ctx);

/* Launch geometry and sizes of this context.  Returns TL_OK or TL_EINVAL.                     */
int tl_get_info(const tl_ctx *ctx, tl_info *info);

/*
 * tl_loglike_batch -- logL[r] (Eq. 5, normalisation included) for r = 0..B-1.
 * ACCURACY.  In the default TL_PRECISION_FP32 mode per-pixel values agree with an FP64 evaluation to
 * ~4e-7 of the image peak and logL to max(1e-3, 1e-6 |logL|) on rows far from the best fit (prior
 * draws), but NOT on rows near the best fit: there |delta logL| was measured at up to 23 x (Tiny),
 * 6.4 x (CSST-like), 2.4 x (HST-like), 2.6 x (survey) that tolerance, because 1e-3 absolute needs
 * every bright pixel to ~1e-8 relative.  TL_PRECISION_FP64 and TL_PRECISION_AUTO
 * (tl_set_precision) meet the tolerance on every row, at 0.32 x / 0.2-0.55 x the FP32 throughput.
 *   params     DEVICE pointer, float [B][P] row-major, caller-owned, read only
 *   B          rows (>= 0; multiple of n_lens)
 *   logL       DEVICE pointer, float [B], caller-owned, written
 *   cuda_stream  stream the kernels are enqueued on.  The call does NOT synchronise.
 * The result is bitwise reproducible (fixed-shape FP64 reduction, no atomics), and the value of a
 * row does not depend on the batch it is evaluated in: calls with few rows (at most
 * tl_info.small_batch_rows = half the SM count, "CPU<->GPU" round trips of a sampler
 * that proposes small batches) spread each row over many CTAs instead of one, 3 launches instead
 * of 2, and return the same bits as a large batch does; so do the rows of the last, mostly empty
 * wave of a larger batch (at most that many rows beyond a multiple of the persistent grid).
 */
int tl_loglike_batch(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream);

/*
 * tl_render_batch -- the blurred model images Im for every row.
 *   images     DEVICE pointer, float [B][ny][nx], caller-owned, written (NaN for invalid rows)
 * Same arithmetic as tl_loglike_batch up to and including the PSF convolution.
 */
int tl_render_batch(tl_ctx *ctx, const float *params, int64_t B, float *images, void *cuda_stream);

/*
 * Serve mode -- a persistent kernel for a sampler that proposes a handful of rows at a time (SURVEY.md 8(f)
 * NEXT-4; the CPU<->GPU round trips, not the likelihood, limit the pipeline).
 * tl_serve_start launches ONE kernel that occupies every SM of the device and polls a request block in pinned,
 * mapped host memory; tl_serve_eval writes the rows and a sequence number into that block and spins until the
 * kernel has written logL back: no cudaMemcpy, no kernel launch and no stream synchronisation per request.
 * The arithmetic is that of tl_loglike_batch (the same device functions in the same order): logL is bit for bit
 * what tl_loglike_batch returns for the same rows.
 *   tl_serve_start(ctx, max_rows, idle_timeout_s)
 *       max_rows        1 .. 16: the most rows one request may hold
 *       idle_timeout_s  (0, 300]: the kernel leaves by itself after this long without a request (and after 120 s
 *                       in any case); the next tl_serve_eval starts it again (one launch).  Every wait inside the
 *                       kernel is bounded in the same way, so a host that goes away cannot leave a spinning GPU.
 *       Contexts: FP32 precision, n_lens = 1, SIE mass model, even supersampling factor, fused path with a
 *       register-blocked PSF size (5, 15, 21, 31, 41); otherwise TL_EINVAL / TL_ESIZE.  Allocates the request
 *       block, per-row scratch for 16 rows and a stream of its own.  TL_EINVAL when already serving.
 *   tl_serve_eval(ctx, params_host, B, logL_host)
 *       params_host  HOST pointer, float [B][P] (need not be pinned: it is copied into the request block)
 *       B            1 .. max_rows
 *       logL_host    HOST pointer, float [B], written (-INFINITY for invalid rows)
 *       Blocking, one request at a time per context (not thread-safe).  TL_ECUDA when the kernel does not answer
 *       within 20 s.
 *   tl_serve_stop(ctx)  tells the kernel to leave, waits for it and frees what tl_serve_start allocated; also done
 *       by tl_destroy.  TL_OK when the context is not serving.
 * WHILE SERVING THE GPU IS TAKEN: kernels launched by anybody else on the device (tl_loglike_batch of this or another
 * context included) only start once the serving kernel has left, i.e. after tl_serve_stop or the idle timeout.
 */
int tl_serve_start(tl_ctx *ctx, int32_t max_rows, double idle_timeout_s);
int tl_serve_eval(tl_ctx *ctx, const float *params_host, int32_t B, float *logL_host);
int tl_serve_stop(tl_ctx *ctx);

/*
 * tl_loglike_batch_noalloc -- tl_loglike_batch (Eq. 5; same steps a0-a7, same kernels,
 * same bits) for callers that may not allocate: code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc.  tl_loglike_batch takes its per-call scratch -- the array of
 * per-row constants that the prologue kernel writes and the fused kernel reads, 1280 bytes per row --
 * from the context's stream-ordered memory pool; this call keeps it in a fixed array in the library's
 * device image instead (TL_NOALLOC_MAX_ROWS rows = 5 MiB, held by every GPU that loads the library
 * until the process exits) and calls no cudaMalloc, cudaFree, cudaMallocAsync, cudaFreeAsync or any
 * other allocating routine.
 *   params, logL, cuda_stream   as for tl_loglike_batch (DEVICE pointers, caller-owned; asynchronous)
 *   B          0 <= B <= TL_NOALLOC_MAX_ROWS, a multiple of n_lens.  B = 0 (params and logL may be NULL)
 *              only resolves the array's device address, which the first call on each device does once
 *              (cudaGetSymbolAddress: no allocation, but make that first call outside graph capture).
 * Returns TL_ESIZE when B > TL_NOALLOC_MAX_ROWS (split a larger batch into several calls on ONE stream)
 * or when the context runs the split path (images too large for one CTA's shared memory: that path
 * needs a binned image per row in global memory); TL_EINVAL for a NULL pointer with B > 0, for B not a
 * multiple of n_lens and for a context whose precision is not TL_PRECISION_FP32; TL_ECUDA as usual.
 * logL is bit for bit tl_loglike_batch's in TL_PRECISION_FP32 mode: every row goes through the fused
 * kernel, whose result the small-batch path of tl_loglike_batch reproduces bitwise.
 * SHARED STATE.  Every context and every call on a device shares the one array, which keeps the
 * contents of the last call; nothing in it has to start at zero (the prologue rewrites every field of
 * rows 0 .. B-1 that the fused kernel reads, and no other row is read).  Calls that can overlap on the
 * GPU -- different streams, or graph branches, without an ordering between them -- RACE on the array and
 * return garbage: order them (one stream, or events).  tl_loglike_batch has no such restriction.
 */
#define TL_NOALLOC_MAX_ROWS 4096
int tl_loglike_batch_noalloc(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream);

/*
 * tl_loglike_linear_batch -- the paper's linear/non-linear split (Eq. 6,
 * :97-129 Eq. 7): for every row the amplitudes s of the N_l + N_s light components are not
 * parameters but are solved as the non-negative least-squares minimiser of
 * || (M s - d) / sigma ||^2, M = B [L_l | L_s] (column k = blurred unit-amplitude image of
 * component k), and logL[r] is Eq. 5 at that optimum.  The I_e entries of the rows are ignored
 * (they may hold anything; a finite |I_e| > 1 is used only as a magnitude hint for the
 * precision refinement).
 *   params   DEVICE pointer, float [B][P], same layout as tl_loglike_batch
 *   logL     DEVICE pointer, float [B], written (-INFINITY for invalid rows)
 *   amps     DEVICE pointer, float [B][N_l + N_s] (lens light first, then sources), written
 *            (NaN for invalid rows), or NULL
 * Asynchronous on cuda_stream; bitwise reproducible.  Two pipelines with identical results
 * (bit for bit): fused (the component images of a row stay in shared memory; chosen when they
 * fit) and staged (component images through global memory; larger images, or
 * tl_options.linear_staged; also calls of at most half the SM count of rows, whose rows it spreads over
 * the whole GPU: 0.08 instead of 0.21 ms for one row of the CSST-like config).  chi^2 at the solved
 * amplitudes is d'Wd - 2 s'b + s'G s from the FP64 Gram quantities.  The NNLS problem is solved on the Gram matrix by the active-set
 * iteration of Bro & De Jong.  Returns TL_OK, TL_EINVAL, TL_ENOMEM, TL_ECUDA,
 * or TL_ESIZE when the PSF tile does not fit in shared memory.
 */
int tl_loglike_linear_batch(tl_ctx *ctx, const float *params, int64_t B, float *logL, float *amps,
                            void *cuda_stream);

/*
 * MGE lens light with linear amplitudes (section 4.3: "we have implemented the
 * Multiple Gaussian Expansion (MGE) model, which can describe arbitrary radial profiles ... in
 * lens galaxies"; the paper gives no formula -- reading G23 of DESIGN.md).  The lens light is
 *     I_l(theta) = sum_{k < n_gauss} a_k exp( -R_p(theta)^2 / (2 sigma_k^2) ),
 * R_p on the ellipses of PAPER.md:143-148 Eq. 10 with one centre and one (e1, e2) for the whole
 * set, fixed dispersions sigma_k, and the a_k >= 0 are linear parameters solved per row together
 * with the source amplitudes (PAPER.md:86-93 Eq. 6, :97-129 Eq. 7), as in
 * tl_loglike_linear_batch but with n_gauss + n_source columns.
 *
 * tl_set_mge -- define the Gaussian set of a context created with n_lens_light = 1.
 *   sigmas     HOST pointer, float [n_gauss], arcsec, finite and > 0 (copied)
 *   n_gauss    1 .. 30
 * Synchronous; not thread-safe with respect to calls in flight on the same context.  May be
 * called again to change the set.  TL_OK, TL_EINVAL (also: n_lens_light != 1), TL_ESIZE,
 * TL_ENOMEM or TL_ECUDA.
 *
 * tl_mge_columns -- n_gauss + n_source (the width of `amps`), or < 0 when no set is defined.
 * tl_mge_chunk_rows -- a call with more rows is processed in chunks of this many (six launches
 *   each, same stream; the blurred component images of a chunk are staged in <= 2 GiB of scratch
 *   from the context's stream-ordered pool; a call halves its chunk when the device cannot give
 *   that much); < 0 when no set is defined.
 *
 * tl_loglike_mge_batch -- logL[r] = Eq. 5 at the NNLS-optimal amplitudes of row r.
 *   params   DEVICE pointer, float [B][P], the context's usual row layout; of the lens-light
 *            block only e1, e2, cx, cy (entries +3..+6) are read -- its I_e, r_e, n and the
 *            I_e of the sources are ignored and may hold anything
 *   logL     DEVICE pointer, float [B], written (-INFINITY for invalid rows)
 *   amps     DEVICE pointer, float [B][n_gauss + n_source] (Gaussians in the order of sigmas,
 *            then sources), written (NaN for invalid rows), or NULL.  Neighbouring Gaussians are
 *            nearly collinear, so individual amplitudes are ill-conditioned; logL and the
 *            fitted image M s are not.
 * Asynchronous on cuda_stream; bitwise reproducible (fixed-order FP64 sums, no atomics).  The
 * NNLS problem is solved on the Gram matrix by the active-set iteration of Bro & De Jong
 * (PAPER.md:123-129).  Returns TL_OK, TL_EINVAL (no set defined, bad pointers, B not a
 * multiple of n_lens), TL_ENOMEM, TL_ECUDA or TL_ESIZE.
 */
int tl_set_mge(tl_ctx *ctx, const float *sigmas, int32_t n_gauss);
/*
 * tl_set_mge_sets -- several Gaussian sets, each with its own ellipticity, position angle and centre
 * ("isophote twists").  The context must have been created with n_lens_light =
 * n_sets (1 or 2): lens-light block j of the parameter row supplies (e1, e2, cx, cy) of set j (its
 * I_e, r_e, n are ignored).  A context with n_lens_light = 2 serves tl_loglike_mge_batch only (the
 * other batch calls return TL_EINVAL).
 *   sigmas      HOST pointer, float [sum_j n_per_set[j]]: the dispersions of set 0, then of set 1
 *   n_per_set   HOST pointer, int32 [n_sets], each >= 1; at most 30 Gaussians in total (the NNLS then
 *               has up to 30 + n_source <= 32 columns)
 * tl_set_mge(ctx, sigmas, n) is tl_set_mge_sets with one set.  Same return codes.
 */
int tl_set_mge_sets(tl_ctx *ctx, const float *sigmas, const int32_t *n_per_set, int32_t n_sets);
int tl_mge_columns(const tl_ctx *ctx);
int64_t tl_mge_chunk_rows(const tl_ctx *ctx);
int tl_loglike_mge_batch(tl_ctx *ctx, const float *params, int64_t B, float *logL, float *amps,
                         void *cuda_stream);

/*
 * tl_loglike_batch_host -- end-to-end convenience for a host-side sampler (PAPER.md:250 names
 * the CPU<->GPU transfers as part of the cost): copies params (HOST, float [B][P], ideally
 * pinned) to the device, runs tl_loglike_batch, copies logL back to logL (HOST, float [B]),
 * and synchronises the stream before returning.
 */
int tl_loglike_batch_host(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream);

/*
 * tl_loglike_batch_host_async / tl_wait -- the same end-to-end call, split so that a host-side
 * sampler can overlap its own work and the upload of the next batch with the kernels of the
 * current one (PAPER.md:250 names the CPU<->GPU transfers, :285 the CPU sampler, as the limit of
 * the whole pipeline).  The context owns two staging slots (pinned host + device buffers, grown on
 * demand and then reused: no allocation per call) and an upload and a download stream of its own.
 *   tl_loglike_batch_host_async
 *     params   HOST pointer, float [B][P]; copied into the slot's pinned buffer before the call
 *              returns, so the caller may reuse it at once
 *     B        rows (>= 1; multiple of n_lens)
 *     logL     HOST pointer, float [B]; written by tl_wait (must stay valid until then)
 *     cuda_stream  stream the kernels run on (the upload runs on the context's own stream and the
 *              kernels wait for it; the download waits for the kernels)
 *     returns the slot (0 or 1) to pass to tl_wait, or a negative error code.  Slots alternate; a
 *     submission that finds its slot still in flight first completes that earlier submission
 *     (its logL buffer is written), so at most two batches are in flight.
 *   tl_wait    blocks until the slot's batch is complete, copies its logL into the caller's buffer and
 *              frees the slot.  TL_OK, TL_EINVAL (slot not in flight) or TL_ECUDA.
 * One submitting thread per context.  tl_loglike_batch_host is submit + wait.
 */
int tl_loglike_batch_host_async(tl_ctx *ctx, const float *params, int64_t B, float *logL, void *cuda_stream);
int tl_wait(tl_ctx *ctx, int slot);

/*
 * tl_set_precision -- choose the arithmetic of later tl_loglike_batch / tl_render_batch /
 * tl_loglike_batch_host(_async) / tl_loglike_linear_batch / tl_loglike_mge_batch calls on this context.
 * In the two linear-amplitude calls both TL_PRECISION_FP64 and TL_PRECISION_AUTO run the FP64 pipeline
 * on every row (with solved amplitudes every row is near its best fit); TL_PRECISION_FP64_LIBM is the
 * FP32 pipeline there.
 *   TL_PRECISION_FP32 (default)  the FP32 kernels: meet the tolerances of DESIGN.md "Tolerances"
 *   TL_PRECISION_FP64            the same forward model in double precision on the device, about
 *                                ten times slower; agrees with an FP64 CPU evaluation to ~1e-9
 *                                relative, i.e. |delta logL| <= 1e-3 also where FP32 cannot
 *                                (rows near the best fit).  Results are still returned as float.
 * Not thread-safe with respect to calls in flight on the same context.  TL_OK or TL_EINVAL.
 */
int tl_set_precision(tl_ctx *ctx, int precision);

/*
 * Benchmark facility.  tl_set_profiling(ctx, 1) makes every later batch call record a pair of
 * CUDA events, on the call's stream, around its dominant kernel (fused path: the fused kernel;
 * split path: the ray-trace kernel) -- for a call that is split into several chunks, around the
 * last chunk's.  tl_last_kernel_ms waits for the second event and returns the elapsed device
 * time of that launch in milliseconds.  Not thread-safe: use one context per measuring thread.
 * Returns TL_OK, TL_EINVAL (no profiled call pending) or TL_ECUDA.
 */
int tl_set_profiling(tl_ctx *ctx, int enable);
int tl_last_kernel_ms(tl_ctx *ctx, float *ms);

/*
 * tl_measure_peaks -- issue-rate micro-benchmarks of the pipes that bound the hot path
 * (DESIGN.md 5.2 "Roofline that bounds it: plain ALU issue"; SURVEY.md 8(d) "verify by
 * micro-benchmark on the box before quoting"): scalar FFMA, packed FFMA2 (fma.rn.f32x2), MUFU,
 * DFMA and mixes of them, one persistent CTA of 1024 threads per SM on the current device.
 *   out        HOST pointer, tl_peak [n_max], written
 *   n_max      capacity of out (11 probes exist)
 *   seed_err4  HOST pointer, double [4], or NULL: worst relative error over [1, 4) of
 *              rcp.approx.f64, of one Newton step on it, of rsqrt.approx.f64, and of one Newton
 *              step on it (the seeds of the FP64 kernels' divisions and square roots)
 * Synchronous (default stream).  Returns the number of probes written (> 0), or TL_EINVAL,
 * TL_ENOMEM, TL_ECUDA.  `python bench.py --peaks` prints the table.
 */
typedef struct {
    char   name[64];           /* instruction mix of one loop trip                              */
    double inst_per_clk_sm;    /* thread-instructions issued per SM clock                       */
    double fma_per_clk_sm;     /* FMAs (FP32 or FP64) retired per SM clock in that mix          */
    double sm_mhz;             /* SM clock the probe ran at (cycles / event time)               */
    double ms;                 /* duration of the probe kernel                                  */
} tl_peak;
int tl_measure_peaks(tl_peak *out, int32_t n_max, double *seed_err4);

/*
 * Guard-word check of the library's scratch memory (compute-sanitizer is not available everywhere): a context
 * created with tl_options.debug_canaries = 1 surrounds every per-call scratch allocation with 256 bytes of
 * 0xA5 and, when the allocation is freed (stream-ordered, at the end of the call), counts the guard words that
 * changed.  tl_debug_canary_errors synchronises the device and returns that count (0 = no kernel of any call so
 * far wrote outside its scratch buffers); tl_debug_canary_selftest writes one word on either side of a test
 * allocation on purpose and returns TL_OK when both hits are counted (the counter is reset afterwards).
 * TL_EINVAL for a context without the option.
 */
int tl_debug_canary_errors(tl_ctx *ctx, int64_t *count);
int tl_debug_canary_selftest(tl_ctx *ctx);

/* Release a context and its device memory (NULL is allowed).                                  */
void tl_destroy(tl_ctx *ctx);

/* Static, never-NULL description of a return code.                                            */
const char *tl_strerror(int code);

/* Library version string, e.g. "tinylens-b200 0.1 (sm_100a)".                                 */
const char *tl_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TINYLENS_H */
