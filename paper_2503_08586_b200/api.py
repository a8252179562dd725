"""Thin Python binding of the C ABI in include/tinylens.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/; PyTorch supplies device memory and
streams.  There is no CPU fallback: if the shared library is missing or no CUDA device is
usable, the calls raise ``TinyLensError``.

The functions carry the C names (``tl_create`` ...); ``LensContext`` is a small RAII wrapper.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("TL_LIB") or os.path.join(_HERE, "libtinylens.so")   # TL_LIB: experiments only

TL_OK, TL_EINVAL, TL_ENOMEM, TL_ECUDA, TL_ESIZE = 0, -1, -2, -3, -4
TL_EDGE_EXTEND, TL_EDGE_ZERO = 0, 1
TL_PRECISION_FP32, TL_PRECISION_FP64, TL_PRECISION_FP64_LIBM, TL_PRECISION_AUTO = 0, 1, 2, 3
TL_MASS_SIE, TL_MASS_EPL = 0, 1


class TinyLensError(RuntimeError):
    def __init__(self, code: int, what: str = ""):
        self.code = code
        msg = tl_strerror(code) if _lib is not None else "library not loaded"
        super().__init__("%s: %s (code %d)" % (what, msg, code))


class tl_config(C.Structure):
    _fields_ = [("ny", C.c_int32), ("nx", C.c_int32), ("pix_scale", C.c_double),
                ("supersample", C.c_int32), ("n_lens_light", C.c_int32), ("n_source", C.c_int32),
                ("edge_mode", C.c_int32), ("n_lens", C.c_int32), ("mass_model", C.c_int32)]


class tl_info(C.Structure):
    _fields_ = [("n_params", C.c_int32), ("path", C.c_int32), ("block_threads", C.c_int32),
                ("ctas_per_sm", C.c_int32), ("grid", C.c_int32), ("smem_bytes", C.c_int32),
                ("n_sm", C.c_int32), ("launches_per_call", C.c_int32),
                ("samples_per_row", C.c_int64), ("conv_fma_per_row", C.c_int64),
                ("logl_const", C.c_double), ("sigma_min", C.c_double),
                ("small_batch_rows", C.c_int32), ("chunk_rows", C.c_int32)]


class tl_options(C.Structure):
    _fields_ = [("small_batch_rows", C.c_int32), ("force_split", C.c_int32), ("block_threads", C.c_int32),
                ("linear_staged", C.c_int32), ("mge_chunk_rows", C.c_int64), ("scratch_keep_bytes", C.c_int64),
                ("refine_tau", C.c_double), ("debug_canaries", C.c_int32), ("reserved", C.c_int32)]


class tl_peak(C.Structure):
    _fields_ = [("name", C.c_char * 64), ("inst_per_clk_sm", C.c_double), ("fma_per_clk_sm", C.c_double),
                ("sm_mhz", C.c_double), ("ms", C.c_double)]


_lib = None


def load(build_if_missing: bool = True):
    """dlopen libtinylens.so (building it in-tree with nvcc when it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and not os.environ.get("TL_LIB"):
        from . import build as _build
        try:
            _build.build()
        except Exception:
            if not os.path.exists(LIB_PATH):
                raise
    if not os.path.exists(LIB_PATH):
        raise OSError("libtinylens.so not found at %s: run `python -m paper_2503_08586_b200.build`" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, fp = C.c_void_p, C.c_int32, C.c_int64, C.POINTER(C.c_float)
    L.tl_create.restype = C.c_int
    L.tl_create.argtypes = [C.POINTER(vp), C.POINTER(tl_config), fp, i32, i32, fp, fp, vp]
    L.tl_create_ex.restype = C.c_int
    L.tl_create_ex.argtypes = [C.POINTER(vp), C.POINTER(tl_config), vp, i32, i32, vp, vp, C.POINTER(tl_options), vp]
    L.tl_param_count.restype = C.c_int; L.tl_param_count.argtypes = [vp]
    L.tl_get_info.restype = C.c_int; L.tl_get_info.argtypes = [vp, C.POINTER(tl_info)]
    L.tl_loglike_batch.restype = C.c_int; L.tl_loglike_batch.argtypes = [vp, vp, i64, vp, vp]
    L.tl_render_batch.restype = C.c_int; L.tl_render_batch.argtypes = [vp, vp, i64, vp, vp]
    L.tl_debug_canary_errors.restype = C.c_int; L.tl_debug_canary_errors.argtypes = [vp, C.POINTER(i64)]
    L.tl_debug_canary_selftest.restype = C.c_int; L.tl_debug_canary_selftest.argtypes = [vp]
    L.tl_serve_start.restype = C.c_int; L.tl_serve_start.argtypes = [vp, i32, C.c_double]
    L.tl_serve_eval.restype = C.c_int; L.tl_serve_eval.argtypes = [vp, vp, i32, vp]
    L.tl_serve_stop.restype = C.c_int; L.tl_serve_stop.argtypes = [vp]
    L.tl_loglike_batch_noalloc.restype = C.c_int; L.tl_loglike_batch_noalloc.argtypes = [vp, vp, i64, vp, vp]
    L.tl_loglike_batch_host.restype = C.c_int; L.tl_loglike_batch_host.argtypes = [vp, vp, i64, vp, vp]
    L.tl_loglike_batch_host_async.restype = C.c_int; L.tl_loglike_batch_host_async.argtypes = [vp, vp, i64, vp, vp]
    L.tl_wait.restype = C.c_int; L.tl_wait.argtypes = [vp, C.c_int]
    L.tl_loglike_linear_batch.restype = C.c_int; L.tl_loglike_linear_batch.argtypes = [vp, vp, i64, vp, vp, vp]
    L.tl_set_mge.restype = C.c_int; L.tl_set_mge.argtypes = [vp, fp, i32]
    L.tl_set_mge_sets.restype = C.c_int; L.tl_set_mge_sets.argtypes = [vp, fp, C.POINTER(i32), i32]
    L.tl_mge_columns.restype = C.c_int; L.tl_mge_columns.argtypes = [vp]
    L.tl_mge_chunk_rows.restype = i64; L.tl_mge_chunk_rows.argtypes = [vp]
    L.tl_loglike_mge_batch.restype = C.c_int; L.tl_loglike_mge_batch.argtypes = [vp, vp, i64, vp, vp, vp]
    L.tl_set_precision.restype = C.c_int; L.tl_set_precision.argtypes = [vp, C.c_int]
    L.tl_set_profiling.restype = C.c_int; L.tl_set_profiling.argtypes = [vp, C.c_int]
    L.tl_last_kernel_ms.restype = C.c_int; L.tl_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.tl_measure_peaks.restype = C.c_int; L.tl_measure_peaks.argtypes = [C.POINTER(tl_peak), i32, C.POINTER(C.c_double)]
    L.tl_destroy.restype = None; L.tl_destroy.argtypes = [vp]
    L.tl_strerror.restype = C.c_char_p; L.tl_strerror.argtypes = [C.c_int]
    L.tl_version.restype = C.c_char_p; L.tl_version.argtypes = []
    _lib = L
    return L


def tl_strerror(code: int) -> str:
    return load().tl_strerror(int(code)).decode()


def tl_version() -> str:
    return load().tl_version().decode()


def _check(code: int, what: str):
    if code != TL_OK:
        raise TinyLensError(code, what)


def _stream_handle(stream) -> int:
    """cudaStream_t of a torch stream (None = torch's current stream)."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _f32c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _host_or_device(a):
    """numpy array / host tensor -> (keep-alive, pointer, size, last two dims); CUDA float32 tensors are passed as they are."""
    try:
        import torch
        if isinstance(a, torch.Tensor) and a.is_cuda:
            if a.dtype != torch.float32 or not a.is_contiguous():
                raise TinyLensError(TL_EINVAL, "tl_create (device arrays must be contiguous float32)")
            return a, a.data_ptr(), a.numel(), tuple(a.shape[-2:])
        if isinstance(a, torch.Tensor):
            a = a.numpy()
    except ImportError:
        pass
    h = _f32c(a)
    return h, h.ctypes.data, h.size, tuple(h.shape[-2:])


def tl_create(ny, nx, pix_scale, supersample, n_lens_light, n_source, psf, data, noise,
              edge_mode=TL_EDGE_EXTEND, n_lens=1, stream=None, mass_model=TL_MASS_SIE, options=None) -> int:
    """-> opaque handle (int).  psf [n_lens,K,K], data/noise [n_lens,ny,nx]: host float32 arrays or CUDA
    float32 tensors.  options: dict of tl_options fields (tl_create_ex), e.g. {"small_batch_rows": 0}."""
    L = load()
    (pk, pp, pn, pshape), (dk, dp_, dn, _), (sk, sp, sn, _) = _host_or_device(psf), _host_or_device(data), _host_or_device(noise)
    K = pshape[-1]
    if pn != n_lens * K * K or pshape[-2] != K:
        raise TinyLensError(TL_EINVAL, "tl_create (psf shape)")
    if dn != n_lens * ny * nx or sn != n_lens * ny * nx:
        raise TinyLensError(TL_EINVAL, "tl_create (data/noise shape)")
    cfg = tl_config(int(ny), int(nx), float(pix_scale), int(supersample), int(n_lens_light),
                    int(n_source), int(edge_mode), int(n_lens), int(mass_model))
    h = C.c_void_p()
    sh = 0
    try:
        import torch
        if torch.cuda.is_available():
            sh = _stream_handle(stream)
    except ImportError:
        pass
    opt = tl_options(small_batch_rows=-1)
    for k, v in (options or {}).items():
        if k not in dict(tl_options._fields_):
            raise TinyLensError(TL_EINVAL, "tl_create (unknown option %r)" % k)
        setattr(opt, k, v)
    _check(L.tl_create_ex(C.byref(h), C.byref(cfg), pp, K, K, dp_, sp, C.byref(opt), sh), "tl_create_ex")
    del pk, dk, sk
    return h.value


def tl_param_count(handle: int) -> int:
    return load().tl_param_count(handle)


def tl_get_info(handle: int) -> dict:
    info = tl_info()
    _check(load().tl_get_info(handle, C.byref(info)), "tl_get_info")
    return {k: getattr(info, k) for k, _ in tl_info._fields_}


def _dev_rows(handle, params):
    import torch
    P = tl_param_count(handle)
    if not (isinstance(params, torch.Tensor) and params.is_cuda and params.dtype == torch.float32
            and params.is_contiguous() and params.dim() == 2 and params.shape[1] == P):
        raise TinyLensError(TL_EINVAL, "params must be a contiguous CUDA float32 tensor [B, %d]" % P)
    return params.shape[0]


def _check_out(t, shape, device, what):
    """A caller-supplied result tensor must be a contiguous CUDA float32 tensor of exactly the shape the kernels write."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == device and t.dtype == torch.float32
            and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise TinyLensError(TL_EINVAL, "%s must be a contiguous CUDA float32 tensor of shape %s on %s" % (what, tuple(shape), device))


def tl_loglike_batch(handle: int, params, out=None, stream=None):
    """params: CUDA float32 [B,P] -> logL CUDA float32 [B] (enqueued on `stream`, no sync)."""
    import torch
    B = _dev_rows(handle, params)
    if out is None:
        out = torch.empty(B, dtype=torch.float32, device=params.device)
    else:
        _check_out(out, (B,), params.device, "out")
    _check(load().tl_loglike_batch(handle, params.data_ptr(), B, out.data_ptr(), _stream_handle(stream)),
           "tl_loglike_batch")
    return out


TL_NOALLOC_MAX_ROWS = 4096


def tl_serve_start(handle: int, max_rows: int = 16, idle_timeout_s: float = 2.0):
    """Launch the persistent serving kernel (include/tinylens.h): the GPU is taken until tl_serve_stop / the timeout."""
    _check(load().tl_serve_start(handle, int(max_rows), float(idle_timeout_s)), "tl_serve_start")


def tl_serve_eval(handle: int, params_host, out_host=None):
    """params_host: numpy float32 [B,P] (B <= max_rows) -> logL numpy float32 [B], through the serving kernel."""
    p = np.ascontiguousarray(params_host, dtype=np.float32)
    if p.ndim != 2:
        raise TinyLensError(TL_EINVAL, "params_host must be [B, P]")
    if out_host is None:
        out_host = np.empty(p.shape[0], np.float32)
    if out_host.dtype != np.float32 or out_host.shape != (p.shape[0],) or not out_host.flags["C_CONTIGUOUS"]:
        raise TinyLensError(TL_EINVAL, "out_host must be a contiguous float32 array of shape (B,)")
    _check(load().tl_serve_eval(handle, p.ctypes.data, p.shape[0], out_host.ctypes.data), "tl_serve_eval")
    return out_host


def tl_serve_stop(handle: int):
    _check(load().tl_serve_stop(handle), "tl_serve_stop")


def tl_loglike_batch_noalloc(handle: int, params, out, stream=None):
    """tl_loglike_batch without any allocation in the library (include/tinylens.h): params CUDA float32
    [B,P], B <= TL_NOALLOC_MAX_ROWS, written into the caller's `out` (CUDA float32 [B]).  Calls that can
    overlap on the GPU race on the library's fixed scratch array: keep them on one stream."""
    B = _dev_rows(handle, params)
    _check_out(out, (B,), params.device, "out")
    code = load().tl_loglike_batch_noalloc(handle, params.data_ptr(), B, out.data_ptr(), _stream_handle(stream))
    if code == TL_ESIZE and B > TL_NOALLOC_MAX_ROWS:
        raise TinyLensError(code, "tl_loglike_batch_noalloc: B = %d exceeds TL_NOALLOC_MAX_ROWS = %d (split the batch "
                            "into several calls on one stream)" % (B, TL_NOALLOC_MAX_ROWS))
    _check(code, "tl_loglike_batch_noalloc")
    return out


def tl_render_batch(handle: int, params, ny: int, nx: int, out=None, stream=None):
    """params: CUDA float32 [B,P] -> images CUDA float32 [B,ny,nx]."""
    import torch
    B = _dev_rows(handle, params)
    if out is None:
        out = torch.empty((B, ny, nx), dtype=torch.float32, device=params.device)
    else:
        _check_out(out, (B, ny, nx), params.device, "out")
    _check(load().tl_render_batch(handle, params.data_ptr(), B, out.data_ptr(), _stream_handle(stream)),
           "tl_render_batch")
    return out


def tl_loglike_linear_batch(handle: int, params, n_comp: int, out=None, amps=None, want_amps=True, stream=None):
    """params: CUDA float32 [B,P] -> (logL CUDA float32 [B], amplitudes CUDA float32 [B,n_comp] or None)."""
    import torch
    B = _dev_rows(handle, params)
    if out is None:
        out = torch.empty(B, dtype=torch.float32, device=params.device)
    else:
        _check_out(out, (B,), params.device, "out")
    if amps is None and want_amps:
        amps = torch.empty((B, n_comp), dtype=torch.float32, device=params.device)
    elif amps is not None:
        _check_out(amps, (B, n_comp), params.device, "amps")
    _check(load().tl_loglike_linear_batch(handle, params.data_ptr(), B, out.data_ptr(),
                                          amps.data_ptr() if amps is not None else None, _stream_handle(stream)),
           "tl_loglike_linear_batch")
    return out, amps


def tl_set_mge(handle: int, sigmas):
    """sigmas: host float32 [n_gauss] (arcsec) -- the Gaussian set of the MGE lens light."""
    sg = _f32c(sigmas).reshape(-1)
    _check(load().tl_set_mge(handle, sg.ctypes.data_as(C.POINTER(C.c_float)), int(sg.size)), "tl_set_mge")


def tl_set_mge_sets(handle: int, sigma_sets):
    """sigma_sets: list of 1-D float arrays (arcsec), one per Gaussian set; set j takes its shape and centre
    from lens-light block j of the parameter rows (the context's n_lens_light must equal len(sigma_sets))."""
    sets = [_f32c(sg).reshape(-1) for sg in sigma_sets]
    allsg = np.concatenate(sets)
    per = (C.c_int32 * len(sets))(*[int(sg.size) for sg in sets])
    _check(load().tl_set_mge_sets(handle, allsg.ctypes.data_as(C.POINTER(C.c_float)), per, len(sets)), "tl_set_mge_sets")


def tl_mge_columns(handle: int) -> int:
    return load().tl_mge_columns(handle)


def tl_mge_chunk_rows(handle: int) -> int:
    return int(load().tl_mge_chunk_rows(handle))


def tl_loglike_mge_batch(handle: int, params, out=None, amps=None, want_amps=True, stream=None):
    """params: CUDA float32 [B,P] -> (logL CUDA float32 [B], amplitudes CUDA float32 [B,n_gauss+n_source] or None)."""
    import torch
    B = _dev_rows(handle, params)
    n_col = tl_mge_columns(handle)
    if n_col < 0:
        raise TinyLensError(TL_EINVAL, "tl_loglike_mge_batch (no Gaussian set: call tl_set_mge)")
    if out is None:
        out = torch.empty(B, dtype=torch.float32, device=params.device)
    else:
        _check_out(out, (B,), params.device, "out")
    if amps is None and want_amps:
        amps = torch.empty((B, n_col), dtype=torch.float32, device=params.device)
    elif amps is not None:
        _check_out(amps, (B, n_col), params.device, "amps")
    _check(load().tl_loglike_mge_batch(handle, params.data_ptr(), B, out.data_ptr(),
                                       amps.data_ptr() if amps is not None else None, _stream_handle(stream)),
           "tl_loglike_mge_batch")
    return out, amps


def tl_loglike_batch_host(handle: int, params_host, out_host=None, stream=None):
    """params_host: host float32 [B,P] (torch CPU tensor, ideally pinned, or numpy) -> host logL [B].
    Host->device copy, kernels, device->host copy and a stream synchronise, all inside the call."""
    import torch
    P = tl_param_count(handle)
    if isinstance(params_host, np.ndarray):
        params_host = torch.from_numpy(_f32c(params_host))
    if params_host.is_cuda or params_host.dtype != torch.float32 or not params_host.is_contiguous() \
            or params_host.dim() != 2 or params_host.shape[1] != P:
        raise TinyLensError(TL_EINVAL, "params_host must be a contiguous host float32 tensor [B, %d]" % P)
    B = params_host.shape[0]
    if out_host is None:
        out_host = torch.empty(B, dtype=torch.float32, pin_memory=True)
    _check(load().tl_loglike_batch_host(handle, params_host.data_ptr(), B, out_host.data_ptr(),
                                        _stream_handle(stream)), "tl_loglike_batch_host")
    return out_host


def _host_rows(handle, params_host):
    import torch
    P = tl_param_count(handle)
    if isinstance(params_host, np.ndarray):
        params_host = torch.from_numpy(_f32c(params_host))
    if params_host.is_cuda or params_host.dtype != torch.float32 or not params_host.is_contiguous() \
            or params_host.dim() != 2 or params_host.shape[1] != P:
        raise TinyLensError(TL_EINVAL, "params_host must be a contiguous host float32 tensor [B, %d]" % P)
    return params_host


def tl_loglike_batch_host_async(handle: int, params_host, out_host, stream=None) -> int:
    """Submit one batch (host float32 [B,P]); out_host (host float32 [B]) is written by tl_wait(slot) and must
    stay alive until then.  Returns the slot."""
    import torch
    params_host = _host_rows(handle, params_host)
    B = params_host.shape[0]
    if not (isinstance(out_host, torch.Tensor) and not out_host.is_cuda and out_host.dtype == torch.float32
            and out_host.is_contiguous() and out_host.numel() == B):
        raise TinyLensError(TL_EINVAL, "out_host must be a contiguous host float32 tensor [B]")
    slot = load().tl_loglike_batch_host_async(handle, params_host.data_ptr(), B, out_host.data_ptr(), _stream_handle(stream))
    if slot < 0:
        raise TinyLensError(slot, "tl_loglike_batch_host_async")
    return slot


def tl_wait(handle: int, slot: int):
    _check(load().tl_wait(handle, int(slot)), "tl_wait")


def tl_set_precision(handle: int, precision: int):
    _check(load().tl_set_precision(handle, int(precision)), "tl_set_precision")


def tl_set_profiling(handle: int, enable: bool):
    _check(load().tl_set_profiling(handle, 1 if enable else 0), "tl_set_profiling")


def tl_last_kernel_ms(handle: int) -> float:
    ms = C.c_float()
    _check(load().tl_last_kernel_ms(handle, C.byref(ms)), "tl_last_kernel_ms")
    return float(ms.value)


def tl_measure_peaks():
    """-> (list of dicts, one per probe; [rcp seed, rcp + Newton, rsqrt seed, rsqrt + Newton] worst relative errors)."""
    arr = (tl_peak * 16)()
    err = (C.c_double * 4)()
    n = load().tl_measure_peaks(arr, 16, err)
    if n < 0:
        raise TinyLensError(n, "tl_measure_peaks")
    return ([{"name": arr[i].name.decode(), "inst_per_clk_sm": arr[i].inst_per_clk_sm, "fma_per_clk_sm": arr[i].fma_per_clk_sm,
              "sm_mhz": arr[i].sm_mhz, "ms": arr[i].ms} for i in range(n)], [float(x) for x in err])


def tl_destroy(handle: Optional[int]):
    if handle:
        load().tl_destroy(handle)


class LensContext:
    """RAII wrapper: ``ctx = LensContext.from_problem(problem); ctx.loglike(params)``."""

    def __init__(self, ny, nx, pix_scale, supersample, n_lens_light, n_source, psf, data, noise,
                 edge_mode=TL_EDGE_EXTEND, n_lens=1, stream=None, mass_model=TL_MASS_SIE, options=None):
        self.ny, self.nx, self.n_lens = int(ny), int(nx), int(n_lens)
        self.n_comp = int(n_lens_light) + int(n_source)
        self.handle = tl_create(ny, nx, pix_scale, supersample, n_lens_light, n_source, psf, data,
                                noise, edge_mode, n_lens, stream, mass_model, options)
        self.n_params = tl_param_count(self.handle)

    @classmethod
    def from_problem(cls, prob, stream=None, options=None):
        w = prob.workload
        return cls(w.ny, w.nx, w.pix_scale, w.supersample, w.n_lens_light, w.n_source,
                   prob.psf, prob.data, prob.noise, w.edge_mode, w.n_lens, stream,
                   getattr(w, "mass_model", TL_MASS_SIE), options)

    def info(self) -> dict:
        return tl_get_info(self.handle)

    def loglike(self, params, out=None, stream=None):
        return tl_loglike_batch(self.handle, params, out, stream)

    def canary_errors(self) -> int:
        """Guard words of the scratch allocations found changed so far (contexts created with options={"debug_canaries": 1})."""
        n = C.c_int64(0)
        _check(load().tl_debug_canary_errors(self.handle, C.byref(n)), "tl_debug_canary_errors")
        return int(n.value)

    def canary_selftest(self):
        _check(load().tl_debug_canary_selftest(self.handle), "tl_debug_canary_selftest")

    def serve_start(self, max_rows=16, idle_timeout_s=2.0):
        tl_serve_start(self.handle, max_rows, idle_timeout_s)

    def serve_eval(self, params_host, out_host=None):
        return tl_serve_eval(self.handle, params_host, out_host)

    def serve_stop(self):
        tl_serve_stop(self.handle)

    def loglike_noalloc(self, params, out, stream=None):
        return tl_loglike_batch_noalloc(self.handle, params, out, stream)

    def render(self, params, out=None, stream=None):
        return tl_render_batch(self.handle, params, self.ny, self.nx, out, stream)

    def loglike_linear(self, params, out=None, amps=None, want_amps=True, stream=None):
        return tl_loglike_linear_batch(self.handle, params, self.n_comp, out, amps, want_amps, stream)

    def set_mge(self, sigmas):
        tl_set_mge(self.handle, sigmas)

    def set_mge_sets(self, sigma_sets):
        tl_set_mge_sets(self.handle, sigma_sets)

    def loglike_mge(self, params, out=None, amps=None, want_amps=True, stream=None):
        return tl_loglike_mge_batch(self.handle, params, out, amps, want_amps, stream)

    def loglike_host(self, params_host, out_host=None, stream=None):
        return tl_loglike_batch_host(self.handle, params_host, out_host, stream)

    def loglike_host_async(self, params_host, out_host, stream=None) -> int:
        slot = tl_loglike_batch_host_async(self.handle, params_host, out_host, stream)
        self._pending = getattr(self, "_pending", {})
        self._pending[slot] = out_host                  # keeps the result buffer alive until wait()
        return slot

    def wait(self, slot: int):
        tl_wait(self.handle, slot)
        return getattr(self, "_pending", {}).pop(slot, None)

    def set_precision(self, precision: int):
        tl_set_precision(self.handle, precision)

    def set_profiling(self, enable: bool = True):
        tl_set_profiling(self.handle, enable)

    def last_kernel_ms(self) -> float:
        return tl_last_kernel_ms(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            tl_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
