"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/tinylens.h declares, validates arguments before touching CUDA, and fails loudly (no
CPU fallback) when no device is usable.  No compute calls are made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tinylens.h")


@pytest.fixture(scope="module")
def api():
    from paper_2503_08586_b200 import api as _api
    _api.load()
    return _api


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tl_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for need in ("tl_create", "tl_render_batch", "tl_loglike_batch", "tl_destroy", "tl_param_count",
                 "tl_strerror"):
        assert need in names


def test_library_exports_every_declared_symbol(api):
    lib = C.CDLL(api.LIB_PATH)
    for name in _declared_functions():
        assert hasattr(lib, name), "libtinylens.so does not export %s" % name


def test_no_torch_types_in_signatures():
    src = open(HEADER).read()
    assert "torch" not in src.lower().replace("pytorch tensors", "")
    assert "at::" not in src and "Tensor" not in src


def test_strerror_and_version(api):
    for code in (0, -1, -2, -3, -4, -99):
        s = api.tl_strerror(code)
        assert isinstance(s, str) and len(s) > 0
    assert "no CPU fallback" in api.tl_strerror(api.TL_ECUDA)
    assert "sm_100a" in api.tl_version()


def _args(ny=8, nx=8, K=3, L=1):
    psf = np.full((L, K, K), 1.0 / (K * K), np.float32)
    data = np.zeros((L, ny, nx), np.float32)
    noise = np.ones((L, ny, nx), np.float32)
    return psf, data, noise


def test_create_rejects_bad_arguments_before_cuda(api):
    psf, data, noise = _args()
    bad = [
        dict(ny=0), dict(nx=-1), dict(pix_scale=0.0), dict(pix_scale=float("nan")), dict(supersample=0),
        dict(supersample=17), dict(n_lens_light=3), dict(n_lens_light=-1), dict(n_source=0), dict(n_source=3), dict(edge_mode=2),
        dict(n_lens=0), dict(mass_model=2), dict(mass_model=-1),
    ]
    base = dict(ny=8, nx=8, pix_scale=0.1, supersample=2, n_lens_light=0, n_source=1, edge_mode=0, n_lens=1,
                mass_model=0)
    lib = api.load()
    fp = C.POINTER(C.c_float)
    for b in bad:
        kw = dict(base); kw.update(b)
        cfg = api.tl_config(kw["ny"], kw["nx"], kw["pix_scale"], kw["supersample"], kw["n_lens_light"],
                            kw["n_source"], kw["edge_mode"], kw["n_lens"], kw["mass_model"])
        h = C.c_void_p(123)
        rc = lib.tl_create(C.byref(h), C.byref(cfg), psf.ctypes.data_as(fp), 3, 3,
                           data.ctypes.data_as(fp), noise.ctypes.data_as(fp), None)
        assert rc == api.TL_EINVAL, (b, rc)
        assert h.value is None
    cfg = api.tl_config(8, 8, 0.1, 2, 0, 1, 0, 1)
    h = C.c_void_p()
    # even PSF, non-square PSF
    p4 = np.ones((1, 4, 4), np.float32)
    assert lib.tl_create(C.byref(h), C.byref(cfg), p4.ctypes.data_as(fp), 4, 4, data.ctypes.data_as(fp),
                         noise.ctypes.data_as(fp), None) == api.TL_EINVAL
    assert lib.tl_create(C.byref(h), C.byref(cfg), psf.ctypes.data_as(fp), 3, 5, data.ctypes.data_as(fp),
                         noise.ctypes.data_as(fp), None) == api.TL_EINVAL
    # null pointers
    assert lib.tl_create(C.byref(h), C.byref(cfg), None, 3, 3, data.ctypes.data_as(fp),
                         noise.ctypes.data_as(fp), None) == api.TL_EINVAL
    assert lib.tl_create(None, C.byref(cfg), psf.ctypes.data_as(fp), 3, 3, data.ctypes.data_as(fp),
                         noise.ctypes.data_as(fp), None) == api.TL_EINVAL
    # noise must be finite and > 0
    for v in (0.0, -1.0, float("inf"), float("nan")):
        n2 = noise.copy(); n2[0, 3, 3] = v
        assert lib.tl_create(C.byref(h), C.byref(cfg), psf.ctypes.data_as(fp), 3, 3, data.ctypes.data_as(fp),
                             n2.ctypes.data_as(fp), None) == api.TL_EINVAL


def test_null_context_calls_are_errors_not_crashes(api):
    lib = api.load()
    assert lib.tl_param_count(None) < 0
    info = api.tl_info()
    assert lib.tl_get_info(None, C.byref(info)) == api.TL_EINVAL
    assert lib.tl_loglike_batch(None, None, 4, None, None) == api.TL_EINVAL
    assert lib.tl_render_batch(None, None, 4, None, None) == api.TL_EINVAL
    assert lib.tl_loglike_batch_host(None, None, 4, None, None) == api.TL_EINVAL
    assert lib.tl_loglike_linear_batch(None, None, 4, None, None, None) == api.TL_EINVAL
    # MGE entry points (NEXT-3)
    sg = np.array([0.1, 0.3], np.float32)
    assert lib.tl_set_mge(None, sg.ctypes.data_as(C.POINTER(C.c_float)), 2) == api.TL_EINVAL
    per = (C.c_int32 * 2)(1, 1)
    assert lib.tl_set_mge_sets(None, sg.ctypes.data_as(C.POINTER(C.c_float)), per, 2) == api.TL_EINVAL
    assert lib.tl_mge_columns(None) < 0
    assert lib.tl_mge_chunk_rows(None) < 0
    assert lib.tl_loglike_mge_batch(None, None, 4, None, None, None) == api.TL_EINVAL
    lib.tl_destroy(None)


def test_create_ex_validates_options_before_cuda(api):
    psf, data, noise = _args()
    lib = api.load()
    cfg = api.tl_config(8, 8, 0.1, 2, 0, 1, 0, 1, 0)
    for bad in (dict(small_batch_rows=-2), dict(block_threads=48), dict(block_threads=1024), dict(mge_chunk_rows=-1),
                dict(scratch_keep_bytes=-5), dict(refine_tau=-1.0), dict(refine_tau=float("nan"))):
        opt = api.tl_options(small_batch_rows=-1)
        for k, v in bad.items():
            setattr(opt, k, v)
        h = C.c_void_p(1)
        rc = lib.tl_create_ex(C.byref(h), C.byref(cfg), psf.ctypes.data, 3, 3, data.ctypes.data, noise.ctypes.data,
                              C.byref(opt), None)
        assert rc == api.TL_EINVAL and h.value is None, bad
    with pytest.raises(api.TinyLensError):
        api.tl_create(8, 8, 0.1, 2, 0, 1, psf, data, noise, options={"no_such_option": 1})


def test_async_host_entry_and_peaks_reject_null(api):
    lib = api.load()
    assert lib.tl_loglike_batch_host_async(None, None, 4, None, None) == api.TL_EINVAL
    assert lib.tl_wait(None, 0) == api.TL_EINVAL
    assert lib.tl_measure_peaks(None, 4, None) == api.TL_EINVAL


def test_library_reads_no_environment_variables():
    """Every tuning knob is a tl_options field (tl_create_ex); nothing in csrc/ calls getenv."""
    csrc = os.path.join(ROOT, "paper_2503_08586_b200", "csrc")
    for f in os.listdir(csrc):
        if f.endswith((".cu", ".cuh", ".h")):
            assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_no_cpu_fallback_without_a_device(api):
    """Without a usable GPU the product path must fail loudly with TL_ECUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present; covered by the gpu tests")
    psf, data, noise = _args()
    with pytest.raises(api.TinyLensError) as ei:
        api.tl_create(8, 8, 0.1, 2, 0, 1, psf, data, noise)
    assert ei.value.code == api.TL_ECUDA


def test_product_path_does_not_import_the_oracle():
    """The package must not reference oracle/ (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_2503_08586_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "tl_oracle" not in src and "liboracle" not in src, f
