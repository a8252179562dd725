"""ctypes wrapper around oracle/tl_oracle.c (the FP64 CPU oracle).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the
CUDA path; the only shared module is the arithmetic-free input generator
(paper_2503_08586_b200.workloads), and only for its `Workload` record.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tl_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


class OrcConfig(C.Structure):
    _fields_ = [("ny", C.c_int32), ("nx", C.c_int32), ("pix_scale", C.c_double),
                ("supersample", C.c_int32), ("n_lens_light", C.c_int32),
                ("n_source", C.c_int32), ("edge_mode", C.c_int32), ("mass_model", C.c_int32)]


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no -ffast-math.  Rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d, i32, i64 = C.c_double, C.c_int32, C.c_int64
        fp, dp, cp = C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(OrcConfig)
        L.orc_gammainc_p.restype = d; L.orc_gammainc_p.argtypes = [d, d]
        L.orc_bn.restype = d; L.orc_bn.argtypes = [d]
        L.orc_shape.restype = None; L.orc_shape.argtypes = [d, d, dp, dp]
        L.orc_sie_deflection.restype = None; L.orc_sie_deflection.argtypes = [d] * 7 + [dp, dp]
        L.orc_epl_deflection.restype = None; L.orc_epl_deflection.argtypes = [d] * 8 + [dp, dp]
        L.orc_shear_deflection.restype = None; L.orc_shear_deflection.argtypes = [d] * 4 + [dp, dp]
        L.orc_sersic.restype = d; L.orc_sersic.argtypes = [d] * 10
        L.orc_row_valid.restype = i32; L.orc_row_valid.argtypes = [cp, fp]
        L.orc_ideal_image.restype = None; L.orc_ideal_image.argtypes = [cp, i32, fp, dp]
        L.orc_convolve.restype = None; L.orc_convolve.argtypes = [i32, i32, i32, dp, fp, i32, dp]
        L.orc_render.restype = i32; L.orc_render.argtypes = [cp, fp, i32, fp, dp]
        L.orc_loglike_from_image.restype = d; L.orc_loglike_from_image.argtypes = [dp, fp, fp, C.c_size_t]
        L.orc_chi2_from_image.restype = d; L.orc_chi2_from_image.argtypes = [dp, fp, fp, C.c_size_t]
        L.orc_loglike.restype = d; L.orc_loglike.argtypes = [cp, fp, i32, fp, fp, fp]
        L.orc_loglike_batch.restype = i32
        L.orc_loglike_batch.argtypes = [cp, i32, fp, i32, fp, fp, fp, i64, dp, i32]
        L.orc_render_batch.restype = i32
        L.orc_render_batch.argtypes = [cp, i32, fp, i32, fp, i64, dp, i32]
        L.orc_nnls_small.restype = None; L.orc_nnls_small.argtypes = [i32, dp, dp, dp]
        L.orc_component_images.restype = i32; L.orc_component_images.argtypes = [cp, fp, i32, fp, dp]
        L.orc_loglike_linear.restype = d; L.orc_loglike_linear.argtypes = [cp, fp, i32, fp, fp, fp, dp]
        L.orc_loglike_linear_batch.restype = i32
        L.orc_loglike_linear_batch.argtypes = [cp, i32, fp, i32, fp, fp, fp, i64, dp, dp, i32]
        L.orc_gauss.restype = d; L.orc_gauss.argtypes = [d] * 7
        L.orc_mge_row_valid.restype = i32; L.orc_mge_row_valid.argtypes = [cp, fp]
        L.orc_mge_component_images.restype = i32
        L.orc_mge_component_images.argtypes = [cp, fp, i32, fp, fp, i32, dp]
        L.orc_nnls_enum.restype = None; L.orc_nnls_enum.argtypes = [i32, dp, dp, dp]
        L.orc_loglike_mge.restype = d; L.orc_loglike_mge.argtypes = [cp, fp, i32, fp, fp, fp, fp, i32, dp]
        L.orc_loglike_mge_batch.restype = i32
        L.orc_loglike_mge_batch.argtypes = [cp, i32, fp, i32, fp, fp, fp, i64, fp, i32, dp, dp, i32]
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def config(ny, nx, pix_scale, supersample, n_lens_light, n_source, edge_mode=0, mass_model=0) -> OrcConfig:
    return OrcConfig(int(ny), int(nx), float(pix_scale), int(supersample), int(n_lens_light),
                     int(n_source), int(edge_mode), int(mass_model))


def config_of(w) -> OrcConfig:
    """OrcConfig from a workloads.Workload-like record."""
    return config(w.ny, w.nx, w.pix_scale, w.supersample, w.n_lens_light, w.n_source, w.edge_mode,
                  getattr(w, "mass_model", 0))


# ---- scalar pieces (each cites the passage in tl_oracle.c) -------------------------------

def gammainc_p(a, x):
    return lib().orc_gammainc_p(float(a), float(x))


def bn(n):
    return lib().orc_bn(float(n))


def shape(e1, e2):
    q, phi = C.c_double(), C.c_double()
    lib().orc_shape(float(e1), float(e2), C.byref(q), C.byref(phi))
    return q.value, phi.value


def sie_deflection(theta_e, q, phi, cx, cy, x, y):
    ax, ay = C.c_double(), C.c_double()
    lib().orc_sie_deflection(float(theta_e), float(q), float(phi), float(cx), float(cy),
                             float(x), float(y), C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def epl_deflection(theta_e, gamma, q, phi, cx, cy, x, y):
    ax, ay = C.c_double(), C.c_double()
    lib().orc_epl_deflection(float(theta_e), float(gamma), float(q), float(phi), float(cx), float(cy),
                             float(x), float(y), C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def shear_deflection(g1, g2, x, y):
    ax, ay = C.c_double(), C.c_double()
    lib().orc_shear_deflection(float(g1), float(g2), float(x), float(y), C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def sersic(i_e, r_e, n, q, phi, cx, cy, x, y, b_n=None):
    b = bn(n) if b_n is None else b_n
    return lib().orc_sersic(float(i_e), float(r_e), float(n), float(b), float(q), float(phi),
                            float(cx), float(cy), float(x), float(y))


def row_valid(cfg: OrcConfig, row) -> bool:
    r = _f32(row)
    return bool(lib().orc_row_valid(C.byref(cfg), _fp(r)))


# ---- images ------------------------------------------------------------------------------

def halo(cfg: OrcConfig, K: int) -> int:
    return (K - 1) // 2 if cfg.edge_mode == 0 else 0


def ideal_image(cfg: OrcConfig, g: int, row) -> np.ndarray:
    r = _f32(row)
    out = np.empty((cfg.ny + 2 * g, cfg.nx + 2 * g), np.float64)
    lib().orc_ideal_image(C.byref(cfg), int(g), _fp(r), _dp(out))
    return out


def convolve(ny, nx, g, img, psf) -> np.ndarray:
    img = np.ascontiguousarray(img, dtype=np.float64)
    p = _f32(psf)
    K = p.shape[0]
    assert p.shape == (K, K) and img.shape == (ny + 2 * g, nx + 2 * g)
    out = np.empty((ny, nx), np.float64)
    lib().orc_convolve(int(ny), int(nx), int(g), _dp(img), _fp(p), int(K), _dp(out))
    return out


def render(cfg: OrcConfig, psf, row) -> np.ndarray:
    p, r = _f32(psf), _f32(row)
    out = np.empty((cfg.ny, cfg.nx), np.float64)
    lib().orc_render(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(r), _dp(out))
    return out


def loglike_from_image(image, data, noise) -> float:
    im = np.ascontiguousarray(image, dtype=np.float64)
    d, s = _f32(data), _f32(noise)
    return lib().orc_loglike_from_image(_dp(im), _fp(d), _fp(s), im.size)


def chi2_from_image(image, data, noise) -> float:
    im = np.ascontiguousarray(image, dtype=np.float64)
    d, s = _f32(data), _f32(noise)
    return lib().orc_chi2_from_image(_dp(im), _fp(d), _fp(s), im.size)


def loglike(cfg: OrcConfig, psf, data, noise, row) -> float:
    p, d, s, r = _f32(psf), _f32(data), _f32(noise), _f32(row)
    return lib().orc_loglike(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(d), _fp(s), _fp(r))


# ---- batches -----------------------------------------------------------------------------

def loglike_batch(cfg: OrcConfig, psf, data, noise, rows, n_lens: int = 1, threads: int = 0):
    """logL [B] float64 and the number of OpenMP threads used."""
    p, d, s, r = _f32(psf), _f32(data), _f32(noise), _f32(rows)
    B = r.shape[0]
    out = np.empty(B, np.float64)
    used = lib().orc_loglike_batch(C.byref(cfg), int(n_lens), _fp(p), int(p.shape[-1]), _fp(d),
                                   _fp(s), _fp(r), B, _dp(out), int(threads))
    return out, used


def render_batch(cfg: OrcConfig, psf, rows, n_lens: int = 1, threads: int = 0) -> np.ndarray:
    p, r = _f32(psf), _f32(rows)
    B = r.shape[0]
    out = np.empty((B, cfg.ny, cfg.nx), np.float64)
    lib().orc_render_batch(C.byref(cfg), int(n_lens), _fp(p), int(p.shape[-1]), _fp(r), B,
                           _dp(out), int(threads))
    return out


def render_for_workloads(w, psf, row) -> np.ndarray:
    """`render` callable for workloads.make_problem (tests / cpu_baseline leg only)."""
    return render(config_of(w), psf, row)


# ---- NEXT-1: linear amplitudes ------------------------------------------

def nnls_small(G, b) -> np.ndarray:
    G = np.ascontiguousarray(G, dtype=np.float64); b = np.ascontiguousarray(b, dtype=np.float64)
    n = b.size
    s = np.zeros(n, np.float64)
    lib().orc_nnls_small(int(n), _dp(G), _dp(b), _dp(s))
    return s


def component_images(cfg: OrcConfig, psf, row) -> np.ndarray:
    p, r = _f32(psf), _f32(row)
    C_ = cfg.n_lens_light + cfg.n_source
    out = np.empty((C_, cfg.ny, cfg.nx), np.float64)
    lib().orc_component_images(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(r), _dp(out))
    return out


def loglike_linear(cfg: OrcConfig, psf, data, noise, row):
    """(logL at the NNLS amplitudes, amplitudes [C])."""
    p, d, s, r = _f32(psf), _f32(data), _f32(noise), _f32(row)
    amps = np.empty(cfg.n_lens_light + cfg.n_source, np.float64)
    ll = lib().orc_loglike_linear(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(d), _fp(s), _fp(r), _dp(amps))
    return ll, amps


def loglike_linear_batch(cfg: OrcConfig, psf, data, noise, rows, n_lens: int = 1, threads: int = 0):
    p, d, s, r = _f32(psf), _f32(data), _f32(noise), _f32(rows)
    B = r.shape[0]
    out = np.empty(B, np.float64)
    amps = np.empty((B, cfg.n_lens_light + cfg.n_source), np.float64)
    lib().orc_loglike_linear_batch(C.byref(cfg), int(n_lens), _fp(p), int(p.shape[-1]), _fp(d), _fp(s), _fp(r),
                                   B, _dp(out), _dp(amps), int(threads))
    return out, amps


# ---- NEXT-3: MGE lens light with linear amplitudes (reading G23) -----------

def gauss(sigma, q, phi, cx, cy, x, y) -> float:
    return lib().orc_gauss(sigma, q, phi, cx, cy, x, y)


def nnls_enum(G, b) -> np.ndarray:
    G = np.ascontiguousarray(G, dtype=np.float64); b = np.ascontiguousarray(b, dtype=np.float64)
    n = b.size
    s = np.zeros(n, np.float64)
    lib().orc_nnls_enum(int(n), _dp(G), _dp(b), _dp(s))
    return s


def mge_component_images(cfg: OrcConfig, psf, row, sigmas) -> np.ndarray:
    p, r, sg = _f32(psf), _f32(row), _f32(sigmas)
    out = np.full((sg.size + cfg.n_source, cfg.ny, cfg.nx), np.nan, np.float64)
    lib().orc_mge_component_images(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(r), _fp(sg), int(sg.size), _dp(out))
    return out


def loglike_mge(cfg: OrcConfig, psf, data, noise, row, sigmas):
    """(logL at the NNLS amplitudes, amplitudes [n_gauss + n_source])."""
    p, d, s, r, sg = _f32(psf), _f32(data), _f32(noise), _f32(row), _f32(sigmas)
    amps = np.empty(sg.size + cfg.n_source, np.float64)
    ll = lib().orc_loglike_mge(C.byref(cfg), _fp(p), int(p.shape[-1]), _fp(d), _fp(s), _fp(r), _fp(sg), int(sg.size),
                               _dp(amps))
    return ll, amps


def loglike_mge_batch(cfg: OrcConfig, psf, data, noise, rows, sigmas, n_lens: int = 1, threads: int = 0):
    p, d, s, r, sg = _f32(psf), _f32(data), _f32(noise), _f32(rows), _f32(sigmas)
    B = r.shape[0]
    out = np.empty(B, np.float64)
    amps = np.empty((B, sg.size + cfg.n_source), np.float64)
    lib().orc_loglike_mge_batch(C.byref(cfg), int(n_lens), _fp(p), int(p.shape[-1]), _fp(d), _fp(s), _fp(r), B,
                                _fp(sg), int(sg.size), _dp(out), _dp(amps), int(threads))
    return out, amps


# ---- NEXT-3, several Gaussian sets (isophote twists; G23) ----------
# The row of a context with n_lens_light = n_sets carries one lens-light block per set; set j takes
# its (e1, e2, cx, cy) from block j (entries +3..+6; I_e, r_e, n ignored).  Plain and slow, out of the
# single-set pieces above: the columns of set j are the Gaussian columns of `mge_component_images`
# on the single-set view of the row (lens | block j | sources); the sources come from the first view.
# The NNLS optimum is taken by its definition (every support enumerated, orc_nnls_enum) up to 16
# columns; beyond that 2^n supports are out of reach and the library routine scipy.optimize.nnls
# (Lawson-Hanson on the whitened design matrix) serves as the step -- pinned against the enumeration
# on random problems of <= 10 columns and against it on MGE problems of <= 16 columns
# (tests/test_oracle_mge_pins.py).

def _single_set_view(cfg: OrcConfig, row, j: int):
    lp = 7 + (1 if cfg.mass_model == 1 else 0)
    r = np.asarray(row, np.float32)
    nll = cfg.n_lens_light
    view = np.concatenate([r[:lp], r[lp + 7 * j: lp + 7 * (j + 1)], r[lp + 7 * nll:]]).astype(np.float32)
    c1 = config(cfg.ny, cfg.nx, cfg.pix_scale, cfg.supersample, 1, cfg.n_source, cfg.edge_mode, cfg.mass_model)
    return c1, view


def mge_sets_component_images(cfg: OrcConfig, psf, row, sigma_sets):
    """Columns of M: the Gaussians of set 0, of set 1, ..., then the sources; None for an invalid row."""
    cols, src = [], None
    for j, sg in enumerate(sigma_sets):
        c1, view = _single_set_view(cfg, row, j)
        if not lib().orc_mge_row_valid(C.byref(c1), _fp(_f32(view))):
            return None
        M = mge_component_images(c1, psf, view, sg)
        cols.append(M[:len(sg)])
        if src is None:
            src = M[len(sg):]
    return np.concatenate(cols + [src], axis=0)


def nnls_design(A, y, enum_max: int = 16) -> np.ndarray:
    """argmin ||A s - y||^2 over s >= 0: enumeration of supports up to enum_max columns, else scipy's nnls."""
    A = np.asarray(A, np.float64); y = np.asarray(y, np.float64)
    if A.shape[1] <= enum_max:
        return nnls_enum(A.T @ A, A.T @ y)
    from scipy.optimize import nnls as _nnls
    return _nnls(A, y, maxiter=50 * A.shape[1])[0]


def loglike_mge_sets(cfg: OrcConfig, psf, data, noise, row, sigma_sets, enum_max: int = 16):
    """(logL of PAPER.md:82 Eq. 5 at the NNLS amplitudes of Eq. 6-7, amplitudes)."""
    M = mge_sets_component_images(cfg, psf, row, sigma_sets)
    n_col = sum(len(s) for s in sigma_sets) + cfg.n_source
    if M is None:
        return -np.inf, np.full(n_col, np.nan)
    sig = np.asarray(noise, np.float64).reshape(-1)
    A = (M.reshape(n_col, -1) / sig).T
    s = nnls_design(A, np.asarray(data, np.float64).reshape(-1) / sig, enum_max)
    return loglike_from_image(np.tensordot(s, M, axes=1), data, noise), s
