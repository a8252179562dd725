"""Seeded synthetic inputs for the batched lens-model likelihood.

This module is the ONE piece shared by the CUDA path's callers (tests, bench.py) and the
FP64 oracle's callers.  It holds no part of the method's arithmetic: it never traces a ray,
evaluates a light profile, convolves or forms a chi^2.  Whenever an input needs a model
image (mock data = model(truth) + noise, "Mock Lens Creation"), the caller
passes a ``render`` callable: tests pass the oracle's renderer, bench.py passes the
library's own ``tl_render_batch``.

What is here:
  * the five BASELINE.json workloads as ``Workload`` records (shapes, pixel scales,
    supersampling, PSF and noise recipes, priors)                     [DESIGN.md "Inputs"]
  * a counter-based RNG (numpy Philox) keyed by  250308586 + 1000*config + stream
  * prior draws -> parameter rows in the boundary's layout (include/tinylens.h):
        theta_E, e1, e2, cx, cy, gamma1, gamma2, [slope gamma when mass_model = MASS_EPL,]
        then per Sersic (lens light first, then sources): I_e, r_e, n, e1, e2, cx, cy
    Drawn (q, phi) are encoded as (e1, e2) with the forward map of PAPER.md:152 Eq. 11.
  * PSF builders sampled at pixel centres, normalised to sum 1 (Gaussian / Moffat)
  * the noise recipe  sigma^2 = bg^2 + max(model, 0) / exptime

The paper's own datasets (Cao et al. 2024 CSST mock catalogue; SLACS HST
images) are not available; these workloads take their shapes, pixel scales,
supersampling and noise character and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Callable, Optional

import numpy as np

SEED_BASE = 250308586

# streams of the counter-based generator
STREAM_TRUTH, STREAM_NOISE, STREAM_BATCH, STREAM_NEAR, STREAM_PSF = 0, 1, 2, 3, 4

EDGE_EXTEND, EDGE_ZERO = 0, 1
MASS_SIE, MASS_EPL = 0, 1


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (index = position in BASELINE.json `configs`)."""
    index: int
    name: str
    ny: int
    nx: int
    pix_scale: float          # arcsec per native pixel
    supersample: int          # S
    psf_size: int             # K (odd)
    psf_kind: str             # "gaussian" | "moffat"
    psf_fwhm: float           # arcsec (survey batch: drawn per lens from psf_fwhm_range)
    psf_beta: float           # Moffat beta
    n_lens_light: int
    n_source: int
    noise_bg: float           # constant sigma (Tiny) or background sigma
    noise_exptime: float      # 0 => constant sigma
    source_amp: tuple         # (lo, hi) of I_e for the source; lo == hi => fixed
    batch: int                # B rows per call (total over lenses)
    n_lens: int = 1
    psf_fwhm_range: Optional[tuple] = None
    edge_mode: int = EDGE_EXTEND
    mass_model: int = MASS_SIE  # MASS_EPL: the row carries the power-law slope (Eq. 12)

    @property
    def n_lens_params(self) -> int:
        return 7 + (1 if self.mass_model == MASS_EPL else 0)

    @property
    def n_params(self) -> int:
        return self.n_lens_params + 7 * self.n_lens_light + 7 * self.n_source

    @property
    def rows_per_lens(self) -> int:
        return self.batch // self.n_lens

    @property
    def halo(self) -> int:
        return (self.psf_size - 1) // 2

    @property
    def samples_per_likelihood(self) -> int:
        h = self.halo if self.edge_mode == EDGE_EXTEND else 0
        return (self.ny + 2 * h) * (self.nx + 2 * h) * self.supersample ** 2

    def with_epl(self) -> "Workload":
        """Same workload with the elliptical power-law mass model (free slope)."""
        return replace(self, mass_model=MASS_EPL)

    def scaled(self, batch: Optional[int] = None, n_lens: Optional[int] = None) -> "Workload":
        """Same workload with a smaller batch / fewer lenses (parity-test sizes)."""
        nl = self.n_lens if n_lens is None else n_lens
        b = self.batch if batch is None else batch
        if b % nl:
            raise ValueError("batch must be a multiple of n_lens")
        return replace(self, batch=b, n_lens=nl)


WORKLOADS = (
    Workload(0, "tiny", 32, 32, 0.1, 1, 5, "gaussian", 0.2, 0.0, 0, 1,
             0.1, 0.0, (10.0, 10.0), 64),
    Workload(1, "csst", 100, 100, 0.074, 4, 21, "gaussian", 0.15, 0.0, 1, 1,
             0.05, 150.0, (1.0, 20.0), 4096),
    Workload(2, "hst", 200, 200, 0.05, 4, 31, "moffat", 0.1, 3.0, 1, 1,
             0.01, 2000.0, (1.0, 20.0), 16384),
    Workload(3, "survey", 64, 64, 0.074, 2, 15, "gaussian", 0.15, 0.0, 1, 1,
             0.05, 150.0, (1.0, 20.0), 512 * 1000, n_lens=1000, psf_fwhm_range=(0.12, 0.2)),
    Workload(4, "large", 400, 400, 0.025, 8, 41, "moffat", 0.1, 3.0, 1, 2,
             0.01, 2000.0, (1.0, 20.0), 65536),
)


def mge_sigmas(w: Workload, n_gauss: int = 10) -> np.ndarray:
    """Dispersions (arcsec, float32) of the MGE lens-light set used by the tests and bench.py
    --mode mge: log-spaced from 0.6 native pixels to half the field of view (input recipe,
    DESIGN.md section 13; the paper gives no set)."""
    lo = 0.6 * w.pix_scale
    hi = 0.5 * w.pix_scale * max(w.ny, w.nx)
    return np.geomspace(lo, hi, int(n_gauss)).astype(np.float32)


def workload(index_or_name) -> Workload:
    for w in WORKLOADS:
        if w.index == index_or_name or w.name == index_or_name:
            return w
    raise KeyError(index_or_name)


def rng_for(config: int, stream: int, sub: int = 0) -> np.random.Generator:
    """Counter-based generator: key = SEED_BASE + 1000*config + stream, counter block = sub."""
    bitgen = np.random.Philox(key=SEED_BASE + 1000 * config + stream, counter=[0, 0, sub, 0])
    return np.random.Generator(bitgen)


# --------------------------------------------------------------------------- parameters

def ellipticity_from_q_phi(q, phi):
    """(e1, e2) = (1-q)/(1+q) (cos 2phi, sin 2phi): the sampler's encoding, Eq. 11."""
    e = (1.0 - q) / (1.0 + q)
    return e * np.cos(2.0 * phi), e * np.sin(2.0 * phi)


def draw_params(w: Workload, rng: np.random.Generator, n: int) -> np.ndarray:
    """n independent prior draws, float32 [n, P] in the boundary's row layout."""
    cols = []
    theta_e = rng.uniform(0.8, 1.5, n)
    q = rng.uniform(0.6, 1.0, n)
    phi = rng.uniform(0.0, np.pi, n)
    cx = rng.uniform(-0.05, 0.05, n)
    cy = rng.uniform(-0.05, 0.05, n)
    g1 = rng.uniform(-0.05, 0.05, n)
    g2 = rng.uniform(-0.05, 0.05, n)
    e1, e2 = ellipticity_from_q_phi(q, phi)
    cols += [theta_e, e1, e2, cx, cy, g1, g2]
    for _ in range(w.n_lens_light):
        amp = rng.uniform(5.0, 50.0, n)
        re = rng.uniform(0.5, 2.0, n)
        ns = rng.uniform(2.0, 6.0, n)
        ql = rng.uniform(0.5, 1.0, n)
        pl = rng.uniform(0.0, np.pi, n)
        l1, l2 = ellipticity_from_q_phi(ql, pl)
        cols += [amp, re, ns, l1, l2, cx, cy]          # centre tied to the mass centre
    for _ in range(w.n_source):
        lo, hi = w.source_amp
        amp = np.full(n, lo) if lo == hi else rng.uniform(lo, hi, n)
        re = rng.uniform(0.1, 0.4, n)
        ns = rng.uniform(0.5, 4.0, n)
        qs = rng.uniform(0.5, 1.0, n)
        ps = rng.uniform(0.0, np.pi, n)
        s1, s2 = ellipticity_from_q_phi(qs, ps)
        sx = rng.uniform(-0.2, 0.2, n)
        sy = rng.uniform(-0.2, 0.2, n)
        cols += [amp, re, ns, s1, s2, sx, sy]
    if w.mass_model == MASS_EPL:
        # drawn last, so that every other parameter equals the SIE workload's draw
        cols.insert(7, rng.uniform(1.6, 2.4, n))
    return np.ascontiguousarray(np.stack(cols, axis=1).astype(np.float32))


def near_truth(truth_row: np.ndarray, rng: np.random.Generator, n: int, rel: float = 1e-3) -> np.ndarray:
    """truth * (1 + rel * N(0,1)) per parameter: the slice where |logL| is small and the
    absolute tolerance is tightest."""
    t = np.asarray(truth_row, dtype=np.float64).reshape(1, -1)
    out = t * (1.0 + rel * rng.standard_normal((n, t.shape[1])))
    return np.ascontiguousarray(out.astype(np.float32))


# --------------------------------------------------------------------------- PSF / noise

def _pixel_offsets(k: int) -> np.ndarray:
    return np.arange(k, dtype=np.float64) - (k - 1) / 2.0


def gaussian_psf(k: int, fwhm_pix: float) -> np.ndarray:
    sig = fwhm_pix / (2.0 * np.sqrt(2.0 * np.log(2.0)))
    o = _pixel_offsets(k)
    g = np.exp(-0.5 * (o[:, None] ** 2 + o[None, :] ** 2) / sig ** 2)
    return (g / g.sum()).astype(np.float32)


def moffat_psf(k: int, fwhm_pix: float, beta: float) -> np.ndarray:
    alpha = fwhm_pix / (2.0 * np.sqrt(2.0 ** (1.0 / beta) - 1.0))
    o = _pixel_offsets(k)
    m = (1.0 + (o[:, None] ** 2 + o[None, :] ** 2) / alpha ** 2) ** (-beta)
    return (m / m.sum()).astype(np.float32)


def make_psf(w: Workload, fwhm: Optional[float] = None) -> np.ndarray:
    f = (w.psf_fwhm if fwhm is None else fwhm) / w.pix_scale
    if w.psf_kind == "gaussian":
        return gaussian_psf(w.psf_size, f)
    return moffat_psf(w.psf_size, f, w.psf_beta)


def noise_map(w: Workload, model: np.ndarray) -> np.ndarray:
    """sigma per pixel: constant, or sqrt(bg^2 + max(model,0)/exptime) (Gaussian approx.)."""
    model = np.asarray(model, dtype=np.float64)
    if w.noise_exptime <= 0.0:
        return np.full(model.shape, w.noise_bg, dtype=np.float64)
    return np.sqrt(w.noise_bg ** 2 + np.maximum(model, 0.0) / w.noise_exptime)


# --------------------------------------------------------------------------- problems

@dataclass
class Problem:
    """Everything `tl_create` needs plus the truth rows (one per lens)."""
    workload: Workload
    psf: np.ndarray       # float32 [n_lens, K, K]
    data: np.ndarray      # float32 [n_lens, ny, nx]
    noise: np.ndarray     # float32 [n_lens, ny, nx]
    truth: np.ndarray     # float32 [n_lens, P]


RenderFn = Callable[[Workload, np.ndarray, np.ndarray], np.ndarray]
"""render(workload_with_n_lens_1, psf[K,K] float32, row[P] float32) -> image [ny,nx]."""


def make_problem(w: Workload, render: RenderFn) -> Problem:
    """Mock data per lens: model(truth) + sigma * N(0,1).

    `render` supplies the model image; this module does not know how it is computed.
    """
    L = w.n_lens
    psf = np.empty((L, w.psf_size, w.psf_size), np.float32)
    data = np.empty((L, w.ny, w.nx), np.float32)
    noise = np.empty((L, w.ny, w.nx), np.float32)
    truth = np.empty((L, w.n_params), np.float32)
    single = replace(w, n_lens=1, batch=1)
    for l in range(L):
        if w.psf_fwhm_range is not None:
            fwhm = rng_for(w.index, STREAM_PSF, l).uniform(*w.psf_fwhm_range)
        else:
            fwhm = None
        psf[l] = make_psf(w, fwhm)
        truth[l] = draw_params(w, rng_for(w.index, STREAM_TRUTH, l), 1)[0]
        model = np.asarray(render(single, psf[l], truth[l]), dtype=np.float64).reshape(w.ny, w.nx)
        sig = noise_map(w, model)
        z = rng_for(w.index, STREAM_NOISE, l).standard_normal(model.shape)
        data[l] = (model + sig * z).astype(np.float32)
        noise[l] = sig.astype(np.float32)
    return Problem(w, psf, data, noise, truth)


def batch_rows(w: Workload, n_per_lens: Optional[int] = None) -> np.ndarray:
    """Prior draws for one call: float32 [n_lens * rows, P], `rows` consecutive rows per lens."""
    n = w.rows_per_lens if n_per_lens is None else n_per_lens
    if w.n_lens == 1:
        return draw_params(w, rng_for(w.index, STREAM_BATCH, 0), n)
    return np.concatenate([draw_params(w, rng_for(w.index, STREAM_BATCH, l), n)
                           for l in range(w.n_lens)], axis=0)


def near_truth_rows(p: Problem, n_per_lens: int = 64, rel: float = 1e-3) -> np.ndarray:
    w = p.workload
    return np.concatenate([near_truth(p.truth[l], rng_for(w.index, STREAM_NEAR, l), n_per_lens, rel)
                           for l in range(w.n_lens)], axis=0)
