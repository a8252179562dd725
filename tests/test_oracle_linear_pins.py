"""Pins of the oracle's linear-amplitude likelihood (Eq. 6-7; NEXT-1): the NNLS
minimiser against a library routine, exact amplitude recovery, optimality, and the clamp at 0."""
import numpy as np
import pytest
from scipy.optimize import nnls as scipy_nnls

from paper_2503_08586_b200 import workloads as W


def test_nnls_matches_library(orc):
    rng = np.random.default_rng(3)
    n_active = 0
    for trial in range(300):
        n = int(rng.integers(1, 4))
        A = rng.normal(size=(12, n))
        if trial % 3 == 0 and n > 1:
            A[:, 1] = A[:, 0] + 0.3 * rng.normal(size=12)          # correlated columns
        y = rng.normal(size=12) + (A @ rng.uniform(-1, 2, n))
        want, _ = scipy_nnls(A, y)
        got = orc.nnls_small(A.T @ A, A.T @ y)
        assert np.allclose(got, want, rtol=1e-9, atol=1e-10), (trial, got, want)
        n_active += int(np.any(want == 0.0))
    assert n_active > 30            # the constraint was active often enough to be tested


def _problem(orc, nl=1, ns=1):
    w = W.Workload(index=8, name="lin", ny=20, nx=24, pix_scale=0.15, supersample=2, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=nl, n_source=ns,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=4)
    return w, W.make_problem(w, orc.render_for_workloads)


def test_noise_free_amplitudes_are_recovered_exactly(orc):
    w, prob = _problem(orc, 1, 2)
    cfg = orc.config_of(w)
    row = prob.truth[0].copy()
    M = orc.component_images(cfg, prob.psf[0], row)
    true_amps = np.array([7.5, 3.25, 11.0])
    data = np.tensordot(true_amps, M, axes=1).astype(np.float32)       # noise-free
    noise = np.full_like(data, 0.1)
    ll, amps = orc.loglike_linear(cfg, prob.psf[0], data, noise, row)
    # data were rounded to float32: amplitudes to that accuracy, chi^2 ~ (rounding/sigma)^2 ~ 0
    assert np.allclose(amps, true_amps, rtol=1e-6)
    const = -0.5 * data.size * np.log(2 * np.pi * 0.1 ** 2)
    assert abs(ll - const) < 1e-6 * abs(const)
    # the I_e entries of the row are ignored
    row2 = row.copy(); row2[7] = 123.0; row2[14] = 0.0; row2[21] = -4.0
    ll2, amps2 = orc.loglike_linear(cfg, prob.psf[0], data, noise, row2)
    assert ll2 == ll and np.array_equal(amps, amps2)


def test_linear_likelihood_is_the_maximum_over_amplitudes(orc):
    w, prob = _problem(orc)
    cfg = orc.config_of(w)
    rows = W.batch_rows(w, 4)
    rng = np.random.default_rng(5)
    for row in rows:
        ll, amps = orc.loglike_linear(cfg, prob.psf[0], prob.data[0], prob.noise[0], row)
        assert np.all(amps >= 0.0)
        at = row.copy(); at[7] = amps[0]; at[14] = amps[1]
        # Eq. 6: the linear likelihood is Eq. 5 at the optimal amplitudes (float32 rounding of them)
        ll_at = orc.loglike(cfg, prob.psf[0], prob.data[0], prob.noise[0], at)
        assert abs(ll - ll_at) <= 1e-5 * max(1.0, abs(ll))
        for _ in range(5):
            other = row.copy(); other[7] = amps[0] * rng.uniform(0, 2); other[14] = amps[1] * rng.uniform(0, 2) + rng.uniform(0, 1)
            assert orc.loglike(cfg, prob.psf[0], prob.data[0], prob.noise[0], other) <= ll + 1e-6 * abs(ll)


def test_negative_unconstrained_amplitude_is_clamped(orc):
    w, prob = _problem(orc)
    cfg = orc.config_of(w)
    row = prob.truth[0].copy()
    M = orc.component_images(cfg, prob.psf[0], row)
    data = (5.0 * M[0] - 2.0 * M[1]).astype(np.float32)          # "negative source"
    noise = np.full_like(data, 0.1)
    ll, amps = orc.loglike_linear(cfg, prob.psf[0], data, noise, row)
    assert amps[1] == 0.0 and amps[0] > 0.0
    # with the source switched off the best lens amplitude is the 1-d weighted projection
    want = (M[0] * data).sum() / (M[0] ** 2).sum()
    assert abs(amps[0] - want) <= 1e-9 * want
    assert orc.loglike_linear(cfg, prob.psf[0], data, noise, np.where(np.arange(21) == 1, 2.0, row).astype(np.float32))[0] == -np.inf
