"""Pins of the oracle's MGE lens light with linear amplitudes (reading G23;
NEXT-3): the Gaussian columns against the Sersic n = 1/2 special case and their analytic flux,
the NNLS enumeration against a library routine, exact amplitude recovery, optimality."""
import math

import numpy as np
from scipy.optimize import nnls as scipy_nnls

from paper_2503_08586_b200 import workloads as W


def _problem(orc, ns=1, S=2):
    w = W.Workload(index=9, name="mge", ny=22, nx=26, pix_scale=0.15, supersample=S, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=1, n_source=ns,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=4)
    return w, W.make_problem(w, orc.render_for_workloads)


def test_gaussian_is_the_sersic_of_index_one_half(orc):
    # Eq. 8 with n = 1/2: I_e exp(-b [(R/r_e)^2 - 1]) and Eq. 9 gives b = ln 2 (P(1, b) = 1 - e^-b),
    # so it is the Gaussian of sigma = r_e / sqrt(2 ln 2) and central brightness 2 I_e
    assert abs(orc.bn(0.5) - math.log(2.0)) < 1e-12
    rng = np.random.default_rng(11)
    for _ in range(50):
        re, q, phi = rng.uniform(0.2, 2.0), rng.uniform(0.3, 1.0), rng.uniform(0, math.pi)
        cx, cy, x, y = rng.uniform(-1, 1, 4)
        want = orc.sersic(0.5, re, 0.5, q, phi, cx, cy, x, y)
        got = orc.gauss(re / math.sqrt(2 * math.log(2.0)), q, phi, cx, cy, x, y)
        assert abs(got - want) <= 1e-13 * max(want, 1e-300) + 1e-300


def test_gaussian_columns_equal_rendered_sersic_one_half(orc):
    # the whole column (grid, supersampling, binning, convolution) through an independent route:
    # orc_render of a row whose lens light is that Sersic and whose source is switched off
    w, prob = _problem(orc)
    cfg = orc.config_of(w)
    row = prob.truth[0].copy()
    sigmas = np.array([0.11, 0.4, 1.3], np.float32)
    M = orc.mge_component_images(cfg, prob.psf[0], row, sigmas)
    assert M.shape == (4, w.ny, w.nx)
    for k, sg in enumerate(sigmas):
        r2 = row.copy()
        r2[7] = 0.5; r2[8] = np.float32(float(sg) * math.sqrt(2 * math.log(2.0))); r2[9] = 0.5
        r2[14] = 0.0
        want = orc.render(cfg, prob.psf[0], r2)
        # r_e was rounded to float32: relative change of the exponent 6e-8 x (R/sigma)^2 / 2
        assert np.allclose(M[k], want, rtol=2e-5, atol=1e-12 * want.max()), k
    # last column = the source at unit amplitude, lens light off
    r3 = row.copy(); r3[7] = 0.0; r3[14] = 1.0
    assert np.allclose(M[3], orc.render(cfg, prob.psf[0], r3), rtol=1e-12, atol=0)
    # I_e, r_e, n of the lens-light block and I_e of the source are ignored
    r4 = row.copy(); r4[7] = -3.0; r4[8] = -1.0; r4[9] = np.nan; r4[14] = 55.0
    assert np.array_equal(orc.mge_component_images(cfg, prob.psf[0], r4, sigmas), M)


def test_gaussian_total_flux(orc):
    # integral of exp(-R_p^2 / 2 sigma^2) over the plane = 2 pi sigma^2 (Eq. 10 has unit determinant);
    # a PSF of unit sum preserves it
    w = W.Workload(index=9, name="mgeflux", ny=81, nx=81, pix_scale=0.1, supersample=4, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.25, psf_beta=0.0, n_lens_light=1, n_source=1,
                   noise_bg=0.05, noise_exptime=0.0, source_amp=(1.0, 1.0), batch=1)
    cfg = orc.config_of(w)
    psf = np.asarray(W.make_psf(w), np.float64).reshape(5, 5)
    psf = (psf / psf.sum()).astype(np.float32)
    row = np.array([1.0, 0.1, 0.05, 0, 0, 0, 0, 1, 1, 1, 0.2, -0.1, 0.03, -0.02, 1, 0.3, 1, 0, 0, 0, 0], np.float32)
    for sg in (0.25, 0.5):
        M = orc.mge_component_images(cfg, psf, row, np.array([sg], np.float32))
        flux = M[0].sum() * w.pix_scale ** 2
        assert abs(flux - 2 * math.pi * sg * sg) < 2e-4 * 2 * math.pi * sg * sg, (sg, flux)


def test_nnls_enum_matches_library(orc):
    rng = np.random.default_rng(4)
    n_active = 0
    for trial in range(120):
        n = int(rng.integers(1, 11))
        A = rng.normal(size=(40, n))
        if trial % 3 == 0 and n > 2:
            A[:, 1] = A[:, 0] + 0.3 * rng.normal(size=40)          # correlated columns
            A[:, 2] = 0.5 * (A[:, 0] + A[:, 1]) + 0.2 * rng.normal(size=40)
        y = rng.normal(size=40) + (A @ rng.uniform(-1, 2, n))
        want, _ = scipy_nnls(A, y)
        got = orc.nnls_enum(A.T @ A, A.T @ y)
        assert np.allclose(got, want, rtol=1e-8, atol=1e-9), (trial, got, want)
        n_active += int(np.any(want == 0.0))
    assert n_active > 40
    # and it agrees with the three-column routine of NEXT-1
    for _ in range(50):
        A = rng.normal(size=(12, 3)); y = rng.normal(size=12)
        assert np.allclose(orc.nnls_enum(A.T @ A, A.T @ y), orc.nnls_small(A.T @ A, A.T @ y), rtol=1e-10, atol=1e-12)


def test_noise_free_amplitudes_are_recovered(orc):
    w, prob = _problem(orc, ns=2)
    cfg = orc.config_of(w)
    row = prob.truth[0].copy()
    sigmas = np.array([0.1, 0.3, 0.9, 2.7], np.float32)
    M = orc.mge_component_images(cfg, prob.psf[0], row, sigmas)
    true_amps = np.array([40.0, 0.0, 6.5, 1.25, 3.0, 11.0])
    data = np.tensordot(true_amps, M, axes=1).astype(np.float32)
    noise = np.full_like(data, 0.1)
    ll, amps = orc.loglike_mge(cfg, prob.psf[0], data, noise, row, sigmas)
    assert np.allclose(amps, true_amps, rtol=1e-4, atol=1e-4)
    const = -0.5 * data.size * np.log(2 * np.pi * 0.1 ** 2)
    assert abs(ll - const) < 1e-6 * abs(const)
    bad = row.copy(); bad[10] = 0.8; bad[11] = 0.7           # |e| >= 1 of the MGE shape
    ll_bad, amps_bad = orc.loglike_mge(cfg, prob.psf[0], data, noise, bad, sigmas)
    assert ll_bad == -np.inf and np.all(np.isnan(amps_bad))


def test_mge_likelihood_is_the_maximum_over_amplitudes(orc):
    w, prob = _problem(orc)
    cfg = orc.config_of(w)
    sigmas = np.geomspace(0.08, 2.5, 7).astype(np.float32)
    rows = W.batch_rows(w, 3)
    rng = np.random.default_rng(6)
    for row in rows:
        ll, amps = orc.loglike_mge(cfg, prob.psf[0], prob.data[0], prob.noise[0], row, sigmas)
        assert np.all(amps >= 0.0) and amps.shape == (8,)
        M = orc.mge_component_images(cfg, prob.psf[0], row, sigmas)
        ll_at = orc.loglike_from_image(np.tensordot(amps, M, axes=1), prob.data[0], prob.noise[0])
        assert abs(ll - ll_at) <= 1e-12 * max(1.0, abs(ll))
        # library NNLS on the whitened design reaches the same optimum
        A = (M.reshape(8, -1) / prob.noise[0].reshape(1, -1).astype(np.float64)).T
        y = (prob.data[0].astype(np.float64) / prob.noise[0]).reshape(-1)
        s_lib, _ = scipy_nnls(A, y)
        ll_lib = orc.loglike_from_image(np.tensordot(s_lib, M, axes=1), prob.data[0], prob.noise[0])
        assert abs(ll - ll_lib) <= 1e-8 * max(1.0, abs(ll))
        for _ in range(5):
            other = amps * rng.uniform(0, 2, 8) + rng.uniform(0, 0.5, 8) * (rng.uniform(size=8) < 0.3)
            assert orc.loglike_from_image(np.tensordot(other, M, axes=1), prob.data[0], prob.noise[0]) <= ll + 1e-9 * abs(ll)
    # a single Gaussian plus a Sersic: the two-column problem agrees with the NEXT-1 oracle run on
    # the equivalent Sersic n = 1/2 lens light
    row = rows[0].copy()
    sg = np.float32(0.4)
    row[8] = np.float32(float(sg) * math.sqrt(2 * math.log(2.0))); row[9] = 0.5
    ll1, a1 = orc.loglike_mge(cfg, prob.psf[0], prob.data[0], prob.noise[0], row, np.array([sg]))
    ll2, a2 = orc.loglike_linear(cfg, prob.psf[0], prob.data[0], prob.noise[0], row)
    assert abs(ll1 - ll2) <= 2e-5 * abs(ll2)
    assert np.allclose(a1, [2 * a2[0], a2[1]], rtol=1e-4, atol=1e-6)


# ---- several Gaussian sets (oracle.loglike_mge_sets) -------------------------------------------

def _two_set_problem(orc):
    w = W.Workload(index=9, name="mge2", ny=20, nx=24, pix_scale=0.15, supersample=2, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=2, n_source=1,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=4)
    w1 = W.Workload(**{**w.__dict__, "n_lens_light": 1})
    rows = W.batch_rows(w, 4)
    # mock data from a single-Sersic lens light (the first lens-light block) + source
    truth1 = np.concatenate([rows[0][:14], rows[0][21:]]).astype(np.float32)
    prob1 = W.make_problem(w1, lambda ww, psf, row: orc.render_for_workloads(ww, psf, truth1))
    return w, prob1, rows


def test_two_identical_sets_equal_one_set(orc):
    """Sets that share shape and centre are one set with the dispersions concatenated."""
    w, prob, rows = _two_set_problem(orc)
    cfg = orc.config_of(w)
    row = rows[1].copy()
    row[14:21] = row[7:14]                                   # block 1 := block 0
    s0, s1 = np.array([0.1, 0.4], np.float32), np.array([0.2, 0.9, 2.0], np.float32)
    ll2, a2 = orc.loglike_mge_sets(cfg, prob.psf[0], prob.data[0], prob.noise[0], row, [s0, s1])
    w1 = W.Workload(**{**w.__dict__, "n_lens_light": 1})
    row1 = np.concatenate([row[:14], row[21:]]).astype(np.float32)
    ll1, a1 = orc.loglike_mge(orc.config_of(w1), prob.psf[0], prob.data[0], prob.noise[0], row1, np.concatenate([s0, s1]))
    assert abs(ll2 - ll1) <= 1e-9 * abs(ll1) and np.allclose(a2, a1, rtol=1e-6, atol=1e-9 * a1.max())


def test_second_set_uses_its_own_shape(orc):
    """The columns of set 1 are Gaussians on ITS ellipses: equal to the single-set columns of a row
    that carries block 1 as its lens light, and different from set 0's when the shapes differ."""
    w, prob, rows = _two_set_problem(orc)
    cfg = orc.config_of(w)
    row = rows[2]
    sg = np.array([0.3, 1.0], np.float32)
    M = orc.mge_sets_component_images(cfg, prob.psf[0], row, [sg, sg])
    assert M.shape == (5, w.ny, w.nx)
    w1 = W.Workload(**{**w.__dict__, "n_lens_light": 1})
    rowb = np.concatenate([row[:7], row[14:21], row[21:]]).astype(np.float32)
    Mb = orc.mge_component_images(orc.config_of(w1), prob.psf[0], rowb, sg)
    assert np.array_equal(M[2:4], Mb[:2]) and np.array_equal(M[4], Mb[2])
    assert np.abs(M[0] - M[2]).max() > 1e-3 * M[0].max()
    # invalid second shape -> invalid row
    bad = row.copy(); bad[17] = 0.9; bad[18] = 0.8
    ll, amps = orc.loglike_mge_sets(cfg, prob.psf[0], prob.data[0], prob.noise[0], bad, [sg, sg])
    assert ll == -np.inf and np.all(np.isnan(amps))


def test_library_nnls_equals_enumeration_on_mge_problems(orc):
    """Beyond 16 columns the oracle takes scipy.optimize.nnls as its step; on MGE problems small
    enough to enumerate (12 nearly collinear columns) both give the same logL and fitted image."""
    w, prob, rows = _two_set_problem(orc)
    cfg = orc.config_of(w)
    sets = [W.mge_sigmas(w, 6), W.mge_sigmas(w, 5)]
    for r in range(3):
        ll_e, a_e = orc.loglike_mge_sets(cfg, prob.psf[0], prob.data[0], prob.noise[0], rows[r], sets, enum_max=16)
        ll_s, a_s = orc.loglike_mge_sets(cfg, prob.psf[0], prob.data[0], prob.noise[0], rows[r], sets, enum_max=0)
        assert np.all(a_e >= 0) and np.all(a_s >= 0)
        assert abs(ll_e - ll_s) <= 1e-8 * abs(ll_e) + 1e-6, (ll_e, ll_s)
        M = orc.mge_sets_component_images(cfg, prob.psf[0], rows[r], sets)
        fe, fs = np.tensordot(a_e, M, axes=1), np.tensordot(a_s, M, axes=1)
        assert np.abs(fe - fs).max() <= 1e-6 * np.abs(fe).max()
        assert ll_e >= ll_s - 1e-6                          # the enumeration is the exact optimum
