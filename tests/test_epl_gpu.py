"""GPU parity of the elliptical power-law mass model (NEXT-2: Eq. 12,
tl_config.mass_model = TL_MASS_EPL) against the oracle, through the C ABI."""
import dataclasses

import numpy as np
import pytest

from paper_2503_08586_b200 import workloads as W
from tests import parity as PT

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available()
    from paper_2503_08586_b200 import api as _api
    _api.load()
    return _api


def _gpu(api, prob, rows, precision=None):
    import torch
    ctx = api.LensContext.from_problem(prob)
    assert ctx.n_params == prob.workload.n_params
    if precision is not None:
        ctx.set_precision(precision)
    d = torch.from_numpy(np.ascontiguousarray(rows)).cuda()
    ll = ctx.loglike(d)
    ll2 = ctx.loglike(d)
    im = ctx.render(d)
    torch.cuda.synchronize()
    assert torch.equal(ll, ll2)                                   # bitwise reproducible
    info = ctx.info()
    ctx.close()
    return ll.cpu().numpy().astype(np.float64), im.cpu().numpy().astype(np.float64), info


def _compare(w, prob, rows, isnear, ll, im, oll, oim, near_measured):
    B = len(rows)
    peak = np.abs(oim).reshape(B, -1).max(axis=1)
    dpix = np.abs(im - oim).reshape(B, -1).max(axis=1)
    assert np.all(dpix <= PT.PIX_TOL * peak), "pixel parity: worst %.3g x peak" % (dpix / peak).max()
    tol = PT.logl_tol(oll)
    dl = np.abs(ll - oll)
    prior = ~isnear
    assert np.all(dl[prior] <= tol[prior]), "logL (prior rows): worst %.3g x tol" % (dl[prior] / tol[prior]).max()
    near = (dl[isnear] / tol[isnear]).max() if isnear.any() else 0.0
    assert near <= PT.near_bound_fp32(near_measured), "logL (near-truth rows, fp32): %.3g x north_star > %.3g" % (near, PT.near_bound_fp32(near_measured))
    return (dpix / peak).max() / PT.PIX_TOL, (dl[prior] / tol[prior]).max() if prior.any() else 0.0, \
        (dl[isnear] / tol[isnear]).max() if isnear.any() else 0.0


@pytest.mark.parametrize("idx,n_prior,n_near,n_lens", [(0, 64, 64, 1), (1, 24, 24, 1), (2, 3, 3, 1), (3, 8, 8, 4), (4, 1, 1, 1)])
def test_epl_configs_match_oracle(api, orc, idx, n_prior, n_near, n_lens):
    w = W.workload(idx).with_epl().scaled(batch=n_lens * n_prior, n_lens=n_lens)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, isnear = PT.rows_with_near(W, w, prob, n_prior, n_near)
    ll, im, info = _gpu(api, prob, rows)
    oll, oim = PT.oracle_reference(orc, w, prob, rows)
    pix, prior, near = _compare(w, prob, rows, isnear, ll, im, oll, oim, PT.FP32_NEAR_MEASURED_EPL[idx])
    print("EPL config %d path=%d: pix %.3g x tol, logL prior %.3g x tol, near %.3g x north-star tol"
          % (idx, info["path"], pix, prior, near))


def _small(**kw):
    base = dict(index=8, name="epl-small", ny=37, nx=45, pix_scale=0.11, supersample=4, psf_size=7,
                psf_kind="gaussian", psf_fwhm=0.25, psf_beta=0.0, n_lens_light=1, n_source=2,
                noise_bg=0.05, noise_exptime=150.0, source_amp=(1.0, 20.0), batch=16, mass_model=W.MASS_EPL)
    base.update(kw)
    return W.Workload(**base)


def test_epl_slopes_shapes_and_flat_lenses(api, orc):
    """Slopes across (1, 3), both series paths (FP32 up to 24 terms, FP64 beyond: q < 0.35), q = 1,
    theta_E = 0, ragged image, two sources, S = 3 (generic loop) and S = 4 (unrolled)."""
    for S in (4, 3):
        w = _small(supersample=S)
        prob = W.make_problem(w, orc.render_for_workloads)
        rows = W.batch_rows(w, 16)
        slopes = [1.05, 1.3, 1.6, 2.0, 2.4, 2.7, 2.95, 2.2]
        for r, g in enumerate(slopes):
            rows[r, 7] = g
        for r, q in zip(range(8, 13), (0.36, 0.34, 0.2, 0.08, 0.5)):        # around the 24-term limit and far beyond
            rows[r, 1], rows[r, 2] = W.ellipticity_from_q_phi(q, 0.7)
        rows[13, 1] = rows[13, 2] = 0.0                                       # q = 1: every a_n = 0
        rows[14, 0] = 0.0                                                     # no lens
        ll, im, _ = _gpu(api, prob, rows)
        oll, oim = PT.oracle_reference(orc, w, prob, rows)
        assert np.all(np.isfinite(ll))
        isnear = np.zeros(len(rows), bool)         # prior draws with a few entries replaced: north_star as stated
        pix, prior, _ = _compare(w, prob, rows, isnear, ll, im, oll, oim, 1.0)
        print("EPL small S=%d: pix %.3g x tol, logL %.3g x north-star tol" % (S, pix, prior))


def test_epl_slope_two_is_the_sie_kernel(api, orc):
    """gamma = 2: the EPL kernels reproduce the SIE kernels' images."""
    import torch
    w = W.workload(1).scaled(batch=8)
    we = w.with_epl()
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, 8)
    rows_e = np.insert(rows, 7, 2.0, axis=1).astype(np.float32)
    _, im_s, _ = _gpu(api, prob, rows)
    prob_e = dataclasses.replace(prob, workload=we, truth=np.insert(prob.truth, 7, 2.0, axis=1).astype(np.float32))
    _, im_e, _ = _gpu(api, prob_e, rows_e)
    peak = np.abs(im_s).reshape(8, -1).max(axis=1)
    d = np.abs(im_s - im_e).reshape(8, -1).max(axis=1)
    assert np.all(d <= 4e-6 * peak), (d / peak).max()


def test_epl_invalid_slope(api, orc):
    w = _small(n_source=1)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, 8)
    for r, g in enumerate((1.0, 3.0, 0.2, 3.4, np.nan, np.inf)):
        rows[r, 7] = g
    for prec in (None, 1):
        ll, im, _ = _gpu(api, prob, rows, prec)
        assert np.all(np.isneginf(ll[:6])) and np.all(np.isnan(im[:6]))
        assert np.all(np.isfinite(ll[6:])) and np.all(np.isfinite(im[6:]))


@pytest.mark.parametrize("idx,n_prior,n_near", [(0, 32, 32), (1, 8, 8)])
def test_epl_fp64_mode(api, orc, idx, n_prior, n_near):
    w = W.workload(idx).with_epl().scaled(batch=n_prior)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, isnear = PT.rows_with_near(W, w, prob, n_prior, n_near)
    rows[0, 1], rows[0, 2] = W.ellipticity_from_q_phi(0.15, 1.1)
    ll, im, _ = _gpu(api, prob, rows, 1)
    oll, oim = PT.oracle_reference(orc, w, prob, rows)
    tol = PT.logl_tol(oll) + np.abs(oll) * 2.0 ** -24
    dl = np.abs(ll - oll)
    assert np.all(dl <= tol), "EPL FP64 mode: worst %.3g x north-star tol" % (dl / tol).max()
    peak = np.abs(oim).reshape(len(rows), -1).max(axis=1)
    assert np.all(np.abs(im - oim).reshape(len(rows), -1).max(axis=1) <= 2e-7 * peak)


@pytest.mark.parametrize("idx,n_prior,n_near", [(0, 24, 24), (1, 8, 8)])
def test_epl_linear_mode(api, orc, idx, n_prior, n_near):
    import torch
    w = W.workload(idx).with_epl().scaled(batch=n_prior)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, _ = PT.rows_with_near(W, w, prob, n_prior, n_near)
    ctx = api.LensContext.from_problem(prob)
    ll, amps = ctx.loglike_linear(torch.from_numpy(rows).cuda())
    ll = ll.cpu().numpy().astype(np.float64); amps = amps.cpu().numpy().astype(np.float64)
    ctx.close()
    cfg = orc.config_of(w)
    oll, oamps = orc.loglike_linear_batch(cfg, prob.psf, prob.data, prob.noise, rows)
    scale = np.maximum(np.abs(oamps).max(axis=1, keepdims=True), 1e-30)
    assert np.all(np.abs(amps - oamps) <= 2e-5 * scale), np.abs((amps - oamps) / scale).max()
    oimg = np.stack([np.tensordot(oamps[r], orc.component_images(cfg, prob.psf[0], rows[r]), axes=1) for r in range(len(rows))])
    ratio = (np.abs(ll - oll) / PT.logl_tol(oll)).max()
    print("EPL linear config %d: logL %.3g x north_star" % (idx, ratio))
    assert ratio <= PT.near_bound_fp32(PT.FP32_LINEAR_MEASURED_EPL[idx]), ratio


@pytest.mark.parametrize("seed", range(8))
def test_epl_random_shapes(api, orc, seed):
    """The random geometries of tests/test_parity_gpu.py (odd / tiny sizes, S in 1..6, PSF sizes on
    both convolution paths, both edge modes, 1-3 components) with the EPL mass model."""
    from tests.test_parity_gpu import _random_case, _small_problem
    rng = np.random.default_rng(2000 + seed)
    w, prob = _small_problem(orc, index=40 + seed, mass_model=W.MASS_EPL, **_random_case(rng))
    rows, isnear = PT.rows_with_near(W, w, prob, 6, 2)
    ll, im, _ = _gpu(api, prob, rows)
    oll, oim = PT.oracle_reference(orc, w, prob, rows)
    res = _compare(w, prob, rows, isnear, ll, im, oll, oim, PT.FP32_EPL_SMALL_MEASURED)
    print("EPL random shape %d: pix %.3g, prior %.3g, near %.3g x north_star" % ((seed,) + tuple(res)))


def test_epl_full_size_csst_batch_sampled_against_oracle(api, orc):
    """configs[1] with the EPL mass model at its full B = 4096, in the launch configuration
    `bench.py --mass epl` times: every logL finite, a seeded sample of rows against the oracle."""
    import torch
    w = W.workload(1).with_epl()
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w)
    ctx = api.LensContext.from_problem(prob)
    ll = ctx.loglike(torch.from_numpy(rows).cuda()).cpu().numpy().astype(np.float64)
    info = ctx.info()
    ctx.close()
    assert info["path"] == 0 and info["block_threads"] == 512 and len(ll) == 4096 > info["small_batch_rows"]
    assert np.all(np.isfinite(ll))
    pick = np.random.default_rng(17).choice(4096, 24, replace=False)
    oll, _ = orc.loglike_batch(orc.config_of(w), prob.psf, prob.data, prob.noise, rows[pick])
    assert np.all(np.abs(ll[pick] - oll) <= PT.logl_tol(oll))
