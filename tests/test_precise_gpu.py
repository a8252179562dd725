"""FP64 validation mode (tl_set_precision(ctx, TL_PRECISION_FP64)): the north_star tolerance
must hold on EVERY row, including the near-truth slice where FP32 arithmetic cannot reach it."""
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


@pytest.mark.parametrize("idx,n_prior,n_near,n_lens", [(0, 64, 64, 1), (1, 16, 16, 1), (2, 2, 4, 1), (3, 6, 6, 3)])
def test_fp64_mode_meets_north_star_everywhere(api, orc, idx, n_prior, n_near, n_lens):
    import torch
    w = W.workload(idx).scaled(batch=n_lens * n_prior, n_lens=n_lens)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, isnear = PT.rows_with_near(W, w, prob, n_prior, n_near)
    ctx = api.LensContext.from_problem(prob)
    d = torch.from_numpy(rows).cuda()
    fast = ctx.loglike(d).cpu().numpy().astype(np.float64)
    ctx.set_precision(api.TL_PRECISION_FP64)
    ll = ctx.loglike(d).cpu().numpy().astype(np.float64)
    im = ctx.render(d).cpu().numpy().astype(np.float64)
    ll2 = ctx.loglike(d).cpu().numpy().astype(np.float64)
    # the same model with CUDA's double math library instead of the hand-ordered polynomials: an
    # independent check of every approximation in csrc/tl_dp.cuh (both results are rounded to float)
    ctx.set_precision(api.TL_PRECISION_FP64_LIBM)
    ll_libm = ctx.loglike(d).cpu().numpy().astype(np.float64)
    im_libm = ctx.render(d).cpu().numpy().astype(np.float64)
    ctx.set_precision(api.TL_PRECISION_FP32)
    back = ctx.loglike(d).cpu().numpy().astype(np.float64)
    ctx.close()
    assert np.array_equal(ll, ll2) and np.array_equal(fast, back)
    assert np.all(np.abs(ll - ll_libm) <= 1e-4 * PT.logl_tol(ll_libm) + np.abs(ll_libm) * 2.0 ** -23)
    assert np.all(np.abs(im - im_libm) <= 2.0 ** -22 * np.abs(im_libm).max())
    oll, oim = PT.oracle_reference(orc, w, prob, rows)
    tol = PT.logl_tol(oll)
    # the result is returned as float: half an ulp of |logL| on top of the tolerance
    tol = tol + np.abs(oll) * 2.0 ** -24
    dl = np.abs(ll - oll)
    assert np.all(dl <= tol), "FP64 mode: worst %.3g x north-star tol" % (dl / tol).max()
    peak = np.abs(oim).reshape(len(rows), -1).max(axis=1)
    dpix = np.abs(im - oim).reshape(len(rows), -1).max(axis=1)
    assert np.all(dpix <= 2e-7 * peak)
    print("config %d FP64 mode: logL %.3g x north-star tol (fast path on the same rows: %.3g x)"
          % (idx, (dl / tol).max(), (np.abs(fast - oll) / tol).max()))


def test_fp64_mode_invalid_rows_and_edges(api, orc):
    import torch
    w = W.Workload(index=9, name="p64", ny=11, nx=14, pix_scale=0.2, supersample=3, psf_size=5,
                   psf_kind="moffat", psf_fwhm=0.3, psf_beta=2.5, n_lens_light=1, n_source=2,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=8, edge_mode=W.EDGE_ZERO)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, 8)
    rows[1, 0] = -1.0; rows[2, 8] = 0.0; rows[3, 4] = np.nan
    rows[4, 1] = rows[4, 2] = 0.0                         # SIS
    ctx = api.LensContext.from_problem(prob)
    ctx.set_precision(api.TL_PRECISION_FP64)
    d = torch.from_numpy(rows).cuda()
    ll = ctx.loglike(d).cpu().numpy().astype(np.float64)
    im = ctx.render(d).cpu().numpy().astype(np.float64)
    ctx.close()
    oll, oim = PT.oracle_reference(orc, w, prob, rows)
    for r in (1, 2, 3):
        assert ll[r] == -np.inf and np.all(np.isnan(im[r]))
    ok = [0, 4, 5, 6, 7]
    assert np.all(np.abs(ll[ok] - oll[ok]) <= PT.logl_tol(oll[ok]) + np.abs(oll[ok]) * 2.0 ** -24)
