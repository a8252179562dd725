"""GPU parity of tl_loglike_mge_batch (NEXT-3: MGE lens light with linear amplitudes,
PAPER.md:291-293 reading G23, amplitudes by PAPER.md:86-129 Eq. 6-7) against the oracle."""
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


def _check(api, orc, w, prob, rows, sigmas, amp_rtol=None, precision=0):
    """precision 0: the FP32 pipeline, held to NEAR_MARGIN x its measured worst (every MGE row is near its
    best fit); TL_PRECISION_FP64 / AUTO: the FP64 pipeline, north_star as stated on every row."""
    import torch
    ctx = api.LensContext.from_problem(prob)
    ctx.set_mge(sigmas)
    ctx.set_precision(precision)
    bound = PT.near_bound_fp32(PT.FP32_MGE_MEASURED) if precision == 0 else 1.0
    d = torch.from_numpy(rows).cuda()
    ll, amps = ctx.loglike_mge(d)
    ll2, _ = ctx.loglike_mge(d, want_amps=False)
    torch.cuda.synchronize()
    assert torch.equal(ll, ll2)                      # bitwise reproducible
    ctx.close()
    ll = ll.cpu().numpy().astype(np.float64); amps = amps.cpu().numpy().astype(np.float64)
    cfg = orc.config_of(w)
    oll, oamps = orc.loglike_mge_batch(cfg, prob.psf, prob.data, prob.noise, rows, sigmas, n_lens=w.n_lens)
    n_col = len(sigmas) + w.n_source
    assert amps.shape == (len(rows), n_col)
    assert np.all(np.isfinite(ll)) and np.all(amps >= 0.0)
    per = len(rows) // w.n_lens
    lens = np.arange(len(rows)) // per
    dl = np.abs(ll - oll)
    tol = PT.logl_tol(oll)
    worst_fit = 0.0
    floors = np.empty(len(rows))
    for r in range(len(rows)):
        M = orc.mge_component_images(cfg, prob.psf[lens[r]], rows[r], sigmas)
        oimg = np.tensordot(oamps[r], M, axes=1)
        floors[r] = PT.fp32_floor(oimg[None], prob.data[lens[r]][None], prob.noise[lens[r]][None], w.supersample)[0]
        # what is unique: the fitted image M s.  The GPU's amplitudes, put through the ORACLE's
        # columns, must reach the oracle's optimum (neighbouring Gaussians are nearly collinear,
        # so the amplitudes themselves are compared only when the set is well separated)
        gimg = np.tensordot(amps[r], M, axes=1)
        ll_at = orc.loglike_from_image(gimg, prob.data[lens[r]], prob.noise[lens[r]])
        assert ll_at <= oll[r] + 1e-9 * abs(oll[r])                 # the oracle's is the maximum
        assert oll[r] - ll_at <= bound * tol[r], (r, oll[r] - ll_at, tol[r])
        worst_fit = max(worst_fit, np.abs(gimg - oimg).max() / oimg.max())
    assert worst_fit <= 1e-4, worst_fit                             # fitted image, relative to its peak
    tn = np.maximum(tol, floors)
    tolf = tol + np.abs(oll) * 2.0 ** -24                           # the result is returned as float
    assert (dl / tolf).max() <= bound, "MGE logL parity (precision %d): worst %.3g x north_star" % (precision, (dl / tolf).max())
    if amp_rtol is not None:
        scale = np.maximum(np.abs(oamps).max(axis=1, keepdims=True), 1e-30)
        assert np.all(np.abs(amps - oamps) <= amp_rtol * scale), np.abs((amps - oamps) / scale).max()
    print("%s MGE (%d columns, precision %d): logL %.3g x north-star tol, %.3g x derived; fitted image %.2e x peak"
          % (w.name, n_col, precision, (dl / tol).max(), (dl / tn).max(), worst_fit))
    return ll, amps, oll, oamps


def test_mge_small_image_well_separated_set(api, orc):
    """Odd-sized image with a ragged tail, sigmas a factor 3 apart: amplitudes are well conditioned."""
    w = W.Workload(index=9, name="mge-small", ny=37, nx=45, pix_scale=0.12, supersample=2, psf_size=7,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=1, n_source=1,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=24)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, _ = PT.rows_with_near(W, w, prob, 16, 8)
    rows[::3, 7] = np.nan; rows[1::3, 8] = -1.0; rows[2::3, 9] = np.inf     # ignored entries
    rows[::2, 14] = np.nan
    sigmas = np.array([0.1, 0.3, 0.9, 2.7], np.float32)
    _check(api, orc, w, prob, rows, sigmas, amp_rtol=2e-4)
    _check(api, orc, w, prob, rows, sigmas, amp_rtol=1e-6, precision=api.TL_PRECISION_FP64)


@pytest.mark.parametrize("precision", [0, 1, 3])
@pytest.mark.parametrize("idx,n_prior,n_near,n_lens,n_gauss", [(1, 6, 6, 1, 10), (3, 4, 4, 3, 8), (4, 1, 1, 1, 6)])
def test_mge_matches_oracle_on_configs(api, orc, idx, n_prior, n_near, n_lens, n_gauss, precision):
    w = W.workload(idx).scaled(batch=n_lens * n_prior, n_lens=n_lens)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows, _ = PT.rows_with_near(W, w, prob, n_prior, n_near)
    _check(api, orc, w, prob, rows, W.mge_sigmas(w, n_gauss), precision=precision)


def test_mge_zero_edge_and_epl(api, orc):
    from dataclasses import replace
    w = replace(W.workload(1).with_epl().scaled(batch=6), ny=40, nx=52, psf_size=9, edge_mode=1)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, 6)
    _check(api, orc, w, prob, rows, W.mge_sigmas(w, 7))
    _check(api, orc, w, prob, rows, W.mge_sigmas(w, 7), precision=api.TL_PRECISION_FP64)


def test_mge_recovers_known_amplitudes_and_flags_invalid_rows(api, orc):
    import torch
    w = W.Workload(index=9, name="mge-rec", ny=48, nx=48, pix_scale=0.1, supersample=2, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.25, psf_beta=0.0, n_lens_light=1, n_source=2,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=8)
    prob = W.make_problem(w, orc.render_for_workloads)
    cfg = orc.config_of(w)
    row = prob.truth[0].copy()
    sigmas = np.array([0.12, 0.36, 1.1], np.float32)
    M = orc.mge_component_images(cfg, prob.psf[0], row, sigmas)
    true_amps = np.array([30.0, 0.0, 4.5, 2.0, 9.0])
    data = np.tensordot(true_amps, M, axes=1).astype(np.float32)[None]
    noise = np.full_like(data, 0.1)
    rows = np.stack([row] * 8)
    rows[1, 0] = -1.0                 # theta_E < 0
    rows[2, 10] = 0.9; rows[2, 11] = 0.9    # |e| >= 1 of the MGE shape
    rows[3, 13] = np.nan              # MGE centre not finite
    rows[4, 16] = 0.0                 # source n = 0
    ctx = api.LensContext(w.ny, w.nx, w.pix_scale, w.supersample, 1, 2, prob.psf, data, noise)
    with pytest.raises(api.TinyLensError):
        ctx.loglike_mge(torch.from_numpy(rows).cuda())          # no Gaussian set yet
    with pytest.raises(api.TinyLensError):
        ctx.set_mge(np.array([0.1, -0.2], np.float32))
    with pytest.raises(api.TinyLensError):
        ctx.set_mge(np.full(31, 0.1, np.float32))          # more than 30 Gaussians
    ctx.set_mge(sigmas)
    ll, amps = ctx.loglike_mge(torch.from_numpy(rows).cuda())
    ll = ll.cpu().numpy(); amps = amps.cpu().numpy()
    ctx.close()
    for r in (1, 2, 3, 4):
        assert ll[r] == -np.inf and np.all(np.isnan(amps[r]))
    const = -0.5 * data.size * np.log(2 * np.pi * 0.1 ** 2)
    for r in (0, 5, 6, 7):
        assert np.allclose(amps[r], true_amps, rtol=2e-4, atol=2e-3), amps[r]
        assert abs(ll[r] - const) <= 1e-3 + 1e-6 * abs(const) + 0.05     # chi^2 ~ (1e-7 x SNR)^2 summed
    # a context without lens light has no MGE
    w0 = W.workload(0)
    p0 = W.make_problem(w0, orc.render_for_workloads)
    c0 = api.LensContext.from_problem(p0)
    with pytest.raises(api.TinyLensError):
        c0.set_mge(sigmas)
    c0.close()


def test_mge_full_size_batch_sampled(api, orc):
    """configs[1] at the batch bench.py --mode mge times (B = 4096, one chunk): the oracle on a
    sample of rows, properties on all of them, and the value of a row does not depend on the batch."""
    import torch
    w = W.workload(1)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w)
    assert rows.shape[0] == 4096
    sigmas = W.mge_sigmas(w, 10)
    ctx = api.LensContext.from_problem(prob)
    ctx.set_mge(sigmas)
    assert api.tl_mge_columns(ctx.handle) == 11 and api.tl_mge_chunk_rows(ctx.handle) >= 4096
    d = torch.from_numpy(rows).cuda()
    ll, amps = ctx.loglike_mge(d)
    sample = np.arange(7, 4096, 273)                       # 15 rows across the batch
    ll_s, amps_s = ctx.loglike_mge(d[torch.from_numpy(sample).cuda()].contiguous())
    torch.cuda.synchronize()
    ctx.close()
    assert torch.equal(ll[sample], ll_s) and torch.equal(amps[sample], amps_s)
    ll = ll.cpu().numpy().astype(np.float64); amps = amps.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(ll)) and np.all(amps >= 0.0) and np.all(np.isfinite(amps))
    cfg = orc.config_of(w)
    oll, oamps = orc.loglike_mge_batch(cfg, prob.psf, prob.data, prob.noise, rows[sample], sigmas)
    tol = PT.logl_tol(oll)
    for t, r in enumerate(sample):
        M = orc.mge_component_images(cfg, prob.psf[0], rows[r], sigmas)
        oimg = np.tensordot(oamps[t], M, axes=1)
        floor = PT.fp32_floor(oimg[None], prob.data[0][None], prob.noise[0][None], w.supersample)[0]
        assert abs(ll[r] - oll[t]) <= PT.near_bound_fp32(PT.FP32_MGE_MEASURED) * tol[t], (r, ll[r] - oll[t], tol[t], floor)
        gimg = np.tensordot(amps[r], M, axes=1)
        assert np.abs(gimg - oimg).max() <= 1e-4 * oimg.max()
    # Eq. 6: the solved likelihood is a maximum over amplitudes, so never below the fixed-amplitude
    # likelihood of a Sersic lens light that the Gaussian set can reproduce poorly -- not comparable;
    # what is comparable: more Gaussians never fit worse than a subset of them
    ctx2 = api.LensContext.from_problem(prob)
    ctx2.set_mge(sigmas[::2])
    ll_sub, _ = ctx2.loglike_mge(d[:256].contiguous())
    ctx2.close()
    ll_sub = ll_sub.cpu().numpy().astype(np.float64)
    assert np.all(ll[:256] >= ll_sub - 1e-3 - 2e-6 * np.abs(ll_sub))


def test_mge_call_is_cuda_graph_capturable(api, orc):
    """NEXT-4: tl_loglike_mge_batch makes no host sync and takes its scratch from the
    stream-ordered allocator, so a sampler can capture the seven launches in a CUDA graph."""
    import torch
    w = W.Workload(index=9, name="mge-graph", ny=30, nx=34, pix_scale=0.12, supersample=2, psf_size=5,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=1, n_source=1,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=40)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w)
    ctx = api.LensContext.from_problem(prob)
    ctx.set_mge(W.mge_sigmas(w, 6))
    d = torch.from_numpy(rows).cuda()
    ref, ref_amps = ctx.loglike_mge(d)
    ref, ref_amps = ref.clone(), ref_amps.clone()
    out, amps = torch.empty_like(ref), torch.empty_like(ref_amps)
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        ctx.loglike_mge(d, out, amps, stream=s)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ctx.loglike_mge(d, out, amps, stream=s)
    out.zero_(); amps.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref) and torch.equal(amps, ref_amps)
    d.copy_(torch.from_numpy(rows[::-1].copy()).cuda())       # new parameters, same buffers
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref.flip(0)) and torch.equal(amps, ref_amps.flip(0))
    del g
    ctx.close()


def test_mge_chunked_call_equals_single_chunk(api, orc):
    """A call larger than the scratch budget is processed in chunks (tl_options.mge_chunk_rows forces
    that here, with a ragged last chunk, on three lenses): identical bits."""
    import torch
    w = W.workload(3).scaled(batch=3 * 14, n_lens=3)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, 14)
    rows[5, 0] = -1.0                                   # an invalid row inside a chunk
    ctx = api.LensContext.from_problem(prob)
    ctx.set_mge(W.mge_sigmas(w, 7))
    d = torch.from_numpy(rows).cuda()
    ll1, am1 = ctx.loglike_mge(d)
    torch.cuda.synchronize()
    ctx2 = api.LensContext.from_problem(prob, options={"mge_chunk_rows": 5})
    ctx2.set_mge(W.mge_sigmas(w, 7))
    assert api.tl_mge_chunk_rows(ctx2.handle) == 5
    ll2, am2 = ctx2.loglike_mge(d)
    torch.cuda.synchronize()
    ctx.close(); ctx2.close()
    assert torch.equal(ll1, ll2) and torch.equal(am1.nan_to_num(-1.0), am2.nan_to_num(-1.0))
    assert ll1[5].item() == -np.inf


# ---- several Gaussian sets with their own shapes (tl_set_mge_sets; "isophote twists") ----

def _two_set_case(orc, n0, n1, ny=36, nx=44, S=2, K=7, batch=12):
    w = W.Workload(index=9, name="mge-sets", ny=ny, nx=nx, pix_scale=0.12, supersample=S, psf_size=K,
                   psf_kind="gaussian", psf_fwhm=0.3, psf_beta=0.0, n_lens_light=2, n_source=1,
                   noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=batch)
    w1 = W.Workload(**{**w.__dict__, "n_lens_light": 1})
    rows = W.batch_rows(w, batch)
    truth1 = np.concatenate([rows[0][:14], rows[0][21:]]).astype(np.float32)
    prob = W.make_problem(w1, lambda ww, psf, row: orc.render_for_workloads(ww, psf, truth1))
    prob = type(prob)(w, prob.psf, prob.data, prob.noise, rows[:1].copy())
    sets = [W.mge_sigmas(w, n0), (W.mge_sigmas(w, n1) * 1.3).astype(np.float32)]
    return w, prob, rows, sets


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("n0,n1", [(6, 5), (14, 12), (16, 14)])
def test_mge_two_sets_match_oracle(api, orc, n0, n1, precision):
    """Two Gaussian sets, each on its own ellipses, 12 / 27 / 31 columns (the last two beyond what the
    oracle can enumerate: scipy's NNLS is its step there, pinned against the enumeration on CPU).
    Compared: logL, and the fitted image through the oracle's own columns."""
    import torch
    w, prob, rows, sets = _two_set_case(orc, n0, n1)
    rows = rows.copy()
    rows[3, 17] = 0.9; rows[3, 18] = 0.9                 # second set's shape invalid -> invalid row
    rows[5, 7:10] = np.nan; rows[5, 14:17] = np.nan      # ignored entries of both blocks
    ctx = api.LensContext.from_problem(prob)
    ctx.set_mge_sets(sets)
    ctx.set_precision(precision)
    bound = PT.near_bound_fp32(PT.FP32_MGE_MEASURED) if precision == 0 else 1.0
    n_col = n0 + n1 + 1
    assert api.tl_mge_columns(ctx.handle) == n_col
    d = torch.from_numpy(rows).cuda()
    ll, amps = ctx.loglike_mge(d)
    ll2, _ = ctx.loglike_mge(d, want_amps=False)
    # a context with two lens-light blocks serves the MGE call only
    with pytest.raises(api.TinyLensError):
        ctx.loglike(d)
    with pytest.raises(api.TinyLensError):
        ctx.set_mge(sets[0])
    ctx.close()
    assert torch.equal(ll, ll2)
    ll = ll.cpu().numpy().astype(np.float64); amps = amps.cpu().numpy().astype(np.float64)
    cfg = orc.config_of(w)
    worst, worst_fit = 0.0, 0.0
    for r in range(len(rows)):
        oll, oamps = orc.loglike_mge_sets(cfg, prob.psf[0], prob.data[0], prob.noise[0], rows[r], sets)
        if r == 3:
            assert oll == -np.inf and ll[r] == -np.inf and np.all(np.isnan(amps[r]))
            continue
        assert np.isfinite(ll[r]) and np.all(amps[r] >= 0.0)
        tol = max(PT.LOGL_ABS, PT.LOGL_REL * abs(oll))
        worst = max(worst, abs(ll[r] - oll) / tol)
        M = orc.mge_sets_component_images(cfg, prob.psf[0], rows[r], sets)
        oimg, gimg = np.tensordot(oamps, M, axes=1), np.tensordot(amps[r], M, axes=1)
        worst_fit = max(worst_fit, np.abs(gimg - oimg).max() / oimg.max())
        # the GPU's amplitudes, through the oracle's columns, reach the oracle's optimum
        ll_at = orc.loglike_from_image(gimg, prob.data[0], prob.noise[0])
        assert oll - ll_at <= bound * tol, (r, oll - ll_at, tol)
    print("two sets (%d + %d Gaussians, %d columns, precision %d): logL %.3g x north_star, fitted image %.2e x peak"
          % (n0, n1, n_col, precision, worst, worst_fit))
    assert worst <= bound and worst_fit <= 1e-4


def test_mge_two_identical_sets_equal_one_set(api, orc):
    """Two sets with the same shape = one set with the dispersions concatenated (logL to FP32 noise;
    the Gaussians are evaluated by the same kernel either way)."""
    import torch
    w, prob, rows, sets = _two_set_case(orc, 4, 3)
    rows = rows.copy()
    rows[:, 14:21] = rows[:, 7:14]
    ctx2 = api.LensContext.from_problem(prob)
    ctx2.set_mge_sets(sets)
    ll2, a2 = ctx2.loglike_mge(torch.from_numpy(rows).cuda())
    ctx2.close()
    w1 = W.Workload(**{**w.__dict__, "n_lens_light": 1})
    prob1 = type(prob)(w1, prob.psf, prob.data, prob.noise, prob.truth)
    rows1 = np.ascontiguousarray(np.concatenate([rows[:, :14], rows[:, 21:]], axis=1))
    ctx1 = api.LensContext.from_problem(prob1)
    ctx1.set_mge(np.concatenate(sets))
    ll1, a1 = ctx1.loglike_mge(torch.from_numpy(rows1).cuda())
    ctx1.close()
    assert torch.equal(ll1, ll2) and torch.equal(a1, a2)
