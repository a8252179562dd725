"""Guard words round the library's scratch memory (tl_options.debug_canaries, include/tinylens.h).

compute-sanitizer cannot be run on this GPU pool (profiles/r2_sanitizers.md), so the library carries a check of
its own for writes outside the per-call scratch buffers: 256 bytes of 0xA5 on either side of every
allocation, compared when it is freed.  Every entry point and every path (fused, small-batch, split, staged,
FP64, AUTO, libm, linear, MGE with one and two sets, host entries) is driven here on several shapes with the
option on; the count must stay 0, and the self-test must see its two deliberate hits.  With the option the
scratch also starts filled with 0xFF (NaN / -1), so a kernel that read scratch nobody wrote would change the
results: they must equal those of a context without the option bit for bit."""
import numpy as np
import pytest

from paper_2503_08586_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available()
    from paper_2503_08586_b200 import api as _api
    _api.load()
    return _api


def _flat_data(w, psf, row):
    return np.full((w.ny, w.nx), 0.3)


CASES = [
    W.workload(1),                                                              # fused path, S = 4, K = 21
    W.workload(3).scaled(batch=24, n_lens=3),                                   # several lenses, S = 2, K = 15
    W.workload(4).scaled(batch=4, n_lens=1),                                    # split path, S = 8, K = 41, two sources
    W.workload(1).with_epl(),
    W.Workload(index=7, name="odd", ny=37, nx=45, pix_scale=0.11, supersample=3, psf_size=9, psf_kind="moffat",
               psf_fwhm=0.3, psf_beta=2.5, n_lens_light=1, n_source=2, noise_bg=0.05, noise_exptime=150.0,
               source_amp=(1.0, 20.0), batch=16),
    W.Workload(index=7, name="zero-edge", ny=20, nx=18, pix_scale=0.2, supersample=2, psf_size=5, psf_kind="gaussian",
               psf_fwhm=0.4, psf_beta=0.0, n_lens_light=0, n_source=1, noise_bg=0.05, noise_exptime=0.0,
               source_amp=(5.0, 5.0), batch=16, edge_mode=W.EDGE_ZERO),
]


@pytest.mark.parametrize("w", CASES, ids=lambda w: "%s%s" % (w.name, "-epl" if w.mass_model else ""))
def test_no_kernel_writes_outside_its_scratch(api, w):
    import torch
    prob = W.make_problem(w, _flat_data)
    ctx = api.LensContext.from_problem(prob, options={"debug_canaries": 1})
    plain = api.LensContext.from_problem(prob)                     # (the scratch of `ctx` starts as NaNs: same results all the same)
    ctx.canary_selftest()                                          # the check sees a word changed on either side
    assert ctx.canary_errors() == 0

    def same(x, y):
        return torch.equal(torch.nan_to_num(x, nan=-7.0), torch.nan_to_num(y, nan=-7.0))
    big = W.batch_rows(w, max(1, 200 // w.n_lens))                 # more rows than half the SMs: the large-batch paths
    small = W.batch_rows(w, 1 if w.n_lens > 1 else 3)              # a few rows: the small-batch routes
    big[1, 0] = -1.0                                               # an invalid row
    for rows in (big, small):
        d = torch.from_numpy(np.ascontiguousarray(rows)).cuda()
        for prec in (api.TL_PRECISION_FP32, api.TL_PRECISION_FP64, api.TL_PRECISION_AUTO, api.TL_PRECISION_FP64_LIBM):
            if prec == api.TL_PRECISION_FP64_LIBM and (w.mass_model or rows is big and w.name == "large"):
                continue
            ctx.set_precision(prec); plain.set_precision(prec)
            assert same(ctx.loglike(d), plain.loglike(d)), (w.name, prec)
            if prec in (api.TL_PRECISION_FP32, api.TL_PRECISION_FP64):
                sub = d[: 2 * w.n_lens].contiguous()
                assert same(ctx.render(sub), plain.render(sub)), (w.name, prec)
            if w.n_lens_light <= 1 and prec != api.TL_PRECISION_FP64_LIBM:
                (la, aa), (lb, ab) = ctx.loglike_linear(d), plain.loglike_linear(d)
                assert same(la, lb) and same(aa, ab), (w.name, prec)
        ctx.set_precision(api.TL_PRECISION_FP32); plain.set_precision(api.TL_PRECISION_FP32)
        assert np.array_equal(ctx.loglike_host(np.ascontiguousarray(rows)), plain.loglike_host(np.ascontiguousarray(rows)))
    torch.cuda.synchronize()
    assert ctx.canary_errors() == 0
    ctx.close(); plain.close()
    # the staged linear pipeline where the fused one would have been taken
    if w.n_lens_light <= 1:
        ctx = api.LensContext.from_problem(prob, options={"debug_canaries": 1, "linear_staged": 1})
        ctx.loglike_linear(torch.from_numpy(np.ascontiguousarray(big)).cuda())
        assert ctx.canary_errors() == 0
        ctx.close()


@pytest.mark.parametrize("idx", [1, 3])
def test_mge_kernels_stay_inside_their_scratch(api, idx):
    import torch
    w = W.workload(idx).scaled(batch=64, n_lens=1) if idx == 3 else W.workload(idx)
    prob = W.make_problem(w, _flat_data)
    ctx = api.LensContext.from_problem(prob, options={"debug_canaries": 1})
    plain = api.LensContext.from_problem(prob)
    ctx.set_mge(W.mge_sigmas(w, 10)); plain.set_mge(W.mge_sigmas(w, 10))
    for n in (160, 3):
        d = torch.from_numpy(np.ascontiguousarray(W.batch_rows(w, n))).cuda()
        for prec in (api.TL_PRECISION_FP32, api.TL_PRECISION_FP64):
            ctx.set_precision(prec); plain.set_precision(prec)
            (la, aa), (lb, ab) = ctx.loglike_mge(d), plain.loglike_mge(d)
            assert torch.equal(la, lb) and torch.equal(aa, ab), (n, prec)
    ctx.set_precision(api.TL_PRECISION_FP32); plain.set_precision(api.TL_PRECISION_FP32)
    ctx.set_mge(W.mge_sigmas(w, 14)); plain.set_mge(W.mge_sigmas(w, 14))   # more than 11 columns: the shared-memory Gram kernel
    d = torch.from_numpy(np.ascontiguousarray(W.batch_rows(w, 100))).cuda()
    (la, aa), (lb, ab) = ctx.loglike_mge(d), plain.loglike_mge(d)
    assert torch.equal(la, lb) and torch.equal(aa, ab)
    torch.cuda.synchronize()
    assert ctx.canary_errors() == 0
    ctx.close(); plain.close()


def test_canary_calls_need_the_option(api):
    w = W.workload(0)
    ctx = api.LensContext.from_problem(W.make_problem(w, _flat_data))
    with pytest.raises(api.TinyLensError):
        ctx.canary_errors()
    with pytest.raises(api.TinyLensError):
        ctx.canary_selftest()
    ctx.close()
