"""Serve mode (NEXT-4: tl_serve_start / tl_serve_eval / tl_serve_stop, csrc/tl_serve.cuh): a persistent kernel
answers small requests through a block of mapped host memory.  It runs the device functions of the small-batch
path in the same order, so logL must be BITWISE tl_loglike_batch's; every wait is bounded (the tests carry a
timeout of their own all the same)."""
import time

import numpy as np
import pytest

from paper_2503_08586_b200 import workloads as W


def _flat_data(w, psf, row):
    return np.full((w.ny, w.nx), 0.3)


def test_serve_calls_reject_null_and_idle_contexts():
    from paper_2503_08586_b200 import api
    L = api.load()
    assert L.tl_serve_start(None, 4, 1.0) == api.TL_EINVAL
    assert L.tl_serve_eval(None, None, 1, None) == api.TL_EINVAL
    assert L.tl_serve_stop(None) == api.TL_EINVAL


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available()
    from paper_2503_08586_b200 import api as _api
    _api.load()
    return _api


CASES = [
    W.workload(1),                                                                       # S = 4, K = 21, 512-thread CTAs
    W.workload(3).scaled(batch=64, n_lens=1),                                            # S = 2, K = 15, 256-thread CTAs
    W.Workload(index=7, name="s8-two-sources", ny=30, nx=34, pix_scale=0.05, supersample=8, psf_size=5, psf_kind="gaussian",
               psf_fwhm=0.12, psf_beta=0.0, n_lens_light=0, n_source=2, noise_bg=0.05, noise_exptime=300.0,
               source_amp=(1.0, 20.0), batch=16, edge_mode=W.EDGE_ZERO),
]


@pytest.mark.gpu
@pytest.mark.timeout(180)
@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_served_requests_equal_loglike_batch_bitwise(api, w):
    import torch
    ctx = api.LensContext.from_problem(W.make_problem(w, _flat_data))
    rows = W.batch_rows(w, 48)
    rows[5, 0] = -1.0                                              # an invalid row: logL = -inf
    rows[7, 1], rows[7, 2] = 0.3, -0.305                           # q = 0.4: the q < 0.5 branch of the SIE
    ref = ctx.loglike(torch.from_numpy(rows).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    with pytest.raises(api.TinyLensError):                         # not serving yet
        ctx.serve_eval(rows[:1])
    ctx.serve_start(max_rows=16, idle_timeout_s=0.5)
    try:
        with pytest.raises(api.TinyLensError):                     # already serving
            ctx.serve_start(max_rows=4, idle_timeout_s=0.5)
        for B in (1, 2, 3, 8, 16):
            for k in range(0, 48 - B + 1, B):
                out = ctx.serve_eval(rows[k:k + B])
                assert np.array_equal(out, ref[k:k + B]), (w.name, B, k, out, ref[k:k + B])
        assert np.isneginf(ctx.serve_eval(rows[5:6])[0])
        with pytest.raises(api.TinyLensError):                     # more rows than max_rows
            ctx.serve_eval(rows[:17])
        time.sleep(1.0)                                            # the kernel leaves after 0.5 s without a request ...
        assert np.array_equal(ctx.serve_eval(rows[:4]), ref[:4])   # ... and the next request starts it again
    finally:
        ctx.serve_stop()
    # the GPU is free again: ordinary calls run, and serving can be started anew
    again = ctx.loglike(torch.from_numpy(rows).cuda()).cpu().numpy()
    assert np.array_equal(again, ref)
    ctx.serve_start(max_rows=2, idle_timeout_s=0.5)
    try:
        assert np.array_equal(ctx.serve_eval(rows[10:12]), ref[10:12])
    finally:
        ctx.serve_stop()
    ctx.close()                                                    # (tl_destroy stops a serving kernel as well)


@pytest.mark.gpu
@pytest.mark.timeout(120)
def test_serve_latency_and_unsupported_contexts(api):
    import torch
    w = W.workload(1)
    prob = W.make_problem(w, _flat_data)
    ctx = api.LensContext.from_problem(prob)
    row = np.ascontiguousarray(W.batch_rows(w, 1))
    out = np.empty(1, np.float32)
    for _ in range(20):
        ctx.loglike_host(row)
    t0 = time.perf_counter()
    for _ in range(200):
        ctx.loglike_host(row)
    t_host = (time.perf_counter() - t0) / 200
    ctx.serve_start(max_rows=1, idle_timeout_s=0.5)
    try:
        for _ in range(50):
            ctx.serve_eval(row, out)
        t0 = time.perf_counter()
        for _ in range(500):
            ctx.serve_eval(row, out)
        t_serve = (time.perf_counter() - t0) / 500
    finally:
        ctx.serve_stop()
    print("one row, host to host: served %.1f us, tl_loglike_batch_host %.1f us" % (1e6 * t_serve, 1e6 * t_host))
    assert t_serve < 0.8 * t_host
    # FP64 precision, EPL and several lenses are not served
    ctx.set_precision(api.TL_PRECISION_FP64)
    with pytest.raises(api.TinyLensError) as ei:
        ctx.serve_start(4, 0.5)
    assert ei.value.code == api.TL_EINVAL
    ctx.close()
    ctx = api.LensContext.from_problem(W.make_problem(w.with_epl(), _flat_data))
    with pytest.raises(api.TinyLensError):
        ctx.serve_start(4, 0.5)
    ctx.close()
    w3 = W.workload(3).scaled(batch=8, n_lens=2)
    ctx = api.LensContext.from_problem(W.make_problem(w3, _flat_data))
    with pytest.raises(api.TinyLensError):
        ctx.serve_start(4, 0.5)
    ctx.close()
