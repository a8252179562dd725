"""tl_loglike_batch_noalloc (include/tinylens.h): the fixed-amplitude likelihood for callers that may
not allocate.  Its per-row constants live in a fixed array of the library's device image
(TL_NOALLOC_MAX_ROWS rows) instead of pool memory; everything else is tl_loglike_batch's fused path,
so logL must be BITWISE what tl_loglike_batch returns -- the bar tests/test_small_batch_gpu.py holds
the small-batch path to -- on every call, whatever the previous call left in the array.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process (the
array's address is resolved on first use) and after the other tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2503_08586_b200 import workloads as W


def _flat_data(w, psf, row):
    return np.full((w.ny, w.nx), 0.3)


def test_null_context_and_size_limit_are_errors_before_cuda():
    from paper_2503_08586_b200 import api
    L = api.load()
    assert L.tl_loglike_batch_noalloc(None, None, 0, None, None) == api.TL_EINVAL
    assert L.tl_loglike_batch_noalloc(None, None, api.TL_NOALLOC_MAX_ROWS + 1, None, None) == api.TL_EINVAL
    assert api.TL_NOALLOC_MAX_ROWS == 4096


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available()
    from paper_2503_08586_b200 import api as _api
    _api.load()
    return _api


def _rows(w, per_lens, seed_shift, bad_row=None):
    assert w.n_lens == 1
    rows = W.batch_rows(w, per_lens + seed_shift)[seed_shift:].copy()
    if bad_row is not None:
        rows[bad_row, 0] = -1.0                                   # theta_E < 0: invalid row, logL = -inf
    return np.ascontiguousarray(rows)


@pytest.mark.gpu
def test_no_alloc_entry_equals_the_existing_path_on_calls_in_a_row(api):
    import torch
    w = W.workload(1)                                             # BASELINE configs[1], the metric's workload
    ctx = api.LensContext.from_problem(W.make_problem(w, _flat_data))
    w0 = W.workload(0)                                            # a second context shares the array
    ctx0 = api.LensContext.from_problem(W.make_problem(w0, _flat_data))
    assert ctx.info()["path"] == 0 and ctx0.info()["path"] == 0

    # two calls in a row on one stream: 300 rows (one invalid), then 37 other rows over the stale array
    d1 = torch.from_numpy(_rows(w, 300, 0, bad_row=5)).cuda()
    d2 = torch.from_numpy(_rows(w, 37, 300)).cuda()
    o1 = torch.full((d1.shape[0],), 7.0, device="cuda")
    o2 = torch.full((d2.shape[0],), 7.0, device="cuda")
    ctx.loglike_noalloc(d1, o1)
    ctx.loglike_noalloc(d2, o2)
    torch.cuda.synchronize()
    e1, e2 = ctx.loglike(d1), ctx.loglike(d2)                     # fused kernel / small-batch path
    torch.cuda.synchronize()
    assert torch.isneginf(o1[5]) and torch.isfinite(o1[6:]).all() and torch.isfinite(o2).all()
    assert torch.equal(o1, e1), (o1 - e1).abs().max().item()
    assert torch.equal(o2, e2), (o2 - e2).abs().max().item()

    # another context (other image size, other P) in between, then the first one again; the largest
    # batch the array holds
    d0 = torch.from_numpy(_rows(w0, 64, 0)).cuda()
    o0 = torch.empty(d0.shape[0], device="cuda")
    dmax = torch.from_numpy(_rows(w, api.TL_NOALLOC_MAX_ROWS, 0)).cuda()
    omax = torch.empty(dmax.shape[0], device="cuda")
    ctx0.loglike_noalloc(d0, o0)                                  # (first launch of this context's kernels: the driver may load code)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    ctx0.loglike_noalloc(d0, o0)
    ctx.loglike_noalloc(dmax, omax)
    ctx.loglike_noalloc(d2, o2.fill_(7.0))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before            # nothing was taken from the device
    assert torch.equal(o0, ctx0.loglike(d0))
    assert torch.equal(omax, ctx.loglike(dmax))
    assert torch.equal(o2, e2)

    # one row more than the array holds: a clear error, nothing launched, `out` untouched
    dbig = torch.cat([dmax, dmax[:1]]).contiguous()
    obig = torch.full((dbig.shape[0],), 7.0, device="cuda")
    with pytest.raises(api.TinyLensError) as ei:
        ctx.loglike_noalloc(dbig, obig)
    assert ei.value.code == api.TL_ESIZE and "TL_NOALLOC_MAX_ROWS" in str(ei.value)
    torch.cuda.synchronize()
    assert (obig == 7.0).all()
    # B = 0 is the explicit "resolve the address" call
    assert api.load().tl_loglike_batch_noalloc(C.c_void_p(ctx.handle), None, 0, None, None) == api.TL_OK

    # only the FP32 fused path is offered
    ctx.set_precision(api.TL_PRECISION_FP64)
    with pytest.raises(api.TinyLensError) as ei:
        ctx.loglike_noalloc(d2, o2)
    assert ei.value.code == api.TL_EINVAL
    ctx.set_precision(api.TL_PRECISION_FP32)
    ctx.close(); ctx0.close()


@pytest.mark.gpu
def test_no_alloc_entry_rejects_split_path_contexts(api):
    import torch
    w = W.workload(4).scaled(batch=2, n_lens=1)                   # 400 x 400 pixels: the binned image does not fit one CTA
    ctx = api.LensContext.from_problem(W.make_problem(w, _flat_data))
    if ctx.info()["path"] == 0:
        ctx.close()
        pytest.skip("this workload runs the fused path")
    d = torch.from_numpy(_rows(w, 2, 0)).cuda()
    o = torch.empty(d.shape[0], device="cuda")
    with pytest.raises(api.TinyLensError) as ei:
        ctx.loglike_noalloc(d, o)
    assert ei.value.code == api.TL_ESIZE
    ctx.close()
