"""Small-batch path (NEXT-4): fewer rows than SMs are spread over many CTAs per row; the result
must be BITWISE the fused kernel's (include/tinylens.h: the value of a row does not depend on the
batch it is evaluated in)."""
import os

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


def _zero_render(w, psf, row):
    return np.full((w.ny, w.nx), 0.3)


def _contexts(api, prob):
    small = api.LensContext.from_problem(prob)
    fused = api.LensContext.from_problem(prob, options={"small_batch_rows": 0})     # fused path whatever B
    return small, fused


CASES = [
    W.workload(0), W.workload(1), W.workload(1).with_epl(), W.workload(3).scaled(batch=8, n_lens=2),
    W.Workload(index=7, name="odd", ny=37, nx=45, pix_scale=0.11, supersample=3, psf_size=15, psf_kind="moffat",
               psf_fwhm=0.3, psf_beta=2.5, n_lens_light=1, n_source=2, noise_bg=0.05, noise_exptime=150.0,
               source_amp=(1.0, 20.0), batch=16),
    # S = 2 with two sources and a 21 x 21 PSF: the three-CTAs-per-SM variant of the fused kernel (no 31 / 41 blocks)
    W.Workload(index=7, name="s2-two-sources", ny=48, nx=56, pix_scale=0.09, supersample=2, psf_size=21, psf_kind="gaussian",
               psf_fwhm=0.25, psf_beta=0.0, n_lens_light=1, n_source=2, noise_bg=0.05, noise_exptime=300.0,
               source_amp=(1.0, 20.0), batch=16),
    W.Workload(index=7, name="zero-edge", ny=20, nx=18, pix_scale=0.2, supersample=2, psf_size=5, psf_kind="gaussian",
               psf_fwhm=0.4, psf_beta=0.0, n_lens_light=0, n_source=1, noise_bg=0.05, noise_exptime=0.0,
               source_amp=(5.0, 5.0), batch=16, edge_mode=W.EDGE_ZERO),
]


@pytest.mark.parametrize("w", CASES, ids=lambda w: "%s%s" % (w.name, "-epl" if w.mass_model else ""))
def test_small_batches_equal_the_fused_kernel_bitwise(api, w):
    import torch
    prob = W.make_problem(w, _zero_render)
    small, fused = _contexts(api, prob)
    n_sm = small.info()["n_sm"]
    # (up to 16 rows per call: one pair of sub-samples per lane, trace_pairs_kernel, where S is even)
    for per_lens in (1, 2, 3, 8, 16 // w.n_lens, 17, n_sm // 2 // w.n_lens):
        rows = W.batch_rows(w, per_lens)
        rows[0, 0] = -1.0 if per_lens == 3 else rows[0, 0]                # an invalid row in one of the batches
        if per_lens in (2, 8):                                            # q = 0.4: the q < 0.5 branch of the SIE
            rows[-1, 1], rows[-1, 2] = 0.3, -0.305
        d = torch.from_numpy(rows).cuda()
        a, b = small.loglike(d), fused.loglike(d)
        ia, ib = small.render(d), fused.render(d)
        torch.cuda.synchronize()
        assert torch.equal(a, b), (w.name, per_lens, (a - b).abs().max().item())
        assert torch.equal(torch.nan_to_num(ia, nan=-7.0), torch.nan_to_num(ib, nan=-7.0))
        if per_lens == 3:
            assert torch.isneginf(a[0]) and torch.isnan(ia[0]).all()
    # one row more than the limit takes the fused kernel on both contexts
    small.close(); fused.close()


def test_small_batch_handoff_stress(api):
    """compute-sanitizer (racecheck) is closed on this GPU pool, so the cross-CTA hand-off of
    conv_small_kernel (__threadfence + a finished-band counter per row; the row's last band reduces
    the stored terms) and the per-row work-queue heads of trace_kernel are hammered instead: 300
    calls of varying small sizes on two streams at once, every result bitwise equal to the fused kernel's."""
    import torch
    w = [c for c in CASES if c.name == "odd"][0]
    prob = W.make_problem(w, _zero_render)
    small, fused = _contexts(api, prob)
    assert small.info()["small_batch_rows"] > 0
    rows = W.batch_rows(w, 40)
    d = torch.from_numpy(rows).cuda()
    want = fused.loglike(d).clone()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    outs = []
    for it in range(150):
        n1, n2 = 1 + (it * 7) % 40, 1 + (it * 11) % 37
        a = small.loglike(d[:n1], stream=s1)
        b = small.loglike(d[40 - n2:], stream=s2)
        outs.append((n1, n2, a, b))
    torch.cuda.synchronize()
    for n1, n2, a, b in outs:
        assert torch.equal(a, want[:n1]) and torch.equal(b, want[40 - n2:]), (n1, n2)
    small.close(); fused.close()


def test_small_batch_latency(api):
    """A handful of rows must not cost a whole row-time of one SM (0.18 ms on configs[1])."""
    import torch
    w = W.workload(1)
    prob = W.make_problem(w, _zero_render)
    small, fused = _contexts(api, prob)
    d = torch.from_numpy(W.batch_rows(w, 4)).cuda()
    out = torch.empty(4, device="cuda")

    def best(ctx):
        for _ in range(5):
            ctx.loglike(d, out)
        torch.cuda.synchronize()
        ts = []
        for _ in range(20):
            e0, e1 = torch.cuda.Event(True), torch.cuda.Event(True)
            e0.record(); ctx.loglike(d, out); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return min(ts)
    ts, tf = best(small), best(fused)
    print("B = 4 on configs[1]: small-batch path %.3f ms, fused kernel %.3f ms" % (ts, tf))
    assert ts < 0.6 * tf
    # the one-row call (30 us measured; the round-1 verdict asked for <= 40 us)
    d = d[:1].contiguous()
    out = out[:1]
    t1 = min(best(small) for _ in range(3))
    print("B = 1 on configs[1]: %.1f us" % (1e3 * t1))
    assert t1 < 0.040
    small.close(); fused.close()
