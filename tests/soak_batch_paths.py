"""Soak run (not collected by pytest): `python tests/soak_batch_paths.py FIRST LAST` -- for seeded random mid-size
shapes (40..120 pixels a side, S = 2 / 4, PSF 5 / 15 / 21, SIE, one lens: the shapes on which the small-batch path, the
tail routing of the last wave, tl_loglike_batch_noalloc and the serving kernel are all available) the value of a row
must not depend on how it is asked for: a 310-row call is the reference, and calls of 1, 5, 17, 74, 75, 149 and 200 of
its rows, the allocation-free entry point and served requests of 1, 3 and 16 rows must return the same bits; the
linear-amplitude mode likewise for 1, 17, 149 and 200 rows, the MGE mode for 1, 7 and 74 rows against 200.  With tl_options.debug_canaries on; prints the seeds that fail."""
import os
import sys
import traceback

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np
import torch

from paper_2503_08586_b200 import api, workloads as W

s0, s1 = int(sys.argv[1]), int(sys.argv[2])
bad = 0
for seed in range(s0, s1):
    rng = np.random.default_rng(70000 + seed)
    kw = dict(index=100 + seed % 50, name="soak", ny=int(rng.integers(40, 121)), nx=int(rng.integers(40, 121)),
              supersample=int(rng.choice([2, 4])), psf_size=int(rng.choice([5, 15, 21])), pix_scale=float(rng.uniform(0.04, 0.12)),
              n_lens_light=int(rng.integers(0, 2)), n_source=int(rng.integers(1, 3)), edge_mode=int(rng.integers(0, 2)),
              psf_kind="gaussian", psf_fwhm=float(rng.uniform(0.1, 0.3)), psf_beta=0.0, noise_bg=0.05, noise_exptime=100.0,
              source_amp=(1.0, 20.0), batch=310)
    try:
        w = W.Workload(**kw)
        prob = W.make_problem(w, lambda ww, psf, row: np.full((ww.ny, ww.nx), 0.3))
        ctx = api.LensContext.from_problem(prob, options={"debug_canaries": 1})
        rows = W.batch_rows(w, 310)
        rows[3, 0] = -1.0
        d = torch.from_numpy(np.ascontiguousarray(rows)).cuda()
        ref = ctx.loglike(d)
        for B in (1, 5, 17, 74, 75, 149, 200):
            got = ctx.loglike(d[:B].contiguous())
            assert torch.equal(got, ref[:B]), ("loglike", B)
            out = torch.empty(B, device="cuda")
            assert torch.equal(ctx.loglike_noalloc(d[:B].contiguous(), out), ref[:B]), ("noalloc", B)
        refl, refa = ctx.loglike_linear(d)
        for B in (1, 17, 149, 200):
            gl, ga = ctx.loglike_linear(d[:B].contiguous())
            assert torch.equal(gl, refl[:B]) and torch.equal(torch.nan_to_num(ga, nan=-7.0), torch.nan_to_num(refa[:B], nan=-7.0)), ("linear", B)
        if w.n_lens_light == 1:                                   # MGE: a few rows (bands of gauss_conv_kernel, thin tiles) against many
            ctx.set_mge(W.mge_sigmas(w, int(rng.integers(3, 11))))
            rm, ra = ctx.loglike_mge(d[:200].contiguous())
            for B in (1, 7, 74):
                gm, ga = ctx.loglike_mge(d[:B].contiguous())
                assert torch.equal(gm, rm[:B]) and torch.equal(torch.nan_to_num(ga, nan=-7.0), torch.nan_to_num(ra[:B], nan=-7.0)), ("mge", B)
        torch.cuda.synchronize()
        refh = ref.cpu().numpy()
        ctx.serve_start(16, 0.5)
        try:
            for k, B in ((0, 1), (2, 3), (20, 16)):
                assert np.array_equal(ctx.serve_eval(rows[k:k + B]), refh[k:k + B]), ("serve", B)
        finally:
            ctx.serve_stop()
        assert ctx.canary_errors() == 0, "canary"
        ctx.close()
    except Exception as e:
        bad += 1
        print("SEED %d FAILED: %r  kw=%r" % (seed, e, kw), flush=True)
        traceback.print_exc(limit=2)
print("soak %d..%d done, %d failures" % (s0, s1, bad))
