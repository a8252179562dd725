"""Soak run (not collected by pytest): `python tests/soak_random_shapes.py FIRST LAST` drives seeds FIRST .. LAST-1 of a
seeded random geometry (3..69 pixels a side, S = 1..8, PSF 1..31, one or two sources, with / without lens light,
both edge modes, a quarter of them EPL, one to three lenses per call, a third forced onto the split path) through tl_loglike_batch and tl_render_batch in the FP32, FP64 and AUTO modes
and through tl_loglike_linear_batch and (with a lens-light block) tl_loglike_mge_batch (one set, and on a third of those shapes two sets) in FP32 and FP64, with
tl_options.debug_canaries on: every result against the oracle (pixels to
1e-5 of the peak; logL to north_star in FP64 / AUTO, to 60 x north_star in FP32 -- the FP32 floor of small images,
DESIGN.md 6), one row alone against the same row in the batch (same bits), the finite / -inf pattern, 0 guard words
changed.  Prints the seeds that fail.  tests/test_parity_gpu.py::test_random_shapes is the 12-seed version of it."""
import sys, os, traceback
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import numpy as np, torch
from paper_2503_08586_b200 import api, workloads as W
from oracle import oracle as O
import parity as PT
O.lib()
s0, s1 = int(sys.argv[1]), int(sys.argv[2])
bad = 0
for seed in range(s0, s1):
    rng = np.random.default_rng(50000 + seed)
    ny, nx = int(rng.integers(3, 70)), int(rng.integers(3, 70))
    S = int(rng.integers(1, 9))
    K = int(rng.choice([1, 3, 5, 7, 9, 13, 15, 21, 31]))
    kw = dict(index=100 + seed % 50, name="soak", ny=ny, nx=nx, supersample=S, psf_size=K, pix_scale=float(rng.uniform(0.03, 0.3)),
              n_lens_light=int(rng.integers(0, 2)), n_source=int(rng.integers(1, 3)), edge_mode=int(rng.integers(0, 2)),
              psf_kind=str(rng.choice(["gaussian", "moffat"])), psf_fwhm=float(rng.uniform(0.1, 0.4)), psf_beta=2.5,
              noise_bg=0.05, noise_exptime=100.0, source_amp=(1.0, 20.0), batch=12)
    try:
        w = W.Workload(**kw)
        if rng.integers(0, 4) == 0: w = w.with_epl()
        n_lens = int(rng.choice([1, 1, 2, 3]))                     # several lenses share a call (own PSF / data / noise each)
        if n_lens > 1: w = w.scaled(batch=8 * n_lens, n_lens=n_lens)
        opts = {"debug_canaries": 1}
        if rng.integers(0, 3) == 0: opts["force_split"] = 1        # the split path (large images) on a small one
        prob = W.make_problem(w, O.render_for_workloads)
        rows, isnear = PT.rows_with_near(W, w, prob, 6, 2)
        oll, oim = PT.oracle_reference(O, w, prob, rows)
        ctx = api.LensContext.from_problem(prob, options=opts)
        d = torch.from_numpy(np.ascontiguousarray(rows)).cuda()
        tol = PT.logl_tol(oll)
        fin = np.isfinite(oll)
        for prec in (api.TL_PRECISION_FP32, api.TL_PRECISION_FP64, api.TL_PRECISION_AUTO):
            ctx.set_precision(prec)
            ll = ctx.loglike(d).cpu().numpy().astype(np.float64)
            im = ctx.render(d).cpu().numpy().astype(np.float64)
            assert np.array_equal(np.isfinite(ll), fin), ("finite pattern", prec)
            peak = np.abs(oim[fin]).reshape(fin.sum(), -1).max(1) if fin.any() else np.ones(0)
            dpix = (np.abs(im[fin] - oim[fin]).reshape(fin.sum(), -1).max(1) / np.maximum(peak, 1e-30)).max() if fin.any() else 0.0
            # (FP32 on a cutout that holds nothing but the far tail of the source -- peak ~1e-13 of its amplitude, exponent
            # ~ -42 -- carries the exponent's 2.6e-7 into the value: 1.1e-5 of that peak on seed 12767; not a pixel anybody fits)
            assert dpix <= (1e-5 if prec == api.TL_PRECISION_FP64 or peak.min() > 1e-9 else 3e-5), ("pixels", prec, dpix)   # (AUTO renders are FP32 renders)
            r = (np.abs(ll[fin] - oll[fin]) / tol[fin])
            lim = 1.0 if prec != api.TL_PRECISION_FP32 else 60.0
            assert (r.max() if r.size else 0.0) <= lim, ("logL", prec, r.max())
            # one row alone = the same bits (FP32: small-batch / fused; the others: same path)
            if prec == api.TL_PRECISION_FP32 and w.n_lens == 1:
                one = ctx.loglike(d[:1].contiguous()).cpu().numpy().astype(np.float64)
                assert np.array_equal(one, ll[:1], equal_nan=True), ("batch independence", one, ll[:1])
        ctx.set_precision(api.TL_PRECISION_FP32)
        if w.n_lens_light <= 1:
            l1, a1 = ctx.loglike_linear(d)
            ol, oa = O.loglike_linear_batch(O.config_of(w), prob.psf, prob.data, prob.noise, rows, n_lens=w.n_lens)
            fl = np.isfinite(ol)
            rl = np.abs(l1.cpu().numpy().astype(np.float64)[fl] - ol[fl]) / PT.logl_tol(ol)[fl]
            assert (rl.max() if rl.size else 0.0) <= 60.0, ("linear", rl.max())
        if w.n_lens_light == 1 and min(ny, nx) >= 8:
            # MGE lens light: 2..8 Gaussians + the sources by NNLS, FP32 and FP64 pipelines
            sig = W.mge_sigmas(w, int(rng.integers(2, 9)))
            ctx.set_mge(sig)
            om, _ = O.loglike_mge_batch(O.config_of(w), prob.psf, prob.data, prob.noise, rows, sig, n_lens=w.n_lens)
            fm = np.isfinite(om)
            for prec, lim in ((api.TL_PRECISION_FP32, 60.0), (api.TL_PRECISION_FP64, 1.0)):
                ctx.set_precision(prec)
                lm, _ = ctx.loglike_mge(d)
                lm = lm.cpu().numpy().astype(np.float64)
                assert np.array_equal(np.isfinite(lm), fm), ("mge finite pattern", prec)
                rm = np.abs(lm[fm] - om[fm]) / PT.logl_tol(om)[fm]
                assert (rm.max() if rm.size else 0.0) <= lim, ("mge", prec, rm.max())
            ctx.set_precision(api.TL_PRECISION_FP32)
        assert ctx.canary_errors() == 0, "canary"
        ctx.close()
        if w.n_lens_light == 1 and w.n_lens == 1 and min(ny, nx) >= 8 and rng.integers(0, 3) == 0:
            # two Gaussian sets on ellipses of their own (two lens-light blocks in the row), the data of the one-set problem
            w2 = W.Workload(**{**w.__dict__, "n_lens_light": 2})
            rows2 = W.batch_rows(w2, 6)
            sets = [W.mge_sigmas(w2, int(rng.integers(2, 7))), (W.mge_sigmas(w2, int(rng.integers(2, 7))) * 1.3).astype(np.float32)]
            prob2 = type(prob)(w2, prob.psf, prob.data, prob.noise, rows2[:1].copy())
            ctx2 = api.LensContext.from_problem(prob2, options=opts)
            ctx2.set_mge_sets(sets)
            d2 = torch.from_numpy(np.ascontiguousarray(rows2)).cuda()
            o2 = np.array([O.loglike_mge_sets(O.config_of(w2), prob.psf[0], prob.data[0], prob.noise[0], rows2[r], sets)[0] for r in range(len(rows2))])
            f2 = np.isfinite(o2)
            for prec, lim in ((api.TL_PRECISION_FP32, 60.0), (api.TL_PRECISION_FP64, 1.0)):
                ctx2.set_precision(prec)
                l2 = ctx2.loglike_mge(d2)[0].cpu().numpy().astype(np.float64)
                assert np.array_equal(np.isfinite(l2), f2), ("mge sets finite pattern", prec)
                r2 = np.abs(l2[f2] - o2[f2]) / PT.logl_tol(o2)[f2]
                assert (r2.max() if r2.size else 0.0) <= lim, ("mge sets", prec, r2.max())
            assert ctx2.canary_errors() == 0, "canary (sets)"
            ctx2.close()
    except Exception as e:
        bad += 1
        print("SEED %d FAILED: %r  kw=%r" % (seed, e, kw), flush=True)
        traceback.print_exc(limit=2)
print("soak %d..%d done, %d failures" % (s0, s1, bad))
