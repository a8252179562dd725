"""Shared helpers of the GPU parity tests: tolerances (north_star + the derived FP32 floor for
near-truth rows) and oracle-side reference computation."""
import numpy as np

# north_star: per-pixel |delta| <= 1e-5 * image peak; |delta logL| <= max(1e-3, 1e-6 |logL|)
PIX_TOL = 1e-5
LOGL_ABS, LOGL_REL = 1e-3, 1e-6
# FP32 evaluation of a Sersic sample carries a relative error of a few
# ulp amplified by b_n u (the exponent), i.e. eps_sample <~ 2^-20; a pixel is the mean of S^2
# samples and the PSF averages further.  To first order  delta logL = sum_i z_i SNR_i eps_i
# (z = (d - m)/sigma, SNR = m/sigma), so for near-truth rows -- where |logL| is small only
# because -chi^2/2 and the Eq. 5 normalisation cancel -- the bound that FP32 arithmetic can
# meet is  4 * eps_pix * sqrt(sum_i z_i^2 SNR_i^2),  eps_pix = 2^-20 / S.
EPS_SAMPLE = 2.0 ** -20


def logl_tol(oll):
    return np.maximum(LOGL_ABS, LOGL_REL * np.abs(oll))


def fp32_floor(oimg, data, noise, S):
    """4 eps_pix sqrt(sum z^2 SNR^2) per row; oimg [B,ny,nx] float64 oracle images."""
    sig = np.asarray(noise, np.float64)
    z = (np.asarray(data, np.float64) - oimg) / sig
    snr = oimg / sig
    return 4.0 * (EPS_SAMPLE / S) * np.sqrt(np.sum((z * snr) ** 2, axis=(1, 2)))


def oracle_reference(orc, w, prob, rows):
    cfg = orc.config_of(w)
    oll, _ = orc.loglike_batch(cfg, prob.psf, prob.data, prob.noise, rows, n_lens=w.n_lens)
    oim = orc.render_batch(cfg, prob.psf, rows, n_lens=w.n_lens)
    return oll, oim


def rows_with_near(W, w, prob, n_prior, n_near):
    """[lens0: n_prior prior draws, n_near near-truth rows][lens1: ...] and the near mask."""
    rows = W.batch_rows(w, n_prior)
    near = W.near_truth_rows(prob, n_near)
    L = w.n_lens
    allrows = np.concatenate([np.concatenate([rows[l * n_prior:(l + 1) * n_prior],
                                              near[l * n_near:(l + 1) * n_near]]) for l in range(L)])
    per = n_prior + n_near
    isnear = (np.arange(len(allrows)) % per) >= n_prior
    return np.ascontiguousarray(allrows), isnear
