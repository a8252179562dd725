"""Shared helpers of the GPU parity tests: tolerances (north_star + the derived FP32 floor for
near-truth rows) and oracle-side reference computation."""
import numpy as np

# north_star: per-pixel |delta| <= 1e-5 * image peak; |delta logL| <= max(1e-3, 1e-6 |logL|)
PIX_TOL = 1e-5
LOGL_ABS, LOGL_REL = 1e-3, 1e-6
# near the truth |logL| is small only because -chi^2/2 and the Eq. 5
# normalisation cancel, while the terms being summed stay large (chi^2 ~ 1e4, sum SNR^2 ~ 1e8),
# so an absolute 1e-3 asks for ~1e-8 relative accuracy of every bright pixel -- below the FP32
# resolution of the pixel value itself.  To first order  delta logL = sum_i z_i SNR_i eps_i
# (z = (d - m)/sigma, SNR = m/sigma, eps = relative error of pixel i).  The FP32 / MUFU
# evaluation of a Sersic sample (profiles/r1_mufu_accuracy.md) has
#   * a random relative error of rms <= 2^-21 per sample (measured 2e-7 .. 5e-7), averaged over
#     the S^2 samples of a pixel, plus the FP32 roundings of the S^2-term bin sum and of the
#     K^2-term convolution sum, which do not shrink with S (measured 1.5e-7 per pixel at
#     S = 4, K = 21):   eps_rnd = 2^-21 / S + 2^-22,
#   * a systematic relative error |eps_coh| <= 2^-22 (measured <= 1.5e-7; MUFU.LG2 / MUFU.EX2
#     biases amplified by b_n u), coherent over the image,
# hence the bound that FP32 arithmetic can meet on such rows,
#   tol = max(north_star, eps_coh |sum_i z_i SNR_i| + 5 eps_rnd sqrt(sum_i z_i^2 SNR_i^2))   (5 sigma: several hundred rows are tested).
EPS_RND = 2.0 ** -21
EPS_COH = 2.0 ** -22
EPS_ACC = 2.0 ** -22


def logl_tol(oll):
    return np.maximum(LOGL_ABS, LOGL_REL * np.abs(oll))


def fp32_floor(oimg, data, noise, S):
    """eps_coh |sum z SNR| + 5 (eps_rnd/S + eps_acc) sqrt(sum z^2 SNR^2) per row; oimg [B,ny,nx] float64 oracle images."""
    sig = np.asarray(noise, np.float64)
    z = (np.asarray(data, np.float64) - oimg) / sig
    snr = oimg / sig
    coh = EPS_COH * np.abs(np.sum(z * snr, axis=(1, 2)))
    rnd = 5.0 * (EPS_RND / S + EPS_ACC) * np.sqrt(np.sum((z * snr) ** 2, axis=(1, 2)))
    return coh + rnd


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
