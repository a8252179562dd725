"""Pins for the FP64 oracle (oracle/tl_oracle.c): closed forms, invariants, library routines,
brute force -- things the paper and the mathematics fix, none of them the oracle's own formula
retyped.  Each test names the passage (PAPER.md line / equation) and the SURVEY.md 8(c) pin.
CPU only; runs in seconds.
"""
import math
import os

import numpy as np
import pytest
import scipy.signal
import scipy.special

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


def _gold():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            out[k] = np.array([float(x) for x in v])
    return out


# ------------------------------------------------------------------ Eq. 9: b_n

def test_bn_closed_forms(orc):
    # PAPER.md:139 Eq. 9.  n = 1/2: gamma(1,b) = 1 - e^-b = 1/2 -> b = ln 2 (closed form).
    assert abs(orc.bn(0.5) - math.log(2.0)) < 1e-14
    # textbook values (exponential n=1, de Vaucouleurs n=4)
    assert abs(orc.bn(1.0) - 1.678346990016661) < 1e-13
    assert abs(orc.bn(4.0) - 7.669249442500804) < 1e-12


def test_bn_against_library_inverse(orc):
    # P(2n, b_n) = 1/2: scipy's inverse regularised incomplete gamma is an independent routine.
    for n in [0.3, 0.36, 0.5, 0.77, 1.0, 1.5, 2.5, 4.0, 6.0, 8.0, 10.0]:
        ref = scipy.special.gammaincinv(2.0 * n, 0.5)
        assert abs(orc.bn(n) - ref) < 1e-12 * max(1.0, ref)
        assert abs(scipy.special.gammainc(2.0 * n, orc.bn(n)) - 0.5) < 1e-13


def test_gammainc_series_against_library(orc):
    for a, x in [(0.6, 0.1), (1.0, 0.7), (3.0, 2.5), (8.0, 7.7), (20.0, 19.0), (2.0, 5.0)]:
        assert abs(orc.gammainc_p(a, x) - scipy.special.gammainc(a, x)) < 1e-13


# ------------------------------------------------------------------ Eq. 11 inverse

def test_shape_roundtrip(orc):
    # PAPER.md:152 Eq. 11 forward map, inverted by the oracle.
    rng = np.random.default_rng(1)
    for _ in range(50):
        q, phi = rng.uniform(0.2, 1.0), rng.uniform(-math.pi / 2, math.pi / 2)
        e = (1 - q) / (1 + q)
        q2, phi2 = orc.shape(e * math.cos(2 * phi), e * math.sin(2 * phi))
        assert abs(q2 - q) < 1e-14
        if q < 0.999:
            assert abs(math.remainder(phi2 - phi, math.pi)) < 1e-12
    assert orc.shape(0.0, 0.0) == (1.0, 0.0)


# ------------------------------------------------------------------ Eq. 12: SIE

def test_sis_closed_form(orc):
    # q = 1: alpha = theta_E (theta - c)/|theta - c|   (SIS; PAPER.md:160 gamma = 2)
    rng = np.random.default_rng(2)
    for _ in range(100):
        te, cx, cy = rng.uniform(0.5, 2), rng.uniform(-.3, .3), rng.uniform(-.3, .3)
        x, y, phi = rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(0, math.pi)
        ax, ay = orc.sie_deflection(te, 1.0, phi, cx, cy, x, y)
        r = math.hypot(x - cx, y - cy)
        assert abs(ax - te * (x - cx) / r) < 1e-12 and abs(ay - te * (y - cy) / r) < 1e-12


def _kappa(te, q, phi, cx, cy, x, y):
    # PAPER.md:158 Eq. 12 with gamma = 2 and R -> R_p of Eq. 10
    c, s = math.cos(phi), math.sin(phi)
    xp = (x - cx) * c + (y - cy) * s
    yp = -(x - cx) * s + (y - cy) * c
    return 0.5 * te / math.sqrt(q * xp * xp + yp * yp / q)


def test_sie_divergence_is_2kappa_and_curl_free(orc):
    # 1/2 div(alpha) = kappa (Poisson equation of lensing) and curl(alpha) = 0, by 4th-order
    # central differences; kappa from Eq. 12 (gamma = 2) with R -> R_p of Eq. 10.
    rng = np.random.default_rng(3)
    h = 1e-3

    def d(f, k):
        return (-f(2 * h)[k] + 8 * f(h)[k] - 8 * f(-h)[k] + f(-2 * h)[k]) / (12 * h)
    n = 0
    for _ in range(80):
        te, q = rng.uniform(0.5, 2), rng.uniform(0.25, 0.98)
        phi, cx, cy = rng.uniform(0, math.pi), rng.uniform(-.2, .2), rng.uniform(-.2, .2)
        x, y = rng.uniform(-3, 3), rng.uniform(-3, 3)
        if math.hypot(x - cx, y - cy) < 0.3:
            continue
        n += 1
        fx = lambda t: orc.sie_deflection(te, q, phi, cx, cy, x + t, y)
        fy = lambda t: orc.sie_deflection(te, q, phi, cx, cy, x, y + t)
        k = _kappa(te, q, phi, cx, cy, x, y)
        assert abs(0.5 * (d(fx, 0) + d(fy, 1)) - k) < 1e-7 * k
        assert abs(d(fy, 0) - d(fx, 1)) < 1e-8
    assert n > 50


def test_sie_major_axis_closed_form(orc):
    # on the major axis (y' = 0): alpha_x' = theta_E sqrt(q)/q' atan(q'/q) sign(x'), alpha_y' = 0
    for q in [0.3, 0.6, 0.9]:
        for phi in [0.0, 0.4, 2.0]:
            te, t = 1.3, 0.9
            for sgn in (1, -1):
                x, y = sgn * t * math.cos(phi), sgn * t * math.sin(phi)
                ax, ay = orc.sie_deflection(te, q, phi, 0, 0, x, y)
                axp = ax * math.cos(phi) + ay * math.sin(phi)
                ayp = -ax * math.sin(phi) + ay * math.cos(phi)
                qp = math.sqrt(1 - q * q)
                assert abs(axp - sgn * te * math.sqrt(q) / qp * math.atan(qp / q)) < 1e-12
                assert abs(ayp) < 1e-12


def test_sie_minor_axis_closed_form(orc):
    # on the minor axis (x' = 0): alpha_y' = theta_E sqrt(q)/q' atanh(q') sign(y')
    q, phi, te = 0.55, 0.7, 1.1
    qp = math.sqrt(1 - q * q)
    x, y = -0.8 * math.sin(phi), 0.8 * math.cos(phi)
    ax, ay = orc.sie_deflection(te, q, phi, 0, 0, x, y)
    ayp = -ax * math.sin(phi) + ay * math.cos(phi)
    assert abs(ayp - te * math.sqrt(q) / qp * math.atanh(qp)) < 1e-12


def test_sie_einstein_normalisation(orc):
    # flux of alpha through the ellipse q x'^2 + y'^2/q = theta_E^2 is 2 * integral(kappa) = 2 pi theta_E^2
    te, q, phi, cx, cy = 1.2, 0.6, 0.5, 0.1, -0.05
    n = 20000
    t = (np.arange(n) + 0.5) * 2 * math.pi / n
    a, b = te / math.sqrt(q), te * math.sqrt(q)
    xp, yp = a * np.cos(t), b * np.sin(t)
    # outward normal * dl = (dy', -dx') dt
    nxp, nyp = b * np.cos(t), a * np.sin(t)
    c, s = math.cos(phi), math.sin(phi)
    tot = 0.0
    for i in range(n):
        x = cx + xp[i] * c - yp[i] * s
        y = cy + xp[i] * s + yp[i] * c
        ax, ay = orc.sie_deflection(te, q, phi, cx, cy, x, y)
        axp, ayp = ax * c + ay * s, -ax * s + ay * c
        tot += (axp * nxp[i] + ayp * nyp[i]) * (2 * math.pi / n)
    assert abs(tot - 2 * math.pi * te * te) < 1e-8


def test_sie_q_to_one_is_continuous_and_centre_is_zero(orc):
    a0 = orc.sie_deflection(1.0, 1.0, 0.3, 0, 0, 0.7, -0.4)
    a1 = orc.sie_deflection(1.0, 1.0 - 1e-9, 0.3, 0, 0, 0.7, -0.4)
    assert abs(a0[0] - a1[0]) < 1e-8 and abs(a0[1] - a1[1]) < 1e-8
    assert orc.sie_deflection(1.0, 0.7, 0.3, 0.1, 0.2, 0.1, 0.2) == (0.0, 0.0)


# ------------------------------------------------------------------ Eq. 13/14: shear, Eq. 1: ray-trace

def test_shear_is_gradient_of_eq13(orc):
    # psi_ext = -1/2 gamma theta^2 cos 2(phi - phi_ext)   (Eq. 13)
    g, pe = 0.07, 0.6
    g1, g2 = g * math.cos(2 * pe), g * math.sin(2 * pe)       # PAPER.md:189 Eq. 14

    def psi(x, y):
        return -0.5 * g * (x * x + y * y) * math.cos(2 * (math.atan2(y, x) - pe))
    x, y, h = 0.8, -1.3, 1e-5
    ax, ay = orc.shear_deflection(g1, g2, x, y)
    assert abs(ax - (psi(x + h, y) - psi(x - h, y)) / (2 * h)) < 1e-9
    assert abs(ay - (psi(x, y + h) - psi(x, y - h)) / (2 * h)) < 1e-9


def _cfg(orc, n=8, scale=0.25, S=1, nl=0, ns=1, edge=0):
    return orc.config(n, n, scale, S, nl, ns, edge)


def test_sis_ring_maps_to_lens_centre(orc):
    # PAPER.md:54 Eq. 1.  Any point on the SIS Einstein ring maps to the lens centre: with the
    # source centred there, ring pixels show the central brightness I_e e^{b_n}.
    te = 0.875                       # 3.5 pixels of 0.25: pixel centres (+-3.5 px, +-0.5 px) are not on it
    cfg = _cfg(orc, n=8, scale=0.25, S=1)
    # pixel centre (x=0.875, y=0.125)? |.| != te.  Use a grid where a pixel centre is on the ring:
    cfg = orc.config(1, 8, 0.25, 1, 0, 1, 0)      # one row, y = 0; x_j = (j - 3.5) * 0.25
    row = np.array([te, 0, 0, 0, 0, 0, 0, 2.0, 0.3, 1.0, 0, 0, 0, 0], np.float32)
    img = orc.ideal_image(cfg, 0, row)
    peak = 2.0 * math.exp(orc.bn(1.0))
    assert abs(img[0, 7] - peak) < 1e-12 * peak      # x = +0.875 = theta_E
    assert abs(img[0, 0] - peak) < 1e-12 * peak      # x = -0.875
    ax, ay = orc.sie_deflection(te, 1.0, 0.0, 0.1, -0.2, 0.1 + te * 0.6, -0.2 + te * 0.8)
    assert abs(0.1 + te * 0.6 - ax - 0.1) < 1e-15 and abs(-0.2 + te * 0.8 - ay + 0.2) < 1e-15


def test_shear_only_gaussian_source_is_analytic(orc):
    # theta_E = 0: beta = theta + Gamma theta is linear; n = 1/2 Sersic = 2 I_e exp(-ln2 R^2/r_e^2)
    g1, g2 = 0.04, -0.03
    q, phi, re, ie, sx, sy = 0.7, 0.4, 0.5, 3.0, 0.1, -0.15
    e = (1 - q) / (1 + q)
    row = np.array([0, 0, 0, 0, 0, g1, g2, ie, re, 0.5, e * math.cos(2 * phi), e * math.sin(2 * phi), sx, sy],
                   np.float32)
    cfg = orc.config(6, 6, 0.2, 1, 0, 1, 0)
    img = orc.ideal_image(cfg, 0, row)
    r = row.astype(np.float64)
    q64 = (1 - math.hypot(r[10], r[11])) / (1 + math.hypot(r[10], r[11]))
    ph64 = 0.5 * math.atan2(r[11], r[10])
    xs = (np.arange(6) - 2.5) * 0.2
    X, Y = np.meshgrid(xs, xs)
    BX = X + r[5] * X + r[6] * Y
    BY = Y + r[6] * X - r[5] * Y
    x1 = (BX - r[12]) * math.cos(ph64) + (BY - r[13]) * math.sin(ph64)
    x2 = -(BX - r[12]) * math.sin(ph64) + (BY - r[13]) * math.cos(ph64)
    ref = 2 * r[7] * np.exp(-math.log(2) * (q64 * x1 ** 2 + x2 ** 2 / q64) / r[8] ** 2)
    assert np.max(np.abs(img - ref)) < 1e-13


# ------------------------------------------------------------------ Eq. 8/10: Sersic

def _sersic_total_flux(ie, re, n, bn):
    return 2 * math.pi * n * ie * re * re * math.exp(bn) * math.gamma(2 * n) / bn ** (2 * n)


@pytest.mark.parametrize("n,q", [(1.0, 0.6), (0.5, 0.8), (2.0, 1.0)])
def test_sersic_total_and_half_flux(orc, n, q):
    # closed form F = 2 pi n I_e r_e^2 e^b Gamma(2n) / b^(2n), independent of q (Eq. 10 has unit
    # Jacobian); half of it inside R_p < r_e ("exactly half").
    ie, re, phi = 1.0, 0.3, 0.35
    e = (1 - q) / (1 + q)
    N, scale = 500, 0.03 if n < 2 else 0.06
    row = np.array([0, 0, 0, 0, 0, 0, 0, ie, re, n, e * math.cos(2 * phi), e * math.sin(2 * phi), 0, 0], np.float32)
    cfg = orc.config(N, N, scale, 4, 1, 0, 0)
    img = orc.ideal_image(cfg, 0, row)
    F = _sersic_total_flux(ie, re, n, orc.bn(n))
    tot = img.sum() * scale ** 2
    assert abs(tot - F) < (2e-4 if n < 2 else 3e-3) * F
    qq, pp = orc.shape(*row[10:12].astype(np.float64))
    xs = (np.arange(N) - (N - 1) / 2) * scale
    X, Y = np.meshgrid(xs, xs)
    x1 = X * math.cos(pp) + Y * math.sin(pp)
    x2 = -X * math.sin(pp) + Y * math.cos(pp)
    inside = (qq * x1 ** 2 + x2 ** 2 / qq) < re * re
    half = img[inside].sum() * scale ** 2
    assert abs(half - 0.5 * F) < 6e-3 * F          # pixel-edge quantisation of the mask


def test_sersic_value_at_re_and_centre(orc):
    # Eq. 8: I(r_e) = I_e; I(0) = I_e e^{b_n}
    b = orc.bn(2.5)
    assert abs(orc.sersic(1.7, 0.4, 2.5, 1.0, 0.0, 0, 0, 0.4, 0.0) - 1.7) < 1e-14
    assert abs(orc.sersic(1.7, 0.4, 2.5, 0.5, 0.3, 0.1, 0.2, 0.1, 0.2) - 1.7 * math.exp(b)) < 1e-12
    # Eq. 10: on the major axis R_p = sqrt(q) r; on the minor axis r / sqrt(q)
    q, phi = 0.5, 0.6
    v = orc.sersic(1.0, 1.0, 1.0, q, phi, 0, 0, math.cos(phi) / math.sqrt(q), math.sin(phi) / math.sqrt(q))
    assert abs(v - 1.0) < 1e-14
    v = orc.sersic(1.0, 1.0, 1.0, q, phi, 0, 0, -math.sin(phi) * math.sqrt(q), math.cos(phi) * math.sqrt(q))
    assert abs(v - 1.0) < 1e-14


def test_bin_is_mean_erf_closed_form(orc):
    # n = 1/2, q = 1: pixel mean of 2 I_e exp(-ln2 r^2/r_e^2) has an erf closed form; the S x S
    # mean converges to it as O(S^-2): pins "bin = mean of the samples" (G9).
    ie, re, scale, N = 1.5, 0.35, 0.2, 6
    row = np.array([0, 0, 0, 0, 0, 0, 0, ie, re, 0.5, 0, 0, 0.03, -0.02], np.float32)
    r = row.astype(np.float64)
    k = math.sqrt(math.log(2)) / r[8]

    def cell(lo, hi, c):
        return math.sqrt(math.pi) / (2 * k) * (math.erf(k * (hi - c)) - math.erf(k * (lo - c)))
    exact = np.empty((N, N))
    for i in range(N):
        for j in range(N):
            x0, y0 = (j - (N - 1) / 2 - 0.5) * scale, (i - (N - 1) / 2 - 0.5) * scale
            exact[i, j] = 2 * r[7] * cell(x0, x0 + scale, r[12]) * cell(y0, y0 + scale, r[13]) / scale ** 2
    errs = []
    for S in (1, 2, 4, 8):
        img = orc.ideal_image(orc.config(N, N, scale, S, 1, 0, 0), 0, row)
        errs.append(np.max(np.abs(img - exact)))
    for a, b in zip(errs, errs[1:]):
        assert 3.5 < a / b < 4.5
    assert errs[-1] < 1e-3 * exact.max()          # (scale/S)^2/24 * laplacian ~ 1.6e-3 at S = 8


def test_bin_leaves_constant_image_unchanged(orc):
    row = np.array([0, 0, 0, 0, 0, 0, 0, 2.0, 1e6, 0.5, 0, 0, 0, 0], np.float32)
    for S in (1, 2, 3, 4, 8):
        img = orc.ideal_image(orc.config(5, 7, 0.1, S, 1, 0, 0), 0, row)
        assert np.max(np.abs(img - 4.0)) < 1e-10


# ------------------------------------------------------------------ Eq. 3: PSF

def test_psf_delta_is_identity_both_modes(orc):
    rng = np.random.default_rng(5)
    K = 5
    psf = np.zeros((K, K), np.float32)
    psf[2, 2] = 1.0
    ext = rng.normal(size=(6 + 4, 7 + 4))
    assert np.array_equal(orc.convolve(6, 7, 2, ext, psf), ext[2:-2, 2:-2])
    img = rng.normal(size=(6, 7))
    assert np.array_equal(orc.convolve(6, 7, 0, img, psf), img)


def test_psf_orientation_delta_image(orc):
    # true convolution (Eq. 3): a delta image reproduces the kernel unflipped
    # around the delta; delta at (2,2), h = 1 -> output (1,2) is K[0,1].
    K = np.arange(1, 10, dtype=np.float32).reshape(3, 3)
    img = np.zeros((5, 5))
    img[2, 2] = 1.0
    out = orc.convolve(5, 5, 0, img, K)
    assert np.array_equal(out[1:4, 1:4], K.astype(np.float64))
    assert out[1, 2] == K[0, 1]


def test_psf_against_library_and_brute_force(orc):
    rng = np.random.default_rng(6)
    for (ny, nx, K) in [(4, 5, 3), (7, 6, 5), (9, 9, 7)]:
        h = (K - 1) // 2
        psf = rng.uniform(size=(K, K)).astype(np.float32)
        ext = rng.normal(size=(ny + 2 * h, nx + 2 * h))
        ref = scipy.signal.convolve2d(ext, psf.astype(np.float64), mode="valid")
        assert np.max(np.abs(orc.convolve(ny, nx, h, ext, psf) - ref)) < 1e-13
        img = rng.normal(size=(ny, nx))
        ref0 = scipy.signal.convolve2d(img, psf.astype(np.float64), mode="same")
        assert np.max(np.abs(orc.convolve(ny, nx, 0, img, psf) - ref0)) < 1e-13
        # brute-force 4-loop straight from Eq. 3
        bf = np.zeros((ny, nx))
        for i in range(ny):
            for j in range(nx):
                for a in range(K):
                    for b in range(K):
                        bf[i, j] += float(psf[a, b]) * ext[i - (a - h) + h, j - (b - h) + h]
        assert np.max(np.abs(orc.convolve(ny, nx, h, ext, psf) - bf)) < 1e-14


def test_psf_separable_gaussian(orc):
    g = np.exp(-0.5 * (np.arange(7) - 3.0) ** 2 / 1.3 ** 2).astype(np.float32)
    g64 = g.astype(np.float64)
    psf64 = np.outer(g64, g64)
    psf = psf64.astype(np.float32)
    rng = np.random.default_rng(7)
    ext = rng.normal(size=(10 + 6, 8 + 6))
    rows = np.apply_along_axis(lambda v: np.convolve(v, g64, mode="valid"), 1, ext)
    both = np.apply_along_axis(lambda v: np.convolve(v, g64, mode="valid"), 0, rows)
    assert np.max(np.abs(orc.convolve(10, 8, 3, ext, psf) - both)) < 1e-6     # psf rounded to FP32


# ------------------------------------------------------------------ Eq. 5: likelihood

def test_chi2_zero_and_n(orc):
    rng = np.random.default_rng(8)
    model = rng.uniform(1, 2, size=(6, 5)).astype(np.float32)
    sig = rng.uniform(0.1, 0.3, size=(6, 5)).astype(np.float32)
    m64 = model.astype(np.float64)
    C = np.sum(np.log(2 * math.pi * sig.astype(np.float64) ** 2))
    assert orc.chi2_from_image(m64, model, sig) == 0.0
    assert abs(orc.loglike_from_image(m64, model, sig) + 0.5 * C) < 1e-12
    # data = model + sigma everywhere -> chi^2 = N  (power-of-two sigma keeps it exact)
    sig2 = np.full((6, 5), 0.25, np.float32)
    data = (model + sig2).astype(np.float32)
    assert abs(orc.chi2_from_image(data.astype(np.float64) - 0.25, data, sig2) - 30.0) < 1e-12


def test_loglike_is_log_of_eq5_product(orc):
    # PAPER.md:82 Eq. 5 as printed: product of normal densities
    rng = np.random.default_rng(9)
    m = rng.normal(size=(3, 3))
    d = rng.normal(size=(3, 3)).astype(np.float32)
    s = rng.uniform(0.5, 1.5, size=(3, 3)).astype(np.float32)
    d64, s64 = d.astype(np.float64), s.astype(np.float64)
    prod = np.prod(np.exp(-0.5 * (d64 - m) ** 2 / s64 ** 2) / np.sqrt(2 * math.pi * s64 ** 2))
    assert abs(orc.loglike_from_image(m, d, s) - math.log(prod)) < 1e-12


# ------------------------------------------------------------------ whole pipeline

def _rows_example():
    lens = [1.25, 0.125, -0.0625, 0.0625, -0.03125, 0.03125, -0.015625]
    src = [2, 0.25, 1.5, -0.125, 0.25, 0.125, 0.0625]
    ll = [3, 0.5, 4, 0.0625, 0.125, 0.0625, -0.03125]
    return np.array(lens + src, np.float32), np.array(lens + ll + src, np.float32)


def test_worked_example_golden(orc):
    """tests/golden/worked_example.txt: a second, independent implementation."""
    g = _gold()
    row, row_ll = _rows_example()
    psf20 = np.array([[0, 1, 0], [2, 12, 3], [0, 2, 0]], np.float32)     # = 20 * K, exact in FP32
    data = np.full((4, 4), 0.5, np.float32)
    sig = np.full((4, 4), 0.25, np.float32)
    q, phi = orc.shape(0.125, -0.0625)
    assert abs(q - g["lens_q"][0]) < 1e-15 and abs(phi - g["lens_phi"][0]) < 1e-15
    assert abs(orc.bn(1.5) - g["bn_1p5"][0]) < 1e-11
    ax, ay = orc.sie_deflection(1.25, q, phi, 0.0625, -0.03125, -1.375, -1.375)
    sx, sy = orc.shear_deflection(0.03125, -0.015625, -1.375, -1.375)
    assert abs(-1.375 - ax - sx - g["beta0_x"][0]) < 1e-14
    assert abs(-1.375 - ay - sy - g["beta0_y"][0]) < 1e-14
    cfg = orc.config(4, 4, 0.5, 2, 0, 1, 0)
    im = orc.render(cfg, psf20, row) / 20.0
    ref = np.stack([g["extend_row%d" % i] for i in range(4)])
    assert np.max(np.abs(im - ref)) < 2e-12
    assert abs(orc.chi2_from_image(im, data, sig) - g["extend_chi2"][0]) < 1e-9
    assert abs(orc.loglike_from_image(im, data, sig) - g["extend_logl"][0]) < 1e-9
    cfgz = orc.config(4, 4, 0.5, 2, 0, 1, 1)
    imz = orc.render(cfgz, psf20, row) / 20.0
    assert np.max(np.abs(imz[1:3, 1:3] - ref[1:3, 1:3])) < 2e-12           # interior identical
    assert np.max(np.abs(np.array([imz[0, 0], imz[0, 3], imz[3, 0], imz[3, 3]]) - g["zero_corners"])) < 2e-12
    assert abs(orc.chi2_from_image(imz, data, sig) - g["zero_chi2"][0]) < 1e-9
    assert abs(orc.loglike_from_image(imz, data, sig) - g["zero_logl"][0]) < 1e-9
    cfgl = orc.config(4, 4, 0.5, 2, 1, 1, 0)
    iml = orc.render(cfgl, psf20, row_ll) / 20.0
    assert abs(iml[1, 1] - g["ll_im11"][0]) < 2e-12 * 10
    assert abs(iml[1, 2] - g["ll_im12"][0]) < 2e-12 * 10
    assert abs(iml[0, 0] - g["ll_im00"][0]) < 2e-12 * 10
    assert abs(orc.chi2_from_image(iml, data, sig) - g["ll_chi2"][0]) < 1e-8
    assert abs(orc.loglike_from_image(iml, data, sig) - g["ll_logl"][0]) < 1e-8


def test_linearity_in_amplitudes(orc):
    row, row_ll = _rows_example()
    psf = np.array([[0, 1, 0], [2, 12, 3], [0, 2, 0]], np.float32) / 32
    cfg = orc.config(6, 6, 0.4, 2, 1, 1, 0)
    a = orc.render(cfg, psf, row_ll)
    r2 = row_ll.copy()
    r2[7] *= 4.0
    r2[14] *= 4.0
    assert np.max(np.abs(orc.render(cfg, psf, r2) - 4.0 * a)) < 1e-12 * a.max()


def test_rotation_by_90_degrees_transposes(orc):
    # rotate every centre by +90 deg ((x,y)->(-y,x)) and every angle by +90 deg ((e1,e2)->(-e1,-e2),
    # (g1,g2)->(-g1,-g2)): on a square grid the ideal image maps as img'[i, j] = img[N-1-j, i].
    _, r = _rows_example()
    rr = r.copy()

    def rot(block_e, block_c):
        rr[block_e] = -r[block_e]
        rr[block_e + 1] = -r[block_e + 1]
        rr[block_c] = -r[block_c + 1]
        rr[block_c + 1] = r[block_c]
    rot(1, 3)
    rr[5], rr[6] = -r[5], -r[6]
    rot(10, 12)
    rot(17, 19)
    N = 6
    cfg = orc.config(N, N, 0.4, 2, 1, 1, 0)
    a = orc.ideal_image(cfg, 0, r)
    b = orc.ideal_image(cfg, 0, rr)
    ref = np.empty_like(a)
    for i in range(N):
        for j in range(N):
            ref[i, j] = a[N - 1 - j, i]
    assert np.max(np.abs(b - ref)) < 1e-11 * a.max()


def test_invalid_rows(orc):
    row, _ = _rows_example()
    cfg = orc.config(4, 4, 0.5, 2, 0, 1, 0)
    psf = np.array([[0, 1, 0], [2, 12, 3], [0, 2, 0]], np.float32) / 20
    data = np.full((4, 4), 0.5, np.float32)
    sig = np.full((4, 4), 0.25, np.float32)
    assert orc.row_valid(cfg, row)
    for idx, val in [(0, -0.1), (1, 0.9), (8, 0.0), (8, -1.0), (9, 0.0), (10, 1.0), (3, np.nan), (7, np.inf)]:
        bad = row.copy()
        bad[idx] = val
        if idx == 1:
            bad[2] = 0.5
        assert not orc.row_valid(cfg, bad), (idx, val)
        assert orc.loglike(cfg, psf, data, sig, bad) == -math.inf
        assert np.all(np.isnan(orc.render(cfg, psf, bad)))
    ok = row.copy()
    ok[0] = 0.0                       # theta_E = 0 is allowed (no lens)
    assert math.isfinite(orc.loglike(cfg, psf, data, sig, ok))


def test_batch_matches_single_and_lens_indexing(orc):
    row, _ = _rows_example()
    cfg = orc.config(4, 4, 0.5, 2, 0, 1, 0)
    rng = np.random.default_rng(11)
    psf = rng.uniform(size=(2, 3, 3)).astype(np.float32)
    data = rng.normal(size=(2, 4, 4)).astype(np.float32)
    sig = rng.uniform(0.2, 0.4, size=(2, 4, 4)).astype(np.float32)
    rows = np.stack([row * (1 + 0.01 * k) for k in range(6)]).astype(np.float32)
    out, used = orc.loglike_batch(cfg, psf, data, sig, rows, n_lens=2)
    assert used >= 1
    for r in range(6):
        l = r // 3
        assert out[r] == orc.loglike(cfg, psf[l], data[l], sig[l], rows[r])
    ims = orc.render_batch(cfg, psf, rows, n_lens=2)
    assert np.array_equal(ims[4], orc.render(cfg, psf[1], rows[4]))
