"""Pins for the oracle's elliptical power-law deflection (NEXT-2; Eq. 12).

The oracle sums Tessore & Metcalf's angular series; nothing here re-types that series.  The
pins are what Eq. 12 and potential theory fix independently of it:
  * gamma = 2 is the SIE, whose closed form the SIE pins already fix;
  * q = 1: the mean convergence inside r of Eq. 12 is (theta_E / r)^(gamma-1), so
    alpha = theta_E (theta_E / r)^(gamma-2) radially;
  * any q: the deflection of a homoeoidal mass distribution as a one-dimensional quadrature
    (Schramm 1990; Keeton 2001), evaluated with scipy.integrate.quad;
  * div alpha = 2 kappa and curl alpha = 0 (alpha is the gradient of a potential whose
    Laplacian is 2 kappa), by central differences;
  * the row layout: an EPL row with slope 2 renders the image of the SIE row.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as O
from paper_2503_08586_b200 import workloads as W


def kappa_epl(theta_e, gamma, q, x, y):
    """Eq. 12 with R -> R_p of Eq. 10 (major axis along x)."""
    rp = math.sqrt(q * x * x + y * y / q)
    return 0.5 * (3.0 - gamma) * (theta_e / rp) ** (gamma - 1.0)


def test_slope_two_is_the_sie():
    rng = np.random.default_rng(5)
    for _ in range(200):
        q = rng.uniform(0.05, 1.0)
        phi = rng.uniform(0, math.pi)
        x, y = rng.uniform(-3, 3, 2)
        a = O.sie_deflection(1.3, q, phi, 0.02, -0.01, x, y)
        b = O.epl_deflection(1.3, 2.0, q, phi, 0.02, -0.01, x, y)
        assert abs(a[0] - b[0]) < 1e-12 and abs(a[1] - b[1]) < 1e-12


def test_circular_closed_form():
    rng = np.random.default_rng(6)
    for _ in range(50):
        g = rng.uniform(1.2, 2.8)
        th = rng.uniform(0.5, 2.0)
        x, y = rng.uniform(-3, 3, 2)
        r = math.hypot(x, y)
        a = th * (th / r) ** (g - 2.0)
        ax, ay = O.epl_deflection(th, g, 1.0, 0.7, 0.0, 0.0, x, y)
        assert abs(ax - a * x / r) < 1e-13 * (1 + a) and abs(ay - a * y / r) < 1e-13 * (1 + a)


def test_homoeoid_quadrature():
    """alpha_x = q x J_0, alpha_y = q y J_1,  J_n = int_0^1 kappa(xi(u)) [1 - (1-q^2) u]^-(n+1/2) du,
    xi(u)^2 = u (x^2 + y^2 / (1 - (1-q^2) u)),  kappa a function of xi^2 = x^2 + y^2/q^2."""
    th = 1.2
    for g, q, x, y in [(2.3, 0.7, 0.9, 0.4), (1.6, 0.5, -0.3, 1.1), (2.0, 0.8, 1.5, -0.2), (2.6, 0.35, 0.5, 0.5),
                       (1.3, 0.9, -1.2, -0.7)]:
        def kap(xi2):
            # R_p^2 = q x^2 + y^2/q = q xi^2
            return 0.5 * (3.0 - g) * (th / math.sqrt(q * xi2)) ** (g - 1.0)

        def J(n):
            def f(u):
                w = 1.0 - (1.0 - q * q) * u
                return kap(u * (x * x + y * y / w)) / w ** (n + 0.5)
            # integrable u^-(g-1)/2 singularity at 0: substitute u = v^m to remove it
            m = 2.0 / (3.0 - g) + 1.0
            val, err = integrate.quad(lambda v: f(v ** m) * m * v ** (m - 1.0), 0.0, 1.0, epsabs=1e-13, epsrel=1e-13,
                                      limit=400)
            return val
        ax, ay = O.epl_deflection(th, g, q, 0.0, 0.0, 0.0, x, y)
        assert abs(ax - q * x * J(0)) < 2e-10 and abs(ay - q * y * J(1)) < 2e-10


def test_divergence_is_two_kappa_and_curl_free():
    th, cx, cy = 1.1, 0.05, -0.03
    h = 1e-3
    for g, q, phi, x, y in [(2.2, 0.6, 0.4, 0.8, 0.5), (1.7, 0.75, 2.1, -1.0, 0.3), (2.5, 0.9, 1.0, 0.2, -1.4)]:
        def a(xx, yy):
            return O.epl_deflection(th, g, q, phi, cx, cy, xx, yy)

        def d(comp, axis, hh):
            p = a(x + hh * (axis == 0), y + hh * (axis == 1))[comp]
            m = a(x - hh * (axis == 0), y - hh * (axis == 1))[comp]
            return (p - m) / (2 * hh)

        def rich(comp, axis):            # Richardson: O(h^4)
            return (4.0 * d(comp, axis, h / 2) - d(comp, axis, h)) / 3.0
        c, s = math.cos(phi), math.sin(phi)
        xp, yp = (x - cx) * c + (y - cy) * s, -(x - cx) * s + (y - cy) * c
        k = kappa_epl(th, g, q, xp, yp)
        assert abs(0.5 * (rich(0, 0) + rich(1, 1)) - k) < 1e-9 * max(k, 1.0)
        assert abs(rich(1, 0) - rich(0, 1)) < 1e-9


def test_centre_and_zero_mass():
    assert O.epl_deflection(1.0, 2.2, 0.7, 0.3, 0.1, 0.2, 0.1, 0.2) == (0.0, 0.0)
    assert O.epl_deflection(0.0, 2.2, 0.7, 0.3, 0.0, 0.0, 0.5, 0.2) == (0.0, 0.0)


def test_row_layout_and_validity():
    w = W.workload(0).scaled(batch=4)
    we = w.with_epl()
    assert we.n_params == w.n_params + 1
    rows = W.draw_params(w, W.rng_for(0, W.STREAM_BATCH, 0), 4)
    rows_e = W.draw_params(we, W.rng_for(0, W.STREAM_BATCH, 0), 4)
    assert np.array_equal(np.delete(rows_e, 7, axis=1), rows)             # same draw, slope inserted
    psf = W.make_psf(w)
    r2 = rows_e.copy()
    r2[:, 7] = 2.0
    for i in range(4):
        a = O.render(O.config_of(w), psf, rows[i])
        b = O.render(O.config_of(we), psf, r2[i])
        assert np.max(np.abs(a - b)) < 1e-12 * np.max(np.abs(a))
        c = O.render(O.config_of(we), psf, rows_e[i])
        assert np.max(np.abs(a - c)) > 1e-4 * np.max(np.abs(a))         # the slope does matter
    cfg = O.config_of(we)
    assert O.row_valid(cfg, rows_e[0])
    for bad in (1.0, 3.0, 0.5, 3.5, np.nan):
        r = rows_e[0].copy()
        r[7] = bad
        assert not O.row_valid(cfg, r)


def test_linear_mode_uses_the_epl_layout():
    w = W.workload(1).scaled(batch=1)
    w = W.Workload(**{**w.__dict__, "ny": 24, "nx": 24, "supersample": 2, "psf_size": 5}).with_epl()
    prob = W.make_problem(w, O.render_for_workloads)
    cfg = O.config_of(w)
    row = prob.truth[0]
    ll, amps = O.loglike_linear(cfg, prob.psf[0], prob.data[0], prob.noise[0], row)
    # at the truth the solved amplitudes are the true I_e up to the noise
    assert abs(amps[0] / row[8] - 1.0) < 0.05 and abs(amps[1] / row[15] - 1.0) < 0.25
    assert ll >= O.loglike(cfg, prob.psf[0], prob.data[0], prob.noise[0], row) - 1e-9


def test_scaling_rotation_and_parity_symmetries():
    """kappa is homogeneous of degree 1 - gamma, so alpha(lambda theta) = lambda^(2-gamma) alpha(theta);
    rotating the lens and the position together rotates the deflection; alpha(-theta) = -alpha(theta)."""
    rng = np.random.default_rng(9)
    for _ in range(40):
        g, q, phi = rng.uniform(1.2, 2.8), rng.uniform(0.2, 1.0), rng.uniform(0, math.pi)
        x, y = rng.uniform(-2, 2, 2)
        lam, rot = rng.uniform(0.3, 3.0), rng.uniform(0, 2 * math.pi)
        ax, ay = O.epl_deflection(1.1, g, q, phi, 0.0, 0.0, x, y)
        sx, sy = O.epl_deflection(1.1, g, q, phi, 0.0, 0.0, lam * x, lam * y)
        f = lam ** (2.0 - g)
        assert abs(sx - f * ax) < 1e-12 * (1 + abs(f * ax)) and abs(sy - f * ay) < 1e-12 * (1 + abs(f * ay))
        c, s = math.cos(rot), math.sin(rot)
        rx, ry = O.epl_deflection(1.1, g, q, phi + rot, 0.0, 0.0, c * x - s * y, s * x + c * y)
        assert abs(rx - (c * ax - s * ay)) < 1e-12 and abs(ry - (s * ax + c * ay)) < 1e-12
        mx, my = O.epl_deflection(1.1, g, q, phi, 0.0, 0.0, -x, -y)
        assert abs(mx + ax) < 1e-14 and abs(my + ay) < 1e-14
        # theta_E scaling: alpha is proportional to theta_E^(gamma-1)
        tx, ty = O.epl_deflection(2.2, g, q, phi, 0.0, 0.0, x, y)
        assert abs(tx - 2.0 ** (g - 1.0) * ax) < 1e-12 * (1 + abs(tx))
