"""Pins for the oracle's Schwarzschild integrals (psi, lensing factor, lag): P1-P7 of DESIGN.md.

Each pin compares oracle/ppm_oracle.c with something other than itself: stored probe values,
scipy.integrate.quad of the *original* integrals Eq 12 / Eq 15 -- the oracle
integrates the regularised forms Eq 32 / 35 --, closed-form limits, and the direct travel-time
integral for inward rays.
"""
import numpy as np
import pytest
from scipy import integrate, optimize

import oracle as o

U0 = 0.3446


def test_gl_rule_is_gauss_legendre():
    x, w = o.gl_rule()
    xr, wr = np.polynomial.legendre.leggauss(len(x))
    assert np.allclose(np.sort(x), xr, atol=1e-15)
    assert np.allclose(w[np.argsort(x)], wr, atol=1e-15)
    assert abs(w.sum() - 2.0) < 1e-15


def test_p1_probe_values(golden):
    fn = dict(psi=o.psi, lag=o.lag, rho=o.rho, lagin=o.lag_total_over_R, dpsi=o.dpsi_dalpha, lf=o.lensing_factor)
    for kind, u, a, val in golden("geodesic_pins.txt"):
        got = fn[kind](float(u), float(a))
        tol = 2e-11 if kind == "lagin" else 1e-11
        assert abs(got - float(val)) <= tol * max(1.0, abs(float(val))), (kind, u, a, got, val)


def _psi_eq12(u, alpha):
    """Eq 12 as printed, with y = R/r: psi = int_0^1 dy / sqrt((1-u)/sin^2 a - y^2 (1 - u y))."""
    A = (1.0 - u) / np.sin(alpha) ** 2
    v, _ = integrate.quad(lambda y: 1.0 / np.sqrt(A - y * y * (1.0 - u * y)), 0.0, 1.0, epsabs=1e-13, epsrel=1e-13,
                          limit=400)
    return v


def _lag_eq15(u, alpha):
    """Eq 15 as printed, y = R/r: (1/R) int dr/(1-Rs/r) {[1 - b^2/r^2 (1-Rs/r)]^-1/2 - 1}."""
    b2 = np.sin(alpha) ** 2 / (1.0 - u)

    def f(y):
        w = 1.0 - u * y
        return (1.0 / np.sqrt(1.0 - b2 * y * y * w) - 1.0) / (y * y * w)
    v, _ = integrate.quad(f, 0.0, 1.0, epsabs=1e-13, epsrel=1e-13, limit=400)
    return v


@pytest.mark.parametrize("u,alpha", [(0.2, 0.4), (U0, 0.3), (U0, 1.0), (U0, 1.5), (0.5, 1.2), (0.55, 1.45), (0.1, 1.3)])
def test_p1_eq32_equals_eq12_and_eq35_equals_eq15(u, alpha):
    assert abs(o.psi(u, alpha) - _psi_eq12(u, alpha)) < 5e-12
    assert abs(o.lag(u, alpha) - _lag_eq15(u, alpha)) < 5e-12


def test_p2_flat_space_limit():
    for a in (0.1, 0.7, 1.4):
        assert abs(o.psi(1e-9, a) - a) < 2e-9
        assert abs(o.lag(1e-9, a) - (1.0 - np.cos(a))) < 2e-9
        assert abs(o.lensing_factor(1e-9, a) - 1.0) < 5e-9
    assert abs(o.psi(1e-9, 0.7) - 0.70000000037) < 1e-10          # probe value, SURVEY P2
    assert abs(o.lag(1e-9, 0.7) - 0.2351578130) < 1e-9


@pytest.mark.parametrize("u,err_pct", [(0.2, 0.199), (U0, 1.056), (0.5, 5.62)])
def test_p3_beloborodov_error_at_limb(u, err_pct):
    """1 - cos(alpha) ~ (1 - cos(psi))(1 - u) (Beloborodov 2002, cited PAPER.md:29): its error in cos(alpha)
    is largest at alpha = pi/2 where it equals the quoted percentages, and vanishes as alpha -> 0."""
    ps = o.psi(u, np.pi / 2)
    cos_alpha_B = 1.0 - (1.0 - np.cos(ps)) * (1.0 - u)
    assert abs(abs(cos_alpha_B) * 100.0 - err_pct) < 0.006
    prev = None
    for a in (1.2, 0.8, 0.4, 0.1):
        e = abs((1.0 - (1.0 - np.cos(o.psi(u, a))) * (1.0 - u)) - np.cos(a))
        assert e < abs(cos_alpha_B)
        if prev is not None:
            assert e < prev
        prev = e
    # scales ~ u^2 as u -> 0
    e1 = abs(1.0 - (1.0 - np.cos(o.psi(0.02, np.pi / 2))) * 0.98)
    e2 = abs(1.0 - (1.0 - np.cos(o.psi(0.01, np.pi / 2))) * 0.99)
    assert 3.0 < e1 / e2 < 5.0


def test_p4_critical_compactness():
    ucrit = optimize.brentq(lambda u: o.psi(u, np.pi / 2) - np.pi, 0.5, 0.6, xtol=1e-14)
    assert abs(ucrit - 0.5680820870) < 2e-10
    assert abs(2.0 / ucrit - 3.52062) < 2e-5          # R = 3.52062 GM/c^2; "GM/(Rc^2) >~ 0.28" PAPER.md:718
    assert abs(1.0 / (2.0 / ucrit) - 0.284) < 1e-3


def test_p5_inward_rays():
    assert abs(o.rho(U0, np.pi / 2) - 1.0) < 1e-15
    for a in (1.6, 1.7, 1.8):
        r = o.rho(U0, a)
        # periastron condition behind Eq 14: rho^2/(1-u/rho) = sin^2(alpha)/(1-u)
        assert abs(r * r / (1.0 - U0 / r) - np.sin(a) ** 2 / (1.0 - U0)) < 1e-14
    # C^1 across alpha = pi/2 for psi and for the total lag
    h = 1e-4
    for f in (o.psi, o.lag_total_over_R):
        left = (f(U0, np.pi / 2) - f(U0, np.pi / 2 - h)) / h
        right = (f(U0, np.pi / 2 + h) - f(U0, np.pi / 2)) / h
        assert abs(left - right) < 5e-4
        cen = (f(U0, np.pi / 2 + h) - f(U0, np.pi / 2 - h)) / (2 * h)
        assert abs(0.5 * (left + right) - cen) < 1e-9
    # probe one-sided slopes
    assert abs((o.psi(U0, np.pi / 2) - o.psi(U0, np.pi / 2 - h)) / h - 1.67572) < 2e-5
    assert abs((o.psi(U0, np.pi / 2 + h) - o.psi(U0, np.pi / 2)) / h - 1.67583) < 2e-5


def _inward_travel_time(u, alpha):
    """2 int_{Rp}^{R} K dr + int_R^inf (K - K0) dr in units R/c, K = 1/((1-Rs/r) sqrt(1 - b^2 (1-Rs/r)/r^2)),
    K0 = 1/(1-Rs/r); R = 1, Rs = u.  Periastron from a root solve (not Eq 14)."""
    b2 = np.sin(alpha) ** 2 / (1.0 - u)

    def D(r):
        return 1.0 - b2 * (1.0 - u / r) / (r * r)
    rp = optimize.brentq(D, 1.5 * u, 1.0, xtol=1e-15, rtol=1e-15)
    # r = rp + s^2 removes the inverse-sqrt end-point singularity
    smax = np.sqrt(1.0 - rp)

    def f_in(s):
        r = rp + s * s
        return 2.0 * s / ((1.0 - u / r) * np.sqrt(max(D(r), 1e-300)))
    t_in, _ = integrate.quad(f_in, 0.0, smax, epsabs=1e-13, epsrel=1e-13, limit=400)

    def f_out(y):        # y = 1/r
        w = 1.0 - u * y
        return (1.0 / np.sqrt(1.0 - b2 * y * y * w) - 1.0) / (y * y * w)
    t_out, _ = integrate.quad(f_out, 0.0, 1.0, epsabs=1e-13, epsrel=1e-13, limit=400)
    return 2.0 * t_in + t_out


@pytest.mark.parametrize("alpha", [1.6, 1.7, 1.8])
def test_p6_inward_lag_is_eq17_not_eq36(alpha):
    direct = _inward_travel_time(U0, alpha)
    assert abs(o.lag_total_over_R(U0, alpha) - direct) < 1e-9
    # Eq 36 as printed (dimensionless, no 2 dt(Rp) - dt(R) and no rho factor) is NOT the travel time (reading R6)
    r = o.rho(U0, alpha)
    eq36 = 2.0 * o.lag(U0 / r, np.pi / 2) - o.lag(U0, np.pi - alpha)
    assert abs(eq36 - direct) > 1e-4


def test_p7_lensing_factor_derivative():
    h = 1e-3
    for u, a in [(U0, 0.3), (U0, 1.0), (U0, 1.5), (0.5, 1.2), (0.2, 0.8)]:
        fd = (-o.psi(u, a + 2 * h) + 8 * o.psi(u, a + h) - 8 * o.psi(u, a - h) + o.psi(u, a - 2 * h)) / (12 * h)
        assert abs(o.dpsi_dalpha_analytic(u, a) - fd) < 2e-10
    # the finite-difference branch (alpha >= pi/2 - 0.05) agrees with the analytic integral where both exist
    for a in (np.pi / 2 - 0.049, np.pi / 2 - 0.02, np.pi / 2 - 0.004):
        assert abs(o.dpsi_dalpha(U0, a) - o.dpsi_dalpha_analytic(U0, a)) < 2e-12
    # LF -> 1 - u as alpha -> 0
    for u in (0.2, U0, 0.5):
        assert abs(o.lensing_factor(u, 1e-4) - (1.0 - u)) < 1e-7


def test_alpha_of_psi_inverts_psi():
    rng = np.random.default_rng(1)
    for _ in range(50):
        u = rng.uniform(0.05, 0.56)
        a = rng.uniform(0.0, np.pi / 2 + 0.08)
        ps = o.psi(u, a)
        a2 = o.alpha_of_psi(u, ps, np.pi / 2 + 0.1)
        assert abs(a2 - a) < 1e-13
    assert o.alpha_of_psi(U0, 3.0, np.pi / 2) is None


@pytest.mark.parametrize("eps", [1e-6, 1e-8, 1e-9, 1e-10, 1e-11])
def test_p5_no_missed_boundary_layer_next_to_the_limb(eps):
    """psi and the lag are smooth in alpha through pi/2 (pin P5: one-sided slopes 1.67572 / 1.67583 and
    2.06989 / 2.07004 at h = 1e-4), so the secant slope over ANY small step must sit between
    them.  The Eq 32/35 integrands have a layer of width ~cos(alpha) at x = 0; a quadrature that does not
    resolve it returns psi(pi/2 - eps) = psi(pi/2) for eps < ~1e-8 (slope 0)."""
    hp = np.pi / 2
    s_psi = (o.psi(U0, hp) - o.psi(U0, hp - eps)) / eps
    s_lag = (o.lag(U0, hp) - o.lag(U0, hp - eps)) / eps
    tol = 3e-4 + 1e-15 / eps          # probe spread + double rounding of the difference
    assert abs(s_psi - 1.675775) < tol
    assert abs(s_lag - 2.069965) < tol
