"""Pins for the oracle's atmosphere interpolation (P11, P12 of DESIGN.md)."""
import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator

import gen
import oracle as o


def _axes():
    return gen.atmosphere_axes()


def _poly_table(deg_T, deg_g, deg_m, deg_x, seed=0):
    """Table whose values are a tensor-product polynomial of the given per-axis degrees."""
    logT, logg, mu, logx = _axes()
    rng = np.random.default_rng(seed)
    cs = [rng.uniform(-1, 1, size=d + 1) for d in (deg_T, deg_g, deg_m, deg_x)]
    ctr = [6.0, 14.2, 0.5, 0.3]

    def f(t, g, m, x):
        return (np.polyval(cs[0], t - ctr[0]) * np.polyval(cs[1], g - ctr[1])
                * np.polyval(cs[2], m - ctr[2]) * np.polyval(cs[3], x - ctr[3]))
    T, G, M, X = np.meshgrid(logT, logg, mu, logx, indexing="ij")
    return o.Atmosphere(logT, logg, mu, logx, f(T, G, M, X)), f


def _random_points(n, seed=1, inside_only=False):
    logT, logg, mu, logx = _axes()
    rng = np.random.default_rng(seed)
    pts = np.stack([rng.uniform(ax[0], ax[-1], size=n) for ax in (logT, logg, mu, logx)], axis=1)
    return pts


@pytest.mark.parametrize("strategy", [1, 2, 3])
def test_p11_reproduces_nodes(strategy):
    logT, logg, mu, logx, vals = gen.synthetic_atmosphere()
    atm = o.Atmosphere(logT, logg, mu, logx, vals)
    rng = np.random.default_rng(2)
    for _ in range(300):
        i, j, k, m = (rng.integers(0, len(a)) for a in (logT, logg, mu, logx))
        v = o.interp4(atm, strategy, logT[i], logg[j], mu[k], logx[m])
        assert abs(v - vals[i, j, k, m]) <= 1e-13 * max(1.0, abs(vals[i, j, k, m]))


def test_p11_strategy_a_reproduces_cubics_everywhere():
    atm, f = _poly_table(3, 3, 3, 3)
    for p in _random_points(300):
        assert abs(o.interp4(atm, 1, *p) - f(*p)) < 1e-11
    # also in the shifted edge stencils
    logT, logg, mu, logx = _axes()
    for p in ([logT[0] + 1e-3, logg[-1] - 1e-3, mu[0] + 1e-4, logx[-1] - 1e-3],
              [logT[-1] - 1e-3, logg[0] + 1e-3, mu[-1] - 1e-5, logx[0] + 1e-3]):
        assert abs(o.interp4(atm, 1, *p) - f(*p)) < 1e-11


def test_p11_strategy_d_local_orders():
    """(d): linear in logT, logg; cubic in mu and logx in the interior; linear for mu <= mu[3], in the last
    mu interval, and in the first / last logx interval (reading R13c)."""
    logT, logg, mu, logx = _axes()
    atm, f = _poly_table(1, 1, 3, 3)
    rng = np.random.default_rng(3)
    for _ in range(300):                                     # interior: exact for (1,1,3,3)
        p = [rng.uniform(logT[0], logT[-1]), rng.uniform(logg[0], logg[-1]),
             rng.uniform(mu[3], mu[-2]), rng.uniform(logx[1], logx[-2])]
        assert abs(o.interp4(atm, 2, *p) - f(*p)) < 1e-11
    atm1, f1 = _poly_table(1, 1, 1, 1)
    for _ in range(200):                                     # everywhere: exact for multilinear
        p = _random_points(1, seed=int(rng.integers(1 << 30)))[0]
        assert abs(o.interp4(atm1, 2, *p) - f1(*p)) < 1e-12
    # NOT exact for a mu-cubic inside the protected zone -> it really is lower order there
    atm3, f3 = _poly_table(0, 0, 3, 0)
    p = [6.0, 14.2, 0.5 * (mu[1] + mu[2]), 0.3]
    lin = f3(6.0, 14.2, mu[1], 0.3) * 0.5 + f3(6.0, 14.2, mu[2], 0.3) * 0.5
    assert abs(o.interp4(atm3, 2, *p) - lin) < 1e-13
    assert abs(o.interp4(atm3, 2, *p) - f3(*p)) > 1e-9
    # logT cubic is not reproduced by (d) but is by (a)
    atmT, fT = _poly_table(3, 0, 0, 0)
    p = [5.93, 14.2, 0.5, 0.3]
    assert abs(o.interp4(atmT, 1, *p) - fT(*p)) < 1e-12
    assert abs(o.interp4(atmT, 2, *p) - fT(*p)) > 1e-7


def test_p11_strategy_c_local_orders():
    """(c) (PAPER.md:537 caption, 551; reading R13e): cubic on all four axes in the interior; linear in the first / last
    interval of logT, logg, logx, for mu <= mu[3] and in the last mu interval."""
    logT, logg, mu, logx = _axes()
    atm, f = _poly_table(3, 3, 3, 3)
    rng = np.random.default_rng(5)
    for _ in range(300):                                     # interior of every axis: exact for tensor cubics
        p = [rng.uniform(logT[1], logT[-2]), rng.uniform(logg[1], logg[-2]),
             rng.uniform(mu[3], mu[-2]), rng.uniform(logx[1], logx[-2])]
        assert abs(o.interp4(atm, 3, *p) - f(*p)) < 1e-11
    atm1, f1 = _poly_table(1, 1, 1, 1)
    for _ in range(200):                                     # everywhere: exact for multilinear
        p = _random_points(1, seed=int(rng.integers(1 << 30)))[0]
        assert abs(o.interp4(atm1, 3, *p) - f1(*p)) < 1e-12
    # first logT interval: linear between the two nodes, not the cubic
    atmT, fT = _poly_table(3, 0, 0, 0)
    tm = 0.5 * (logT[0] + logT[1])
    lin = 0.5 * (fT(logT[0], 14.2, 0.5, 0.3) + fT(logT[1], 14.2, 0.5, 0.3))
    assert abs(o.interp4(atmT, 3, tm, 14.2, 0.5, 0.3) - lin) < 1e-13
    assert abs(o.interp4(atmT, 3, tm, 14.2, 0.5, 0.3) - fT(tm, 14.2, 0.5, 0.3)) > 1e-9
    # interior logT: (c) agrees with (a), differs from (d)
    p = [5.93, 14.2, 0.5, 0.3]
    assert abs(o.interp4(atmT, 3, *p) - o.interp4(atmT, 1, *p)) < 1e-13
    assert abs(o.interp4(atmT, 3, *p) - o.interp4(atmT, 2, *p)) > 1e-7
    # protected small-mu zone as in (d)
    atm3, f3 = _poly_table(0, 0, 3, 0)
    q = [6.0, 14.2, 0.5 * (mu[1] + mu[2]), 0.3]
    assert abs(o.interp4(atm3, 3, *q) - o.interp4(atm3, 2, *q)) < 1e-13


def test_p11_continuity_across_nodes_and_zone_boundary():
    logT, logg, mu, logx, vals = gen.synthetic_atmosphere()
    atm = o.Atmosphere(logT, logg, mu, logx, vals)
    eps = 1e-10
    for strategy in (1, 2, 3):
        for k in (1, 2, 3, 4, 30, 65):                       # mu nodes incl. the protected-zone edge mu[3]
            a = o.interp4(atm, strategy, 6.03, 14.21, mu[k] - eps, 0.77)
            b = o.interp4(atm, strategy, 6.03, 14.21, mu[k] + eps, 0.77)
            assert abs(a - b) < 1e-7
        for m in (1, 2, 80, 164):
            a = o.interp4(atm, strategy, 6.03, 14.21, 0.4, logx[m] - eps)
            b = o.interp4(atm, strategy, 6.03, 14.21, 0.4, logx[m] + eps)
            assert abs(a - b) < 1e-7
        # clamping outside the table (reading R13b): constant continuation
        assert o.interp4(atm, strategy, 6.03, 14.21, 0.001, 2.5) == o.interp4(atm, strategy, 6.03, 14.21, mu[0], logx[-1])
        assert o.interp4(atm, strategy, 4.0, 20.0, 0.4, -5.0) == o.interp4(atm, strategy, logT[0], logg[-1], 0.4, logx[0])


def test_p11_1d_is_textbook_four_point_lagrange():
    _, _, mu, _ = _axes()
    rng = np.random.default_rng(5)
    y = rng.normal(size=len(mu))
    for x in rng.uniform(mu[0], mu[-1], size=40):
        i = min(np.searchsorted(mu, x, side="right") - 1, len(mu) - 2)
        s = min(max(i - 1, 0), len(mu) - 4)
        ref = float(BarycentricInterpolator(mu[s:s + 4], y[s:s + 4])(x))   # textbook 4-point Lagrange
        assert abs(o.interp1(mu, y, x, o.AX_CUBIC_SHIFT) - ref) < 1e-10
        # mixed rule: linear where protected
        if i < 3 or i == len(mu) - 2:
            t = (x - mu[i]) / (mu[i + 1] - mu[i])
            assert abs(o.interp1(mu, y, x, o.AX_MU_PROTECTED) - ((1 - t) * y[i] + t * y[i + 1])) < 1e-13
        else:
            assert abs(o.interp1(mu, y, x, o.AX_MU_PROTECTED) - ref) < 1e-10


def test_p12_unperturbed_table_is_planck_times_limb_darkening():
    """With the perturbation switched off the table is log10[(2k^3/h^3c^2) x^3/(e^x-1) (1+2.06mu)/3.06], so the
    table path must reproduce the closed-form blackbody (Eq C.5) times the limb factor to interpolation error."""
    logT, logg, mu, logx, vals = gen.synthetic_atmosphere(amplitude=0.0)
    atm = o.Atmosphere(logT, logg, mu, logx, vals)
    assert abs(np.log10(2.0 * o.KB_KEV_K ** 3 / (o.H_KEV_S ** 3 * o.C_CM_S ** 2)) - 10.30387) < 1e-5
    assert abs(o.TWO_OVER_H3C2 / 3.1459490373e31 - 1.0) < 1e-8
    rng = np.random.default_rng(7)
    for _ in range(200):
        lt = rng.uniform(5.2, 6.7)
        m = rng.uniform(0.05, 1.0)
        kT = o.KB_KEV_K * 10.0 ** lt
        Ep = kT * 10.0 ** rng.uniform(-1.2, 1.9)
        bb = o.intensity(0, None, lt, 14.2, Ep, m)
        ref = bb * (1.0 + 2.06 * m) / 3.06
        for strategy, tol in ((1, 2e-5), (2, 2e-5)):      # cubic-in-logx interpolation error of the Wien tail
            got = o.intensity(strategy, atm, lt, 14.2, Ep, m)
            assert abs(got / ref - 1.0) < tol
    # the closed form itself: Planck photon-energy intensity
    E, kT = 1.0, 0.3
    assert abs(o.intensity(0, None, gen.log10T_of_kT(kT), 14.0, E, 0.5)
               - o.TWO_OVER_H3C2 * E ** 3 / np.expm1(E / kT)) < 1e-3 * 1e-12 * o.TWO_OVER_H3C2
