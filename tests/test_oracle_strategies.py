"""Pins P21-P23 of the oracle's SURVEY 8(f) widenings:
  P21  Interp of Eq 46 at order 3 (reading R11b): textbook 4-point Lagrange on the periodic template, linear next to the
       visibility edge, error order N_fp^-4 instead of N_fp^-2, same limit.
  P22  table interpolation applied to the intensity I/T^3 = 10^table (reading R13g) with the four strategies of
       PAPER.md:551 (a, b = a + clip, c, d): nodes, polynomials, clip identity, agreement with the log-domain reading.
  P23  the two Table 3 geometries on a table that is steep towards the limb: negative lobes under (a),
       zero "holes" under (b), clean profiles under (c) and (d) -- the paper's qualitative finding.
"""
import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator

import gen
import oracle as o

LT = gen.log10T_of_kT(0.3)


# ------------------------------------------------------------------------------------------------- P21
def _toy_template(n_fp=24, hidden=()):
    """A hand-made periodic template with non-uniform, strictly increasing phi_o."""
    i = np.arange(n_fp + 1)
    phio = i / n_fp + 0.01 * np.sin(2 * np.pi * i / n_fp) + 0.03
    F = 2.0 + np.cos(2 * np.pi * i / n_fp)
    F[list(hidden)] = 0.0
    F[n_fp] = F[0]
    y = 1.0 + 0.3 * np.sin(2 * np.pi * i / n_fp + 0.4)
    y[n_fp] = y[0]
    return phio, F, y


def test_p21_order3_is_four_point_lagrange_with_periodic_wrap():
    n_fp = 24
    phio, F, y = _toy_template(n_fp)
    rng = np.random.default_rng(1)
    for phi_p in np.concatenate([rng.uniform(phio[0], phio[n_fp], 40), [phio[0] + 1e-9, phio[n_fp] - 1e-9]]):
        v, i = o.phase_interp(phio, F, y, phi_p, 3)
        assert phio[i] <= phi_p < phio[i + 1]
        xs, ys = [], []
        for k in (i - 1, i, i + 1, i + 2):
            if k < 0:
                xs.append(phio[k + n_fp] - 1.0); ys.append(y[k + n_fp])
            elif k > n_fp:
                xs.append(phio[k - n_fp] + 1.0); ys.append(y[k - n_fp])
            else:
                xs.append(phio[k]); ys.append(y[k])
        assert abs(v - BarycentricInterpolator(xs, ys)(phi_p)) < 1e-13
        # order 1: the linear rule of reading R11
        v1, i1 = o.phase_interp(phio, F, y, phi_p, 1)
        t = (phi_p - phio[i]) / (phio[i + 1] - phio[i])
        assert i1 == i and abs(v1 - (y[i] + (y[i + 1] - y[i]) * t)) < 1e-15
    # nodes are reproduced
    for i in range(n_fp):
        assert abs(o.phase_interp(phio, F, y, phio[i], 3)[0] - y[i]) < 1e-14
    # a cubic in phi_o is reproduced exactly away from the wrap
    c = lambda x: 0.7 - 1.1 * x + 2.3 * x ** 2 - 0.9 * x ** 3
    for phi_p in rng.uniform(phio[2], phio[n_fp - 2], 20):
        assert abs(o.phase_interp(phio, F, c(phio), phi_p, 3)[0] - c(phi_p)) < 1e-13


def test_p21_order3_reverts_to_linear_next_to_hidden_entries():
    n_fp = 24
    hidden = (9, 10, 11, 12, 13)
    phio, F, y = _toy_template(n_fp, hidden)
    for i in range(n_fp):
        phi_p = 0.5 * (phio[i] + phio[i + 1])
        stencil = [(i - 1) % n_fp, i, i + 1, (i + 2) if i + 2 <= n_fp else 1]
        near = any(F[k] == 0.0 for k in stencil)
        v3 = o.phase_interp(phio, F, y, phi_p, 3)[0]
        v1 = o.phase_interp(phio, F, y, phi_p, 1)[0]
        if near:
            assert v3 == v1
        else:
            assert abs(v3 - v1) > 1e-6
        assert o.phase_interp(phio, F, F, phi_p, 3)[0] >= 0.0              # F_p never overshoots below zero at the edge


def test_p21_error_order_rises_from_2_to_4():
    ci = np.cos(np.deg2rad(50.0))
    p = gen.pack_params(1.4, 12.0, 400.0, ci, 0.2, spots=[(0.6, 0.0, 0.2, LT)])          # always visible
    E = np.array([0.3, 1.0, 3.0])
    cfg = lambda n, order: dict(n_spots=1, n_theta=6, n_phi=6, n_phase=16, n_fp=n, emission=0, oblate=1, phase_interp=order)
    ref1, _ = o.evaluate(cfg(4096, 1), E, p)
    ref3, _ = o.evaluate(cfg(4096, 3), E, p)
    assert np.max(np.abs(ref3 / ref1 - 1.0)) < 2e-6                                       # same limit
    err = {1: [], 3: []}
    for order in (1, 3):
        for n in (24, 48, 96):
            f, s = o.evaluate(cfg(n, order), E, p)
            assert s == 0
            err[order].append(np.abs(f - ref3).sum() / ref3.sum())
    assert 3.0 < err[1][0] / err[1][1] < 5.5 and 3.0 < err[1][1] / err[1][2] < 5.5       # N_fp^-2
    assert 11.0 < err[3][0] / err[3][1] < 22.0 and 11.0 < err[3][1] / err[3][2] < 22.0   # N_fp^-4
    assert err[3][2] < 1e-2 * err[1][2]


# ------------------------------------------------------------------------------------------------- P22
@pytest.fixture(scope="module")
def steep():
    tab = gen.steep_limb_atmosphere()
    return tab, o.Atmosphere(*tab)


def test_p22_linear_domain_reproduces_node_intensities(steep):
    (logT, logg, mu, logx, vals), atm = steep
    rng = np.random.default_rng(2)
    for _ in range(40):
        a, b, c, d = (rng.integers(0, n) for n in vals.shape)
        for strat in (1, 2, 3, 4):
            got = o.interp4_domain(atm, strat, 1, logT[a], logg[b], mu[c], logx[d])
            assert abs(got / 10.0 ** vals[a, b, c, d] - 1.0) < 1e-12


def test_p22_linear_domain_reproduces_polynomial_intensities():
    """If I/T^3 is a tensor-product polynomial of the local order, interpolating the INTENSITY is exact (it would not be
    exact for the logarithm): cubic on every axis for strategy a away from nothing (shifted stencils stay cubic)."""
    logT = np.linspace(5.0, 6.0, 7); logg = np.linspace(13.5, 14.5, 6)
    mu = np.array([0.0, 0.1, 0.25, 0.45, 0.6, 0.8, 0.9, 1.0]); logx = np.linspace(-1.0, 1.0, 9)
    pT = lambda t: 2.0 + 0.3 * (t - 5.5) - 0.2 * (t - 5.5) ** 3
    pg = lambda g: 1.5 + 0.4 * (g - 14.0) ** 2
    pm = lambda m: 1.0 + 2.0 * m - 0.5 * m ** 3
    px = lambda x: 3.0 + x + 0.6 * x ** 2 + 0.3 * x ** 3
    I = pT(logT)[:, None, None, None] * pg(logg)[None, :, None, None] * pm(mu)[None, None, :, None] * px(logx)[None, None, None, :]
    assert I.min() > 0
    atm = o.Atmosphere(logT, logg, mu, logx, np.log10(I))
    rng = np.random.default_rng(3)
    for _ in range(50):
        t, g, m, x = rng.uniform(5.0, 6.0), rng.uniform(13.5, 14.5), rng.uniform(0.0, 1.0), rng.uniform(-1.0, 1.0)
        exact = pT(t) * pg(g) * pm(m) * px(x)
        assert abs(o.interp4_domain(atm, 1, 1, t, g, m, x) / exact - 1.0) < 1e-12          # strategy a: cubic everywhere
    # strategy d: linear in T and g -> exact only for a table that is linear in them
    I2 = (1.0 + 0.2 * (logT - 5.0))[:, None, None, None] * (1.0 + 0.1 * (logg - 13.5))[None, :, None, None] \
        * pm(mu)[None, None, :, None] * px(logx)[None, None, None, :]
    atm2 = o.Atmosphere(logT, logg, mu, logx, np.log10(I2))
    for _ in range(50):
        t, g = rng.uniform(5.0, 6.0), rng.uniform(13.5, 14.5)
        m, x = rng.uniform(mu[3], mu[-2]), rng.uniform(logx[1], logx[-2])                   # cubic zones of mu and logx
        exact = (1.0 + 0.2 * (t - 5.0)) * (1.0 + 0.1 * (g - 13.5)) * pm(m) * px(x)
        assert abs(o.interp4_domain(atm2, 2, 1, t, g, m, x) / exact - 1.0) < 1e-12


def test_p22_strategy_b_is_strategy_a_clipped(steep):
    _, atm = steep
    rng = np.random.default_rng(4)
    kT6 = o.KB_KEV_K * 1e6
    neg = 0
    for _ in range(300):
        mu = 10.0 ** rng.uniform(-3.2, -1.4)
        Ep = kT6 * 10.0 ** rng.uniform(-1.2, 1.0)
        g = rng.uniform(13.8, 14.6)
        a = o.intensity(1, atm, 6.0, g, Ep, mu, domain=1)
        b = o.intensity(4, atm, 6.0, g, Ep, mu, domain=1)
        assert b == max(a, 0.0)
        neg += a < 0
        assert o.intensity(4, atm, 6.0, g, Ep, mu, domain=0) == o.intensity(1, atm, 6.0, g, Ep, mu, domain=0) > 0   # R13f
        # strategies c and d are linear in mu here (protected zone mu <= mu[3] = 0.04): between the node values, positive
        assert o.intensity(3, atm, 6.0, g, Ep, mu, domain=1) > 0 and o.intensity(2, atm, 6.0, g, Ep, mu, domain=1) > 0
    assert neg > 50                                     # the steep table does drive the cubic stencil below zero


def test_p22_both_domains_agree_on_a_smooth_table():
    atm = o.Atmosphere(*gen.synthetic_atmosphere())
    rng = np.random.default_rng(5)
    for _ in range(100):
        t, g, m, x = rng.uniform(5.3, 6.6), rng.uniform(13.9, 14.5), rng.uniform(0.1, 0.95), rng.uniform(-1.0, 1.2)
        for strat in (1, 2, 3):
            lin = o.interp4_domain(atm, strat, 1, t, g, m, x)
            log = 10.0 ** o.interp4_domain(atm, strat, 0, t, g, m, x)
            assert abs(lin / log - 1.0) < (2e-3 if strat == 2 else 5e-4)       # both are interpolation-error close to the truth


# ------------------------------------------------------------------------------------------------- P23
@pytest.mark.parametrize("which", [1, 2])
def test_p23_table3_geometries_lobes_holes_and_clean_profiles(which, steep):
    _, atm = steep
    conf = gen.config_interp_test(which, n_cells=8, n_phase=64, n_energy=16)
    f = {}
    for em in (1, 4, 3, 2):
        cfg = dict(conf["cfg"], emission=em, interp_domain=1)
        f[em], st = o.evaluate(cfg, conf["energies"], conf["params"][0], atm)
        assert st == 0
    peak = f[2].max()
    assert f[1].min() < -1e-2 * peak and (f[1] < 0).sum() > 100             # (a): pronounced negative intensities
    soft, hard = f[1][:, :8], f[1][:, 8:]
    assert (soft < 0).sum() > (hard < 0).sum()                              # predominantly in the soft band
    assert f[4].min() == 0.0 and (f[4] == 0).sum() > 50                     # (b): zero-intensity "holes"
    assert np.all(f[4] >= f[1] - 1e-12 * peak)                               # (OpenMP sums are not order-stable)
    for em in (3, 2):                                                       # (c), (d): physically consistent profiles
        # (bins 17 decades below the peak can still dip below zero: the cubic along log x overshoots in the Wien tail
        # when it acts on the intensity instead of its logarithm)
        assert f[em].min() > -1e-12 * peak and (f[em] > 0).mean() > 0.85 and np.all(f[em][np.abs(f[1]) > 1e-9 * peak] > 0)
    # in the logarithmic reading (R13a) every strategy is positive and (b) is (a) (R13f)
    g1, _ = o.evaluate(dict(conf["cfg"], emission=1), conf["energies"], conf["params"][0], atm)
    g4, _ = o.evaluate(dict(conf["cfg"], emission=4), conf["energies"], conf["params"][0], atm)
    assert g1.min() > 0 and np.allclose(g1, g4, rtol=1e-12, atol=0)
