"""Pins for the oracle's per-cell temperature map (reading R24).  The map path has a plain definition
in terms of the uniform-temperature path, which is pinned elsewhere (P8-P13): (i) a constant map equals the uniform
spot; (ii) maps with disjoint supports add; (iii) on the HEALPix mesh, which every spot shares, a two-temperature map
equals the sum of two masked uniform spots pixel for pixel; (iv) NaN cells do not emit."""
import numpy as np
import pytest

import gen
import oracle as o


@pytest.fixture(scope="module")
def atm():
    return o.Atmosphere(*gen.synthetic_atmosphere())


def _conf(emission=2):
    c = gen.config_c3(n_cells=14, n_phase=10, n_energy=12)
    return dict(c["cfg"], emission=emission), c["energies"], c["params"][0]


@pytest.mark.parametrize("emission", [2, 1, 3])                     # strategies d, a, c: linear / cubic / cubic-linedge in log T
def test_constant_map_equals_uniform_spot(atm, emission):
    cfg, E, p = _conf(emission)
    f0, _ = o.evaluate(cfg, E, p, atm)
    tm = np.empty((2, 14, 14))
    tm[0], tm[1] = p[8 + 3], p[16 + 3]
    f1, st = o.evaluate(cfg, E, p, atm, tmap=tm)
    assert st == 0 and np.max(np.abs(f1 / f0 - 1)) < 1e-13
    q = p.copy()
    q[[8 + 3, 16 + 3]] = 5.5                                        # the spot's own temperature is ignored with a map
    f2, _ = o.evaluate(cfg, E, q, atm, tmap=tm)
    assert np.array_equal(f1 == 0, f2 == 0) and np.max(np.abs(f2 / f1 - 1)) < 1e-13


def test_disjoint_maps_add_and_nan_cells_do_not_emit(atm):
    cfg, E, p = _conf()
    rng = np.random.default_rng(8)
    tm = rng.uniform(5.8, 6.4, size=(2, 14, 14))
    sel = rng.random((2, 14, 14)) < 0.5
    a, b = np.where(sel, tm, np.nan), np.where(sel, np.nan, tm)
    fa, _ = o.evaluate(cfg, E, p, atm, tmap=a)
    fb, _ = o.evaluate(cfg, E, p, atm, tmap=b)
    f, _ = o.evaluate(cfg, E, p, atm, tmap=tm)
    assert f.max() > 0 and np.max(np.abs((fa + fb) / f - 1)) < 1e-12
    fn, _ = o.evaluate(cfg, E, p, atm, tmap=np.full((2, 14, 14), np.nan))
    assert np.all(fn == 0)


@pytest.mark.parametrize("emission", [2, 1, 3])
def test_two_temperature_map_on_healpix_equals_two_masked_spots(atm, emission):
    """Inner cap at T1 + surrounding ring at T2.  As spots: a cap (zeta = 0.15) and a cap (zeta = 0.4) with that inner
    cap omitted; as a map: one spot (zeta = 0.4) whose pixels carry T1 inside the inner cap and T2 outside."""
    nside = 12
    E = gen.logspace(0.2, 8.0, 10)
    th, ph = 1.1, 0.7
    T1, T2 = 6.35, 5.95
    base = dict(n_theta=4 * nside - 1, n_phi=4 * nside, n_phase=8, n_fp=192, emission=emission, oblate=1, mesh=1)
    p2 = gen.pack_params(1.4, 12.0, 300.0, 0.5, 0.2, spots=[(th, ph, 0.15, T1), (th, ph, 0.4, T2, th, ph, 0.15)])
    f_spots, st = o.evaluate(dict(base, n_spots=2), E, p2, atm)
    inner = o.spot_mask_healpix(o.spot(th, ph, 0.15, T1), nside).astype(bool)
    outer = o.spot_mask_healpix(o.spot(th, ph, 0.4, T2), nside).astype(bool)
    tm = np.where(inner, T1, np.where(outer, T2, np.nan))[None]
    p1 = gen.pack_params(1.4, 12.0, 300.0, 0.5, 0.2, spots=[(th, ph, 0.4, 0.0)])
    f_map, st1 = o.evaluate(dict(base, n_spots=1), E, p1, atm, tmap=tm)
    assert st == 0 and st1 == 0 and f_spots.max() > 0
    assert np.max(np.abs(f_map / f_spots - 1)) < 1e-12
    # and the temperatures matter: swapping them changes the spectrum
    tm2 = np.where(inner, T2, np.where(outer, T1, np.nan))[None]
    f_sw, _ = o.evaluate(dict(base, n_spots=1), E, p1, atm, tmap=tm2)
    assert np.max(np.abs(f_sw / f_map - 1)) > 0.1
