"""Pins for the oracle's full evaluation: star scalars (P14), occultation (P8), invariants of the
discrete algorithm (P9), absolute scale against a closed form (P10), convergence (P13), fold (P15)
and Poisson likelihood (P16).  See DESIGN.md for the statements."""
import numpy as np
import pytest
from scipy import stats

import gen
import oracle as o


# ---------------------------------------------------------------------------------------- P14
def test_p14_star_and_row_scalars(golden):
    for M, Re, nu, q, th_deg, val, tol in golden("star_pins.txt"):
        M, Re, nu, th, val, tol = float(M), float(Re), float(nu), np.deg2rad(float(th_deg)), float(val), float(tol)
        st = o.star(M, Re, nu, True)
        th = max(th, 1e-9)
        rw = o.row(st, o.Box(th, th, np.pi, 0.1), 1, 0)
        got = dict(Rs_km=st.Rs_cm / 1e5, x=st.x, Obar2=st.Obar2, o2=st.o2, Rpole_km=st.Re_cm * (1 + st.o2) / 1e5,
                   u=rw.u, f=rw.f, beta=rw.beta, log10g=rw.log10g)[q]
        assert abs(got - val) <= tol * 1.01, (M, Re, nu, q, th_deg, got, val)


def test_row_geometry_identities():
    st = o.star(1.4, 12.0, 300.0, True)
    sp = o.spot(1.2, 0.3, 0.4, 6.0)
    bx = o.spot_box(sp, 32, 32)
    assert abs(bx.W - np.arcsin(np.sin(0.4) / np.sin(1.2))) < 1e-15
    tot = 0.0
    for j in range(32):
        r = o.row(st, bx, 32, j)
        assert abs(r.coseta ** 2 + r.sineta ** 2 - 1.0) < 1e-15
        assert abs(r.sineta / r.coseta - r.f) < 1e-15
        assert abs(r.gamma - 1.0 / np.sqrt(1.0 - r.beta ** 2)) < 1e-15
        # numerical dR/dtheta vs Eq 2
        h = 1e-6
        R = lambda t: st.Re_cm * (1.0 + st.o2 * np.cos(t) ** 2)
        f_num = (R(r.theta + h) - R(r.theta - h)) / (2 * h) / (r.R_cm * np.sqrt(1.0 - r.u))
        assert abs(f_num - r.f) < 1e-9
        tot += r.dcos
    assert abs(tot - (np.cos(0.8) - np.cos(1.6))) < 1e-15
    # sphere mode (reading R20)
    ss = o.star(1.4, 12.0, 300.0, False)
    rs = o.row(ss, bx, 32, 5)
    assert rs.f == 0.0 and rs.R_cm == ss.Re_cm and abs(rs.log10g - np.log10(ss.g0_cgs)) < 1e-15


def test_mask_cap_ring_and_area():
    sp = o.spot(1.0, 0.5, 0.3, 6.0)
    m = o.spot_mask(sp, 200, 200)
    bx = o.spot_box(sp, 200, 200)
    # centre-in area of the cap -> 2 pi (1 - cos zeta)
    area = 0.0
    for j in range(200):
        e0 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * j / 200
        e1 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (j + 1) / 200
        area += m[j].sum() * (np.cos(e0) - np.cos(e1)) * bx.dphi
    assert abs(area / (2 * np.pi * (1 - np.cos(0.3))) - 1.0) < 5e-3
    assert 0.77 < m.mean() < 0.80                               # ~ pi/4 of the bounding box
    # brute-force check of every cell with an independent vector formula
    th = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (np.arange(200) + 0.5) / 200
    ph = 0.5 - bx.W + (np.arange(200) + 0.5) * bx.dphi
    TH, PH = np.meshgrid(th, ph, indexing="ij")
    n = np.stack([np.sin(TH) * np.cos(PH), np.sin(TH) * np.sin(PH), np.cos(TH)], -1)
    c = np.array([np.sin(1.0) * np.cos(0.5), np.sin(1.0) * np.sin(0.5), np.cos(1.0)])
    sep = np.arccos(np.clip(n @ c, -1, 1))
    safe = np.abs(sep - 0.3) > 1e-9
    assert np.array_equal((sep <= 0.3)[safe], m.astype(bool)[safe])
    # ring: omitted inner cap removes cells
    thm, phm = gen.workloads._offset_point(1.0, 0.5, 0.05, 1.1)
    m2 = o.spot_mask(o.spot(1.0, 0.5, 0.3, 6.0, thm, phm, 0.12), 200, 200)
    cm = np.array([np.sin(thm) * np.cos(phm), np.sin(thm) * np.sin(phm), np.cos(thm)])
    sepm = np.arccos(np.clip(n @ cm, -1, 1))
    safe2 = safe & (np.abs(sepm - 0.12) > 1e-9)
    assert np.array_equal(((sep <= 0.3) & ~(sepm <= 0.12))[safe2], m2.astype(bool)[safe2])
    assert m2.sum() < m.sum()
    # polar cap uses the full azimuth range
    assert abs(o.spot_box(o.spot(0.05, 0.0, 0.1, 6.0), 8, 8).W - np.pi) < 1e-15


# ---------------------------------------------------------------------------------------- helpers
def _bb_cfg(n_cells=16, n_phase=32, n_fp=192, oblate=0, n_spots=1):
    return dict(n_spots=n_spots, n_theta=n_cells, n_phi=n_cells, n_phase=n_phase, n_fp=n_fp, emission=0, oblate=oblate)


E3 = np.array([0.3, 1.0, 3.0])
LT = gen.log10T_of_kT(0.3)


def _run(cfg, p, E=E3, atm=None):
    flux, status = o.evaluate(cfg, E, p, atm)
    assert status == 0
    return flux


# ---------------------------------------------------------------------------------------- P8
def test_p8_fully_occulted_spot_gives_exact_zero():
    ci = np.cos(0.3)
    p = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[(2.9, 0.0, 0.1, LT)])
    flux = _run(_bb_cfg(oblate=1), p)
    assert np.all(flux == 0.0)


# ---------------------------------------------------------------------------------------- P9
def test_p9_invariants():
    ci = np.cos(np.deg2rad(60.0))
    cfg = _bb_cfg(n_cells=12, n_phase=32, oblate=1)
    base = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[(0.7, 0.4, 0.25, LT)])
    f0 = _run(cfg, base)
    assert f0.min() > 0
    # (i) phi_c shift by 2 pi n / N_ph  <->  circular shift by n bins (Eq 45 depends on phi_out + phi_m/2pi only)
    n = 5
    p = base.copy(); p[9] += 2 * np.pi * n / 32
    f1 = _run(cfg, p)
    assert np.allclose(f1, np.roll(f0, -n, axis=0), rtol=1e-11, atol=0)
    # same with the phase-offset parameter
    p = base.copy(); p[6] = n / 32
    assert np.allclose(_run(cfg, p), np.roll(f0, -n, axis=0), rtol=1e-11, atol=0)
    # (ii) north-south mirror
    p = gen.pack_params(1.4, 12.0, 300.0, -ci, 0.2, spots=[(np.pi - 0.7, 0.4, 0.25, LT)])
    assert np.allclose(_run(cfg, p), f0, rtol=1e-10, atol=0)
    # (v) flux ~ D^-2
    p = base.copy(); p[4] *= 2.0
    assert np.allclose(_run(cfg, p) * 4.0, f0, rtol=1e-13, atol=0)
    # (iv) two spots = sum of the single-spot results
    s2 = (1.9, 2.0, 0.3, LT + 0.1)
    pa = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[(0.7, 0.4, 0.25, LT)])
    pb = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[s2])
    pab = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[(0.7, 0.4, 0.25, LT), s2])
    cfg2 = _bb_cfg(n_cells=12, n_phase=32, oblate=1, n_spots=2)
    assert np.allclose(_run(cfg2, pab), _run(cfg, pa) + _run(cfg, pb), rtol=1e-13, atol=0)
    # (vii) mirrored spot moved by half a turn -> half-period circular shift
    p = gen.pack_params(1.4, 12.0, 300.0, -ci, 0.2, spots=[(np.pi - 0.7, 0.4 + np.pi, 0.25, LT)])
    assert np.allclose(_run(cfg, p), np.roll(f0, -16, axis=0), rtol=1e-10, atol=0)


def test_p9_symmetry_without_rotation():
    """(iii) nu -> 0: F_t(phase) is symmetric about the phase at which the spot centre crosses the observer meridian."""
    cfg = _bb_cfg(n_cells=12, n_phase=32, oblate=0)
    p = gen.pack_params(1.4, 12.0, 0.0, 0.5, 0.2, spots=[(0.9, 0.0, 0.3, LT)])
    f = _run(cfg, p)
    # spot centre crosses the meridian at phase 0: F(k) = F(N-k)
    assert np.allclose(f[1:], f[1:][::-1], rtol=1e-10, atol=0)
    # with rotation the Doppler boost breaks the symmetry
    p[2] = 400.0
    f = _run(cfg, p)
    assert np.max(np.abs(f[1:] / f[1:][::-1] - 1.0)) > 1e-2


def test_p9_axisymmetric_cap_is_phase_independent():
    """(vi) cap centred on the rotation axis: constant in phase when the azimuth cell count is a multiple of N_ph."""
    cfg = _bb_cfg(n_cells=32, n_phase=16, oblate=1)
    p = gen.pack_params(1.4, 12.0, 300.0, 0.6, 0.2, spots=[(0.0, 0.0, 0.3, LT)])
    f = _run(cfg, p)
    assert np.max(np.abs(f / f[0:1] - 1.0)) < 1e-12


# ---------------------------------------------------------------------------------------- P10
def test_p10_absolute_scale_against_closed_form(golden):
    pins = {(q, float(E)): float(v) for q, E, v in golden("cap_flux_pins.txt")}
    M, Rkm, zeta, kT, Dkpc = 1.4, 12.0, 0.2, 0.3, 0.2
    st = o.star(M, Rkm, 0.0, False)
    u = st.Rs_cm / st.Re_cm
    assert abs(u - 0.344545842258) < 1e-11
    a_z = o.alpha_of_psi(u, zeta, np.pi / 2)
    assert abs(a_z - pins[("alpha_zeta", 0.0)]) < 1e-11
    D_cm = Dkpc * 1e3 * o.PC_CM

    def closed(E):
        Ep = E / np.sqrt(1 - u)
        Ibb = o.TWO_OVER_H3C2 * Ep ** 3 / np.expm1(Ep / kT)
        return np.sqrt(1 - u) * Ibb / E * np.pi * st.Re_cm ** 2 * np.sin(a_z) ** 2 / D_cm ** 2
    for E in (0.3, 1.0, 3.0):
        assert abs(closed(E) / pins[("flux", E)] - 1.0) < 1e-9
    # the discrete oracle converges to it (cap centred on the line of sight: i = 0, theta_c = 0)
    errs = []
    for N in (8, 16, 32):
        cfg = _bb_cfg(n_cells=N, n_phase=4, n_fp=8, oblate=0)
        p = gen.pack_params(M, Rkm, 0.0, 1.0, Dkpc, spots=[(0.0, 0.0, zeta, gen.log10T_of_kT(kT))])
        f = _run(cfg, p)
        assert np.max(np.abs(f / f[0:1] - 1.0)) < 1e-12
        errs.append(np.max(np.abs(f[0] / np.array([closed(E) for E in E3]) - 1.0)))
    assert errs[2] < 2e-4 and errs[0] > errs[1] > errs[2]
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0      # midpoint rule in theta: 2nd order


def test_p2_flat_space_small_spot():
    """M -> 0, nu = 0: F(E) = I_bb(E)/E * sum_cells cos(psi_cell) dS_cell / D^2 (Eq 21 with u = 0, delta = gamma = 1,
    d cos(alpha)/d cos(psi) = 1, sigma = alpha = psi)."""
    Dkpc, kT, zeta = 0.2, 0.3, 0.05
    i_obs, th_c = 0.5, 0.9
    N = 16
    cfg = _bb_cfg(n_cells=N, n_phase=8, n_fp=2048, oblate=0)
    p = gen.pack_params(1e-8, 12.0, 0.0, np.cos(i_obs), Dkpc, spots=[(th_c, 0.0, zeta, gen.log10T_of_kT(kT))])
    f = _run(cfg, p)
    sp = o.spot(th_c, 0.0, zeta, 0.0)
    mask = o.spot_mask(sp, N, N)
    bx = o.spot_box(sp, N, N)
    st = o.star(1e-8, 12.0, 0.0, False)
    D_cm = Dkpc * 1e3 * o.PC_CM
    for k in range(8):
        proj = 0.0
        for j in range(N):
            r = o.row(st, bx, N, j)
            for m in range(N):
                if mask[j, m]:
                    phi = -bx.W + (m + 0.5) * bx.dphi + 2 * np.pi * k / 8
                    cpsi = np.sin(i_obs) * np.sin(r.theta) * np.cos(phi) + np.cos(i_obs) * np.cos(r.theta)
                    proj += max(cpsi, 0.0) * r.dcos * bx.dphi * st.Re_cm ** 2
        for e, E in enumerate(E3):
            ref = o.TWO_OVER_H3C2 * E ** 3 / np.expm1(E / kT) / E * proj / D_cm ** 2
            assert abs(f[k, e] / ref - 1.0) < 2e-6     # template interpolation error ~ (2 pi / N_fp)^2 / 8


# ---------------------------------------------------------------------------------------- P13
def test_p13_convergence_in_nfp_and_cells():
    ci = np.cos(np.deg2rad(60.0))
    p = gen.pack_params(1.4, 12.0, 300.0, ci, 0.2, spots=[(0.7, 0.0, 0.25, LT)])
    ref = _run(_bb_cfg(n_cells=8, n_phase=16, n_fp=2048, oblate=1), p)
    e = [np.abs(_run(_bb_cfg(n_cells=8, n_phase=16, n_fp=n, oblate=1), p) - ref).sum() / ref.sum() for n in (64, 128, 256)]
    assert e[0] > e[1] > e[2]
    assert 2.8 < e[0] / e[1] < 5.5 and 2.8 < e[1] / e[2] < 5.5          # linear Interp: error ~ 1/N_fp^2
    # cells: centre-in mask -> first-order convergence; total (phase-averaged) flux settles
    tot = [(_run(_bb_cfg(n_cells=n, n_phase=16, n_fp=192, oblate=1), p)).mean(axis=0) for n in (16, 32, 64, 128)]
    d = [np.max(np.abs(tot[i] / tot[3] - 1.0)) for i in range(3)]
    assert d[2] < d[0] and d[2] < 1e-2


# ---------------------------------------------------------------------------------------- domain / status
def test_status_codes():
    cfg = _bb_cfg()
    ok = gen.pack_params(1.4, 12.0, 200.0, 0.5, 0.2, spots=[(0.7, 0.0, 0.2, LT)])
    bad_u = ok.copy(); bad_u[0] = 2.6                    # u_eq = 0.64 > 0.56
    f, s = o.evaluate(cfg, E3, bad_u)
    assert s & 1 and np.all(np.isnan(f))
    bad_nan = ok.copy(); bad_nan[3] = np.nan
    assert o.evaluate(cfg, E3, bad_nan)[1] & 2
    bad_spot = ok.copy(); bad_spot[10] = 0.0
    assert o.evaluate(cfg, E3, bad_spot)[1] & 4


# ---------------------------------------------------------------------------------------- P15 / P16
def test_p15_fold_conserves_row_sums():
    E = gen.logspace(0.2, 12.0, 60)
    rsp = gen.synthetic_response(E, n_channel=1500)
    rng = np.random.default_rng(3)
    flux = rng.uniform(0.1, 1.0, size=(4, 60))
    NH = 0.7
    counts = o.fold(flux, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], NH, 1500)
    full_rows = (rsp["first_chan"] >= 0) & (rsp["first_chan"] + rsp["rsp_band"].shape[1] <= 1500)
    # dense reference
    dense = np.zeros((60, 1500))
    for e in range(60):
        for w in range(rsp["rsp_band"].shape[1]):
            c = rsp["first_chan"][e] + w
            if 0 <= c < 1500:
                dense[e, c] = rsp["rsp_band"][e, w]
    ref = (flux * np.exp(-NH * rsp["tau_ref"])[None, :]) @ dense
    assert np.allclose(counts, ref, rtol=1e-13, atol=1e-300)
    # rows of K sum to 1 => channel-summed counts = sum_e F ATT w A
    att = np.exp(-NH * rsp["tau_ref"])
    assert np.allclose(dense.sum(axis=1)[full_rows], (rsp["w"] * rsp["area"])[full_rows], rtol=1e-12)
    # N_H = 0, A = 1: channel-summed counts = trapezoid integral of F_t over E
    band1 = rsp["rsp_band"] / rsp["area"][:, None]
    c1 = o.fold(flux, rsp["first_chan"], band1, rsp["tau_ref"], 0.0, 1500)
    keep = full_rows
    fl = flux * keep[None, :]
    c1 = o.fold(fl, rsp["first_chan"], band1, rsp["tau_ref"], 0.0, 1500)
    assert np.allclose(c1.sum(axis=1), (fl * rsp["w"][None, :]).sum(axis=1), rtol=1e-12)
    w_trap = rsp["w"]
    assert abs((w_trap * np.ones(60)).sum() - (E[-1] - E[0])) < 1e-12
    del att


def test_p16_loglike_is_poisson_logpmf():
    rng = np.random.default_rng(4)
    counts = rng.uniform(0.0, 3.0, size=(8, 20))
    counts[0, 0] = 0.0
    bkg = rng.uniform(0.01, 0.2, size=20)
    t_exp = 50.0
    m = t_exp * counts / 8 + bkg[None, :]
    d = rng.poisson(m).astype(float)
    ll = o.loglike(counts, d, bkg, t_exp)
    assert abs(ll - stats.poisson.logpmf(d, m).sum()) < 1e-9 * abs(ll)
    # 0 ln 0 := 0 ; -inf when m = 0 < d
    d0 = d.copy(); d0[0, 0] = 0.0
    assert np.isfinite(o.loglike(counts, d0, None, t_exp))
    d1 = d.copy(); d1[0, 0] = 2.0
    assert o.loglike(counts, d1, None, t_exp) == -np.inf
    # large counts: -2 (lnL(m) - lnL(d)) ~ chi^2
    m_big = rng.uniform(2e3, 5e3, size=(8, 20))
    d_big = rng.poisson(m_big).astype(float)
    ll_m = o.loglike(m_big * 8, d_big, None, 1.0)
    ll_d = o.loglike(d_big * 8, d_big, None, 1.0)
    chi2 = ((m_big - d_big) ** 2 / m_big).sum()
    assert abs(-2 * (ll_m - ll_d) / chi2 - 1.0) < 0.02
    # Eq 56-57 helper
    assert abs(o.chi2(m_big, d_big) - 1e6 / m_big.sum() * chi2) < 1e-9 * chi2


# ---------------------------------------------------------------------------------------- beaming laws
def test_beaming_laws_closed_form_and_linearity(golden):
    """Blackbody with the parametric beaming laws prop. to cos^2(sigma'), sin^2(sigma') (reading R23).
    Face-on cap of pin P10 (non-rotating sphere, sigma' = alpha): integrating Eq 21 over the cap gives
      F_cos2 / F_iso = (1 + cos^2 a_z) / 2,   F_sin2 / F_iso = sin^2(a_z) / 2,
    with a_z the emission angle at the cap's rim; and for ANY geometry F_iso = F_cos2 + F_sin2 (the laws add to 1)."""
    pins = {(q, float(E)): float(v) for q, E, v in golden("cap_flux_pins.txt")}
    a_z = pins[("alpha_zeta", 0.0)]
    p = gen.pack_params(1.4, 12.0, 0.0, 1.0, 0.2, spots=[(0.0, 0.0, 0.2, LT)])
    f = {}
    for b in (0, 1, 2):
        cfg = dict(_bb_cfg(n_cells=256, n_phase=2, n_fp=8, oblate=0), beaming=b)
        f[b] = _run(cfg, p)[0]
    assert np.max(np.abs(f[1] / f[0] / ((1 + np.cos(a_z) ** 2) / 2) - 1)) < 2e-5
    assert np.max(np.abs(f[2] / f[0] / (np.sin(a_z) ** 2 / 2) - 1)) < 2e-3          # rim-weighted: mask edge error
    # linearity on a rotating oblate geometry
    p2 = gen.pack_params(1.4, 12.0, 400.0, np.cos(1.1), 0.2, spots=[(0.8, 0.3, 0.6, LT)])
    g = {b: _run(dict(_bb_cfg(n_cells=24, n_phase=16, oblate=1), beaming=b), p2) for b in (0, 1, 2)}
    assert np.max(np.abs((g[1] + g[2]) / g[0] - 1)) < 1e-13
    assert np.all(g[1] >= 0) and np.all(g[2] >= 0) and g[2].max() > 0
