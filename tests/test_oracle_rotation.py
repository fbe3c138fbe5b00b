"""Pins P17-P21 for the parts of the oracle's ring template (oracle/ppm_oracle.c: orc_template, O3 + O4) that the
non-rotating pins P2 / P10 cannot see: the Doppler factor and its sign, the powers of delta and the gamma of Eq 40,
z = 1/(delta sqrt(1-u)), the sign of nu * Delta t in phi_o, the sin(eta) term of Eq 39, the invisible-range fill of
Eq 41-44, and the Obar^6 terms of Eq 10.

Every pin compares the oracle with something built *outside* it: unit vectors of Table 1-2, the
Lorentz transformation of Appendix A, the arrival-time relation of Appendix B,
the surface equation Eq 7, or Eq 41-44 written out on the oracle's own *visible* entries.
"""
import numpy as np
import pytest

import gen
import oracle as o

C = o.C_CM_S


def _unit(v):
    return v / np.linalg.norm(v)


def _vectors(inc, theta, phi):
    """Table 1-2 in the frame of Fig 1: z = rotation axis, observer in the x-z plane, the patch rotates towards
    increasing azimuth (reading R17)."""
    k = np.array([np.sin(inc), 0.0, np.cos(inc)])                                  # to the observer
    r = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    th = np.array([np.cos(theta) * np.cos(phi), np.cos(theta) * np.sin(phi), -np.sin(theta)])
    ph = np.array([-np.sin(phi), np.cos(phi), 0.0])                                # velocity direction beta-hat
    return k, r, th, ph


# ------------------------------------------------------------------------------------------------- P17
def test_p17_rotating_spot_in_flat_space_is_a_moving_blackbody():
    """Flat-space limit (M -> 0) of a small spot on a rapidly rotating SPHERE, whole evaluation against first principles.

    Derivation (not from the oracle's code).  A patch of rest-frame (comoving) area dS' moves with velocity beta along
    phi-hat and emits a blackbody of temperature T in its rest frame.  (1) I/E^3 is Lorentz invariant, so in the static
    frame the patch shows a blackbody of temperature delta*T, delta = 1/(gamma (1 - beta cos xi)), cos xi = beta-hat . k-hat
    (Eq 19; App. A): I(E) = (2/h^3 c^2) E^3 / expm1(E / (delta k T)).  (2) Photons leaving during the
    static-frame interval dt_emit arrive during dt_rec = (1 - beta cos xi) dt_emit = dt_emit / (gamma delta) (Eq B.8,
    PAPER.md:1009).  (3) In the static frame the patch is length-contracted along its motion, which lies in the surface:
    dS = dS'/gamma with dS' = gamma R^2 dcos(theta) dphi (the "gamma R^2 ... dcos(theta) dphi" of Eq 21).
    Photon rate per detector area, per energy, at distance D, in arrival time:
        F(E) = [I(E)/E] * cos(sigma) dS / D^2 * (gamma delta)
             = gamma * delta * cos(sigma) * (2/h^3 c^2) E^2 / expm1(E/(delta k T)) * R^2 dcos(theta) dphi / D^2,
    with cos(sigma) = r-hat . k-hat (sphere, straight rays).  "Approaching patches (cos xi > 0) are boosted"
    (PAPER.md:224).  Arrival phase: a photon from the point beneath the observer has zero delay and any other photon
    arrives LATER by the extra path R (1 - cos psi)/c, so a cell with azimuth phi_m that emits at
    phase t (azimuth phi_m + 2 pi t) is seen at phase t + nu R (1 - cos psi)/c.

    Fixes: the sign of cos xi, the exponent of delta and the gamma in F, z = 1/delta, the sign of nu*Delta t."""
    M, Rkm, nu, inc, Dkpc, kT = 1e-8, 12.0, 600.0, np.deg2rad(35.0), 0.2, 0.3
    th_c, zeta, N, n_phase, n_fp = np.deg2rad(48.0), 0.04, 6, 16, 4096
    E = np.array([0.3, 1.0, 3.0])
    cfg = dict(n_spots=1, n_theta=N, n_phi=N, n_phase=n_phase, n_fp=n_fp, emission=0, oblate=0)
    p = gen.pack_params(M, Rkm, nu, np.cos(inc), Dkpc, spots=[(th_c, 0.3, zeta, gen.log10T_of_kT(kT))])
    flux, status = o.evaluate(cfg, E, p)
    assert status == 0 and flux.min() > 0

    sp = o.spot(th_c, 0.3, zeta, 0.0)
    mask = o.spot_mask(sp, N, N)                      # pinned by brute-force unit vectors in test_oracle_model.py
    bx = o.spot_box(sp, N, N)
    R = Rkm * 1e5
    D = Dkpc * 1e3 * o.PC_CM
    ref = np.zeros_like(flux)
    for j in range(N):
        e0 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * j / N
        e1 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (j + 1) / N
        theta, dcos = 0.5 * (e0 + e1), np.cos(e0) - np.cos(e1)
        beta = 2 * np.pi * nu * R * np.sin(theta) / C
        gam = 1.0 / np.sqrt(1.0 - beta * beta)
        for m in range(N):
            if not mask[j, m]:
                continue
            phi_m = 0.3 - bx.W + (m + 0.5) * bx.dphi
            for k in range(n_phase):
                t = k / n_phase                                              # emission phase: fixed point of the arrival map
                for _ in range(60):
                    kv, rv, _, _ = _vectors(inc, theta, phi_m + 2 * np.pi * t)
                    t = k / n_phase - nu * R * (1.0 - rv @ kv) / C
                kv, rv, _, pv = _vectors(inc, theta, phi_m + 2 * np.pi * t)
                cos_sigma = rv @ kv
                assert cos_sigma > 0.05                                      # geometry chosen always visible
                delta = 1.0 / (gam * (1.0 - beta * (pv @ kv)))
                ref[k] += gam * delta * cos_sigma * o.TWO_OVER_H3C2 * E ** 2 / np.expm1(E / (delta * kT)) \
                    * R * R * dcos * bx.dphi / D ** 2
    # N_fp = 4096: linear template interpolation error ~ (2 pi / N_fp)^2 / 8 x O(E/kT) ~ 1e-6; u = 2.5e-9
    assert np.max(np.abs(flux / ref - 1.0)) < 1e-5
    # the rotation terms matter at the 10 % level here, so the pin has teeth
    assert np.max(ref[:, 2]) / np.min(ref[:, 2]) > 1.3


# ------------------------------------------------------------------------------------------------- P18
@pytest.mark.parametrize("theta", [0.5, 1.25, 2.1])
def test_p18_template_angles_against_unit_vectors(theta):
    """Oblate, fast, compact star: for every visible template entry rebuild cos(sigma) = n-hat . k0-hat and
    cos(xi) = beta-hat . k0-hat from the vectors of Table 1 and compare with what the template stores.
      * k0-hat lies in the plane of r-hat and k-hat at angle alpha from r-hat (Table 2: alpha = angle(r, k0)).
      * n-hat is the normal of the surface r = R(theta) of Eq 7: gradient of r - R(theta) with proper lengths
        dr/sqrt(1-u) and r dtheta, i.e. n ~ r-hat - [R'(theta) / (R sqrt(1-u))] theta-hat; R' by central differences of
        Eq 7 here, so neither Eq 2-3 nor Eq 39 is retyped.
      * delta from Eq 19 with cos xi = phi-hat . k0-hat and beta from Eq 18; stored: z = 1/(delta sqrt(1-u)), mu = delta cos sigma.
    Fixes the sin(eta) term of Eq 39 (sign and magnitude), cos(xi) (Table 2) in curved space, mu and z of Eq 40; and the
    lag's sign: phi_o - phi/2pi = nu Delta t >= 0, smallest where the patch is closest to the observer."""
    M, Rkm, nu, inc = 1.8, 11.0, 600.0, 1.0
    st = o.star(M, Rkm, nu, True)
    n_fp = 48
    rw = o.row(st, o.Box(theta - 0.01, theta + 0.01, np.pi, 0.1), 1, 0)
    assert abs(rw.theta - theta) < 1e-15 and abs(rw.sineta) > 1e-3
    tpl = o.template(st, rw, np.cos(inc), 1.0, 1.0, n_fp)
    Rf = lambda t: st.Re_cm * (1.0 + st.o2 * np.cos(t) ** 2)                  # Eq 7
    h = 1e-5
    slope = (Rf(theta + h) - Rf(theta - h)) / (2 * h) / (Rf(theta) * np.sqrt(1.0 - rw.u))
    beta = 2 * np.pi * nu * Rf(theta) * np.sin(theta) / (C * np.sqrt(1.0 - rw.u))   # Eq 18
    gam = 1.0 / np.sqrt(1.0 - beta ** 2)
    lag = tpl["phio"][:n_fp] - np.arange(n_fp) / n_fp
    nvis = 0
    for i in range(n_fp):
        if not tpl["vis"][i]:
            continue
        nvis += 1
        k, r, th, ph = _vectors(inc, theta, 2 * np.pi * i / n_fp)
        cpsi = r @ k
        e = _unit(k - cpsi * r)
        a = tpl["alpha"][i]
        k0 = np.cos(a) * r + np.sin(a) * e
        n = _unit(r - slope * th)
        cos_sigma = n @ k0
        delta = 1.0 / (gam * (1.0 - beta * (ph @ k0)))
        assert abs(1.0 / (tpl["z"][i] * np.sqrt(1.0 - rw.u)) - delta) < 1e-12
        assert abs(tpl["mu"][i] - delta * cos_sigma) < 1e-9                   # R' by finite differences: 1e-10
        assert lag[i] > 0.0
    assert nvis >= n_fp // 2
    vis = tpl["vis"][:n_fp].astype(bool)
    psi = np.arccos(np.clip([_vectors(inc, theta, 2 * np.pi * i / n_fp)[1] @ _vectors(inc, theta, 0.0)[0]
                             for i in range(n_fp)], -1, 1))
    order = np.argsort(psi[vis])
    assert np.all(np.diff(lag[vis][order]) > -1e-15)                          # later the further from the sub-observer point
    # approaching side (phi < 0, i.e. i_fp > N_fp/2) is blueshifted: smaller z than the mirror entry on the receding side
    for i in range(1, n_fp // 2):
        if vis[i] and vis[n_fp - i]:
            assert tpl["z"][n_fp - i] < tpl["z"][i]


# ------------------------------------------------------------------------------------------------- P19
@pytest.mark.parametrize("oblate", [0, 1])
def test_p19_invisible_range_fill_eq_41_44(oblate):
    """Partially visible ring: Eq 41-44 written out on the template's own visible entries.
    Sphere: the invisible set is exactly {psi > psi(u, pi/2)} (psi pinned by P1); visibility is even in phi."""
    M, Rkm, nu, inc, theta, n_fp = 1.4, 12.0, 300.0, 1.3, 2.2, 96
    st = o.star(M, Rkm, nu, bool(oblate))
    rw = o.row(st, o.Box(theta - 0.01, theta + 0.01, np.pi, 0.1), 1, 0)
    tpl = o.template(st, rw, np.cos(inc), 3e20, 1e-4, n_fp)
    vis = tpl["vis"][:n_fp].astype(bool)
    assert tpl["visible"] and vis[0] and 10 < (~vis).sum() < n_fp - 10
    inv = np.flatnonzero(~vis)
    a, b = inv.min(), inv.max()
    assert np.array_equal(inv, np.arange(a, b + 1))                           # contiguous (reading R9)
    assert b == n_fp - a                                                       # even in phi
    if not oblate:
        phi = 2 * np.pi * np.arange(n_fp) / n_fp
        psi = np.arccos(np.sin(inc) * np.sin(theta) * np.cos(phi) + np.cos(inc) * np.cos(theta))
        assert np.array_equal(vis, psi <= o.psi(rw.u, np.pi / 2))
    F, z, po, mu = tpl["F"], tpl["z"], tpl["phio"], tpl["mu"]
    assert np.all(F[:a] > 0) and np.all(F[b + 1:] > 0) and np.all(mu[:a] > 0) and np.all(mu[b + 1:] > 0)
    x0, x1 = a - 1, b + 1                                                      # points of disappearance / reappearance
    for i in range(a, b + 1):
        assert F[i] == 0.0 and mu[i] == 0.0                                    # Eq 41
        Lz = z[x0] + (z[x1] - z[x0]) * (i - x0) / (x1 - x0)                    # Eq 42 with Eq 44
        Lp = po[x0] + (po[x1] - po[x0]) * (i - x0) / (x1 - x0)                 # Eq 43
        assert abs(z[i] - Lz) < 1e-15 and abs(po[i] - Lp) < 1e-15
    assert np.all(np.diff(po) > 0)                                             # phi_o stays strictly increasing (Eq 45-46 need it)
    assert z[x0] > 0.5 and z[x1] > 0.5 and abs(po[n_fp] - po[0] - 1.0) < 1e-15 and F[n_fp] == F[0]
    # the neighbours of the range are genuine (unfilled) template values: z = 1/(delta sqrt(1-u)) within Doppler bounds
    zs = 1.0 / np.sqrt(1.0 - rw.u)
    assert zs / (rw.gamma * (1 + rw.beta)) / 1.0001 < z[x1] < z[x0] < zs * rw.gamma * (1 + rw.beta) * 1.0001


def test_p19_convergence_in_nfp_on_a_partially_visible_ring():
    """P13 repeated on a ring that is hidden for part of the rotation: the evaluation still converges as N_fp grows
    (at least first order: the limb is a kink of F, where linear interpolation loses one order locally)."""
    cfg = lambda n: dict(n_spots=1, n_theta=6, n_phi=6, n_phase=16, n_fp=n, emission=0, oblate=1)
    p = gen.pack_params(1.4, 12.0, 300.0, np.cos(1.3), 0.2, spots=[(2.2, 0.4, 0.15, gen.log10T_of_kT(0.3))])
    E = np.array([0.3, 1.0, 3.0])
    ref, s = o.evaluate(cfg(4096), E, p)
    assert s == 0 and (ref == 0).any() and (ref > 0).any()                    # hidden at some output phases, seen at others
    err = []
    for n in (64, 128, 256, 512):
        f, _ = o.evaluate(cfg(n), E, p)
        err.append(np.abs(f - ref).sum() / ref.sum())
    assert err[0] > err[1] > err[2] > err[3]
    assert err[0] / err[2] > 3.5 and err[1] / err[3] > 3.5


# ------------------------------------------------------------------------------------------------- P20
def test_p20_effective_gravity_eq10_all_nine_coefficients():
    """Eq 10 evaluated from a coefficient table typed from the paper, at Obar^2 = 0.0713 (M = 2, R_e = 11 km,
    600 Hz) where the Obar^6 terms move log10 g by 5e-5 -- far above this test's tolerance."""
    st = o.star(2.0, 11.0, 600.0, True)
    O2, x = st.Obar2, st.x
    assert abs(O2 - 0.07127) < 1e-5 and abs(x - 0.2685) < 1e-4               # P14 probe values
    # rows: [coefficient of x^0, x^1, x^2] for Obar^2, Obar^4, Obar^6
    c_sin = np.array([[-0.791, 0.776, 0.0], [0.0, -1.315, 2.431], [0.0, -1.172, 0.0]])
    c_cos = np.array([[1.138, -1.431, 0.0], [0.0, 0.653, -2.864], [0.0, 0.975, 0.0]])
    c_abs = np.array([0.0, 13.47, -27.13])                                     # Obar^4 only
    xp = np.array([1.0, x, x * x])
    Op = np.array([O2, O2 ** 2, O2 ** 3])
    e4 = O2 ** 2 * (c_abs @ xp)
    for th in (1e-9, 0.4, np.pi / 4, 1.1, np.pi / 2, 2.3):
        s2, c2 = np.sin(th) ** 2, np.cos(th) ** 2
        ratio = 1.0 + s2 * (Op @ (c_sin @ xp)) + c2 * (Op @ (c_cos @ xp) - e4) + abs(np.cos(th)) * e4
        rw = o.row(st, o.Box(th, th, np.pi, 0.1), 1, 0)
        assert abs(rw.log10g - np.log10(st.g0_cgs * ratio)) < 1e-13
    # the Obar^6 terms are visible at this spin: dropping them moves g by > 1e-5
    drop6 = 1.0 + 1.0 * (Op[:2] @ (c_sin @ xp)[:2])
    assert abs(drop6 / (1.0 + Op @ (c_sin @ xp)) - 1.0) > 1e-5
    # gravity is enhanced at the poles and reduced at the equator
    g_pole = o.row(st, o.Box(1e-9, 1e-9, np.pi, 0.1), 1, 0).log10g
    g_eq = o.row(st, o.Box(np.pi / 2, np.pi / 2, np.pi, 0.1), 1, 0).log10g
    assert g_pole > np.log10(st.g0_cgs) > g_eq
