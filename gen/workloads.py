"""Synthetic workloads C1..C5 / T of BASELINE.json, generated with numpy PCG64 streams.

Every array an evaluation consumes is produced here and handed unchanged to BOTH the CPU
oracle and the CUDA path ("identical seeded inputs" = identical arrays).  The shapes, ranges
and structure follow what the paper states (atmosphere axes PAPER.md:249; resolution tiers
Table 4; energy grid Eq 50; star / observer settings
PAPER.md:486, 573-575; ring = emitter + nested non-concentric mask PAPER.md:575) -- they stand
in for the NSX-H table, NICER response, tbnew table and benchmark spot parameters, none of
which are available.  Nothing here evaluates the model.
"""
import numpy as np

SEED0 = 20251007

# physical constants used ONLY to lay out synthetic data (CODATA 2019 exact SI)
_C = 299792458.0
_H = 6.62607015e-34
_KB = 1.380649e-23
_E = 1.602176634e-19
_GMSUN = 1.32712440018e20

N_SPOT_PARAMS = 8
N_STAR_PARAMS = 8


def linspace(lo, hi, n):
    """Eq 30-31."""
    i = np.arange(n, dtype=np.float64)
    return lo + (hi - lo) * i / (n - 1)


def logspace(lo, hi, n):
    """Eq 48-49."""
    i = np.arange(n, dtype=np.float64)
    return np.exp(np.log(lo) + (np.log(hi) - np.log(lo)) * i / (n - 1))


def pack_params(M, Re_km, nu, cos_i, D_kpc, NH20=0.0, phase0=0.0, spots=()):
    """[M, R_eq, nu, cos i, D, N_H/1e20, phase offset, 0] + per spot
    [theta_c, phi_c, zeta, log10T, theta_m, phi_m, zeta_m, 0]."""
    v = [M, Re_km, nu, cos_i, D_kpc, NH20, phase0, 0.0]
    for s in spots:
        s = list(s) + [0.0] * (7 - len(s))
        v += s[:7] + [0.0]
    return np.asarray(v, dtype=np.float64)


def log10T_of_kT(kT_keV):
    return float(np.log10(kT_keV / (_KB / _E / 1e3)))


# ------------------------------------------------------------------------------------------
# synthetic 4-D atmosphere table (BASELINE.json configs[1])
# ------------------------------------------------------------------------------------------
def atmosphere_axes():
    logT = linspace(5.1, 6.8, 35)
    logg = linspace(13.7, 14.7, 11)
    j = np.arange(67, dtype=np.float64)
    mu = 0.01 + 0.99 * (1.0 - np.cos(np.pi * j / 66.0)) / 2.0      # extra nodes near both ends
    mu[-1] = 1.0
    logx = linspace(-1.3, 2.0, 166)
    return logT, logg, mu, logx


def synthetic_atmosphere(seed=SEED0, amplitude=0.05):
    """log10 of Planck x limb darkening (1+2.06 mu)/3.06 x (1 + amplitude * P), P a seeded
    low-order Fourier perturbation with |P| <= 1.  Returns (logT, logg, mu, logx, values[35][11][67][166])."""
    logT, logg, mu, logx = atmosphere_axes()
    rng = np.random.Generator(np.random.PCG64(seed))
    nterm = 8
    ks = np.zeros((nterm, 4), dtype=np.int64)
    for n in range(nterm):
        while True:
            k = rng.integers(0, 3, size=4)
            if k.any():
                break
        ks[n] = k
    ph = rng.uniform(0.0, 2.0 * np.pi, size=nterm)
    a = rng.uniform(0.0, 1.0, size=nterm)
    a /= np.abs(a).sum()
    s = [(ax - ax[0]) / (ax[-1] - ax[0]) for ax in (logT, logg, mu, logx)]
    S = np.meshgrid(*s, indexing="ij")
    P = np.zeros(S[0].shape)
    for n in range(nterm):
        P += a[n] * np.cos(2.0 * np.pi * sum(ks[n, d] * S[d] for d in range(4)) + ph[n])
    kB = _KB / _E / 1e3
    h = _H / _E / 1e3
    c = _C * 100.0
    const = 2.0 * kB ** 3 / (h ** 3 * c ** 2)
    x = 10.0 ** logx
    planck = const * x ** 3 / np.expm1(x)
    limb = (1.0 + 2.06 * mu) / 3.06
    vals = np.log10(planck[None, None, None, :] * limb[None, None, :, None] * (1.0 + amplitude * P))
    return logT, logg, mu, logx, np.ascontiguousarray(vals)


def steep_limb_atmosphere(seed=SEED0, amplitude=0.05, a0=1.2):
    """Table for the interpolation-strategy study: same axes and Planck x perturbation
    as synthetic_atmosphere, but (i) the mu axis reaches 1e-6 with a few widely spaced nodes near 0 -- mu = 1e-6, 1e-3,
    1e-2, then 64 cosine-spaced nodes on [0.04, 1] ("mu in [1e-6, 1] with extra nodes near mu ~ 0, 1") --
    and (ii) the angular law is steep towards the limb, exp(-a(x) (1-mu)/(mu+0.03)) with a(x) = a0 / (1 + x/3), stronger in
    the soft band.  On such nodes a cubic Lagrange stencil applied to the INTENSITY overshoots below zero inside the first
    intervals of the mu axis (the paper's artefact); the NSX-H table itself is not available."""
    logT, logg, _, logx = atmosphere_axes()
    j = np.arange(64, dtype=np.float64)
    mu = np.concatenate([[1e-6, 1e-3, 1e-2], 0.04 + 0.96 * (1.0 - np.cos(np.pi * j / 63.0)) / 2.0])
    mu[-1] = 1.0
    _, _, mu0, _, base = synthetic_atmosphere(seed, amplitude)
    # strip synthetic_atmosphere's own limb law (its perturbation P is kept as laid out on the normalised axes)
    limb0 = (1.0 + 2.06 * mu0) / 3.06
    core = base - np.log10(limb0)[None, None, :, None]
    x = 10.0 ** logx
    a = a0 / (1.0 + x / 3.0)
    law = -a[None, :] * (1.0 - mu[:, None]) / (mu[:, None] + 0.03) / np.log(10.0)      # log10 of the angular law
    vals = core + law[None, None, :, :]
    return logT, logg, mu, logx, np.ascontiguousarray(vals)


def config_interp_test(which, n_cells=32, n_phase=128, n_energy=128):
    """The two atmosphere-interpolation test geometries of Table 3: one point-like hotspot of angular
    radius 0.01 rad at T = 1e6 K, M = 1.4, R_e = 12 km, 600 Hz, D = 150 pc; Test 1: theta_c = 1.983, i = 0.01;
    Test 2: theta_c = pi - 0.01, i = 0.964.  Energies: the paper's grid, Eq 50.  Strategy / domain are set by the caller."""
    theta_c, inc = {1: (1.983, 0.01), 2: (np.pi - 0.01, 0.964)}[which]
    cfg = _cfg(1, n_cells, n_cells, n_phase, max(192, 2 * n_phase), 2, 1)
    E = logspace(0.1, 5.215, n_energy)
    p = pack_params(1.4, 12.0, 600.0, np.cos(inc), 0.15, spots=[(theta_c, 0.0, 0.01, 6.0)])
    return dict(name="interp_test_%d" % which, cfg=cfg, energies=E, params=p[None, :], needs_table=True)


# ------------------------------------------------------------------------------------------
# configs
# ------------------------------------------------------------------------------------------
def _cfg(n_spots, n_theta, n_phi, n_phase, n_fp, emission, oblate):
    return dict(n_spots=n_spots, n_theta=n_theta, n_phi=n_phi, n_phase=n_phase, n_fp=n_fp,
                emission=emission, oblate=oblate)


def config_c1():
    """Tiny: sphere, closed-form blackbody, nothing random."""
    cfg = _cfg(1, 16, 16, 32, 192, 0, 0)
    E = logspace(0.3, 3.0, 8)
    p = pack_params(1.4, 12.0, 200.0, np.cos(np.deg2rad(60.0)), 0.2,
                    spots=[(np.deg2rad(40.0), 0.0, 0.2, log10T_of_kT(0.3))])
    return dict(name="C1", cfg=cfg, energies=E, params=p[None, :], needs_table=False)


def config_c2(n_cells=64, n_phase=128, n_energy=64, seed=SEED0 + 2):
    """Oblate star, one cap, cubic interpolation on all four table axes (strategy a)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    cos_i = rng.uniform(0.05, 0.95)
    cfg = _cfg(1, n_cells, n_cells, n_phase, max(192, 2 * n_phase), 1, 1)
    E = logspace(0.2, 12.0, n_energy)
    p = pack_params(1.4, 12.0, 300.0, cos_i, 0.15, spots=[(np.deg2rad(70.0), 0.0, 0.3, 6.1)])
    return dict(name="C2", cfg=cfg, energies=E, params=p[None, :], needs_table=True)


def _offset_point(theta_c, phi_c, dist, chi):
    """Point at angular distance `dist` from (theta_c, phi_c) at position angle chi (spherical trig)."""
    ct = np.cos(theta_c) * np.cos(dist) + np.sin(theta_c) * np.sin(dist) * np.cos(chi)
    theta = np.arccos(np.clip(ct, -1.0, 1.0))
    dphi = np.arctan2(np.sin(chi) * np.sin(dist) * np.sin(theta_c), np.cos(dist) - np.cos(theta_c) * ct)
    return float(theta), float(phi_c + dphi)


def config_c3(n_cells=128, n_phase=256, n_energy=128, seed=SEED0 + 3):
    """Two spots, one a seeded ring with cool temperature; mixed-order interpolation (strategy d)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    cos_i = rng.uniform(0.05, 0.95)
    th2 = rng.uniform(1.7, 2.3)
    ph2 = rng.uniform(0.0, 2.0 * np.pi)
    logT2 = rng.uniform(5.15, 5.30)
    chi = rng.uniform(0.0, 2.0 * np.pi)
    thm, phm = _offset_point(th2, ph2, 0.05, chi)
    cfg = _cfg(2, n_cells, n_cells, n_phase, max(192, 2 * n_phase), 2, 1)
    E = logspace(0.1, 5.215, n_energy)                       # the paper's grid, Eq 50
    p = pack_params(1.4, 12.0, 300.0, cos_i, 0.15,
                    spots=[(np.deg2rad(70.0), 0.0, 0.3, 6.1),
                           (th2, ph2, 0.4, logT2, thm, phm, 0.15)])
    return dict(name="C3", cfg=cfg, energies=E, params=p[None, :], needs_table=True)


def config_c4(n_cells=512, n_phase=512, n_energy=256, seed=SEED0 + 4):
    """Extreme geometry: tiny polar spot + huge equatorial spot, i = 85 deg, near-critical compactness."""
    rng = np.random.Generator(np.random.PCG64(seed))
    ph1 = rng.uniform(0.0, 2.0 * np.pi)
    cfg = _cfg(2, n_cells, n_cells, n_phase, max(192, 2 * n_phase), 2, 1)
    E = logspace(0.2, 12.0, n_energy)
    p = pack_params(2.0, 11.0, 600.0, np.cos(np.deg2rad(85.0)), 0.15,
                    spots=[(0.05, ph1, 0.02, 6.2), (1.75, 0.0, 1.2, 6.0)])
    return dict(name="C4", cfg=cfg, energies=E, params=p[None, :], needs_table=True)


def _outside_prior_support(M, Re_km, nu):
    """SURVEY.md 8(d) support of the C5 prior: a draw is rejected when u_pole = R_S / R(theta = 0) > 0.55 or
    beta_eq >= 0.5, with R(0) = R_e (1 + o2) of Eq 7-8 and beta_eq of Eq 18.
    This only defines which synthetic vectors exist; neither implementation calls it."""
    GM = M * _GMSUN
    Re = Re_km * 1.0e3
    Rs = 2.0 * GM / (_C * _C)
    x = GM / (_C * _C * Re)
    Ob2 = (2.0 * np.pi * nu) ** 2 * Re ** 3 / GM
    o2 = Ob2 * (-0.788 + 1.030 * x)
    R_pole = Re * (1.0 + o2)
    if not (R_pole > Rs and Re > Rs):
        return True
    u_pole = Rs / R_pole
    beta_eq = 2.0 * np.pi * nu * Re / (_C * np.sqrt(1.0 - Rs / Re))
    return bool(u_pole > 0.55 or beta_eq >= 0.5)


def c5_params(n_vec=1024, seed=SEED0 + 5):
    """Seeded parameter vectors from uniform priors; a vector is re-drawn while it lies outside the prior support
    of SURVEY.md 8(d) (u_pole > 0.55 or beta_eq >= 0.5; the raw priors reach unphysical u > 1), which keeps every
    vector inside the supported domain u <= 0.56 of reading R4."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = np.zeros((n_vec, N_STAR_PARAMS + 2 * N_SPOT_PARAMS))
    for b in range(n_vec):
        while True:
            M = rng.uniform(1.0, 3.0)
            Re = rng.uniform(8.0, 16.0)
            nu = rng.uniform(200.0, 700.0)
            cos_i = rng.uniform(0.0, 1.0)
            NH = rng.uniform(0.05, 3.0)
            sp = []
            for s in range(2):
                th = rng.uniform(0.1, np.pi - 0.1)
                ze = rng.uniform(0.05, 1.0)
                lt = rng.uniform(5.6, 6.5)
                ph = 0.0 if s == 0 else rng.uniform(0.0, 2.0 * np.pi)
                sp.append((th, ph, ze, lt))
            if not _outside_prior_support(M, Re, nu):
                break
        out[b] = pack_params(M, Re, nu, cos_i, 0.15, NH, 0.0, sp)
    return out


def config_c5(n_vec=1024, n_cells=256, n_phase=128, n_energy=300, seed=SEED0 + 5):
    cfg = _cfg(2, n_cells, n_cells, n_phase, max(192, 2 * n_phase), 2, 1)
    E = logspace(0.2, 12.0, n_energy)
    return dict(name="C5", cfg=cfg, energies=E, params=c5_params(n_vec, seed), needs_table=True)


def config_t():
    """North-star target: vector 0 of C5 evaluated alone (2 x 256x256 cells, 128 phases, 300 energies)."""
    c = config_c5(n_vec=1)
    c["name"] = "T"
    return c


# ------------------------------------------------------------------------------------------
# synthetic response (readings R15, R16)
# ------------------------------------------------------------------------------------------
def synthetic_response(energies, n_channel=1500, chan_width=0.01, sigma=0.1, seed=SEED0 + 5):
    """Banded RSP0[e][c] = w_e * A(E_e) * K[e][c]; K Gaussian (sigma keV) in channel-centre energy,
    truncated at |E_c - E_e| <= 5 sigma and renormalised to row sum 1.
    Returns dict(first_chan[int32 nE], rsp_band[nE][W], tau_ref[nE], n_channel, area[nE], w[nE])."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    b = rng.uniform(-1.0, 1.0, size=3)
    th = rng.uniform(0.0, 2.0 * np.pi, size=3)
    E = np.asarray(energies, dtype=np.float64)
    nE = len(E)
    area = 1800.0 * np.exp(-(np.log(E / 1.5)) ** 2 / (2 * 0.8 ** 2))
    ripple = sum(b[n] * np.sin((n + 1) * np.pi * np.log(E / 0.2) / np.log(60.0) + th[n]) for n in range(3))
    area = area * (1.0 + 0.1 * ripple)
    w = np.zeros(nE)
    w[1:-1] = 0.5 * (E[2:] - E[:-2])
    w[0] = 0.5 * (E[1] - E[0])
    w[-1] = 0.5 * (E[-1] - E[-2])
    centres = (np.arange(n_channel) + 0.5) * chan_width
    W = int(round(2 * 5 * sigma / chan_width)) + 1
    first = np.zeros(nE, dtype=np.int32)
    band = np.zeros((nE, W))
    for e in range(nE):
        c0 = int(np.floor((E[e] - 5 * sigma) / chan_width + 0.5))
        first[e] = c0
        ch = c0 + np.arange(W)
        ok = (ch >= 0) & (ch < n_channel)
        Ec = (ch + 0.5) * chan_width
        k = np.where(ok & (np.abs(Ec - E[e]) <= 5 * sigma + 1e-12), np.exp(-(Ec - E[e]) ** 2 / (2 * sigma ** 2)), 0.0)
        if k.sum() > 0:
            k = k / k.sum()
        band[e] = w[e] * area[e] * k
    tau_ref = 0.024 * E ** (-2.5)
    del centres
    return dict(first_chan=first, rsp_band=np.ascontiguousarray(band), tau_ref=tau_ref, n_channel=n_channel,
                area=area, w=w)


def synthetic_counts(n_phase, n_channel, total=1.0e6, bkg_frac=0.05, seed=SEED0 + 7):
    """Seeded Poisson counts of a smooth pulse x spectrum shape, for throughput runs (bench.py) where
    the data only have to look like an observation: a 1e6-count exposure with a
    single-peaked pulse and a thermal-looking channel spectrum, plus a flat background carrying
    `bkg_frac` of the source counts.  Returns (data[n_phase][n_channel], bkg[n_channel]).
    Parity tests draw their data from the ORACLE's model instead (tests/test_gpu_parity.py)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    k = np.arange(n_phase, dtype=np.float64) / n_phase
    Ec = (np.arange(n_channel, dtype=np.float64) + 0.5) * 0.01
    pulse = 1.0 + 0.35 * np.cos(2.0 * np.pi * (k - 0.2)) + 0.08 * np.cos(4.0 * np.pi * (k - 0.1))
    spec = Ec ** 2 * np.exp(-Ec / 0.35) * np.exp(-(0.25 / Ec) ** 2.5)
    m = pulse[:, None] * spec[None, :]
    m *= total / m.sum()
    bkg = np.full(n_channel, bkg_frac * total / (n_phase * n_channel))
    data = rng.poisson(m + bkg[None, :]).astype(np.float64)
    return data, bkg


def smooth_temperature_map(cfg, params, amplitude=0.05, seed=SEED0 + 9):
    """Seeded smooth per-cell temperature maps log10 T[B][n_spots][n_theta][n_phi] for ppm_evaluate_map: each spot's own
    log10 T (params) modulated over its mesh by +- `amplitude` dex of low-order structure (the paper's maps come from a
    physical surface-heating model, which is not available; the table's log T node spacing is 0.05 dex,
    so amplitude 0.05 spans 2-3 intervals per row and 0.3 about a dozen).  No NaN holes."""
    rng = np.random.Generator(np.random.PCG64(seed))
    B = params.shape[0]
    ns, nt, nphi = cfg["n_spots"], cfg["n_theta"], cfg["n_phi"]
    j = np.arange(nt, dtype=np.float64)[:, None] / nt
    m = np.arange(nphi, dtype=np.float64)[None, :] / nphi
    out = np.empty((B, ns, nt, nphi))
    for b in range(B):
        for s in range(ns):
            a, c = rng.uniform(0.0, 2.0 * np.pi, size=2)
            out[b, s] = params[b, 8 + 8 * s + 3] + amplitude * np.sin(2.0 * np.pi * j + a) * np.cos(2.0 * np.pi * m + c)
    return out
