"""ctypes front end of oracle/ppm_oracle.c (the CPU oracle).  TEST INFRASTRUCTURE.

Argument marshalling only; every number is computed by the C file.  Citations are in the C
source next to each function.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_u8p = C.POINTER(C.c_uint8)


class Star(C.Structure):
    _fields_ = [("GM", C.c_double), ("Rs_cm", C.c_double), ("Re_cm", C.c_double), ("x", C.c_double),
                ("Obar2", C.c_double), ("o2", C.c_double), ("g0_cgs", C.c_double), ("nu", C.c_double),
                ("oblate", C.c_int)]


class Row(C.Structure):
    _fields_ = [("theta", C.c_double), ("dcos", C.c_double), ("R_cm", C.c_double), ("u", C.c_double),
                ("f", C.c_double), ("coseta", C.c_double), ("sineta", C.c_double), ("beta", C.c_double),
                ("gamma", C.c_double), ("log10g", C.c_double), ("c_dt_cm", C.c_double)]


class Spot(C.Structure):
    _fields_ = [("theta_c", C.c_double), ("phi_c", C.c_double), ("zeta", C.c_double), ("log10T", C.c_double),
                ("theta_m", C.c_double), ("phi_m", C.c_double), ("zeta_m", C.c_double)]


class Box(C.Structure):
    _fields_ = [("theta_lo", C.c_double), ("theta_hi", C.c_double), ("W", C.c_double), ("dphi", C.c_double)]


class _Atm(C.Structure):
    _fields_ = [("nT", C.c_int32), ("ng", C.c_int32), ("nmu", C.c_int32), ("nx", C.c_int32),
                ("logT", _dp), ("logg", _dp), ("mu", _dp), ("logx", _dp), ("values", _dp)]


class _Config(C.Structure):
    _fields_ = [("n_spots", C.c_int32), ("n_theta", C.c_int32), ("n_phi", C.c_int32), ("n_phase", C.c_int32),
                ("n_fp", C.c_int32), ("n_energy", C.c_int32), ("emission", C.c_int32), ("oblate", C.c_int32),
                ("mesh", C.c_int32), ("beaming", C.c_int32), ("phase_interp", C.c_int32), ("interp_domain", C.c_int32)]


def _sig(name, res, args):
    f = getattr(_lib, name)
    f.restype = res
    f.argtypes = args
    return f


_const = _sig("orc_const", C.c_double, [C.c_int])
_psi = _sig("orc_psi", C.c_double, [C.c_double, C.c_double])
_dpsi = _sig("orc_dpsi_dalpha", C.c_double, [C.c_double, C.c_double])
_dpsi_an = _sig("orc_dpsi_dalpha_analytic", C.c_double, [C.c_double, C.c_double])
_lag = _sig("orc_lag", C.c_double, [C.c_double, C.c_double])
_rho = _sig("orc_rho", C.c_double, [C.c_double, C.c_double])
_lag_tot_R = _sig("orc_lag_total_over_R", C.c_double, [C.c_double, C.c_double])
_lag_tot = _sig("orc_lag_total", C.c_double, [C.c_double] * 4)
_alpha_of_psi = _sig("orc_alpha_of_psi", C.c_int, [C.c_double, C.c_double, C.c_double, _dp])
_gl_rule = _sig("orc_gl_rule", None, [C.POINTER(C.c_int), _dp, _dp])
_star_init = _sig("orc_star_init", None, [C.c_double, C.c_double, C.c_double, C.c_int, C.POINTER(Star)])
_spot_box = _sig("orc_spot_box", None, [C.POINTER(Spot), C.c_int, C.c_int, C.POINTER(Box)])
_row_init = _sig("orc_row_init", None, [C.POINTER(Star), C.POINTER(Box), C.c_int, C.c_int, C.POINTER(Row)])
_spot_mask = _sig("orc_spot_mask", C.c_int, [C.POINTER(Spot), C.c_int, C.c_int, _u8p])
_spot_mask_margin = _sig("orc_spot_mask_margin", C.c_double, [C.POINTER(Spot), C.c_int, C.c_int])
_template = _sig("orc_template", C.c_int,
                 [C.POINTER(Star), C.POINTER(Row), C.c_double, C.c_double, C.c_double, C.c_int,
                  _dp, _dp, _dp, _dp, _u8p, _dp, _dp, _dp])
_interp1 = _sig("orc_interp1", C.c_double, [_dp, _dp, C.c_int, C.c_double, C.c_int])
_interp4 = _sig("orc_interp4", C.c_double, [C.POINTER(_Atm), C.c_int] + [C.c_double] * 4)
_intensity = _sig("orc_intensity", C.c_double, [C.c_int, C.POINTER(_Atm)] + [C.c_double] * 4)
_interp4_dom = _sig("orc_interp4_domain", C.c_double, [C.POINTER(_Atm), C.c_int, C.c_int] + [C.c_double] * 4)
_intensity_dom = _sig("orc_intensity_domain", C.c_double, [C.c_int, C.c_int, C.POINTER(_Atm)] + [C.c_double] * 4)
_phase_interp = _sig("orc_phase_interp", C.c_double, [C.c_int, _dp, _dp, _dp, C.c_double, C.c_int, C.POINTER(C.c_int)])
_evaluate = _sig("orc_evaluate", C.c_int,
                 [C.POINTER(_Config), _dp, _dp, C.POINTER(_Atm), _ip, C.c_int, _dp, _dp])
_evaluate_map = _sig("orc_evaluate_map", C.c_int,
                     [C.POINTER(_Config), _dp, _dp, C.POINTER(_Atm), _dp, _ip, C.c_int, _dp, _dp])
_fold = _sig("orc_fold", None, [_dp, C.c_int, C.c_int, C.c_int, C.c_int, _ip, _dp, _dp, C.c_double, _dp])
_loglike = _sig("orc_loglike", C.c_double, [_dp, _dp, _dp, C.c_int, C.c_int, C.c_double])
_hp_ring = _sig("orc_healpix_ring", None, [C.c_int, C.c_int, _dp, C.POINTER(C.c_int), _dp, _dp])
_hp_mask = _sig("orc_spot_mask_healpix", C.c_int, [C.POINTER(Spot), C.c_int, _u8p])
_hp_row = _sig("orc_row_init_healpix", None, [C.POINTER(Star), C.c_int, C.c_int, C.POINTER(Row)])
_chi2 = _sig("orc_chi2", C.c_double, [_dp, _dp, C.c_size_t])
_u32p = C.POINTER(C.c_uint32)
_i64p = C.POINTER(C.c_int64)
_philox = _sig("orc_philox4x32_10", None, [_u32p, _u32p, _u32p])
_chain_random = _sig("orc_chain_random", None, [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _dp, _dp, _dp, _dp])
_chain_run = _sig("orc_chain_run", None,
                  [C.POINTER(_Config), _dp, C.POINTER(_Atm), C.c_int, C.c_int, _ip, _dp, _dp, _dp, _dp, C.c_double, C.c_int,
                   _dp, _dp, _dp, _dp, C.c_uint64, C.c_uint64, C.c_int, _dp, _dp, _i64p, _i64p, _dp])
_nthreads = _sig("orc_num_threads", C.c_int, [])
_set_nthreads = _sig("orc_set_num_threads", None, [C.c_int])

AX_LINEAR, AX_CUBIC_SHIFT, AX_CUBIC_LINEDGE, AX_MU_PROTECTED = 0, 1, 2, 3


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp)


# ---- constants -------------------------------------------------------------------------
C_CM_S = _const(0)
H_KEV_S = _const(1)
KB_KEV_K = _const(2)
GM_SUN = _const(3)
PC_CM = _const(4)
TWO_OVER_H3C2 = _const(5)


# ---- geodesic integrals ----------------------------------------------------------------
def psi(u, alpha):
    return _psi(u, alpha)


def dpsi_dalpha(u, alpha):
    return _dpsi(u, alpha)


def dpsi_dalpha_analytic(u, alpha):
    return _dpsi_an(u, alpha)


def lag(u, alpha):
    """G(u, alpha) = c dt_p / R for an outgoing ray (Eq 15/35)."""
    return _lag(u, alpha)


def rho(u, alpha):
    return _rho(u, alpha)


def lag_total_over_R(u, alpha):
    """c Delta t / R with R_e := R (Eq 15 outgoing, Eq 17 inward)."""
    return _lag_tot_R(u, alpha)


def lag_total(Re, Rs, R, alpha):
    return _lag_tot(Re, Rs, R, alpha)


def alpha_of_psi(u, psi_t, alpha_max):
    out = C.c_double()
    rc = _alpha_of_psi(u, psi_t, alpha_max, C.byref(out))
    return None if rc else out.value


def lensing_factor(u, alpha):
    """d cos(alpha) / d cos(psi) = sin(alpha) / (sin(psi) dpsi/dalpha)."""
    ps = _psi(u, alpha)
    return np.sin(alpha) / (np.sin(ps) * _dpsi(u, alpha))


def gl_rule():
    n = C.c_int()
    x = np.zeros(64)
    w = np.zeros(64)
    _gl_rule(C.byref(n), _p(x), _p(w))
    return x[:n.value].copy(), w[:n.value].copy()


# ---- star / rows / cells ---------------------------------------------------------------
def star(M, Re_km, nu, oblate=True):
    s = Star()
    _star_init(M, Re_km, nu, int(bool(oblate)), C.byref(s))
    return s


def spot(theta_c, phi_c, zeta, log10T, theta_m=0.0, phi_m=0.0, zeta_m=0.0):
    return Spot(theta_c, phi_c, zeta, log10T, theta_m, phi_m, zeta_m)


def spot_box(sp, n_theta, n_phi):
    b = Box()
    _spot_box(C.byref(sp), n_theta, n_phi, C.byref(b))
    return b


def row(st, bx, n_theta, j):
    r = Row()
    _row_init(C.byref(st), C.byref(bx), n_theta, j, C.byref(r))
    return r


def spot_mask(sp, n_theta, n_phi):
    m = np.zeros((n_theta, n_phi), dtype=np.uint8)
    _spot_mask(C.byref(sp), n_theta, n_phi, m.ctypes.data_as(_u8p))
    return m


def spot_mask_margin(sp, n_theta, n_phi):
    """min over the box grid's cells of the distance to a mask decision boundary (in cos of the separation)."""
    return _spot_mask_margin(C.byref(sp), n_theta, n_phi)


def healpix_ring(nside, i):
    """Ring i = 1 .. 4 nside - 1 of the HEALPix ring scheme (Eq 24-29): -> (cos theta, npix, phi of pixel 1, dphi)."""
    z, p0, dp = C.c_double(), C.c_double(), C.c_double()
    n = C.c_int()
    _hp_ring(int(nside), int(i), C.byref(z), C.byref(n), C.byref(p0), C.byref(dp))
    return z.value, n.value, p0.value, dp.value


def spot_mask_healpix(sp, nside):
    m = np.zeros((4 * nside - 1, 4 * nside), dtype=np.uint8)
    _hp_mask(C.byref(sp), int(nside), m.ctypes.data_as(_u8p))
    return m


def row_healpix(st, nside, j):
    r = Row()
    _hp_row(C.byref(st), int(nside), int(j), C.byref(r))
    return r


def template(st, rw, cosi, D_cm, dOmega, n_fp):
    """Ring template (O3+O4).  Returns dict(F, z, phio, mu, vis, margin, alpha, lf, visible)."""
    F, z, po, mu, al, lf = (np.zeros(n_fp + 1) for _ in range(6))
    vis = np.zeros(n_fp + 1, dtype=np.uint8)
    mg = C.c_double()
    ok = _template(C.byref(st), C.byref(rw), cosi, D_cm, dOmega, n_fp, _p(F), _p(z), _p(po), _p(mu),
                   vis.ctypes.data_as(_u8p), C.byref(mg), _p(al), _p(lf))
    return dict(F=F, z=z, phio=po, mu=mu, vis=vis, margin=mg.value, alpha=al, lf=lf, visible=bool(ok))


# ---- atmosphere ------------------------------------------------------------------------
class Atmosphere:
    """Holds the 4-D table log10(I/T^3)[logT][logg][mu][logx] (C order) for the oracle."""

    def __init__(self, logT, logg, mu, logx, values):
        self.logT, self.logg, self.mu, self.logx = map(_f64, (logT, logg, mu, logx))
        self.values = _f64(values)
        assert self.values.shape == (len(self.logT), len(self.logg), len(self.mu), len(self.logx))
        self.c = _Atm(len(self.logT), len(self.logg), len(self.mu), len(self.logx),
                      _p(self.logT), _p(self.logg), _p(self.mu), _p(self.logx), _p(self.values))


def interp1(ax, y, x, rule):
    ax, y = _f64(ax), _f64(y)
    return _interp1(_p(ax), _p(y), len(ax), float(x), int(rule))


def interp4(atm, strategy, logT, logg, mu, logx):
    return _interp4(C.byref(atm.c), int(strategy), logT, logg, mu, logx)


def intensity(emission, atm, log10T, log10g, Ep, mu, domain=0):
    ap = C.byref(atm.c) if atm is not None else None
    if domain:
        return _intensity_dom(int(emission), int(domain), ap, log10T, log10g, Ep, mu)
    return _intensity(int(emission), ap, log10T, log10g, Ep, mu)


def interp4_domain(atm, strategy, domain, logT, logg, mu, logx):
    return _interp4_dom(C.byref(atm.c), int(strategy), int(domain), logT, logg, mu, logx)


def phase_interp(phio, F, y, phi_p, order):
    """Interp of Eq 46 on a periodic template (n_fp + 1 entries): -> (value, bracket index)."""
    phio, F, y = _f64(phio), _f64(F), _f64(y)
    i = C.c_int()
    v = _phase_interp(len(phio) - 1, _p(phio), _p(F), _p(y), float(phi_p), int(order), C.byref(i))
    return v, i.value


# ---- evaluation ------------------------------------------------------------------------
def evaluate(cfg, energies, params, atm=None, phase_sel=None, return_margin=False, tmap=None):
    """cfg: dict(n_spots,n_theta,n_phi,n_phase,n_fp,n_energy?,emission,oblate).  params: 1-D vector.
    Returns (flux[n_k][n_energy], status[, margin])."""
    energies = _f64(energies)
    params = _f64(params)
    c = _Config(cfg["n_spots"], cfg["n_theta"], cfg["n_phi"], cfg["n_phase"], cfg["n_fp"],
                len(energies), cfg["emission"], int(cfg.get("oblate", 1)), int(cfg.get("mesh", 0)),
                int(cfg.get("beaming", 0)), int(cfg.get("phase_interp", 0)), int(cfg.get("interp_domain", 0)))
    assert params.shape == (8 + 8 * cfg["n_spots"],)
    if cfg["emission"] != 0:
        assert atm is not None
    if phase_sel is not None:
        sel = np.ascontiguousarray(phase_sel, dtype=np.int32)
        nk, selp = len(sel), sel.ctypes.data_as(_ip)
    else:
        nk, selp = cfg["n_phase"], None
    flux = np.zeros((nk, len(energies)))
    mg = C.c_double()
    ap = C.byref(atm.c) if atm is not None else None
    if tmap is not None:                       # per-cell log10 T map [n_spots][n_theta][n_phi], NaN = not emitting
        tmap = _f64(tmap)
        assert tmap.shape == (cfg["n_spots"], cfg["n_theta"], cfg["n_phi"])
        status = _evaluate_map(C.byref(c), _p(energies), _p(params), ap, _p(tmap), selp, nk, _p(flux), C.byref(mg))
    else:
        status = _evaluate(C.byref(c), _p(energies), _p(params), ap, selp, nk, _p(flux), C.byref(mg))
    if return_margin:
        return flux, status, mg.value
    return flux, status


def fold(flux, first_chan, rsp_band, tau_ref, NH20, n_channel):
    flux = _f64(flux)
    rsp_band = _f64(rsp_band)
    tau_ref = _f64(tau_ref)
    fc = np.ascontiguousarray(first_chan, dtype=np.int32)
    n_phase, n_energy = flux.shape
    band_w = rsp_band.shape[1]
    counts = np.zeros((n_phase, n_channel))
    _fold(_p(flux), n_phase, n_energy, n_channel, band_w, fc.ctypes.data_as(_ip), _p(rsp_band), _p(tau_ref),
          float(NH20), _p(counts))
    return counts


def loglike(counts, data, bkg, exposure_s):
    counts, data = _f64(counts), _f64(data)
    n_phase, n_channel = counts.shape
    b = _f64(bkg) if bkg is not None else None
    return _loglike(_p(counts), _p(data), _p(b) if b is not None else None, n_phase, n_channel, float(exposure_s))


def chi2(m, d):
    m, d = _f64(m).ravel(), _f64(d).ravel()
    return _chi2(_p(m), _p(d), m.size)


def philox4x32_10(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    _philox(c.ctypes.data_as(_u32p), k.ctypes.data_as(_u32p), out.ctypes.data_as(_u32p))
    return out


def chain_random(seed, t, walker, stream):
    """-> (u0, u1, n0, n1) of counter (t, walker, stream) under key `seed` (reading R26)."""
    v = [C.c_double() for _ in range(4)]
    _chain_random(int(seed), int(t), int(walker), int(stream), *[C.byref(x) for x in v])
    return tuple(x.value for x in v)


def chain_run(cfg, energies, atm, rsp, data, bkg, exposure_s, params, loglike, lo, hi, sigma, beta, seed, t0, n_steps):
    """Reference sampler loop (O10).  params [W][P] and loglike [W] are updated in place.
    -> (accepted [W], swapped [W], margin)."""
    energies = _f64(energies)
    c = _Config(cfg["n_spots"], cfg["n_theta"], cfg["n_phi"], cfg["n_phase"], cfg["n_fp"], len(energies), cfg["emission"],
                int(cfg.get("oblate", 1)), int(cfg.get("mesh", 0)), int(cfg.get("beaming", 0)),
                int(cfg.get("phase_interp", 0)), int(cfg.get("interp_domain", 0)))
    assert params.dtype == np.float64 and params.flags.c_contiguous and loglike.dtype == np.float64
    W = params.shape[0]
    fc = np.ascontiguousarray(rsp["first_chan"], dtype=np.int32)
    band, tau = _f64(rsp["rsp_band"]), _f64(rsp["tau_ref"])
    data, bkg = _f64(data), _f64(bkg)
    lo, hi, sigma, beta = _f64(lo), _f64(hi), _f64(sigma), _f64(beta)
    acc = np.zeros(W, dtype=np.int64)
    swp = np.zeros(W, dtype=np.int64)
    mg = C.c_double()
    _chain_run(C.byref(c), _p(energies), C.byref(atm.c) if atm is not None else None, int(rsp["n_channel"]), band.shape[1],
               fc.ctypes.data_as(_ip), _p(band), _p(tau), _p(data), _p(bkg), float(exposure_s), W, _p(lo), _p(hi), _p(sigma),
               _p(beta), int(seed), int(t0), int(n_steps), _p(params), _p(loglike), acc.ctypes.data_as(_i64p),
               swp.ctypes.data_as(_i64p), C.byref(mg))
    return acc, swp, mg.value


def num_threads():
    return _nthreads()


def set_num_threads(n):
    _set_nthreads(int(n))
