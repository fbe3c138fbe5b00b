"""-m gpu: each step S0-S3 of the CUDA path against the oracle's own routine for that step
(row scalars, cell mask, psi/lag lookup, ring template), read back through ppm_debug_*."""
import numpy as np
import pytest

import gen
import oracle as o
from gpu_common import gpu_flux

pytestmark = pytest.mark.gpu


def _small(conf, n_cells, n_phase, n_energy):
    conf = dict(conf)
    conf["cfg"] = dict(conf["cfg"], n_theta=n_cells, n_phi=n_cells, n_phase=n_phase, n_fp=max(192, 2 * n_phase))
    conf["energies"] = gen.logspace(conf["energies"][0], conf["energies"][-1], n_energy)
    return conf


def _spots(conf):
    p = conf["params"][0]
    return [o.spot(*p[8 + 8 * s: 8 + 8 * s + 7]) for s in range(conf["cfg"]["n_spots"])]


@pytest.mark.parametrize("name", ["c2", "c3", "c4"])
def test_rows_and_mask(name):
    conf = _small(getattr(gen, "config_" + name)(), 48, 32, 16)
    conf["cfg"]["n_phi"] = 41                                   # ragged azimuth count
    _, status, ctx = gpu_flux(conf)
    assert status[0] == 0
    rows = ctx.debug_rows()
    mask = ctx.debug_mask()
    p = conf["params"][0]
    st = o.star(p[0], p[1], p[2], conf["cfg"]["oblate"])
    nt, nphi = conf["cfg"]["n_theta"], conf["cfg"]["n_phi"]
    for s, sp in enumerate(_spots(conf)):
        bx = o.spot_box(sp, nt, nphi)
        m_ref = o.spot_mask(sp, nt, nphi)
        # the inequality is decided in separately rounded multiplies / adds on both sides, but cos() comes from two math
        # libraries: a cell within a few ulp of the boundary would be undefined -- none of the seeded configs has one
        assert o.spot_mask_margin(sp, nt, nphi) > 1e-13
        assert np.array_equal(mask[s * nt:(s + 1) * nt], m_ref)                # bit-exact index work
        for j in range(nt):
            r = o.row(st, bx, nt, j)
            ref = np.array([r.theta, r.dcos, r.R_cm, r.u, r.f, r.coseta, r.sineta, r.beta, r.gamma, r.log10g,
                            r.c_dt_cm, r.dcos * bx.dphi, np.pi / 2 + abs(np.arctan(r.f))])
            got = rows[s * nt + j, :13]
            scale = np.maximum(np.abs(ref), 1e-300)
            tol = np.full(13, 1e-13)
            tol[10] = 1e-9                                       # c dt(R): cancellation R_e - R, absolute 1e-9 R
            err = np.abs(got - ref) / scale
            err[10] = abs(got[10] - ref[10]) / r.R_cm
            err[4] = abs(got[4] - ref[4])                        # f can be ~0
            err[6] = abs(got[6] - ref[6])
            assert np.all(err <= tol), (name, s, j, err)
            assert rows[s * nt + j, 14] == m_ref[j].sum()


@pytest.mark.parametrize("name", ["c2", "c4"])
def test_lookup_against_quadrature(name):
    conf = _small(getattr(gen, "config_" + name)(), 24, 32, 8)
    _, _, ctx = gpu_flux(conf)
    rows = ctx.debug_rows()
    rng = np.random.default_rng(5)
    worst = np.zeros(3)
    for r in range(0, rows.shape[0], 5):
        if rows[r, 14] == 0:
            continue
        u, amax, psimax = rows[r, 3], rows[r, 12], rows[r, 13]
        al = np.concatenate([rng.uniform(1e-6, amax, 24), [1e-7, 1e-3, np.pi / 2 - 1e-9, np.pi / 2, amax]])
        al = al[al <= amax]
        psi, dpsi, lag = ctx.debug_lookup(r, al)
        psi_o = np.array([o.psi(u, a) for a in al])
        dpsi_o = np.array([o.dpsi_dalpha(u, a) for a in al])
        lag_o = np.array([o.lag_total_over_R(u, a) for a in al])       # R_e := R, i.e. without c dt(R)
        worst = np.maximum(worst, [np.max(np.abs(psi - psi_o) / psi_o), np.max(np.abs(dpsi - dpsi_o) / dpsi_o),
                                   np.max(np.abs(lag - lag_o))])
        assert abs(psimax - o.psi(u, amax)) <= 1e-13 * psimax
    assert worst[0] <= 1e-13 and worst[1] <= 2e-11 and worst[2] <= 1e-13, worst


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_template_against_oracle(name):
    conf = getattr(gen, "config_" + name)()
    if name != "c1":
        conf = _small(conf, 24, 64, 8)
    _, _, ctx = gpu_flux(conf)
    tm = ctx.debug_template()
    rows = ctx.debug_rows()
    p = conf["params"][0]
    st = o.star(p[0], p[1], p[2], conf["cfg"]["oblate"])
    nt, nphi, nfp = conf["cfg"]["n_theta"], conf["cfg"]["n_phi"], ctx.n_fp
    D_cm = p[4] * 1e3 * o.PC_CM
    checked = 0
    for s, sp in enumerate(_spots(conf)):
        bx = o.spot_box(sp, nt, nphi)
        for j in range(0, nt, 3):
            r = s * nt + j
            if rows[r, 14] == 0:
                continue
            rw = o.row(st, bx, nt, j)
            ref = o.template(st, rw, p[3], D_cm, rw.dcos * bx.dphi, nfp)
            assert bool(rows[r, 15]) == ref["visible"]
            if ref["margin"] < 1e-9:
                continue                                           # visibility flip guard (reading R22)
            for q, key in enumerate(("F", "z", "phio", "mu")):
                a, b = tm[r, q], ref[key]
                assert np.array_equal(a == 0, b == 0), (name, r, key)
                nz = b != 0
                if nz.any():
                    tol = 1e-13 if key in ("z", "phio") else 3e-11
                    # phi_o is a phase in cycles of order 1 whose first entry can sit next to 0: its error
                    # scale is absolute (what Eq 45-46 consume); everything else is compared relatively
                    scale = np.maximum(np.abs(b[nz]), 1.0) if key == "phio" else np.abs(b[nz])
                    assert np.max(np.abs(a[nz] - b[nz]) / scale) <= tol, (name, r, key)
            checked += 1
    assert checked > 0
