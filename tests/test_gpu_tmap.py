"""-m gpu: per-cell temperature maps (ppm_evaluate_map, reading R24) against the oracle."""
import numpy as np
import pytest

import gen
import oracle as o
from gpu_common import make_ctx, max_rel_err, oracle_atm

pytestmark = pytest.mark.gpu
TOL = 1e-9


def _gpu_map(conf, tmap, ctx=None):
    import torch
    ctx = ctx or make_ctx(conf)
    p = torch.as_tensor(conf["params"], dtype=torch.float64, device="cuda").contiguous()
    tm = torch.as_tensor(np.ascontiguousarray(tmap), dtype=torch.float64, device="cuda")
    flux, status = ctx.evaluate_map(p, tm)
    torch.cuda.synchronize()
    return flux.cpu().numpy(), status.cpu().numpy(), ctx


def _smooth_map(cfg, rng, lo=5.7, hi=6.5, holes=0.1):
    """Seeded smooth map over each spot's mesh spanning many log T intervals (node spacing 0.05), with NaN holes."""
    ns, nt, nphi = cfg["n_spots"], cfg["n_theta"], cfg["n_phi"]
    j = np.arange(nt)[:, None] / nt
    m = np.arange(nphi)[None, :] / nphi
    out = np.empty((ns, nt, nphi))
    for s in range(ns):
        a, b, c = rng.uniform(0, 2 * np.pi, 3)
        f = 0.5 + 0.25 * np.sin(2 * np.pi * j + a) * np.cos(2 * np.pi * m + b) + 0.25 * np.sin(4 * np.pi * (j + m) + c)
        out[s] = lo + (hi - lo) * f
    out[rng.random(out.shape) < holes] = np.nan
    return out


@pytest.mark.parametrize("mesh", [0, 1])
def test_smooth_map_matches_oracle(mesh):
    conf = gen.config_c3(n_cells=36, n_phase=21, n_energy=70)
    if mesh:
        nside = 20
        conf["cfg"] = dict(conf["cfg"], n_theta=4 * nside - 1, n_phi=4 * nside, mesh=1)
    rng = np.random.default_rng(31 + mesh)
    tmap = _smooth_map(conf["cfg"], rng)
    g, st, ctx = _gpu_map(conf, tmap[None])
    ref, so = o.evaluate(conf["cfg"], conf["energies"], conf["params"][0], oracle_atm(), tmap=tmap)
    assert st[0] == 0 and so == 0 and ref.max() > 0
    assert max_rel_err(g[0], ref) <= TOL
    # the mask of emitting cells = geometric mask AND finite map entry (bit-exact index work)
    mask = ctx.debug_mask()
    nt = conf["cfg"]["n_theta"]
    for s in range(2):
        sp = o.spot(*conf["params"][0, 8 + 8 * s: 8 + 8 * s + 7])
        geo = o.spot_mask_healpix(sp, conf["cfg"]["n_phi"] // 4) if mesh else o.spot_mask(sp, nt, conf["cfg"]["n_phi"])
        assert np.array_equal(mask[s * nt:(s + 1) * nt].astype(bool), geo.astype(bool) & np.isfinite(tmap[s]))


def test_constant_map_equals_uniform_evaluate_and_batch_of_maps():
    import torch
    conf = gen.config_c5(n_vec=3, n_cells=20, n_phase=12, n_energy=40)
    ctx = make_ctx(conf)
    p = torch.as_tensor(conf["params"], device="cuda")
    f_uni, _ = ctx.evaluate(p)
    cfg = conf["cfg"]
    tmap = np.empty((3, 2, cfg["n_theta"], cfg["n_phi"]))
    for b in range(3):
        tmap[b, 0], tmap[b, 1] = conf["params"][b, 8 + 3], conf["params"][b, 16 + 3]
    g, st, _ = _gpu_map(conf, tmap, ctx)
    assert np.all(st == 0)
    fu = f_uni.cpu().numpy()
    for b in range(3):
        assert max_rel_err(g[b], fu[b]) <= 1e-12
    # temperatures below / above the table's log T axis clamp on the axis but keep their own kT and T^3 (reading R13b)
    tmap2 = tmap.copy()
    tmap2[:, 0] = 5.02
    tmap2[:, 1] = 6.87
    g2, st2, _ = _gpu_map(conf, tmap2, ctx)
    ref, _ = o.evaluate(cfg, conf["energies"], conf["params"][1], oracle_atm(), tmap=tmap2[1])
    assert max_rel_err(g2[1], ref) <= TOL
    # all-NaN map: nothing emits
    g3, st3, _ = _gpu_map(conf, np.full_like(tmap, np.nan), ctx)
    assert np.all(st3 == 0) and np.all(g3 == 0.0)


def test_map_mode_needs_table_emission_and_fp64():
    import paper_2510_07764_b200 as ppm
    import torch
    conf = gen.config_c1()                                                      # closed-form blackbody: no table to map onto
    ctx = make_ctx(conf)
    cfg = conf["cfg"]
    tm = torch.full((1, cfg["n_spots"], cfg["n_theta"], cfg["n_phi"]), 6.0, dtype=torch.float64, device="cuda")
    with pytest.raises(ppm.PPMError):
        ctx.evaluate_map(torch.as_tensor(conf["params"], device="cuda"), tm)
    conf = gen.config_c2(n_cells=8, n_phase=8, n_energy=8)
    ctx = make_ctx(conf, precision=1)
    tm = torch.full((1, 1, 8, 8), 6.0, dtype=torch.float64, device="cuda")
    with pytest.raises(ppm.PPMError):
        ctx.evaluate_map(torch.as_tensor(conf["params"], device="cuda"), tm)


@pytest.mark.parametrize("emission", [1, 3, 4])
@pytest.mark.parametrize("mesh,n_energy", [(0, 70), (1, 70), (0, 300)])
def test_cubic_in_log_T_strategies_match_oracle(emission, mesh, n_energy):
    """Temperature maps under strategies a, c and b: cubic Lagrange in log T -- four node slices per
    interval, stencil shifted inward (a, b) or linear (c) in the first / last log T interval -- on smooth seeded maps that
    reach both ends of the log T axis; 300 energies run as two energy tiles of five energies per lane."""
    conf = gen.config_c3(n_cells=28, n_phase=21, n_energy=n_energy)
    conf["cfg"] = dict(conf["cfg"], emission=emission)
    if n_energy == 300:
        conf["energies"] = gen.logspace(0.2, 12.0, 300)
    if mesh:
        nside = 16
        conf["cfg"] = dict(conf["cfg"], n_theta=4 * nside - 1, n_phi=4 * nside, mesh=1)
    rng = np.random.default_rng(300 + 10 * emission + mesh)
    tmap = _smooth_map(conf["cfg"], rng, lo=5.12, hi=6.78, holes=0.08)
    g, st, ctx = _gpu_map(conf, tmap[None])
    ref, so = o.evaluate(conf["cfg"], conf["energies"], conf["params"][0], oracle_atm(), tmap=tmap)
    assert st[0] == 0 and so == 0 and ref.max() > 0
    assert max_rel_err(g[0], ref) <= TOL


def test_cubic_map_constant_equals_uniform_and_window_status():
    """A constant map reproduces the uniform-temperature evaluate of the same strategy; temperatures inside the axis's
    clamp range but outside the axis still work (own kT, clamped table coordinate); a row whose window exceeds the four
    slice buffers gives PPM_STATUS_MAP_WINDOW and a NaN flux for that vector only."""
    import torch
    conf = gen.config_c5(n_vec=2, n_cells=20, n_phase=12, n_energy=40)
    conf["cfg"] = dict(conf["cfg"], emission=1)
    ctx = make_ctx(conf)
    p = torch.as_tensor(conf["params"], device="cuda")
    f_uni, _ = ctx.evaluate(p)
    cfg = conf["cfg"]
    tmap = np.empty((2, 2, cfg["n_theta"], cfg["n_phi"]))
    for b in range(2):
        tmap[b, 0], tmap[b, 1] = conf["params"][b, 8 + 3], conf["params"][b, 16 + 3]
    g, st, _ = _gpu_map(conf, tmap, ctx)
    fu = f_uni.cpu().numpy()
    assert np.all(st == 0)
    for b in range(2):
        assert max_rel_err(g[b], fu[b]) <= 1e-11
    tmap2 = tmap.copy()
    tmap2[:, 0] = 5.02                                                           # just outside the axis at both ends
    tmap2[:, 1] = 6.87
    g2, st2, _ = _gpu_map(conf, tmap2, ctx)
    ref, _ = o.evaluate(cfg, conf["energies"], conf["params"][1], oracle_atm(), tmap=tmap2[1])
    assert np.all(st2 == 0) and max_rel_err(g2[1], ref) <= TOL
    tmap3 = tmap.copy()
    tmap3[1, 0, 3:6, ::2] = 9.0                                                  # 2.2 dex above the axis: the last interval's window
                                                                                 # runs from column 0 to its own top, > 130 columns
    g3, st3, _ = _gpu_map(conf, tmap3, ctx)
    assert st3[0] == 0 and max_rel_err(g3[0], fu[0]) <= 1e-11
    assert st3[1] == 8 and np.all(np.isnan(g3[1]))


@pytest.mark.parametrize("mesh", [0, 1])
def test_fp32_map_matches_oracle(mesh):
    """precision = 1 (FP32 interpolation and exponential, tolerance 1e-4 per bin: the paper's production precision) with a
    temperature map: reference exponents per (row, log T interval); smooth seeded maps over many intervals, both meshes."""
    conf = gen.config_c3(n_cells=36, n_phase=21, n_energy=70)
    if mesh:
        nside = 20
        conf["cfg"] = dict(conf["cfg"], n_theta=4 * nside - 1, n_phi=4 * nside, mesh=1)
    rng = np.random.default_rng(131 + mesh)
    tmap = _smooth_map(conf["cfg"], rng)
    g, st, _ = _gpu_map(conf, tmap[None], make_ctx(conf, precision=1))
    ref, so = o.evaluate(conf["cfg"], conf["energies"], conf["params"][0], oracle_atm(), tmap=tmap)
    assert st[0] == 0 and so == 0 and ref.max() > 0
    assert max_rel_err(g[0], ref) <= 1e-4


def test_fp32_map_target_size_edges_and_status():
    """FP32 maps at the T size (300 energies, clamped upper energies) against the FP64 map kernel (itself at 1e-9 of the
    oracle); temperatures slightly outside the axis work, an interval spanning more than 0.5 dex gives the status bit."""
    conf = gen.config_t()
    cfg = conf["cfg"]
    tmap = gen.smooth_temperature_map(cfg, conf["params"], 0.3)
    g64, st64, _ = _gpu_map(conf, tmap)
    g32, st32, ctx32 = _gpu_map(conf, tmap, make_ctx(conf, precision=1))
    assert st64[0] == 0 and st32[0] == 0 and max_rel_err(g32[0], g64[0]) <= 1e-4
    t2 = np.array(tmap, copy=True)
    t2[0, 0, 100:140, ::3] = 4.85                                                # 0.25 dex below the axis: still inside FP32's range
    g64b, _, _ = _gpu_map(conf, t2)
    g32b, st32b, _ = _gpu_map(conf, t2, ctx32)
    assert st32b[0] == 0 and max_rel_err(g32b[0], g64b[0]) <= 1e-4
    t3 = np.array(tmap, copy=True)
    t3[0, 1, 50:60, ::2] = 7.6                                                   # 0.8 dex above the axis
    g32c, st32c, _ = _gpu_map(conf, t3, ctx32)
    assert st32c[0] == 8 and np.all(np.isnan(g32c[0]))


def test_rows_split_between_the_windowed_and_the_full_width_launch():
    """Temperatures far outside the table's log T axis keep their own kT (reading R13b), which moves the row's logx
    window by tens of columns: such rows do not fit the windowed slice buffers and go to the full-width launch, the
    others to the windowed one; the two launches add into the same tiles."""
    conf = gen.config_c3(n_cells=30, n_phase=32, n_energy=64)
    cfg = conf["cfg"]
    rng = np.random.default_rng(77)
    tmap = _smooth_map(cfg, rng, lo=5.9, hi=6.3, holes=0.05)
    tmap[0, 4:9, ::3] = 4.2                       # 0.9 dex below the axis: window wider than the buffers
    tmap[1, 20:24, 1::2] = 7.6                    # 0.8 dex above
    g, st, _ = _gpu_map(conf, tmap[None])
    ref, so = o.evaluate(cfg, conf["energies"], conf["params"][0], oracle_atm(), tmap=tmap)
    assert st[0] == 0 and so == 0 and max_rel_err(g[0], ref) <= TOL
