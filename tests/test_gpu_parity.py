"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element on the same
seeded inputs.  Bar (BASELINE.json north_star): max relative error per (phase, energy) bin 1e-9."""
import numpy as np
import pytest

import gen
import oracle as o
from gpu_common import chi2_eq56, gpu_flux, make_ctx, max_rel_err, oracle_flux, report

pytestmark = pytest.mark.gpu
TOL = 1e-9


def test_c1_tiny_full():
    conf = gen.config_c1()
    g, st, _ = gpu_flux(conf)
    ref, so = oracle_flux(conf)
    assert st[0] == 0 and so == 0
    assert ref.max() > 0
    assert max_rel_err(g[0], ref) <= TOL


def test_c2_cubic_full():
    conf = gen.config_c2()
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


def test_c3_mixed_reduced_and_ragged():
    conf = gen.config_c3(n_cells=40, n_phase=37, n_energy=77)     # ragged tails in every dimension
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


def test_c3_full_size_every_phase():
    """C3 at BASELINE.json's full size, every (phase, energy) bin against the oracle, with the chi^2 of Eq 56-57."""
    conf = gen.config_c3()
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    err = max_rel_err(g[0], ref)
    report("c3_full", max_rel_err=err, chi2=chi2_eq56(g[0], ref), bins=int(ref.size))
    assert st[0] == 0 and err <= TOL


def test_c4_extreme_reduced():
    conf = gen.config_c4(n_cells=48, n_phase=64, n_energy=96)
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


def test_target_full_size_every_phase():
    """The north-star evaluation T (2 x 256x256 cells, 128 phases x 300 energies) in the launch configuration bench.py
    times: every bin of the flux against the oracle; folded counts and chi^2 (Eq 56-57) on the 128 x 1500 count plane."""
    import torch
    conf = gen.config_t()
    rsp = gen.synthetic_response(conf["energies"])
    ctx = make_ctx(conf)
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    p = torch.as_tensor(conf["params"], device="cuda")
    flux, st = ctx.evaluate(p)
    counts = ctx.fold_response(flux, p)
    g, c = flux.cpu().numpy()[0], counts.cpu().numpy()[0]
    ref, _ = oracle_flux(conf)
    cref = o.fold(ref, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][0, 5], rsp["n_channel"])
    err, cerr = max_rel_err(g, ref), max_rel_err(c, cref)
    report("T_full", max_rel_err=err, max_rel_err_counts=cerr, chi2_counts=chi2_eq56(c, cref), bins=int(ref.size))
    assert int(st[0]) == 0 and err <= TOL and cerr <= TOL
    assert chi2_eq56(c, cref) < 1e-9                    # Delta ln L ~ chi^2 / 2 at 1e6 counts: far below anything a sampler sees
    assert np.all(np.isfinite(g)) and np.all(g >= 0)


def test_batch_matches_single_and_status_codes():
    conf = gen.config_c5(n_vec=5, n_cells=24, n_phase=16, n_energy=40)
    P = conf["params"].copy()
    P[1, 1] = 4.0            # R_eq = 4 km: compactness out of domain -> status 1
    P[3, 10] = -0.5          # zeta < 0 -> status 4
    conf["params"] = P
    g, st, ctx = gpu_flux(conf)
    assert list(st) == [0, 1, 0, 4, 0]
    assert np.all(np.isnan(g[1])) and np.all(np.isnan(g[3]))
    for b in (0, 2, 4):
        ref, so = oracle_flux(conf, b)
        assert so == 0 and max_rel_err(g[b], ref) <= TOL
    assert o.evaluate(conf["cfg"], conf["energies"], P[1], None if conf["cfg"]["emission"] == 0 else
                      __import__("gpu_common").oracle_atm())[1] == 1
    # host-buffer entry point gives the same numbers
    gh, sh = ctx.evaluate_host(P)
    assert np.array_equal(sh, st) and np.array_equal(np.isnan(gh), np.isnan(g))
    assert np.array_equal(gh[[0, 2, 4]], g[[0, 2, 4]])             # deterministic: bit-identical re-run


def test_batch_larger_than_the_sub_batch():
    """B = 2 SB + 1: the context's scratch budget is shrunk (ppm_config.scratch_mb) so that the batch is processed in three
    sub-batches, the last one ragged -- the loop C5's 1024 vectors take.  Every vector against the oracle, through
    ppm_evaluate, ppm_evaluate_host and ppm_loglike_host (ln L against the oracle's fold + ln L)."""
    import torch
    conf = gen.config_c5(n_vec=5, n_cells=24, n_phase=16, n_energy=300, seed=gen.SEED0 + 31)
    rsp = gen.synthetic_response(conf["energies"])
    ctx = make_ctx(conf, scratch_mb=14)
    assert ctx.sub_batch() == 2
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    refs = [oracle_flux(conf, b)[0] for b in range(5)]
    p = torch.as_tensor(conf["params"], device="cuda")
    flux, st = ctx.evaluate(p)
    g = flux.cpu().numpy()
    assert np.all(st.cpu().numpy() == 0)
    errs = [max_rel_err(g[b], refs[b]) for b in range(5)]
    assert max(errs) <= TOL, errs
    gh, sh = ctx.evaluate_host(conf["params"])
    assert np.array_equal(gh, g) and np.all(sh == 0)
    cref = [o.fold(refs[b], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][b, 5], rsp["n_channel"])
            for b in range(5)]
    expo = 1e6 / (cref[0].sum() / 16)
    bkg = np.full(rsp["n_channel"], 0.05 * 1e6 / (16 * rsp["n_channel"]))
    data = np.random.default_rng(5).poisson(expo * cref[0] / 16 + bkg).astype(np.float64)
    llh, sth = ctx.loglike_host(conf["params"], torch.as_tensor(data, device="cuda"), torch.as_tensor(bkg, device="cuda"), expo)
    for b in range(5):
        assert abs(llh[b] - o.loglike(cref[b], data, bkg, expo)) <= 1e-9 * data.sum(), b
    # the same context with the whole batch in one sub-batch gives bit-identical numbers
    ctx1 = make_ctx(conf)
    assert ctx1.sub_batch() == 5
    g1 = ctx1.evaluate(p)[0].cpu().numpy()
    assert np.array_equal(g1, g)
    report("batch_2sb_plus_1", max_rel_err=max(errs), sub_batch=2, batch=5)


def test_occluded_spot_is_exactly_zero_and_empty_batch():
    import torch
    E = gen.logspace(0.3, 3.0, 8)
    cfg = dict(n_spots=1, n_theta=8, n_phi=8, n_phase=16, n_fp=192, emission=0, oblate=0)
    p = gen.pack_params(1.4, 12.0, 200.0, np.cos(0.3), 0.2, spots=[(2.9, 0.0, 0.1, 6.5)])     # pin P8 geometry
    conf = dict(cfg=cfg, energies=E, params=p[None, :])
    g, st, ctx = gpu_flux(conf)
    assert st[0] == 0 and np.all(g == 0.0)
    ref, _ = oracle_flux(conf)
    assert np.all(ref == 0.0)
    empty = torch.empty((0, ctx.P), dtype=torch.float64, device="cuda")
    f, s = ctx.evaluate(empty)
    assert f.shape[0] == 0
    import paper_2510_07764_b200 as ppm
    with pytest.raises(ppm.PPMError):
        ctx.evaluate(torch.zeros((2, ctx.P), dtype=torch.float64, device="cuda"))   # B > max_batch
    with pytest.raises(ppm.PPMError):
        ppm.PPM(dict(cfg, emission=2), E).evaluate(torch.zeros((1, ctx.P), dtype=torch.float64, device="cuda"))


def test_fold_and_loglike():
    import torch
    conf = gen.config_c5(n_vec=3, n_cells=16, n_phase=8, n_energy=300)
    rsp = gen.synthetic_response(conf["energies"])
    ctx = make_ctx(conf)
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    p = torch.as_tensor(conf["params"], device="cuda")
    flux, _ = ctx.evaluate(p)
    counts = ctx.fold_response(flux, p)
    fh = flux.cpu().numpy()
    ch = counts.cpu().numpy()
    cref = [o.fold(fh[b], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][b, 5], rsp["n_channel"])
            for b in range(3)]
    for b in range(3):
        assert max_rel_err(ch[b], cref[b]) <= 1e-13
    expo = 1e6 / (cref[0].sum() / 8)
    bkg = np.full(rsp["n_channel"], 0.05 * 1e6 / (8 * rsp["n_channel"]))
    rng = np.random.default_rng(11)
    data = rng.poisson(expo * cref[0] / 8 + bkg).astype(np.float64)
    ll = ctx.loglike(counts, torch.as_tensor(data, device="cuda"), torch.as_tensor(bkg, device="cuda"), expo)
    ll = ll.cpu().numpy()
    for b in range(3):
        ref = o.loglike(cref[b], data, bkg, expo)
        assert abs(ll[b] - ref) <= 1e-9 * data.sum(), (b, ll[b], ref)
    # host-buffer one-call path
    llh, sth = ctx.loglike_host(conf["params"], torch.as_tensor(data, device="cuda"),
                                torch.as_tensor(bkg, device="cuda"), expo)
    assert np.array_equal(llh, ll) and np.all(sth == 0)
    # -inf when the model is zero where data are not
    ll0 = ctx.loglike(torch.zeros_like(counts), torch.as_tensor(data, device="cuda"), None, expo).cpu().numpy()
    assert np.all(np.isneginf(ll0))


def test_c4_full_size_sampled_phases():
    """C4 at BASELINE.json's full size (2 x 512x512 cells, 512 phases x 256 energies, N_fp = 1024) in the launch
    configuration bench.py times; the oracle computes 16 of the 512 output phases (a full C4 oracle run is ~1 core-hour)."""
    conf = gen.config_c4()
    g, st, _ = gpu_flux(conf)
    sel = [5 + 33 * i for i in range(16)]                # 16 of 512 phases, one in every warp slot (k mod 16 all distinct)
    assert sorted(k % 16 for k in sel) == list(range(16)) and max(sel) < 512
    ref, _ = oracle_flux(conf, phase_sel=sel)
    assert st[0] == 0 and ref.max() > 0
    err = max_rel_err(g[0][sel], ref)
    report("c4_16_phases", max_rel_err=err, chi2=chi2_eq56(g[0][sel], ref), bins=int(ref.size))
    assert err <= TOL
    assert np.all(np.isfinite(g[0])) and np.all(g[0] >= 0)


def test_c5_loglike_parity_and_profile_counters():
    """S0-S7 end to end on C5 vectors (cells reduced to 64x64 per spot so that the oracle runs every phase):
    flux, folded counts and ln L against the oracle; data drawn from the ORACLE's model of vector 0."""
    import torch
    conf = gen.config_c5(n_vec=3, n_cells=64)
    rsp = gen.synthetic_response(conf["energies"])
    ctx = make_ctx(conf)
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    nph = conf["cfg"]["n_phase"]
    oflux = [oracle_flux(conf, b)[0] for b in range(3)]
    ocnt = [o.fold(oflux[b], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][b, 5], rsp["n_channel"])
            for b in range(3)]
    expo = 1e6 / (ocnt[0].sum() / nph)                               # 1e6 source counts from the reference vector
    bkg = np.full(rsp["n_channel"], 0.05 * 1e6 / (nph * rsp["n_channel"]))
    data = np.random.default_rng(gen.SEED0 + 55).poisson(expo * ocnt[0] / nph + bkg).astype(np.float64)
    p = torch.as_tensor(conf["params"], device="cuda")
    ctx.profile_enable(True)
    flux, status = ctx.evaluate(p)
    counts = ctx.fold_response(flux, p)
    ll = ctx.loglike(counts, torch.as_tensor(data, device="cuda"), torch.as_tensor(bkg, device="cuda"), expo)
    prof, triples = ctx.profile_read()
    ctx.profile_enable(False)
    assert np.all(status.cpu().numpy() == 0)
    fh, ch, llh = flux.cpu().numpy(), counts.cpu().numpy(), ll.cpu().numpy()
    for b in range(3):
        assert max_rel_err(fh[b], oflux[b]) <= TOL
        assert max_rel_err(ch[b], ocnt[b]) <= TOL
        ref = o.loglike(ocnt[b], data, bkg, expo)
        assert abs(llh[b] - ref) <= 1e-9 * data.sum(), (b, llh[b], ref)
    assert llh[0] > llh[1] and llh[0] > llh[2]                        # the data were drawn from vector 0
    # the device-side unit counter: accumulated (cell, phase) pairs x energies; bounded by active cells x phases x energies
    assert prof["cells"][1] == 1 and prof["cells"][0] > 0
    nE = len(conf["energies"])
    n_act = sum(int(ctx.debug_mask(b).sum()) for b in range(3))
    assert 0 < triples <= n_act * nph * nE and triples % nE == 0


@pytest.mark.parametrize("emission", [1, 2])
def test_table_edges_below_and_above_the_logx_axis(emission):
    """Energies from far below to far above the table's log10(E/kT) range: coordinates clamp at both ends (reading
    R13b), the window of intervals holds the first and the last interval of the axis (linear in strategy d, shifted
    cubic stencil in strategy a), and 333 energies span two energy tiles with a ragged tail."""
    conf = gen.config_c2(n_cells=20, n_phase=19, n_energy=333)
    conf["cfg"] = dict(conf["cfg"], emission=emission)
    conf["energies"] = gen.logspace(0.002, 40.0, 333)
    conf["params"] = conf["params"].copy()
    conf["params"][0, 8 + 3] = 6.45                                  # hot spot: x = E/kT reaches below 10^-1.3
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


@pytest.mark.parametrize("emission", [1, 2])
def test_table_edges_on_the_uniform_energy_path(emission):
    """The same sweep across both ends of the logx axis with 320 energies = one full tile of a log-uniform grid: the cell
    kernel steps its coordinate from energy group to energy group (EnergyCoord, UNI = true) through the clamped-low,
    the plain and the clamped-high energy loops."""
    conf = gen.config_c2(n_cells=20, n_phase=19, n_energy=320)
    conf["cfg"] = dict(conf["cfg"], emission=emission)
    conf["energies"] = gen.logspace(0.002, 40.0, 320)
    conf["params"] = conf["params"].copy()
    conf["params"][0, 8 + 3] = 6.45
    g, st, ctx = gpu_flux(conf)
    assert ctx.uniform_energy()
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


def test_uniform_and_general_energy_paths():
    """Log-uniform grids (all BASELINE.json configs) take the stepped-coordinate kernel, with a ragged last energy group
    (120 = 3 x 32 + 24 energies); a grid that is uniform in E (an instrument's channel grid) is not log-uniform and takes
    the kernel that holds one coordinate per energy.  Both against the oracle."""
    for name in ("c2", "c3", "c4"):
        small = getattr(gen, "config_" + name)(n_cells=8, n_phase=8)
        assert make_ctx(small).uniform_energy(), name
    assert make_ctx(gen.config_t()).uniform_energy()
    conf = gen.config_c3(n_cells=24, n_phase=20, n_energy=120)
    g, st, ctx = gpu_flux(conf)
    assert ctx.uniform_energy()
    ref, _ = oracle_flux(conf)
    e_uni = max_rel_err(g[0], ref)
    lin = dict(conf, energies=np.linspace(0.25, 9.0, 120))
    g2, st2, ctx2 = gpu_flux(lin)
    assert not ctx2.uniform_energy()
    ref2, _ = oracle_flux(lin)
    e_gen = max_rel_err(g2[0], ref2)
    # two full energy tiles (640 = 2 x 320 energies) on the stepped coordinate: each tile anchors its own lanes
    two = gen.config_c2(n_cells=12, n_phase=9, n_energy=640)
    two["energies"] = gen.logspace(0.1, 15.0, 640)
    g3, st3, ctx3 = gpu_flux(two)
    assert ctx3.uniform_energy()
    ref3, _ = oracle_flux(two)
    e_two = max_rel_err(g3[0], ref3)
    report("energy_paths", uniform=e_uni, general=e_gen, two_tiles=e_two)
    assert st[0] == 0 and st2[0] == 0 and st3[0] == 0 and e_uni <= TOL and e_gen <= TOL and e_two <= TOL


def test_narrow_energy_band_uses_a_small_window():
    """8 energies in a narrow band: the per-pair window is a few intervals (NPL = 1 variant of the cell kernel)."""
    conf = gen.config_c3(n_cells=24, n_phase=16, n_energy=8)
    conf["energies"] = gen.logspace(1.0, 1.6, 8)
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL


TOL32 = 1e-4      # north_star: "1e-4 on any FP32-interpolation path"


@pytest.mark.parametrize("name,kw", [("c2", {}), ("c3", dict(n_cells=40, n_phase=37, n_energy=77)),
                                     ("c4", dict(n_cells=48, n_phase=64, n_energy=96))])
def test_fp32_interpolation_path(name, kw):
    conf = getattr(gen, "config_" + name)(**kw)
    g, st, _ = gpu_flux(conf, precision=1)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0
    err = max_rel_err(g[0], ref)
    assert err <= TOL32, err
    g64, _, _ = gpu_flux(conf)
    assert np.array_equal(g[0] == 0, g64[0] == 0)


def test_fp32_path_target_full_size_and_edges():
    conf = gen.config_t()
    g, st, _ = gpu_flux(conf, precision=1)
    sel = [3, 77]
    ref, _ = oracle_flux(conf, phase_sel=sel)
    assert st[0] == 0 and max_rel_err(g[0][sel], ref) <= TOL32
    # both ends of the logx axis, two energy tiles, strategy a
    conf = gen.config_c2(n_cells=20, n_phase=19, n_energy=333)
    conf["energies"] = gen.logspace(0.002, 40.0, 333)
    conf["params"] = conf["params"].copy()
    conf["params"][0, 8 + 3] = 6.45
    g, st, _ = gpu_flux(conf, precision=1)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL32


def test_strategy_c_cubic_with_linear_edges():
    """emission = 3 (strategy c): C3's cool ring sits in the first logT intervals (linear there),
    the hot cap in the interior (cubic in logT and logg)."""
    conf = gen.config_c3(n_cells=32, n_phase=24, n_energy=70)
    conf["cfg"] = dict(conf["cfg"], emission=3)
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and max_rel_err(g[0], ref) <= TOL
    conf2 = dict(conf, cfg=dict(conf["cfg"], emission=2))
    g2, _, _ = gpu_flux(conf2)
    assert np.max(np.abs(g2[0] - g[0]) / np.maximum(g[0], 1e-300)) > 1e-7      # and it differs from strategy d


def test_terms_that_underflow_take_the_guarded_loop():
    """A table whose high-x half lies 300 decades lower: there F_p T^3 10^v < 2^-1000, the exponent add of the fast
    2^y would wrap; such pairs must take the guarded loop and contribute (numerically) nothing, and the bins the
    oracle resolves as normal numbers must still agree to 1e-9."""
    import oracle as orc
    import paper_2510_07764_b200 as ppm
    import torch
    logT, logg, mu, logx, vals = gen.synthetic_atmosphere()
    vals = vals.copy()
    vals[..., 120:] -= 300.0
    conf = gen.config_c3(n_cells=24, n_phase=16, n_energy=60)
    ctx = ppm.PPM(conf["cfg"], conf["energies"], max_batch=1)
    ctx.load_atmosphere(logT, logg, mu, logx, vals)
    flux, st = ctx.evaluate(torch.as_tensor(conf["params"], device="cuda"))
    g = flux.cpu().numpy()[0]
    ref, _ = orc.evaluate(conf["cfg"], conf["energies"], conf["params"][0], orc.Atmosphere(logT, logg, mu, logx, vals))
    assert int(st[0]) == 0 and np.all(np.isfinite(g)) and np.all(g >= 0)
    big = ref > 1e-250
    assert big.any() and (~big).any()
    assert np.max(np.abs(g[big] - ref[big]) / ref[big]) <= TOL
    assert np.all(g[~big] <= 1e-240)


@pytest.mark.parametrize("emission,precision", [(0, 0), (2, 0), (2, 1)])
def test_healpix_mesh(emission, precision):
    """mesh = 1: the paper's HEALPix ring mesh over the whole surface (Eq 24-29), two spots (cap + ring with an omitted
    cap) selected by the centre-in mask; masks bit-exact, flux at the path's tolerance."""
    nside = 24
    conf = gen.config_c3(n_cells=8, n_phase=21, n_energy=40)
    conf["cfg"] = dict(conf["cfg"], n_theta=4 * nside - 1, n_phi=4 * nside, mesh=1, emission=emission)
    if emission == 0:
        conf["params"] = conf["params"].copy()
        conf["params"][0, [8 + 3, 16 + 3]] = 6.4
    g, st, ctx = gpu_flux(conf, precision=precision)
    ref, so = oracle_flux(conf)
    assert st[0] == 0 and so == 0 and ref.max() > 0
    assert max_rel_err(g[0], ref) <= (TOL32 if precision else TOL)
    mask = ctx.debug_mask()
    nt = 4 * nside - 1
    for s in range(2):
        sp = o.spot(*conf["params"][0, 8 + 8 * s: 8 + 8 * s + 7])
        assert np.array_equal(mask[s * nt:(s + 1) * nt], o.spot_mask_healpix(sp, nside))
    rows = ctx.debug_rows()
    assert np.allclose(rows[:nt, 11], np.pi / (3 * nside ** 2), rtol=1e-15)      # equal-area pixels


@pytest.mark.parametrize("beaming", [1, 2])
def test_blackbody_beaming_laws(beaming):
    """cos^2 / sin^2 beaming on the OS1-like set-up: M = 1.4, R = 12 km, D = 200 pc, kT = 0.35 keV,
    monochromatic 1 keV, extended spot zeta = 1 rad, oblate star at 400 Hz."""
    E = np.array([1.0])
    cfg = dict(n_spots=1, n_theta=40, n_phi=40, n_phase=32, n_fp=192, emission=0, oblate=1, beaming=beaming)
    p = gen.pack_params(1.4, 12.0, 400.0, np.cos(np.deg2rad(70.0)), 0.2,
                        spots=[(np.deg2rad(50.0), 0.0, 1.0, gen.log10T_of_kT(0.35))])
    conf = dict(cfg=cfg, energies=E, params=p[None, :])
    g, st, _ = gpu_flux(conf)
    ref, _ = oracle_flux(conf)
    assert st[0] == 0 and ref.max() > 0 and max_rel_err(g[0], ref) <= TOL


@pytest.mark.parametrize("name,kw,emission", [("c1", {}, 0), ("c3", dict(n_cells=40, n_phase=37, n_energy=77), 2),
                                              ("c4", dict(n_cells=48, n_phase=64, n_energy=96), 2),
                                              ("c2", dict(n_cells=32, n_phase=32, n_energy=64), 1)])
def test_phase_interp_order3(name, kw, emission):
    """phase_interp = 3 (reading R11b): 4-point Lagrange Interp of Eq 46 with periodic wrap, linear next to
    hidden template entries (C3's ring and C4's big spot are partly occulted), against the oracle's orc_phase_interp;
    a coarse template (N_fp = 64) makes the order matter."""
    conf = getattr(gen, "config_" + name)(**kw)
    conf["cfg"] = dict(conf["cfg"], phase_interp=3, n_fp=64)
    g, st, _ = gpu_flux(conf)
    ref, so = oracle_flux(conf)
    assert st[0] == 0 and so == 0 and ref.max() > 0
    err = max_rel_err(g[0], ref)
    assert err <= TOL, err
    lin, _ = oracle_flux(dict(conf, cfg=dict(conf["cfg"], phase_interp=1)))
    assert np.max(np.abs(lin - ref)) > 1e-6 * ref.max()                    # and it is not the linear rule
    report("phase_interp3_" + name, max_rel_err=err)
    if emission == 2:                                                      # the FP32-interpolation path shares step A
        g32, _, _ = gpu_flux(conf, precision=1)
        assert max_rel_err(g32[0], ref) <= TOL32


def test_bench_line_contract():
    """bench.py prints one JSON line with the keys the driver and the judge read (small workload, no CPU baseline)."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "C2", "--batch", "2", "--steps", "3",
                          "--warmup", "3", "--no-cpu-baseline"], capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["steps"] == 3 and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["gpu_launches"] >= 3 * 10 and "workload" in d["config"]
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s"
    assert abs(r["algorithmic_frac"] - r["algorithmic_achieved"] / r["peak"]) < 1e-12
    if r["frac"] is None:                          # no ncu capture for this (workload, batch, kernel source): nothing is made up
        assert r["achieved"] is None and r["traffic"] is None and r["executed_flop_per_unit"] is None
    else:
        assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["frac"] <= 1.0
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 2 * 16 * 8 and e["d2h_bytes_per_step"] == 2 * 12


def test_random_prior_vectors_sweep():
    """48 seeded vectors from C5's priors (M 1-3, R 8-16 km, 200-700 Hz, any inclination, spot radii up to 1 rad) at
    reduced grid size, every bin against the oracle: FP64 path at 1e-9, FP32-interpolation path at 1e-4."""
    import torch
    conf = gen.config_c5(n_vec=48, n_cells=16, n_phase=20, n_energy=40, seed=gen.SEED0 + 77)
    refs = [oracle_flux(conf, b) for b in range(48)]
    for precision, tol in ((0, TOL), (1, TOL32)):
        ctx = make_ctx(conf, precision=precision)
        flux, status = ctx.evaluate(torch.as_tensor(conf["params"], device="cuda"))
        g, st = flux.cpu().numpy(), status.cpu().numpy()
        for b, (ref, so) in enumerate(refs):
            assert st[b] == so == 0
            assert max_rel_err(g[b], ref) <= tol, (precision, b)


def test_step_is_capturable_in_a_cuda_graph():
    """The device-pointer calls neither synchronise nor allocate after their first use: evaluate + fold + ln L can be
    captured into a CUDA graph on the context's stream and replayed, bit-identical to the eager run."""
    import torch
    conf = gen.config_c5(n_vec=2, n_cells=24, n_phase=16, n_energy=300)
    rsp = gen.synthetic_response(conf["energies"])
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = make_ctx(conf)
        ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
        p = torch.as_tensor(conf["params"], device="cuda")
        d_h, b_h = gen.synthetic_counts(16, rsp["n_channel"])
        data, bkg = torch.as_tensor(d_h, device="cuda"), torch.as_tensor(b_h, device="cuda")
        flux = torch.empty((2, 16, 300), dtype=torch.float64, device="cuda")
        st = torch.empty((2,), dtype=torch.int32, device="cuda")
        counts = torch.empty((2, 16, rsp["n_channel"]), dtype=torch.float64, device="cuda")
        ll = torch.empty((2,), dtype=torch.float64, device="cuda")

        def step():
            ctx.evaluate(p, flux, st)
            ctx.fold_response(flux, p, counts)
            ctx.loglike(counts, data, bkg, 1.0e6, ll)
        step()
        torch.cuda.synchronize()
        ref = ll.clone()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            step()
        ll.zero_()
        flux.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(ll, ref) and bool(torch.isfinite(ll).all()) and float(flux.max()) > 0
