"""-m gpu: the device-resident sampler loop (ppm_chain_*, reading R26) against the oracle's reference chain
on the same seeded inputs: same proposals (same counter-based generator on both sides), same accept / exchange
decisions, states and ln L within the path's tolerance; graph replay is deterministic and restartable."""
import numpy as np
import pytest

import gen
import oracle as o
from gpu_common import atmosphere, oracle_atm, report

pytestmark = pytest.mark.gpu


def _setup(W, n_cells=6, n_phase=8):
    import torch
    import paper_2510_07764_b200 as ppm
    conf = gen.config_c5(n_vec=W, n_cells=n_cells, n_phase=n_phase, n_energy=300, seed=gen.SEED0 + 91)
    cfg, E = conf["cfg"], conf["energies"]
    rsp = gen.synthetic_response(E)
    f0, _ = o.evaluate(cfg, E, conf["params"][0], oracle_atm())
    c0 = o.fold(f0, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][0, 5], rsp["n_channel"])
    expo = 2e4 / (c0.sum() / n_phase)
    bkg = np.full(rsp["n_channel"], 0.05 * 2e4 / (n_phase * rsp["n_channel"]))
    data = np.random.default_rng(7).poisson(expo * c0 / n_phase + bkg).astype(np.float64)
    P = conf["params"].shape[1]
    lo, hi, sig = np.full(P, -1e30), np.full(P, 1e30), np.zeros(P)
    for k, (a, b, s) in {0: (1.0, 3.0, 0.02), 1: (8.0, 16.0, 0.1), 3: (0.0, 1.0, 0.01), 8: (0.1, 3.0, 0.01), 10: (0.05, 1.0, 0.01),
                         11: (5.6, 6.5, 0.005)}.items():
        lo[k], hi[k], sig[k] = a, b, s
    ctx = ppm.PPM(cfg, E, max_batch=W)
    ctx.load_atmosphere(*atmosphere())
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    d_dev, b_dev = torch.as_tensor(data, device="cuda"), torch.as_tensor(bkg, device="cuda")
    return conf, cfg, E, rsp, expo, bkg, data, lo, hi, sig, ctx, d_dev, b_dev


def test_chain_matches_the_reference_chain():
    W, n_steps, seed = 4, 8, 424242
    conf, cfg, E, rsp, expo, bkg, data, lo, hi, sig, ctx, d_dev, b_dev = _setup(W)
    beta = np.array([1.0, 0.7, 0.4, 0.2])
    ctx.chain_create(conf["params"], lo, hi, sig, d_dev, b_dev, expo, beta=beta, seed=seed)
    p0, ll0, acc0, swp0, t0 = ctx.chain_read()
    assert t0 == 0 and acc0.sum() == 0 and np.array_equal(p0, conf["params"])
    # reference: start from the oracle's own ln L of the same states
    params = np.ascontiguousarray(conf["params"].copy())
    ll = np.empty(W)
    for w in range(W):
        f, st = o.evaluate(cfg, E, params[w], oracle_atm())
        assert st == 0
        c = o.fold(f, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], params[w, 5], rsp["n_channel"])
        ll[w] = o.loglike(c, data, bkg, expo)
    assert np.max(np.abs(ll0 - ll)) <= 1e-9 * data.sum()
    acc, swp, margin = o.chain_run(cfg, E, oracle_atm(), rsp, data, bkg, expo, params, ll, lo, hi, sig, beta, seed, 0, n_steps)
    assert margin > 1e-5                                 # every decision of the reference run is robust against 1e-9 in ln L
    ctx.chain_run(n_steps)
    p, l, a, s, t = ctx.chain_read()
    assert t == n_steps
    assert np.array_equal(a, acc) and np.array_equal(s, swp)                     # same decisions (integer work: exact)
    assert acc.sum() > 0 and swp.sum() > 0
    assert np.max(np.abs(p - params)) <= 1e-12                                   # same proposals (libm-level differences)
    assert np.max(np.abs(l - ll)) <= 1e-9 * data.sum()
    report("chain_vs_reference", steps=n_steps, walkers=W, accepted=int(acc.sum()), swapped=int(swp.sum()),
           max_abs_dlnL=float(np.max(np.abs(l - ll))), margin=float(margin))
    # the chain's ln L is the likelihood of its states (fresh evaluation through the host-buffer entry)
    ll_h, st_h = ctx.loglike_host(p, d_dev, b_dev, expo)
    assert np.all(st_h == 0) and np.array_equal(ll_h, l)


def test_chain_is_deterministic_restartable_and_respects_the_prior():
    W, seed = 6, 99
    conf, cfg, E, rsp, expo, bkg, data, lo, hi, sig, ctx, d_dev, b_dev = _setup(W)
    ctx.chain_create(conf["params"], lo, hi, sig, d_dev, b_dev, expo, seed=seed)
    ctx.chain_run(10)
    r1 = ctx.chain_read()
    ctx.chain_create(conf["params"], lo, hi, sig, d_dev, b_dev, expo, seed=seed)
    ctx.chain_run(4)
    ctx.chain_run(6)
    r2 = ctx.chain_read()
    for x, y in zip(r1, r2):
        assert np.array_equal(x, y)
    assert r1[4] == 10 and r1[2].sum() > 0
    moving = sig > 0
    assert np.all(r1[0][:, moving] >= lo[moving]) and np.all(r1[0][:, moving] <= hi[moving])
    assert np.array_equal(np.sort(r1[0][:, ~moving], axis=0), np.sort(conf["params"][:, ~moving], axis=0))
    # another seed gives another chain
    ctx.chain_create(conf["params"], lo, hi, sig, d_dev, b_dev, expo, seed=seed + 1)
    ctx.chain_run(10)
    assert not np.array_equal(ctx.chain_read()[0], r1[0])
    # a box that no proposal can stay in: nothing is accepted, ln L untouched
    lo2, hi2 = lo.copy(), hi.copy()
    for k in np.flatnonzero(moving):
        lo2[k], hi2[k] = conf["params"][:, k].min() - 1e-12, conf["params"][:, k].max() + 1e-12
    ctx.chain_create(conf["params"], lo2, hi2, sig * 100, d_dev, b_dev, expo, seed=seed)
    before = ctx.chain_read()
    ctx.chain_run(5)
    after = ctx.chain_read()
    assert after[2].sum() == 0 and np.array_equal(np.sort(after[1]), np.sort(before[1]))
