"""Pins P24 for the reference sampler loop of the oracle (oracle/ppm_oracle.c O10; reading R26): the counter-based
generator against its published known-answer vectors and against cuRAND's host implementation of the same generator,
the uniform / normal variates against their distributions, and the Metropolis / replica-exchange rules against their
definitions on a chain whose likelihood the test computes itself with the (separately pinned) oracle pieces."""
import ctypes as C
import glob

import numpy as np
import pytest
from scipy import stats

import gen
import oracle as o


def test_p24_philox_known_answers():
    """Philox4x32-10, known-answer vectors of the Random123 distribution (Salmon, Moraes, Dror & Shaw 2011, kat_vectors)."""
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    for ctr, key, out in kat:
        assert tuple(int(x) for x in o.philox4x32_10(ctr, key)) == out


def test_p24_philox_equals_curand_host_generator():
    libs = sorted(glob.glob("/usr/local/cuda/lib64/libcurand.so*"))
    if not libs:
        pytest.skip("libcurand not found")
    lib = C.CDLL(libs[0])
    gen_h = C.c_void_p()
    if lib.curandCreateGeneratorHost(C.byref(gen_h), 161) != 0:          # CURAND_RNG_PSEUDO_PHILOX4_32_10
        pytest.skip("cuRAND host generator unavailable")
    for seed in (0, 0x299f31d0a4093822, 20251007):
        assert lib.curandSetPseudoRandomGeneratorSeed(gen_h, C.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(gen_h, C.c_ulonglong(0)) == 0
        out = np.zeros(16, dtype=np.uint32)
        assert lib.curandGenerate(gen_h, out.ctypes.data_as(C.POINTER(C.c_uint32)), C.c_size_t(16)) == 0
        key = (seed & 0xffffffff, seed >> 32)
        # cuRAND's host generator walks the subsequence word of the counter (ctr[2]) from block to block
        mine = np.concatenate([o.philox4x32_10((0, 0, i, 0), key) for i in range(4)])
        assert np.array_equal(out, mine)
    lib.curandDestroyGenerator(gen_h)


def test_p24_variates():
    n = 40000
    u, nm = [], []
    for t in range(n):
        u0, u1, n0, n1 = o.chain_random(20251007, t, 3, 0)
        u += [u0, u1]; nm += [n0, n1]
    u, nm = np.array(u), np.array(nm)
    assert 0.0 < u.min() and u.max() < 1.0
    assert stats.kstest(u, "uniform").pvalue > 1e-3 and stats.kstest(nm, "norm").pvalue > 1e-3
    assert abs(np.corrcoef(nm[0::2], nm[1::2])[0, 1]) < 0.02                 # the two Box-Muller normals are independent
    # different walkers / streams / seeds give different numbers; same counter gives the same
    a = o.chain_random(1, 5, 0, 0)
    assert a == o.chain_random(1, 5, 0, 0) and a != o.chain_random(1, 5, 1, 0) and a != o.chain_random(1, 5, 0, 1)
    assert a != o.chain_random(2, 5, 0, 0) and a != o.chain_random(1, 6, 0, 0)
    # Box-Muller written out
    u0, u1, n0, n1 = a
    assert abs(n0 - np.sqrt(-2 * np.log(u0)) * np.cos(2 * np.pi * u1)) < 1e-15
    assert abs(n1 - np.sqrt(-2 * np.log(u0)) * np.sin(2 * np.pi * u1)) < 1e-15


def _setup(W=4):
    conf = gen.config_c5(n_vec=W, n_cells=6, n_phase=8, n_energy=300, seed=gen.SEED0 + 91)
    cfg = conf["cfg"]
    E = conf["energies"]
    rsp = gen.synthetic_response(E)
    atm = o.Atmosphere(*gen.synthetic_atmosphere())

    def lnl(p, data, bkg, expo):
        f, st = o.evaluate(cfg, E, p, atm)
        if st:
            return -np.inf
        c = o.fold(f, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], p[5], rsp["n_channel"])
        return o.loglike(c, data, bkg, expo)
    f0, _ = o.evaluate(cfg, E, conf["params"][0], atm)
    c0 = o.fold(f0, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], conf["params"][0, 5], rsp["n_channel"])
    expo = 2e4 / (c0.sum() / 8)
    bkg = np.full(rsp["n_channel"], 0.05 * 2e4 / (8 * rsp["n_channel"]))
    data = np.random.default_rng(7).poisson(expo * c0 / 8 + bkg).astype(np.float64)
    P = conf["params"].shape[1]
    lo, hi, sig = np.full(P, -1e30), np.full(P, 1e30), np.zeros(P)
    for k, (a, b, s) in {0: (1.0, 3.0, 0.02), 1: (8.0, 16.0, 0.1), 3: (0.0, 1.0, 0.01), 8: (0.1, 3.0, 0.01), 10: (0.05, 1.0, 0.01),
                         11: (5.6, 6.5, 0.005)}.items():
        lo[k], hi[k], sig[k] = a, b, s
    return conf, cfg, E, rsp, atm, lnl, data, bkg, expo, lo, hi, sig


def test_p24_chain_follows_the_metropolis_and_exchange_rules():
    """The oracle's chain re-derived step by step in the test from its definition (reading R26), with the likelihood
    from the separately pinned evaluate / fold / loglike and the random numbers from the pinned generator."""
    W, n_steps, seed = 4, 6, 424242
    conf, cfg, E, rsp, atm, lnl, data, bkg, expo, lo, hi, sig = _setup(W)
    beta = np.array([1.0, 0.7, 0.4, 0.2])
    P = conf["params"].shape[1]
    params = np.ascontiguousarray(conf["params"].copy())
    ll = np.array([lnl(params[w], data, bkg, expo) for w in range(W)])
    p_ref, ll_ref = params.copy(), ll.copy()
    acc, swp, margin = o.chain_run(cfg, E, atm, rsp, data, bkg, expo, params, ll, lo, hi, sig, beta, seed, 0, n_steps)
    acc_ref, swp_ref = np.zeros(W, int), np.zeros(W, int)
    for t in range(n_steps):
        for w in range(W):
            prop = p_ref[w].copy()
            for k in range(P):
                if sig[k] > 0:
                    _, _, n0, n1 = o.chain_random(seed, t, w, k // 2)
                    prop[k] += sig[k] * (n1 if k % 2 else n0)
            if np.any(prop < lo) or np.any(prop > hi):
                continue
            lp = lnl(prop, data, bkg, expo)
            u0 = o.chain_random(seed, t, w, 0x10000)[0]
            if np.isfinite(lp) and np.log(u0) < beta[w] * (lp - ll_ref[w]):
                p_ref[w], ll_ref[w] = prop, lp
                acc_ref[w] += 1
        for i in range(t % 2, W - 1, 2):
            u0 = o.chain_random(seed, t, i, 0x10001)[0]
            if np.log(u0) < (beta[i] - beta[i + 1]) * (ll_ref[i + 1] - ll_ref[i]):
                p_ref[[i, i + 1]] = p_ref[[i + 1, i]]
                ll_ref[[i, i + 1]] = ll_ref[[i + 1, i]]
                swp_ref[[i, i + 1]] += 1
    assert margin > 1e-6                                                     # no decision of this run was a coin flip
    assert np.array_equal(acc, acc_ref) and np.array_equal(swp, swp_ref)
    assert np.allclose(params, p_ref, rtol=0, atol=1e-14) and np.allclose(ll, ll_ref, rtol=1e-12)
    assert acc.sum() > 0 and acc.sum() < W * n_steps                          # both outcomes occurred
    # restartable: two runs of 3 steps = one run of 6
    p2 = np.ascontiguousarray(conf["params"].copy())
    l2 = np.array([lnl(p2[w], data, bkg, expo) for w in range(W)])
    a1, s1, _ = o.chain_run(cfg, E, atm, rsp, data, bkg, expo, p2, l2, lo, hi, sig, beta, seed, 0, 3)
    a2, s2, _ = o.chain_run(cfg, E, atm, rsp, data, bkg, expo, p2, l2, lo, hi, sig, beta, seed, 3, 3)
    assert np.array_equal(p2, params) and np.array_equal(a1 + a2, acc) and np.array_equal(s1 + s2, swp)


def test_p24_box_prior_and_fixed_parameters():
    W = 2
    conf, cfg, E, rsp, atm, lnl, data, bkg, expo, lo, hi, sig = _setup(W)
    params = np.ascontiguousarray(conf["params"].copy())
    ll = np.array([lnl(params[w], data, bkg, expo) for w in range(W)])
    # a box so tight around the start that every proposal leaves it: nothing is ever accepted
    lo2, hi2 = lo.copy(), hi.copy()
    for k in np.flatnonzero(sig > 0):
        lo2[k], hi2[k] = params[:, k].min() - 1e-12, params[:, k].max() + 1e-12
    before = params.copy()
    acc, swp, _ = o.chain_run(cfg, E, atm, rsp, data, bkg, expo, params, ll, lo2, hi2, sig * 100, np.ones(W), 5, 0, 5)
    # (at equal temperatures an exchange has ratio 0 and always happens: the states only trade places)
    assert acc.sum() == 0 and np.array_equal(np.sort(params, axis=0), np.sort(before, axis=0))
    # parameters with sigma = 0 never move
    acc, _, _ = o.chain_run(cfg, E, atm, rsp, data, bkg, expo, params, ll, lo, hi, sig, np.ones(W), 5, 0, 4)
    fixed = sig == 0
    assert np.array_equal(np.sort(params[:, fixed], axis=0), np.sort(before[:, fixed], axis=0))
