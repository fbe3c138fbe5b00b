"""-m gpu: the interpolation-strategy study of PAPER.md:492-561 on the CUDA path: the four strategies
a, b, c, d with the table interpolation applied to the intensity (interp_domain = 1, reading R13g) on the two Table 3
geometries, against the oracle.

Parity metric for interp_domain = 1 (DESIGN reading R22b): under strategy a the terms of a bin have both signs and the
bin can cancel to (nearly) zero, so |gpu - oracle| is taken relative to the bin's sum of |terms|, which the oracle gives
as 2 F_b - F_a (strategy b sums the positive terms only).  Bar: 1e-9 of that."""
import numpy as np
import pytest

import gen
import oracle as o
from gpu_common import max_rel_err, report

pytestmark = pytest.mark.gpu
TOL = 1e-9


@pytest.fixture(scope="module")
def steep():
    tab = gen.steep_limb_atmosphere()
    return tab, o.Atmosphere(*tab)


def _gpu(conf, tab, emission, domain):
    import torch
    import paper_2510_07764_b200 as ppm
    cfg = dict(conf["cfg"], emission=emission, interp_domain=domain)
    ctx = ppm.PPM(cfg, conf["energies"], max_batch=1)
    ctx.load_atmosphere(*tab)
    flux, st = ctx.evaluate(torch.as_tensor(conf["params"], device="cuda"))
    torch.cuda.synchronize()
    assert int(st[0]) == 0
    return flux.cpu().numpy()[0]


@pytest.mark.parametrize("which", [1, 2])
def test_table3_geometries_four_strategies(which, steep):
    tab, atm = steep
    conf = gen.config_interp_test(which, n_cells=12, n_phase=64, n_energy=40)
    ref = {}
    for em in (1, 4, 3, 2):
        ref[em], st = o.evaluate(dict(conf["cfg"], emission=em, interp_domain=1), conf["energies"], conf["params"][0], atm)
        assert st == 0
    scale = 2.0 * ref[4] - ref[1]                       # sum of |terms| per bin under the cubic stencils
    assert np.all(scale > 0) and ref[1].min() < 0 and (ref[4] == 0).any()
    worst = {}
    for em in (1, 4, 3, 2):
        g = _gpu(conf, tab, em, 1)
        s = scale if em in (1, 4) else np.maximum(np.abs(ref[em]), 1e-6 * np.abs(ref[em]).max())
        worst[em] = float(np.max(np.abs(g - ref[em]) / s))
        assert worst[em] <= TOL, (em, worst[em])
    # the qualitative finding on the device: lobes, holes, clean
    ga, gb, gd = _gpu(conf, tab, 1, 1), _gpu(conf, tab, 4, 1), _gpu(conf, tab, 2, 1)
    assert ga.min() < -1e-2 * gd.max() and gb.min() == 0.0 and (gb == 0).sum() > 0 and gd.min() > -1e-12 * gd.max()
    # bins that are exactly 0 in the oracle under clipping are exactly 0 on the device
    assert np.all(gb[ref[4] == 0] == 0.0)
    report("table3_test%d" % which, **{"strategy_%s" % k: v for k, v in zip("abcd", (worst[1], worst[4], worst[3], worst[2]))})
    # log-domain reading (R13a/R13f): b == a, all positive
    la, lb = _gpu(conf, tab, 1, 0), _gpu(conf, tab, 4, 0)
    assert np.array_equal(la, lb) and la.min() > 0


@pytest.mark.parametrize("name,kw", [("c2", dict(n_cells=24, n_phase=32, n_energy=64)),
                                     ("c3", dict(n_cells=40, n_phase=37, n_energy=77)),
                                     ("c4", dict(n_cells=48, n_phase=64, n_energy=96))])
@pytest.mark.parametrize("emission", [1, 2, 3])
def test_intensity_domain_on_the_standard_table(name, kw, emission):
    """interp_domain = 1 on the smooth synthetic table (ragged sizes, ring, occultation, both table ends): plain per-bin
    relative error where the flux is not negligible; the Wien tail (> 12 decades below the peak), where the cubic along
    log x can cancel, relative to the peak."""
    conf = getattr(gen, "config_" + name)(**kw)
    tab = gen.synthetic_atmosphere()
    ref, st = o.evaluate(dict(conf["cfg"], emission=emission, interp_domain=1), conf["energies"], conf["params"][0],
                         o.Atmosphere(*tab))
    g = _gpu(conf, tab, emission, 1)
    assert st == 0 and ref.max() > 0
    big = np.abs(ref) > 1e-12 * ref.max()
    assert np.max(np.abs(g[big] - ref[big]) / np.abs(ref[big])) <= TOL
    assert np.max(np.abs(g[~big] - ref[~big])) <= 1e-20 * ref.max() if (~big).any() else True
    assert np.all(g[ref == 0] == 0)
