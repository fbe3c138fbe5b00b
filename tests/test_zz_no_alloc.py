"""-m gpu: ppm_loglike_noalloc (include/ppm.h, csrc/ppm_noalloc.cu) -- the allocation-free Poisson ln L whose scratch is a
static __device__ array -- against the existing path ppm_loglike, on two calls in a row that share that array.
Collected last on purpose (file name): the suite runs with pytest -x, so a failure here hides nothing after it."""
import numpy as np
import pytest

import gen
from gpu_common import make_ctx

pytestmark = pytest.mark.gpu


def _counts_and_data(n_vec, seed):
    """Folded counts of a small C5-like batch through the existing path, and seeded Poisson data drawn from vector 0."""
    import torch
    conf = gen.config_c5(n_vec=n_vec, n_cells=16, n_phase=8, n_energy=300)
    rsp = gen.synthetic_response(conf["energies"])
    ctx = make_ctx(conf)
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    p = torch.as_tensor(conf["params"], device="cuda")
    flux, status = ctx.evaluate(p)
    counts = ctx.fold_response(flux, p)
    torch.cuda.synchronize()
    assert int(status.sum()) == 0
    c0 = counts[0].cpu().numpy()
    expo = 1e6 / (c0.sum() / 8)
    bkg = np.full(rsp["n_channel"], 0.05 * 1e6 / (8 * rsp["n_channel"]))
    data = np.random.default_rng(seed).poisson(expo * c0 / 8 + bkg).astype(np.float64)
    return ctx, counts, torch.as_tensor(data, device="cuda"), torch.as_tensor(bkg, device="cuda"), expo


def test_noalloc_loglike_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    import paper_2510_07764_b200 as ppm
    ctx, counts, data, bkg, expo = _counts_and_data(5, 21)
    tol = 1e-9 * float(data.sum())                       # the bar of test_fold_and_loglike
    # call 1: all five vectors
    ref1 = ctx.loglike(counts, data, bkg, expo)
    out1 = torch.full((5,), 123.0, dtype=torch.float64, device="cuda")
    ppm.loglike_noalloc(counts, data, bkg, expo, out1)
    # call 2 right behind it, fewer vectors, other data, background and exposure: the shared scratch still holds call 1's
    # sums (the background keeps the model positive where the flipped data are, so ln L stays finite)
    data2 = torch.flip(data, dims=(0,)).contiguous()
    bkg2 = (3.0 * bkg).contiguous()
    ref2 = ctx.loglike(counts[1:4].contiguous(), data2, bkg2, 0.5 * expo)
    out2 = torch.full((3,), 123.0, dtype=torch.float64, device="cuda")
    ppm.loglike_noalloc(counts[1:4].contiguous(), data2, bkg2, 0.5 * expo, out2)
    torch.cuda.synchronize()
    r1, o1, r2, o2 = (t.cpu().numpy() for t in (ref1, out1, ref2, out2))
    assert np.all(np.isfinite(r1)) and np.all(np.isfinite(r2))
    assert np.max(np.abs(o1 - r1)) <= tol and np.max(np.abs(o2 - r2)) <= tol
    assert np.array_equal(o1, r1) and np.array_equal(o2, r2)         # same arithmetic, same summation order: same bits
    # -inf where the model is zero and the data are not, as on the existing path
    out3 = torch.empty((5,), dtype=torch.float64, device="cuda")
    ppm.loglike_noalloc(torch.zeros_like(counts), data, None, expo, out3)
    assert np.all(np.isneginf(out3.cpu().numpy()))


def test_noalloc_loglike_rejects_batches_beyond_the_static_maximum():
    import torch
    import paper_2510_07764_b200 as ppm
    n = ppm.NOALLOC_MAX_BATCH
    data = torch.ones((2, 3), dtype=torch.float64, device="cuda")
    big = torch.ones((n + 1, 2, 3), dtype=torch.float64, device="cuda")
    out = torch.zeros((n + 1,), dtype=torch.float64, device="cuda")
    with pytest.raises(ppm.PPMError, match="PPM_NOALLOC_MAX_BATCH"):
        ppm.loglike_noalloc(big, data, None, 1.0, out)
    # the maximum itself is accepted: ln L = sum d ln m - m - lgamma(d + 1) with m = exposure * counts / n_phase = 0.5, d = 1
    ok = torch.empty((n,), dtype=torch.float64, device="cuda")
    ppm.loglike_noalloc(big[:n].contiguous(), data, None, 1.0, ok)
    torch.cuda.synchronize()
    assert np.allclose(ok.cpu().numpy(), 6 * (np.log(0.5) - 0.5), rtol=0, atol=1e-12)
