"""Helpers shared by the -m gpu parity tests: run one workload through the C ABI (CUDA path) and
through the oracle on the same seeded arrays."""
import functools

import numpy as np

import gen
import oracle as o


@functools.lru_cache(maxsize=1)
def atmosphere():
    return gen.synthetic_atmosphere()


@functools.lru_cache(maxsize=1)
def oracle_atm():
    return o.Atmosphere(*atmosphere())


def make_ctx(conf, max_batch=None, precision=0, scratch_mb=0):
    import paper_2510_07764_b200 as ppm
    B = conf["params"].shape[0]
    ctx = ppm.PPM(conf["cfg"], conf["energies"], max_batch=max_batch or B, precision=precision, scratch_mb=scratch_mb)
    if conf["cfg"]["emission"] != 0:
        ctx.load_atmosphere(*atmosphere())
    return ctx


def gpu_flux(conf, ctx=None, precision=0):
    import torch
    ctx = ctx or make_ctx(conf, precision=precision)
    p = torch.as_tensor(conf["params"], dtype=torch.float64, device="cuda").contiguous()
    flux, status = ctx.evaluate(p)
    torch.cuda.synchronize()
    return flux.cpu().numpy(), status.cpu().numpy(), ctx


def oracle_flux(conf, b=0, phase_sel=None):
    atm = oracle_atm() if conf["cfg"]["emission"] != 0 else None
    f, st = o.evaluate(conf["cfg"], conf["energies"], conf["params"][b], atm, phase_sel=phase_sel)
    return f, st


def max_rel_err(g, ref):
    """reading R22: max |g-o|/|o| over bins with o != 0; bins with o = 0 must have g = 0."""
    g, ref = np.asarray(g), np.asarray(ref)
    nz = ref != 0
    assert np.all(g[~nz] == 0.0), "bins that are exactly 0 in the oracle must be 0 on the GPU"
    if not nz.any():
        return 0.0
    return float(np.max(np.abs(g[nz] - ref[nz]) / np.abs(ref[nz])))


def chi2_eq56(model, ref):
    """Eq 56-57 between two non-negative arrays: both scaled to a total of 1e6 'counts' of the
    reference, chi^2 = K sum (m - d)^2 / m with m = reference (oracle), d = the other (GPU)."""
    return o.chi2(np.asarray(ref, dtype=np.float64), np.asarray(model, dtype=np.float64))


def report(name, **values):
    """Append one line to gpurun_out/parity_report.jsonl (when that folder exists): the numbers DESIGN.md quotes."""
    import json
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    d = os.path.join(root, "gpurun_out")
    if os.path.isdir(d):
        with open(os.path.join(d, "parity_report.jsonl"), "a") as f:
            f.write(json.dumps(dict(test=name, **{k: (float(v) if isinstance(v, (float, np.floating)) else v)
                                                   for k, v in values.items()})) + "\n")
