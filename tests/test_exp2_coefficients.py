"""CPU check of the degree-8 polynomial the table cell kernel uses for 2^f, |f| <= 1/2 (ppm_cells.cuh: exp2_frac_scaled): the
coefficients are parsed from the CUDA source and evaluated in the kernel's Horner order against numpy.exp2; the claimed
bound (max relative error 1.1e-12, three orders below the 1e-9 parity bar) is asserted.  Also the FP32 helper constants."""
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _coefficients():
    src = open(os.path.join(ROOT, "paper_2510_07764_b200", "csrc", "ppm_cells.cuh")).read()
    body = re.search(r"double exp2_frac_scaled\(double f, int n\).*?\{(.*?)return", src, flags=re.S).group(1)
    c = [float(x) for x in re.findall(r"(?:double p = |fma\(p, f, )([-+]?\d+\.?\d*(?:[eE][-+]?\d+)?)", body)]
    assert len(c) == 9
    return c


def test_exp2_polynomial_error_bound():
    c = _coefficients()
    assert c[-1] == 1.0 and abs(c[-2] - np.log(2.0)) < 1e-10                   # 2^f = 1 + f ln 2 + ...
    f = np.linspace(-0.5, 0.5, 200001)
    p = np.full_like(f, c[0])
    for ck in c[1:]:
        p = p * f + ck                                                        # the kernel's Horner chain (FMA there)
    rel = np.abs(p / np.exp2(f) - 1.0)
    assert rel.max() < 1.1e-12, rel.max()
    assert rel.max() > 1e-13                                                  # degree 8, not more: the bound is tight
    # round-to-nearest split used by the kernel: y = n + f with n = rint(y) through the 1.5 * 2^52 constant
    y = np.random.default_rng(0).uniform(-900.0, 900.0, 100000)
    magic = 6755399441055744.0
    r = y + magic
    n = (r - magic)
    assert np.all(np.abs(y - n) <= 0.5) and np.all(n == np.rint(y))
