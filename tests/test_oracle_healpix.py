"""Pins for the oracle's HEALPix ring mesh (Eq 24-29).  No HEALPix library is available, so the
formulas are pinned by what the equal-area isolatitude construction fixes: pixel counts, the equal-area ring edges,
the north-south mirror, the azimuth layout, full-sphere coverage and the closed-form flux of a face-on cap (P10)."""
import numpy as np
import pytest

import gen
import oracle as o


@pytest.mark.parametrize("nside", [1, 2, 5, 8, 37])
def test_ring_counts_areas_and_mirror(nside):
    rings = [o.healpix_ring(nside, i) for i in range(1, 4 * nside)]
    npix = np.array([r[1] for r in rings])
    z = np.array([r[0] for r in rings])
    assert npix.sum() == 12 * nside ** 2
    assert np.all(np.diff(z) < 0)                                     # rings ordered north -> south
    # equal area: the sphere above the lower edge of ring i holds cum(i) pixels of area 4 pi / (12 N^2), so
    # z_edge(i) = 1 - 2 cum(i) / (12 N^2); every ring centre lies strictly inside its own band
    cum = np.cumsum(npix)
    z_edge = np.concatenate([[1.0], 1.0 - 2.0 * cum / (12.0 * nside ** 2)])
    assert abs(z_edge[-1] + 1.0) < 1e-14
    assert np.all(z < z_edge[:-1]) and np.all(z > z_edge[1:])
    # Eq 28-29: southern rings mirror the northern ones
    for i in range(1, 2 * nside):
        a, b = rings[i - 1], rings[4 * nside - i - 1]
        assert a[0] == -b[0] and a[1:] == b[1:]
    assert abs(rings[2 * nside - 1][0]) < 1e-15                       # the equator ring
    # azimuths: uniform, covering the circle once; Eq 25 / 27 for pixel 1
    for i, (zz, n, p0, dp) in enumerate(rings, start=1):
        assert abs(n * dp - 2 * np.pi) < 1e-14
        iN = min(i, 4 * nside - i)
        if iN < nside:
            assert n == 4 * iN and abs(p0 - np.pi / (2 * iN) * 0.5) < 1e-15
            assert abs(abs(zz) - (1 - iN ** 2 / (3 * nside ** 2))) < 1e-15            # Eq 24
        else:
            assert n == 4 * nside
            assert abs(p0 - np.pi / (2 * nside) * (1 - ((iN - nside + 1) % 2) / 2)) < 1e-15   # Eq 27
            assert abs(abs(zz) - (4 / 3 - 2 * iN / (3 * nside))) < 1e-15              # Eq 26


def test_masks_full_sphere_cap_and_ring():
    nside = 16
    full = o.spot_mask_healpix(o.spot(1.0, 0.3, np.pi, 6.0), nside)
    assert full.sum() == 12 * nside ** 2
    for j in range(4 * nside - 1):
        assert full[j].sum() == o.healpix_ring(nside, j + 1)[1]       # entries past a ring's pixel count stay 0
    cap = o.spot_mask_healpix(o.spot(1.2, 0.5, 0.4, 6.0), nside)
    area = cap.sum() * np.pi / (3 * nside ** 2)
    assert abs(area / (2 * np.pi * (1 - np.cos(0.4))) - 1) < 0.02     # equal-area pixels: count x pixel area ~ cap area
    ring = o.spot_mask_healpix(o.spot(1.2, 0.5, 0.4, 6.0, 1.25, 0.5, 0.15), nside)
    assert 0 < ring.sum() < cap.sum() and not np.any(ring & ~cap)
    # brute force: centre-in test written out with unit vectors
    th = np.arccos([o.healpix_ring(nside, j + 1)[0] for j in range(4 * nside - 1)])
    c = np.array([np.sin(1.2) * np.cos(0.5), np.sin(1.2) * np.sin(0.5), np.cos(1.2)])
    for j in range(0, 4 * nside - 1, 3):
        _, n, p0, dp = o.healpix_ring(nside, j + 1)
        ph = p0 + dp * np.arange(n)
        v = np.stack([np.sin(th[j]) * np.cos(ph), np.sin(th[j]) * np.sin(ph), np.full(n, np.cos(th[j]))], axis=1)
        sep = np.arccos(np.clip(v @ c, -1, 1))
        safe = np.abs(sep - 0.4) > 1e-9
        assert np.array_equal(cap[j, :n][safe].astype(bool), (sep <= 0.4)[safe])


def test_p10_absolute_scale_on_the_healpix_mesh(golden):
    """The face-on cap of pin P10 (closed form, tests/golden/cap_flux_pins.txt) on HEALPix: converges ~ 1/N_side
    (centre-in mask), phase independent."""
    pins = {(q, float(E)): float(v) for q, E, v in golden("cap_flux_pins.txt")}
    E3 = np.array([0.3, 1.0, 3.0])
    ref = np.array([pins[("flux", E)] for E in E3])
    errs = []
    for nside in (32, 64, 128):
        cfg = dict(n_spots=1, n_theta=4 * nside - 1, n_phi=4 * nside, n_phase=4, n_fp=8, emission=0, oblate=0, mesh=1)
        p = gen.pack_params(1.4, 12.0, 0.0, 1.0, 0.2, spots=[(0.0, 0.0, 0.2, gen.log10T_of_kT(0.3))])
        f, st = o.evaluate(cfg, E3, p)
        assert st == 0 and np.max(np.abs(f / f[0:1] - 1.0)) < 1e-12
        errs.append(np.max(np.abs(f[0] / ref - 1.0)))
    assert errs[2] < 0.02 and errs[2] < errs[0]


def test_healpix_and_box_meshes_agree_for_a_large_cap():
    """Two discretisations of the same cap give the same pulse profile up to their (first-order) edge errors."""
    E = gen.logspace(0.3, 3.0, 4)
    p = gen.pack_params(1.4, 12.0, 300.0, np.cos(1.0), 0.2, spots=[(0.9, 0.4, 0.5, gen.log10T_of_kT(0.3))])
    box = dict(n_spots=1, n_theta=96, n_phi=96, n_phase=8, n_fp=192, emission=0, oblate=1)
    hp = dict(n_spots=1, n_theta=4 * 64 - 1, n_phi=4 * 64, n_phase=8, n_fp=192, emission=0, oblate=1, mesh=1)
    fb, _ = o.evaluate(box, E, p)
    fh, _ = o.evaluate(hp, E, p)
    assert np.max(np.abs(fh / fb - 1.0)) < 0.02
