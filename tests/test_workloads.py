"""Host logic: the seeded input generators (shapes, ranges, determinism, recipe facts)."""
import math

import numpy as np

from paper_1706_02261_b200 import workloads as wl


def test_configs_match_baseline_shapes():
    c = wl.CONFIGS
    assert (c["C1"].Nx, c["C1"].Nz, c["C1"].dx, c["C1"].lam) == (128, 128, 0.1, 0.5)
    assert (c["C2"].Nx, c["C2"].Nz, c["C2"].dx, c["C2"].lam, c["C2"].NA) == (256, 256, 0.2, 0.488, 0.1)
    assert (c["C3"].Nx, c["C3"].Nz, c["C3"].emitters, c["C3"].spacing) == (512, 512, 10, 8.0)
    assert (c["C4"].Nx, c["C4"].Nz, c["C4"].emitters, c["C4"].n_cells) == (1024, 1024, 32, 2000)
    assert (c["C5"].Nx, c["C5"].Nz, c["C5"].batch) == (512, 512, 16)
    assert all(w.n0 == 1.33 for w in c.values())


def test_dn_deterministic_and_in_range():
    w = wl.config("C1").with_nz(16)
    a = wl.make_dn(w).numpy()
    b = wl.make_dn(w).numpy()
    assert a.dtype == np.float32 and a.shape == (16, 128, 128)
    assert np.array_equal(a, b)
    nz = a[a != 0]
    assert nz.size > 0 and nz.min() >= 0.01 - 1e-7 and nz.max() <= 0.05 + 1e-7


def test_noise_statistics_and_smoothness():
    w = wl.tiny(N=32, Nz=32, n_cells=0, noise_sigma_um=0.6, noise_amp=0.005, dx=0.2, dz=0.2)
    v = wl.make_dn(w).numpy().astype(np.float64)
    assert abs(v.std() - 0.005) < 1e-4
    # blurred with sigma = 3 voxels: neighbouring voxels strongly correlated, periodic along every axis
    for ax in range(3):
        r = np.mean(v * np.roll(v, 1, axis=ax)) / np.mean(v * v)
        assert r > 0.9


def test_painter_order_later_cell_overwrites():
    w = wl.tiny(N=32, Nz=32, n_cells=40, r_lo=1.0, r_hi=2.5)
    v = wl.make_dn(w).numpy()
    rng = np.random.default_rng(w.seed)
    centres, radii, vals = wl._cell_params(w, rng)
    # brute force, voxel by voxel, in painter's order
    ref = np.zeros_like(v)
    zz, yy, xx = np.mgrid[0:w.Nz, 0:w.Ny, 0:w.Nx]
    for (cx, cy, cz), (rx, ry, rz), val in zip(centres, radii, vals):
        inside = (((xx * w.dx - cx) / rx) ** 2 + ((yy * w.dx - cy) / ry) ** 2
                  + ((zz * w.dz - cz) / rz) ** 2) <= 1.0
        ref[inside] = np.float32(val)
    assert np.array_equal(v, ref)


def test_fields():
    g = wl.make_field(wl.config("C1"))
    assert g.shape == (1, 128, 128) and g.dtype == np.complex64
    assert g[0, 64, 64] == 1.0 and abs(g[0, 64, 84] - math.exp(-1.0)) < 1e-6   # r = 2 um = w0
    s = wl.make_field(wl.config("C2"))[0]
    assert np.array_equal(s[:, 0], s[:, 100])                                  # flat in x
    assert abs(np.abs(s[:, 0]).argmax() - 128) <= 0
    b = wl.make_field(wl.config("C5"))
    assert b.shape == (16, 512, 512)
    assert wl.make_field(wl.config("C4")) is None
