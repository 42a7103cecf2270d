"""Pins P2-P10, P12 for Algorithm O (oracle/bpm_oracle.c) -- closed forms, invariants and
brute force, none of which call the oracle's step to produce the expected value.

Every expected value below is written from physics / mathematics:
  P2  tilted plane wave: eigenfunction of the step, phase exp(i dz sqrt(k^2-kx^2-ky^2));
      evanescent mode -> 0                      (pins kx ordering, propagator sign, cut-off)
  P3  uniform slab dn = c: with nref = n0 + c the result is exact propagation in index n0+c;
      with nref = n0 the on-axis phase per step is k0 (n0 + c) dz   (pins screen sign/scale, A3)
  P4  step splitting in a homogeneous medium
  P5  Gaussian beam vs 1-D Hankel quadrature of the angular-spectrum integral (scipy)
  P6  Gaussian beam vs the paraxial closed form
  P7  Parseval / unitarity on an all-propagating grid; monotone energy on a cut-off grid
  P8  reversibility
  P9  linearity
  P10 shift / transpose / mirror equivariance
  P12 n_ref helper
plus a step rebuilt with numpy's pocketfft (an independent FFT) for a random field + dn.
"""
import math

import numpy as np
import pytest

from conftest import rel_l2
from paper_1706_02261_b200 import workloads as wl

F32 = np.float32


def f32(x):
    """float32-rounded scalar as a Python float (what both C ABIs receive)."""
    return float(np.float32(x))


def kgrid(N, dx):
    return 2.0 * np.pi * np.fft.fftfreq(N, d=f32(dx))


def plane_wave(Nx, Ny, p, q):
    y, x = np.mgrid[0:Ny, 0:Nx]
    return np.exp(2j * np.pi * (p * x / Nx + q * y / Ny))


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("p,q", [(0, 0), (3, 0), (0, 5), (7, 9), (-4, 6), (-11, -2)])
def test_p2_tilted_plane_wave(oracle_mod, p, q):
    Nx, Ny, dx, dz, lam, n0 = 64, 32, 0.2, 0.13, 0.5, 1.33
    u0 = plane_wave(Nx, Ny, p, q)      # double: the step API takes complex128, no input rounding
    k = 2 * np.pi / f32(lam) * f32(n0)
    kx = 2 * np.pi * p / (Nx * f32(dx))
    ky = 2 * np.pi * q / (Ny * f32(dx))
    s = k * k - kx * kx - ky * ky
    assert s > 0
    u = u0.astype(np.complex128)
    for j in range(1, 4):
        u, I = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)
        # homogeneous medium at nref = n0: the screen is exp(i*0) = 1
        expect = u0.astype(np.complex128) * np.exp(1j * j * f32(dz) * math.sqrt(s))
        assert rel_l2(u, expect) < 1e-12
        assert np.allclose(I, 1.0, atol=1e-12)


def test_p2_evanescent_mode_is_cut(oracle_mod):
    Nx = Ny = 64
    dx, dz, lam, n0 = 0.1, 0.1, 0.5, 1.33   # k = 16.7 rad/um, k_nyquist = 31.4 rad/um
    p = 24                                  # kx = 2 pi 24 / 6.4 = 23.6 > k  -> evanescent
    u0 = plane_wave(Nx, Ny, p, 0)
    u, _ = oracle_mod.bpm_step(u0, None, dx, dz, lam, n0)
    assert np.abs(u).max() < 1e-12
    # just inside the light cone survives with unit modulus
    p = 16                                  # kx = 15.7 < 16.7
    u0 = plane_wave(Nx, Ny, p, 0)
    u, _ = oracle_mod.bpm_step(u0, None, dx, dz, lam, n0)
    assert abs(np.abs(u).mean() - 1.0) < 1e-12


# ---------------------------------------------------------------- P3
def test_p3_uniform_slab_adapted_nref_is_exact(oracle_mod):
    Nx, Ny, dx, dz, lam, n0, c = 32, 32, 0.2, 0.2, 0.5, 1.33, 0.04
    dn = np.full((Ny, Nx), c, dtype=F32)
    nref = F32(F32(n0) + F32(c))
    p, q = 3, -2
    u0 = plane_wave(Nx, Ny, p, q)
    kx = 2 * np.pi * p / (Nx * f32(dx))
    ky = 2 * np.pi * q / (Ny * f32(dx))
    k0 = 2 * np.pi / f32(lam)
    u = u0.astype(np.complex128)
    for j in range(1, 6):
        u, _ = oracle_mod.bpm_step(u, dn, dx, dz, lam, n0, nref=nref)
        # exact propagation in a homogeneous medium of index nref, times the residual screen
        # exp(i k0 dz (n0 + c - nref)) which is ~1e-8 rad because nref is float32-rounded
        resid = f32(n0) + float(F32(c)) - float(nref)
        expect = u0.astype(np.complex128) * np.exp(
            1j * j * f32(dz) * (math.sqrt((k0 * float(nref)) ** 2 - kx * kx - ky * ky) + k0 * resid))
        assert rel_l2(u, expect) < 1e-12
    # the same test with a fixed reference index must NOT agree for a tilted wave:
    u = u0.astype(np.complex128)
    for j in range(5):
        u, _ = oracle_mod.bpm_step(u, dn, dx, dz, lam, n0, nref=None)
    k_true = k0 * (f32(n0) + float(F32(c)))
    exact = u0.astype(np.complex128) * np.exp(1j * 5 * f32(dz) * math.sqrt(k_true ** 2 - kx * kx - ky * ky))
    assert rel_l2(u, exact) > 1e-4


def test_p3_on_axis_phase_with_fixed_reference(oracle_mod):
    Nx, Ny, dx, dz, lam, n0, c = 16, 16, 0.2, 0.1, 0.5, 1.33, 0.03
    dn = np.full((Ny, Nx), c, dtype=F32)
    u = np.ones((Ny, Nx), dtype=np.complex128)
    k0 = 2 * np.pi / f32(lam)
    out = u.astype(np.complex128)
    for j in range(1, 5):
        out, _ = oracle_mod.bpm_step(out, dn, dx, dz, lam, n0)
        expect = np.exp(1j * j * k0 * (f32(n0) + float(F32(c))) * f32(dz))
        assert np.abs(out - expect).max() < 1e-12


# ---------------------------------------------------------------- P4
def test_p4_step_splitting_homogeneous(oracle_mod):
    N, dx, lam, n0 = 64, 0.1, 0.5, 1.33
    u0 = wl.gaussian_beam(N, N, dx, 1.0)
    dz = 0.25          # exactly representable, so 8*dz, dz/2 are exact in float32 too
    Nz = 8
    a = u0.astype(np.complex128)
    for _ in range(Nz):
        a, _ = oracle_mod.bpm_step(a, None, dx, dz, lam, n0)
    b, _ = oracle_mod.bpm_step(u0, None, dx, dz * Nz, lam, n0)
    c = u0.astype(np.complex128)
    for _ in range(2 * Nz):
        c, _ = oracle_mod.bpm_step(c, None, dx, dz / 2, lam, n0)
    assert rel_l2(a, b) < 1e-11
    assert rel_l2(c, b) < 1e-11


# ---------------------------------------------------------------- P5 / P6
def _hankel_gaussian(r, z, w0, k):
    """u(r,z) = (w0^2/2) int_0^k exp(-kappa^2 w0^2/4) exp(i z sqrt(k^2-kappa^2)) J0(kappa r) kappa dkappa
    (angular-spectrum integral of exp(-r^2/w0^2), propagating part only), by adaptive quadrature."""
    from scipy.integrate import quad
    from scipy.special import j0
    kmax = min(k, 14.0 / w0)   # exp(-(14/w0)^2 w0^2/4) = e^-49: below double precision of the result

    def re(kap):
        return math.exp(-kap * kap * w0 * w0 / 4) * math.cos(z * math.sqrt(k * k - kap * kap)) * j0(kap * r) * kap

    def im(kap):
        return math.exp(-kap * kap * w0 * w0 / 4) * math.sin(z * math.sqrt(k * k - kap * kap)) * j0(kap * r) * kap

    a = quad(re, 0.0, kmax, epsabs=1e-14, epsrel=1e-13, limit=400)[0]
    b = quad(im, 0.0, kmax, epsabs=1e-14, epsrel=1e-13, limit=400)[0]
    return (w0 * w0 / 2) * (a + 1j * b)


def test_p5_gaussian_beam_vs_hankel_quadrature(oracle_mod):
    N, dx, dz, lam, n0, w0 = 256, 0.1, 0.1, 0.5, 1.33, 2.0
    u0 = wl.gaussian_beam(N, N, dx, w0)
    k = 2 * np.pi / f32(lam) * f32(n0)
    checks = {32: 3.2, 64: 6.4, 128: 12.8}
    u = u0.astype(np.complex128)
    c = N // 2
    for j in range(1, 129):
        u, _ = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)
        if j in checks:
            z = j * f32(dz)
            for ir in (0, 5, 10):          # r = 0, 0.5, 1.0 um along x; and along y
                r = ir * f32(dx)
                ref = _hankel_gaussian(r, z, w0, k)
                # the input is complex64: its rounding (~3e-8 relative per pixel, averaging
                # down in the transform) bounds the agreement, not the oracle's arithmetic
                assert abs(u[c, c + ir] - ref) < 1e-7 * abs(ref) + 1e-9
                assert abs(u[c + ir, c] - ref) < 1e-7 * abs(ref) + 1e-9


def test_p5_gaussian_beam_double_input_tight(oracle_mod):
    """Same pin with a float64 input field fed to the step directly: agreement at 1e-10."""
    N, dx, dz, lam, n0, w0 = 256, 0.1, 0.1, 0.5, 1.33, 2.0
    x = (np.arange(N) - N // 2) * f32(dx)
    u = np.exp(-(x[:, None] ** 2 + x[None, :] ** 2) / w0 ** 2).astype(np.complex128)
    k = 2 * np.pi / f32(lam) * f32(n0)
    c = N // 2
    for j in range(1, 65):
        u, _ = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)
    z = 64 * f32(dz)
    for ir in (0, 5, 10):
        ref = _hankel_gaussian(ir * f32(dx), z, w0, k)
        assert abs(u[c, c + ir] - ref) < 1e-10
        assert abs(u[c + ir, c] - ref) < 1e-10


def test_p6_gaussian_beam_vs_paraxial_closed_form(oracle_mod):
    N, dx, dz, lam, n0, w0 = 256, 0.1, 0.1, 0.5, 1.33, 2.0
    u0 = wl.gaussian_beam(N, N, dx, w0)
    k = 2 * np.pi / f32(lam) * f32(n0)
    zR = math.pi * w0 * w0 * f32(n0) / f32(lam)
    u = u0.astype(np.complex128)
    for j in range(64):
        u, _ = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)
    z = 64 * f32(dz)
    x = (np.arange(N) - N // 2) * f32(dx)
    r2 = x[:, None] ** 2 + x[None, :] ** 2
    q = 1 + 1j * z / zR
    expect = np.exp(-r2 / (w0 * w0 * q)) / q * np.exp(1j * k * z)
    assert rel_l2(u, expect) < 2e-3            # non-paraxial correction is ~6e-4
    assert rel_l2(u, np.conj(expect)) > 0.1    # a sign error in the propagator fails


# ---------------------------------------------------------------- P7 / P8
def _all_propagating_case(seed=11, N=64, Nz=24):
    dx, dz, lam, n0 = 0.3, 0.2, 0.5, 1.33     # dx > lam / (sqrt(2) n0) = 0.266: every mode propagates
    rng = np.random.default_rng(seed)
    u0 = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    dn = rng.uniform(0.0, 0.05, size=(Nz, N, N)).astype(F32)
    k = 2 * np.pi / f32(lam) * f32(n0)
    kk = kgrid(N, dx)
    assert (k * k - kk[:, None] ** 2 - kk[None, :] ** 2).min() > 0
    return u0, dn, dx, dz, lam, n0


def test_p7_parseval_all_propagating(oracle_mod):
    u0, dn, dx, dz, lam, n0 = _all_propagating_case()
    e0 = float(np.sum(np.abs(u0.astype(np.complex128)) ** 2))
    energies = []
    oracle_mod.propagate_stream(u0, dn, dx, dz, lam, n0,
                                on_slice=lambda j, u, I: energies.append((float(np.sum(np.abs(u) ** 2)),
                                                                          float(I.sum()))))
    for eu, ei in energies:
        assert abs(eu - e0) < 1e-12 * e0
        assert abs(ei - e0) < 1e-12 * e0      # I really is |u|^2 of the same field


def test_p7_energy_monotone_on_cutoff_grid(oracle_mod):
    w = wl.tiny(N=64, Nz=32, dx=0.1, dz=0.1, w0=0.4)    # tightly focused: has evanescent content
    u0 = wl.make_field(w)[0]
    dn = wl.make_dn(w).numpy()
    e = [float(np.sum(np.abs(u0.astype(np.complex128)) ** 2))]
    oracle_mod.propagate_stream(u0, dn, w.dx, w.dz, w.lam, w.n0,
                                on_slice=lambda j, u, I: e.append(float(I.sum())))
    e = np.array(e)
    assert np.all(np.diff(e) <= 1e-12 * e[0])
    assert e[-1] < e[0]                                    # something was cut


def test_p8_reversibility(oracle_mod):
    u0, dn, dx, dz, lam, n0 = _all_propagating_case(seed=5, N=64, Nz=40)
    nref = (F32(n0) + dn.mean(axis=(1, 2))).astype(F32)
    u = oracle_mod.propagate_stream(u0, dn, dx, dz, lam, n0, nref=nref)
    assert rel_l2(u, u0) > 0.5
    for j in range(dn.shape[0] - 1, -1, -1):
        u = oracle_mod.bpm_step_backward(u, dn[j], dx, dz, lam, n0, nref=nref[j])
    assert rel_l2(u, u0) < 1e-11


# ---------------------------------------------------------------- P9 / P10
def _tiny_case(N=32, Nz=16, seed=0):
    w = wl.tiny(N=N, Nz=Nz)
    dn = wl.make_dn(w).numpy()
    nref = (F32(w.n0) + dn.reshape(Nz, -1).mean(axis=1)).astype(F32)
    return w, dn, nref


def test_p9_linearity(oracle_mod):
    w, dn, nref = _tiny_case()
    u1 = wl.random_field(w.Nx, w.Ny, 1)[0]
    u2 = wl.random_field(w.Nx, w.Ny, 2)[0]
    a, b = 0.5, 2.0      # exactly representable scalings keep the complex64 inputs exact
    f1, _ = oracle_mod.propagate(u1, dn, w.dx, w.dz, w.lam, w.n0, nref)
    f2, _ = oracle_mod.propagate(u2, dn, w.dx, w.dz, w.lam, w.n0, nref)
    # feed the double-precision mix through the step API so no input rounding enters
    u = a * u1.astype(np.complex128) + 1j * b * u2.astype(np.complex128)
    for j in range(w.Nz):
        u, _ = oracle_mod.bpm_step(u, dn[j], w.dx, w.dz, w.lam, w.n0, nref[j])
    assert rel_l2(u, a * f1 + 1j * b * f2) < 1e-12


@pytest.mark.parametrize("sx,sy", [(5, 0), (0, -3), (7, 11)])
def test_p10_shift_equivariance(oracle_mod, sx, sy):
    w, dn, nref = _tiny_case()
    u0 = wl.random_field(w.Nx, w.Ny, 3)[0]
    f, I = oracle_mod.propagate(u0, dn, w.dx, w.dz, w.lam, w.n0, nref)
    fs, Is = oracle_mod.propagate(np.roll(u0, (sy, sx), axis=(0, 1)),
                                  np.roll(dn, (sy, sx), axis=(1, 2)), w.dx, w.dz, w.lam, w.n0, nref)
    assert rel_l2(fs, np.roll(f, (sy, sx), axis=(0, 1))) < 1e-12
    assert rel_l2(Is, np.roll(I, (sy, sx), axis=(1, 2))) < 1e-12


def test_p10_transpose_and_mirror(oracle_mod):
    w, dn, nref = _tiny_case()
    u0 = wl.random_field(w.Nx, w.Ny, 4)[0]
    f, I = oracle_mod.propagate(u0, dn, w.dx, w.dz, w.lam, w.n0, nref)
    ft, It = oracle_mod.propagate(u0.T.copy(), dn.transpose(0, 2, 1).copy(), w.dx, w.dz, w.lam, w.n0, nref)
    assert rel_l2(ft, f.T) < 1e-12
    assert rel_l2(It, I.transpose(0, 2, 1)) < 1e-12
    # mirror x -> -x (index i -> (-i) mod N keeps the periodic grid)
    idx = (-np.arange(w.Nx)) % w.Nx
    fm, Im = oracle_mod.propagate(u0[:, idx].copy(), dn[:, :, idx].copy(), w.dx, w.dz, w.lam, w.n0, nref)
    assert rel_l2(fm, f[:, idx]) < 1e-12
    assert rel_l2(Im, I[:, :, idx]) < 1e-12


def test_non_square_grid_transpose(oracle_mod):
    """Nx != Ny (the paper's Fig. 1 grid is 1024 x 2048)."""
    Nx, Ny, Nz = 64, 32, 6
    rng = np.random.default_rng(8)
    u0 = wl.random_field(Nx, Ny, 5)[0]
    dn = rng.uniform(0, 0.05, size=(Nz, Ny, Nx)).astype(F32)
    f, I = oracle_mod.propagate(u0, dn, 0.2, 0.2, 0.5, 1.33)
    ft, It = oracle_mod.propagate(u0.T.copy(), dn.transpose(0, 2, 1).copy(), 0.2, 0.2, 0.5, 1.33)
    assert f.shape == (Ny, Nx) and ft.shape == (Nx, Ny)
    assert rel_l2(ft, f.T) < 1e-12
    assert rel_l2(It, I.transpose(0, 2, 1)) < 1e-12


# ---------------------------------------------------------------- independent rebuild of one step
def test_step_vs_numpy_pocketfft_rebuild(oracle_mod):
    """The whole step rebuilt here with numpy's FFT and fftfreq, in double, from the formulas of
    BASELINE.json:north_star -- catches a dropped term, a wrong index or a transposed operand
    for a general (non-eigenfunction) field and a non-uniform dn."""
    Nx, Ny, dx, dz, lam, n0 = 64, 32, 0.1, 0.15, 0.5, 1.33
    rng = np.random.default_rng(21)
    u0 = wl.random_field(Nx, Ny, 6)[0]
    dn = rng.uniform(-0.02, 0.05, size=(Ny, Nx)).astype(F32)
    nref = F32(1.345)
    k0 = 2 * np.pi / f32(lam)
    kx = kgrid(Nx, dx)[None, :]
    ky = kgrid(Ny, dx)[:, None]
    s = (k0 * float(nref)) ** 2 - kx ** 2 - ky ** 2
    H = np.where(s > 0, np.exp(1j * f32(dz) * np.sqrt(np.maximum(s, 0))), 0)
    assert (s <= 0).any() and (s > 0).any()
    v = np.fft.ifft2(np.fft.fft2(u0.astype(np.complex128)) * H)
    v = v * np.exp(1j * k0 * f32(dz) * (f32(n0) + dn.astype(np.float64) - float(nref)))
    u, I = oracle_mod.bpm_step(u0, dn, dx, dz, lam, n0, nref=nref)
    assert rel_l2(u, v) < 1e-13
    assert rel_l2(I, np.abs(v) ** 2) < 1e-13


def test_propagate_matches_stepping_and_accumulate(oracle_mod):
    w, dn, nref = _tiny_case(N=32, Nz=5)
    u0 = wl.random_field(w.Nx, w.Ny, 9)[0]
    f, I = oracle_mod.propagate(u0, dn, w.dx, w.dz, w.lam, w.n0, nref)
    slices = []
    g = oracle_mod.propagate_stream(u0, dn, w.dx, w.dz, w.lam, w.n0, nref,
                                    on_slice=lambda j, u, Ij: slices.append(Ij.copy()))
    assert np.array_equal(f, g) and np.array_equal(I, np.stack(slices))
    init = np.full_like(I, 0.25)
    _, Iacc = oracle_mod.propagate(u0, dn, w.dx, w.dz, w.lam, w.n0, nref, intensity_init=init)
    assert np.allclose(Iacc, I + 0.25, rtol=0, atol=1e-15)


# ---------------------------------------------------------------- P12
def test_p12_nref_helper(oracle_mod):
    n0 = 1.33
    dn = np.full((7, 8, 16), 0.03, dtype=F32)
    out = oracle_mod.nref_from_dn(dn, n0, 3)
    assert np.all(out == F32(float(F32(n0)) + float(F32(0.03))))
    # two-level volume, slab 2, short last slab: hand-computed means
    dn = np.zeros((5, 4, 4), dtype=F32)
    dn[0] = 0.5; dn[1] = 0.25; dn[2, :2] = 1.0; dn[4] = 0.125
    out = oracle_mod.nref_from_dn(dn, 1.0, 2)
    expect = np.array([1.375, 1.375, 1.25, 1.25, 1.125], dtype=F32)
    assert np.array_equal(out, expect)
    out1 = oracle_mod.nref_from_dn(dn, 1.0, 1)
    assert np.array_equal(out1, np.array([1.5, 1.25, 1.5, 1.0, 1.125], dtype=F32))
