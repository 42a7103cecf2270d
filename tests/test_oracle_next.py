"""Pins for the oracle functions of the NEXT rows (oracle/bpm_oracle.c, end of file).

Every expected value is a closed form, an invariant, plain array slicing, an independent library
routine (numpy's pocketfft, scipy's Bessel functions) or a composition of oracle functions that are
pinned elsewhere (tests/test_oracle_bpm.py) -- never the function under test:
  N1  refocus: tilted plane wave picks up exp(i dz sqrt(k^2 - k_perp^2)) for either sign of dz and is cut
      when evanescent; refocus(L) equals L / dz homogeneous Algorithm-O steps (P4); refocus(-dz) undoes
      refocus(dz) on an all-propagating grid; an on-grid emitter refocused away and back peaks at its pixel
  N2  tiles: array slicing with wrap-around; on-grid emitter -> tile centre value 1
  N3  backward propagation: undoes the forward run (P8) and records the forward run's intensities
  N4  light sheet: forward propagation by z_focus restores the Gaussian waist; amplitude against the
      paraxial cylindrical Gaussian beam; uniform in x
  N5  annular pupil: NA_in = 0 is Algorithm M; spectrum support; thin annulus -> J0(k0 NA r)
  N6  image formation: delta object -> the PSF tile of the nearest emitter at the right place; one emitter
      -> plain periodic convolution (numpy FFT); linearity in S
"""
import math

import numpy as np
import pytest

from conftest import rel_l2

F32 = np.float32


def f32(x):
    return float(np.float32(x))


def plane_wave(Nx, Ny, p, q):
    y, x = np.mgrid[0:Ny, 0:Nx]
    return np.exp(2j * np.pi * (p * x / Nx + q * y / Ny))


# ---------------------------------------------------------------- N1 refocus
@pytest.mark.parametrize("p,q,dz", [(0, 0, 0.7), (3, -2, 1.37), (5, 4, -2.13), (-7, 1, -0.4)])
def test_n1_refocus_plane_wave_closed_form(oracle_mod, p, q, dz):
    Nx, Ny, dx, lam, n = 64, 32, 0.2, 0.5, 1.36
    u0 = plane_wave(Nx, Ny, p, q)
    k = 2 * np.pi / f32(lam) * f32(n)
    kx, ky = 2 * np.pi * p / (Nx * f32(dx)), 2 * np.pi * q / (Ny * f32(dx))
    s = k * k - kx * kx - ky * ky
    assert s > 0
    u = oracle_mod.refocus(u0, dx, dz, lam, n)
    assert rel_l2(u, u0 * np.exp(1j * f32(dz) * math.sqrt(s))) < 1e-12
    assert rel_l2(u, u0 * np.exp(-1j * f32(dz) * math.sqrt(s))) > 1e-2     # the sign of dz matters


def test_n1_refocus_cuts_evanescent_modes_for_both_signs(oracle_mod):
    Nx, Ny, dx, lam, n = 64, 64, 0.1, 0.5, 1.33          # dx = lam / 5: bins beyond ~17 are evanescent
    u0 = plane_wave(Nx, Ny, 25, 3)
    for dz in (0.5, -0.5):
        assert np.abs(oracle_mod.refocus(u0, dx, dz, lam, n)).max() < 1e-12


def test_n1_refocus_equals_chained_homogeneous_steps(oracle_mod):
    rng = np.random.default_rng(3)
    N, dx, dz, lam, n0, steps = 32, 0.1, 0.1, 0.5, 1.33, 9
    u0 = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    u = u0.astype(np.complex128)
    for _ in range(steps):
        u, _ = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)                 # pinned by P2-P5
    L = float(np.float32(np.float32(dz) * steps))
    # the distance is passed as float32: use a step for which steps * dz is exact in float32 arithmetic
    assert abs(L - steps * f32(dz)) < 1e-7
    v = oracle_mod.refocus(u0, dx, steps * f32(dz), lam, n0)
    assert rel_l2(v, u) < 1e-6                                               # float32 rounding of L: k dL ~ 1e-7 rad
    # exact variant: dz = 0.125 (a binary fraction) makes steps * dz exact
    u = u0.astype(np.complex128)
    for _ in range(8):
        u, _ = oracle_mod.bpm_step(u, None, dx, 0.125, lam, n0)
    assert rel_l2(oracle_mod.refocus(u0, dx, 1.0, lam, n0), u) < 1e-11


def test_n1_refocus_inverts_itself_when_all_modes_propagate(oracle_mod):
    rng = np.random.default_rng(4)
    N, dx, lam, n = 64, 0.3, 0.5, 1.33                   # dx > lam / (sqrt2 n): nothing is cut
    u0 = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    away = oracle_mod.refocus(u0, dx, 7.5, lam, n)
    assert rel_l2(away, u0) > 0.5
    assert rel_l2(oracle_mod.refocus(away, dx, -7.5, lam, n), u0) < 1e-11


def test_n1_emitter_refocused_to_its_plane_peaks_at_its_pixel(oracle_mod):
    N, dx, lam, n0, NA = 64, 0.2, 0.5, 1.33, 0.8
    pos = np.array([[4 * 0.2, -6 * 0.2]], dtype=F32)     # on-grid: pixel (32 + 4, 32 - 6)
    u0 = oracle_mod.multiplex_psf(pos, None, None, NA, N, N, dx, lam)
    away = oracle_mod.refocus(u0, dx, 6.0, lam, n0)
    assert np.abs(away).max() < 0.5                      # defocused
    back = oracle_mod.refocus(away, dx, -6.0, lam, n0)   # NA 0.8 < n0: the whole pupil propagates
    iy, ix = np.unravel_index(np.argmax(np.abs(back)), back.shape)
    assert (ix, iy) == (36, 26)
    assert abs(back[26, 36] - 1.0) < 1e-11


# ---------------------------------------------------------------- N2 tiles
def test_n2_tiles_are_array_slices_with_wraparound(oracle_mod):
    rng = np.random.default_rng(8)
    Np, Ny, Nx, dx, T = 3, 16, 32, 0.25, 6
    vol = rng.standard_normal((Np, Ny, Nx))
    pos = np.array([[0.0, 0.0], [3.1 * dx, -2.6 * dx], [-16 * dx, 7 * dx], [15.4 * dx, -8 * dx]], dtype=F32)
    tiles = oracle_mod.extract_tiles(vol, pos, dx, T)
    assert tiles.shape == (4, Np, T, T)
    for e, (x, y) in enumerate(pos):
        cx = int(math.floor(float(x) / f32(dx) + 0.5)) + Nx // 2
        cy = int(math.floor(float(y) / f32(dx) + 0.5)) + Ny // 2
        shifted = np.roll(vol, (-(cy - T // 2), -(cx - T // 2)), axis=(1, 2))   # window start -> index 0
        assert np.array_equal(tiles[e], shifted[:, :T, :T])
    cplx = vol + 1j * rng.standard_normal(vol.shape)
    tc = oracle_mod.extract_tiles(cplx, pos, dx, T)
    assert np.array_equal(tc.real, tiles) and np.array_equal(tc.imag, oracle_mod.extract_tiles(cplx.imag, pos, dx, T))


def test_n2_on_grid_emitters_sit_at_their_tile_centres(oracle_mod):
    N, dx, lam, NA, T = 128, 0.2, 0.5, 0.8, 8
    pos = np.array([[-20 * dx, 12 * dx], [24 * dx, -30 * dx]], dtype=F32)     # far apart: side lobes ~1e-3
    u0 = oracle_mod.multiplex_psf(pos, None, None, NA, N, N, dx, lam)
    tiles = oracle_mod.extract_tiles(u0, pos, dx, T)
    for e in range(2):
        t = np.abs(tiles[e, 0])
        assert np.unravel_index(np.argmax(t), t.shape) == (T // 2, T // 2)
        assert abs(t[T // 2, T // 2] - 1.0) < 5e-3


# ---------------------------------------------------------------- N3 backward
def test_n3_backward_undoes_forward_and_records_the_same_planes(oracle_mod):
    rng = np.random.default_rng(5)
    N, Nz, dx, dz, lam, n0 = 32, 12, 0.3, 0.2, 0.5, 1.33          # all modes propagate
    u0 = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    dn = rng.uniform(0.0, 0.05, size=(Nz, N, N)).astype(F32)
    nref = (F32(n0) + dn.mean(axis=(1, 2))).astype(F32)
    uf, If = oracle_mod.propagate(u0, dn, dx, dz, lam, n0, nref=nref)           # pinned by P2-P10
    ub, Ib = oracle_mod.propagate_backward(uf.astype(np.complex64), dn, dx, dz, lam, n0, nref=nref)
    assert rel_l2(ub, u0) < 2e-7                                   # complex64 rounding of the hand-over field
    assert rel_l2(Ib, If) < 4e-7
    # step by step against the pinned single step (P8), no rounding in between
    u = uf.copy()
    for j in range(Nz - 1, -1, -1):
        u = oracle_mod.bpm_step_backward(u, dn[j], dx, dz, lam, n0, nref=nref[j])
    assert rel_l2(u, u0) < 1e-11


def test_n3_backward_on_a_cutoff_grid_loses_exactly_the_evanescent_part(oracle_mod):
    N, dx, dz, lam, n0 = 32, 0.1, 0.1, 0.5, 1.33
    rng = np.random.default_rng(6)
    u0 = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)
    dn = np.zeros((1, N, N), dtype=F32)
    ub, _ = oracle_mod.propagate_backward(u0, dn, dx, dz, lam, n0)
    k = 2 * np.pi / f32(lam) * f32(n0)
    kk = 2 * np.pi * np.fft.fftfreq(N, d=f32(dx))
    live = (k * k - kk[None, :] ** 2 - kk[:, None] ** 2) > 0
    U0 = np.fft.fft2(u0.astype(np.complex128))
    kz = np.sqrt(np.where(live, k * k - kk[None, :] ** 2 - kk[:, None] ** 2, 0.0))
    expect = np.fft.ifft2(np.where(live, U0 * np.exp(-1j * f32(dz) * kz), 0.0))
    assert rel_l2(ub, expect) < 1e-12


# ---------------------------------------------------------------- N4 light sheet
def test_n4_light_sheet_focuses_to_its_gaussian_waist(oracle_mod):
    Nx, Ny, dx, lam, n0, NA = 8, 256, 0.2, 0.488, 1.33, 0.1
    zf = 25.6
    g = oracle_mod.lightsheet(Nx, Ny, dx, lam, n0, NA, zf)
    assert np.abs(g - g[:, :1]).max() == 0.0                      # flat in x
    w0 = f32(lam) / (np.pi * f32(NA))
    y = (np.arange(Ny) - Ny // 2) * f32(dx)
    waist = np.exp(-(y * y) / (w0 * w0))
    at_focus = oracle_mod.refocus(g, dx, zf, lam, n0)             # refocus is pinned by N1
    assert rel_l2(at_focus[:, 0], waist) < 1e-10                  # evanescent content of the waist ~ e^-600
    assert rel_l2(g[:, 0], waist) > 0.3                           # and it really was defocused
    # chained Algorithm-O steps do the same (128 steps of 0.2 um)
    u = g.copy()
    for _ in range(128):
        u, _ = oracle_mod.bpm_step(u, None, dx, 0.2, lam, n0)
    assert rel_l2(u[:, 0], waist) < 1e-5                          # 128 float32-rounded step lengths vs 25.6f


def test_n4_light_sheet_against_the_paraxial_cylindrical_beam(oracle_mod):
    Nx, Ny, dx, lam, n0, NA, zf = 4, 512, 0.2, 0.488, 1.33, 0.1, 25.6
    g = oracle_mod.lightsheet(Nx, Ny, dx, lam, n0, NA, zf)[:, 0]
    w0 = f32(lam) / (np.pi * f32(NA))
    zR = np.pi * w0 * w0 * f32(n0) / f32(lam)
    z = -f32(zf)
    y = (np.arange(Ny) - Ny // 2) * f32(dx)
    q = 1 + 1j * z / zR
    k = 2 * np.pi / f32(lam) * f32(n0)
    expect = np.exp(-(y * y) / (w0 * w0 * q)) / np.sqrt(q) * np.exp(1j * k * z)     # 1-D (cylindrical) Gaussian beam
    assert rel_l2(g, expect) < 3e-3
    assert rel_l2(g, np.conj(expect)) > 0.1


# ---------------------------------------------------------------- N5 annular pupil
def test_n5_annular_pupil_reduces_to_algorithm_m_and_has_annular_support(oracle_mod):
    N, dx, lam = 64, 0.2, 0.5
    rng = np.random.default_rng(9)
    pos = rng.uniform(-4, 4, size=(5, 2)).astype(F32)
    ph = rng.uniform(0, 2 * np.pi, size=5).astype(F32)
    am = rng.uniform(0.5, 1.5, size=5).astype(F32)
    a = oracle_mod.multiplex_annular(pos, ph, am, 0.0, 0.8, N, N, dx, lam)
    b = oracle_mod.multiplex_psf(pos, ph, am, 0.8, N, N, dx, lam)              # pinned by P11
    assert rel_l2(a, b) < 1e-13
    ring = oracle_mod.multiplex_annular(pos, ph, am, 0.5, 0.8, N, N, dx, lam)
    U = np.fft.fft2(ring)
    kk = 2 * np.pi * np.fft.fftfreq(N, d=f32(dx))
    k2 = kk[None, :] ** 2 + kk[:, None] ** 2
    k0 = 2 * np.pi / f32(lam)
    outside = (k2 > (k0 * f32(0.8)) ** 2) | (k2 < (k0 * f32(0.5)) ** 2)
    assert np.abs(U[outside]).max() < 1e-9 * np.abs(U).max()
    assert np.abs(U[~outside]).min() > 0


def test_n5_thin_annulus_is_a_bessel_beam(oracle_mod):
    from scipy.special import j0
    N, dx, lam = 512, 0.1, 0.5
    NA_in, NA_out = 0.59, 0.61
    u = oracle_mod.multiplex_annular(np.zeros((1, 2), dtype=F32), None, None, NA_in, NA_out, N, N, dx, lam)
    c = N // 2
    assert abs(u[c, c] - 1.0) < 1e-12                             # the normalisation of Algorithm M
    r = np.arange(0, 40) * f32(dx)
    k0 = 2 * np.pi / f32(lam)
    prof = u[c, c:c + 40].real
    assert np.abs(prof - j0(k0 * 0.6 * r)).max() < 3e-2           # finite ring width and pixelation (2 px wide ring)
    assert np.abs(prof - j0(k0 * 0.5 * r)).max() > 0.2            # the radius of the ring matters
    assert np.abs(u[c, c:c + 40].imag).max() < 1e-12


# ---------------------------------------------------------------- N6 image formation
def test_n6_delta_object_gives_the_tile_of_the_nearest_emitter(oracle_mod):
    rng = np.random.default_rng(12)
    Nx, Ny, dx, T = 32, 16, 0.5, 5
    pos = np.array([[-4.0, -2.0], [4.0, 2.0], [4.0, -2.0]], dtype=F32)
    psf = rng.uniform(0, 1, size=(3, T, T))
    for (sx, sy, owner) in [(8, 4, 0), (25, 12, 1), (23, 3, 2), (0, 0, 0)]:
        S = np.zeros((Ny, Nx))
        S[sy, sx] = 2.5
        # nearest emitter by brute force, periodic distance, lowest index on ties
        px, py = (sx - Nx // 2) * f32(dx), (sy - Ny // 2) * f32(dx)
        d = []
        for e in range(3):
            ddx = (px - float(pos[e, 0]) + Nx * f32(dx) / 2) % (Nx * f32(dx)) - Nx * f32(dx) / 2
            ddy = (py - float(pos[e, 1]) + Ny * f32(dx) / 2) % (Ny * f32(dx)) - Ny * f32(dx) / 2
            d.append(ddx * ddx + ddy * ddy)
        assert int(np.argmin(d)) == owner
        img = oracle_mod.image_formation(S, pos, dx, psf)
        expect = np.zeros((Ny, Nx))
        for ty in range(T):
            for tx in range(T):
                expect[(sy + ty - T // 2) % Ny, (sx + tx - T // 2) % Nx] = 2.5 * psf[owner, ty, tx]
        assert np.abs(img - expect).max() < 1e-15


def test_n6_single_emitter_is_a_plain_convolution_and_the_map_is_linear(oracle_mod):
    rng = np.random.default_rng(13)
    Nx, Ny, dx, T = 32, 32, 0.5, 7
    S1, S2 = rng.uniform(0, 1, size=(2, Ny, Nx))
    psf = rng.uniform(0, 1, size=(1, T, T))
    pos1 = np.zeros((1, 2), dtype=F32)
    img = oracle_mod.image_formation(S1, pos1, dx, psf)
    kern = np.zeros((Ny, Nx))
    for ty in range(T):
        for tx in range(T):
            kern[(ty - T // 2) % Ny, (tx - T // 2) % Nx] = psf[0, ty, tx]
    conv = np.fft.ifft2(np.fft.fft2(S1) * np.fft.fft2(kern)).real              # periodic convolution, numpy's FFT
    assert rel_l2(img, conv) < 1e-13
    pos4 = np.array([[-4, -4], [4, -4], [-4, 4], [4, 4]], dtype=F32)
    psf4 = rng.uniform(0, 1, size=(4, T, T))
    a = oracle_mod.image_formation(S1, pos4, dx, psf4)
    b = oracle_mod.image_formation(S2, pos4, dx, psf4)
    c = oracle_mod.image_formation(2 * S1 - 3 * S2, pos4, dx, psf4)
    assert rel_l2(c, 2 * a - 3 * b) < 1e-13
    # energy bookkeeping: every source pixel spreads S * sum(psf of its owner); owner by brute force
    yy, xx = np.mgrid[0:Ny, 0:Nx]
    L = Nx * f32(dx)
    d2 = []
    for e in range(4):
        ddx = ((xx - Nx // 2) * f32(dx) - float(pos4[e, 0]) + L / 2) % L - L / 2
        ddy = ((yy - Ny // 2) * f32(dx) - float(pos4[e, 1]) + L / 2) % L - L / 2
        d2.append(ddx * ddx + ddy * ddy)
    owner = np.argmin(np.stack(d2), axis=0)                       # first minimum = lowest index on ties
    assert abs(a.sum() - float((S1 * psf4.sum(axis=(1, 2))[owner]).sum())) < 1e-12 * a.sum()
