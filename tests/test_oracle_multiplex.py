"""Pin P11 for Algorithm M (oracle_multiplex_psf) and P9's multiplexing premise.

Expected values come from: a brute-force direct sum over the pupil written here in numpy;
symmetry / normalisation facts (on-grid unit emitter has value 1 at its own pixel, real and
symmetric about it; spectrum exactly zero outside the NA disk); the Airy amplitude
2 J1(v)/v on a fine grid; and the paper's premise that a multiplexed run
equals the sum of single-emitter runs, checked by brute force through Algorithm O.
"""
import numpy as np
import pytest

from conftest import rel_l2
from paper_1706_02261_b200 import workloads as wl

F32 = np.float32


def f32(x):
    return float(np.float32(x))


def direct_sum(pos, phase, amp, NA, Nx, Ny, dx, lam):
    """u0(r) = (1/|P|) sum_{k in P} sum_e a_e exp(i phi_e) exp(i k.(r - r_e)), brute force."""
    dx, lam, NA = f32(dx), f32(lam), f32(NA)
    kx = 2 * np.pi * np.fft.fftfreq(Nx, d=dx)
    ky = 2 * np.pi * np.fft.fftfreq(Ny, d=dx)
    KX, KY = np.meshgrid(kx, ky, indexing="xy")
    P = (KX ** 2 + KY ** 2) <= (2 * np.pi / lam * NA) ** 2
    ks = np.stack([KX[P], KY[P]], axis=1)                       # [|P|][2]
    xs = (np.arange(Nx) - Nx // 2) * dx
    ys = (np.arange(Ny) - Ny // 2) * dx
    out = np.zeros((Ny, Nx), dtype=np.complex128)
    for e in range(pos.shape[0]):
        xe, ye = float(pos[e, 0]), float(pos[e, 1])
        ph = 0.0 if phase is None else float(phase[e])
        a = 1.0 if amp is None else float(amp[e])
        ex = np.exp(1j * np.outer(ks[:, 0], xs - xe))           # [|P|][Nx]
        ey = np.exp(1j * np.outer(ks[:, 1], ys - ye))           # [|P|][Ny]
        out += a * np.exp(1j * ph) * np.einsum("ky,kx->yx", ey, ex)
    return out / P.sum(), P


def test_single_on_grid_emitter(oracle_mod):
    N, dx, lam, NA = 32, 0.2, 0.5, 0.8
    pos = np.array([[3 * f32(dx), -2 * f32(dx)]], dtype=F32)    # exactly on pixel (N/2+3, N/2-2)
    u = oracle_mod.multiplex_psf(pos, None, None, NA, N, N, dx, lam)
    cy, cx = N // 2 - 2, N // 2 + 3
    assert abs(u[cy, cx] - 1.0) < 1e-6          # float32 position -> ~1e-7 of a pixel off-grid
    assert np.abs(u).max() <= abs(u[cy, cx]) + 1e-12
    # symmetric about the emitter, real up to the sub-pixel residual
    for d in (1, 2, 5):
        assert abs(u[cy, cx + d] - u[cy, cx - d]) < 1e-6
        assert abs(u[cy + d, cx] - u[cy - d, cx]) < 1e-6
    assert np.abs(u.imag).max() < 1e-6
    # spectrum exactly zero outside the NA disk (numpy FFT as the independent transform)
    U = np.fft.fft2(u)
    k = 2 * np.pi * np.fft.fftfreq(N, d=f32(dx))
    outside = (k[None, :] ** 2 + k[:, None] ** 2) > (2 * np.pi / f32(lam) * f32(NA)) ** 2
    assert np.abs(U[outside]).max() < 1e-10 * np.abs(U).max()
    inside_mod = np.abs(U[~outside])
    assert np.allclose(inside_mod, inside_mod[0], rtol=1e-10)   # uniform pupil, no apodisation


def test_subpixel_emitters_vs_direct_sum(oracle_mod):
    Nx, Ny, dx, lam, NA = 16, 16, 0.2, 0.5, 0.8
    rng = np.random.default_rng(3)
    pos = rng.uniform(-1.0, 1.0, size=(3, 2)).astype(F32)
    phase = rng.uniform(0, 2 * np.pi, size=(3,)).astype(F32)
    amp = rng.uniform(0.5, 2.0, size=(3,)).astype(F32)
    u = oracle_mod.multiplex_psf(pos, phase, amp, NA, Nx, Ny, dx, lam)
    ref, P = direct_sum(pos, phase, amp, NA, Nx, Ny, dx, lam)
    assert 4 < P.sum() < Nx * Ny
    assert rel_l2(u, ref) < 1e-12


def test_non_square_subpixel_vs_direct_sum(oracle_mod):
    Nx, Ny, dx, lam, NA = 32, 16, 0.25, 0.5, 0.6
    pos = np.array([[0.37, -0.81], [-2.2, 0.4]], dtype=F32)
    phase = np.array([0.3, 2.1], dtype=F32)
    u = oracle_mod.multiplex_psf(pos, phase, None, NA, Nx, Ny, dx, lam)
    ref, _ = direct_sum(pos, phase, None, NA, Nx, Ny, dx, lam)
    assert rel_l2(u, ref) < 1e-12


def test_airy_amplitude_on_fine_grid(oracle_mod):
    """Radial profile of one emitter -> 2 J1(v)/v, v = k0 NA r (pupil-edge pixelation ~2e-3)."""
    from scipy.special import j1
    N, dx, lam, NA = 1024, 0.02, 0.5, 0.8
    u = oracle_mod.multiplex_psf(np.zeros((1, 2), dtype=F32), None, None, NA, N, N, dx, lam)
    c = N // 2
    r = np.arange(1, 120) * f32(dx)
    v = 2 * np.pi / f32(lam) * f32(NA) * r
    airy = 2 * j1(v) / v
    assert np.abs(u[c, c + 1:c + 120].real - airy).max() < 5e-3
    assert np.abs(u[c + 1:c + 120, c].real - airy).max() < 5e-3
    assert abs(u[c, c] - 1.0) < 1e-12


def test_p9_multiplexed_run_equals_sum_of_single_runs(oracle_mod):
    """The paper's premise: independent PSFs can be calculated in one
    multiplexed simulation.  Brute force on 32 x 32 x 16 with 4 emitters."""
    w = wl.tiny(N=32, Nz=16)
    dn = wl.make_dn(w).numpy()
    nref = (F32(w.n0) + dn.reshape(w.Nz, -1).mean(axis=1)).astype(F32)
    pos = np.array([[-1.6, -1.6], [1.6, -1.6], [-1.6, 1.6], [1.7, 1.5]], dtype=F32)
    phase = np.array([0.1, 1.3, 2.9, 4.4], dtype=F32)
    NA = 0.8

    def run(u0):
        u = u0.copy()
        for j in range(w.Nz):
            u, _ = oracle_mod.bpm_step(u, dn[j], w.dx, w.dz, w.lam, w.n0, nref[j])
        return u

    multi = run(oracle_mod.multiplex_psf(pos, phase, None, NA, w.Nx, w.Ny, w.dx, w.lam))
    singles = sum(run(oracle_mod.multiplex_psf(pos[e:e + 1], phase[e:e + 1], None, NA,
                                               w.Nx, w.Ny, w.dx, w.lam)) for e in range(4))
    assert rel_l2(multi, singles) < 1e-12


def test_workload_emitter_grids():
    for name, M in (("C3", 100), ("C4", 1024)):
        w = wl.config(name)
        pos, phase, amp = wl.make_emitters(w)
        assert pos.shape == (M, 2) and phase.shape == (M,) and np.all(amp == 1)
        assert abs(pos.mean()) < 1e-5
        L = w.Nx * w.dx
        assert np.abs(pos).max() < L / 2
        assert 0 <= phase.min() and phase.max() < 2 * np.pi + 1e-6
    # C4's grid tiles the field periodically: spacing * emitters == L
    w = wl.config("C4")
    assert abs(w.spacing * w.emitters - w.Nx * w.dx) < 1e-9
