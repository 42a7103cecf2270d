"""-m gpu: the building blocks of the CUDA path against the oracle, each on its own
(SURVEY section 4 tier T1): 2-D FFT, propagator table, multiplexed input field, n_ref helper."""
import numpy as np
import pytest
import torch

from conftest import rel_l2
from gpu_common import need_gpu
from paper_1706_02261_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# one 2-D complex64 FFT against the double oracle: rounding of ~log2(N) butterfly levels
FFT_TOL = 5e-7


@pytest.mark.parametrize("Nx,Ny,B", [(32, 32, 1), (64, 32, 3), (32, 128, 2), (128, 128, 1), (256, 64, 2),
                                      (512, 256, 1), (256, 512, 2), (1024, 128, 1), (128, 1024, 1),
                                      (512, 512, 5), (1024, 1024, 2),
                                      (2048, 1024, 1), (1024, 2048, 1), (2048, 2048, 1), (2048, 256, 2), (256, 2048, 1)])
def test_fft2_matches_oracle(oracle_mod, Nx, Ny, B):
    bb = need_gpu()
    f = wl.random_field(Nx, Ny, seed=Nx * 7 + Ny, batch=B)
    d = torch.from_numpy(f).cuda()
    bb.fft2(d, -1)
    torch.cuda.synchronize()
    bb.device_status()
    got = d.cpu().numpy()
    for b in range(B):
        assert rel_l2(got[b], oracle_mod.fft2(f[b], -1)) < FFT_TOL
    d2 = torch.from_numpy(f).cuda()
    bb.fft2(d2, +1)
    got = d2.cpu().numpy()
    for b in range(B):
        assert rel_l2(got[b], oracle_mod.fft2(f[b], +1)) < FFT_TOL
    bb.fft2(d, +1)                    # inverse of the forward result: back to the input
    assert rel_l2(d.cpu().numpy(), f) < 2 * FFT_TOL


def test_fft2_of_a_delta_and_a_plane_wave():
    """Closed forms, independent of the oracle: delta -> ones; plane wave -> one bin."""
    bb = need_gpu()
    Nx, Ny = 256, 128
    d = torch.zeros((Ny, Nx), dtype=torch.complex64, device="cuda")
    d[0, 0] = 1.0
    bb.fft2(d, -1)
    assert torch.allclose(d, torch.ones_like(d), atol=1e-6)
    y, x = np.mgrid[0:Ny, 0:Nx]
    p, q = 37, -11
    pw = np.exp(2j * np.pi * (p * x / Nx + q * y / Ny)).astype(np.complex64)
    d = torch.from_numpy(pw).cuda()
    bb.fft2(d, -1)
    got = d.cpu().numpy()
    expect = np.zeros_like(got)
    expect[q % Ny, p % Nx] = Nx * Ny
    assert np.abs(got - expect).max() < 2e-6 * Nx * Ny


@pytest.mark.parametrize("Nx,Ny,dx,dz,lam,nref", [(128, 128, 0.1, 0.1, 0.5, 1.33), (256, 64, 0.2, 0.2, 0.488, 1.3412),
                                                   (512, 512, 0.2, 0.2, 0.5, 1.35), (1024, 1024, 0.1, 0.1, 0.5, 1.3372)])
def test_propagator_table(oracle_mod, Nx, Ny, dx, dz, lam, nref):
    """H = spectrum of one oracle step applied to a delta (dn = 0): the cut-off pattern must be
    identical (a decision taken in double on both sides), values equal to float32 rounding."""
    bb = need_gpu()
    delta = np.zeros((Ny, Nx), dtype=np.complex128)
    delta[0, 0] = 1.0
    u1, _ = oracle_mod.bpm_step(delta, None, dx, dz, lam, 1.33, nref=nref, want_intensity=False)
    # undo the homogeneous screen exp(i k0 dz (n0 - nref)) the step applies after the propagator
    k0 = 2 * np.pi / float(np.float32(lam))
    u1 = u1 * np.exp(-1j * k0 * float(np.float32(dz)) * (float(np.float32(1.33)) - float(np.float32(nref))))
    H = oracle_mod.fft2(u1, -1)
    got = bb.propagator_table(Nx, Ny, dx, dz, lam, nref).cpu().numpy().astype(np.complex128) * (Nx * Ny)
    evan = np.abs(H) < 0.5
    assert np.array_equal(got == 0, evan)
    assert 0 < evan.sum() < evan.size or dx > 0.25
    assert np.abs(got - H).max() < 1.5e-7
    assert np.abs(np.abs(got[~evan]) - 1).max() < 1.5e-7


@pytest.mark.parametrize("cfg", ["C3", "C4"])
def test_multiplex_psf_matches_oracle(oracle_mod, cfg):
    bb = need_gpu()
    w = wl.config(cfg)
    pos, ph, amp = wl.make_emitters(w)
    ref = oracle_mod.multiplex_psf(pos, ph, amp, w.NA, w.Nx, w.Ny, w.dx, w.lam)
    got = bb.multiplex_psf(torch.from_numpy(pos).cuda(), torch.from_numpy(ph).cuda(), torch.from_numpy(amp).cuda(),
                           w.NA, w.Nx, w.Ny, w.dx, w.lam)
    bb.device_status()
    assert rel_l2(got.cpu().numpy(), ref) < 2e-6
    # band limit: nothing outside the NA disk (exact zeros were transformed; allow FFT rounding)
    spec = got.clone()
    bb.fft2(spec, -1)
    k = 2 * np.pi * np.fft.fftfreq(w.Nx, d=float(np.float32(w.dx)))
    outside = (k[None, :] ** 2 + k[:, None] ** 2) > (2 * np.pi / float(np.float32(w.lam)) * float(np.float32(w.NA))) ** 2
    s = spec.cpu().numpy()
    assert np.abs(s[outside]).max() < 1e-5 * np.abs(s).max()


def test_multiplex_psf_defaults_subpixel_and_nonsquare(oracle_mod):
    bb = need_gpu()
    rng = np.random.default_rng(5)
    pos = rng.uniform(-5, 5, size=(7, 2)).astype(np.float32)      # off-grid positions
    ref = oracle_mod.multiplex_psf(pos, None, None, 0.6, 256, 128, 0.15, 0.5)
    got = bb.multiplex_psf(torch.from_numpy(pos).cuda(), None, None, 0.6, 256, 128, 0.15, 0.5)
    assert rel_l2(got.cpu().numpy(), ref) < 2e-6
    # the paper's own lateral grid (1024 x 2048): 2048-point lines
    ref = oracle_mod.multiplex_psf(pos, None, None, 0.8, 2048, 1024, 0.1, 0.5)
    got = bb.multiplex_psf(torch.from_numpy(pos).cuda(), None, None, 0.8, 2048, 1024, 0.1, 0.5)
    assert rel_l2(got.cpu().numpy(), ref) < 2e-6
    one = np.zeros((1, 2), dtype=np.float32)                      # on-grid unit emitter: value 1 at its pixel
    got = bb.multiplex_psf(torch.from_numpy(one).cuda(), None, None, 0.8, 128, 128, 0.1, 0.5).cpu().numpy()
    assert abs(got[64, 64] - 1.0) < 1e-5


@pytest.mark.parametrize("slab", [1, 5, 32, 1000])
def test_nref_from_dn(oracle_mod, slab):
    bb = need_gpu()
    w = wl.config("C1").with_nz(70)
    dn = wl.make_dn(w)
    ref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, slab)
    got = bb.nref_from_dn(dn.cuda(), w.n0, slab).numpy()
    # means are taken in double on both sides (different summation order): equal to 1 float32 ulp
    assert np.abs(got.astype(np.float64) - ref.astype(np.float64)).max() <= 1.2e-7 * 1.4
    const = torch.full((6, 64, 32), 0.02, device="cuda")
    assert np.array_equal(bb.nref_from_dn(const, 1.33, 4).numpy(),
                          np.full(6, np.float32(np.float64(np.float32(1.33)) + np.float64(np.float32(0.02)))))


def test_a_misspelt_environment_switch_is_rejected(monkeypatch):
    """The diagnostic BB_* switches are read when a plan is made; a BB_* name the library does not know fails
    the call (it would otherwise be ignored silently), and the message names it."""
    bb = need_gpu()
    bb.shutdown()
    monkeypatch.setenv("BB_DISABLE_K61", "1")
    f = torch.zeros((1, 256, 256), dtype=torch.complex64, device="cuda")
    with pytest.raises(bb.BBError) as e:
        bb.fft2(f, -1)
    assert e.value.status == 1 and "BB_DISABLE_K61" in str(e.value)
    monkeypatch.delenv("BB_DISABLE_K61")
    bb.fft2(f, -1)
    torch.cuda.synchronize()
    bb.shutdown()
