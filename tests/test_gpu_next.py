"""-m gpu: parity of the NEXT rows and of the 2048-point lines with the oracle,
through the C ABI: backward (phase-conjugate) propagation, homogeneous through-focus stacks, refocus,
PSF tile extraction, light-sheet and Bessel generators, image formation."""
import numpy as np
import pytest
import torch

from conftest import rel_l2
from gpu_common import need_gpu
from paper_1706_02261_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def small_tol(nz):
    return 2e-6 + 2.5e-7 * nz


def _case(Nx, Ny, Nz, B, seed=3):
    w = wl.tiny(N=Nx, Nz=Nz, n_cells=10, r_lo=0.5, r_hi=3.0)
    w = wl.dataclasses.replace(w, Ny=Ny)
    dn = wl.make_dn(w)
    f0 = wl.random_field(Nx, Ny, seed=seed + Nx + Ny, batch=B)
    return w, dn, f0


# ---------------------------------------------------------------- 2048-point lines (class radix 8)
@pytest.mark.parametrize("Nx,Ny,Nz,B", [(2048, 256, 2, 1), (256, 2048, 2, 1), (2048, 1024, 2, 1), (1024, 2048, 2, 1),
                                         (2048, 2048, 2, 1), (2048, 512, 3, 2)])
def test_2048_point_lines(oracle_mod, Nx, Ny, Nz, B):
    bb = need_gpu()
    w, dn, f0 = _case(Nx, Ny, Nz, B)
    nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, 1)
    d = torch.from_numpy(f0).cuda()
    I = torch.full((Nz, Ny, Nx), float("nan"), device="cuda")
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref)
    torch.cuda.synchronize()
    bb.device_status()
    Io = 0.0
    for b in range(B):
        uo, Ib = oracle_mod.propagate(f0[b], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert rel_l2(d[b].cpu().numpy(), uo) < small_tol(Nz)
        Io = Io + Ib
    assert rel_l2(I.cpu().numpy(), Io) < 2 * small_tol(Nz)


@pytest.mark.parametrize("Nx,Ny,B,per_field,Nz", [(2048, 1024, 2, False, 2), (1024, 2048, 3, True, 2),
                                                  # host runs of more than one z-chunk (chunks of 4 slices on these grids)
                                                  (2048, 1024, 2, False, 6), (2048, 1024, 2, True, 5)])
def test_batches_too_large_for_the_batch_kernel_run_field_by_field(oracle_mod, Nx, Ny, B, per_field, Nz):
    """ceil(Ny / SMs) * Nx > 8192: the batch variant cannot hold the screen factors of a CTA's rows; summed and
    per-field intensities, on top of existing contents (BB_ACCUMULATE).  The host-buffer entry point walks the
    fields inside its chunk loop (each dn chunk is uploaded once) and must give the same bits."""
    bb = need_gpu()
    w, dn, f0 = _case(Nx, Ny, Nz, B, seed=17)
    nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, 1)
    d = torch.from_numpy(f0).cuda()
    shape = ((B,) if per_field else ()) + (Nz, Ny, Nx)
    I0 = np.random.default_rng(1).uniform(0, 1, size=shape).astype(np.float32)
    I = torch.from_numpy(I0).cuda()
    flags = bb.ACCUMULATE | (bb.INTENSITY_PER_FIELD if per_field else 0)
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=flags)
    torch.cuda.synchronize()
    assert "false" in bb.last_kernel()                      # the single-field variant did the work
    Io = np.zeros((B, Nz, Ny, Nx))
    for b in range(B):
        uo, Io[b] = oracle_mod.propagate(f0[b], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert rel_l2(d[b].cpu().numpy(), uo) < small_tol(Nz)
    expect = (Io if per_field else Io.sum(axis=0)) + I0.astype(np.float64)
    assert rel_l2(I.cpu().numpy(), expect) < 2 * small_tol(Nz)
    # the host-buffer entry point takes the same route: bit-identical
    fh = torch.from_numpy(f0.copy()).pin_memory()
    Ih = torch.from_numpy(I0.copy()).pin_memory()
    bb.propagate(fh, dn.pin_memory(), w.dx, w.dz, w.lam, w.n0, intensity=Ih, nref=nref, flags=flags)
    assert torch.equal(fh, d.cpu()) and torch.equal(Ih, I.cpu())


@pytest.mark.parametrize("cfg", ["C2", "C3", "2048x512", "512x2048"])
def test_8_point_thread_kernel(oracle_mod, monkeypatch, cfg):
    """BB_USE_K8=1 routes propagations to the 8-point-thread kernel (otherwise it only runs the transform
    programs of 2048-point lines): every class radix, 1 .. 8."""
    bb = need_gpu()
    bb.shutdown()
    monkeypatch.setenv("BB_USE_K8", "1")
    try:
        if "x" in cfg:
            nx, ny = (int(v) for v in cfg.split("x"))
            w = wl.dataclasses.replace(wl.tiny(N=nx, Nz=6, n_cells=10, r_lo=0.5, r_hi=3.0), Ny=ny, nref_slab=2)
        else:
            w = wl.config(cfg).with_nz(6)
        dn = wl.make_dn(w)
        f0 = wl.random_field(w.Nx, w.Ny, seed=5, batch=1)
        nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, 2)
        d = torch.from_numpy(f0).cuda()
        I = torch.empty((6, w.Ny, w.Nx), device="cuda")
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref)
        torch.cuda.synchronize()
        assert "bpm8_kernel" in bb.last_kernel()
        uo, Io = oracle_mod.propagate(f0[0], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert rel_l2(d[0].cpu().numpy(), uo) < small_tol(6)
        assert rel_l2(I.cpu().numpy(), Io) < 2 * small_tol(6)
    finally:
        bb.shutdown()


# ---------------------------------------------------------------- NEXT-4 backward propagation
@pytest.mark.parametrize("Nx,Ny,Nz,B", [(64, 128, 7, 1), (128, 128, 5, 2), (256, 256, 9, 1), (512, 256, 6, 3),
                                         (1024, 1024, 3, 1), (2048, 256, 2, 1)])
def test_backward_matches_oracle(oracle_mod, Nx, Ny, Nz, B):
    bb = need_gpu()
    w, dn, f0 = _case(Nx, Ny, Nz, B, seed=9)
    nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, 2)
    d = torch.from_numpy(f0).cuda()
    I = torch.full((B, Nz, Ny, Nx), float("nan"), device="cuda")
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref,
                 flags=bb.BACKWARD | bb.INTENSITY_PER_FIELD)
    torch.cuda.synchronize()
    bb.device_status()
    for b in range(B):
        uo, Io = oracle_mod.propagate_backward(f0[b], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert rel_l2(d[b].cpu().numpy(), uo) < small_tol(Nz)
        assert rel_l2(I[b].cpu().numpy(), Io) < 2 * small_tol(Nz)


@pytest.mark.parametrize("N", [128, 256])
def test_forward_then_backward_recovers_the_input(N):
    """All-propagating grid (tests/test_oracle_bpm.py: dx = 0.3 um at lambda 0.5, n 1.33): the phase-conjugate
    run undoes the forward run to float32 rounding, and records the same planes."""
    bb = need_gpu()
    rng = np.random.default_rng(5)
    Nz, dx, dz, lam, n0 = 24, 0.3, 0.2, 0.5, 1.33
    u0 = (rng.standard_normal((1, N, N)) + 1j * rng.standard_normal((1, N, N))).astype(np.complex64)
    dn = torch.from_numpy(rng.uniform(0.0, 0.05, size=(Nz, N, N)).astype(np.float32)).cuda()
    nref = (np.float32(n0) + dn.mean(dim=(1, 2)).cpu().numpy()).astype(np.float32)
    d = torch.from_numpy(u0).cuda()
    If = torch.empty((Nz, N, N), device="cuda")
    Ib = torch.empty((Nz, N, N), device="cuda")
    bb.propagate(d, dn, dx, dz, lam, n0, intensity=If, nref=nref)
    assert rel_l2(d.cpu().numpy(), u0) > 0.5
    bb.propagate(d, dn, dx, dz, lam, n0, intensity=Ib, nref=nref, flags=bb.BACKWARD)
    torch.cuda.synchronize()
    assert rel_l2(d.cpu().numpy(), u0) < 2e-5
    assert rel_l2(Ib.cpu().numpy(), If.cpu().numpy()) < 4e-5


def test_backward_through_the_host_buffer_entry_point(oracle_mod):
    bb = need_gpu()
    w, dn, f0 = _case(256, 256, 40, 1, seed=2)          # 40 slices of 256 KiB: several chunks of the streaming pipeline? no: one
    w = wl.dataclasses.replace(w)                        # (chunking is exercised by the 1024^2 case below)
    nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, 8)
    fh = torch.from_numpy(f0.copy()).pin_memory()
    Ih = torch.empty((40, 256, 256), dtype=torch.float32).pin_memory()
    bb.propagate(fh, dn.pin_memory(), w.dx, w.dz, w.lam, w.n0, intensity=Ih, nref=nref, flags=bb.BACKWARD)
    d = torch.from_numpy(f0).cuda()
    I = torch.empty((40, 256, 256), device="cuda")
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=bb.BACKWARD)
    torch.cuda.synchronize()
    assert torch.equal(fh, d.cpu()) and torch.equal(Ih, I.cpu())
    # 1024^2: 8 slices per 32 MiB chunk -> 3 chunks, processed from the far end
    w, dn, f0 = _case(1024, 1024, 20, 1, seed=4)
    fh = torch.from_numpy(f0.copy()).pin_memory()
    Ih = torch.empty((20, 1024, 1024), dtype=torch.float32).pin_memory()
    bb.propagate(fh, dn.pin_memory(), w.dx, w.dz, w.lam, w.n0, intensity=Ih, flags=bb.BACKWARD)
    d = torch.from_numpy(f0).cuda()
    I = torch.empty((20, 1024, 1024), device="cuda")
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, flags=bb.BACKWARD)
    torch.cuda.synchronize()
    assert torch.equal(fh, d.cpu()) and torch.equal(Ih, I.cpu())


# ---------------------------------------------------------------- NEXT-1 refocus, through-focus stack, tiles
@pytest.mark.parametrize("Nx,Ny,B,dz", [(128, 64, 1, 3.7), (256, 256, 2, -12.8), (1024, 512, 1, -25.6), (512, 512, 3, 51.2),
                                         (2048, 256, 1, -6.4), (256, 256, 1, 0.0)])
def test_refocus_matches_oracle(oracle_mod, Nx, Ny, B, dz):
    bb = need_gpu()
    f0 = wl.random_field(Nx, Ny, seed=11 + Nx, batch=B)
    d = torch.from_numpy(f0).cuda()
    bb.refocus(d, 0.1, dz, 0.5, 1.33)
    torch.cuda.synchronize()
    for b in range(B):
        assert rel_l2(d[b].cpu().numpy(), oracle_mod.refocus(f0[b], 0.1, dz, 0.5, 1.33)) < 1e-6


@pytest.mark.parametrize("N,B", [(128, 1), (256, 2), (512, 1)])
def test_homogeneous_through_focus_stack(oracle_mod, N, B):
    bb = need_gpu()
    Nz, dx, dz, lam, n0 = 8, 0.2, 0.4, 0.5, 1.33
    f0 = wl.random_field(N, N, seed=N, batch=B)
    d = torch.from_numpy(f0).cuda()
    I = torch.full((Nz, N, N), float("nan"), device="cuda")
    bb.propagate(d, None, dx, dz, lam, n0, intensity=I, flags=bb.HOMOGENEOUS, nz=Nz)
    torch.cuda.synchronize()
    Io = np.zeros((Nz, N, N))
    for b in range(B):
        u = f0[b].astype(np.complex128)
        for j in range(Nz):
            u, Ij = oracle_mod.bpm_step(u, None, dx, dz, lam, n0)
            Io[j] += Ij
        assert rel_l2(d[b].cpu().numpy(), u) < small_tol(Nz)
    assert rel_l2(I.cpu().numpy(), Io) < 2 * small_tol(Nz)


def test_psf_tiles_of_a_refocused_multiplexed_field(oracle_mod):
    """C3's emitter grid (10 x 10, 8 um pitch) on a 512^2 field: propagate through a sample, refocus the exit
    field onto the emitter plane, cut the tiles -- each stage against the oracle; the gather itself bit-exact."""
    bb = need_gpu()
    w = wl.config("C3").with_nz(8)
    pos, ph, amp = wl.make_emitters(w)
    pos_d = torch.from_numpy(pos).cuda()
    u = bb.multiplex_psf(pos_d, torch.from_numpy(ph).cuda(), torch.from_numpy(amp).cuda(), w.NA, w.Nx, w.Ny, w.dx, w.lam)[None]
    dn = wl.make_dn(w)
    bb.propagate(u, dn.cuda(), w.dx, w.dz, w.lam, w.n0)
    exit_field = u.clone()
    bb.refocus(u, w.dx, -8 * w.dz, w.lam, w.n0)
    T = 32
    tiles = bb.extract_tiles(u, pos_d, w.dx, T)
    stack = torch.empty((5, w.Ny, w.Nx), device="cuda")
    v = exit_field.clone()
    bb.refocus(v, w.dx, -10 * w.dz, w.lam, w.n0)
    bb.propagate(v, None, w.dx, w.dz, w.lam, w.n0, intensity=stack, flags=bb.HOMOGENEOUS, nz=5)
    vol_tiles = bb.extract_tiles(stack, pos_d, w.dx, T)
    torch.cuda.synchronize()
    assert tiles.shape == (100, 1, T, T) and vol_tiles.shape == (100, 5, T, T)
    # the gathers: exactly the oracle's windows of the same arrays
    assert np.array_equal(tiles.cpu().numpy(), oracle_mod.extract_tiles(u[0].cpu().numpy(), pos, w.dx, T).astype(np.complex64))
    assert np.array_equal(vol_tiles.cpu().numpy(), oracle_mod.extract_tiles(stack.cpu().numpy(), pos, w.dx, T).astype(np.float32))
    # the chain: oracle from the same emitters
    uo = oracle_mod.multiplex_psf(pos, ph, amp, w.NA, w.Nx, w.Ny, w.dx, w.lam).astype(np.complex64)
    uo, _ = oracle_mod.propagate(uo, dn.numpy(), w.dx, w.dz, w.lam, w.n0, want_intensity=False)
    uo = oracle_mod.refocus(uo, w.dx, -8 * w.dz, w.lam, w.n0)
    assert rel_l2(tiles.cpu().numpy(), oracle_mod.extract_tiles(uo, pos, w.dx, T)) < 1e-5
    # every refocused emitter image peaks inside its tile, near the centre
    t = np.abs(tiles.cpu().numpy()[:, 0])
    peak = np.array([np.unravel_index(np.argmax(a), a.shape) for a in t])
    assert np.abs(peak - T // 2).max() <= 2


# ---------------------------------------------------------------- NEXT-2 illumination generators
@pytest.mark.parametrize("Nx,Ny,dx,lam,NA,zf", [(256, 256, 0.2, 0.488, 0.1, 25.6), (128, 512, 0.1, 0.5, 0.3, 10.0),
                                                 (512, 256, 0.2, 0.5, 0.2, 0.0), (256, 1024, 0.1, 0.5, 0.15, -20.0)])
def test_lightsheet_matches_oracle(oracle_mod, Nx, Ny, dx, lam, NA, zf):
    bb = need_gpu()
    g = bb.lightsheet(Nx, Ny, dx, lam, 1.33, NA, zf)
    torch.cuda.synchronize()
    assert rel_l2(g.cpu().numpy(), oracle_mod.lightsheet(Nx, Ny, dx, lam, 1.33, NA, zf)) < 2e-6


@pytest.mark.parametrize("N,NA_in,NA,M", [(256, 0.55, 0.6, 1), (512, 0.4, 0.8, 7), (256, 0.0, 0.8, 5)])
def test_bessel_lattice_matches_oracle(oracle_mod, N, NA_in, NA, M):
    bb = need_gpu()
    dx, lam = 0.1, 0.5
    rng = np.random.default_rng(N + M)
    pos = np.stack([(np.arange(M) - (M - 1) / 2) * 2.37, rng.uniform(-1, 1, M)], axis=1).astype(np.float32)
    ph = rng.uniform(0, 2 * np.pi, M).astype(np.float32)
    u = bb.multiplex_annular(torch.from_numpy(pos).cuda(), torch.from_numpy(ph).cuda(), None, NA_in, NA, N, N, dx, lam)
    torch.cuda.synchronize()
    assert rel_l2(u.cpu().numpy(), oracle_mod.multiplex_annular(pos, ph, None, NA_in, NA, N, N, dx, lam)) < 2e-6


# ---------------------------------------------------------------- NEXT-3 image formation
@pytest.mark.parametrize("Nx,Ny,T,G", [(64, 32, 5, 2), (256, 256, 16, 4), (512, 512, 32, 10), (128, 256, 9, 3),
                                       # the kernel's other paths: more emitters in a CTA's halo than it stages (cells of
                                       # 8 px under 16-px tiles: ~28 owners > 16 slots), more than its 64-entry owner set
                                       # holds (cells of 4 px: ~72 owners), tiles above the 48 KB default shared memory
                                       # (T = 64: 6 staged tiles, 152 KB), and T = 96 (one slot: every mixed halo gathers)
                                       (256, 256, 16, 32), (256, 256, 16, 64), (256, 256, 64, 2), (256, 128, 96, 3)])
def test_image_formation_matches_oracle(oracle_mod, Nx, Ny, T, G):
    bb = need_gpu()
    rng = np.random.default_rng(T + G)
    dx = 0.2
    gx = (np.arange(G) - (G - 1) / 2) * (Nx * dx / G)
    gy = (np.arange(G) - (G - 1) / 2) * (Ny * dx / G)
    pos = np.stack(np.meshgrid(gx, gy), axis=-1).reshape(-1, 2).astype(np.float32)
    psf = rng.uniform(0, 1, size=(G * G, T, T)).astype(np.float32)
    S = rng.uniform(0, 1, size=(Ny, Nx)).astype(np.float32)
    img = bb.image_formation(torch.from_numpy(S).cuda(), torch.from_numpy(pos).cuda(), dx, torch.from_numpy(psf).cuda())
    torch.cuda.synchronize()
    assert rel_l2(img.cpu().numpy(), oracle_mod.image_formation(S, pos, dx, psf)) < 2e-6
    # a delta object on a cell boundary: the nearest-emitter decision (ties included) must be the oracle's
    S0 = np.zeros((Ny, Nx), dtype=np.float32)
    S0[Ny // 2, Nx // 2] = 1.0
    S0[0, 0] = 2.0
    img = bb.image_formation(torch.from_numpy(S0).cuda(), torch.from_numpy(pos).cuda(), dx, torch.from_numpy(psf).cuda())
    assert np.array_equal(img.cpu().numpy(), oracle_mod.image_formation(S0, pos, dx, psf).astype(np.float32))


def test_next_rows_argument_checks():
    bb = need_gpu()
    f = torch.zeros((1, 256, 256), dtype=torch.complex64, device="cuda")
    with pytest.raises(bb.BBError) as e:
        bb.refocus(f, 0.1, float("nan"), 0.5, 1.33)
    assert e.value.status == 1
    with pytest.raises(bb.BBError) as e:
        bb.propagate(f, None, 0.1, 0.1, 0.5, 1.33, flags=bb.HOMOGENEOUS, nz=2, nref=[1.33, 1.33])
    assert e.value.status == 1
    with pytest.raises(bb.BBError) as e:
        bb.extract_tiles(torch.zeros((1, 16, 16), device="cuda"), torch.zeros((1, 2), device="cuda"), 0.1, 17)
    assert e.value.status == 1
    with pytest.raises(bb.BBError) as e:
        bb.multiplex_annular(torch.zeros((1, 2), device="cuda"), None, None, 0.9, 0.8, 256, 256, 0.1, 0.5)
    assert e.value.status == 1
    g = torch.zeros((1, 2048, 128), dtype=torch.complex64, device="cuda")
    with pytest.raises(bb.BBError) as e:
        bb.refocus(g, 0.1, 1.0, 0.5, 1.33)
    assert e.value.status == 2
