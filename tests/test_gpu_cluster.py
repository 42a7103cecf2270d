"""-m gpu: the cluster kernel for small grids (csrc/bb_kernelsc.cuh; the field
resident in the distributed shared memory of one thread-block cluster) against the oracle, through
the C ABI: every shape it serves, both cluster sizes, both exchange forms, both thread forms, the
flags, batches, chunked host runs, and the dispatch rule."""
import numpy as np
import pytest
import torch

from conftest import rel_l2
from gpu_common import need_gpu
from paper_1706_02261_b200 import workloads as wl
from test_gpu_bpm import run_both, small_tol

pytestmark = pytest.mark.gpu

KC_ENV = ("BB_DISABLE_KC", "BB_KC_CS", "BB_KC_MODE", "BB_KC_PT", "BB_KC_FORCE")


@pytest.fixture
def kc_env(monkeypatch):
    """Sets the diagnostic switches of the cluster kernel for one test (they are read when a plan is made)."""
    bb = need_gpu()

    def set_env(**kw):
        for k in KC_ENV:
            monkeypatch.delenv(k, raising=False)
        for k, v in kw.items():
            monkeypatch.setenv(k, str(v))
        bb.shutdown()
        return bb

    yield set_env
    for k in KC_ENV:
        monkeypatch.delenv(k, raising=False)
    bb.shutdown()


def problem(oracle_mod, Nx, Ny, Nz, B, seed=5, slab=2):
    w = wl.tiny(N=Nx, Nz=Nz, n_cells=10, r_lo=0.5, r_hi=3.0)
    w = wl.dataclasses.replace(w, Ny=Ny)
    dn = wl.make_dn(w)
    f0 = wl.random_field(Nx, Ny, seed=seed, batch=B)
    nref = oracle_mod.nref_from_dn(dn.numpy(), w.n0, slab)
    return w, dn, f0, nref


@pytest.mark.parametrize("Nx,Ny", [(128, 128), (256, 128), (128, 256), (256, 256)])
@pytest.mark.parametrize("cs", [16, 8])
@pytest.mark.parametrize("mode", [1, 0])
def test_every_shape_cluster_size_and_exchange_form(oracle_mod, kc_env, Nx, Ny, cs, mode):
    """Bulk copies counted on mbarriers (mode 1, the default) and plain remote stores between cluster
    barriers (mode 0); clusters of 16 (non-portable size) and 8 CTAs.  256 x 256 does not fit 8 CTAs:
    the library must then fall back to the grid kernel and still be right."""
    bb = kc_env(BB_KC_CS=cs, BB_KC_MODE=mode, BB_KC_FORCE=1)
    Nz = 9
    w, dn, f0, nref = problem(oracle_mod, Nx, Ny, Nz, 1, seed=Nx + 2 * Ny + cs)
    u, I, uo, Io = run_both(bb, oracle_mod, w, dn, f0, nref)
    name = bb.last_kernel()
    if (Nx, Ny, cs) == (256, 256, 8):
        assert "bpm16_kernel" in name
    else:
        assert name == "bb::bpmc_kernel<%d,%d,%d,%d,%d>" % (Nx, Ny, cs, mode, 16 if (Nx, Ny) == (256, 256) else 8)
    assert rel_l2(u[0], uo[0]) < small_tol(Nz)
    assert rel_l2(I, Io) < 2 * small_tol(Nz)


def test_dispatch_rule(oracle_mod, kc_env):
    """A 128-point side: cluster kernel.  256 x 256: the 16-point-thread grid kernel unless forced.
    Anything else: never.  BB_DISABLE_KC: the grid kernels everywhere (and they still agree with the oracle)."""
    bb = kc_env()
    seen = {}
    for Nx, Ny in [(128, 128), (256, 128), (128, 256), (256, 256), (64, 128), (512, 128)]:
        w, dn, f0, nref = problem(oracle_mod, Nx, Ny, 2, 1)
        d = torch.from_numpy(f0.copy()).cuda()
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        seen[(Nx, Ny)] = bb.last_kernel()
    for shape in [(128, 128), (256, 128), (128, 256)]:
        assert "bpmc_kernel" in seen[shape], seen
    for shape in [(256, 256), (64, 128), (512, 128)]:
        assert "bpmc_kernel" not in seen[shape], seen
    bb = kc_env(BB_DISABLE_KC=1)
    Nz = 6
    w, dn, f0, nref = problem(oracle_mod, 128, 128, Nz, 2)
    u, I, uo, Io = run_both(bb, oracle_mod, w, dn, f0, nref)
    assert "bpm_kernel" in bb.last_kernel()
    assert rel_l2(u[1], uo[1]) < small_tol(Nz) and rel_l2(I, Io) < 2 * small_tol(Nz)


def test_16_point_threads_reproduce_the_grid_kernel_bit_for_bit(oracle_mod, kc_env):
    """On 256 x 256 the cluster kernel with 16-point threads does the arithmetic of the 16-point-thread
    grid kernel in the same order: identical bits, field and intensity; the 8-point form agrees to rounding."""
    Nz = 12
    w, dn, f0, nref = problem(oracle_mod, 256, 256, Nz, 1, seed=77)
    out = {}
    for key, env in (("grid", dict(BB_DISABLE_KC=1)), ("c16", dict(BB_KC_FORCE=1)), ("c8", dict(BB_KC_FORCE=1, BB_KC_PT=8))):
        bb = kc_env(**env)
        d = torch.from_numpy(f0.copy()).cuda()
        I = torch.empty(dn.shape, device="cuda")
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref)
        out[key] = (d.cpu(), I.cpu(), bb.last_kernel())
    assert "bpm16_kernel" in out["grid"][2] and out["c16"][2].endswith(",16>") and out["c8"][2].endswith(",8>")
    assert torch.equal(out["grid"][0], out["c16"][0]) and torch.equal(out["grid"][1], out["c16"][1])
    assert rel_l2(out["c8"][0].numpy(), out["grid"][0].numpy().astype(np.complex128)) < 1e-5


@pytest.mark.parametrize("Nx,Ny", [(128, 128), (256, 128)])
@pytest.mark.parametrize("inten", ["summed", "per_field", "accumulate", "none"])
def test_batches_one_cluster_per_field(oracle_mod, kc_env, Nx, Ny, inten):
    """21 fields (more clusters than the device holds at once).  Summed intensity: the clusters add into
    slices the library has zeroed (atomics: tolerance, bb.h); per-field volumes; BB_ACCUMULATE on top of
    existing contents; no intensity at all."""
    bb = kc_env()
    Nz, B = 5, 21
    w, dn, f0, nref = problem(oracle_mod, Nx, Ny, Nz, B, seed=31)
    if inten == "none":
        d = torch.from_numpy(f0.copy()).cuda()
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert "bpmc_kernel" in bb.last_kernel()
        for b in (0, 7, 20):
            uo, _ = oracle_mod.propagate(f0[b], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
            assert rel_l2(d[b].cpu().numpy(), uo) < small_tol(Nz)
        return
    flags = {"summed": 0, "per_field": bb.INTENSITY_PER_FIELD, "accumulate": bb.ACCUMULATE}[inten]
    init = np.random.default_rng(3).uniform(0, 5, size=tuple(dn.shape)) if inten == "accumulate" else None
    u, I, uo, Io = run_both(bb, oracle_mod, w, dn, f0, nref, flags=flags, intensity_init=init)
    assert "bpmc_kernel" in bb.last_kernel()
    for b in range(B):
        assert rel_l2(u[b], uo[b]) < small_tol(Nz)
    assert rel_l2(I, Io) < 2 * small_tol(Nz)
    assert not np.isnan(I).any()


@pytest.mark.parametrize("flag", ["backward", "per_phase", "homogeneous"])
def test_flags_on_the_cluster_kernel(oracle_mod, kc_env, flag):
    bb = kc_env()
    Nz = 7
    w, dn, f0, nref = problem(oracle_mod, 128, 256, Nz, 1, seed=13)
    d = torch.from_numpy(f0.copy()).cuda()
    I = torch.empty(dn.shape, device="cuda")
    if flag == "backward":
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=bb.BACKWARD)
        uo, Io = oracle_mod.propagate_backward(f0[0], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
    elif flag == "per_phase":
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=bb.LAUNCH_PER_PHASE)
        uo, Io = oracle_mod.propagate(f0[0], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
    else:
        bb.propagate(d, None, w.dx, w.dz, w.lam, w.n0, intensity=I, flags=bb.HOMOGENEOUS, nz=Nz)
        uo, Io = oracle_mod.propagate(f0[0], np.zeros(dn.shape, np.float32), w.dx, w.dz, w.lam, w.n0)
    assert "bpmc_kernel" in bb.last_kernel()
    assert rel_l2(d.cpu().numpy()[0], uo) < small_tol(Nz)
    assert rel_l2(I.cpu().numpy(), Io) < 2 * small_tol(Nz)


def test_forward_then_backward_returns_the_input(kc_env):
    """All-propagating grid (dx > lambda / 2n: no mode is cut), so the phase-conjugate run undoes the forward one."""
    bb = kc_env()
    w = wl.tiny(N=128, Nz=40, n_cells=10, r_lo=0.5, r_hi=3.0)
    w = wl.dataclasses.replace(w, dx=0.3, dz=0.3)
    dn = wl.make_dn(w).cuda()
    f0 = wl.random_field(w.Nx, w.Ny, seed=4, batch=1)
    d = torch.from_numpy(f0.copy()).cuda()
    bb.propagate(d, dn, w.dx, w.dz, w.lam, w.n0)
    assert rel_l2(d.cpu().numpy(), f0) > 0.1
    bb.propagate(d, dn, w.dx, w.dz, w.lam, w.n0, flags=bb.BACKWARD)
    assert rel_l2(d.cpu().numpy(), f0) < 2e-5


@pytest.mark.parametrize("backward", [False, True])
def test_host_buffers_in_several_chunks(oracle_mod, kc_env, backward):
    """bb_propagate_host cuts 128^2 x 1100 slices into chunks of 512: every launch but the first starts from the
    field in global memory half way through a step, every launch but the last leaves it there (forward: launches
    start and end on row phases; backward: they end on column phases).  Same bits as the one-launch device run."""
    bb = kc_env()
    Nz = 1100
    w, dn, f0, nref = problem(oracle_mod, 128, 128, Nz, 1, seed=2, slab=64)
    flags = bb.BACKWARD if backward else 0
    d = torch.from_numpy(f0.copy()).cuda()
    I = torch.empty(dn.shape, device="cuda")
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=flags)
    assert "bpmc_kernel" in bb.last_kernel()
    fh = torch.from_numpy(f0.copy()).pin_memory()
    Ih = torch.empty(dn.shape).pin_memory()
    bb.propagate(fh, dn.pin_memory(), w.dx, w.dz, w.lam, w.n0, intensity=Ih, nref=nref, flags=flags)
    assert torch.equal(fh, d.cpu()) and torch.equal(Ih, I.cpu())
    ofn = oracle_mod.propagate_backward if backward else oracle_mod.propagate
    uo, Io = ofn(f0[0], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
    assert rel_l2(fh.numpy()[0], uo) < 1e-4 and rel_l2(Ih.numpy(), Io) < 1e-4


def test_repeated_runs_are_bit_identical(kc_env):
    bb = kc_env()
    w = wl.config("C1")
    dn = wl.make_dn(w).cuda()
    f0 = torch.from_numpy(wl.make_field(w)).cuda()
    outs = []
    for _ in range(3):
        d = f0.clone()
        I = torch.empty(dn.shape, device="cuda")
        bb.propagate(d, dn, w.dx, w.dz, w.lam, w.n0, intensity=I)
        outs.append((d.cpu(), I.cpu()))
    assert "bpmc_kernel" in bb.last_kernel()
    for d, I in outs[1:]:
        assert torch.equal(d, outs[0][0]) and torch.equal(I, outs[0][1])


def test_summed_intensity_of_a_large_batch_with_a_wide_dynamic_range(oracle_mod, kc_env):
    """64 clusters add their |u|^2 into the same slices with global float atomics, in whatever order they
    arrive (bb.h: tolerance contract 1e-4, not bit-reproducible).  Field amplitudes span four decades, so
    the addends of one pixel span eight: the order of the additions matters as much as it ever will."""
    bb = kc_env()
    Nz, B = 12, 64
    w, dn, f0, nref = problem(oracle_mod, 128, 128, Nz, B, seed=64)
    amp = np.logspace(-2, 2, B).astype(np.float32)
    np.random.default_rng(1).shuffle(amp)
    f0 = (f0 * amp[:, None, None]).astype(np.complex64)
    d = torch.from_numpy(f0.copy()).cuda()
    I = torch.full(dn.shape, 7.0, device="cuda")                       # the call zeroes the slices itself
    bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref)
    torch.cuda.synchronize()
    bb.device_status()
    assert "bpmc_kernel" in bb.last_kernel()
    Io = np.zeros(dn.shape, dtype=np.float64)
    for b in range(B):
        uo, Ib = oracle_mod.propagate(f0[b], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        Io += Ib
        if b in (0, 31, 63):
            assert rel_l2(d[b].cpu().numpy(), uo) < small_tol(Nz)
    assert rel_l2(I.cpu().numpy(), Io) < 1e-4
    # pixel by pixel as well: no slice is dominated by a few lost small addends
    assert np.abs(I.cpu().numpy() - Io).max() <= 1e-4 * Io.max()


def test_a_traced_batch_stays_inside_the_trace_buffer(oracle_mod, kc_env):
    """bb_probe_trace's buffer has one row per SM.  A batch on the cluster kernel launches 16 CTAs per
    field -- 12 fields are 192 CTAs, more rows than the buffer has -- so it must run untraced and leave the
    buffer and the guard words behind it alone; a single field (16 CTAs) is traced."""
    bb = kc_env()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    Nz, phases = 4, 16
    guard = 4096
    raw = torch.zeros(phases * sms * 6 + guard, dtype=torch.int64, device="cuda")
    raw[phases * sms * 6:] = -12345
    buf = raw[:phases * sms * 6].view(phases, sms, 6)
    try:
        bb.probe_trace(buf)
        w, dn, f0, nref = problem(oracle_mod, 128, 128, Nz, 12, seed=3)
        d = torch.from_numpy(f0.copy()).cuda()
        bb.propagate(d, dn.cuda(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        torch.cuda.synchronize()
        assert "bpmc_kernel" in bb.last_kernel()
        assert int((raw[phases * sms * 6:] != -12345).sum()) == 0 and int((buf != 0).sum()) == 0
        uo, _ = oracle_mod.propagate(f0[11], dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        assert rel_l2(d[11].cpu().numpy(), uo) < small_tol(Nz)
        d1 = torch.from_numpy(f0[:1].copy()).cuda()
        bb.propagate(d1, dn.cuda(), w.dx, w.dz, w.lam, w.n0, nref=nref)
        torch.cuda.synchronize()
        assert int((buf != 0).sum()) > 0                               # the single field was traced
        assert int((raw[phases * sms * 6:] != -12345).sum()) == 0
    finally:
        bb.probe_trace(None)
