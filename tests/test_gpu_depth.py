"""-m gpu: parity at depth for what round 2 added ("the slope is the real check").

  * BB_BACKWARD on the headline grid (1024 x 1024, C4's phantom and emitters) for 256 slices against
    ``oracle.propagate_backward`` (Fig. 2c; line 33), with the same bound on the error growth
    per step as the forward run of tests/test_gpu_bpm.py;
  * a batch at the headline size: 4 multiplexed 1024 x 1024 fields through 128 slices of the shared volume
    (north_star item 4), every field and the summed intensity volume;
  * the detection chain emitters -> sample -> refocus -> PSF tiles at C3's full depth of 512 slices
    (PAPER.md lines 29-31).
"""
import numpy as np
import pytest
import torch

from conftest import rel_l2
from gpu_common import StreamCompare, gpu_inputs, need_gpu, oracle_field0
from paper_1706_02261_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-4          # BASELINE.json north_star: relative L2 on the final field and on the intensity volume


def test_backward_at_depth_on_the_headline_grid(oracle_mod):
    bb = need_gpu()
    w = wl.config("C4").with_nz(256)
    dn, f_gpu = gpu_inputs(w, bb)
    f0 = oracle_field0(w, oracle_mod)
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    I = torch.empty(dn.shape, device="cuda")
    bb.propagate(f_gpu, dn, w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=bb.BACKWARD)
    torch.cuda.synchronize()
    bb.device_status()
    assert "bpm16_kernel<4,4" in bb.last_kernel()
    uo, Io = oracle_mod.propagate_backward(f0[0], dn.cpu().numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref)
    cmp_I = StreamCompare()
    for j in range(w.Nz - 1, -1, -1):                      # the order the run visits the slices in
        cmp_I.add(I[j].cpu().numpy(), Io[j])
    err_u = rel_l2(f_gpu[0].cpu().numpy(), uo)
    # slice Nz-1-i is recorded after i steps: the line through the origin of (intensity error / 2) against i
    i = np.arange(w.Nz, dtype=np.float64)
    slope = float(np.sum(i * (np.array(cmp_I.curve) / 2)) / np.sum(i * i))
    print("\nbackward 1024^2 x %d: field rel-L2 %.3e, intensity rel-L2 %.3e, growth per step %.2e" % (w.Nz, err_u, cmp_I.rel, slope))
    assert err_u < TOL and cmp_I.rel < TOL
    assert slope <= 6e-8, slope


def test_a_batch_of_four_fields_at_the_headline_size(oracle_mod):
    bb = need_gpu()
    B = 4
    w = wl.config("C4").with_nz(128)
    pos, ph, amp = wl.make_emitters(w)
    phases = [ph] + [np.random.default_rng(1000 + b).uniform(0, 2 * np.pi, size=ph.shape).astype(np.float32) for b in range(1, B)]
    dn = wl.make_dn(w, device="cuda").cuda()
    pos_d, amp_d = torch.from_numpy(pos).cuda(), torch.from_numpy(amp).cuda()
    f_gpu = torch.stack([bb.multiplex_psf(pos_d, torch.from_numpy(p).cuda(), amp_d, w.NA, w.Nx, w.Ny, w.dx, w.lam)
                         for p in phases]).contiguous()
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    I = torch.empty(dn.shape, device="cuda")
    bb.propagate(f_gpu, dn, w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref)
    torch.cuda.synchronize()
    bb.device_status()
    assert "bpm16_kernel<4,4" in bb.last_kernel() and bb.last_kernel().endswith("true>")     # the batch variant
    dn_h = dn.cpu().numpy()
    Io = None
    for b in range(B):
        u0 = oracle_mod.multiplex_psf(pos, phases[b], amp, w.NA, w.Nx, w.Ny, w.dx, w.lam).astype(np.complex64)
        uo, Ib = oracle_mod.propagate(u0, dn_h, w.dx, w.dz, w.lam, w.n0, nref=nref)
        Io = Ib if Io is None else Io + Ib
        e = rel_l2(f_gpu[b].cpu().numpy(), uo)
        print("\nfield %d of %d, 1024^2 x %d: rel-L2 %.3e" % (b, B, w.Nz, e))
        assert e < TOL
    cmp_I = StreamCompare()
    for j in range(w.Nz):
        cmp_I.add(I[j].cpu().numpy(), Io[j])
    print("summed intensity rel-L2 %.3e (last slice %.2e)" % (cmp_I.rel, cmp_I.curve[-1]))
    assert cmp_I.rel < TOL and max(cmp_I.curve) < TOL


def test_detection_chain_at_full_c3_depth(oracle_mod):
    """C3 (10 x 10 emitters, 512 x 512, 512 slices): through the whole sample, back onto the emitter plane through
    the refocusing lens (one signed free-space step of -512 dz), PSF tiles cut around every emitter."""
    bb = need_gpu()
    w = wl.config("C3")
    pos, ph, amp = wl.make_emitters(w)
    pos_d = torch.from_numpy(pos).cuda()
    u = bb.multiplex_psf(pos_d, torch.from_numpy(ph).cuda(), torch.from_numpy(amp).cuda(), w.NA, w.Nx, w.Ny, w.dx, w.lam)[None]
    dn = wl.make_dn(w)
    nref = bb.nref_from_dn(dn.cuda(), w.n0, w.nref_slab).numpy()
    bb.propagate(u, dn.cuda(), w.dx, w.dz, w.lam, w.n0, nref=nref)
    bb.refocus(u, w.dx, -w.Nz * w.dz, w.lam, w.n0)
    T = 32
    tiles = bb.extract_tiles(u, pos_d, w.dx, T)
    torch.cuda.synchronize()
    bb.device_status()
    uo = oracle_mod.multiplex_psf(pos, ph, amp, w.NA, w.Nx, w.Ny, w.dx, w.lam).astype(np.complex64)
    uo, _ = oracle_mod.propagate(uo, dn.numpy(), w.dx, w.dz, w.lam, w.n0, nref=nref, want_intensity=False)
    uo = oracle_mod.refocus(uo, w.dx, -w.Nz * w.dz, w.lam, w.n0)
    assert rel_l2(u[0].cpu().numpy(), uo) < TOL
    assert np.array_equal(tiles.cpu().numpy(), oracle_mod.extract_tiles(u[0].cpu().numpy(), pos, w.dx, T).astype(np.complex64))
    e = rel_l2(tiles.cpu().numpy(), oracle_mod.extract_tiles(uo, pos, w.dx, T))
    print("\nC3 chain at %d slices: tiles rel-L2 %.3e" % (w.Nz, e))
    assert e < TOL
