"""``bb_nref_from_dn_static`` against ``bb_nref_from_dn``.

The static entry point is for users who must not allocate while the GPU is busy: a pipeline that
prepares n_ref of the next sample on a side stream during a propagation (``cudaMalloc`` / ``cudaFree``
wait for the whole device and would stall it), or a process whose allocator already owns almost all
device memory.  Its per-slice partial sums sit in a fixed 512 KiB array inside the library, shared by
all calls on a device and never cleared -- so the test makes TWO calls in a row, the second on a
different, shallower volume with another slab length, and compares each with the allocating path
within the 1-ulp tolerance ``test_gpu_blocks.py::test_nref_from_dn`` uses for that path.

The file sorts last on purpose: ``pytest -x`` stops at the first failure, and a failure here should
not hide the parity tests.  It runs the same in a fresh process (first use of the array on the
device) and after every other test (after ``bb_shutdown`` calls and the other kernels).
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1706_02261_b200 import workloads as wl
from gpu_common import need_gpu

ULP = 1.2e-7 * 1.4          # one float32 ulp at n ~ 1.33 .. 1.4, as in test_nref_from_dn


@pytest.mark.gpu
def test_static_nref_matches_the_allocating_path_on_two_calls_in_a_row():
    bb = need_gpu()
    w = wl.config("C1")
    dn_a = wl.make_dn(w.with_nz(70)).cuda()                        # 70 x 128 x 128
    dn_b = (wl.make_dn(w.with_nz(33)).cuda() * 3.0 + 0.01).contiguous()   # shallower, other values
    out_a = torch.full((70,), -1.0, device="cuda")
    out_b = torch.full((33,), -1.0, device="cuda")
    want_a = bb.nref_from_dn(dn_a, w.n0, 5).numpy()
    want_b = bb.nref_from_dn(dn_b, w.n0, 1000).numpy()
    torch.cuda.synchronize()

    n_launch = bb.launch_count()
    bb.nref_from_dn_static(dn_a, w.n0, 5, out_a)                   # first call (in a fresh process: the set-up)
    free_before = torch.cuda.mem_get_info()[0]
    bb.nref_from_dn_static(dn_b, w.n0, 1000, out_b)                # second call sees the first one's partial sums
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert bb.launch_count() == n_launch + 4                       # its own kernels ran: two per call
    got_a, got_b = out_a.cpu().numpy(), out_b.cpu().numpy()
    assert np.abs(got_a.astype(np.float64) - want_a.astype(np.float64)).max() <= ULP
    assert np.abs(got_b.astype(np.float64) - want_b.astype(np.float64)).max() <= ULP
    assert len(set(got_b.tolist())) == 1 and len(set(got_a.tolist())) > 1      # one slab / 14 slabs
    assert free_after == free_before, "device memory in use changed across a call that must not allocate"
    # and once more on the first volume: the deeper call after the shallower one
    out_a.fill_(-1.0)
    bb.nref_from_dn_static(dn_a, w.n0, 5, out_a)
    torch.cuda.synchronize()
    assert np.array_equal(out_a.cpu().numpy(), got_a)


@pytest.mark.gpu
def test_static_nref_refuses_volumes_deeper_than_its_scratch():
    bb = need_gpu()
    lib = bb.load()
    nz = bb.static_max_nz() + 1
    assert bb.static_max_nz() == 4096
    small = torch.zeros((4, 8, 8), device="cuda")
    out = torch.zeros(4, device="cuda")
    rc = lib.bb_nref_from_dn_static(ctypes.c_void_p(small.data_ptr()), 8, 8, nz, 1.33, 1,
                                    ctypes.c_void_p(out.data_ptr()), None)
    assert rc == 1 and "BB_STATIC_MAX_NZ" in lib.bb_last_error().decode()
    # the limit itself is accepted (a thin volume: 4096 x 8 x 8)
    deep = torch.full((4096, 8, 8), 0.02, device="cuda")
    out = torch.empty(4096, device="cuda")
    bb.nref_from_dn_static(deep, 1.33, 7, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(),
                          np.full(4096, np.float32(np.float64(np.float32(1.33)) + np.float64(np.float32(0.02)))))
