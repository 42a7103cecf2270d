"""Helpers shared by the ``-m gpu`` parity tests: they call the CUDA path only through the
binding of the C ABI and the oracle only through ``oracle``; inputs come from ``workloads``."""
import numpy as np
import pytest
import torch

from paper_1706_02261_b200 import workloads as wl


def need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1706_02261_b200 import build, binding
    build.build_library()
    return binding


class StreamCompare:
    """Accumulates ||a - b||^2 and ||b||^2 slice by slice (b = oracle, double)."""

    def __init__(self):
        self.num = 0.0
        self.den = 0.0
        self.curve = []

    def add(self, a, b):
        a = np.asarray(a, dtype=np.float64)
        n = float(np.sum((a - b) ** 2))
        d = float(np.sum(b ** 2))
        self.num += n
        self.den += d
        self.curve.append((n / d) ** 0.5 if d > 0 else 0.0)

    @property
    def rel(self):
        return (self.num / self.den) ** 0.5


def gpu_inputs(w: wl.Workload, bb, dn_device="cuda"):
    """dn (CUDA float32), initial field(s) (CUDA complex64 [B][Ny][Nx]) and host copies."""
    dn = wl.make_dn(w, device=dn_device).cuda()
    f = wl.make_field(w)
    if f is None:
        pos, ph, amp = wl.make_emitters(w)
        f_gpu = bb.multiplex_psf(torch.from_numpy(pos).cuda(), torch.from_numpy(ph).cuda(),
                                 torch.from_numpy(amp).cuda(), w.NA, w.Nx, w.Ny, w.dx, w.lam)[None].contiguous()
    else:
        f_gpu = torch.from_numpy(f).cuda()
    return dn, f_gpu


def oracle_field0(w: wl.Workload, oracle):
    """The oracle's own input field for workload w (Algorithm M for multiplex workloads)."""
    f = wl.make_field(w)
    if f is not None:
        return f
    pos, ph, amp = wl.make_emitters(w)
    u0 = oracle.multiplex_psf(pos, ph, amp, w.NA, w.Nx, w.Ny, w.dx, w.lam)
    return u0.astype(np.complex64)[None]
