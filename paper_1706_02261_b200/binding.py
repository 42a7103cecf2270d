"""ctypes binding of ``libbiobeam_b200.so`` (``include/bb.h``): argument marshalling only.

Every function takes torch tensors (device memory and streams are torch's; all arithmetic
runs in the library's CUDA kernels) and has the name of the C entry point without ``bb_``.
There is no fallback: if the shared library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbiobeam_b200.so")

ACCUMULATE = 1
INTENSITY_PER_FIELD = 2
LAUNCH_PER_PHASE = 4
BACKWARD = 8
HOMOGENEOUS = 16

EXPORTS = ("bb_propagate", "bb_propagate_ex", "bb_propagate_host", "bb_nref_from_dn",
           "bb_multiplex_psf", "bb_fft2", "bb_propagator_table", "bb_last_error", "bb_version",
           "bb_shutdown", "bb_launch_count", "bb_device_status", "bb_probe_l2_bandwidth", "bb_probe_fp32", "bb_probe_trace",
           "bb_last_kernel", "bb_nref_from_dn_static", "bb_static_max_nz", "bb_multiplex_annular", "bb_lightsheet", "bb_refocus", "bb_extract_tiles", "bb_image_formation")

STATUS_NAMES = {0: "BB_OK", 1: "BB_ERR_INVALID_ARG", 2: "BB_ERR_UNSUPPORTED_SHAPE", 3: "BB_ERR_CUDA",
                4: "BB_ERR_OOM", 5: "BB_ERR_ARCH", 6: "BB_ERR_INTERNAL"}


class BBError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, str(status)), message))
        self.status = status


class _Opts(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_int), ("batch", ctypes.c_int),
                ("nref", ctypes.POINTER(ctypes.c_float)), ("flags", ctypes.c_uint),
                ("stream", ctypes.c_void_p)]


_lib = None


def load() -> ctypes.CDLL:
    """Loads the shared library (built by ``paper_1706_02261_b200.build``); raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            "%s not found: build it with `python -m paper_1706_02261_b200.build` "
            "(there is no fallback implementation)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, fp, i, f = ctypes.c_void_p, ctypes.POINTER(ctypes.c_float), ctypes.c_int, ctypes.c_float
    lib.bb_propagate.argtypes = [vp, vp, i, i, i, f, f, f, f, vp]
    lib.bb_propagate_ex.argtypes = [vp, vp, i, i, i, f, f, f, f, vp, ctypes.POINTER(_Opts)]
    lib.bb_propagate_host.argtypes = [vp, vp, i, i, i, f, f, f, f, vp, ctypes.POINTER(_Opts)]
    lib.bb_nref_from_dn.argtypes = [vp, i, i, i, f, i, fp, vp]
    lib.bb_nref_from_dn_static.argtypes = [vp, i, i, i, f, i, vp, vp]
    lib.bb_multiplex_psf.argtypes = [vp, vp, vp, i, f, i, i, f, f, vp, vp]
    lib.bb_multiplex_annular.argtypes = [vp, vp, vp, i, f, f, i, i, f, f, vp, vp]
    lib.bb_lightsheet.argtypes = [i, i, f, f, f, f, f, vp, vp]
    lib.bb_refocus.argtypes = [vp, i, i, i, f, f, f, f, vp]
    lib.bb_extract_tiles.argtypes = [vp, i, i, i, i, vp, i, f, i, vp, vp]
    lib.bb_image_formation.argtypes = [vp, i, i, vp, i, f, vp, i, vp, vp]
    lib.bb_fft2.argtypes = [vp, i, i, i, i, vp]
    lib.bb_propagator_table.argtypes = [i, i, f, f, f, f, vp, vp]
    lib.bb_probe_l2_bandwidth.argtypes = [ctypes.c_ulonglong, i, i, ctypes.POINTER(ctypes.c_double)]
    lib.bb_probe_fp32.argtypes = [i, i, ctypes.POINTER(ctypes.c_double)]
    lib.bb_probe_trace.argtypes = [ctypes.c_void_p, i]
    lib.bb_last_error.restype = ctypes.c_char_p
    lib.bb_last_kernel.restype = ctypes.c_char_p
    lib.bb_launch_count.restype = ctypes.c_ulonglong
    lib.bb_shutdown.restype = None
    _lib = lib
    return lib


def _check(rc: int):
    if rc != 0:
        raise BBError(rc, load().bb_last_error().decode("utf-8", "replace"))


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _field_shape(field: torch.Tensor):
    if field.dtype != torch.complex64 or not field.is_contiguous():
        raise TypeError("field must be a contiguous complex64 tensor [B][Ny][Nx] or [Ny][Nx]")
    if field.dim() == 2:
        return 1, field.shape[0], field.shape[1]
    if field.dim() == 3:
        return field.shape[0], field.shape[1], field.shape[2]
    raise TypeError("field must be [B][Ny][Nx] or [Ny][Nx]")


def _f32(t: torch.Tensor, name: str):
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous float32 tensor" % name)
    return t


def propagate(field: torch.Tensor, dn: torch.Tensor, dx: float, dz: float, lam: float, n0: float,
              intensity: Optional[torch.Tensor] = None, nref=None, flags: int = 0, stream=None, nz=None):
    """``bb_propagate_ex`` (CUDA tensors; asynchronous on ``stream``) or ``bb_propagate_host``
    (CPU tensors, pinned for overlap; synchronous).  ``field`` is updated in place.
    ``nref``: None or a sequence / CPU tensor of Nz floats."""
    lib = load()
    B, Ny, Nx = _field_shape(field)
    on_gpu = field.is_cuda
    if dn is None:
        if not flags & HOMOGENEOUS or nz is None:
            raise TypeError("dn may be None only with HOMOGENEOUS and nz = number of steps")
        Nz = int(nz)
    else:
        _f32(dn, "dn")
        if dn.dim() != 3 or dn.shape[1] != Ny or dn.shape[2] != Nx:
            raise TypeError("dn must be [Nz][%d][%d]" % (Ny, Nx))
        Nz = dn.shape[0]
    if (dn is not None and dn.is_cuda != on_gpu) or (intensity is not None and intensity.is_cuda != on_gpu):
        raise TypeError("field, dn and intensity must all be CUDA tensors or all CPU tensors")
    if intensity is not None:
        _f32(intensity, "intensity")
        want = (B * Nz if flags & INTENSITY_PER_FIELD else Nz) * Ny * Nx
        if intensity.numel() != want:
            raise TypeError("intensity has %d elements, expected %d" % (intensity.numel(), want))
    opts = _Opts()
    opts.struct_size = ctypes.sizeof(_Opts)
    opts.batch = B
    opts.flags = flags
    nref_buf = None
    if nref is not None:
        nref_buf = (ctypes.c_float * Nz)(*[float(x) for x in nref])
        opts.nref = ctypes.cast(nref_buf, ctypes.POINTER(ctypes.c_float))
    iptr = ctypes.c_void_p(intensity.data_ptr()) if intensity is not None else None
    dnp = ctypes.c_void_p(dn.data_ptr()) if dn is not None else None
    if on_gpu:
        opts.stream = _stream_ptr(stream)
        with torch.cuda.device(field.device):
            rc = lib.bb_propagate_ex(ctypes.c_void_p(field.data_ptr()), dnp, Nx, Ny, Nz,
                                     dx, dz, lam, n0, iptr, ctypes.byref(opts))
    else:
        rc = lib.bb_propagate_host(ctypes.c_void_p(field.data_ptr()), dnp, Nx, Ny, Nz,
                                   dx, dz, lam, n0, iptr, ctypes.byref(opts))
    _check(rc)
    return field, intensity


def propagate_simple(field: torch.Tensor, dn: torch.Tensor, dx, dz, lam, n0, intensity=None):
    """The flat ``bb_propagate`` entry point (B = 1, n_ref = n0, default stream)."""
    lib = load()
    B, Ny, Nx = _field_shape(field)
    if B != 1:
        raise TypeError("bb_propagate takes one field")
    _f32(dn, "dn")
    with torch.cuda.device(field.device):
        rc = lib.bb_propagate(ctypes.c_void_p(field.data_ptr()), ctypes.c_void_p(dn.data_ptr()), Nx, Ny, dn.shape[0],
                              dx, dz, lam, n0,
                              ctypes.c_void_p(intensity.data_ptr()) if intensity is not None else None)
    _check(rc)
    return field, intensity


def nref_from_dn(dn: torch.Tensor, n0: float, slab: int, stream=None) -> torch.Tensor:
    lib = load()
    _f32(dn, "dn")
    Nz, Ny, Nx = dn.shape
    out = (ctypes.c_float * Nz)()
    with torch.cuda.device(dn.device):
        _check(lib.bb_nref_from_dn(ctypes.c_void_p(dn.data_ptr()), Nx, Ny, Nz, n0, slab, out, _stream_ptr(stream)))
    return torch.tensor(list(out), dtype=torch.float32)


def static_max_nz() -> int:
    return int(load().bb_static_max_nz())


def nref_from_dn_static(dn: torch.Tensor, n0: float, slab: int, out: torch.Tensor, stream=None) -> torch.Tensor:
    """``bb_nref_from_dn_static``: n_ref per slice into ``out``, a CUDA float32 tensor of Nz elements that
    the CALLER supplies -- this wrapper creates no tensor, because the entry point exists for callers that
    must not allocate (see ``include/bb.h``).  Asynchronous on ``stream``; at most ``static_max_nz()`` slices."""
    lib = load()
    _f32(dn, "dn")
    _f32(out, "out")
    Nz, Ny, Nx = dn.shape
    if not dn.is_cuda or not out.is_cuda or out.device != dn.device or out.numel() != Nz:
        raise TypeError("dn and out must be CUDA tensors on one device, out with Nz = %d elements" % Nz)
    with torch.cuda.device(dn.device):
        _check(lib.bb_nref_from_dn_static(ctypes.c_void_p(dn.data_ptr()), Nx, Ny, Nz, n0, slab,
                                          ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def multiplex_psf(pos: torch.Tensor, phase: Optional[torch.Tensor], amp: Optional[torch.Tensor], NA: float,
                  Nx: int, Ny: int, dx: float, lam: float, out: Optional[torch.Tensor] = None, stream=None):
    lib = load()
    _f32(pos, "pos")
    if pos.dim() != 2 or pos.shape[1] != 2:
        raise TypeError("pos must be [M][2]")
    M = pos.shape[0]
    for t, n in ((phase, "phase"), (amp, "amp")):
        if t is not None and (_f32(t, n).numel() != M):
            raise TypeError("%s must have M elements" % n)
    if out is None:
        out = torch.empty((Ny, Nx), dtype=torch.complex64, device=pos.device)
    p = lambda t: ctypes.c_void_p(t.data_ptr()) if t is not None else None
    with torch.cuda.device(pos.device):
        _check(lib.bb_multiplex_psf(p(pos), p(phase), p(amp), M, NA, Nx, Ny, dx, lam, p(out), _stream_ptr(stream)))
    return out


def multiplex_annular(pos: torch.Tensor, phase: Optional[torch.Tensor], amp: Optional[torch.Tensor], NA_in: float, NA: float,
                      Nx: int, Ny: int, dx: float, lam: float, out: Optional[torch.Tensor] = None, stream=None):
    """``bb_multiplex_annular``: Bessel-beam foci / lattices (annular pupil NA_in <= |k|/k0 <= NA)."""
    lib = load()
    _f32(pos, "pos")
    M = pos.shape[0]
    if out is None:
        out = torch.empty((Ny, Nx), dtype=torch.complex64, device=pos.device)
    p = lambda t: ctypes.c_void_p(t.data_ptr()) if t is not None else None
    with torch.cuda.device(pos.device):
        _check(lib.bb_multiplex_annular(p(pos), p(phase), p(amp), M, NA_in, NA, Nx, Ny, dx, lam, p(out), _stream_ptr(stream)))
    return out


def lightsheet(Nx: int, Ny: int, dx: float, lam: float, n0: float, NA: float, z_focus: float, device="cuda", stream=None):
    """``bb_lightsheet``: input-plane field of a cylindrical Gaussian sheet focused z_focus behind the plane."""
    out = torch.empty((Ny, Nx), dtype=torch.complex64, device=device)
    with torch.cuda.device(out.device):
        _check(load().bb_lightsheet(Nx, Ny, dx, lam, n0, NA, z_focus, ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def refocus(field: torch.Tensor, dx: float, dz: float, lam: float, n: float, stream=None) -> torch.Tensor:
    """``bb_refocus``: in-place free-space propagation over the signed distance dz in index n."""
    B, Ny, Nx = _field_shape(field)
    with torch.cuda.device(field.device):
        _check(load().bb_refocus(ctypes.c_void_p(field.data_ptr()), Nx, Ny, B, dx, dz, lam, n, _stream_ptr(stream)))
    return field


def extract_tiles(src: torch.Tensor, pos: torch.Tensor, dx: float, T: int, stream=None) -> torch.Tensor:
    """``bb_extract_tiles``: src [Np][Ny][Nx] (or [Ny][Nx]), float32 or complex64 -> [M][Np][T][T]."""
    if src.dim() == 2:
        src = src[None]
    if src.dtype not in (torch.float32, torch.complex64) or not src.is_contiguous() or src.dim() != 3:
        raise TypeError("src must be a contiguous float32 or complex64 tensor [Np][Ny][Nx]")
    _f32(pos, "pos")
    Np, Ny, Nx = src.shape
    M = pos.shape[0]
    out = torch.empty((M, Np, T, T), dtype=src.dtype, device=src.device)
    with torch.cuda.device(src.device):
        _check(load().bb_extract_tiles(ctypes.c_void_p(src.data_ptr()), 2 if src.dtype == torch.complex64 else 1, Nx, Ny, Np,
                                       ctypes.c_void_p(pos.data_ptr()), M, dx, T, ctypes.c_void_p(out.data_ptr()),
                                       _stream_ptr(stream)))
    return out


def image_formation(source: torch.Tensor, pos: torch.Tensor, dx: float, psf: torch.Tensor, stream=None) -> torch.Tensor:
    """``bb_image_formation``: source [Ny][Nx] float32, psf [M][T][T] float32 -> image [Ny][Nx]."""
    _f32(source, "source"); _f32(pos, "pos"); _f32(psf, "psf")
    Ny, Nx = source.shape
    M, T = psf.shape[0], psf.shape[1]
    if pos.shape[0] != M or psf.shape[2] != T:
        raise TypeError("psf must be [M][T][T] with M = number of emitters")
    out = torch.empty_like(source)
    with torch.cuda.device(source.device):
        _check(load().bb_image_formation(ctypes.c_void_p(source.data_ptr()), Nx, Ny, ctypes.c_void_p(pos.data_ptr()), M, dx,
                                         ctypes.c_void_p(psf.data_ptr()), T, ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def fft2(field: torch.Tensor, sign: int = -1, stream=None) -> torch.Tensor:
    lib = load()
    B, Ny, Nx = _field_shape(field)
    with torch.cuda.device(field.device):
        _check(lib.bb_fft2(ctypes.c_void_p(field.data_ptr()), Nx, Ny, B, sign, _stream_ptr(stream)))
    return field


def propagator_table(Nx: int, Ny: int, dx: float, dz: float, lam: float, nref: float, device="cuda", stream=None):
    lib = load()
    out = torch.empty((Ny, Nx), dtype=torch.complex64, device=device)
    with torch.cuda.device(out.device):
        _check(lib.bb_propagator_table(Nx, Ny, dx, dz, lam, nref, ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def probe_l2_bandwidth(nbytes: int = 32 << 20, iters: int = 200, mode: int = 0) -> float:
    """GB/s of an L2-resident copy (mode 0) or read (mode 1); see ``bb_probe_l2_bandwidth``."""
    out = ctypes.c_double()
    _check(load().bb_probe_l2_bandwidth(nbytes, iters, mode, ctypes.byref(out)))
    return out.value


def probe_fp32(iters: int = 20000, packed=False) -> float:
    """TFLOP/s of the scalar (``packed`` False / 0) or packed (True / 1) FP32 FMA pipe, or of the library's butterfly
    mix run from registers (2); see ``bb_probe_fp32``."""
    out = ctypes.c_double()
    _check(load().bb_probe_fp32(iters, int(packed), ctypes.byref(out)))
    return out.value


def device_status():
    _check(load().bb_device_status())


def last_kernel() -> str:
    return load().bb_last_kernel().decode()


def launch_count() -> int:
    return int(load().bb_launch_count())


def version() -> int:
    return int(load().bb_version())


def shutdown():
    load().bb_shutdown()


def probe_trace(buf: Optional[torch.Tensor]) -> None:
    """Switch the persistent kernel's timeline on (``buf``: CUDA int64 [phases][grid][6]) or off (None);
    see ``bb_probe_trace``."""
    if buf is None:
        _check(load().bb_probe_trace(None, 0))
        return
    if not (buf.is_cuda and buf.dtype == torch.int64 and buf.is_contiguous() and buf.dim() == 3 and buf.shape[2] == 6):
        raise ValueError("trace buffer must be a contiguous CUDA int64 tensor [phases][grid][6]")
    _check(load().bb_probe_trace(buf.data_ptr(), int(buf.shape[0])))
