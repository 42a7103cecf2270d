"""ctypes marshalling for ``bpm_oracle.c`` -- TEST INFRASTRUCTURE (see package docstring).

No arithmetic of the method happens here: every function converts its numpy
arguments to the C layout, calls the C routine of the same name and returns
double-precision results.  Float32 / complex64 inputs are passed as such and
promoted to double inside the C code (never through NumPy scalar promotion,
which would silently compute in single precision).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bpm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

_f32p = ctypes.POINTER(ctypes.c_float)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False, sanitize: bool | None = None) -> str:
    """Compile ``bpm_oracle.c`` into ``oracle/liboracle.so`` with gcc (IEEE double, OpenMP).

    ``sanitize`` (default: the environment variable ``ORACLE_SANITIZE=1``) builds ``liboracle_san.so`` with
    AddressSanitizer and UndefinedBehaviorSanitizer instead -- same source, same
    floating-point flags; run the CPU tests against it as
    ``ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 pytest -m "not gpu"``.
    """
    if sanitize is None:
        sanitize = os.environ.get("ORACLE_SANITIZE", "") == "1"
    lib = os.path.join(_HERE, "liboracle_san.so") if sanitize else _LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(_SRC)):
        return lib
    tmp = lib + ".tmp%d" % os.getpid()
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] \
        if sanitize else ["-O2"]
    cmd = ["gcc", *opt, "-std=c11", "-fPIC", "-shared", "-fopenmp",
           "-ffp-contract=off", "-fno-fast-math", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


def _load():
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        lib = ctypes.CDLL(build())
        lib.oracle_dft2_bruteforce.argtypes = [_f64p, _f64p, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.oracle_dft2_bruteforce.restype = None
        lib.oracle_fft1.argtypes = [_f64p, ctypes.c_int, ctypes.c_int]
        lib.oracle_fft2.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.oracle_bpm_step.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, _f32p,
                                        ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                        ctypes.c_float, ctypes.c_float, _f64p]
        lib.oracle_bpm_step_backward.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, _f32p,
                                                 ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                                 ctypes.c_float, ctypes.c_float]
        lib.oracle_propagate.argtypes = [_f32p, _f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                         ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                         _f32p, _f64p, _f64p, ctypes.c_int]
        lib.oracle_multiplex_psf.argtypes = [_f32p, _f32p, _f32p, ctypes.c_int, ctypes.c_float,
                                             ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, _f64p]
        lib.oracle_nref_from_dn.argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                            ctypes.c_float, ctypes.c_int, _f32p]
        lib.oracle_propagate_backward.argtypes = [_f32p, _f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                  ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                                  _f32p, _f64p, _f64p]
        lib.oracle_refocus.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float,
                                       ctypes.c_float, ctypes.c_float]
        lib.oracle_extract_tiles.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f32p,
                                             ctypes.c_int, ctypes.c_float, ctypes.c_int, _f64p]
        lib.oracle_lightsheet.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                          ctypes.c_float, ctypes.c_float, _f64p]
        lib.oracle_multiplex_annular.argtypes = [_f32p, _f32p, _f32p, ctypes.c_int, ctypes.c_float, ctypes.c_float,
                                                 ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, _f64p]
        lib.oracle_image_formation.argtypes = [_f64p, ctypes.c_int, ctypes.c_int, _f32p, ctypes.c_int, ctypes.c_float,
                                               _f64p, ctypes.c_int, _f64p]
        _lib = lib
        return lib


def num_threads() -> int:
    """Threads the OpenMP loops will use (OMP_NUM_THREADS or the affinity mask)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        try:
            return max(1, int(env.split(",")[0]))
        except ValueError:
            pass
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _c128(a) -> np.ndarray:
    """Own, C-contiguous complex128 copy (complex64 -> complex128 is exact)."""
    return np.array(a, dtype=np.complex128, order="C", copy=True)


def _p64(a: np.ndarray):
    return a.ctypes.data_as(_f64p)


def _p32(a):
    return None if a is None else a.ctypes.data_as(_f32p)


def _f32(a, shape=None):
    if a is None:
        return None
    b = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None and b.shape != tuple(shape):
        raise ValueError("expected shape %r, got %r" % (tuple(shape), b.shape))
    return b


def _sf(x) -> float:
    """A scalar rounded to float32 (what the C ABI of both sides receives), as a Python float."""
    return float(np.float32(x))


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError("%s failed with status %d (sizes must be powers of two)" % (what, rc))


def dft2_bruteforce(a, sign: int = -1) -> np.ndarray:
    a = _c128(a)
    Ny, Nx = a.shape
    out = np.empty_like(a)
    _load().oracle_dft2_bruteforce(_p64(a), _p64(out), Nx, Ny, int(sign))
    return out


def fft1(a, sign: int = -1) -> np.ndarray:
    a = _c128(a)
    _check(_load().oracle_fft1(_p64(a), a.shape[0], int(sign)), "oracle_fft1")
    return a


def fft2(a, sign: int = -1) -> np.ndarray:
    a = _c128(a)
    Ny, Nx = a.shape
    _check(_load().oracle_fft2(_p64(a), Nx, Ny, int(sign)), "oracle_fft2")
    return a


def bpm_step(u, dn_slice, dx, dz, lam, n0, nref=None, want_intensity=True):
    """One Algorithm-O step on a complex128 field (returns new field, intensity)."""
    u = _c128(u)
    Ny, Nx = u.shape
    dn_slice = _f32(dn_slice, (Ny, Nx))
    I = np.empty((Ny, Nx), dtype=np.float64) if want_intensity else None
    nr = _sf(n0 if nref is None else nref)
    _check(_load().oracle_bpm_step(_p64(u), Nx, Ny, _p32(dn_slice),
                                   _sf(dx), _sf(dz), _sf(lam),
                                   _sf(n0), nr, None if I is None else _p64(I)),
           "oracle_bpm_step")
    return u, I


def bpm_step_backward(u, dn_slice, dx, dz, lam, n0, nref=None):
    u = _c128(u)
    Ny, Nx = u.shape
    dn_slice = _f32(dn_slice, (Ny, Nx))
    nr = _sf(n0 if nref is None else nref)
    _check(_load().oracle_bpm_step_backward(_p64(u), Nx, Ny, _p32(dn_slice),
                                            _sf(dx), _sf(dz), _sf(lam),
                                            _sf(n0), nr),
           "oracle_bpm_step_backward")
    return u


def propagate(field, dn, dx, dz, lam, n0, nref=None, want_intensity=True, intensity_init=None):
    """Whole propagation of one complex64 field through dn[Nz][Ny][Nx] (float32).

    Returns (final field complex128 [Ny][Nx], intensity float64 [Nz][Ny][Nx] or None).
    ``intensity_init`` (float64 volume) switches to accumulate mode (I += |u|^2).
    """
    f = np.ascontiguousarray(field, dtype=np.complex64)
    Ny, Nx = f.shape
    dn = _f32(dn)
    if dn.ndim != 3 or dn.shape[1:] != (Ny, Nx):
        raise ValueError("dn must be [Nz][Ny][Nx]")
    Nz = dn.shape[0]
    nref = _f32(nref, (Nz,))
    out = np.empty((Ny, Nx), dtype=np.complex128)
    accumulate = 0
    I = None
    if intensity_init is not None:
        I = np.array(intensity_init, dtype=np.float64, order="C", copy=True)
        accumulate = 1
    elif want_intensity:
        I = np.empty((Nz, Ny, Nx), dtype=np.float64)
    rc = _load().oracle_propagate(f.view(np.float32).ctypes.data_as(_f32p), _p32(dn), Nx, Ny, Nz,
                                  _sf(dx), _sf(dz), _sf(lam), _sf(n0),
                                  _p32(nref), _p64(out), None if I is None else _p64(I), accumulate)
    _check(rc, "oracle_propagate")
    return out, I


def propagate_stream(field, dn, dx, dz, lam, n0, nref=None, on_slice=None, z_range=None):
    """Same steps as :func:`propagate`, one C step per slice, calling
    ``on_slice(j, u_complex128, I_float64)`` after each so that a 4 GiB volume can be
    compared slice by slice without materialising it in double.  Returns the final field.
    """
    u = _c128(np.ascontiguousarray(field, dtype=np.complex64))
    Ny, Nx = u.shape
    Nz = dn.shape[0]
    nref = _f32(nref, (Nz,))
    lib = _load()
    I = np.empty((Ny, Nx), dtype=np.float64)
    j0, j1 = (0, Nz) if z_range is None else z_range
    for j in range(j0, j1):
        sl = _f32(dn[j], (Ny, Nx))
        nr = _sf(n0 if nref is None else nref[j])
        _check(lib.oracle_bpm_step(_p64(u), Nx, Ny, _p32(sl), _sf(dx), _sf(dz),
                                   _sf(lam), _sf(n0), nr, _p64(I)),
               "oracle_bpm_step")
        if on_slice is not None:
            on_slice(j, u, I)
    return u


def multiplex_psf(pos, phase, amp, NA, Nx, Ny, dx, lam) -> np.ndarray:
    pos = _f32(pos)
    if pos.ndim != 2 or pos.shape[1] != 2:
        raise ValueError("pos must be [M][2]")
    M = pos.shape[0]
    phase = _f32(phase, (M,))
    amp = _f32(amp, (M,))
    out = np.empty((Ny, Nx), dtype=np.complex128)
    rc = _load().oracle_multiplex_psf(_p32(pos), _p32(phase), _p32(amp), M, _sf(NA),
                                      Nx, Ny, _sf(dx), _sf(lam), _p64(out))
    _check(rc, "oracle_multiplex_psf")
    return out


def nref_from_dn(dn, n0, slab) -> np.ndarray:
    dn = _f32(dn)
    Nz, Ny, Nx = dn.shape
    out = np.empty((Nz,), dtype=np.float32)
    _check(_load().oracle_nref_from_dn(_p32(dn), Nx, Ny, Nz, _sf(n0), int(slab), _p32(out)),
           "oracle_nref_from_dn")
    return out


def propagate_backward(field, dn, dx, dz, lam, n0, nref=None, want_intensity=True):
    """Time-reversed propagation (``oracle_propagate_backward``): returns (field at z = 0, I[Nz][Ny][Nx] or None)."""
    f = np.ascontiguousarray(field, dtype=np.complex64)
    Ny, Nx = f.shape
    dn = _f32(dn)
    Nz = dn.shape[0]
    nref = _f32(nref, (Nz,))
    out = np.empty((Ny, Nx), dtype=np.complex128)
    I = np.empty((Nz, Ny, Nx), dtype=np.float64) if want_intensity else None
    rc = _load().oracle_propagate_backward(f.view(np.float32).ctypes.data_as(_f32p), _p32(dn), Nx, Ny, Nz,
                                           _sf(dx), _sf(dz), _sf(lam), _sf(n0), _p32(nref), _p64(out),
                                           None if I is None else _p64(I))
    _check(rc, "oracle_propagate_backward")
    return out, I


def refocus(u, dx, dz, lam, n) -> np.ndarray:
    """One homogeneous-medium step of SIGNED length dz (``oracle_refocus``)."""
    u = _c128(u)
    Ny, Nx = u.shape
    _check(_load().oracle_refocus(_p64(u), Nx, Ny, _sf(dx), _sf(dz), _sf(lam), _sf(n)), "oracle_refocus")
    return u


def extract_tiles(src, pos, dx, T) -> np.ndarray:
    """T x T windows around the emitters of every plane of ``src`` ([Np][Ny][Nx] or [Ny][Nx], real or
    complex): returns [M][Np][T][T] (``oracle_extract_tiles``)."""
    a = np.asarray(src)
    if a.ndim == 2:
        a = a[None]
    cplx = np.iscomplexobj(a)
    a = np.ascontiguousarray(a, dtype=np.complex128 if cplx else np.float64)
    Np, Ny, Nx = a.shape
    pos = _f32(pos)
    M = pos.shape[0]
    out = np.empty((M, Np, T, T), dtype=a.dtype)
    _check(_load().oracle_extract_tiles(_p64(a), 2 if cplx else 1, Nx, Ny, Np, _p32(pos), M, _sf(dx), int(T), _p64(out)),
           "oracle_extract_tiles")
    return out


def lightsheet(Nx, Ny, dx, lam, n0, NA, z_focus) -> np.ndarray:
    out = np.empty((Ny, Nx), dtype=np.complex128)
    _check(_load().oracle_lightsheet(Nx, Ny, _sf(dx), _sf(lam), _sf(n0), _sf(NA), _sf(z_focus), _p64(out)),
           "oracle_lightsheet")
    return out


def multiplex_annular(pos, phase, amp, NA_in, NA_out, Nx, Ny, dx, lam) -> np.ndarray:
    pos = _f32(pos)
    M = pos.shape[0]
    phase = _f32(phase, (M,))
    amp = _f32(amp, (M,))
    out = np.empty((Ny, Nx), dtype=np.complex128)
    _check(_load().oracle_multiplex_annular(_p32(pos), _p32(phase), _p32(amp), M, _sf(NA_in), _sf(NA_out),
                                            Nx, Ny, _sf(dx), _sf(lam), _p64(out)), "oracle_multiplex_annular")
    return out


def image_formation(S, pos, dx, psf) -> np.ndarray:
    """Camera image of one object plane with a piecewise-constant spatially varying PSF
    (``oracle_image_formation``): S [Ny][Nx], psf [M][T][T]."""
    S = np.ascontiguousarray(S, dtype=np.float64)
    psf = np.ascontiguousarray(psf, dtype=np.float64)
    Ny, Nx = S.shape
    pos = _f32(pos)
    M, T = psf.shape[0], psf.shape[1]
    out = np.empty((Ny, Nx), dtype=np.float64)
    _check(_load().oracle_image_formation(_p64(S), Nx, Ny, _p32(pos), M, _sf(dx), _p64(psf), T, _p64(out)),
           "oracle_image_formation")
    return out
