"""Host-side checks of the C-ABI library that need no GPU: it builds for sm_100a, exports
every symbol ``include/bb.h`` declares, rejects bad arguments before touching the device,
and has no fallback when there is no device."""
import ctypes
import os
import re
import shutil

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "bb.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bb_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
        pytest.skip("nvcc not available")
    from paper_1706_02261_b200 import build, binding
    build.build_library()
    return binding.load()


def test_header_declares_the_boundary():
    syms = declared_symbols()
    for name in ("bb_propagate", "bb_propagate_ex", "bb_propagate_host", "bb_multiplex_psf",
                 "bb_nref_from_dn", "bb_last_error", "bb_version", "bb_shutdown"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_1706_02261_b200 import binding
    for name in declared_symbols():
        assert hasattr(lib, name), "libbiobeam_b200.so does not export %s" % name
    assert set(declared_symbols()) == set(binding.EXPORTS)
    assert lib.bb_version() >= 100


def test_library_holds_sm100a_code_only(lib):
    from paper_1706_02261_b200 import binding
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    import subprocess
    out = subprocess.run([cuobjdump, "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_oracle_and_library_share_nothing():
    """Neither side imports the other; the binding never references the oracle."""
    pkg = os.path.join(ROOT, "paper_1706_02261_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("``oracle``", "").replace("nor the oracle", "").lower() \
                    or f == "workloads.py", "%s mentions the oracle" % f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1706_02261_b200" not in txt and "from paper_1706_02261_b200" not in txt
            assert "bb.h" not in txt


def _opts(lib, batch=1, flags=0, size=None):
    from paper_1706_02261_b200.binding import _Opts
    o = _Opts()
    o.struct_size = ctypes.sizeof(_Opts) if size is None else size
    o.batch = batch
    o.flags = flags
    return o


def test_argument_checks_come_before_any_device_work(lib):
    """Bad arguments return their status without a CUDA call (works on a GPU-less box)."""
    fake = ctypes.c_void_p(4096)
    err = lambda: lib.bb_last_error().decode()
    assert lib.bb_propagate(None, fake, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None) == 1 and "field" in err()
    assert lib.bb_propagate(fake, None, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None) == 1
    assert lib.bb_propagate(fake, fake, 128, 128, 0, 0.1, 0.1, 0.5, 1.33, None) == 1
    assert lib.bb_propagate(fake, fake, 128, 128, 4, -0.1, 0.1, 0.5, 1.33, None) == 1
    assert lib.bb_propagate(fake, fake, 128, 128, 4, 0.1, 0.0, 0.5, 1.33, None) == 1
    assert lib.bb_propagate(fake, fake, 128, 128, 4, 0.1, 0.1, float("nan"), 1.33, None) == 1
    assert lib.bb_propagate(fake, fake, 128, 128, 4, 0.1, 0.1, 0.5, 0.0, None) == 1
    for nx, ny in ((100, 128), (128, 96), (16, 128), (2048, 128), (128, 4096), (0, 128)):
        assert lib.bb_propagate(fake, fake, nx, ny, 4, 0.1, 0.1, 0.5, 1.33, None) == 2, (nx, ny)
    o = _opts(lib, batch=0)
    assert lib.bb_propagate_ex(fake, fake, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None, ctypes.byref(o)) == 1
    o = _opts(lib, flags=64)
    assert lib.bb_propagate_ex(fake, fake, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None, ctypes.byref(o)) == 1
    o = _opts(lib, size=8)
    assert lib.bb_propagate_ex(fake, fake, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None, ctypes.byref(o)) == 1
    o = _opts(lib)
    bad = (ctypes.c_float * 4)(1.33, 1.33, -1.0, 1.33)
    o.nref = ctypes.cast(bad, ctypes.POINTER(ctypes.c_float))
    assert lib.bb_propagate_host(fake, fake, 128, 128, 4, 0.1, 0.1, 0.5, 1.33, None, ctypes.byref(o)) == 1
    assert lib.bb_fft2(None, 128, 128, 1, -1, None) == 1
    assert lib.bb_fft2(fake, 128, 128, 1, 0, None) == 1
    assert lib.bb_fft2(fake, 128, 100, 1, -1, None) == 2
    assert lib.bb_multiplex_psf(None, None, None, 4, 0.8, 128, 128, 0.1, 0.5, fake, None) == 1
    assert lib.bb_multiplex_psf(fake, None, None, 0, 0.8, 128, 128, 0.1, 0.5, fake, None) == 1
    assert lib.bb_multiplex_psf(fake, None, None, 4, -0.8, 128, 128, 0.1, 0.5, fake, None) == 1
    assert lib.bb_nref_from_dn(None, 128, 128, 4, 1.33, 2, None, None) == 1
    assert lib.bb_nref_from_dn_static(None, 128, 128, 4, 1.33, 2, fake, None) == 1
    assert lib.bb_nref_from_dn_static(fake, 128, 128, lib.bb_static_max_nz() + 1, 1.33, 2, fake, None) == 1 \
        and "BB_STATIC_MAX_NZ" in err()
    assert lib.bb_propagator_table(128, 128, 0.1, 0.1, 0.5, 1.33, None, None) == 1


def test_no_fallback_without_a_device(lib):
    """On a box without a usable sm_100 device a valid call fails loudly (there is no CPU path)."""
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    fake = ctypes.c_void_p(4096)
    rc = lib.bb_fft2(fake, 128, 128, 1, -1, None)
    assert rc in (3, 5) and lib.bb_last_error().decode() != ""


def test_binding_rejects_wrong_tensors(lib):
    from paper_1706_02261_b200 import binding as bb
    f = torch.zeros((64, 64), dtype=torch.complex64)
    dn = torch.zeros((4, 64, 32), dtype=torch.float32)
    with pytest.raises(TypeError):
        bb.propagate(f, dn, 0.1, 0.1, 0.5, 1.33)
    with pytest.raises(TypeError):
        bb.propagate(f.to(torch.complex128), torch.zeros((4, 64, 64)), 0.1, 0.1, 0.5, 1.33)
    with pytest.raises(TypeError):
        bb.propagate(f, torch.zeros((4, 64, 64), dtype=torch.float64), 0.1, 0.1, 0.5, 1.33)
    with pytest.raises(TypeError):
        bb.propagate(f, torch.zeros((4, 64, 64)), 0.1, 0.1, 0.5, 1.33, intensity=torch.zeros((3, 64, 64)))
