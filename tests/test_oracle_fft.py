"""Pin P1: the oracle's own FFT against things that are not the oracle's FFT.

* the O(N^2) DFT written straight from the definition (oracle_dft2_bruteforce is a
  separate routine in the same C file: four nested loops over cos/sin, no FFT code);
* numpy's pocketfft (an independent library);
* a DFT evaluated here in numpy from the definition (outer-product matrices);
* structural facts: delta -> constant, single mode -> delta at the right bin (pins the
  sign convention and the [y][x] index order), inverse carries 1/(Nx Ny).
"""
import numpy as np
import pytest

from conftest import rel_l2


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _dft2_numpy_definition(a, sign):
    Ny, Nx = a.shape
    y = np.arange(Ny)
    x = np.arange(Nx)
    Wy = np.exp(sign * 2j * np.pi * np.outer(y, y) / Ny)   # [q][y]
    Wx = np.exp(sign * 2j * np.pi * np.outer(x, x) / Nx)   # [x][p]
    out = Wy @ a @ Wx
    if sign > 0:
        out = out / (Nx * Ny)
    return out


@pytest.mark.parametrize("shape", [(4, 4), (8, 8), (8, 16), (16, 16), (32, 32), (2, 64), (1, 8)])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft2_vs_bruteforce_and_definition(oracle_mod, shape, sign):
    a = _rand(shape, seed=hash(shape) % 1000 + (sign > 0))
    got = oracle_mod.fft2(a, sign)
    assert rel_l2(got, oracle_mod.dft2_bruteforce(a, sign)) < 1e-12
    assert rel_l2(got, _dft2_numpy_definition(a, sign)) < 1e-12


@pytest.mark.parametrize("shape", [(128, 128), (256, 64), (512, 1024)])
def test_fft2_vs_pocketfft(oracle_mod, shape):
    a = _rand(shape, seed=7)
    assert rel_l2(oracle_mod.fft2(a, -1), np.fft.fft2(a)) < 1e-13
    assert rel_l2(oracle_mod.fft2(a, +1), np.fft.ifft2(a)) < 1e-13


@pytest.mark.parametrize("n", [1, 2, 4, 64, 2048])
def test_fft1_vs_pocketfft(oracle_mod, n):
    a = _rand((n,), seed=n)
    assert rel_l2(oracle_mod.fft1(a, -1), np.fft.fft(a)) < 1e-13
    assert rel_l2(oracle_mod.fft1(a, +1), np.fft.ifft(a)) < 1e-13


def test_roundtrip_and_normalisation(oracle_mod):
    a = _rand((64, 32), seed=3)
    assert rel_l2(oracle_mod.fft2(oracle_mod.fft2(a, -1), +1), a) < 1e-13
    # forward is unnormalised: DC bin of an all-ones array is Nx*Ny (reading A7)
    ones = np.ones((16, 8), dtype=np.complex128)
    F = oracle_mod.fft2(ones, -1)
    assert abs(F[0, 0] - 128.0) < 1e-12 and np.abs(F).sum() - 128.0 < 1e-10
    # inverse carries 1/(Nx Ny): delta at DC -> constant 1/(Nx Ny)
    d = np.zeros((16, 8), dtype=np.complex128)
    d[0, 0] = 1.0
    assert np.allclose(oracle_mod.fft2(d, +1), 1.0 / 128.0, atol=1e-15)


def test_sign_convention_and_axis_order(oracle_mod):
    """u = exp(+2 pi i (p x/Nx + q y/Ny)) must land in bin [q][p] of the forward transform
    (kernel exp(-i k.r), array [y][x]); a transposed or sign-flipped FFT fails this."""
    Ny, Nx, p, q = 16, 32, 5, 3
    y, x = np.mgrid[0:Ny, 0:Nx]
    u = np.exp(2j * np.pi * (p * x / Nx + q * y / Ny))
    F = oracle_mod.fft2(u, -1)
    assert abs(F[q, p] - Nx * Ny) < 1e-9
    F[q, p] = 0
    assert np.abs(F).max() < 1e-9


def test_non_power_of_two_rejected(oracle_mod):
    with pytest.raises(ValueError):
        oracle_mod.fft2(np.zeros((6, 8), dtype=np.complex128), -1)
