"""Pins for the oracle's own DFT (oracle steps O3/O5; Eq. 3).

P-a: the DFT *definition* evaluated as an O(N^2) matrix product (sign -, unnormalised forward;
sign +, 1/N inverse), on power-of-two, radix-3, 5-smooth and prime shapes; plus numpy.fft as an
independent library cross-check on a size too big for the brute force.  A wrong sign, a missing
1/N, a transposed axis or a bad twiddle index fails here.
"""
import numpy as np
import pytest

from oracle import asm_oracle as orc


def dft_matrix(n, sign):
    k = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(k, k) / n)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 8, 9, 12, 16, 27, 49, 64, 96, 97, 100, 384])
def test_dft1_matches_definition(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    fwd = dft_matrix(n, -1) @ x
    inv = dft_matrix(n, +1) @ x            # oracle_dft1 is unnormalised both ways
    scale = max(1.0, np.abs(fwd).max())
    assert np.abs(orc.dft1(x) - fwd).max() / scale < 1e-12
    assert np.abs(orc.dft1(x, inverse=True) - inv).max() / scale < 1e-12


@pytest.mark.parametrize("shape", [(2, 2), (8, 8), (48, 36), (27, 64), (30, 50), (64, 64),
                                   (7, 11), (1, 16), (16, 1), (24, 32)])
def test_dft2_matches_bruteforce(shape):
    ny, nx = shape
    rng = np.random.default_rng(ny * 1000 + nx)
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    # U[ky,kx] = sum_y sum_x a[y,x] exp(-2 pi i (kx x/Nx + ky y/Ny))
    fwd = dft_matrix(ny, -1) @ a @ dft_matrix(nx, -1).T
    inv = dft_matrix(ny, +1) @ a @ dft_matrix(nx, +1).T / (ny * nx)
    assert np.abs(orc.dft2(a) - fwd).max() / np.abs(fwd).max() < 1e-12
    assert np.abs(orc.dft2(a, inverse=True) - inv).max() / np.abs(inv).max() < 1e-12


def test_dft2_axes_not_transposed():
    """a single spatial frequency along x must land in row 0, column kx (x is the fast axis)."""
    ny, nx, kx0 = 12, 16, 3
    x = np.arange(nx)
    a = np.tile(np.exp(2j * np.pi * kx0 * x / nx), (ny, 1))
    U = orc.dft2(a)
    expect = np.zeros((ny, nx), complex)
    expect[0, kx0] = ny * nx
    assert np.abs(U - expect).max() < 1e-9


def test_dft2_roundtrip_and_library():
    rng = np.random.default_rng(7)
    a = rng.standard_normal((384, 512)) + 1j * rng.standard_normal((384, 512))
    U = orc.dft2(a)
    ref = np.fft.fft2(a)
    assert np.abs(U - ref).max() / np.abs(ref).max() < 1e-13
    assert np.abs(orc.dft2(U, inverse=True) - a).max() < 1e-12


def test_dft2_linearity_and_shift_theorem():
    rng = np.random.default_rng(8)
    a = rng.standard_normal((18, 20)) + 1j * rng.standard_normal((18, 20))
    sy, sx = 5, 3
    U = orc.dft2(a)
    Us = orc.dft2(np.roll(a, (sy, sx), axis=(0, 1)))
    ky = np.arange(18)[:, None]
    kx = np.arange(20)[None, :]
    assert np.abs(Us - U * np.exp(-2j * np.pi * (ky * sy / 18 + kx * sx / 20))).max() < 1e-10
