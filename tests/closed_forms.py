"""Closed forms used as size-independent pins (SURVEY.md 8(c) P-i, P-j), evaluated in fp64 with numpy /
scipy only -- no code from oracle/ or from the CUDA path.  tests/test_oracle_physics.py checks them
against the oracle on small grids; tests/test_parity_gpu.py evaluates them at sampled points of the
full-size grids (C4, C5), where no host oracle fits."""
import numpy as np
from scipy.special import jv


def signed_bin(k, n):
    """DFT bin k (any integer) -> its signed representative in [-n/2, n/2) (numpy fftfreq order)."""
    k = np.mod(k, n)
    return np.where(k < (n + 1) // 2, k, k - n)


def transfer(kx, ky, ny, nx, pitch, lam, z):
    """H at signed bins (kx, ky): exp(i 2 pi z sqrt(1/lam^2 - fx^2 - fy^2)), 0 where evanescent."""
    fx = np.asarray(kx, dtype=np.float64) / (nx * pitch)
    fy = np.asarray(ky, dtype=np.float64) / (ny * pitch)
    arg = 1.0 / lam ** 2 - fx ** 2 - fy ** 2
    return np.where(arg >= 0, np.exp(2j * np.pi * z * np.sqrt(np.maximum(arg, 0.0))), 0.0)


def grating_phase(ny, nx, a, b, m1, m2, c, y, x):
    """Phi = c + m1 sin(2 pi a x/nx) + m2 sin(2 pi b y/ny) with the arguments reduced exactly (integers)."""
    tx = np.mod(a * np.asarray(x, dtype=np.int64), nx) / float(nx)
    ty = np.mod(b * np.asarray(y, dtype=np.int64), ny) / float(ny)
    return c + m1 * np.sin(2 * np.pi * tx) + m2 * np.sin(2 * np.pi * ty)


def grating_field(ny, nx, pitch, lam, z, a, b, m1, m2, c, sy, sx, K=25):
    """P-j: u0 = exp(i Phi) = e^{ic} sum_k sum_l J_k(m1) J_l(m2) e^{2 pi i (k a x/nx + l b y/ny)} (Jacobi-Anger).
    On the grid every term is the DFT basis vector of bin (k a mod nx, l b mod ny), an eigenvector of the
    circular propagation operator, so u = e^{ic} sum J_k J_l H(wrap(k a), wrap(l b)) e^{...}: exact for any
    a, b (orders that alias are propagated at their aliased frequency, as the DFT does).  Evaluated at the
    sample points (sy, sx); J_K(m) must be negligible at the truncation K."""
    ks = np.arange(-K, K + 1)
    Hkl = transfer(signed_bin(ks * a, nx)[None, :], signed_bin(ks * b, ny)[:, None], ny, nx, pitch, lam, z)  # [l, k]
    Mkl = Hkl * jv(ks, m2)[:, None] * jv(ks, m1)[None, :]
    sx = np.asarray(sx, dtype=np.int64)
    sy = np.asarray(sy, dtype=np.int64)
    ex = np.exp(2j * np.pi * (np.mod(ks[None, :] * a * sx[:, None], nx) / float(nx)))   # [s, k]
    ey = np.exp(2j * np.pi * (np.mod(ks[None, :] * b * sy[:, None], ny) / float(ny)))   # [s, l]
    return np.exp(1j * c) * np.einsum("sl,lk,sk->s", ey, Mkl, ex), Hkl
