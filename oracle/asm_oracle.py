"""fp64 CPU oracle for ASM forward + adjoint: Python face of oracle/asm_oracle.c.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from
paper_2505_22313_b200 and shares no code with the CUDA path.

Each function follows one step of SURVEY.md section 8(c)'s oracle algorithm (O0..O10), i.e. the
paper's Eq. (1)-(4), the row-column 2-D DFT of PAPER.md:200 and the
back-propagation of PAPER.md:124/200, in that order, one C call per step so the composition can
be checked against the paper by eye.  numpy only holds the arrays.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_i64, _dbl, _int, _ptr = C.c_int64, C.c_double, C.c_int, C.c_void_p
_lib.oracle_dft1.argtypes = [_i64, _ptr, _ptr, _int]
_lib.oracle_dft1.restype = _int
_lib.oracle_dft2.argtypes = [_i64, _i64, _ptr, _int]
_lib.oracle_dft2.restype = _int
_lib.oracle_phase_field.argtypes = [_i64, _ptr, _dbl, _dbl, _ptr]
_lib.oracle_phase_field.restype = None
_lib.oracle_transfer_multiply.argtypes = [_i64, _i64, _ptr, _dbl, _dbl, _dbl, _int]
_lib.oracle_transfer_multiply.restype = None
_lib.oracle_transfer_function.argtypes = [_i64, _i64, _ptr, _dbl, _dbl, _dbl]
_lib.oracle_transfer_function.restype = None
_lib.oracle_gaussian_multiply.argtypes = [_i64, _i64, _ptr, _dbl]
_lib.oracle_gaussian_multiply.restype = None
_lib.oracle_intensity.argtypes = [_i64, _ptr, _ptr]
_lib.oracle_intensity.restype = None
_lib.oracle_l2_loss.argtypes = [_i64, _ptr, _ptr]
_lib.oracle_l2_loss.restype = _dbl
_lib.oracle_seed.argtypes = [_i64, _ptr, _ptr, _ptr]
_lib.oracle_seed.restype = None
_lib.oracle_phase_adjoint.argtypes = [_i64, _ptr, _ptr, _dbl, _dbl, _ptr]
_lib.oracle_phase_adjoint.restype = None
_lib.oracle_num_threads.argtypes = []
_lib.oracle_num_threads.restype = _int


def _p(a: np.ndarray):
    return a.ctypes.data_as(_ptr)


def _c128(a) -> np.ndarray:
    """fresh C-contiguous complex128 copy"""
    return np.array(a, dtype=np.complex128, order="C", copy=True)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_lib.oracle_num_threads())


# --------------------------------------------------------------------------------------------
# DFTs (O3 / O5)
# --------------------------------------------------------------------------------------------
def dft1(x, inverse: bool = False) -> np.ndarray:
    """X[k] = sum_n x[n] exp(-/+ 2 pi i k n / N), unnormalised in both directions."""
    x = _c128(x)
    out = np.empty_like(x)
    rc = _lib.oracle_dft1(x.size, _p(x), _p(out), int(inverse))
    if rc:
        raise RuntimeError(f"oracle_dft1 failed ({rc})")
    return out


def dft2(a, inverse: bool = False) -> np.ndarray:
    """O3 (forward, unnormalised, sign -) / O5 (inverse, 1/N, sign +); rows then columns."""
    a = _c128(a)
    if a.ndim != 2:
        raise ValueError("dft2 wants a 2-D array [ny, nx]")
    rc = _lib.oracle_dft2(a.shape[0], a.shape[1], _p(a), int(inverse))
    if rc:
        raise RuntimeError(f"oracle_dft2 failed ({rc})")
    return a


def _dft2_inplace(a: np.ndarray, inverse: bool) -> None:
    rc = _lib.oracle_dft2(a.shape[0], a.shape[1], _p(a), int(inverse))
    if rc:
        raise RuntimeError(f"oracle_dft2 failed ({rc})")


# --------------------------------------------------------------------------------------------
# Steps
# --------------------------------------------------------------------------------------------
def prefilter(h, sigma_px: float) -> np.ndarray:
    """O0 (and, being self-adjoint, O10): Re IDFT2( Ghat * DFT2(h) ), Ghat the periodic Gaussian
    spectrum exp(-2 pi^2 sigma^2 ((kx/Nx)^2 + (ky/Ny)^2)).  BASELINE.json config 3; the form of
    the MTF model of PAPER.md:184."""
    a = _c128(h)
    _dft2_inplace(a, False)
    _lib.oracle_gaussian_multiply(a.shape[0], a.shape[1], _p(a), float(sigma_px))
    _dft2_inplace(a, True)
    return np.ascontiguousarray(a.real)


def phase_field(h, lam: float, n_refr: float) -> np.ndarray:
    """O1 + O2: u0 = exp(i 2 pi (n-1) h / lambda).  Eq. (1), (2) with E_in = 1."""
    h = _f64(h)
    u0 = np.empty(h.shape, dtype=np.complex128)
    _lib.oracle_phase_field(h.size, _p(h), float(lam), float(n_refr), _p(u0))
    return u0


def transfer_function(ny: int, nx: int, pitch: float, lam: float, z: float) -> np.ndarray:
    """H[ky,kx] in DFT bin order (O4)."""
    H = np.empty((ny, nx), dtype=np.complex128)
    _lib.oracle_transfer_function(ny, nx, _p(H), float(pitch), float(lam), float(z))
    return H


def propagate(u0, pitch: float, lam: float, z: float, conj_h: bool = False) -> np.ndarray:
    """O3-O5, Eq. (3): IDFT2( H (or conj H) * DFT2(u0) ).  With conj_h this is the adjoint A^H
    (O8): the 1/N of the forward's inverse and the N of its adjoint cancel into one IDFT2."""
    a = _c128(u0)
    _dft2_inplace(a, False)
    _lib.oracle_transfer_multiply(a.shape[0], a.shape[1], _p(a), float(pitch), float(lam),
                                  float(z), int(conj_h))
    _dft2_inplace(a, True)
    return a


def intensity(u) -> np.ndarray:
    """O6: I = Re(u)^2 + Im(u)^2."""
    u = np.ascontiguousarray(u, dtype=np.complex128)
    out = np.empty(u.shape, dtype=np.float64)
    _lib.oracle_intensity(u.size, _p(u), _p(out))
    return out


def l2_loss(inten, target) -> float:
    """O6: (1/N) sum (I - T)^2 for one wavelength."""
    inten, target = _f64(inten), _f64(target)
    return float(_lib.oracle_l2_loss(inten.size, _p(inten), _p(target)))


# --------------------------------------------------------------------------------------------
# Whole path
# --------------------------------------------------------------------------------------------
def forward(h, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float,
            target=None, sigma_px: float = 0.0, keep_field: bool = True) -> dict:
    """O0-O6 for every wavelength.  Returns dict(I=[L,ny,nx], u=[L,ny,nx] or None, loss=float or
    None, h_eff=[ny,nx]) with loss = sum_lambda (1/N) sum (I_lambda - T)^2 when target is given."""
    h = _f64(h)
    h_eff = prefilter(h, sigma_px) if sigma_px > 0.0 else h                      # O0
    L = len(lambdas)
    I = np.empty((L,) + h.shape, dtype=np.float64)
    u_all = np.empty((L,) + h.shape, dtype=np.complex128) if keep_field else None
    loss = 0.0 if target is not None else None
    for l, (lam, n) in enumerate(zip(lambdas, n_refr)):
        u0 = phase_field(h_eff, lam, n)                                          # O1, O2
        u = propagate(u0, pitch, lam, z)                                         # O3, O4, O5
        del u0
        I[l] = intensity(u)                                                      # O6
        if keep_field:
            u_all[l] = u
        if target is not None:
            loss += l2_loss(I[l], target)                                        # O6
    return {"I": I, "u": u_all, "loss": loss, "h_eff": h_eff}


def adjoint(h, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float,
            target=None, dLdI=None, sigma_px: float = 0.0) -> np.ndarray:
    """O7-O10: dL/dh for L = sum_lambda (1/N) sum (I_lambda - T)^2 (target given) or for a caller's
    dL/dI [L,ny,nx].  Recomputes the forward field (the oracle keeps nothing between calls)."""
    if (target is None) == (dLdI is None):
        raise ValueError("give exactly one of target, dLdI")
    h = _f64(h)
    npts = h.size
    h_eff = prefilter(h, sigma_px) if sigma_px > 0.0 else h                      # O0
    grad = np.zeros(h.shape, dtype=np.float64)
    for l, (lam, n) in enumerate(zip(lambdas, n_refr)):
        u0 = phase_field(h_eff, lam, n)                                          # O1, O2
        u = propagate(u0, pitch, lam, z)                                         # O3-O5
        if target is not None:
            gI = 2.0 * (intensity(u) - _f64(target)) / npts                      # O7: dL/dI
        else:
            gI = _f64(dLdI[l])
        gu = np.empty_like(u)
        _lib.oracle_seed(npts, _p(u), _p(gI), _p(gu))                            # O7: 2 gI u
        del u, gI
        gu0 = propagate(gu, pitch, lam, z, conj_h=True)                          # O8
        del gu
        _lib.oracle_phase_adjoint(npts, _p(u0), _p(gu0), float(lam), float(n), _p(grad))  # O9
    if sigma_px > 0.0:
        grad = prefilter(grad, sigma_px)                                         # O10
    return grad
