"""fp64 CPU oracle for linear (non-circular) ASM propagation: 2x zero padding and the band-limited transfer
function.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may
import this.  It imports nothing from paper_2505_22313_b200 and shares no code with the CUDA path.  Plain numpy
in double precision around the steps of oracle/asm_oracle (its DFT, its transfer multiply).

What it computes, in the order of the method the paper cites for it (Matsushima & Shimobaba 2009,
"Band-limited angular spectrum method ..."; the paper itself only says that it propagates with the ASM,
PAPER.md:104-108, and names the grids of Table 2):

  1. the aperture field u0 [ny, nx] is embedded in the top-left corner of a [2 ny, 2 nx] window, zero elsewhere
     (zero amplitude, NOT zero phase: outside the DOE no light enters the window);
  2. the window is propagated circularly: F^-1{ F{.} (x) H' } with H' = H on the window's own frequency grid
     (f = k / (2 n pitch)), clipped to the rectangle |fx| <= u_limit, |fy| <= v_limit when band_limit is set;
  3. the result is cropped to the aperture [ny, nx]; I, the loss (mean over the aperture) and dL/dh live there.

  u_limit = 1 / ( lambda sqrt( (2 du z)^2 + 1 ) ),  du = 1 / (2 nx pitch)  (the window's frequency sampling),
  v_limit likewise with dv = 1 / (2 ny pitch): beyond it the phase of H advances by more than pi between
  neighbouring frequency samples, i.e. the sampled H aliases.

READINGS: aperture in the corner rather than centred (a circular shift of input and output by the
same amount, i.e. the same operator); the limit is applied per axis as in the reference; `<=` keeps the bin that
sits exactly on the limit.

Pins (tests/test_oracle_linear.py, -m "not gpu"): the padded result against the brute-force spatial (linear)
convolution with the impulse response on tiny grids -- no wrap-around; the band limit against the local-frequency
criterion evaluated by finite differences of H's unwrapped phase; adjoint against central finite differences and
<A x, y> = <x, A^H y>.
"""
from __future__ import annotations

from typing import Sequence

import numpy as np

from . import asm_oracle as asm


def band_limits(ny: int, nx: int, pitch: float, lam: float, z: float):
    """(u_limit, v_limit) of the [2 ny, 2 nx] window: 1 / (lambda sqrt((2 du z)^2 + 1))."""
    du, dv = 1.0 / (2.0 * nx * pitch), 1.0 / (2.0 * ny * pitch)
    return (1.0 / (lam * np.sqrt((2.0 * du * z) ** 2 + 1.0)), 1.0 / (lam * np.sqrt((2.0 * dv * z) ** 2 + 1.0)))


def window_frequencies(n: int, pitch: float) -> np.ndarray:
    """signed-bin frequencies of a length-n DFT: k / (n pitch), k < (n+1)/2 ? k : k - n (asm_oracle's convention)."""
    k = np.arange(n)
    return np.where(k < (n + 1) // 2, k, k - n) / (n * pitch)


def band_mask(ny: int, nx: int, pitch: float, lam: float, z: float) -> np.ndarray:
    """[2 ny, 2 nx] boolean mask of the frequency bins the band limit keeps."""
    ul, vl = band_limits(ny, nx, pitch, lam, z)
    fx, fy = window_frequencies(2 * nx, pitch), window_frequencies(2 * ny, pitch)
    return (np.abs(fy)[:, None] <= vl) & (np.abs(fx)[None, :] <= ul)


def propagate_linear(u0, pitch: float, lam: float, z: float, band_limit: bool = True, conj_h: bool = False) -> np.ndarray:
    """Steps 1-3 for one wavelength: [ny, nx] complex -> [ny, nx] complex.  With conj_h the adjoint operator
    (crop^T = zero embedding, pad^T = crop: the same three steps with conj H)."""
    u0 = np.asarray(u0, dtype=np.complex128)
    ny, nx = u0.shape
    w = np.zeros((2 * ny, 2 * nx), dtype=np.complex128)
    w[:ny, :nx] = u0                                                   # 1. embed, zero amplitude outside
    W = asm.dft2(w)                                                    # 2. F
    H = asm.transfer_function(2 * ny, 2 * nx, pitch, lam, z)           #    H on the window's grid (evanescent bins 0)
    if band_limit:
        H = np.where(band_mask(ny, nx, pitch, lam, z), H, 0.0)
    W *= np.conj(H) if conj_h else H
    w = asm.dft2(W, inverse=True)                                      #    F^-1
    return np.ascontiguousarray(w[:ny, :nx])                           # 3. crop


def forward(h, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float, target=None,
            band_limit: bool = True) -> dict:
    """Eq. (1)-(4) with the padded propagation: I [L, ny, nx], u [L, ny, nx], loss = sum_lambda mean_aperture (I - T)^2."""
    h = np.asarray(h, dtype=np.float64)
    L = len(lambdas)
    I = np.empty((L,) + h.shape)
    u_all = np.empty((L,) + h.shape, dtype=np.complex128)
    loss = 0.0 if target is not None else None
    for l, (lam, n) in enumerate(zip(lambdas, n_refr)):
        u = propagate_linear(asm.phase_field(h, lam, n), pitch, lam, z, band_limit)
        u_all[l] = u
        I[l] = asm.intensity(u)
        if target is not None:
            loss += asm.l2_loss(I[l], target)
    return {"I": I, "u": u_all, "loss": loss}


def adjoint(h, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float, target=None, dLdI=None,
            band_limit: bool = True) -> np.ndarray:
    """dL/dh [ny, nx] for the L2 loss over the aperture (target) or a caller's dL/dI [L, ny, nx]."""
    if (target is None) == (dLdI is None):
        raise ValueError("give exactly one of target, dLdI")
    h = np.asarray(h, dtype=np.float64)
    grad = np.zeros(h.shape)
    for l, (lam, n) in enumerate(zip(lambdas, n_refr)):
        u0 = asm.phase_field(h, lam, n)
        u = propagate_linear(u0, pitch, lam, z, band_limit)
        gI = 2.0 * (asm.intensity(u) - np.asarray(target, dtype=np.float64)) / h.size if target is not None \
            else np.asarray(dLdI[l], dtype=np.float64)
        gu0 = propagate_linear(2.0 * gI * u, pitch, lam, z, band_limit, conj_h=True)
        grad += (2.0 * np.pi * (n - 1.0) / lam) * np.imag(np.conj(u0) * gu0)
    return grad
