"""fp64 CPU oracle for the design loop around the ASM path.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline
leg may import this.  It imports nothing from paper_2505_22313_b200 and shares no code with the CUDA
path.  Plain numpy in double precision, one function per step, in the paper's order:

  super-resolved design variable  PAPER.md:51, 141 ("zero-order interpolation, i.e., nearest upsampling"),
                                  259-260, 264: the optimised layout l lives on a coarse feature grid and is
                                  nearest-neighbour up-sampled r x r to the simulation grid; 10-bit / 8-bit
                                  gray-level layouts are levels times a height step.
  penalty, Eq. (6) PAPER.md:130-139   L_p = L_si-mse + beta L_energy, beta = 5e-3.
  optimiser        PAPER.md:130, 141  Adam [Kingma 2014], learning rate 1e-2 on a cosine schedule that decays
                                      to zero in 3000 iterations.

READING (flagged in DESIGN.md "Readings"): the definitions of L_si-mse and L_energy are "given in the
Supplementary Material", which is not in /root/reference.  This oracle takes
    L_si-mse(I, T) = (1/N) sum (s I - T)^2   with the least-squares scale  s = <I,T> / <I,I>
(the scale that minimises it, so the term is invariant under I -> alpha I), and
    L_energy(I)    = 1 - (1/N) sum I
(the fraction of the unit incident energy that does not arrive: >= 0 because |H| <= 1), per wavelength,
summed over wavelengths as Eq. (4) says.

Pins (tests/test_oracle_design.py, -m "not gpu"): scale invariance and optimality of s; the energy term on a
lossless grid; dL/dI and the whole chain dL/dl against central finite differences; the up-sample / sum-pool
pair as an adjoint pair (<U l, g> = <l, U^T g>) and against np.kron; Adam against its closed-form first step
and against torch.optim.Adam + CosineAnnealingLR (a library implementation) over several steps.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from . import asm_oracle as asm


# --------------------------------------------------------------------------------------------
# super-resolved design variable
# --------------------------------------------------------------------------------------------
def layout_to_height(layout, step: float = 1.0) -> np.ndarray:
    """Gray-level layout (any integer or float dtype) -> heights in metres: h = level * step."""
    return np.asarray(layout, dtype=np.float64) * float(step)


def upsample_nearest(coarse, r: int) -> np.ndarray:
    """U: [Y, X] -> [Y r, X r], every coarse feature repeated r x r (zero-order interpolation)."""
    c = np.asarray(coarse, dtype=np.float64)
    out = np.empty((c.shape[0] * r, c.shape[1] * r), dtype=np.float64)
    for dy in range(r):
        for dx in range(r):
            out[dy::r, dx::r] = c
    return out


def sumpool(fine, r: int) -> np.ndarray:
    """U^T: [Y r, X r] -> [Y, X], the sum over every r x r block (the adjoint of upsample_nearest)."""
    f = np.asarray(fine, dtype=np.float64)
    out = np.zeros((f.shape[0] // r, f.shape[1] // r), dtype=np.float64)
    for dy in range(r):
        for dx in range(r):
            out += f[dy::r, dx::r]
    return out


# --------------------------------------------------------------------------------------------
# Eq. (6): L_p = L_si-mse + beta L_energy  (one wavelength)
# --------------------------------------------------------------------------------------------
def simse_energy_loss(inten, target, beta: float):
    """-> (L_p, s, dL_p/dI).  s = <I,T>/<I,I>; dL/dI = (2 s / N)(s I - T) - beta / N: the term through
    ds/dI vanishes because s minimises the first term (d/ds = 0)."""
    I = np.asarray(inten, dtype=np.float64)
    T = np.asarray(target, dtype=np.float64)
    n = I.size
    it, ii = float(np.sum(I * T)), float(np.sum(I * I))
    s = it / ii if ii > 0.0 else 0.0
    r = s * I - T
    loss = float(np.sum(r * r)) / n + beta * (1.0 - float(np.sum(I)) / n)
    gI = (2.0 * s / n) * r - beta / n
    return loss, s, gI


# --------------------------------------------------------------------------------------------
# whole path with the design-loop pieces
# --------------------------------------------------------------------------------------------
def forward(layout, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float, target,
            beta: float, upsample: int = 1, step: float = 1.0, sigma_px: float = 0.0) -> dict:
    """layout [Y, X] -> h = U(level * step) -> Eq. (1)-(3) per wavelength (asm_oracle) -> I -> sum_lambda L_p."""
    h = upsample_nearest(layout_to_height(layout, step), upsample)
    f = asm.forward(h, pitch, lambdas, n_refr, z, sigma_px=sigma_px, keep_field=False)
    loss, scales = 0.0, []
    for l in range(len(lambdas)):
        lp, s, _ = simse_energy_loss(f["I"][l], target, beta)
        loss += lp
        scales.append(s)
    return {"I": f["I"], "loss": loss, "scales": scales, "h": h}


def adjoint(layout, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float], z: float, target,
            beta: float, upsample: int = 1, step: float = 1.0, sigma_px: float = 0.0) -> np.ndarray:
    """dL/d(coarse height) [Y, X] = U^T dL/dh: dL/dI from Eq. (6) per wavelength, back through the ASM
    adjoint (asm_oracle.adjoint, caller-supplied dL/dI), then the sum-pool."""
    h = upsample_nearest(layout_to_height(layout, step), upsample)
    f = asm.forward(h, pitch, lambdas, n_refr, z, sigma_px=sigma_px, keep_field=False)
    gI = np.stack([simse_energy_loss(f["I"][l], target, beta)[2] for l in range(len(lambdas))])
    g = asm.adjoint(h, pitch, lambdas, n_refr, z, dLdI=gI, sigma_px=sigma_px)
    return sumpool(g, upsample)


def adjoint_l2(layout, pitch, lambdas, n_refr, z, target, upsample: int = 1, step: float = 1.0,
               sigma_px: float = 0.0) -> np.ndarray:
    """The same with the plain L2 penalty of the five benchmark configurations."""
    h = upsample_nearest(layout_to_height(layout, step), upsample)
    return sumpool(asm.adjoint(h, pitch, lambdas, n_refr, z, target=target, sigma_px=sigma_px), upsample)


# --------------------------------------------------------------------------------------------
# Adam with a cosine learning-rate schedule (Kingma & Ba 2014, Algorithm 1)
# --------------------------------------------------------------------------------------------
def cosine_lr(lr0: float, it: int, total: int) -> float:
    """lr0 (1 + cos(pi it / total)) / 2 for the 0-based iteration `it`: lr0 at 0, zero at `total`."""
    return lr0 * 0.5 * (1.0 + np.cos(np.pi * min(it, total) / total))


def adam_step(theta, grad, m, v, lr0: float, beta1: float, beta2: float, eps: float, it: int, total: int):
    """One Adam update of the design variable, 0-based iteration `it` (bias correction uses t = it + 1):
    m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;  theta <- theta - lr_it (m / (1-b1^t)) / (sqrt(v / (1-b2^t)) + eps)."""
    g = np.asarray(grad, dtype=np.float64)
    m = beta1 * np.asarray(m, dtype=np.float64) + (1.0 - beta1) * g
    v = beta2 * np.asarray(v, dtype=np.float64) + (1.0 - beta2) * g * g
    t = it + 1
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    theta = np.asarray(theta, dtype=np.float64) - cosine_lr(lr0, it, total) * mhat / (np.sqrt(vhat) + eps)
    return theta, m, v
