"""Pins for oracle/linear_oracle.py: 2x zero-padded, band-limited ASM propagation
(Matsushima & Shimobaba 2009).  None of the pins re-types the oracle's formula: brute-force linear
convolution in the spatial domain (numpy.fft only supplies the impulse response), the sampling criterion behind
the band limit checked by finite differences of H's phase, finite differences and <A x, y> = <x, A^H y>."""
import numpy as np
import pytest

from oracle import asm_oracle as asm
from oracle import linear_oracle as lin

PITCH, LAM = 0.4e-6, 550e-9


@pytest.mark.parametrize("ny,nx,z,bl", [(6, 5, 3e-6, False), (8, 12, 20e-6, False), (8, 12, 20e-6, True), (9, 7, 60e-6, True)])
def test_padded_propagation_is_the_linear_convolution_with_the_impulse_response(ny, nx, z, bl):
    """out[y, x] = sum_{y', x'} u0[y', x'] k[y - y', x - x'] with k the window's impulse response and NO index
    wrapping inside the aperture: every offset |y - y'| < ny, |x - x'| < nx is a distinct sample of k."""
    rng = np.random.default_rng(ny * 100 + nx)
    u0 = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    H = asm.transfer_function(2 * ny, 2 * nx, PITCH, LAM, z)
    if bl:
        H = H * lin.band_mask(ny, nx, PITCH, LAM, z)
    k = np.fft.ifft2(H)                                   # library inverse DFT: impulse response of the window
    ref = np.zeros((ny, nx), dtype=np.complex128)
    for y in range(ny):
        for x in range(nx):
            s = 0.0
            for yp in range(ny):
                for xp in range(nx):
                    s += u0[yp, xp] * k[(y - yp) % (2 * ny), (x - xp) % (2 * nx)]
            ref[y, x] = s
    out = lin.propagate_linear(u0, PITCH, LAM, z, band_limit=bl)
    assert np.abs(out - ref).max() <= 1e-12 * np.abs(ref).max()


def test_no_wrap_around_unlike_the_circular_operator():
    """A point source in one corner: circular propagation on the bare grid folds the far side of its diffraction
    pattern back in, the padded operator does not (it equals the window's impulse response there)."""
    ny = nx = 16
    z = 40e-6
    u0 = np.zeros((ny, nx), dtype=np.complex128)
    u0[0, 0] = 1.0
    out = lin.propagate_linear(u0, PITCH, LAM, z, band_limit=False)
    k = np.fft.ifft2(asm.transfer_function(2 * ny, 2 * nx, PITCH, LAM, z))
    assert np.abs(out - k[:ny, :nx]).max() < 1e-13
    circ = asm.propagate(u0, PITCH, LAM, z)
    assert np.abs(circ - out).max() > 1e-3               # the two operators genuinely differ


@pytest.mark.parametrize("n,z", [(64, 200e-6), (256, 2e-3), (48, 5e-3)])
def test_band_limit_is_where_the_sampled_phase_of_H_starts_to_alias(n, z):
    """Kept bins advance H's phase by at most pi per frequency sample (the sampling criterion), the clipped ones by
    more: checked with a central difference of the phase 2 pi z sqrt(1/lambda^2 - u^2) at every bin."""
    ul, vl = lin.band_limits(n, n, PITCH, LAM, z)
    assert abs(ul - vl) < 1e-9 * ul
    du = 1.0 / (2 * n * PITCH)
    u = np.abs(lin.window_frequencies(2 * n, PITCH))
    prop = u < 1.0 / LAM - 2 * du                         # inside the propagating band, away from its edge
    phase = lambda f: 2 * np.pi * z * np.sqrt(1.0 / LAM ** 2 - f ** 2)
    eps = du * 1e-3
    adv = np.abs(phase(u[prop] + eps) - phase(u[prop] - eps)) / (2 * eps) * du   # |d phase / du| du
    kept = u[prop] <= ul
    assert kept.any() and (~kept).any()
    assert adv[kept].max() <= np.pi * (1 + 1e-6)
    assert adv[~kept].min() > np.pi * (1 - 1e-6)
    mask = lin.band_mask(n, n, PITCH, LAM, z)
    assert mask.shape == (2 * n, 2 * n) and mask[0, 0] and np.array_equal(mask[0], np.abs(lin.window_frequencies(2 * n, PITCH)) <= ul)


def test_adjoint_is_the_adjoint_and_the_gradient_matches_finite_differences():
    ny, nx, z = 10, 12, 30e-6
    rng = np.random.default_rng(7)
    x = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    y = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    Ax = lin.propagate_linear(x, PITCH, LAM, z, True)
    AHy = lin.propagate_linear(y, PITCH, LAM, z, True, conj_h=True)
    assert abs(np.vdot(y, Ax) - np.vdot(AHy, x)) <= 1e-12 * abs(np.vdot(y, Ax))
    h = rng.random((ny, nx)) * 1.0e-6
    T = rng.random((ny, nx))
    lambdas, n_refr = (450e-9, 633e-9), (1.5, 1.46)
    g = lin.adjoint(h, PITCH, lambdas, n_refr, z, target=T)
    for (iy, ix) in ((0, 0), (3, 7), (9, 11), (5, 0)):
        d = 1e-10
        hp, hm = h.copy(), h.copy()
        hp[iy, ix] += d
        hm[iy, ix] -= d
        fd = (lin.forward(hp, PITCH, lambdas, n_refr, z, target=T)["loss"] - lin.forward(hm, PITCH, lambdas, n_refr, z, target=T)["loss"]) / (2 * d)
        assert abs(fd - g[iy, ix]) <= 2e-6 * np.abs(g).max(), (iy, ix, fd, g[iy, ix])
    # caller-supplied dL/dI: linear in it
    dLdI = rng.standard_normal((2, ny, nx))
    g1 = lin.adjoint(h, PITCH, lambdas, n_refr, z, dLdI=dLdI)
    g2 = lin.adjoint(h, PITCH, lambdas, n_refr, z, dLdI=2 * dLdI)
    assert np.abs(g2 - 2 * g1).max() <= 1e-12 * np.abs(g1).max()


def test_loss_is_the_mean_over_the_aperture():
    ny, nx, z = 6, 8, 10e-6
    rng = np.random.default_rng(3)
    h, T = rng.random((ny, nx)) * 1e-6, rng.random((ny, nx))
    out = lin.forward(h, PITCH, [LAM], [1.5], z, target=T)
    assert abs(out["loss"] - np.mean((out["I"][0] - T) ** 2)) < 1e-15
    assert np.allclose(out["I"][0], np.abs(out["u"][0]) ** 2)
