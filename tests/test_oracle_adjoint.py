"""Pins for the oracle's adjoint path (O7-O10; "solved by back-propagation",
PAPER.md:200 "backward pass is realized by another ... 2-D FFT").

P-g central finite differences of L w.r.t. single pixels (with evanescent bins, with the
pre-filter, with three wavelengths, and in caller-supplied dL/dI mode); P-h <Ax,y> = <x,A^H y>;
P-i closed-form gradient for a tilted plane wave with a cosine target; P-k tiling of the gradient.
A dropped factor 2, a missing conj on H, a wrong sign on Im(conj(u0) g) or a missing 1/N fails.
"""
import numpy as np
import pytest

from oracle import asm_oracle as orc


def fd_grad(h, pix, eps, loss_fn):
    g = []
    for (y, x) in pix:
        hp, hm = h.copy(), h.copy()
        hp[y, x] += eps
        hm[y, x] -= eps
        g.append((loss_fn(hp) - loss_fn(hm)) / (2 * eps))
    return np.array(g)


@pytest.mark.parametrize("sigma,lams", [(0.0, [550e-9]), (0.0, [450e-9, 550e-9, 650e-9]),
                                        (1.5, [550e-9]), (1.5, [500e-9, 600e-9])])
def test_adjoint_matches_central_differences(sigma, lams):
    rng = np.random.default_rng(11)
    ny, nx, pitch, z = 24, 32, 0.25e-6, 30e-6           # evanescent bins present at 0.25 um
    ns = [1.5] * len(lams)
    h = rng.random((ny, nx)) * 1.1e-6
    T = rng.random((ny, nx)) * 2
    grad = orc.adjoint(h, pitch, lams, ns, z, target=T, sigma_px=sigma)
    pix = [(0, 0), (3, 7), (23, 31), (12, 16), (5, 30)]
    fd = fd_grad(h, pix, 1e-12, lambda hh: orc.forward(hh, pitch, lams, ns, z, target=T,
                                                       sigma_px=sigma, keep_field=False)["loss"])
    an = np.array([grad[p] for p in pix])
    assert np.abs(an - fd).max() / np.abs(an).max() < 1e-6


def test_adjoint_with_caller_dLdI_matches_central_differences():
    rng = np.random.default_rng(12)
    ny, nx, pitch, z, lams, ns = 18, 20, 0.5e-6, 50e-6, [450e-9, 650e-9], [1.5, 1.45]
    h = rng.random((ny, nx)) * 1.2e-6
    w = rng.standard_normal((2, ny, nx))                  # L = sum w * I  =>  dL/dI = w
    grad = orc.adjoint(h, pitch, lams, ns, z, dLdI=w)
    pix = [(0, 0), (9, 10), (17, 19), (4, 15)]
    fd = fd_grad(h, pix, 1e-12, lambda hh: float((w * orc.forward(hh, pitch, lams, ns, z,
                                                                  keep_field=False)["I"]).sum()))
    an = np.array([grad[p] for p in pix])
    assert np.abs(an - fd).max() / np.abs(an).max() < 1e-6


def test_dot_product_test_of_propagator_and_its_adjoint():
    rng = np.random.default_rng(13)
    ny, nx, pitch, lam, z = 40, 36, 0.25e-6, 550e-9, 0.4e-3
    x = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    y = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    Ax = orc.propagate(x, pitch, lam, z)
    AHy = orc.propagate(y, pitch, lam, z, conj_h=True)
    assert abs(np.vdot(y, Ax) - np.vdot(AHy, x)) < 1e-12 * abs(np.vdot(y, Ax))


def test_tilted_plane_wave_gradient_closed_form():
    """P-i: u0 = DFT basis vector (a,b), T = 1 - tau cos(theta), theta = 2 pi (p x/Nx + q y/Ny):
    dL/dh = (2 pi (n-1)/lam) (2 tau/N) Im[ H0 (conj(H+) e^{i theta} + conj(H-) e^{-i theta}) ]."""
    ny, nx, pitch, lam, n, z = 96, 128, 0.25e-6, 550e-9, 1.5, 2e-3
    a, b, p, q, tau = 20, 9, 5, -4, 0.3
    y, x = np.mgrid[0:ny, 0:nx]
    h = lam / (n - 1) * np.mod(a * x / nx + b * y / ny, 1.0)
    theta = 2 * np.pi * (p * x / nx + q * y / ny)
    T = 1 - tau * np.cos(theta)
    grad = orc.adjoint(h, pitch, [lam], [n], z, target=T)

    def H(kx, ky):
        r = 1 / lam ** 2 - (kx / (nx * pitch)) ** 2 - (ky / (ny * pitch)) ** 2
        return np.exp(2j * np.pi * z * np.sqrt(r)) if r >= 0 else 0.0

    H0, Hp, Hm = H(a, b), H(a + p, b + q), H(a - p, b - q)
    N = ny * nx
    ref = (2 * np.pi * (n - 1) / lam) * (2 * tau / N) * np.imag(
        H0 * (np.conj(Hp) * np.exp(1j * theta) + np.conj(Hm) * np.exp(-1j * theta)))
    assert np.abs(grad - ref).max() / np.abs(ref).max() < 1e-9


def test_periodic_tiling_invariance_gradient():
    rng = np.random.default_rng(14)
    py, px, R = 24, 32, 2
    pitch, lam, n, z = 0.25e-6, 550e-9, 1.5, 1e-3
    h = rng.random((py, px)) * 1.1e-6
    T = rng.random((py, px)) * 2
    gs = orc.adjoint(h, pitch, [lam], [n], z, target=T)
    gb = orc.adjoint(np.tile(h, (R, R)), pitch, [lam], [n], z, target=np.tile(T, (R, R)))
    assert np.abs(R * R * gb - np.tile(gs, (R, R))).max() < 1e-11 * np.abs(gs).max()


def test_gradient_is_zero_at_perfect_target():
    rng = np.random.default_rng(15)
    h = rng.random((16, 16)) * 1e-6
    I = orc.forward(h, 1e-6, [532e-9], [1.46], 1e-3)["I"][0]
    g = orc.adjoint(h, 1e-6, [532e-9], [1.46], 1e-3, target=I)
    assert np.abs(g).max() == 0.0
