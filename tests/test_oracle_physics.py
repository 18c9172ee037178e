"""Pins for the oracle's ASM forward path (O0-O6) against what mathematics fixes.

The paper prints no worked numerical example of Eq. (1)-(4), so every pin is a
closed form, an invariant or a special case (SURVEY.md section 8(c) pins P-b .. P-f, P-i .. P-k).
Chosen so that a plausible mistake fails one of them: sign of H or of the DFT (P-b, P-f, P-i),
frequency sampling / evanescent cut (P-c, P-e, P-i, P-j), missing 1/N (P-b, P-e), H's z
dependence (P-d), wrong phase constant in Eq. (1) (P-b, P-j), loss normalisation (P-k).
"""
import numpy as np
import pytest
from scipy.special import jv

from oracle import asm_oracle as orc


def H_closed(fx, fy, lam, z):
    """north_star's transfer function evaluated directly at a frequency pair."""
    a = 1.0 / lam ** 2 - fx ** 2 - fy ** 2
    return np.where(a >= 0, np.exp(2j * np.pi * z * np.sqrt(np.abs(a))), 0.0)


def sbin(k, n):
    return k if k < (n + 1) // 2 else k - n


# ---------------------------------------------------------------------------------- P-b
@pytest.mark.parametrize("c", [0.0, 0.3e-6, 1.1e-6])
def test_plane_wave_stays_uniform_with_phase_eikz(c):
    ny, nx, pitch, lam, n, z = 24, 32, 1e-6, 532e-9, 1.46, 1e-3
    h = np.full((ny, nx), c)
    out = orc.forward(h, pitch, [lam], [n], z)
    expect = np.exp(2j * np.pi * (n - 1) * c / lam) * np.exp(2j * np.pi * z / lam)
    assert np.abs(out["u"][0] - expect).max() < 1e-9
    assert np.abs(out["I"][0] - 1.0).max() < 1e-12


# ---------------------------------------------------------------------------------- P-c
def test_z0_is_identity_without_evanescent_bins():
    rng = np.random.default_rng(1)
    ny, nx, pitch, lam = 32, 48, 1e-6, 532e-9          # pitch >= lam/sqrt(2): no bin is cut
    u0 = np.exp(2j * np.pi * rng.random((ny, nx)))
    assert np.abs(orc.propagate(u0, pitch, lam, 0.0) - u0).max() < 1e-13


def test_z0_is_band_projector_with_evanescent_bins():
    rng = np.random.default_rng(2)
    ny, nx, pitch, lam = 32, 48, 0.25e-6, 550e-9       # pitch < lam/2: corners are evanescent
    u0 = np.exp(2j * np.pi * rng.random((ny, nx)))
    p1 = orc.propagate(u0, pitch, lam, 0.0)
    p2 = orc.propagate(p1, pitch, lam, 0.0)
    assert np.abs(p1 - u0).max() > 0.1                  # it is not the identity ...
    assert np.abs(p2 - p1).max() < 1e-13                # ... it is idempotent
    H = orc.transfer_function(ny, nx, pitch, lam, 0.0)
    ncut = sum(1 for ky in range(ny) for kx in range(nx)
               if (sbin(kx, nx) / (nx * pitch)) ** 2 + (sbin(ky, ny) / (ny * pitch)) ** 2 > 1 / lam ** 2)
    assert ncut > 0 and int((H == 0).sum()) == ncut
    assert np.all((H == 0) | (np.abs(H - 1) < 1e-15))


# ---------------------------------------------------------------------------------- P-d
def test_composition_in_z():
    rng = np.random.default_rng(3)
    ny, nx, pitch, lam = 64, 96, 0.25e-6, 550e-9
    u0 = np.exp(2j * np.pi * rng.random((ny, nx)))
    z1, z2 = 0.3e-3, 0.7e-3
    a = orc.propagate(orc.propagate(u0, pitch, lam, z1), pitch, lam, z2)
    b = orc.propagate(u0, pitch, lam, z1 + z2)
    assert np.abs(a - b).max() < 1e-10


# ---------------------------------------------------------------------------------- P-e
def test_parseval_over_propagating_band():
    rng = np.random.default_rng(4)
    ny, nx, lam, z = 48, 64, 550e-9, 2e-3
    u0 = np.exp(2j * np.pi * rng.random((ny, nx)))
    # no bins cut: energy conserved exactly
    u = orc.propagate(u0, 1e-6, lam, z)
    assert abs((np.abs(u) ** 2).sum() - ny * nx) < 1e-9 * ny * nx
    # bins cut: energy = (1/N) sum over propagating bins |U|^2
    pitch = 0.25e-6
    u = orc.propagate(u0, pitch, lam, z)
    U = np.fft.fft2(u0)
    fy = np.fft.fftfreq(ny, pitch)[:, None]
    fx = np.fft.fftfreq(nx, pitch)[None, :]
    band = (1 / lam ** 2 - fx ** 2 - fy ** 2) >= 0
    assert abs((np.abs(u) ** 2).sum() - (np.abs(U[band]) ** 2).sum() / (ny * nx)) < 1e-9 * ny * nx


def test_white_field_mean_intensity_is_band_fraction():
    """SURVEY.md P-e side fact: uniform random phase at pitch 0.25 um, 550 nm -> mean(I) ~ pi (pitch/lam)^2."""
    rng = np.random.default_rng(5)
    n, pitch, lam = 512, 0.25e-6, 550e-9
    h = rng.random((n, n)) * lam / 0.5
    out = orc.forward(h, pitch, [lam], [1.5], 1e-3, keep_field=False)
    assert abs(out["I"].mean() - np.pi * (pitch / lam) ** 2) < 5e-3


# ---------------------------------------------------------------------------------- P-f
def test_gaussian_beam_matches_paraxial_closed_form():
    n, pitch, lam, w0, z = 1024, 0.5e-6, 0.55e-6, 20e-6, 0.5e-3
    c = (np.arange(n) - n // 2) * pitch
    X, Y = np.meshgrid(c, c)
    r2 = X ** 2 + Y ** 2
    u = orc.propagate(np.exp(-r2 / w0 ** 2), pitch, lam, z)
    k = 2 * np.pi / lam
    zR = np.pi * w0 ** 2 / lam
    w = w0 * np.sqrt(1 + (z / zR) ** 2)
    R = z * (1 + (zR / z) ** 2)
    ref = (w0 / w) * np.exp(-r2 / w ** 2) * np.exp(1j * (k * z + k * r2 / (2 * R) - np.arctan(z / zR)))
    assert np.linalg.norm(u - ref) / np.linalg.norm(ref) < 1e-4


# ---------------------------------------------------------------------------------- P-i
def test_tilted_plane_wave_is_an_eigenfunction():
    ny, nx, pitch, lam, n, z = 96, 128, 0.25e-6, 550e-9, 1.5, 2e-3
    for (a, b) in [(20, 9), (-17, 30), (60, 40)]:       # the last one is evanescent
        y, x = np.mgrid[0:ny, 0:nx]
        frac = np.mod(a * x / nx + b * y / ny, 1.0)
        h = lam / (n - 1) * frac                         # Phi = 2 pi frac  ->  u0 = basis vector (a,b)
        out = orc.forward(h, pitch, [lam], [n], z)
        Hab = H_closed(a / (nx * pitch), b / (ny * pitch), lam, z)
        u0 = np.exp(2j * np.pi * (a * x / nx + b * y / ny))
        assert np.abs(out["u"][0] - Hab * u0).max() < 1e-9
        assert np.abs(out["I"][0] - abs(Hab) ** 2).max() < 1e-9
    assert abs(H_closed(60 / (nx * pitch), 40 / (ny * pitch), lam, z)) == 0.0


# ---------------------------------------------------------------------------------- P-j
def test_sinusoidal_phase_grating_jacobi_anger():
    ny, nx, pitch, lam, n, z = 96, 128, 0.25e-6, 550e-9, 1.5, 0.2e-3
    a, b, m1, m2, K = 3, 2, 2.0, 1.5, 20
    c = m1 + m2 + 0.1
    y, x = np.mgrid[0:ny, 0:nx]
    phi = c + m1 * np.sin(2 * np.pi * a * x / nx) + m2 * np.sin(2 * np.pi * b * y / ny)
    h = phi * lam / (2 * np.pi * (n - 1))
    assert h.min() >= 0
    out = orc.forward(h, pitch, [lam], [n], z)
    ref = np.zeros((ny, nx), complex)
    for k in range(-K, K + 1):
        for l in range(-K, K + 1):
            Hkl = H_closed(k * a / (nx * pitch), l * b / (ny * pitch), lam, z)
            ref += jv(k, m1) * jv(l, m2) * Hkl * np.exp(2j * np.pi * (k * a * x / nx + l * b * y / ny))
    ref *= np.exp(1j * c)
    assert np.abs(out["u"][0] - ref).max() < 1e-11
    # some orders must have crossed the evanescent cut for this to test the mask
    assert 1 / lam ** 2 < (K * a / (nx * pitch)) ** 2


def test_phase_grating_closed_form_with_aliased_orders():
    """The evaluator the GPU suite uses at C4 / C5 size (tests/closed_forms.py): grating frequencies so high
    that most orders alias (k a > nx/2) and a good part of them is evanescent; against the oracle at every
    point of a small grid."""
    from closed_forms import grating_field, grating_phase
    ny, nx, pitch, lam, n, z = 96, 128, 0.25e-6, 550e-9, 1.5, 0.3e-3
    a, b, m1, m2 = 37, 29, 1.8, 1.3
    c = m1 + m2
    y, x = np.mgrid[0:ny, 0:nx]
    h = grating_phase(ny, nx, a, b, m1, m2, c, y, x) * lam / (2 * np.pi * (n - 1))
    assert h.min() >= 0 and h.max() <= 1.1e-6
    out = orc.forward(h, pitch, [lam], [n], z)
    ref, Hkl = grating_field(ny, nx, pitch, lam, z, a, b, m1, m2, c, y.ravel(), x.ravel())
    assert np.abs(out["u"][0].ravel() - ref).max() < 1e-11
    cut = np.mean(Hkl == 0)
    assert 0.1 < cut < 0.9          # the evanescent mask is exercised on both sides


# ---------------------------------------------------------------------------------- P-k
def test_periodic_tiling_invariance_forward():
    rng = np.random.default_rng(6)
    py, px, R = 24, 32, 3
    pitch, lam, n, z = 0.25e-6, 550e-9, 1.5, 1e-3
    h = rng.random((py, px)) * 1.1e-6
    T = rng.random((py, px)) * 2
    small = orc.forward(h, pitch, [lam], [n], z, target=T)
    big = orc.forward(np.tile(h, (R, R)), pitch, [lam], [n], z, target=np.tile(T, (R, R)))
    assert np.abs(big["I"][0] - np.tile(small["I"][0], (R, R))).max() < 1e-11
    assert abs(big["loss"] - small["loss"]) < 1e-12 * max(1.0, small["loss"])


# ---------------------------------------------------------------------------------- multi-lambda / loss
def test_loss_is_sum_over_lambda_of_pixel_mean():
    rng = np.random.default_rng(7)
    ny, nx = 16, 20
    h = rng.random((ny, nx)) * 1.2e-6
    T = rng.random((ny, nx))
    lams, ns = [450e-9, 550e-9, 650e-9], [1.5, 1.5, 1.5]
    out = orc.forward(h, 0.5e-6, lams, ns, 1e-3, target=T)
    by_hand = sum(((out["I"][l] - T) ** 2).mean() for l in range(3))
    assert abs(out["loss"] - by_hand) < 1e-13 * by_hand
    single = orc.forward(h, 0.5e-6, lams[1:2], ns[1:2], 1e-3, target=T)
    assert np.abs(single["I"][0] - out["I"][1]).max() == 0.0


# ---------------------------------------------------------------------------------- O0 pre-filter
def test_prefilter_equals_circular_convolution_with_sampled_gaussian():
    rng = np.random.default_rng(8)
    ny, nx, sigma = 40, 48, 3.0
    h = rng.random((ny, nx))
    dy = np.minimum(np.arange(ny), ny - np.arange(ny))[:, None].astype(float)
    dx = np.minimum(np.arange(nx), nx - np.arange(nx))[None, :].astype(float)
    # wrapped, sampled Gaussian (sum over images), normalised to unit DC
    g = np.zeros((ny, nx))
    for my in (-1, 0, 1):
        for mx in (-1, 0, 1):
            yy = (np.arange(ny)[:, None] + my * ny).astype(float)
            xx = (np.arange(nx)[None, :] + mx * nx).astype(float)
            g += np.exp(-(yy ** 2 + xx ** 2) / (2 * sigma ** 2))
    g /= g.sum()
    ref = np.zeros_like(h)
    for sy in range(ny):                                  # direct O(N^2) circular convolution
        for sx in range(nx):
            ref += g[sy, sx] * np.roll(h, (sy, sx), axis=(0, 1))
    out = orc.prefilter(h, sigma)
    assert np.abs(out - ref).max() < 1e-12
    assert abs(out.mean() - h.mean()) < 1e-14            # unit DC gain
    assert dy.shape and dx.shape
