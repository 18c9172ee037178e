"""Pins for oracle/design_oracle.py: the paper's penalty Eq. (6)
(reading of the missing supplement in DESIGN.md), the super-resolved design variable
 and Adam with a cosine schedule.  None of the pins re-types
the oracle's own formula: invariants, finite differences, np.kron, and torch.optim as a library reference."""
import numpy as np
import pytest
import torch

from oracle import asm_oracle as asm
from oracle import design_oracle as des


# ------------------------------------------------------------------------------ Eq. (6)
def test_simse_is_scale_invariant_and_s_is_the_minimiser():
    rng = np.random.default_rng(1)
    I, T = rng.random((12, 20)) * 3, rng.random((12, 20))
    L0, s0, _ = des.simse_energy_loss(I, T, 0.0)
    for alpha in (0.01, 0.5, 7.0):
        L, s, _ = des.simse_energy_loss(alpha * I, T, 0.0)
        assert abs(L - L0) < 1e-14 and abs(s * alpha - s0) < 1e-13      # L(alpha I) = L(I): scale invariant
    # any other scale gives a larger mean squared error
    for ds in (-0.1, -1e-3, 1e-3, 0.1):
        assert np.mean(((s0 + ds) * I - T) ** 2) > L0
    # a target that IS a scaled copy of I is matched exactly
    assert des.simse_energy_loss(I, 2.5 * I, 0.0)[0] < 1e-28
    # plain MSE when the best scale is 1: T = I + noise orthogonal to I
    n = rng.standard_normal(I.shape)
    n -= I * np.sum(n * I) / np.sum(I * I)
    L1, s1, _ = des.simse_energy_loss(I, I + n, 0.0)
    assert abs(s1 - 1.0) < 1e-13 and abs(L1 - np.mean(n ** 2)) < 1e-13


def test_energy_term_counts_the_light_that_does_not_arrive():
    rng = np.random.default_rng(2)
    T = rng.random((16, 16))
    beta = 5e-3
    # lossless grid (pitch >= lambda/sqrt 2: no evanescent bin): all of the unit incident energy arrives
    h = rng.random((16, 16)) * 1e-6
    out = asm.forward(h, 1e-6, [532e-9], [1.46], 1e-3)
    assert abs(out["I"][0].mean() - 1.0) < 1e-12
    L, s, _ = des.simse_energy_loss(out["I"][0], T, beta)
    L_no, _, _ = des.simse_energy_loss(out["I"][0], T, 0.0)
    assert abs(L - L_no) < 1e-14
    # half of the energy missing costs beta / 2, whatever its distribution (the first term is scale invariant)
    L_half, _, _ = des.simse_energy_loss(0.5 * out["I"][0], T, beta)
    assert abs((L_half - L_no) - beta * 0.5) < 1e-14
    # a grid with evanescent bins loses energy: the term is positive
    out2 = asm.forward(h, 0.25e-6, [550e-9], [1.5], 1e-4)
    assert des.simse_energy_loss(out2["I"][0], T, 1.0)[0] - des.simse_energy_loss(out2["I"][0], T, 0.0)[0] > 0.05


def test_dLdI_against_central_differences():
    rng = np.random.default_rng(3)
    I, T = rng.random((6, 7)) + 0.2, rng.random((6, 7))
    beta = 5e-3
    _, _, g = des.simse_energy_loss(I, T, beta)
    for (y, x) in [(0, 0), (2, 5), (5, 6), (3, 3)]:
        e = 1e-6
        Ip, Im = I.copy(), I.copy()
        Ip[y, x] += e
        Im[y, x] -= e
        fd = (des.simse_energy_loss(Ip, T, beta)[0] - des.simse_energy_loss(Im, T, beta)[0]) / (2 * e)
        assert abs(fd - g[y, x]) < 1e-9 * max(1.0, abs(g[y, x])) + 1e-11


# ------------------------------------------------------------------------------ super-resolved design variable
@pytest.mark.parametrize("r", [1, 2, 4, 8])
def test_upsample_is_kron_and_sumpool_is_its_adjoint(r):
    rng = np.random.default_rng(4)
    c = rng.random((5, 7))
    up = des.upsample_nearest(c, r)
    assert np.array_equal(up, np.kron(c, np.ones((r, r))))
    g = rng.random(up.shape)
    assert abs(np.sum(up * g) - np.sum(c * des.sumpool(g, r))) < 1e-12          # <U c, g> = <c, U^T g>
    assert np.array_equal(des.sumpool(up, r), c * r * r) or np.allclose(des.sumpool(up, r), c * r * r, rtol=1e-15)
    assert np.array_equal(des.layout_to_height(np.array([[0, 255]], dtype=np.uint8), 2e-9), np.array([[0.0, 510e-9]]))


@pytest.mark.parametrize("r,sigma", [(2, 0.0), (4, 0.0), (2, 1.5)])
def test_whole_chain_gradient_against_central_differences(r, sigma):
    """d(sum_lambda L_p)/d(coarse height) through up-sampling, (pre-filter,) ASM and Eq. (6)."""
    rng = np.random.default_rng(5)
    Y, X = 6, 8
    pitch, lams, ns, z, beta = 0.25e-6, [450e-9, 650e-9], [1.5, 1.48], 40e-6, 5e-3
    c = rng.random((Y, X)) * 1.0e-6
    T = rng.random((Y * r, X * r)) * 2
    g = des.adjoint(c, pitch, lams, ns, z, T, beta, upsample=r, sigma_px=sigma)
    assert g.shape == (Y, X)
    for (y, x) in [(0, 0), (3, 4), (5, 7)]:
        e = 2e-12
        cp, cm = c.copy(), c.copy()
        cp[y, x] += e
        cm[y, x] -= e
        fd = (des.forward(cp, pitch, lams, ns, z, T, beta, r, 1.0, sigma)["loss"]
              - des.forward(cm, pitch, lams, ns, z, T, beta, r, 1.0, sigma)["loss"]) / (2 * e)
        assert abs(fd - g[y, x]) <= 2e-6 * np.abs(g).max(), (fd, g[y, x])
    # integer layouts: the same heights through (levels, step)
    lev = rng.integers(0, 256, (Y, X)).astype(np.uint8)
    a = des.forward(lev, pitch, lams, ns, z, T, beta, r, 4e-9, sigma)["loss"]
    b = des.forward(lev.astype(np.float64) * 4e-9, pitch, lams, ns, z, T, beta, r, 1.0, sigma)["loss"]
    assert a == b
    # and the L2 penalty of the benchmark configurations pools the same way
    g2 = des.adjoint_l2(c, pitch, lams, ns, z, T, upsample=r, sigma_px=sigma)
    full = asm.adjoint(des.upsample_nearest(c, r), pitch, lams, ns, z, target=T, sigma_px=sigma)
    assert np.allclose(g2, full.reshape(Y, r, X, r).sum(axis=(1, 3)), rtol=1e-13, atol=0)


# ------------------------------------------------------------------------------ Adam + cosine schedule
def test_adam_first_step_closed_form_and_schedule_end_points():
    g = np.array([3.0, -0.02, 1e-5])
    th, m, v = des.adam_step(np.zeros(3), g, np.zeros(3), np.zeros(3), 1e-2, 0.9, 0.999, 1e-8, 0, 3000)
    # first step: m_hat = g, v_hat = g^2  =>  theta moves by lr * g / (|g| + eps) ~ lr * sign(g)
    assert np.allclose(th, -1e-2 * g / (np.abs(g) + 1e-8), rtol=1e-12)
    assert np.allclose(m, 0.1 * g) and np.allclose(v, 0.001 * g * g)
    assert des.cosine_lr(1e-2, 0, 3000) == 1e-2
    assert abs(des.cosine_lr(1e-2, 1500, 3000) - 0.5e-2) < 1e-18
    assert abs(des.cosine_lr(1e-2, 3000, 3000)) < 1e-18


def test_adam_against_torch_optim_with_cosine_annealing():
    """Library cross-check: torch.optim.Adam + CosineAnnealingLR (eta_min 0) on a fixed gradient sequence."""
    rng = np.random.default_rng(6)
    total, steps = 40, 25
    th0 = rng.standard_normal(17)
    grads = rng.standard_normal((steps, 17)) * np.array([1e-3] * 8 + [10.0] * 9)
    p = torch.nn.Parameter(torch.tensor(th0, dtype=torch.float64))
    opt = torch.optim.Adam([p], lr=1e-2, betas=(0.9, 0.999), eps=1e-8)
    sched = torch.optim.lr_scheduler.CosineAnnealingLR(opt, T_max=total, eta_min=0.0)
    th, m, v = th0.copy(), np.zeros(17), np.zeros(17)
    for it in range(steps):
        p.grad = torch.tensor(grads[it], dtype=torch.float64)
        opt.step()
        sched.step()
        th, m, v = des.adam_step(th, grads[it], m, v, 1e-2, 0.9, 0.999, 1e-8, it, total)
        assert np.allclose(th, p.detach().numpy(), rtol=1e-11, atol=1e-14), it
