"""GPU parity of the design-loop pieces against oracle/design_oracle.py, through
the C-ABI: the paper's penalty Eq. (6) (DOP_LOSS_SIMSE), the super-resolved design variable (nearest
up-sampling fused into the first pass's read, deterministic sum-pool of dL/dh, 8 / 16-bit gray-level
layouts) and the Adam + cosine-schedule epilogue.  Same bars as tests/test_parity_gpu.py."""
import numpy as np
import pytest
import torch

from conftest import max_rel_peak, rel_l2
from oracle import design_oracle as des
from paper_2505_22313_b200 import dop, synth

pytestmark = pytest.mark.gpu
TOL_L2, TOL_PEAK, TOL_LOSS = 1e-5, 1e-4, 1e-5
DEV = "cuda:0"
BETA = 5e-3


def check(a, b, what):
    e2, ep = rel_l2(a, b), max_rel_peak(a, b)
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{what}: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"


def digits(text):
    return tuple(int(v) for v in text.split(","))


def make_layout(cfg, r, dtype):
    """coarse layout of the config's height recipe on the [ny/r][nx/r] feature grid, in the requested dtype"""
    coarse = synth.make_height(cfg.scaled(cfg.ny // r, cfg.nx // r), DEV)
    if dtype == dop.DOP_LAYOUT_F32:
        return coarse, 1.0
    levels = 255 if dtype == dop.DOP_LAYOUT_U8 else 1023            # 8-bit, or the paper's 10-bit layouts
    step = cfg.h_max / levels
    q = torch.round(coarse / step).clamp_(0, levels)
    return q.to(torch.uint8 if dtype == dop.DOP_LAYOUT_U8 else torch.uint16), step


def run(cfg, layout, T, loss_mode, r=1, dtype=dop.DOP_LAYOUT_F32, step=0.0, tuning=None, lambdas=None, n_refr=None):
    lambdas = cfg.lambdas if lambdas is None else lambdas
    n_refr = cfg.n_refr if n_refr is None else n_refr
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, lambdas, n_refr, cfg.z, loss_mode, cfg.sigma_px, dop.DOP_WRITE_INTENSITY,
                    DEV, tuning=tuning, energy_beta=BETA, upsample=r, layout_dtype=dtype, layout_step=step)
    inten = torch.full((len(lambdas), cfg.ny, cfg.nx), float("nan"), dtype=torch.float32, device=DEV)
    grad = torch.full((cfg.ny // r, cfg.nx // r), float("nan"), dtype=torch.float32, device=DEV)
    loss = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
    plan.fwd(layout, T, inten, loss)
    plan.adj(layout, None, grad)
    torch.cuda.synchronize()
    text = plan.describe()
    plan.close()
    return inten.cpu().numpy(), float(loss.item()), grad.cpu().numpy(), text


@pytest.mark.parametrize("ny,nx,xd,yd,sigma", [
    (96, 128, "", "", 0.0), (384, 512, "", "", 0.0), (64, 2048, "16,128", "", 0.0), (256, 8192, "", "", 0.0),
    (8, 16384, "", "", 0.0),            # cluster row kernels
    (48, 96, "", "", 0.0),              # generic kernel (3 * 2^k rows)
    (256, 512, "", "", 2.0),            # with the pre-filter
])
def test_simse_energy_loss_against_the_oracle(ny, nx, xd, yd, sigma):
    """DOP_LOSS_SIMSE: I, L and dL/dh for Eq. (6) with three wavelengths."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["C2"].scaled(ny, nx), sigma_px=sigma, pitch=0.3e-6, z=2e-3)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    tun = dop.make_tuning(xdigits=digits(xd) if xd else (), ydigits=digits(yd) if yd else ())
    I, L, g, text = run(cfg, h, T, dop.DOP_LOSS_SIMSE, tuning=tun)
    assert "si-mse+energy" in text and "plane sums" in text
    hn, Tn = h.cpu().numpy(), T.cpu().numpy()
    ref = des.forward(hn, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, Tn, BETA, sigma_px=sigma)
    gref = des.adjoint(hn, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, Tn, BETA, sigma_px=sigma)
    check(I, ref["I"], "intensity")
    assert abs(L - ref["loss"]) <= TOL_LOSS * abs(ref["loss"]), (L, ref["loss"])
    check(g, gref, "dL/dh")


@pytest.mark.parametrize("loss_mode", [dop.DOP_LOSS_L2, dop.DOP_LOSS_SIMSE])
@pytest.mark.parametrize("ny,nx,r,dtype,xd,sigma", [
    (128, 256, 2, dop.DOP_LAYOUT_F32, "", 0.0),
    (256, 512, 4, dop.DOP_LAYOUT_F32, "", 0.0),
    (256, 1024, 8, dop.DOP_LAYOUT_U8, "", 0.0),          # row-type last x pass
    (64, 4096, 8, dop.DOP_LAYOUT_U16, "16,256", 0.0),    # column-type last x pass (two x digits)
    (64, 4096, 4, dop.DOP_LAYOUT_F32, "64,64", 0.0),
    (16, 16384, 8, dop.DOP_LAYOUT_U16, "", 0.0),         # cluster row kernels
    (256, 512, 1, dop.DOP_LAYOUT_U8, "", 0.0),           # gray levels without up-sampling
    (256, 512, 4, dop.DOP_LAYOUT_U16, "", 1.5),          # up-sampling, then the fabrication pre-filter (Eq. 5's shape)
    (64, 4096, 2, dop.DOP_LAYOUT_F32, "16,256", 2.0),
])
def test_super_resolved_layout_against_the_oracle(ny, nx, r, dtype, xd, sigma, loss_mode):
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["C4"].scaled(ny, nx), sigma_px=sigma, z=1e-3)
    layout, step = make_layout(cfg, r, dtype)
    T = synth.make_target(cfg, DEV)
    tun = dop.make_tuning(xdigits=digits(xd) if xd else ())
    I, L, g, text = run(cfg, layout, T, loss_mode, r, dtype, step if dtype != dop.DOP_LAYOUT_F32 else 0.0, tun)
    assert f"upsample={r}" in text
    ln, Tn = layout.cpu().numpy(), T.cpu().numpy()
    if loss_mode == dop.DOP_LOSS_SIMSE:
        ref = des.forward(ln, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, Tn, BETA, r, step, sigma)
        gref = des.adjoint(ln, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, Tn, BETA, r, step, sigma)
        Lref, Iref = ref["loss"], ref["I"]
    else:
        from oracle import asm_oracle as asm
        hf = des.upsample_nearest(des.layout_to_height(ln, step), r)
        f = asm.forward(hf, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, target=Tn, sigma_px=sigma, keep_field=False)
        Lref, Iref = f["loss"], f["I"]
        gref = des.adjoint_l2(ln, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, Tn, r, step, sigma)
    assert g.shape == (ny // r, nx // r)
    check(I, Iref, "intensity")
    assert abs(L - Lref) <= TOL_LOSS * abs(Lref)
    check(g, gref, "dL/dl (sum-pooled)")


def test_pooled_gradient_is_bitwise_repeatable():
    cfg = synth.CONFIGS["C4"].scaled(512, 2048)
    layout, step = make_layout(cfg, 4, dop.DOP_LAYOUT_F32)
    T = synth.make_target(cfg, DEV)
    a = run(cfg, layout, T, dop.DOP_LOSS_SIMSE, 4)
    b = run(cfg, layout, T, dop.DOP_LOSS_SIMSE, 4)
    assert np.array_equal(a[2], b[2]) and a[1] == b[1] and np.array_equal(a[0], b[0])


@pytest.mark.parametrize("ny,nx,r,sigma,nlam", [(128, 256, 1, 0.0, 2), (256, 512, 4, 0.0, 1), (64, 4096, 1, 0.0, 1),
                                                (128, 256, 1, 1.5, 1), (8, 16384, 2, 0.0, 1)])
def test_adam_cosine_epilogue_against_the_oracle(ny, nx, r, sigma, nlam):
    """Three design iterations (fwd + adj_adam) with Eq. (6), lr on the cosine schedule: layout, m, v and the
    loss of every iteration against the oracle's loop."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["C4"].scaled(ny, nx), sigma_px=sigma, z=1e-3)
    lambdas, n_refr = ((550e-9, 640e-9), (1.5, 1.49)) if nlam == 2 else (cfg.lambdas, cfg.n_refr)
    layout, _ = make_layout(cfg, r, dop.DOP_LAYOUT_F32)
    T = synth.make_target(cfg, DEV)
    lr0, b1, b2, total = 1e-2 * cfg.h_max, 0.9, 0.999, 5
    plan = dop.Plan(ny, nx, cfg.pitch, lambdas, n_refr, cfg.z, dop.DOP_LOSS_SIMSE, sigma, 0, DEV, energy_beta=BETA, upsample=r)
    grad = torch.zeros_like(layout)
    m, v = torch.zeros_like(layout), torch.zeros_like(layout)
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    lo = layout.cpu().numpy().astype(np.float64)
    mo, vo = np.zeros_like(lo), np.zeros_like(lo)
    Tn = T.cpu().numpy()
    eps = None
    for it in range(3):
        plan.fwd(layout, T, None, loss)
        torch.cuda.synchronize()
        go = des.adjoint(lo, cfg.pitch, lambdas, n_refr, cfg.z, Tn, BETA, r, 1.0, sigma)
        if eps is None:
            eps = 1e-3 * float(np.abs(go).max())     # in the unit of the gradient
        Lo = des.forward(lo, cfg.pitch, lambdas, n_refr, cfg.z, Tn, BETA, r, 1.0, sigma)["loss"]
        assert abs(float(loss.item()) - Lo) <= 2e-5 * abs(Lo), (it, float(loss.item()), Lo)
        plan.adj_adam(layout, None, grad, m, v, lr0, b1, b2, eps, it, total)
        torch.cuda.synchronize()
        lo, mo, vo = des.adam_step(lo, go, mo, vo, lr0, b1, b2, eps, it, total)
        check(grad.cpu().numpy(), go, f"it {it}: dL/dl")
        check(m.cpu().numpy(), mo, f"it {it}: m")
        check(v.cpu().numpy(), vo, f"it {it}: v")
        # the update itself (layout change since the start), not just the layout, must agree
        check(layout.cpu().numpy().astype(np.float64), lo, f"it {it}: layout")
    plan.close()


def test_design_options_are_validated():
    ok = dict(ny=64, nx=64, pitch=1e-6, lambdas=[550e-9], n_refr=[1.5], z=1e-3)
    for kw, status in ((dict(upsample=3), dop.DOP_ERR_INVALID_ARG), (dict(upsample=8, ny=60), dop.DOP_ERR_UNSUPPORTED_SIZE),
                       (dict(layout_dtype=7), dop.DOP_ERR_INVALID_ARG),
                       (dict(layout_dtype=dop.DOP_LAYOUT_U8, layout_step=0.0), dop.DOP_ERR_INVALID_ARG),
                       (dict(loss=dop.DOP_LOSS_SIMSE, energy_beta=-1.0), dop.DOP_ERR_INVALID_ARG),
                       (dict(upsample=8, ny=48, nx=48), dop.DOP_ERR_UNSUPPORTED_SIZE)):   # pooling needs the fast kernels
        with pytest.raises(dop.DopError) as e:
            dop.dop_plan_create(**{**ok, **kw})
        assert e.value.status == status, kw
