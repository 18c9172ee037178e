"""Parity of the padded / band-limited propagation mode (dop_plan_desc.pad = 2, band_limit; SURVEY.md 8(f)-3,
PAPER.md:436) against oracle/linear_oracle.py, element by element on the same seeded inputs, through the C-ABI."""
import numpy as np
import pytest
import torch

from conftest import max_rel_peak, rel_l2
from oracle import linear_oracle as lin
from paper_2505_22313_b200 import dop, synth

pytestmark = pytest.mark.gpu
TOL_L2, TOL_PEAK, TOL_LOSS = 1e-5, 1e-4, 1e-5
DEV = "cuda:0"


def check(a, b, what):
    e2, ep = rel_l2(a, b), max_rel_peak(a, b)
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{what}: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"


@pytest.mark.parametrize("ny,nx,z,bl", [(6, 10, 20e-6, 0), (48, 64, 0.2e-3, 1), (96, 200, 1e-3, 1), (512, 384, 2e-3, 0),
                                        (512, 384, 2e-3, 1), (300, 1000, 5e-3, 1), (2048, 4096, 20e-3, 1),
                                        (256, 8192, 5e-3, 1), (96, 16384, 5e-3, 0)])   # two x digits: aperture masked by the TMA unit
def test_padded_l2_path_against_the_linear_oracle(ny, nx, z, bl):
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    lambdas, n_refr = (550e-9, 633e-9), (1.5, 1.47)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    plan = dop.Plan(ny, nx, cfg.pitch, lambdas, n_refr, z, dop.DOP_LOSS_L2, 0.0, dop.DOP_WRITE_INTENSITY, DEV, pad=2, band_limit=bl)
    text = plan.describe()
    assert "pad=2" in text
    if nx >= 8192:   # the window's x axis has two digits: the fused x passes run on the TMA kernels, not on the generic one
        assert "col tma" in [l for l in text.splitlines() if "loss,seed" in l][0], text
    inten = torch.full((2, ny, nx), float("nan"), dtype=torch.float32, device=DEV)
    grad = torch.full_like(h, float("nan"))
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    plan.fwd(h, T, inten, loss)
    plan.adj(h, None, grad)
    torch.cuda.synchronize()
    plan.close()
    hn, Tn = h.cpu().numpy(), T.cpu().numpy()
    ref = lin.forward(hn, cfg.pitch, lambdas, n_refr, z, target=Tn, band_limit=bool(bl))
    gref = lin.adjoint(hn, cfg.pitch, lambdas, n_refr, z, target=Tn, band_limit=bool(bl))
    check(inten.cpu().numpy(), ref["I"], "intensity")
    check(grad.cpu().numpy(), gref, "dL/dh")
    assert abs(loss.item() - ref["loss"]) <= TOL_LOSS * abs(ref["loss"])


@pytest.mark.parametrize("ny,nx,bl", [(40, 56, 1), (384, 640, 1), (384, 640, 0)])
def test_padded_field_and_caller_seeded_adjoint(ny, nx, bl):
    """DOP_LOSS_NONE with pad = 2: the cropped field u, I, and the adjoint of a caller-supplied dL/dI."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    z, lambdas, n_refr = 1e-3, (550e-9,), (1.5,)
    h = synth.make_height(cfg, DEV)
    dLdI = synth.uniform_plane(91, 5, ny, nx, DEV).view(1, ny, nx).contiguous() - 0.5
    plan = dop.Plan(ny, nx, cfg.pitch, lambdas, n_refr, z, dop.DOP_LOSS_NONE, 0.0, 0, DEV, pad=2, band_limit=bl)
    inten = torch.empty((1, ny, nx), dtype=torch.float32, device=DEV)
    grad = torch.empty_like(h)
    plan.fwd(h, None, inten, None)
    torch.cuda.synchronize()
    u = plan.field().cpu().numpy()
    plan.adj(h, dLdI, grad)
    torch.cuda.synchronize()
    plan.close()
    hn = h.cpu().numpy()
    ref = lin.forward(hn, cfg.pitch, lambdas, n_refr, z, band_limit=bool(bl))
    check(u, ref["u"], "field u")
    check(inten.cpu().numpy(), ref["I"], "intensity")
    check(grad.cpu().numpy(), lin.adjoint(hn, cfg.pitch, lambdas, n_refr, z, dLdI=dLdI.cpu().numpy(), band_limit=bool(bl)), "dL/dh")


def test_pad_arguments_are_validated():
    args = (64, 64, 0.25e-6, (550e-9,), (1.5,), 1e-3)
    for kw in (dict(pad=3), dict(band_limit=1), dict(pad=2, prefilter_sigma_px=2.0), dict(pad=2, upsample=2),
               dict(pad=2, loss=dop.DOP_LOSS_SIMSE)):
        with pytest.raises(dop.DopError) as e:
            dop.dop_plan_create(*args, **kw)
        assert e.value.status == dop.DOP_ERR_INVALID_ARG
    hnd, ws = dop.dop_plan_create(*args, pad=2, band_limit=1)
    assert ws >= 4 * 64 * 64 * 8   # the workspace holds the 2x window
    dop.dop_plan_destroy(hnd)
