"""Parity of the CUDA path (through the C-ABI, via the thin binding) against the fp64 oracle,
element by element on the same seeded inputs (the same bytes go to both sides).

Bars (BASELINE.json north_star): rel-L2 <= 1e-5 and max-abs/peak <= 1e-4
for the complex64 field u and the intensity I; this suite applies the same two bars to dL/dh and
|L - L_ref|/|L_ref| <= 1e-5 to the loss.
"""
import os

import numpy as np
import pytest
import torch

from conftest import max_rel_peak, rel_l2
from oracle import asm_oracle as orc
from paper_2505_22313_b200 import dop, synth

pytestmark = pytest.mark.gpu

TOL_L2, TOL_PEAK, TOL_LOSS = 1e-5, 1e-4, 1e-5
DEV = "cuda:0"


def check(a, b, what):
    e2, ep = rel_l2(a, b), max_rel_peak(a, b)
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{what}: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"
    return e2, ep


def digits(text):
    return tuple(int(v) for v in text.split(","))


def run_l2(cfg, h, T, lambdas=None, n_refr=None, write_i=True, tuning=None):
    lambdas = cfg.lambdas if lambdas is None else lambdas
    n_refr = cfg.n_refr if n_refr is None else n_refr
    flags = dop.DOP_WRITE_INTENSITY if write_i else 0
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, lambdas, n_refr, cfg.z, dop.DOP_LOSS_L2, cfg.sigma_px, flags, DEV,
                    tuning=tuning)
    inten = torch.full((len(lambdas), cfg.ny, cfg.nx), float("nan"), dtype=torch.float32, device=DEV) if write_i else None
    grad = torch.full_like(h, float("nan"))
    loss = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
    plan.fwd(h, T, inten, loss)
    plan.adj(h, None, grad)
    torch.cuda.synchronize()
    out = (None if inten is None else inten.cpu().numpy(), float(loss.item()), grad.cpu().numpy())
    plan.close()
    return out


def oracle_l2(cfg, h, T, lambdas=None, n_refr=None):
    lambdas = cfg.lambdas if lambdas is None else lambdas
    n_refr = cfg.n_refr if n_refr is None else n_refr
    hn, Tn = h.cpu().numpy(), T.cpu().numpy()
    f = orc.forward(hn, cfg.pitch, lambdas, n_refr, cfg.z, target=Tn, sigma_px=cfg.sigma_px, keep_field=False)
    g = orc.adjoint(hn, cfg.pitch, lambdas, n_refr, cfg.z, target=Tn, sigma_px=cfg.sigma_px)
    return f["I"], f["loss"], g


# ------------------------------------------------------------------------------------------------
# small and medium grids: several tiles, ragged tails, radix 3, one- two- and three-digit axes
# ------------------------------------------------------------------------------------------------
SHAPES = [(2, 2), (2, 3), (3, 2), (4, 6), (16, 16), (48, 36), (27, 64), (96, 128), (384, 512), (1024, 768),
          (1536, 2048), (2048, 1024), (243, 256), (4096, 512), (512, 16384), (18, 20736),
          # general sizes: radix 5 / 7 / 11 / 13 / 67 butterflies, one- and two-digit axes
          (5, 7), (25, 49), (150, 140), (67, 335), (143, 121), (1340, 640), (2880, 2000), (600, 7000)]


@pytest.mark.parametrize("ny,nx", SHAPES)
def test_field_intensity_and_caller_seeded_adjoint(ny, nx):
    """DOP_LOSS_NONE: field u (read from the workspace), I, then adj with a caller-supplied dL/dI."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)          # pitch 0.25 um: evanescent bins present
    z = 2e-3
    lambdas, n_refr = (550e-9, 633e-9), (1.5, 1.47)
    h = synth.make_height(cfg, DEV)
    dLdI = synth.uniform_plane(77, 5, 2 * ny, nx, DEV).view(2, ny, nx).contiguous() - 0.5
    plan = dop.Plan(ny, nx, cfg.pitch, lambdas, n_refr, z, dop.DOP_LOSS_NONE, 0.0, 0, DEV)
    inten = torch.empty((2, ny, nx), dtype=torch.float32, device=DEV)
    grad = torch.empty_like(h)
    plan.fwd(h, None, inten, None)
    torch.cuda.synchronize()
    u = plan.field().cpu().numpy()
    plan.adj(h, dLdI, grad)
    torch.cuda.synchronize()
    plan.close()
    hn = h.cpu().numpy()
    ref = orc.forward(hn, cfg.pitch, lambdas, n_refr, z)
    check(u, ref["u"], "field u")
    check(inten.cpu().numpy(), ref["I"], "intensity")
    gref = orc.adjoint(hn, cfg.pitch, lambdas, n_refr, z, dLdI=dLdI.cpu().numpy())
    check(grad.cpu().numpy(), gref, "dL/dh")


@pytest.mark.parametrize("ny,nx", [(2, 2), (6, 4), (96, 128), (384, 512), (1536, 1024), (512, 6144),
                                   (35, 55), (670, 1280), (900, 3600)])
def test_fused_l2_loss_path(ny, nx):
    # C2's blurred-noise recipe degenerates (zero range) on grids smaller than its blur: tiny grids use C1's
    cfg = synth.CONFIGS["C2" if ny * nx >= 4096 else "C1"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T)
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)
    # without the optional intensity output the loss and gradient are unchanged
    _, L2, g2 = run_l2(cfg, h, T, write_i=False)
    assert L2 == L and np.array_equal(g2, g)


@pytest.mark.parametrize("ny,nx,tun", [(256, 1024, {}),                      # row kernel (one x digit)
                                       (64, 8192, {"xdigits": (256, 32)}),   # h -> exp(i Phi) and dL/dh on the TMA kernels
                                       (64, 8192, {"xdigits": (256, 32), "no_tma": 1}),
                                       (64, 16384, {}),                      # thread-block-cluster row pass
                                       (35, 55, {})])                        # generic kernel
def test_exp_i_phi_over_several_turns_of_either_sign(ny, nx, tun):
    """F1/F2 and A5 on heights between -4 and +4 turns of phase (the configurations stay within 0..1.2 turns): the
    exact residue Phi/2pi - rint(Phi/2pi) and the hardware sine / cosine behind it (reading 9) in every kernel
    family, against the oracle's fp64 exp(i Phi)."""
    cfg = synth.CONFIGS["C2"].scaled(ny, nx)
    lam, n = cfg.lambdas[1], cfg.n_refr[1]
    turn = lam / (n - 1.0)                                       # height of one turn of phase
    h = ((synth.uniform_plane(91, 3, ny, nx, DEV).view(ny, nx) - 0.5) * (8.0 * turn)).contiguous()
    T = synth.make_target(cfg, DEV)
    tuning = dop.make_tuning(**tun) if tun else None
    I, L, g = run_l2(cfg, h, T, lambdas=(lam,), n_refr=(n,), tuning=tuning)
    Ir, Lr, gr = oracle_l2(cfg, h, T, lambdas=(lam,), n_refr=(n,))
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("ny,nx,sigma,no_stencil", [(48, 64, 3.0, 0), (384, 512, 3.0, 0), (384, 512, 3.0, 1), (1024, 1536, 3.0, 0),
                                                    (1024, 1536, 3.0, 1), (256, 640, 0.7, 0), (256, 640, 2.1, 0), (512, 512, 4.0, 0), (512, 512, 5.5, 0)])
def test_prefilter_path(ny, nx, sigma, no_stencil):
    """F0 / A6 against the oracle's spectral definition: as the separable spatial stencil (blur.cu; 2.05 <= sigma <= 4 px,
    ny % 32 == 0) and in the spectral form (dop_tuning.no_stencil, ragged shapes, larger sigma)."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["C3"].scaled(ny, nx), sigma_px=sigma)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    assert len(np.unique(h.cpu().numpy())) <= 256     # 256 gray levels
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, sigma, 0, DEV,
                    tuning=dop.make_tuning(no_stencil=no_stencil))
    stencil = "blur-x" in plan.describe()
    plan.close()
    assert stencil == (not no_stencil and 2.05 <= sigma <= 4.0 and ny % 32 == 0)
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(no_stencil=no_stencil))
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("xd,yd", [("16,8", "4,12"), ("2,4,16", "3,4,4"), ("128", "48")])
def test_every_digit_decomposition_gives_the_same_answer(xd, yd):
    """The multi-pass (four-step) decomposition used for 65536-point lines, forced on a small grid."""
    cfg = synth.CONFIGS["C5"].scaled(48, 128)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(xdigits=digits(xd), ydigits=digits(yd)))
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


KERNEL_FAMILIES = [
    # (ny, nx, DOP_YDIGITS, DOP_XDIGITS): every digit length of every specialised kernel family
    (256, 1024, "16,16", "16,64"),        # column 16 (tile / H / lane), row 64
    (1024, 4096, "32,32", "32,128"),      # column 32, row 128
    (4096, 64, "64,64", "64"),            # column 64 (tile, H), single-digit row 64
    (16, 16384, "16", "64,256"),          # column 64 (lane), staged row 256
    (16384, 64, "128,128", "64"),         # column 128 (tile, H)
    (16, 32768, "16", "128,256"),         # column 128 (lane)
    (65536, 32, "256,256", "32"),         # column 256 with 32-column bundles (tile), column 256 (H)
    (16, 131072, "16", "256,512"),        # column 256 (lane), row 512 (runs of 2)
    (8192, 64, "512,16", "64"),           # column 512 (tile)
    (8192, 64, "16,512", "64"),           # column 512 (H)
    (2, 524288, "2", "512,1024"),         # column 512 (lane), row 1024
    (256, 2048, "16,16", "2048"),         # row 2048
    (128, 4096, "128", "4096"),           # row 4096
    (64, 8192, "64", "8192"),             # row 8192 (config 2's)
    (768, 128, "48,16", "128"),           # 3 x 16
    (1536, 128, "96,16", "128"),          # 3 x 32
    (3072, 128, "192,16", "128"),         # 3 x 64
    (6144, 128, "384,16", "128"),         # 3 x 128 (config 5's)
    (16, 49152, "16", "16,48,64"),        # 3 x 16 with per-lane boundary twiddles
]


@pytest.mark.parametrize("family", ["tma", "ldg", "generic"])
@pytest.mark.parametrize("ny,nx,yd,xd", KERNEL_FAMILIES)
def test_every_kernel_family_against_the_oracle(ny, nx, yd, xd, family):
    """Forces digit decompositions so that each instantiated digit length of every kernel family runs the
    fused L2 path and is compared with the oracle: "tma" = the default routing (column passes through the
    persistent TMA pipeline, tma_col.cuh), "ldg" = the register-blocked LDG/STG kernels alone
    (dop_tuning.no_tma: column tile / H / per-lane variants, staged and unstaged row tiles, 3 x 2^k),
    "generic" = the same plans on the generic shared-memory kernel at full digit lengths."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    tun = dop.make_tuning(xdigits=digits(xd), ydigits=digits(yd), force_generic=int(family == "generic"),
                          no_tma=int(family == "ldg"), no_cluster=1)
    I, L, g = run_l2(cfg, h, T, tuning=tun)
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("tun", [
    dict(no_tma=1, col_nb=32), dict(no_tma=1, col_nb=64), dict(tma_nb=32), dict(tma_nb=16, tma_stages=3),
    dict(no_tma=1, prefetch_waves=-1), dict(no_tma=1, prefetch_waves=3), dict(force_generic=1, tile_pts=1024),
    dict(force_generic=1, tile_pts=16384), dict(slab_mb=1, slab_streams=3), dict(no_mirror=1), dict(no_mirror=1, tma_nb=32),
])
def test_tuning_knobs_only_change_the_rounding_order(tun):
    """include/dop.h: no dop_tuning field changes a result beyond rounding order.  Every knob on a grid with two
    x digits and two y digits (the L2 loss pass is then a column-type pass whose CTA count follows the bundle
    width: the loss partials must match what is launched), against the oracle."""
    cfg = synth.CONFIGS["C4"].scaled(4096, 16384)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(xdigits=(128, 128), ydigits=(64, 64), no_cluster=1, **tun))
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("ny,yd,nx,xd", [(6144, "384,16", 64, "64"), (12288, "48,256", 64, "64"), (8192, "16,512", 128, "128"),
                                         (32768, "2,128,128", 64, "64"), (4096, "64,64", 4096, "64,64"),
                                         (2048, "16,128", 8192, "32,256"), (512, "8,64", 16384, "2,64,128")])
def test_H_on_mirrored_tile_pairs_against_the_oracle(ny, yd, nx, xd):
    """The (x) H pass evaluates H once per group of up to four kx- / ky-mirrored tiles (tma_hpair_kernel): every
    last-digit length, a 3 * 2^k first digit, one-, two- and three-digit axes, against the oracle; and bitwise
    identical to the unpaired pass (same H values, same arithmetic)."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    tun = dict(ydigits=digits(yd), xdigits=digits(xd), no_cluster=1)
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, tuning=dop.make_tuning(**tun))
    text = plan.describe()
    plan.close()
    assert "tma" in [l for l in text.splitlines() if "*H*" in l][0] and "H on mirrored tiles" in text, text
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(**tun))
    I0, L0, g0 = run_l2(cfg, h, T, tuning=dop.make_tuning(no_mirror=1, **tun))
    assert np.array_equal(I, I0) and np.array_equal(g, g0) and L == L0   # same H values, same arithmetic
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("ny,yd,nx,xd", [
    (450, "225,2", 1800, "2,900"),        # 225 as a y digit (ragged last column tile), 900 as the row-type last x digit
    (10000, "", 72, ""),                  # 625 as a y digit (the planner's 625 . 16; ragged last column tile)
    (7, "", 5000, "2,2500"),              # 2500 as the last x digit (ragged last row tile)
    (64, "64", 900, "4,225"),             # 225 as the last x digit
    (64, "64", 1250, "2,625"),            # 625 as the last x digit (odd line length: 8-byte staging)
    (900, "2,225,2", 7200, "2,225,16"),   # 225 as a middle digit of both axes (x: lines = 16 < tile width, per-line twiddles)
    (3600, "225,16", 14400, "16,900"),    # the digit pairs the planner picks for the paper's 28 800 grid, on the TMA kernels
])
def test_smooth_digit_passes_against_the_oracle(ny, yd, nx, xd):
    """Plain passes of the 5-smooth digits 225, 625, 900, 2500 (the paper's 28 800 and 40 000 grids)
    on the register-step kernels (smooth.cu), column- and row-type, forward and inverse, against the oracle and
    against the generic kernel running the same schedule (dop_tuning.no_smooth)."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    tun = dict(ydigits=digits(yd) if yd else (), xdigits=digits(xd) if xd else ())
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, tuning=dop.make_tuning(**tun))
    text = plan.describe()
    plan.close()
    plain = [l for l in text.splitlines() if l.endswith(("[x-fwd]", "[x-inv]", "[y-fwd]", "[y-inv]"))]
    for L in (225, 625, 900, 2500):
        for l in plain:
            if f" L={L} " in l:
                assert " smooth " in l, text
    assert any(" smooth " in l for l in plain), text
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, tuning=dop.make_tuning(no_smooth=1, **tun))
    assert " smooth " not in plan.describe()
    plan.close()
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(**tun))
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)
    I0, L0, g0 = run_l2(cfg, h, T, tuning=dop.make_tuning(no_smooth=1, **tun))
    check(I, I0, "intensity against the generic kernel")
    check(g, g0, "dL/dh against the generic kernel")


@pytest.mark.parametrize("ny,nx", [(8, 16384), (6, 32768), (4, 65536), (96, 65536)])
def test_cluster_row_passes_against_the_oracle(ny, nx):
    """Rows of 16 M points (M = 1024, 2048, 4096) run their two x digit passes as ONE thread-block-cluster
    pass (cluster_row.cuh; DSMEM all-to-all between a radix-16 step and the M-point line transforms):
    fused L2 path, caller-seeded path (field u readable) and pre-filter, all against the oracle, and
    against the same plan with the cluster kernels switched off (dop_tuning.no_cluster)."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    force = dop.make_tuning(cluster_force=1)
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, 0.0, 0, DEV, tuning=force)
    text = plan.describe()
    plan.close()
    assert "x0+x1 L=16x%d" % (nx // 16) in text and "row cluster=%d" % {1024: 2, 2048: 4, 4096: 8}[nx // 16] in text
    I, L, g = run_l2(cfg, h, T, tuning=force)
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)
    I2, L2, g2 = run_l2(cfg, h, T, tuning=dop.make_tuning(no_cluster=1))
    I4, L4, g4 = run_l2(cfg, h, T, tuning=dop.make_tuning(cluster_force=1, cluster_dsmem=1))
    check(I4, Ir, "intensity (DSMEM exchange)")
    check(g4, gr, "dL/dh (DSMEM exchange)")
    if nx == 65536:  # clusters of 16 CTAs of 256 threads
        for dsmem in (0, 1):
            I5, L5, g5 = run_l2(cfg, h, T, tuning=dop.make_tuning(cluster_force=1, cluster_lines=1, cluster_dsmem=dsmem))
            check(I5, Ir, "intensity (clusters of 16)")
            check(g5, gr, "dL/dh (clusters of 16)")
    check(I2, Ir, "intensity (two digit passes)")
    check(I, I2, "cluster vs digit passes")
    check(g, g2, "cluster vs digit passes, dL/dh")
    # caller-seeded path: field u, I, then adj with dL/dI
    dLdI = synth.uniform_plane(78, 5, ny, nx, DEV).view(1, ny, nx).contiguous() - 0.5
    plan = dop.Plan(ny, nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_NONE, 0.0, 0, DEV, tuning=force)
    inten = torch.empty((1, ny, nx), dtype=torch.float32, device=DEV)
    grad = torch.empty_like(h)
    plan.fwd(h, None, inten, None)
    torch.cuda.synchronize()
    u = plan.field().cpu().numpy()
    plan.adj(h, dLdI, grad)
    torch.cuda.synchronize()
    plan.close()
    hn = h.cpu().numpy()
    ref = orc.forward(hn, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z)
    check(u, ref["u"], "field u")
    check(inten.cpu().numpy(), ref["I"], "intensity (LOSS_NONE)")
    check(grad.cpu().numpy(), orc.adjoint(hn, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dLdI=dLdI.cpu().numpy()), "dL/dh")
    # pre-filter (real-plane load / store variants)
    cfg3 = synth.CONFIGS["C3"].scaled(ny, nx)
    h3, T3 = synth.make_height(cfg3, DEV), synth.make_target(cfg3, DEV)
    I3, L3, g3 = run_l2(cfg3, h3, T3, tuning=force)
    I3r, L3r, g3r = oracle_l2(cfg3, h3, T3)
    check(I3, I3r, "intensity (pre-filter)")
    check(g3, g3r, "dL/dh (pre-filter)")
    assert abs(L3 - L3r) <= TOL_LOSS * abs(L3r)


def test_slab_schedule_gives_the_same_answer():
    """dop_tuning.slab_mb: multi-pass segments run slab by slab on auxiliary streams (fork / join on the
    caller's stream); 1 MiB slabs split this grid into 16 column slabs and 16 row slabs."""
    cfg = synth.CONFIGS["C4"].scaled(1024, 2048)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I0, L0, g0 = run_l2(cfg, h, T, tuning=dop.make_tuning(xdigits=(16, 128)))
    I1, L1, g1 = run_l2(cfg, h, T, tuning=dop.make_tuning(xdigits=(16, 128), slab_mb=1))
    # same kernels on the same tiles, only the launch grouping differs: bit-identical
    assert np.array_equal(I0, I1) and np.array_equal(g0, g1) and L0 == L1
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I1, Ir, "intensity")
    check(g1, gr, "dL/dh")
    assert abs(L1 - Lr) <= TOL_LOSS * abs(Lr)


@pytest.mark.parametrize("z,h_float", [(2e-3, 1), (0.4, 0), (-0.4, 0), (0.28, 0), (0.28, 1)])
def test_both_phase_paths_of_H(z, h_float):
    """H's phase is taken in 32-bit fixed point while |z|/lambda < 2^19 turns and through the fp32
    fraction otherwise (or with dop_tuning.h_float): both against the oracle, on both sides of the
    switch (0.28 m / 550 nm = 509 091 turns < 2^19 = 524 288 <= 0.4 m / 550 nm)."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["C4"].scaled(512, 256), z=z)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T, tuning=dop.make_tuning(h_float=h_float))
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "intensity")
    check(g, gr, "dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


def test_calls_capture_into_a_cuda_graph():
    """dop_propagate_fwd / _adj only enqueue kernels on the caller's stream (dop.h "Asynchrony"), so a
    warmed-up pair captures into a CUDA graph; replays give the bit-identical result."""
    cfg = synth.CONFIGS["C1"].scaled(256, 512)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, 0.0, 0, DEV)
    grad = torch.empty_like(h)
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    plan.fwd(h, T, None, loss)
    plan.adj(h, None, grad)
    torch.cuda.synchronize()
    g0, l0 = grad.clone(), loss.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        plan.fwd(h, T, None, loss)
        plan.adj(h, None, grad)
    for _ in range(2):
        grad.zero_()
        loss.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(grad, g0) and torch.equal(loss, l0)
    del graph
    plan.close()


def test_degenerate_inputs():
    """z = 0 (identity on a grid without evanescent bins), flat height (plane wave), negative z."""
    cfg = synth.CONFIGS["C1"].scaled(64, 96)
    h = synth.make_height(cfg, DEV)
    plan = dop.Plan(64, 96, cfg.pitch, cfg.lambdas, cfg.n_refr, 0.0, dop.DOP_LOSS_NONE, 0.0, 0, DEV)
    inten = torch.empty((1, 64, 96), dtype=torch.float32, device=DEV)
    plan.fwd(h, None, inten, None)
    torch.cuda.synchronize()
    u = plan.field().cpu().numpy()[0]
    plan.close()
    u0 = orc.phase_field(h.cpu().numpy(), cfg.lambdas[0], cfg.n_refr[0])
    check(u, u0, "z=0 identity")
    assert np.abs(inten.cpu().numpy() - 1).max() < 1e-5
    flat = torch.full((64, 96), 0.3e-6, dtype=torch.float32, device=DEV)
    for z in (1e-3, -1e-3):
        plan = dop.Plan(64, 96, cfg.pitch, cfg.lambdas, cfg.n_refr, z, dop.DOP_LOSS_NONE, 0.0, 0, DEV)
        plan.fwd(flat, None, inten, None)
        torch.cuda.synchronize()
        u = plan.field().cpu().numpy()[0]
        plan.close()
        lam, n = cfg.lambdas[0], cfg.n_refr[0]
        expect = np.exp(2j * np.pi * (n - 1) * float(flat[0, 0].item()) / lam) * np.exp(2j * np.pi * z / lam)
        assert np.abs(u - expect).max() < 1e-5          # plane wave picks up e^{ikz} (P-b)


def test_state_and_argument_errors_on_device():
    cfg = synth.CONFIGS["C1"].scaled(32, 32)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    plan = dop.Plan(32, 32, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, 0.0, 0, DEV)
    grad = torch.empty_like(h)
    with pytest.raises(dop.DopError) as e:
        plan.adj(h, None, grad)
    assert e.value.status == dop.DOP_ERR_STATE
    with pytest.raises(dop.DopError) as e:
        plan.fwd(h, None, None, None)                   # L2 needs a target
    assert e.value.status == dop.DOP_ERR_INVALID_ARG
    plan.fwd(h, T, None, None)                          # d_loss may be NULL
    plan.adj(h, None, grad)
    with pytest.raises(dop.DopError):
        plan.adj(h, None, grad)                         # one adj per fwd
    torch.cuda.synchronize()
    plan.close()


def test_repeatable_bitwise():
    cfg = synth.CONFIGS["C2"].scaled(768, 1024)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    a = run_l2(cfg, h, T)
    b = run_l2(cfg, h, T)
    assert np.array_equal(a[0], b[0]) and a[1] == b[1] and np.array_equal(a[2], b[2])


@pytest.mark.parametrize("ny,nx,yd,xd", [
    (64, 16384, "64", "64,256"),     # staged row tiles, warp-local exchanges only (256-point rows)
    (512, 1024, "32,16", "1024"),    # row tiles with one CTA-wide and one warp-local exchange
    (256, 8192, "16,16", "8192"),    # 8192-point rows (runs of 2 slots, CTA-wide exchanges)
    (65536, 32, "256,256", "32"),    # 32-column bundles
    (6144, 128, "384,16", "128"),    # 3 x 128
    (2048, 65536, "32,64", "16,4096"),  # cluster row passes (DSMEM exchanges between 8 CTAs)
    (4096, 16384, "64,64", "16,1024"),  # cluster of 2
])
def test_repeatable_bitwise_under_load(ny, nx, yd, xd):
    """A missing barrier (the row kernels synchronise most exchanges with __syncwarp only) would show
    as run-to-run differences: the full grid keeps every SM busy with several CTAs, 8 repeats."""
    cfg = synth.CONFIGS["C4"].scaled(ny, nx)
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, cfg.lambdas, cfg.n_refr, cfg.z, dop.DOP_LOSS_L2, 0.0,
                    dop.DOP_WRITE_INTENSITY, DEV,
                    tuning=dop.make_tuning(xdigits=digits(xd), ydigits=digits(yd), cluster_force=1))
    inten = torch.empty((1, ny, nx), dtype=torch.float32, device=DEV)
    grad = torch.empty_like(h)
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    ref = None
    for _ in range(8):
        plan.fwd(h, T, inten, loss)
        plan.adj(h, None, grad)
        torch.cuda.synchronize()
        cur = (inten.clone(), grad.clone(), loss.clone())
        if ref is None:
            ref = cur
        else:
            assert all(torch.equal(a, b) for a, b in zip(ref, cur))
    plan.close()


# ------------------------------------------------------------------------------------------------
# BASELINE.json configurations at full size, in the launch configuration bench.py times
# ------------------------------------------------------------------------------------------------
def test_C1_full_size_against_the_oracle():
    cfg = synth.CONFIGS["C1"]
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T)
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, "C1 intensity")
    check(g, gr, "C1 dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)


def tiled_case(name, py, px, lambdas_idx=None):
    """Pin P-k: tile a py x px problem R times; spectrum lives on multiples of R where
    the big grid's H equals the small grid's, so I_big = tile(I_small), L_big = L_small,
    Ry Rx grad_big = tile(grad_small).  The small problem comes from the full oracle."""
    cfg = synth.CONFIGS[name]
    ry, rx = cfg.ny // py, cfg.nx // px
    small = cfg.scaled(py, px)
    hs, Ts = synth.make_height(small, DEV), synth.make_target(small, DEV)
    lambdas = cfg.lambdas if lambdas_idx is None else tuple(cfg.lambdas[i] for i in lambdas_idx)
    n_refr = cfg.n_refr[:len(lambdas)]
    # the oracle works on the small grid with the small grid's pitch: same frequencies on bins R k
    Ir, Lr, gr = oracle_l2(small, hs, Ts, lambdas, n_refr)
    h, T = synth.tile_plane(hs, ry, rx), synth.tile_plane(Ts, ry, rx)
    write_i = cfg.write_intensity
    flags = dop.DOP_WRITE_INTENSITY if write_i else 0
    plan = dop.Plan(cfg.ny, cfg.nx, cfg.pitch, lambdas, n_refr, cfg.z, dop.DOP_LOSS_L2, cfg.sigma_px, flags, DEV)
    inten = torch.empty((len(lambdas), cfg.ny, cfg.nx), dtype=torch.float32, device=DEV) if write_i else None
    grad = torch.empty_like(h)
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    plan.fwd(h, T, inten, loss)
    plan.adj(h, None, grad)
    torch.cuda.synchronize()
    plan.close()
    assert abs(float(loss.item()) - Lr) <= TOL_LOSS * abs(Lr)
    # every tile of the big result must equal the small one; compare all tiles on the device, one tile-row at a time
    def cmp_tiles(big, small_np, what):
        sm = torch.from_numpy(np.ascontiguousarray(small_np)).to(DEV)
        num = 0.0
        peak = 0.0
        for iy in range(ry):
            blk = big[iy * py:(iy + 1) * py].view(py, rx, px).permute(1, 0, 2).double() - sm
            num += float((blk ** 2).sum().item())
            peak = max(peak, float(blk.abs().max().item()))
            del blk
        e2 = np.sqrt(num) / (float((sm ** 2).sum().sqrt().item()) * np.sqrt(ry * rx))
        ep = peak / float(sm.abs().max().item())
        assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{name} tiled {what}: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"

    cmp_tiles(grad, gr / (ry * rx), "dL/dh")
    if inten is not None:
        for l in range(len(lambdas)):
            cmp_tiles(inten[l], Ir[l], "I")


def test_C2_full_size_tiled():
    tiled_case("C2", 1024, 2048)


def test_C3_full_size_tiled_with_prefilter():
    tiled_case("C3", 2048, 1024)


def plane_wave_case(name, a, b, p, q, tau=0.25, nsamp=4096):
    """Pin P-i at full size: h = (lambda/(n-1)) frac(a x/Nx + b y/Ny) makes u0 the DFT basis vector
    (a,b), so u = H(a,b) u0, I = |H|^2, and with T = 1 - tau cos(theta) the gradient has the closed
    form of SURVEY.md 8(c) P-i, evaluated in fp64 at sampled points."""
    cfg = synth.CONFIGS[name]
    ny, nx, lam, n, z, pitch = cfg.ny, cfg.nx, cfg.lambdas[0], cfg.n_refr[0], cfg.z, cfg.pitch
    ys = torch.arange(ny, device=DEV, dtype=torch.int64)[:, None]
    xs = torch.arange(nx, device=DEV, dtype=torch.int64)[None, :]
    h = torch.empty((ny, nx), dtype=torch.float32, device=DEV)
    T = torch.empty((ny, nx), dtype=torch.float32, device=DEV)
    rows = max(1, (1 << 26) // nx)
    for y0 in range(0, ny, rows):
        yy = ys[y0:y0 + rows]
        # exact rational phase: (a x Ny + b y Nx) mod (Nx Ny) / (Nx Ny), in int64 then fp64
        num = (a * xs * ny + b * yy * nx) % (nx * ny)
        h[y0:y0 + rows] = ((lam / (n - 1)) * (num.double() / float(nx * ny))).float()
        th = (p * xs * ny + q * yy * nx) % (nx * ny)
        T[y0:y0 + rows] = (1.0 - tau * torch.cos(2 * np.pi * th.double() / float(nx * ny))).float()
    flags = dop.DOP_WRITE_INTENSITY if cfg.write_intensity else 0
    plan = dop.Plan(ny, nx, pitch, (lam,), (n,), z, dop.DOP_LOSS_L2, 0.0, flags, DEV)
    inten = torch.empty((1, ny, nx), dtype=torch.float32, device=DEV) if flags else None
    grad = torch.empty_like(h)
    loss = torch.zeros(1, dtype=torch.float64, device=DEV)
    plan.fwd(h, T, inten, loss)
    plan.adj(h, None, grad)
    torch.cuda.synchronize()
    plan.close()

    def H(ka, kb):
        arg = 1 / lam ** 2 - (ka / (nx * pitch)) ** 2 - (kb / (ny * pitch)) ** 2
        return np.exp(2j * np.pi * z * np.sqrt(arg)) if arg >= 0 else 0.0

    H0, Hp, Hm = H(a, b), H(a + p, b + q), H(a - p, b - q)
    assert abs(H0) == 1.0 and abs(Hp) == 1.0 and abs(Hm) == 1.0
    rng = np.random.default_rng(11)
    sy, sx = rng.integers(0, ny, nsamp), rng.integers(0, nx, nsamp)
    th = 2 * np.pi * (((p * sx * ny + q * sy * nx) % (nx * ny)) / float(nx * ny))
    N = float(nx * ny)
    gref = (2 * np.pi * (n - 1) / lam) * (2 * tau / N) * np.imag(
        H0 * (np.conj(Hp) * np.exp(1j * th) + np.conj(Hm) * np.exp(-1j * th)))
    gs = grad[torch.from_numpy(sy).to(DEV), torch.from_numpy(sx).to(DEV)].double().cpu().numpy()
    # conditioning of the pin itself: the two sidebands must not cancel in Im[.] (for some (p,q,z)
    # they do to a few percent, which only amplifies fp32 noise relative to a vanishing reference)
    A, B = H0 * np.conj(Hp), H0 * np.conj(Hm)
    assert np.hypot(A.imag + B.imag, A.real - B.real) >= 0.5, "ill-conditioned plane-wave pin: choose other p, q"
    # loss: I == 1 exactly, so L = mean (tau cos)^2 = tau^2/2
    assert abs(float(loss.item()) - tau * tau / 2) <= TOL_LOSS * tau * tau / 2
    e2 = np.linalg.norm(gs - gref) / np.linalg.norm(gref)
    ep = np.abs(gs - gref).max() / np.abs(gref).max()
    # (the closed form assumes the ideal ramp; storing h in fp32 perturbs the phase by ~4e-7 rad, well below the bar)
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{name} plane-wave dL/dh: {e2:.3e} {ep:.3e}"
    if inten is not None:
        Is = inten[0][torch.from_numpy(sy).to(DEV), torch.from_numpy(sx).to(DEV)].cpu().numpy()
        assert np.abs(Is - 1.0).max() <= 1e-4


def test_C2_full_size_plane_wave_closed_form():
    plane_wave_case("C2", 1203, -877, 345, 210)


HUGE = pytest.mark.skipif(os.environ.get("DOP_SKIP_HUGE") == "1" or not torch.cuda.is_available()
                          or torch.cuda.get_device_properties(0).total_memory < 150e9,
                          reason="needs ~130 GB of device memory")


@HUGE
def test_C4_full_size_tiled():
    tiled_case("C4", 2048, 4096)


@HUGE
def test_C5_full_size_tiled():
    tiled_case("C5", 3072, 2048)


@HUGE
def test_C5_full_size_plane_wave_closed_form():
    plane_wave_case("C5", 5001, -3 * 2111, 1234, 3 * 779)


@HUGE
def test_C4_full_size_plane_wave_closed_form():
    plane_wave_case("C4", 5001, -6333, 1234, 2337)


def grating_case(name, a, b, m1=1.8, m2=1.3, nsamp=100000, expect_cut=True):
    """Pin P-j at full size on the GPU: a two-sinusoid phase grating; the field u
    (DOP_LOSS_NONE, read from the workspace) against the Jacobi-Anger closed form of
    tests/closed_forms.py in fp64 at ~1e5 sampled points.  a, b are so large that the 51 x 51 orders
    land all over the spectrum, on both sides of the evanescent cut."""
    from closed_forms import grating_field
    cfg = synth.CONFIGS[name]
    ny, nx, lam, n, z, pitch = cfg.ny, cfg.nx, cfg.lambdas[0], cfg.n_refr[0], cfg.z, cfg.pitch
    c = m1 + m2
    assert c + m1 + m2 <= 2 * np.pi * (n - 1) * cfg.h_max / lam       # 0 <= h <= h_max
    xs = torch.arange(nx, device=DEV, dtype=torch.int64)
    sinx = m1 * torch.sin(2 * np.pi * ((a * xs) % nx).double() / nx)
    h = torch.empty((ny, nx), dtype=torch.float32, device=DEV)
    rows = max(1, (1 << 26) // nx)
    for y0 in range(0, ny, rows):
        ys = torch.arange(y0, min(ny, y0 + rows), device=DEV, dtype=torch.int64)
        siny = m2 * torch.sin(2 * np.pi * ((b * ys) % ny).double() / ny)
        h[y0:y0 + rows] = ((c + siny[:, None] + sinx[None, :]) * (lam / (2 * np.pi * (n - 1)))).float()
    plan = dop.Plan(ny, nx, pitch, (lam,), (n,), z, dop.DOP_LOSS_NONE, 0.0, 0, DEV)
    inten = torch.empty((1, ny, nx), dtype=torch.float32, device=DEV)
    plan.fwd(h, None, inten, None)
    torch.cuda.synchronize()
    rng = np.random.default_rng(17)
    sy, sx = rng.integers(0, ny, nsamp), rng.integers(0, nx, nsamp)
    ty, tx = torch.from_numpy(sy).to(DEV), torch.from_numpy(sx).to(DEV)
    us = plan.field()[0][ty, tx].cpu().numpy().astype(np.complex128)
    Is = inten[0][ty, tx].cpu().numpy().astype(np.float64)
    plan.close()
    ref, Hkl = grating_field(ny, nx, pitch, lam, z, a, b, m1, m2, c, sy, sx)
    if expect_cut:
        assert 0.05 < np.mean(Hkl == 0) < 0.95, "orders must fall on both sides of the evanescent cut"
    e2 = np.linalg.norm(us - ref) / np.linalg.norm(ref)
    ep = np.abs(us - ref).max() / np.abs(ref).max()
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{name} grating field: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"
    Ir = np.abs(ref) ** 2
    e2 = np.linalg.norm(Is - Ir) / np.linalg.norm(Ir)
    ep = np.abs(Is - Ir).max() / Ir.max()
    assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{name} grating intensity: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"


def test_C2_full_size_phase_grating_closed_form():
    grating_case("C2", 1511, 977, expect_cut=False)   # (pitch 0.5 um: this grid holds no evanescent bin)


@HUGE
def test_C4_full_size_phase_grating_closed_form():
    grating_case("C4", 14011, 9007)


@HUGE
def test_C5_full_size_phase_grating_closed_form():
    grating_case("C5", 14011, 3 * 4001)


@pytest.mark.slow
@pytest.mark.parametrize("name", ["C2", "C3"])
def test_full_size_on_the_bench_inputs_against_the_oracle(name):
    """Pin P-l ("C1-C3 always"): the bench's own seeded inputs at full size, in the launch
    configuration bench.py times, element by element against the full-size fp64 oracle: every wavelength
    for C2, pre-filter on for C3 (about 20 s / 70 s of oracle time on 16 host cores)."""
    cfg = synth.CONFIGS[name]
    h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)
    I, L, g = run_l2(cfg, h, T)
    Ir, Lr, gr = oracle_l2(cfg, h, T)
    check(I, Ir, f"{name} intensity")
    check(g, gr, f"{name} dL/dh")
    assert abs(L - Lr) <= TOL_LOSS * abs(Lr)
