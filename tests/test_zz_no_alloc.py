"""dop_prefilter_noalloc (include/dop.h): the stencil pre-filter F0 / A6 with its scratch plane in the library's static
device array instead of the caller's workspace -- for callers that cannot call cudaMalloc.

Collected last on purpose (the suite runs with pytest -x): it must pass alone in a fresh process and after the
other tests, so it makes no assumption about what the shared array holds when it starts.

The GPU test checks the new entry point against the existing path twice in a row, on two different seeded inputs:
  existing path   plan(sigma).fwd / .adj: F0 and A6 run inside the propagate calls, scratch in the workspace;
  new entry       h_eff = noalloc(h), plan(sigma = 0).fwd(h_eff) / .adj, dL/dh = noalloc(dL/dh_eff);
intensity, loss and gradient of the two must agree within the suite's bars (they run the same kernels with the same
taps, so in practice bit for bit), and h_eff itself is compared with the oracle's spectral definition.
"""
import ctypes as C
import dataclasses

import numpy as np
import pytest

from conftest import max_rel_peak, rel_l2

TOL_L2, TOL_PEAK, TOL_LOSS = 1e-5, 1e-4, 1e-5
DEV = "cuda:0"
SIGMA = 3.0


def test_limit_and_argument_errors_are_reported_before_anything_is_enqueued():
    """Host-only: sizes beyond DOP_NOALLOC_MAX_POINTS and plans without a stencil pre-filter are rejected with their
    own status (the device pointers are never dereferenced: the checks precede every CUDA call)."""
    from paper_2505_22313_b200 import dop
    fake = C.c_void_p(0x1000)
    lam, nr = (550e-9,), (1.5,)
    big, _ = dop.dop_plan_create(2048, 4096, 0.25e-6, lam, nr, 1e-3, dop.DOP_LOSS_L2, SIGMA)     # 8 Mi points
    assert 2048 * 4096 > dop.DOP_NOALLOC_MAX_POINTS
    st = dop._lib.dop_prefilter_noalloc(big, fake, fake, None)
    assert st == dop.DOP_ERR_NOALLOC_LIMIT
    assert "DOP_NOALLOC_MAX_POINTS" in dop.dop_status_string(st) and "4194304" in dop.dop_status_string(st)
    dop.dop_plan_destroy(big)
    for sigma in (0.0, 0.7, 5.5):                                                                  # no stencil form
        p, _ = dop.dop_plan_create(512, 512, 0.25e-6, lam, nr, 1e-3, dop.DOP_LOSS_L2, sigma)
        assert dop._lib.dop_prefilter_noalloc(p, fake, fake, None) == dop.DOP_ERR_INVALID_ARG
        dop.dop_plan_destroy(p)
    ok, _ = dop.dop_plan_create(2048, 2048, 0.25e-6, lam, nr, 1e-3, dop.DOP_LOSS_L2, SIGMA)       # exactly the limit
    assert 2048 * 2048 == dop.DOP_NOALLOC_MAX_POINTS
    assert dop._lib.dop_prefilter_noalloc(ok, None, fake, None) == dop.DOP_ERR_INVALID_ARG
    assert dop._lib.dop_prefilter_noalloc(None, fake, fake, None) == dop.DOP_ERR_INVALID_ARG
    dop.dop_plan_destroy(ok)


@pytest.mark.gpu
def test_noalloc_prefilter_matches_the_plan_path_on_two_calls_in_a_row():
    import torch
    from oracle import asm_oracle as orc
    from paper_2505_22313_b200 import dop, synth

    ny, nx = 1024, 1536  # several tiles of both stencil kernels
    base = dataclasses.replace(synth.CONFIGS["C3"].scaled(ny, nx), sigma_px=SIGMA)
    with_pre = dop.Plan(ny, nx, base.pitch, base.lambdas, base.n_refr, base.z, dop.DOP_LOSS_L2, SIGMA,
                        dop.DOP_WRITE_INTENSITY, DEV)
    assert "blur-x" in with_pre.describe()
    no_pre = dop.Plan(ny, nx, base.pitch, base.lambdas, base.n_refr, base.z, dop.DOP_LOSS_L2, 0.0,
                      dop.DOP_WRITE_INTENSITY, DEV)
    assert "blur" not in no_pre.describe()

    def bars(a, b, what):
        e2, ep = rel_l2(a, b), max_rel_peak(a, b)
        assert e2 <= TOL_L2 and ep <= TOL_PEAK, f"{what}: rel-L2 {e2:.3e}, max-abs/peak {ep:.3e}"

    first_heff = None
    for call, index in enumerate((base.index, base.index + 7)):   # two calls in a row, different inputs
        cfg = dataclasses.replace(base, index=index)
        h, T = synth.make_height(cfg, DEV), synth.make_target(cfg, DEV)

        # existing path: F0 and A6 inside the propagate calls
        I_a = torch.full((1, ny, nx), float("nan"), dtype=torch.float32, device=DEV)
        g_a = torch.full_like(h, float("nan"))
        L_a = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
        with_pre.fwd(h, T, I_a, L_a)
        with_pre.adj(h, None, g_a)

        # new entry: F0, the unfiltered plan, A6 (in place on the gradient)
        heff = torch.full_like(h, float("nan"))
        dop.dop_prefilter_noalloc(with_pre.handle, h, heff)
        I_b = torch.full((1, ny, nx), float("nan"), dtype=torch.float32, device=DEV)
        g_b = torch.full_like(h, float("nan"))
        L_b = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
        no_pre.fwd(heff, T, I_b, L_b)
        no_pre.adj(heff, None, g_b)
        dop.dop_prefilter_noalloc(with_pre.handle, g_b, g_b)
        torch.cuda.synchronize()

        bars(I_b.cpu().numpy(), I_a.cpu().numpy(), f"call {call}: intensity")
        bars(g_b.cpu().numpy(), g_a.cpu().numpy(), f"call {call}: dL/dh")
        assert abs(L_b.item() - L_a.item()) <= TOL_LOSS * abs(L_a.item())
        # ... and the filtered plane itself against the oracle's spectral definition
        bars(heff.cpu().numpy(), orc.prefilter(h.cpu().numpy(), SIGMA), f"call {call}: h_eff")
        if call == 0:
            first_heff = (h, heff.clone())
    # the array keeps the last call's contents: a repeat of the first input must not see them
    h0, want = first_heff
    again = torch.empty_like(h0)
    dop.dop_prefilter_noalloc(with_pre.handle, h0, again)
    torch.cuda.synchronize()
    assert torch.equal(again, want)
    with_pre.close()
    no_pre.close()
