"""The C-ABI boundary (include/dop.h) without a GPU: libdop.so loads, exports every symbol the
header declares, dop_plan_create validates and plans on the host alone, and the propagate calls
fail loudly (never fall back to a CPU path) when no sm_100 device is present."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2505_22313_b200 import build as dop_build
from paper_2505_22313_b200 import dop

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dop.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dop_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared_symbols()
    assert {"dop_plan_create", "dop_propagate_fwd", "dop_propagate_adj", "dop_plan_destroy"} <= set(names)
    lib = C.CDLL(dop_build.build())
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(dop.EXPORTS)


def test_status_strings():
    for s in range(0, 7):
        assert dop.dop_status_string(s).startswith("DOP_")
    assert "UNKNOWN" in dop.dop_status_string(99)


@pytest.mark.parametrize("ny,nx", [(1024, 1024), (8192, 8192), (16384, 16384), (65536, 65536), (98304, 65536),
                                   (2, 2), (3, 2), (2, 3), (6, 4), (384, 512), (1536, 2048), (19683, 4)])
def test_plan_create_supported_sizes(ny, nx):
    plan, ws = dop.dop_plan_create(ny, nx, 0.25e-6, [550e-9], [1.5], 1e-3)
    try:
        assert ws >= ny * nx * 8
        text = dop.dop_plan_describe(plan)
        assert f"ny={ny} nx={nx}" in text
        # every digit product reproduces the axis length
        for axis, n in (("x", nx), ("y", ny)):
            line = [l for l in text.splitlines() if l.startswith(f"{axis}-digits:")][0]
            prod = 1
            for m in re.findall(r" (\d+)\(st=", line):
                prod *= int(m)
            assert prod == n
        assert dop.dop_plan_launch_count(plan) >= 5
    finally:
        dop.dop_plan_destroy(plan)


def test_workspace_sizes_fit_the_memory_plan():
    """SURVEY.md 8(a) memory plan: C5 = 48 GiB field + 3 x 24 GiB planes < 180 GB; C4 with I output."""
    plan, ws = dop.dop_plan_create(98304, 65536, 0.25e-6, [550e-9], [1.5], 0.1)
    dop.dop_plan_destroy(plan)
    n = 98304 * 65536
    assert ws < n * 8 + (64 << 20)
    assert ws + 3 * n * 4 < 180e9
    plan, ws = dop.dop_plan_create(65536, 65536, 0.25e-6, [550e-9], [1.5], 0.05, flags=dop.DOP_WRITE_INTENSITY)
    dop.dop_plan_destroy(plan)
    assert ws + 4 * (1 << 32) * 4 < 180e9
    # pre-filter adds one fp32 plane, n_lambda multiplies the fields
    plan, ws3 = dop.dop_plan_create(512, 512, 0.5e-6, [450e-9, 550e-9, 650e-9], [1.5] * 3, 1e-3)
    dop.dop_plan_destroy(plan)
    plan, ws1 = dop.dop_plan_create(512, 512, 0.5e-6, [550e-9], [1.5], 1e-3)
    dop.dop_plan_destroy(plan)
    plan, wsp = dop.dop_plan_create(512, 512, 0.5e-6, [550e-9], [1.5], 1e-3, prefilter_sigma_px=3.0)
    dop.dop_plan_destroy(plan)
    assert ws3 - ws1 >= 2 * 512 * 512 * 8 and wsp - ws1 >= 512 * 512 * 4


@pytest.mark.parametrize("kw,status", [
    (dict(ny=1024, nx=1042), dop.DOP_ERR_UNSUPPORTED_SIZE),     # 1042 = 2 x 521: a prime factor above 127
    (dict(ny=1, nx=64), dop.DOP_ERR_UNSUPPORTED_SIZE),
    (dict(ny=64, nx=0), dop.DOP_ERR_UNSUPPORTED_SIZE),
    (dict(ny=131, nx=64), dop.DOP_ERR_UNSUPPORTED_SIZE),        # 131 is prime
    (dict(pitch=0.0), dop.DOP_ERR_INVALID_ARG),
    (dict(pitch=float("nan")), dop.DOP_ERR_INVALID_ARG),
    (dict(lambdas=[]), dop.DOP_ERR_INVALID_ARG),
    (dict(lambdas=[-1.0]), dop.DOP_ERR_INVALID_ARG),
    (dict(z=float("inf")), dop.DOP_ERR_INVALID_ARG),
    (dict(loss=7), dop.DOP_ERR_INVALID_ARG),
    (dict(prefilter_sigma_px=-1.0), dop.DOP_ERR_INVALID_ARG),
    (dict(flags=0x80), dop.DOP_ERR_INVALID_ARG),
])
def test_plan_create_rejects_bad_descriptions(kw, status):
    args = dict(ny=64, nx=64, pitch=1e-6, lambdas=[550e-9], n_refr=[1.5], z=1e-3)
    args.update(kw)
    if len(args["n_refr"]) != len(args["lambdas"]):
        args["n_refr"] = [1.5] * len(args["lambdas"])
    with pytest.raises(dop.DopError) as e:
        dop.dop_plan_create(**args)
    assert e.value.status == status


def test_null_arguments():
    lib = dop._lib
    assert lib.dop_plan_create(None, None, None) == dop.DOP_ERR_INVALID_ARG
    assert lib.dop_plan_destroy(None) == dop.DOP_ERR_INVALID_ARG
    assert lib.dop_propagate_fwd(None, None, None, None, None, None, None) == dop.DOP_ERR_INVALID_ARG
    assert lib.dop_propagate_adj(None, None, None, None, None, None) == dop.DOP_ERR_INVALID_ARG
    plan, _ = dop.dop_plan_create(64, 64, 1e-6, [550e-9], [1.5], 1e-3)
    try:
        fake = C.c_void_p(4096)
        # adj before fwd
        assert lib.dop_propagate_adj(plan, fake, None, fake, fake, None) == dop.DOP_ERR_STATE
        # L2 needs a target; missing workspace
        assert lib.dop_propagate_fwd(plan, fake, None, None, None, fake, None) == dop.DOP_ERR_INVALID_ARG
        assert lib.dop_propagate_fwd(plan, fake, fake, None, None, None, None) == dop.DOP_ERR_WORKSPACE
    finally:
        dop.dop_plan_destroy(plan)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_without_a_device():
    """Without a CUDA device the propagate call must fail (DOP_ERR_CUDA / DOP_ERR_ARCH), never compute."""
    plan, _ = dop.dop_plan_create(64, 64, 1e-6, [550e-9], [1.5], 1e-3)
    try:
        fake = C.c_void_p(4096)
        st = dop._lib.dop_propagate_fwd(plan, fake, fake, None, None, fake, None)
        assert st in (dop.DOP_ERR_CUDA, dop.DOP_ERR_ARCH)
    finally:
        dop.dop_plan_destroy(plan)


def _digits(text):
    return tuple(int(v) for v in text.split(","))


def test_launch_count_follows_the_slab_schedule():
    """dop_plan_launch_count is exact for whole-array launches and for the slab schedule."""
    args = (1024, 2048, 0.25e-6, (550e-9,), (1.5,), 1e-3, dop.DOP_LOSS_L2, 0.0, 0)
    h, _ = dop.dop_plan_create(*args, tuning=dop.make_tuning(xdigits=(16, 128)))
    base = dop.dop_plan_launch_count(h)
    dop.dop_plan_destroy(h)
    assert base == 13 + 1  # 13 passes (x 16.128, y 32.32) + the loss reduction
    h, _ = dop.dop_plan_create(*args, tuning=dop.make_tuning(xdigits=(16, 128), slab_mb=1))
    n = dop.dop_plan_launch_count(h)
    dop.dop_plan_destroy(h)
    # x segments: rows of 16 KiB -> 64 rows per slab -> 16 slabs; y segments: columns of 8 KiB -> 128 -> 16 slabs
    assert n == 13 * 16 + 1


@pytest.mark.parametrize("ny,nx,yd,xd,tun,expect", [
    (65536, 32, "256,256", "32", {}, ["y0 L=256 tile=32x256 col tma stages=2", "y1 L=256 tile=16x256 col tma stages=3"]),
    (65536, 32, "256,256", "32", {"no_tma": 1}, ["y0 L=256 tile=32x256 col pow2", "y1 L=256 tile=16x256 col pow2"]),
    (16, 131072, "16", "256,512", {}, ["x0 L=256 tile=32x256 col tma stages=2 ctas=256 smem=196608 B/pt=12",
                                      "x0 L=256 tile=16x256 col tma stages=3 ctas=512 smem=147456 B/pt=20",
                                      "x0 L=256 tile=32x256 col tma stages=2 ctas=256 smem=196608 B/pt=16 [x-inv,grad]",
                                      "x1 L=512 tile=8x512 row pow2"]),
    (16, 131072, "16", "256,512", {"no_tma": 1}, ["x0 L=256 tile=16x256 col pow2 ctas=512 smem=32768 B/pt=12"]),
    (6144, 128, "384,16", "128", {}, ["y0 L=384 tile=32x384 col tma stages=2", "x0 L=128 tile=32x128 row pow2"]),
    (6144, 128, "384,16", "128", {"no_tma": 1}, ["y0 L=384 tile=32x384 col pow2"]),
    (64, 8192, "64", "8192", {}, ["x0 L=8192 tile=1x8192 row pow2", "y0 L=64 tile=16x64 col tma stages=3"]),
    (64, 8192, "64", "8192", {"tma_nb": 32, "tma_stages": 3}, ["y0 L=64 tile=32x64 col tma stages=3"]),
])
def test_plan_routes_digits_to_the_specialised_kernels(ny, nx, yd, xd, tun, expect):
    """dop_plan_describe names, per pass, the tile shape and the kernel family the plan chose: column passes
    go to the persistent TMA pipeline (tma_col.cuh) unless dop_tuning.no_tma asks for the LDG/STG kernels."""
    h, _ = dop.dop_plan_create(ny, nx, 0.25e-6, (550e-9,), (1.5,), 1e-3, dop.DOP_LOSS_L2, 0.0, 0,
                               tuning=dop.make_tuning(xdigits=_digits(xd), ydigits=_digits(yd), no_cluster=1, **tun))
    text = dop.dop_plan_describe(h)
    dop.dop_plan_destroy(h)
    for e in expect:
        assert e in text, (e, text)


def test_cluster_row_passes_in_the_plan():
    """Rows of 16 M points can run their x digit pair (16, M) as ONE thread-block-cluster pass (one read
    + one write of the field per x transform pair).  Default where measured faster (nx = 16384, clusters
    of 2: config 3); dop_tuning.cluster_force selects them at 65536 too: 144 instead of 208 B/point."""
    h, _ = dop.dop_plan_create(16384, 16384, 0.25e-6, (550e-9,), (1.5,), 0.01)
    text = dop.dop_plan_describe(h)
    dop.dop_plan_destroy(h)
    assert "x0+x1 L=16x1024 tile=8x1024 row cluster=2" in text and "algorithmic_bytes_per_point=144" in text, text
    h, _ = dop.dop_plan_create(98304, 65536, 0.25e-6, (550e-9,), (1.5,), 0.1)
    text = dop.dop_plan_describe(h)
    dop.dop_plan_destroy(h)
    assert "cluster" not in text and "algorithmic_bytes_per_point=208" in text, text
    h, _ = dop.dop_plan_create(98304, 65536, 0.25e-6, (550e-9,), (1.5,), 0.1, tuning=dop.make_tuning(cluster_force=1))
    text = dop.dop_plan_describe(h)
    assert dop.dop_plan_launch_count(h) == 9 + 1
    dop.dop_plan_destroy(h)
    assert "x0+x1 L=16x4096 tile=2x4096 row cluster=8" in text and "algorithmic_bytes_per_point=144" in text, text


def test_the_library_reads_no_environment_variable(monkeypatch):
    """dop.h: no ambient state.  The round-1 environment knobs must be inert; tuning is explicit."""
    args = (1024, 2048, 0.25e-6, (550e-9,), (1.5,), 1e-3, dop.DOP_LOSS_L2, 0.0, 0)
    h, _ = dop.dop_plan_create(*args)
    ref = dop.dop_plan_describe(h)
    dop.dop_plan_destroy(h)
    for k, v in (("DOP_XDIGITS", "16,128"), ("DOP_YDIGITS", "4,256"), ("DOP_FORCE_GENERIC", "1"), ("DOP_COL_NB", "64"),
                 ("DOP_SLAB_MB", "1"), ("DOP_TILE_PTS", "256"), ("DOP_H_FLOAT", "1"), ("DOP_PREFETCH_WAVES", "7")):
        monkeypatch.setenv(k, v)
    h, _ = dop.dop_plan_create(*args)
    assert dop.dop_plan_describe(h) == ref
    dop.dop_plan_destroy(h)
    src = os.path.join(ROOT, "paper_2505_22313_b200", "csrc")
    for f in os.listdir(src):
        assert "getenv" not in open(os.path.join(src, f)).read(), f


@pytest.mark.parametrize("tun,status", [
    (dict(xdigits=(16, 100)), dop.DOP_ERR_UNSUPPORTED_SIZE),        # product != nx
    (dict(xdigits=(2, 1024)), None),                                # fine: 2 x 1024
    (dict(xdigits=(1024, 2)), dop.DOP_ERR_UNSUPPORTED_SIZE),        # a non-last x digit is limited to 512
    (dict(ydigits=(1024,)), dop.DOP_ERR_UNSUPPORTED_SIZE),          # y digits are limited to 512
    (dict(col_nb=48), dop.DOP_ERR_INVALID_ARG),
    (dict(tile_pts=100), dop.DOP_ERR_INVALID_ARG),
    (dict(prefetch_waves=65), dop.DOP_ERR_INVALID_ARG),
])
def test_tuning_is_validated(tun, status):
    """A forced decomposition obeys the same limits as the automatic split: the launch
    can then never ask for more shared memory than a CTA has."""
    args = (1024, 2048, 0.25e-6, (550e-9,), (1.5,), 1e-3, dop.DOP_LOSS_L2, 0.0, 0)
    if status is None:
        h, _ = dop.dop_plan_create(*args, tuning=dop.make_tuning(**tun))
        dop.dop_plan_destroy(h)
        return
    with pytest.raises(dop.DopError) as e:
        dop.dop_plan_create(*args, tuning=dop.make_tuning(**tun))
    assert e.value.status == status


def test_loss_scratch_matches_the_launched_loss_pass():
    """with a forced column bundle width the loss pass launches fewer, wider CTAs;
    the scratch and the final reduce must count the CTAs actually launched."""
    for tun, ctas in ((dict(no_tma=1), 512), (dict(no_tma=1, col_nb=32), 256), (dict(no_tma=1, col_nb=64), 128),
                      (dict(), 512), (dict(tma_nb=32), 256)):
        h, _ = dop.dop_plan_create(64, 16384, 0.25e-6, (550e-9,), (1.5,), 1e-3, dop.DOP_LOSS_L2, 0.0, 0,
                                   tuning=dop.make_tuning(xdigits=(128, 128), no_cluster=1, **tun))
        text = dop.dop_plan_describe(h)
        dop.dop_plan_destroy(h)
        line = [l for l in text.splitlines() if "loss,seed" in l][0]
        assert f"ctas={ctas} " in line, line
        assert f"loss_tiles={ctas}" in text, text


@pytest.mark.parametrize("ny,nx,expect", [
    (3600, 3600, ["x-digits: 3600(", "radix=5.5.3.3.4.4", "y1 L=16 tile=32x16 col tma"]),                  # PAPER.md:274 Table 2
    (28800, 28800, ["x-digits: 32(st=900,radix=4.4.2) 900(st=1,radix=5.3.2.5.3.2)", "y-digits: 225(st=128,radix=5.3.5.3) 128(",
                    "x0 L=32 tile=32x32 col tma", "y1 L=128 tile=16x128 col tma", "x1 L=900 tile=8x900 row smooth",
                    "y0 L=225 tile=32x225 col smooth"]),
    (40000, 40000, ["x-digits: 16(st=2500,radix=4.4) 2500(st=1,radix=5.5.2.5.5.2)", "y-digits: 625(st=64,radix=5.5.5.5) 64(",
                    "x0 L=16 tile=32x16 col tma", "y1 L=64 tile=16x64 col tma", "x1 L=2500 tile=4x2500 row smooth",
                    "y0 L=625 tile=16x625 col smooth"]),
    (128640, 85760, ["x-digits: 64(st=1340,radix=4.4.4) 1340(st=1,radix=67.5.4)", "y-digits: 384(st=335", "335(st=1,radix=67.5)",
                     "x0 L=64 tile=16x64 col tma", "y0 L=384 tile=32x384 col tma"]),
])
def test_the_papers_own_grid_sizes_plan(ny, nx, expect):
    """the grids of PAPER.md:270-280 (Table 2) factor into digits with prime factors 5 and 67; the
    plan puts the fused passes (first x digit, last y digit) on power-of-two digits, i.e. on the specialised
    kernels -- a ragged last column tile (225 or 335 lines) is clipped by the TMA unit --, runs the plain passes of the
    5-smooth digits 225 / 625 / 900 / 2500 on the register-step kernels (smooth.cu) and gives the prime 67 to the generic
    kernel's direct butterflies.  128 640 x 85 760 (the paper's 16-GPU grid) fits one B200 in place: field 82.2 GiB."""
    h, ws = dop.dop_plan_create(ny, nx, 0.5e-6, (520.6e-9,), (1.5,), 0.06)
    text = dop.dop_plan_describe(h)
    dop.dop_plan_destroy(h)
    for e in expect:
        assert e in text, (e, text)
    assert ws >= ny * nx * 8


def test_pad_and_band_limit_arguments_are_validated():
    """dop_plan_desc.pad / band_limit: host-side validation and the window-sized workspace."""
    args = (64, 64, 0.25e-6, (550e-9,), (1.5,), 1e-3)
    for kw in (dict(pad=3), dict(band_limit=1), dict(pad=2, prefilter_sigma_px=2.0), dict(pad=2, upsample=2),
               dict(pad=2, loss=dop.DOP_LOSS_SIMSE)):
        with pytest.raises(dop.DopError) as e:
            dop.dop_plan_create(*args, **kw)
        assert e.value.status == dop.DOP_ERR_INVALID_ARG
    hnd, ws = dop.dop_plan_create(*args, pad=2, band_limit=1)
    text = dop.dop_plan_describe(hnd)
    dop.dop_plan_destroy(hnd)
    assert ws >= 4 * 64 * 64 * 8 and "grid ny=128 nx=128" in text and "pad=2 band_limit=1" in text
    # the x passes are pruned to the aperture rows: half the CTAs of the full window
    line = [l for l in text.splitlines() if "h->u0" in l][0]
    assert "ctas=2 " in line, line   # 64 aperture rows of 128 points = 2 tiles of 32 lines (the window has 128 rows)
