"""Thin ctypes binding of the C-ABI library (include/dop.h): same names, argument marshalling
only -- every step of the hot path runs in the CUDA kernels of libdop.so.  PyTorch appears here
only as the owner of device memory and streams.  There is no CPU fallback: if libdop.so is
missing or no sm_100 device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import torch

from . import build as _build

DOP_OK = 0
DOP_ERR_INVALID_ARG = 1
DOP_ERR_UNSUPPORTED_SIZE = 2
DOP_ERR_WORKSPACE = 3
DOP_ERR_STATE = 4
DOP_ERR_ARCH = 5
DOP_ERR_CUDA = 6
DOP_ERR_NOALLOC_LIMIT = 7
DOP_NOALLOC_MAX_POINTS = 4 * 1024 * 1024
DOP_LOSS_NONE = 0
DOP_LOSS_L2 = 1
DOP_LOSS_SIMSE = 2
DOP_LAYOUT_F32 = 0
DOP_LAYOUT_U8 = 1
DOP_LAYOUT_U16 = 2
DOP_WRITE_INTENSITY = 0x1
_LAYOUT_TORCH = {DOP_LAYOUT_F32: torch.float32, DOP_LAYOUT_U8: torch.uint8, DOP_LAYOUT_U16: torch.uint16}


class dop_tuning(C.Structure):
    _fields_ = [
        ("n_xdigits", C.c_int32), ("xdigits", C.c_int64 * 4), ("n_ydigits", C.c_int32), ("ydigits", C.c_int64 * 4),
        ("force_generic", C.c_int32), ("col_nb", C.c_int32), ("prefetch_waves", C.c_int32), ("slab_mb", C.c_int32),
        ("slab_streams", C.c_int32), ("h_float", C.c_int32), ("tile_pts", C.c_int32), ("no_cluster", C.c_int32),
        ("no_mirror", C.c_int32), ("cluster_dsmem", C.c_int32), ("cluster_lines", C.c_int32), ("cluster_force", C.c_int32),
        ("no_tma", C.c_int32), ("tma_nb", C.c_int32), ("tma_stages", C.c_int32), ("no_stencil", C.c_int32), ("no_smooth", C.c_int32),
    ]


class dop_plan_desc(C.Structure):
    _fields_ = [
        ("ny", C.c_int64), ("nx", C.c_int64), ("pitch", C.c_double), ("n_lambda", C.c_int32),
        ("lambda_", C.POINTER(C.c_double)), ("n_refr", C.POINTER(C.c_double)), ("z", C.c_double),
        ("loss", C.c_int), ("prefilter_sigma_px", C.c_double), ("flags", C.c_uint32),
        ("tuning", C.POINTER(dop_tuning)),
        ("energy_beta", C.c_double), ("upsample", C.c_int32), ("layout_dtype", C.c_int32), ("layout_step", C.c_double),
        ("pad", C.c_int32), ("band_limit", C.c_int32),
    ]


class dop_adam(C.Structure):
    _fields_ = [("lr0", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double), ("eps", C.c_double),
                ("iter", C.c_int64), ("total_iters", C.c_int64)]


def make_tuning(xdigits: Sequence[int] = (), ydigits: Sequence[int] = (), **fields) -> dop_tuning:
    """dop_tuning from keyword arguments (marshalling only): xdigits / ydigits = forced digit
    decompositions, every other keyword is the struct field of that name (include/dop.h)."""
    t = dop_tuning()
    t.n_xdigits, t.n_ydigits = len(xdigits), len(ydigits)
    for i, v in enumerate(xdigits):
        t.xdigits[i] = int(v)
    for i, v in enumerate(ydigits):
        t.ydigits[i] = int(v)
    for k, v in fields.items():
        if k not in dict(dop_tuning._fields_) or k in ("n_xdigits", "n_ydigits"):
            raise TypeError(f"dop_tuning has no field {k!r}")
        setattr(t, k, int(v))
    return t


class DopError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {dop_status_string(status)}")


def _load() -> C.CDLL:
    path = _build.LIB
    if not os.path.exists(path):
        path = _build.build()
    lib = C.CDLL(path)
    vp = C.c_void_p
    lib.dop_plan_create.argtypes = [C.POINTER(vp), C.POINTER(dop_plan_desc), C.POINTER(C.c_size_t)]
    lib.dop_plan_create.restype = C.c_int
    lib.dop_propagate_fwd.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.dop_propagate_fwd.restype = C.c_int
    lib.dop_propagate_adj.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.dop_propagate_adj.restype = C.c_int
    lib.dop_propagate_adj_adam.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(dop_adam), vp, vp]
    lib.dop_propagate_adj_adam.restype = C.c_int
    lib.dop_prefilter_noalloc.argtypes = [vp, vp, vp, vp]
    lib.dop_prefilter_noalloc.restype = C.c_int
    lib.dop_plan_destroy.argtypes = [vp]
    lib.dop_plan_destroy.restype = C.c_int
    lib.dop_status_string.argtypes = [C.c_int]
    lib.dop_status_string.restype = C.c_char_p
    lib.dop_plan_describe.argtypes = [vp, C.c_char_p, C.c_size_t]
    lib.dop_plan_describe.restype = C.c_size_t
    lib.dop_plan_launch_count.argtypes = [vp]
    lib.dop_plan_launch_count.restype = C.c_int64
    lib.dop_plan_set_profiling.argtypes = [vp, C.c_int]
    lib.dop_plan_set_profiling.restype = C.c_int
    lib.dop_plan_get_pass_times.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_double), C.c_int64]
    lib.dop_plan_get_pass_times.restype = C.c_int64
    lib.dop_plan_pass_name.argtypes = [vp, C.c_int64]
    lib.dop_plan_pass_name.restype = C.c_char_p
    return lib


_lib = _load()
EXPORTS = ("dop_plan_create", "dop_propagate_fwd", "dop_propagate_adj", "dop_propagate_adj_adam", "dop_prefilter_noalloc", "dop_plan_destroy",
           "dop_status_string", "dop_plan_describe", "dop_plan_launch_count",
           "dop_plan_set_profiling", "dop_plan_get_pass_times", "dop_plan_pass_name")


def dop_status_string(status: int) -> str:
    return _lib.dop_status_string(int(status)).decode()


def _ptr(t: Optional[torch.Tensor], dtype, what: str) -> Optional[int]:
    """device pointer of a contiguous CUDA tensor (None stays NULL)"""
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TypeError(f"{what}: need a contiguous CUDA tensor of {dtype}")
    return t.data_ptr()


def dop_plan_create(ny: int, nx: int, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float],
                    z: float, loss: int = DOP_LOSS_L2, prefilter_sigma_px: float = 0.0, flags: int = 0,
                    tuning: Optional[dop_tuning] = None, energy_beta: float = 0.0, upsample: int = 0,
                    layout_dtype: int = DOP_LAYOUT_F32, layout_step: float = 0.0, pad: int = 0, band_limit: int = 0):
    """-> (plan handle, workspace_bytes).  Host-only; raises DopError on a bad description."""
    nl = len(lambdas)
    lam = (C.c_double * max(nl, 1))(*[float(v) for v in lambdas])
    nr = (C.c_double * max(nl, 1))(*[float(v) for v in n_refr])
    d = dop_plan_desc(int(ny), int(nx), float(pitch), nl, lam, nr, float(z), int(loss),
                      float(prefilter_sigma_px), int(flags),
                      C.pointer(tuning) if tuning is not None else None,
                      float(energy_beta), int(upsample), int(layout_dtype), float(layout_step), int(pad), int(band_limit))
    out, ws = C.c_void_p(), C.c_size_t(0)
    st = _lib.dop_plan_create(C.byref(out), C.byref(d), C.byref(ws))
    if st != DOP_OK:
        raise DopError(st, "dop_plan_create")
    return out, int(ws.value)


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def dop_propagate_fwd(plan, d_height, d_target=None, d_intensity=None, d_loss=None, d_workspace=None,
                      stream=None, layout_dtype: int = DOP_LAYOUT_F32) -> None:
    st = _lib.dop_propagate_fwd(plan, _ptr(d_height, _LAYOUT_TORCH[layout_dtype], "d_height"),
                                _ptr(d_target, torch.float32, "d_target"),
                                _ptr(d_intensity, torch.float32, "d_intensity"),
                                _ptr(d_loss, torch.float64, "d_loss"),
                                None if d_workspace is None else d_workspace.data_ptr(), _stream(stream))
    if st != DOP_OK:
        raise DopError(st, "dop_propagate_fwd")


def dop_propagate_adj(plan, d_height, d_dLdI=None, d_grad_height=None, d_workspace=None, stream=None,
                      layout_dtype: int = DOP_LAYOUT_F32) -> None:
    st = _lib.dop_propagate_adj(plan, _ptr(d_height, _LAYOUT_TORCH[layout_dtype], "d_height"),
                                _ptr(d_dLdI, torch.float32, "d_dLdI"),
                                _ptr(d_grad_height, torch.float32, "d_grad_height"),
                                None if d_workspace is None else d_workspace.data_ptr(), _stream(stream))
    if st != DOP_OK:
        raise DopError(st, "dop_propagate_adj")


def dop_propagate_adj_adam(plan, d_layout, d_dLdI, d_grad_height, d_m, d_v, lr0: float, beta1: float, beta2: float,
                           eps: float, it: int, total_iters: int, d_workspace=None, stream=None) -> None:
    hp = dop_adam(float(lr0), float(beta1), float(beta2), float(eps), int(it), int(total_iters))
    st = _lib.dop_propagate_adj_adam(plan, _ptr(d_layout, torch.float32, "d_layout"), _ptr(d_dLdI, torch.float32, "d_dLdI"),
                                     _ptr(d_grad_height, torch.float32, "d_grad_height"), _ptr(d_m, torch.float32, "d_m"),
                                     _ptr(d_v, torch.float32, "d_v"), C.byref(hp),
                                     None if d_workspace is None else d_workspace.data_ptr(), _stream(stream))
    if st != DOP_OK:
        raise DopError(st, "dop_propagate_adj_adam")


def dop_prefilter_noalloc(plan, d_in, d_out, stream=None) -> None:
    """The stencil pre-filter through the library's static scratch array (no allocation; include/dop.h)."""
    st = _lib.dop_prefilter_noalloc(plan, _ptr(d_in, torch.float32, "d_in"), _ptr(d_out, torch.float32, "d_out"),
                                    _stream(stream))
    if st != DOP_OK:
        raise DopError(st, "dop_prefilter_noalloc")


def dop_plan_destroy(plan) -> None:
    st = _lib.dop_plan_destroy(plan)
    if st != DOP_OK:
        raise DopError(st, "dop_plan_destroy")


def dop_plan_describe(plan) -> str:
    n = _lib.dop_plan_describe(plan, None, 0)
    buf = C.create_string_buffer(n + 1)
    _lib.dop_plan_describe(plan, buf, n + 1)
    return buf.value.decode()


def dop_plan_launch_count(plan) -> int:
    return int(_lib.dop_plan_launch_count(plan))


def dop_plan_set_profiling(plan, enable: bool) -> None:
    st = _lib.dop_plan_set_profiling(plan, int(bool(enable)))
    if st != DOP_OK:
        raise DopError(st, "dop_plan_set_profiling")


def dop_plan_get_pass_times(plan):
    """-> list of (name, ms, algorithmic bytes per point) for every launch of the last fwd(+adj)."""
    n = int(_lib.dop_plan_get_pass_times(plan, None, None, 0))
    ms = (C.c_float * max(n, 1))()
    bpp = (C.c_double * max(n, 1))()
    _lib.dop_plan_get_pass_times(plan, ms, bpp, n)
    return [(_lib.dop_plan_pass_name(plan, i).decode(), float(ms[i]), float(bpp[i])) for i in range(n)]


class Plan:
    """Convenience owner of a plan handle and its torch-allocated workspace (marshalling only)."""

    def __init__(self, ny: int, nx: int, pitch: float, lambdas: Sequence[float], n_refr: Sequence[float],
                 z: float, loss: int = DOP_LOSS_L2, prefilter_sigma_px: float = 0.0, flags: int = 0,
                 device: str = "cuda:0", tuning: Optional[dop_tuning] = None, energy_beta: float = 0.0,
                 upsample: int = 0, layout_dtype: int = DOP_LAYOUT_F32, layout_step: float = 0.0, pad: int = 0,
                 band_limit: int = 0):
        self.ny, self.nx, self.n_lambda, self.loss, self.flags = int(ny), int(nx), len(lambdas), loss, flags
        self.pad = 2 if pad == 2 else 1
        self.layout_dtype = layout_dtype
        self.handle, self.workspace_bytes = dop_plan_create(ny, nx, pitch, lambdas, n_refr, z, loss,
                                                            prefilter_sigma_px, flags, tuning, energy_beta, upsample,
                                                            layout_dtype, layout_step, pad, band_limit)
        self.device = torch.device(device)
        self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
        self.launches = dop_plan_launch_count(self.handle)

    def describe(self) -> str:
        return dop_plan_describe(self.handle)

    def fwd(self, height, target=None, intensity=None, loss=None, stream=None) -> None:
        dop_propagate_fwd(self.handle, height, target, intensity, loss, self.workspace, stream, self.layout_dtype)

    def adj(self, height, dLdI=None, grad=None, stream=None) -> None:
        dop_propagate_adj(self.handle, height, dLdI, grad, self.workspace, stream, self.layout_dtype)

    def adj_adam(self, layout, dLdI, grad, m, v, lr0, beta1, beta2, eps, it, total_iters, stream=None) -> None:
        dop_propagate_adj_adam(self.handle, layout, dLdI, grad, m, v, lr0, beta1, beta2, eps, it, total_iters,
                               self.workspace, stream)

    def field(self) -> torch.Tensor:
        """complex64 view [n_lambda, ny, nx] of the workspace fields (valid after a DOP_LOSS_NONE fwd); with
        pad = 2 the aperture corner of each [2 ny, 2 nx] window."""
        wy, wx = self.ny * self.pad, self.nx * self.pad
        n = wy * wx
        stride = (n * 8 + 255) // 256 * 256
        out = []
        for l in range(self.n_lambda):
            raw = self.workspace[l * stride: l * stride + n * 8].view(torch.float32).view(wy, wx, 2)
            out.append(torch.view_as_complex(raw)[: self.ny, : self.nx])
        return torch.stack(out)

    def close(self) -> None:
        if self.handle is not None:
            dop_plan_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
