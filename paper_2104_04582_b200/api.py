"""Thin Python binding of libfew_b200 (include/few.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch supplies device buffers and the current stream.
Function names and argument meaning mirror include/few.h.  There is no CPU fallback: importing this module fails
loudly when libfew_b200.so is missing and cannot be built, and `context()` fails when no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

_PKG = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_PKG, "libfew_b200.so")

FEW_OK = 0
SYMBOLS = ["few_create", "few_destroy", "few_strerror", "few_last_error", "few_version", "few_device_status", "few_ylm",
           "few_ylm_modes", "few_spline_fit_workspace", "few_spline_fit", "few_spline_fit_dd", "few_select_modes_workspace", "few_select_modes",
           "few_sum_waveform_workspace", "few_sum_waveform", "few_waveform_workspace", "few_waveform", "few_waveform_host",
           "few_fp64_peak_probe", "few_launch_count", "few_profile_enable", "few_profile_sum_ms", "few_sum_waveform_ex", "few_frame_constants",
           "few_frame_rotate", "few_inner_products_workspace", "few_inner_products", "few_inner_products_static", "few_waveform_ssb", "few_sum_direct_workspace",
           "few_sum_direct", "few_sum_waveform_kerr", "few_waveform_kerr", "few_spline_fit_ragged", "few_spline_fit_dd_ragged",
           "few_select_modes_ragged", "few_sum_waveform_ragged", "few_waveform_ragged", "few_waveform_host_ragged",
           "few_max_steps_for_modes", "few_set_max_steps", "few_sum_waveform_workspace_ex", "few_waveform_workspace_ex"]


class FewError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib.few_strerror(code).decode()
        detail = _lib.few_last_error().decode()
        super().__init__(f"{where}: {msg}" + (f" ({detail})" if detail else ""))


def _load() -> C.CDLL:
    if not os.path.exists(_SO):
        _build.build()          # raises if nvcc is missing: no fallback
    lib = C.CDLL(_SO)
    vp, i, d, ll, sz = C.c_void_p, C.c_int, C.c_double, C.c_longlong, C.c_size_t
    sig = {
        "few_create": (i, [C.POINTER(vp), i]),
        "few_destroy": (i, [vp]),
        "few_strerror": (C.c_char_p, [i]),
        "few_last_error": (C.c_char_p, []),
        "few_version": (i, []),
        "few_device_status": (i, [vp, C.POINTER(i), vp]),
        "few_ylm": (i, [i, i, d, d, C.POINTER(d)]),
        "few_ylm_modes": (i, [vp, vp, vp, vp, vp, i, i, vp, vp, vp]),
        "few_spline_fit_workspace": (sz, [i, i]),
        "few_spline_fit": (i, [vp, vp, vp, i, i, i, vp, vp, sz, vp]),
        "few_spline_fit_dd": (i, [vp, vp, vp, i, i, i, vp, vp]),
        "few_select_modes_workspace": (sz, [i, i, i]),
        "few_select_modes": (i, [vp, vp, vp, vp, vp, d, i, i, i, vp, vp, vp, sz, vp]),
        "few_sum_waveform_workspace": (sz, [i, i, i, ll]),
        "few_sum_waveform": (i, [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, d, d, ll, vp, i, i, i, vp, sz, vp]),
        "few_waveform_workspace": (sz, [i, i, i, ll]),
        "few_waveform_workspace_ex": (sz, [i, i, i, ll, i]),
        "few_sum_waveform_workspace_ex": (sz, [i, i, i, ll, i]),
        "few_set_max_steps": (i, [vp, i]),
        "few_max_steps_for_modes": (i, [vp, vp, vp, i]),
        "few_waveform": (i, [vp] * 10 + [d, d, d, ll, i, i, i, vp, vp, vp, vp, sz, vp]),
        "few_waveform_kerr": (i, [vp] * 11 + [d, d, d, ll, i, i, i, vp, vp, vp, vp, sz, vp]),
        "few_waveform_host": (i, [vp] * 10 + [d, d, d, ll, i, i, i, vp, vp, vp]),
        "few_sum_waveform_ex": (i, [vp] * 13 + [d, d, ll, vp, vp, vp, i, i, i, vp, sz, vp]),
        "few_sum_waveform_kerr": (i, [vp, vp, vp, vp, i] + [vp] * 10 + [d, d, ll, vp, vp, vp, i, i, i, vp, sz, vp]),
        "few_spline_fit_ragged": (i, [vp, vp, vp, vp, i, i, i, vp, vp, sz, vp]),
        "few_spline_fit_dd_ragged": (i, [vp, vp, vp, vp, i, i, i, vp, vp]),
        "few_select_modes_ragged": (i, [vp, vp, vp, vp, vp, vp, d, i, i, i, vp, vp, vp, sz, vp]),
        "few_sum_waveform_ragged": (i, [vp, vp, vp, vp, vp, i] + [vp] * 10 + [d, d, ll, vp, vp, vp, i, i, i, vp, sz, vp]),
        "few_waveform_ragged": (i, [vp] * 11 + [d, d, d, ll, i, i, i, vp, vp, vp, vp, sz, vp]),
        "few_waveform_host_ragged": (i, [vp] * 11 + [d, d, d, ll, i, i, i, vp, vp, vp]),
        "few_frame_constants": (i, [vp, vp, vp, i, vp, vp, vp, vp]),
        "few_frame_rotate": (i, [vp, vp, vp, i, ll, vp, vp]),
        "few_inner_products_workspace": (sz, [i, ll]),
        "few_inner_products": (i, [vp, vp, vp, i, ll, d, vp, vp, sz, vp]),
        "few_inner_products_static": (i, [vp, vp, vp, i, ll, d, vp, vp]),
        "few_waveform_ssb": (i, [vp] * 9 + [d, d, d, ll, i, i, i, vp, vp, vp, vp, vp, vp, sz, vp]),
        "few_sum_direct_workspace": (sz, [i, i]),
        "few_sum_direct": (i, [vp] * 10 + [ll, i, i, vp, vp, sz, vp]),
        "few_fp64_peak_probe": (i, [vp, i, i, i, vp, vp]),
        "few_launch_count": (i, [vp, C.POINTER(C.c_longlong)]),
        "few_profile_enable": (i, [vp, i]),
        "few_profile_sum_ms": (i, [vp, C.POINTER(C.c_float)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


_lib = _load()
_ctx: dict[int, C.c_void_p] = {}


def context(device: int | None = None) -> C.c_void_p:
    """few_ctx of a CUDA device (created once per device)."""
    if not torch.cuda.is_available():
        raise RuntimeError("libfew_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    dev = torch.cuda.current_device() if device is None else int(device)
    if dev not in _ctx:
        h = C.c_void_p()
        rc = _lib.few_create(C.byref(h), dev)
        if rc != FEW_OK:
            raise FewError(rc, "few_create")
        _ctx[dev] = h
    return _ctx[dev]


def _chk(rc: int, where: str):
    if rc != FEW_OK:
        raise FewError(rc, where)


def _p(x: torch.Tensor | None, dtype=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if x is None:
        return None
    if not (x.is_cuda and x.is_contiguous()):
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and x.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {x.dtype}")
    return C.c_void_p(x.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ws(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)   # torch CUDA allocations are 512-B aligned


def few_version() -> int:
    return int(_lib.few_version())


def few_device_status(raise_on_error: bool = True) -> int:
    bits = C.c_int(0)
    rc = _lib.few_device_status(context(), C.byref(bits), _stream())
    if rc != FEW_OK and raise_on_error:
        raise FewError(rc, "few_device_status")
    return rc


def few_ylm(l: int, m: int, theta: float, phi: float) -> complex:
    out = (C.c_double * 2)()
    _chk(_lib.few_ylm(int(l), int(m), float(theta), float(phi), out), "few_ylm")
    return complex(out[0], out[1])


def few_ylm_modes(theta, phi, l, m):
    """theta, phi [n_src] f64; l, m [n_modes] i32 -> (ylm_plus, ylm_minus) complex128 [n_src, n_modes]."""
    n_src, n_modes = theta.shape[0], l.shape[0]
    yp = torch.empty((n_src, n_modes), dtype=torch.complex128, device=theta.device)
    ym = torch.empty_like(yp)
    _chk(_lib.few_ylm_modes(context(), _p(theta, torch.float64), _p(phi, torch.float64), _p(l, torch.int32), _p(m, torch.int32),
                            n_src, n_modes, _p(yp), _p(ym), _stream()), "few_ylm_modes")
    return yp, ym


def few_spline_fit(t, y, out=None, workspace=None):
    """t [n_src, n_t] f64; y [n_src, n_t, n_sys] f64 (or complex128 [n_src, n_t, n_modes], viewed as 2 n_modes systems)
    -> coef [n_src, n_t-1, 4, n_sys]."""
    if y.dtype == torch.complex128:
        y = torch.view_as_real(y).reshape(y.shape[0], y.shape[1], -1)
    n_src, n_t, n_sys = y.shape
    coef = out if out is not None else torch.empty((n_src, max(n_t - 1, 0), 4, n_sys), dtype=torch.float64, device=y.device)
    ws = workspace if workspace is not None else _ws(_lib.few_spline_fit_workspace(n_src, n_t), y.device)
    _chk(_lib.few_spline_fit(context(), _p(t, torch.float64), _p(y, torch.float64), n_src, n_t, n_sys, _p(coef, torch.float64),
                             _p(ws), ws.numel(), _stream()), "few_spline_fit")
    return coef


def few_spline_fit_dd(t, y, out=None):
    """y [n_src, n_t, n_sys] f64 -> coef_dd [n_src, n_t-1, 4, n_sys, 2] (hi, lo)."""
    n_src, n_t, n_sys = y.shape
    coef = out if out is not None else torch.empty((n_src, max(n_t - 1, 0), 4, n_sys, 2), dtype=torch.float64, device=y.device)
    _chk(_lib.few_spline_fit_dd(context(), _p(t, torch.float64), _p(y, torch.float64), n_src, n_t, n_sys, _p(coef, torch.float64),
                                _stream()), "few_spline_fit_dd")
    return coef


def few_select_modes(amp, m, ylm_plus, ylm_minus, eps: float, workspace=None, keep_idx=None, n_keep=None):
    """amp [n_src, n_t, n_modes] c128 -> (keep_idx [n_src, n_modes] i32 ascending, padded -1; n_keep [n_src] i32)."""
    n_src, n_t, n_modes = amp.shape
    keep = keep_idx if keep_idx is not None else torch.empty((n_src, n_modes), dtype=torch.int32, device=amp.device)
    nk = n_keep if n_keep is not None else torch.empty((n_src,), dtype=torch.int32, device=amp.device)
    need = _lib.few_select_modes_workspace(n_src, n_t, n_modes)
    ws = workspace if workspace is not None else _ws(need, amp.device)
    _chk(_lib.few_select_modes(context(), _p(amp, torch.complex128), _p(m, torch.int32), _p(ylm_plus), _p(ylm_minus), float(eps),
                               n_src, n_t, n_modes, _p(keep), _p(nk), _p(ws), ws.numel(), _stream()), "few_select_modes")
    return keep, nk


def few_sum_waveform(t, coef_amp, coef_phase_dd, l, m, n, keep_idx, n_keep, ylm_plus, ylm_minus, t0: float, dt: float,
                     n_samples: int, scale=None, out=None, workspace=None):
    """-> h [n_src, n_samples] complex128 = h_+ - i h_x."""
    n_src, n_t = t.shape
    n_modes = l.shape[0]
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    need = few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples)
    ws = workspace if workspace is not None else _ws(need, t.device)
    _chk(_lib.few_sum_waveform(context(), _p(t, torch.float64), _p(coef_amp, torch.float64), _p(coef_phase_dd, torch.float64),
                               _p(l, torch.int32), _p(m, torch.int32), _p(n, torch.int32), _p(keep_idx), _p(n_keep),
                               _p(ylm_plus, torch.complex128), _p(ylm_minus, torch.complex128), _p(scale), float(t0), float(dt),
                               int(n_samples), _p(h), n_src, n_t, n_modes, _p(ws), ws.numel(), _stream()), "few_sum_waveform")
    return h


def few_sum_waveform_ex(t, coef_amp, coef_phase_dd, l, m, n, keep_idx, n_keep, ylm_plus, ylm_minus, t0: float, dt: float,
                        n_samples: int, scale=None, factor=None, d=None, want_inner: bool = False, want_h: bool = True,
                        out=None, workspace=None):
    """few_sum_waveform with the complex per-source `factor` [n_src] c128 and the fused PSD = 1 inner products against
    d [n_src, n_samples] c128.  -> (h or None, inner [n_src, 3] f64 or None)."""
    n_src, n_t = t.shape
    n_modes = l.shape[0]
    h = None
    if want_h:
        h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    inner = torch.empty((n_src, 3), dtype=torch.float64, device=t.device) if (want_inner or d is not None) else None
    need = few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples)
    ws = workspace if workspace is not None else _ws(need, t.device)
    _chk(_lib.few_sum_waveform_ex(context(), _p(t, torch.float64), _p(coef_amp, torch.float64), _p(coef_phase_dd, torch.float64),
                                  _p(l, torch.int32), _p(m, torch.int32), _p(n, torch.int32), _p(keep_idx), _p(n_keep),
                                  _p(ylm_plus, torch.complex128), _p(ylm_minus, torch.complex128), _p(scale), _p(factor),
                                  float(t0), float(dt), int(n_samples), _p(h), _p(d), _p(inner), n_src, n_t, n_modes, _p(ws),
                                  ws.numel(), _stream()), "few_sum_waveform_ex")
    return h, inner


def few_sum_waveform_kerr(t, coef_amp, coef_phase_dd, l, m, k, n, keep_idx, n_keep, ylm_plus, ylm_minus, t0: float, dt: float,
                          n_samples: int, scale=None, factor=None, d=None, want_inner: bool = False, want_h: bool = True,
                          out=None, workspace=None):
    """Summation for Kerr-shaped mode lists: coef_phase_dd [n_src, n_t-1, 4, n_phase, 2] with n_phase = 3 (Phi_phi, Phi_theta,
    Phi_r) or 2; k [n_modes] i32 or None.  -> (h or None, inner or None)."""
    n_src, n_t = t.shape
    n_modes = l.shape[0]
    n_phase = int(coef_phase_dd.shape[3])
    h = None
    if want_h:
        h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    inner = torch.empty((n_src, 3), dtype=torch.float64, device=t.device) if (want_inner or d is not None) else None
    need = few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples)
    ws = workspace if workspace is not None else _ws(need, t.device)
    _chk(_lib.few_sum_waveform_kerr(context(), _p(t, torch.float64), _p(coef_amp, torch.float64), _p(coef_phase_dd, torch.float64),
                                    n_phase, _p(l, torch.int32), _p(m, torch.int32), _p(k), _p(n, torch.int32), _p(keep_idx),
                                    _p(n_keep), _p(ylm_plus, torch.complex128), _p(ylm_minus, torch.complex128), _p(scale),
                                    _p(factor), float(t0), float(dt), int(n_samples), _p(h), _p(d), _p(inner), n_src, n_t, n_modes,
                                    _p(ws), ws.numel(), _stream()), "few_sum_waveform_kerr")
    return h, inner


def few_frame_constants(sky, mu_over_dl=None):
    """sky [n_src, 4] f64 = (theta_S, phi_S, theta_K, phi_K) -> (theta [n_src], phi [n_src], factor [n_src] c128)."""
    n_src = sky.shape[0]
    theta = torch.empty(n_src, dtype=torch.float64, device=sky.device)
    phi = torch.empty_like(theta)
    factor = torch.empty(n_src, dtype=torch.complex128, device=sky.device)
    _chk(_lib.few_frame_constants(context(), _p(sky, torch.float64), _p(mu_over_dl), n_src, _p(theta), _p(phi), _p(factor), _stream()),
         "few_frame_constants")
    return theta, phi, factor


def few_frame_rotate(h, factor, out=None):
    """h [n_src, n_samples] c128, factor [n_src] c128 -> factor[:, None] * h (a separate pass; `out` may be h)."""
    n_src, n_samples = h.shape
    o = out if out is not None else torch.empty_like(h)
    _chk(_lib.few_frame_rotate(context(), _p(h, torch.complex128), _p(factor, torch.complex128), n_src, int(n_samples), _p(o),
                               _stream()), "few_frame_rotate")
    return o


def few_inner_products(d, h, dt: float, workspace=None):
    """d, h [n_src, n_samples] c128 -> inner [n_src, 3] f64 = (<d|h>, imaginary companion, <h|h>), PSD = 1."""
    n_src, n_samples = h.shape
    inner = torch.empty((n_src, 3), dtype=torch.float64, device=h.device)
    ws = workspace if workspace is not None else _ws(_lib.few_inner_products_workspace(n_src, int(n_samples)), h.device)
    _chk(_lib.few_inner_products(context(), _p(d, torch.complex128), _p(h, torch.complex128), n_src, int(n_samples), float(dt),
                                 _p(inner), _p(ws), ws.numel(), _stream()), "few_inner_products")
    return inner


INNER_STATIC_MAX_CHUNKS = 16384     # FEW_INNER_STATIC_MAX_CHUNKS of include/few.h


def few_inner_products_static(d, h, dt: float, out, use_context: bool = True):
    """few_inner_products without a workspace, for callers that may not allocate device memory (code running where the CUDA
    runtime refuses allocations, a sampler whose memory pool must not grow, a plug-in without an allocator of its own).

    d, h [n_src, n_samples] c128 and the result buffer `out` [n_src, 3] f64 are the caller's; this binding allocates nothing
    either, which is why `out` is required.  The partial sums go to a 512 KB array built into the library, so the call is
    limited to n_src * ceil(n_samples / 2048) <= INNER_STATIC_MAX_CHUNKS (FewError with FEW_ERR_LIMIT beyond) and two calls
    that could run at the same time on one GPU (two streams, two threads) would corrupt each other: keep them on one stream.
    The first call on a device looks up the array's device address; make it before any stream capture.
    use_context=False passes ctx = NULL, as a caller that never ran few_create (which allocates) would.  Returns `out`."""
    n_src, n_samples = h.shape
    if tuple(out.shape) != (n_src, 3):
        raise ValueError("out must be [n_src, 3]")
    ctx = context() if use_context else None
    _chk(_lib.few_inner_products_static(ctx, _p(d, torch.complex128), _p(h, torch.complex128), n_src, int(n_samples), float(dt),
                                        _p(out, torch.float64), _stream()), "few_inner_products_static")
    return out


def few_waveform_ssb(t, phase, amp, l, m, n, sky, eps: float, t0: float, dt: float, n_samples: int, mu_over_dl=None, d=None,
                     want_inner: bool = False, want_h: bool = True, out=None, keep_idx=None, n_keep=None, workspace=None):
    """Whole path in the detector frame.  -> (h or None, inner or None)."""
    n_src, n_t, n_modes = amp.shape
    h = None
    if want_h:
        h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    inner = torch.empty((n_src, 3), dtype=torch.float64, device=t.device) if (want_inner or d is not None) else None
    ws = workspace if workspace is not None else _ws(few_waveform_workspace(n_src, n_t, n_modes, n_samples), t.device)
    _chk(_lib.few_waveform_ssb(context(), _p(t, torch.float64), _p(phase, torch.float64), _p(amp, torch.complex128),
                               _p(l, torch.int32), _p(m, torch.int32), _p(n, torch.int32), _p(sky, torch.float64), _p(mu_over_dl),
                               float(eps), float(t0), float(dt), int(n_samples), n_src, n_t, n_modes, _p(h), _p(d), _p(inner),
                               _p(keep_idx), _p(n_keep), _p(ws), ws.numel(), _stream()), "few_waveform_ssb")
    return h, inner


def few_sum_direct(amp, phase, l, m, n, ylm_plus, ylm_minus, scale=None, factor=None, out=None, workspace=None):
    """Direct summation.  amp [n_src, N, K] c128, phase [n_src, N, 2] f64 -> h [n_src, N] c128."""
    n_src, n_samples, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, n_samples), dtype=torch.complex128, device=amp.device)
    ws = workspace if workspace is not None else _ws(_lib.few_sum_direct_workspace(n_src, n_modes), amp.device)
    _chk(_lib.few_sum_direct(context(), _p(amp, torch.complex128), _p(phase, torch.float64), _p(l, torch.int32), _p(m, torch.int32),
                             _p(n, torch.int32), _p(ylm_plus, torch.complex128), _p(ylm_minus, torch.complex128), _p(scale),
                             _p(factor), int(n_samples), n_src, n_modes, _p(h), _p(ws), ws.numel(), _stream()), "few_sum_direct")
    return h


_max_steps: dict[int, int] = {}     # the bound set per device through few_set_max_steps (the binding's own workspace sizes follow it)


def few_max_steps_for_modes(m, n, k=None) -> int:
    """Most summation steps any kept subset of the mode list (m, k, n: CPU i32 tensors, k optional) can produce (HOST helper)."""
    rc = int(_lib.few_max_steps_for_modes(_hp(m, torch.int32), _hp(k, torch.int32), _hp(n, torch.int32), int(m.numel())))
    if rc < 0:
        raise FewError(rc, "few_max_steps_for_modes")
    return rc


def few_set_max_steps(max_steps: int) -> None:
    """Bound the summation's steps per source on the current device's context (0 = default): smaller workspaces, see few.h."""
    _chk(_lib.few_set_max_steps(context(), int(max_steps)), "few_set_max_steps")
    _max_steps[torch.cuda.current_device()] = int(max_steps)


def _cap() -> int:
    return _max_steps.get(torch.cuda.current_device(), 0) if torch.cuda.is_available() else 0


def few_sum_waveform_workspace(n_src: int, n_t: int, n_modes: int, n_samples: int, max_steps: int | None = None) -> int:
    """Bytes few_sum_waveform* needs; max_steps None = the bound currently set on this device's context."""
    return int(_lib.few_sum_waveform_workspace_ex(n_src, n_t, n_modes, int(n_samples), _cap() if max_steps is None else int(max_steps)))


def few_waveform_workspace(n_src: int, n_t: int, n_modes: int, n_samples: int, max_steps: int | None = None) -> int:
    """Bytes few_waveform* needs; max_steps None = the bound currently set on this device's context."""
    return int(_lib.few_waveform_workspace_ex(n_src, n_t, n_modes, int(n_samples), _cap() if max_steps is None else int(max_steps)))


def few_waveform(t, phase, amp, l, m, n, theta, phi, eps: float, t0: float, dt: float, n_samples: int, scale=None,
                 out=None, keep_idx=None, n_keep=None, workspace=None):
    """Whole path on device tensors.  -> h [n_src, n_samples] complex128 (keep_idx / n_keep are filled if given)."""
    n_src, n_t, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    ws = workspace if workspace is not None else _ws(few_waveform_workspace(n_src, n_t, n_modes, n_samples), t.device)
    _chk(_lib.few_waveform(context(), _p(t, torch.float64), _p(phase, torch.float64), _p(amp, torch.complex128), _p(l, torch.int32),
                           _p(m, torch.int32), _p(n, torch.int32), _p(theta, torch.float64), _p(phi, torch.float64), _p(scale),
                           float(eps), float(t0), float(dt), int(n_samples), n_src, n_t, n_modes, _p(h), _p(keep_idx), _p(n_keep),
                           _p(ws), ws.numel(), _stream()), "few_waveform")
    return h


def few_waveform_kerr(t, phase, amp, l, m, k, n, theta, phi, eps: float, t0: float, dt: float, n_samples: int, scale=None,
                      out=None, keep_idx=None, n_keep=None, workspace=None):
    """Whole path for Kerr-shaped mode lists: phase [n_src, n_t, 3] = (Phi_phi, Phi_theta, Phi_r), k [n_modes] i32."""
    n_src, n_t, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    ws = workspace if workspace is not None else _ws(few_waveform_workspace(n_src, n_t, n_modes, n_samples), t.device)
    _chk(_lib.few_waveform_kerr(context(), _p(t, torch.float64), _p(phase, torch.float64), _p(amp, torch.complex128), _p(l, torch.int32),
                                _p(m, torch.int32), _p(k, torch.int32), _p(n, torch.int32), _p(theta, torch.float64),
                                _p(phi, torch.float64), _p(scale), float(eps), float(t0), float(dt), int(n_samples), n_src, n_t, n_modes,
                                _p(h), _p(keep_idx), _p(n_keep), _p(ws), ws.numel(), _stream()), "few_waveform_kerr")
    return h


def _hp(x, dtype):
    """Host pointer of a contiguous CPU tensor."""
    if x is None:
        return None
    if x.is_cuda or not x.is_contiguous() or x.dtype != dtype:
        raise ValueError(f"expected a contiguous CPU tensor of dtype {dtype}")
    return C.c_void_p(x.data_ptr())


def few_waveform_host(t, phase, amp, l, m, n, theta, phi, eps: float, t0: float, dt: float, n_samples: int, scale=None,
                      out=None, keep_idx=None, n_keep=None, device: int | None = None):
    """Whole path on HOST tensors (pinned recommended): H2D, kernels, D2H inside the library.  -> h (CPU) [n_src, n_samples]."""
    n_src, n_t, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, pin_memory=True)
    _chk(_lib.few_waveform_host(context(device), _hp(t, torch.float64), _hp(phase, torch.float64), _hp(amp, torch.complex128),
                                _hp(l, torch.int32), _hp(m, torch.int32), _hp(n, torch.int32), _hp(theta, torch.float64),
                                _hp(phi, torch.float64), _hp(scale, torch.float64), float(eps), float(t0), float(dt), int(n_samples),
                                n_src, n_t, n_modes, _hp(h, torch.complex128), _hp(keep_idx, torch.int32), _hp(n_keep, torch.int32)),
         "few_waveform_host")
    return h


# ---- ragged batches (few.h "Ragged batches"): padded arrays with n_t = the largest knot count, n_t_src [n_src] i32 per source

def few_spline_fit_ragged(t, y, n_t_src, out=None, workspace=None):
    """few_spline_fit on padded t [n_src, n_t], y [n_src, n_t, n_sys]; rows k >= n_t_src[s] - 1 of coef are left untouched."""
    if y.dtype == torch.complex128:
        y = torch.view_as_real(y).reshape(y.shape[0], y.shape[1], -1)
    n_src, n_t, n_sys = y.shape
    coef = out if out is not None else torch.zeros((n_src, max(n_t - 1, 0), 4, n_sys), dtype=torch.float64, device=y.device)
    ws = workspace if workspace is not None else _ws(_lib.few_spline_fit_workspace(n_src, n_t), y.device)
    _chk(_lib.few_spline_fit_ragged(context(), _p(t, torch.float64), _p(y, torch.float64), _p(n_t_src, torch.int32), n_src, n_t, n_sys,
                                    _p(coef, torch.float64), _p(ws), ws.numel(), _stream()), "few_spline_fit_ragged")
    return coef


def few_spline_fit_dd_ragged(t, y, n_t_src, out=None):
    n_src, n_t, n_sys = y.shape
    coef = out if out is not None else torch.zeros((n_src, max(n_t - 1, 0), 4, n_sys, 2), dtype=torch.float64, device=y.device)
    _chk(_lib.few_spline_fit_dd_ragged(context(), _p(t, torch.float64), _p(y, torch.float64), _p(n_t_src, torch.int32), n_src, n_t, n_sys,
                                       _p(coef, torch.float64), _stream()), "few_spline_fit_dd_ragged")
    return coef


def few_select_modes_ragged(amp, m, ylm_plus, ylm_minus, n_t_src, eps: float, workspace=None, keep_idx=None, n_keep=None):
    n_src, n_t, n_modes = amp.shape
    keep = keep_idx if keep_idx is not None else torch.empty((n_src, n_modes), dtype=torch.int32, device=amp.device)
    nk = n_keep if n_keep is not None else torch.empty((n_src,), dtype=torch.int32, device=amp.device)
    ws = workspace if workspace is not None else _ws(_lib.few_select_modes_workspace(n_src, n_t, n_modes), amp.device)
    _chk(_lib.few_select_modes_ragged(context(), _p(amp, torch.complex128), _p(m, torch.int32), _p(ylm_plus), _p(ylm_minus),
                                      _p(n_t_src, torch.int32), float(eps), n_src, n_t, n_modes, _p(keep), _p(nk), _p(ws), ws.numel(),
                                      _stream()), "few_select_modes_ragged")
    return keep, nk


def few_sum_waveform_ragged(t, n_t_src, coef_amp, coef_phase_dd, l, m, k, n, keep_idx, n_keep, ylm_plus, ylm_minus, t0: float,
                            dt: float, n_samples: int, scale=None, factor=None, d=None, want_inner: bool = False,
                            want_h: bool = True, out=None, workspace=None):
    """few_sum_waveform_kerr with per-source knot counts.  -> (h or None, inner or None)."""
    n_src, n_t = t.shape
    n_modes = l.shape[0]
    n_phase = int(coef_phase_dd.shape[3])
    h = None
    if want_h:
        h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    inner = torch.empty((n_src, 3), dtype=torch.float64, device=t.device) if (want_inner or d is not None) else None
    ws = workspace if workspace is not None else _ws(few_sum_waveform_workspace(n_src, n_t, n_modes, n_samples), t.device)
    _chk(_lib.few_sum_waveform_ragged(context(), _p(t, torch.float64), _p(n_t_src, torch.int32), _p(coef_amp, torch.float64),
                                      _p(coef_phase_dd, torch.float64), n_phase, _p(l, torch.int32), _p(m, torch.int32), _p(k),
                                      _p(n, torch.int32), _p(keep_idx), _p(n_keep), _p(ylm_plus, torch.complex128),
                                      _p(ylm_minus, torch.complex128), _p(scale), _p(factor), float(t0), float(dt), int(n_samples),
                                      _p(h), _p(d), _p(inner), n_src, n_t, n_modes, _p(ws), ws.numel(), _stream()),
         "few_sum_waveform_ragged")
    return h, inner


def few_waveform_ragged(t, n_t_src, phase, amp, l, m, n, theta, phi, eps: float, t0: float, dt: float, n_samples: int, scale=None,
                        out=None, keep_idx=None, n_keep=None, workspace=None):
    """Whole path on device tensors, sources with their own knot counts.  -> h [n_src, n_samples] complex128."""
    n_src, n_t, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, device=t.device)
    ws = workspace if workspace is not None else _ws(few_waveform_workspace(n_src, n_t, n_modes, n_samples), t.device)
    _chk(_lib.few_waveform_ragged(context(), _p(t, torch.float64), _p(n_t_src, torch.int32), _p(phase, torch.float64),
                                  _p(amp, torch.complex128), _p(l, torch.int32), _p(m, torch.int32), _p(n, torch.int32),
                                  _p(theta, torch.float64), _p(phi, torch.float64), _p(scale), float(eps), float(t0), float(dt),
                                  int(n_samples), n_src, n_t, n_modes, _p(h), _p(keep_idx), _p(n_keep), _p(ws), ws.numel(), _stream()),
         "few_waveform_ragged")
    return h


def few_waveform_host_ragged(t, n_t_src, phase, amp, l, m, n, theta, phi, eps: float, t0: float, dt: float, n_samples: int,
                             scale=None, out=None, keep_idx=None, n_keep=None, device: int | None = None):
    """Whole path on HOST tensors, sources with their own knot counts (n_t_src: CPU i32).  -> h (CPU) [n_src, n_samples]."""
    n_src, n_t, n_modes = amp.shape
    h = out if out is not None else torch.empty((n_src, int(n_samples)), dtype=torch.complex128, pin_memory=True)
    _chk(_lib.few_waveform_host_ragged(context(device), _hp(t, torch.float64), _hp(n_t_src, torch.int32), _hp(phase, torch.float64),
                                       _hp(amp, torch.complex128), _hp(l, torch.int32), _hp(m, torch.int32), _hp(n, torch.int32),
                                       _hp(theta, torch.float64), _hp(phi, torch.float64), _hp(scale, torch.float64), float(eps),
                                       float(t0), float(dt), int(n_samples), n_src, n_t, n_modes, _hp(h, torch.complex128),
                                       _hp(keep_idx, torch.int32), _hp(n_keep, torch.int32)), "few_waveform_host_ragged")
    return h


def few_fp64_peak_probe(blocks: int, threads: int, iters: int, sink=None):
    sink = sink if sink is not None else torch.empty(blocks * threads, dtype=torch.float64, device="cuda")
    _chk(_lib.few_fp64_peak_probe(context(), blocks, threads, iters, _p(sink), _stream()), "few_fp64_peak_probe")
    return 2.0 * 16 * iters * blocks * threads   # FLOPs launched


def few_launch_count(device: int | None = None) -> int:
    """Kernels launched by the library through this device's context so far."""
    n = C.c_longlong(0)
    _chk(_lib.few_launch_count(context(device), C.byref(n)), "few_launch_count")
    return int(n.value)


def few_profile_enable(on: bool = True) -> None:
    _chk(_lib.few_profile_enable(context(), int(bool(on))), "few_profile_enable")


def few_profile_sum_ms() -> float:
    """Duration (ms) of the most recent few_sum_kernel launch, from the library's own CUDA events on the launch stream."""
    ms = C.c_float(0.0)
    _chk(_lib.few_profile_sum_ms(context(), C.byref(ms)), "few_profile_sum_ms")
    return float(ms.value)
