"""CPU oracle for the FEW interpolated mode summation -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy/ctypes front end of `few_oracle.c` (plain C, gcc).  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import this package.  It imports nothing from
`paper_2104_04582_b200` and shares no code with the CUDA path.

Functions (each follows the passage cited in few_oracle.c):
  spline_fit(t, y)            O1, FP64
  spline_fit_ext(t, y)        O1, x87 extended    PAPER.md:153 + DESIGN.md R13
  ylm(l, m, theta, phi)       O2
  select_modes(...)           O3
  sum_waveform(...)           O4                  PAPER.md:155-159, Eq. (9), Eq. (10)
  frame(qS, phiS, qK, phiK)   O5                  PAPER.md:69-102 Eq. (4)-(8)
  frame_apply(h, factor)      O5
  inner(d, h, dt)             O6                  PAPER.md:283-296 Eq. (15)-(17), PSD = 1
  sum_direct(...)             O7
  sum_waveform_kerr(...)      O8                  PAPER.md:54 Eq. (1), 438-444 Eq. (19), Eq. (9) with k
  waveform(workload)          chain O2 -> O3 -> O1 -> O4 in the paper's pipeline order
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "few_oracle.c")
_SO = os.path.join(_HERE, "libfew_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile few_oracle.c with gcc (-ffp-contract=off: every FP64 product and sum is rounded separately)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-std=c11",
                               _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _ptr(a, typ=_dp):
    return None if a is None else a.ctypes.data_as(typ)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.oracle_spline_fit.argtypes = [_dp, _dp, C.c_int, C.c_int, _dp]
        L.oracle_spline_fit_ext.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_void_p]
        L.oracle_ylm.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _dp]
        L.oracle_swsh.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp]
        L.oracle_select_modes.argtypes = [_dp, _ip, _dp, _dp, C.c_double, C.c_int, C.c_int, _ip, _ip, _dp]
        L.oracle_sum_waveform.argtypes = [_dp, _dp, C.c_void_p, _ip, _ip, _ip, _ip, C.c_int, _dp, _dp, C.c_double,
                                          C.c_int, C.c_double, C.c_double, C.c_longlong, C.c_longlong, C.c_int,
                                          C.c_int, _dp]
        L.oracle_frame.argtypes = [C.c_double] * 5 + [_dp]
        L.oracle_frame_apply.argtypes = [_dp, C.c_longlong, _dp, _dp]
        L.oracle_inner.argtypes = [_dp, _dp, C.c_longlong, C.c_double, _dp]
        L.oracle_sum_direct.argtypes = [_dp, _dp, _ip, _ip, _ip, _dp, _dp, C.c_double, C.c_int, C.c_longlong, C.c_int, _dp]
        L.oracle_sum_waveform_kerr.argtypes = [_dp, _dp, C.c_void_p, C.c_int, _ip, _ip, _ip, _ip, _ip, C.c_int, _dp, _dp,
                                               C.c_double, C.c_int, C.c_double, C.c_double, C.c_longlong, C.c_longlong,
                                               C.c_int, C.c_int, _dp]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


_ERR = {-1: "n_t < 4", -2: "t not strictly increasing"}


def spline_fit(t, y):
    """O1 in FP64.  t [n_t], y [n_t, n_sys] -> coef [n_t-1, 4, n_sys] (c0, c1, c2, c3)."""
    t = np.ascontiguousarray(t, np.float64); y = np.ascontiguousarray(y, np.float64)
    n_t, n_sys = y.shape
    coef = np.empty((max(n_t - 1, 0), 4, n_sys), np.float64)
    rc = lib().oracle_spline_fit(_ptr(t), _ptr(y), n_t, n_sys, _ptr(coef))
    if rc: raise ValueError(_ERR[rc])
    return coef


def spline_fit_ext(t, y):
    """O1 in x87 extended precision -> np.longdouble coef [n_t-1, 4, n_sys]."""
    assert np.finfo(np.longdouble).nmant == 63, "oracle needs x87 80-bit long double"
    t = np.ascontiguousarray(t, np.float64); y = np.ascontiguousarray(y, np.float64)
    n_t, n_sys = y.shape
    coef = np.empty((max(n_t - 1, 0), 4, n_sys), np.longdouble)
    rc = lib().oracle_spline_fit_ext(_ptr(t), _ptr(y), n_t, n_sys, coef.ctypes.data)
    if rc: raise ValueError(_ERR[rc])
    return coef


def ylm(l: int, m: int, theta: float, phi: float, s: int = -2) -> complex:
    out = np.empty(2)
    rc = lib().oracle_swsh(int(s), int(l), int(m), float(theta), float(phi), _ptr(out))
    if rc: raise ValueError("need l >= |s| and |m| <= l")
    return complex(out[0], out[1])


def ylm_modes(l, m, theta: float, phi: float):
    """Y+_j = -2Y_{l_j, m_j}, Y-_j = -2Y_{l_j, -m_j} for a mode list -> two complex128 [n_modes]."""
    yp = np.array([ylm(a, b, theta, phi) for a, b in zip(l, m)], np.complex128)
    ym = np.array([ylm(a, -b, theta, phi) for a, b in zip(l, m)], np.complex128)
    return yp, ym


def _c2d(z):
    return None if z is None else np.ascontiguousarray(z, np.complex128).view(np.float64)


def select_modes(amp, m, ylm_plus, ylm_minus, eps: float):
    """O3.  amp [n_t, n_modes] complex -> (keep_idx ascending int32 [n_keep], margin float64 [n_modes])."""
    a = _c2d(amp); n_t, n_modes = amp.shape
    m = np.ascontiguousarray(m, np.int32)
    yp, ym = _c2d(ylm_plus), _c2d(ylm_minus)
    keep = np.empty(n_modes, np.int32); nk = C.c_int(0); margin = np.empty(n_modes)
    lib().oracle_select_modes(_ptr(a), _ptr(m, _ip), _ptr(yp), _ptr(ym), float(eps), n_t, n_modes, _ptr(keep, _ip),
                              C.byref(nk), _ptr(margin))
    return keep[: nk.value].copy(), margin


def sum_waveform(t, coef_amp, coef_phase_ext, l, m, n, keep_idx, ylm_plus, ylm_minus, t0, dt, n_samples,
                 scale: float = 1.0, fold: bool = True, i0: int = 0):
    """O4.  coef_amp [n_t-1, 4, 2*n_modes] float64, coef_phase_ext [n_t-1, 4, 2] longdouble -> h complex128 [n_samples]."""
    t = np.ascontiguousarray(t, np.float64)
    ca = np.ascontiguousarray(coef_amp, np.float64)
    cp = np.ascontiguousarray(coef_phase_ext, np.longdouble)
    l, m, n = (np.ascontiguousarray(x, np.int32) for x in (l, m, n))
    n_t, n_modes = t.shape[0], l.shape[0]
    assert ca.shape == (n_t - 1, 4, 2 * n_modes) and cp.shape == (n_t - 1, 4, 2)
    k = None if keep_idx is None else np.ascontiguousarray(keep_idx, np.int32)
    yp = _c2d(ylm_plus)
    ym = _c2d(ylm_minus if ylm_minus is not None else np.zeros(n_modes, np.complex128))
    h = np.empty((int(n_samples), 2), np.float64)
    rc = lib().oracle_sum_waveform(_ptr(t), _ptr(ca), cp.ctypes.data, _ptr(l, _ip), _ptr(m, _ip), _ptr(n, _ip),
                                   _ptr(k, _ip), 0 if k is None else len(k), _ptr(yp), _ptr(ym), float(scale),
                                   int(bool(fold)), float(t0), float(dt), int(i0), int(n_samples), n_t, n_modes, _ptr(h))
    if rc: raise ValueError(_ERR[rc])
    return h.view(np.complex128)[:, 0]


def frame(qS: float, phiS: float, qK: float, phiK: float, mu_over_dl: float = 1.0):
    """O5.  -> (theta_src, phi_src, factor) with factor = -(mu/d_L) exp(+2 i psi) (complex)."""
    out = np.empty(4)
    lib().oracle_frame(float(qS), float(phiS), float(qK), float(phiK), float(mu_over_dl), _ptr(out))
    return float(out[0]), float(out[1]), complex(out[2], out[3])


def frame_apply(h, factor: complex):
    """O5.  h complex128 [n] -> factor * h."""
    hin = np.ascontiguousarray(h, np.complex128).reshape(-1)
    out = np.empty_like(hin)
    f = np.array([factor.real, factor.imag])
    lib().oracle_frame_apply(_ptr(hin.view(np.float64)), hin.shape[0], _ptr(f), _ptr(out.view(np.float64)))
    return out.reshape(np.shape(h))


def inner(d, h, dt: float):
    """O6.  -> (<d|h>, imaginary companion, <h|h>) for PSD = 1."""
    d = np.ascontiguousarray(d, np.complex128).reshape(-1); h = np.ascontiguousarray(h, np.complex128).reshape(-1)
    assert d.shape == h.shape
    out = np.empty(3)
    lib().oracle_inner(_ptr(d.view(np.float64)), _ptr(h.view(np.float64)), d.shape[0], float(dt), _ptr(out))
    return float(out[0]), float(out[1]), float(out[2])


def overlap(a, b, dt: float = 1.0) -> float:
    """Eq. (17) with O6's inner product."""
    ab = inner(a, b, dt)[0]
    return ab / np.sqrt(inner(a, a, dt)[0] * inner(b, b, dt)[0])


def sum_direct(amp, phase, l, m, n, ylm_plus, ylm_minus, scale: float = 1.0, fold: bool = True):
    """O7.  amp [N, K] complex128, phase [N, 2] float64 -> h complex128 [N]."""
    a = _c2d(amp); N, K = amp.shape
    ph = np.ascontiguousarray(phase, np.float64); assert ph.shape == (N, 2)
    l, m, n = (np.ascontiguousarray(x, np.int32) for x in (l, m, n))
    yp = _c2d(ylm_plus)
    ym = _c2d(ylm_minus if ylm_minus is not None else np.zeros(K, np.complex128))
    h = np.empty((N, 2), np.float64)
    lib().oracle_sum_direct(_ptr(a), _ptr(ph), _ptr(l, _ip), _ptr(m, _ip), _ptr(n, _ip), _ptr(yp), _ptr(ym), float(scale),
                            int(bool(fold)), N, K, _ptr(h))
    return h.view(np.complex128)[:, 0]


def sum_waveform_kerr(t, coef_amp, coef_phase_ext, l, m, k, n, keep_idx, ylm_plus, ylm_minus, t0, dt, n_samples,
                      scale: float = 1.0, fold: bool = True, i0: int = 0):
    """O8.  coef_phase_ext [n_t-1, 4, n_ph] longdouble with n_ph = 3 (Phi_phi, Phi_theta, Phi_r) or 2; k int32 [n_modes] or None."""
    t = np.ascontiguousarray(t, np.float64)
    ca = np.ascontiguousarray(coef_amp, np.float64)
    cp = np.ascontiguousarray(coef_phase_ext, np.longdouble)
    l, m, n = (np.ascontiguousarray(x, np.int32) for x in (l, m, n))
    kk = None if k is None else np.ascontiguousarray(k, np.int32)
    n_t, n_modes, n_ph = t.shape[0], l.shape[0], cp.shape[2]
    assert ca.shape == (n_t - 1, 4, 2 * n_modes) and cp.shape == (n_t - 1, 4, n_ph)
    kp = None if keep_idx is None else np.ascontiguousarray(keep_idx, np.int32)
    yp = _c2d(ylm_plus)
    ym = _c2d(ylm_minus if ylm_minus is not None else np.zeros(n_modes, np.complex128))
    h = np.empty((int(n_samples), 2), np.float64)
    rc = lib().oracle_sum_waveform_kerr(_ptr(t), _ptr(ca), cp.ctypes.data, n_ph, _ptr(l, _ip), _ptr(m, _ip), _ptr(kk, _ip),
                                        _ptr(n, _ip), _ptr(kp, _ip), 0 if kp is None else len(kp), _ptr(yp), _ptr(ym),
                                        float(scale), int(bool(fold)), float(t0), float(dt), int(i0), int(n_samples), n_t,
                                        n_modes, _ptr(h))
    if rc: raise ValueError(_ERR.get(rc, f"oracle error {rc}"))
    return h.view(np.complex128)[:, 0]


def waveform(w, *, windows=None, return_parts: bool = False):
    """Whole path for a synth.Workload, in the paper's order: harmonics, mode selection, spline
    fits, interpolated summation.  `windows` = list of (i0, n) sample ranges (default: the whole grid).
    Returns h [n_src][len(windows)] arrays (or a single [n_src, n_samples] array), plus parts on request."""
    hs, parts = [], []
    for s in range(w.n_src):
        yp, ym = ylm_modes(w.l, w.m, float(w.theta[s]), float(w.phi[s]))
        keep, margin = select_modes(w.amp[s], w.m, yp, ym, w.eps)
        ca = spline_fit(w.t[s], _c2d(w.amp[s]))
        cp = spline_fit_ext(w.t[s], w.phase[s])
        wins = windows if windows is not None else [(0, w.n_samples)]
        hw = [sum_waveform(w.t[s], ca, cp, w.l, w.m, w.n, keep, yp, ym, w.t0, w.dt, nn, i0=i0) for (i0, nn) in wins]
        hs.append(hw if windows is not None else hw[0])
        parts.append(dict(ylm_plus=yp, ylm_minus=ym, keep_idx=keep, margin=margin, coef_amp=ca, coef_phase=cp))
    out = hs if windows is not None else np.stack(hs)
    return (out, parts) if return_parts else out
