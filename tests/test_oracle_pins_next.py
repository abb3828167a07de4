"""Pins of the oracle functions of the SURVEY.md section 8(f) rows (no GPU, no CUDA path):
  P12  oracle.frame / frame_apply   detector-frame transformation, Eq. (4)-(8)
  P13  oracle.inner                 PSD = 1 inner product, Eq. (15)-(17)
  P14  oracle.sum_direct            direct summation, PAPER.md:151, 248
Each check rebuilds the quantity by a route that shares nothing with few_oracle.c (vector geometry, an FFT, a closed form,
mpmath), so a wrong sign, a swapped angle or a dropped factor fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2104_04582_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_facts.txt")


def paper_angles():
    """(theta_S, phi_S, theta_K, phi_K) the paper uses for all its tests."""
    v = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 2 and line[0].startswith("angles_"):
            v[line[0]] = float(line[1])
    return v["angles_theta_S"], v["angles_phi_S"], v["angles_theta_K"], v["angles_phi_K"]


def unit(q, p):
    return np.array([math.sin(q) * math.cos(p), math.sin(q) * math.sin(p), math.cos(q)])


ANGLES = [paper_angles(), (1.0, 0.3, 2.2, 4.0), (2.9, 1.0, 0.2, 1.5), (0.3, 6.0, 0.31, 5.9), (1.5707, 3.0, 1.0, 3.0 + 1e-3)]


# ---------------------------------------------------------------- P12: frame
@pytest.mark.parametrize("ang", ANGLES)
def test_p12_frame_matches_wave_frame_geometry(ang):
    """Eq. (8) (as tan psi, R22) against the wave frame BUILT from Eq. (4)-(6) with cross products: x_w = R x S / |.|
    makes the angle psi with e_theta(S-sky) towards e_phi, i.e. x_w = cos psi e_theta + sin psi e_phi."""
    qS, pS, qK, pK = ang
    th, ph, f = oracle.frame(qS, pS, qK, pK)
    R, S = unit(qS, pS), unit(qK, pK)
    xw = np.cross(R, S); xw /= np.linalg.norm(xw)                                    # Eq. (6)
    e_th = np.array([math.cos(qS) * math.cos(pS), math.cos(qS) * math.sin(pS), -math.sin(qS)])
    e_ph = np.array([-math.sin(pS), math.cos(pS), 0.0])
    psi = math.atan2(xw @ e_ph, xw @ e_th)
    cond = 1.0 / np.linalg.norm(np.cross(R, S))                                      # the frame degenerates as S -> +-R
    assert abs(f - (-np.exp(2j * psi))) <= 1e-14 * cond
    assert abs(abs(f) - 1.0) <= 1e-15
    assert abs(math.cos(th) - (-(R @ S))) <= 1e-15
    assert ph == -math.pi / 2
    # source frame of Eq. (7): the direction to the observer has azimuth -pi/2 there, as the paper says it must.
    # (the line of sight seen from the source is -R; Eq. (7)'s y axis is built from +R.)
    zs = S
    xs = xw
    ys = (R - (R @ S) * S); ys /= np.linalg.norm(ys)
    nhat = -R
    assert abs(math.atan2(nhat @ ys, nhat @ xs) - ph) <= 1e-13 * cond
    assert abs(math.acos(np.clip(nhat @ zs, -1, 1)) - th) <= 1e-13 * cond


def test_p12_frame_is_a_spin2_rotation_of_the_polarisation_tensor():
    """h_ij = h_+ e+_ij + h_x ex_ij built on the wave-frame basis (x_w, y_w) and projected on the basis rotated by psi
    about the line of sight -- onto the right-handed pair (e_theta, -e_phi) at the sky position -- gives (h_+ - i h_x) e^{+2 i psi}:
    the rotation 'by twice the polarization angle'."""
    qS, pS, qK, pK = paper_angles()
    _, _, f = oracle.frame(qS, pS, qK, pK)
    R, S = unit(qS, pS), unit(qK, pK)
    xw = np.cross(R, S); xw /= np.linalg.norm(xw)
    yw = S - (S @ R) * R; yw /= np.linalg.norm(yw)
    e_th = np.array([math.cos(qS) * math.cos(pS), math.cos(qS) * math.sin(pS), -math.sin(qS)])
    e_ph = np.array([-math.sin(pS), math.cos(pS), 0.0])
    psi = math.atan2(xw @ e_ph, xw @ e_th)
    rng = np.random.default_rng(12)
    hp, hx = rng.normal(size=2)
    H = hp * (np.outer(xw, xw) - np.outer(yw, yw)) + hx * (np.outer(xw, yw) + np.outer(yw, xw))
    # rotate the basis by +psi from x_w towards y_w
    p = math.cos(psi) * xw + math.sin(psi) * yw
    q = -math.sin(psi) * xw + math.cos(psi) * yw
    hp2 = 0.5 * (p @ H @ p - q @ H @ q)
    hx2 = 0.5 * (p @ H @ q + q @ H @ p)
    assert np.linalg.norm(p - e_th) <= 1e-14 and np.linalg.norm(q + e_ph) <= 1e-14
    got = oracle.frame_apply(np.array([hp - 1j * hx]), -f)[0]       # -f = e^{+2 i psi}: undo the pi phase shift of PAPER.md:98
    assert abs(got - (hp2 - 1j * hx2)) <= 1e-14


def test_p12_frame_invariances_and_scale():
    qS, pS, qK, pK = paper_angles()
    th, ph, f = oracle.frame(qS, pS, qK, pK)
    # a common rotation of the sky about z changes nothing
    th2, _, f2 = oracle.frame(qS, pS + 0.7, qK, pK + 0.7)
    assert abs(th - th2) <= 1e-15 and abs(f - f2) <= 2e-15
    # mu/d_L scales the factor (Eq. (10))
    _, _, f3 = oracle.frame(qS, pS, qK, pK, 3.5e-3)
    assert abs(f3 - 3.5e-3 * f) <= 1e-18
    # swapping the roles of the two directions flips the viewing hemisphere symmetrically: cos theta is symmetric in R, S
    th4, _, _ = oracle.frame(qK, pK, qS, pS)
    assert abs(th - th4) <= 1e-15
    # apply: plain complex product, norm preserved
    h = np.random.default_rng(3).normal(size=64) + 1j * np.random.default_rng(4).normal(size=64)
    out = oracle.frame_apply(h, f)
    assert np.max(np.abs(out - f * h)) <= 1e-15
    assert abs(np.linalg.norm(out) - np.linalg.norm(h)) <= 1e-14 * np.linalg.norm(h)


def test_p12_frame_chain_equals_waveform_at_source_angles():
    """SSB-frame waveform = factor x the Eq. (10) sum evaluated at (theta_src, phi_src): the oracle chain composes."""
    w = synth.make_config(0)
    qS, pS, qK, pK = paper_angles()
    th, ph, f = oracle.frame(qS, pS, qK, pK, 2.0)
    w.theta[:] = th; w.phi[:] = ph
    h_src = oracle.waveform(w)[0]
    h_ssb = oracle.frame_apply(h_src, f)
    assert abs(np.linalg.norm(h_ssb) - 2.0 * np.linalg.norm(h_src)) <= 1e-13 * np.linalg.norm(h_ssb)
    # e^{+2 i psi}: h_+ and h_x of the SSB frame are the pair rotated by 2 psi (with the pi phase shift and mu/d_L = 2)
    c2, s2 = (-f / 2.0).real, (-f / 2.0).imag
    hp, hx = h_src.real * 2.0, -h_src.imag * 2.0
    assert np.max(np.abs(h_ssb.real - (-(c2 * hp + s2 * hx)))) <= 1e-13 * np.max(np.abs(h_ssb))
    assert np.max(np.abs(-h_ssb.imag - (-(-s2 * hp + c2 * hx)))) <= 1e-13 * np.max(np.abs(h_ssb))


# ---------------------------------------------------------------- P13: inner products with PSD = 1
def test_p13_inner_equals_frequency_domain_form_of_eq16():
    """Eq. (16) evaluated as printed -- 4 Re int_0^inf conj(a~) b~ df with S_n = 1, a~ = dt * DFT, df = 1/(N dt), summed over the
    two polarisations -- equals the time-domain sum the oracle computes (Parseval).  The zero and Nyquist bins are their own
    mirrors and carry half weight in the one-sided integral."""
    rng = np.random.default_rng(13)
    N, dt = 4096, 10.0
    a = rng.normal(size=N) + 1j * rng.normal(size=N)
    b = rng.normal(size=N) + 1j * rng.normal(size=N)
    got = oracle.inner(a, b, dt)
    tot = 0.0
    for ar, br in ((a.real, b.real), (-a.imag, -b.imag)):          # h_+ and h_x
        A, B = np.fft.rfft(ar) * dt, np.fft.rfft(br) * dt
        wgt = np.ones(N // 2 + 1); wgt[0] = wgt[-1] = 0.5
        tot += 4.0 * np.real(np.sum(wgt * np.conj(A) * B)) / (N * dt)
    assert abs(got[0] - tot) <= 1e-12 * abs(tot) + 1e-9
    assert abs(got[0] - 2 * dt * np.real(np.vdot(a, b))) <= 1e-13 * 2 * dt * np.linalg.norm(a) * np.linalg.norm(b)
    assert abs(got[1] - 2 * dt * np.imag(np.vdot(a, b))) <= 1e-13 * 2 * dt * np.linalg.norm(a) * np.linalg.norm(b)
    assert abs(got[2] - 2 * dt * np.linalg.norm(b) ** 2) <= 1e-13 * got[2]


def test_p13_overlap_properties_eq17():
    rng = np.random.default_rng(14)
    a = rng.normal(size=1000) + 1j * rng.normal(size=1000)
    b = rng.normal(size=1000) + 1j * rng.normal(size=1000)
    assert abs(oracle.overlap(a, a) - 1.0) <= 1e-15
    assert abs(oracle.overlap(a, -a) + 1.0) <= 1e-15
    assert abs(oracle.overlap(a, 3.0 * a) - 1.0) <= 1e-15                        # normalised: amplitude drops out
    assert abs(oracle.overlap(a, b) - oracle.overlap(b, a)) <= 1e-15            # symmetric
    assert abs(oracle.overlap(a, b)) < 0.2                                       # independent noise: nearly orthogonal
    # Eq. (15): -1/2 <d-h|d-h> expands into the three sums the oracle returns
    dh, _, hh = oracle.inner(a, b, 10.0)
    dd = oracle.inner(a, a, 10.0)[2]
    lhs = -0.5 * oracle.inner(a - b, a - b, 10.0)[2]
    assert abs(lhs - (-0.5 * (dd - 2 * dh + hh))) <= 1e-12 * abs(lhs)


def test_p13_mismatch_of_mode_selected_waveform_follows_paper_power_law():
    """Fig. 3: mismatch ~1e-2 at eps = 1e-1 and falling like a power law: overlap of the eps-selected config-0-like
    waveform with the all-mode one, through O6."""
    w = synth.make_config(0)
    h_all = oracle.waveform(w)[0]
    mm = []
    for eps in (1e-1, 1e-2, 1e-3):
        w.eps = eps
        mm.append(1.0 - oracle.overlap(oracle.waveform(w)[0], h_all, w.dt))
    assert mm[0] >= mm[1] >= mm[2] >= 0.0
    assert mm[0] < 0.3 and mm[2] < 3e-3


# ---------------------------------------------------------------- P14: direct summation
@pytest.mark.parametrize("l,m,n", [(2, 2, 0), (3, 1, -4), (5, 0, 7), (10, 10, 30)])
def test_p14_direct_single_mode_closed_form(l, m, n):
    N = 257
    tt = np.arange(N) * 10.0
    om_phi, om_r = 3.1e-3, 1.9e-3
    phase = np.stack([om_phi * tt, om_r * tt], axis=1)
    a = 0.37 * np.exp(0.9j)
    amp = np.full((N, 1), a)
    yp, ym = oracle.ylm_modes([l], [m], 0.7, 1.1)
    got = oracle.sum_direct(amp, phase, [l], [m], [n], yp, ym, scale=1.5)
    th = m * phase[:, 0].astype(np.longdouble) + n * phase[:, 1].astype(np.longdouble)
    E = (np.cos(th) - 1j * np.sin(th)).astype(np.complex128)
    want = yp[0] * a * E + ((-1) ** l * ym[0] * np.conj(a * E) if m > 0 else 0.0)
    assert np.max(np.abs(got - 1.5 * want)) <= 1e-14 * abs(a)


def test_p14_direct_equals_interpolated_sum_on_dense_spline_values():
    """Feed the direct sum with the interpolated path's own splines evaluated at every sample (amplitudes in FP64, phases
    rounded to FP64): both loops must agree to the FP64 rounding of the dense phases, |m Phi| * 2^-53."""
    w = synth.make_config(0)
    s = 0
    yp, ym = oracle.ylm_modes(w.l, w.m, float(w.theta[s]), float(w.phi[s]))
    ca = oracle.spline_fit(w.t[s], np.ascontiguousarray(w.amp[s]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[s], w.phase[s])
    N = 1500
    h_int = oracle.sum_waveform(w.t[s], ca, cp, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, N)
    ti = w.t0 + np.arange(N) * w.dt
    k = np.clip(np.searchsorted(w.t[s], ti, side="right") - 1, 0, len(w.t[s]) - 2)
    dx = ti - w.t[s][k]
    A = np.empty((N, w.n_modes), np.complex128)
    c = ca[k]                                                  # [N, 4, 2 n_modes]
    val = ((c[:, 3] * dx[:, None] + c[:, 2]) * dx[:, None] + c[:, 1]) * dx[:, None] + c[:, 0]
    A = val[:, 0::2] + 1j * val[:, 1::2]
    dxl = dx.astype(np.longdouble)[:, None]
    cpk = cp[k]
    ph = (((cpk[:, 3] * dxl + cpk[:, 2]) * dxl + cpk[:, 1]) * dxl + cpk[:, 0]).astype(np.float64)
    h_dir = oracle.sum_direct(A, ph, w.l, w.m, w.n, yp, ym)
    tol = 4 * np.max(np.abs(ph)) * 2.0 ** -53 * np.max(np.abs(w.m)) * np.sum(np.abs(A[0]) * np.abs(yp)) * 2
    assert np.max(np.abs(h_dir - h_int)) <= tol


def test_p14_direct_mpmath_bruteforce_and_fold():
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    rng = np.random.default_rng(140)
    modes = [(2, 2, 1), (2, 0, -3), (3, 1, 0), (4, 3, -2)]
    l, m, n = (np.array(x, np.int32) for x in zip(*modes))
    N, K = 5, len(modes)
    amp = rng.normal(size=(N, K)) + 1j * rng.normal(size=(N, K))
    phase = rng.uniform(1e4, 1e6, size=(N, 2))
    yp, ym = oracle.ylm_modes(l, m, 1.3, 0.4)
    got = oracle.sum_direct(amp, phase, l, m, n, yp, ym, scale=0.5)
    for i in range(N):
        tot = mp.mpc(0)
        for j in range(K):
            th = int(m[j]) * mp.mpf(float(phase[i, 0])) + int(n[j]) * mp.mpf(float(phase[i, 1]))
            W = mp.mpc(float(amp[i, j].real), float(amp[i, j].imag)) * mp.expj(-th)
            tot += mp.mpc(float(yp[j].real), float(yp[j].imag)) * W
            if m[j] > 0:
                tot += (-1) ** int(l[j]) * mp.mpc(float(ym[j].real), float(ym[j].imag)) * mp.conj(W)
        assert abs(complex(tot * mp.mpf("0.5")) - got[i]) <= 1e-15 * np.sum(np.abs(amp[i]))
    # fold = explicit list with the (l, -m, -n) mirrors (Eq. (9)), fold switched off
    le, me, ne, cols, ypl = [], [], [], [], []
    for j, (lj, mj, nj) in enumerate(modes):
        le.append(lj); me.append(mj); ne.append(nj); cols.append(amp[:, j]); ypl.append(yp[j])
        if mj > 0:
            le.append(lj); me.append(-mj); ne.append(-nj); cols.append((-1) ** lj * np.conj(amp[:, j])); ypl.append(ym[j])
    h2 = oracle.sum_direct(np.stack(cols, axis=1), phase, le, me, ne, np.array(ypl), None, scale=0.5, fold=False)
    assert np.max(np.abs(h2 - got)) <= 1e-14 * np.max(np.sum(np.abs(amp), axis=1))


# ---------------------------------------------------------------- P15: Kerr-shaped summation (k index, third phase)
def _kerr_small(seed=1):
    w = synth.make_kerr(n_samples=300, n_t=12, l_max=3, k_max=2, n_max=2, t0=2_000_000.0, seed=seed)
    yp, ym = oracle.ylm_modes(w.l, w.m, 0.7, 1.1)
    ca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[0], w.phase[0])
    return w, yp, ym, ca, cp


def test_p15_kerr_sum_reduces_to_schwarzschild_sum():
    """k = 0 everywhere (or two phases): O8 is O4, bit for bit."""
    w, yp, ym, ca, cp = _kerr_small()
    k0 = np.zeros_like(w.k)
    cp2 = np.ascontiguousarray(cp[:, :, [0, 2]])
    ref = oracle.sum_waveform(w.t[0], ca, cp2, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, w.n_samples)
    assert np.array_equal(oracle.sum_waveform_kerr(w.t[0], ca, cp, w.l, w.m, k0, w.n, None, yp, ym, w.t0, w.dt, w.n_samples), ref)
    assert np.array_equal(oracle.sum_waveform_kerr(w.t[0], ca, cp2, w.l, w.m, None, w.n, None, yp, ym, w.t0, w.dt, w.n_samples), ref)


@pytest.mark.parametrize("l,m,k,n", [(2, 2, 1, 0), (3, 1, -2, 4), (4, 0, 3, -1), (5, 5, -1, -3)])
def test_p15_kerr_single_mode_closed_form(l, m, k, n):
    """Constant amplitude, linear phases (splines of lines are exact): h = a Y+ e^{-i w t} + [m>0] (-1)^{l+k} conj(a) Y- e^{+i w t},
    w = m Om_phi + k Om_theta + n Om_r."""
    t = np.linspace(0.0, 5000.0, 9)
    om = np.array([3.1e-3, 2.3e-3, 1.9e-3])
    a = 0.6 * np.exp(-0.4j)
    ca = oracle.spline_fit(t, np.tile(np.array([[a.real, a.imag]]), (9, 1)))
    cp = oracle.spline_fit_ext(t, t[:, None] * om[None, :])
    yp, ym = oracle.ylm_modes([l], [m], 1.0, 2.0)
    got = oracle.sum_waveform_kerr(t, ca, cp, [l], [m], [k], [n], None, yp, ym, 0.0, 12.5, 400)
    ti = 12.5 * np.arange(400)
    wt = (m * om[0] + k * om[1] + n * om[2]) * ti
    want = a * yp[0] * np.exp(-1j * wt) + ((-1) ** (l + k) * np.conj(a) * ym[0] * np.exp(1j * wt) if m > 0 else 0.0)
    assert np.max(np.abs(got - want)) <= 1e-13


def test_p15_kerr_fold_equals_explicit_mirror_list_and_mpmath():
    """Eq. (9) with k: the folded sum equals the un-folded sum over a list that also holds (l, -m, -k, -n) with amplitude
    (-1)^{l+k} conj(A) and harmonic Y_{l,-m}; one sample recomputed with 40-digit mpmath from the extended coefficients."""
    mp = pytest.importorskip("mpmath")
    w, yp, ym, ca, cp = _kerr_small(seed=2)
    h = oracle.sum_waveform_kerr(w.t[0], ca, cp, w.l, w.m, w.k, w.n, None, yp, ym, w.t0, w.dt, w.n_samples)
    le, me, ke, ne, ypl, cols = [], [], [], [], [], []
    A = np.ascontiguousarray(w.amp[0])
    for j in range(w.n_modes):
        le.append(w.l[j]); me.append(w.m[j]); ke.append(w.k[j]); ne.append(w.n[j]); ypl.append(yp[j]); cols.append(A[:, j])
        if w.m[j] > 0:
            le.append(w.l[j]); me.append(-w.m[j]); ke.append(-w.k[j]); ne.append(-w.n[j]); ypl.append(ym[j])
            cols.append((-1) ** int(w.l[j] + w.k[j]) * np.conj(A[:, j]))
    ca2 = oracle.spline_fit(w.t[0], np.ascontiguousarray(np.stack(cols, axis=1)).view(np.float64))
    h2 = oracle.sum_waveform_kerr(w.t[0], ca2, cp, le, me, ke, ne, None, np.array(ypl), None, w.t0, w.dt, w.n_samples, fold=False)
    assert np.max(np.abs(h2 - h)) <= 1e-13 * np.max(np.abs(h))
    # mpmath at one sample
    mp.mp.dps = 40
    i = 137
    ti = w.t0 + i * w.dt
    seg = int(np.searchsorted(w.t[0], ti, side="right") - 1)
    dx = mp.mpf(float(ti - w.t[0][seg]))
    horner = lambda c: ((c[3] * dx + c[2]) * dx + c[1]) * dx + c[0]
    ld = lambda x: mp.mpf(float(x)) + mp.mpf(float(x - np.longdouble(float(x))))      # exact: 64-bit mantissa = two doubles
    P = [horner([ld(cp[seg, p, q]) for p in range(4)]) for q in range(3)]
    tot = mp.mpc(0)
    for j in range(w.n_modes):
        Ar = horner([mp.mpf(float(ca[seg, p, 2 * j])) for p in range(4)])
        Ai = horner([mp.mpf(float(ca[seg, p, 2 * j + 1])) for p in range(4)])
        th = int(w.m[j]) * P[0] + int(w.k[j]) * P[1] + int(w.n[j]) * P[2]
        W = mp.mpc(Ar, Ai) * mp.expj(-th)
        tot += mp.mpc(float(yp[j].real), float(yp[j].imag)) * W
        if w.m[j] > 0:
            tot += (-1) ** int(w.l[j] + w.k[j]) * mp.mpc(float(ym[j].real), float(ym[j].imag)) * mp.conj(W)
    assert abs(complex(tot) - h[i]) <= 1e-13 * np.max(np.abs(h))
