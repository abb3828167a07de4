"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

P1..P11 follow DESIGN.md "Oracle pins".  Each check is chosen so that a plausible mistake in oracle/few_oracle.c
(a dropped term, a wrong sign or index, a transposed operand) fails at least one of them.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2104_04582_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_facts.txt")


def paper_facts():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def eval_spline(t, coef, x):
    """Evaluate coef [n_seg, 4, n_sys] at points x -> [len(x), n_sys] (numpy, for the checks only)."""
    k = np.clip(np.searchsorted(t, x, side="right") - 1, 0, len(t) - 2)
    dx = (x - t[k])[:, None].astype(coef.dtype)
    c = coef[k]
    return c[:, 0] + dx * (c[:, 1] + dx * (c[:, 2] + dx * c[:, 3]))


GRIDS = {
    "uniform": np.linspace(0.0, 9.0, 10),
    "nonuniform": np.array([0.0, 0.4, 1.5, 1.7, 3.1, 4.9, 5.0, 7.3, 8.8, 9.0]),
    "shrinking": synth.sparse_grid(10.0, 25, uniform=False),
    "four": np.array([0.0, 1.0, 2.5, 3.0]),
}


# ---------------------------------------------------------------- P1: cubic reproduction (north_star: 1e-13)
@pytest.mark.parametrize("grid", list(GRIDS))
@pytest.mark.parametrize("fit", ["f64", "ext"])
def test_p1_notaknot_reproduces_cubics(grid, fit):
    t = GRIDS[grid]
    a = np.array([[0.3, -1.2, 0.7, 2.0], [-0.11, 0.5, -2.0, 0.25], [0.0, 0.0, 1.0, 0.0]]).T  # x^3, x^2, x, 1 per system
    y = np.stack([np.polyval(a[:, q], t) for q in range(a.shape[1])], axis=1)
    coef = (oracle.spline_fit if fit == "f64" else oracle.spline_fit_ext)(t, y)
    for q in range(a.shape[1]):
        p = np.poly1d(a[:, q])
        scale = np.max(np.abs(y[:, q])) + 1.0
        assert np.max(np.abs(coef[:, 1, q] - p.deriv(1)(t[:-1]))) <= 1e-13 * scale * len(t)
        assert np.max(np.abs(coef[:, 2, q] - p.deriv(2)(t[:-1]) / 2)) <= 1e-13 * scale * len(t)
        assert np.max(np.abs(coef[:, 3, q] - p.deriv(3)(t[:-1]) / 6)) <= 1e-12 * scale * len(t)
        xs = np.linspace(t[0], t[-1], 301)
        assert np.max(np.abs(eval_spline(t, coef, xs)[:, q] - p(xs))) <= 1e-13 * scale * len(t)


# ---------------------------------------------------------------- P2: independent formulation + invariants
def dense_notaknot_slopes(t, y):
    """Un-eliminated system: 3-term third-derivative-continuity rows at both ends, dense LU with pivoting."""
    n = len(t); h = np.diff(t); d = np.diff(y) / h
    A = np.zeros((n, n)); b = np.zeros(n)
    for i in range(1, n - 1):
        A[i, i - 1], A[i, i], A[i, i + 1] = h[i], 2 * (h[i - 1] + h[i]), h[i - 1]
        b[i] = 3 * (h[i] * d[i - 1] + h[i - 1] * d[i])
    # c3 on segment i = (s_i + s_{i+1} - 2 d_i)/h_i^2 ; continuity of c3 across t_1 and t_{n-2}
    A[0, 0], A[0, 1], A[0, 2] = 1 / h[0] ** 2, 1 / h[0] ** 2 - 1 / h[1] ** 2, -1 / h[1] ** 2
    b[0] = 2 * d[0] / h[0] ** 2 - 2 * d[1] / h[1] ** 2
    A[-1, -3], A[-1, -2], A[-1, -1] = 1 / h[-2] ** 2, 1 / h[-2] ** 2 - 1 / h[-1] ** 2, -1 / h[-1] ** 2
    b[-1] = 2 * d[-2] / h[-2] ** 2 - 2 * d[-1] / h[-1] ** 2
    return np.linalg.solve(A, b)


@pytest.mark.parametrize("grid", list(GRIDS))
def test_p2_dense_lu_and_continuity(grid):
    t = GRIDS[grid]
    rng = np.random.default_rng(5)
    y = rng.normal(size=(len(t), 4))
    coef = oracle.spline_fit(t, y)
    coef_e = oracle.spline_fit_ext(t, y)
    h = np.diff(t)
    assert np.array_equal(coef[:, 0, :], y[:-1])                      # c0 bit-copy
    for q in range(4):
        s = dense_notaknot_slopes(t, y[:, q])
        tol = 1e-12 * (np.max(np.abs(s)) + 1)
        assert np.max(np.abs(coef[:, 1, q] - s[:-1])) <= tol
        assert np.max(np.abs(np.asarray(coef_e[:, 1, q], float) - s[:-1])) <= tol
    c = coef_e.astype(np.float64)
    hh = h[:, None]
    end_val = c[:, 0] + hh * (c[:, 1] + hh * (c[:, 2] + hh * c[:, 3]))
    end_d1 = c[:, 1] + hh * (2 * c[:, 2] + 3 * hh * c[:, 3])
    end_d2 = 2 * c[:, 2] + 6 * hh * c[:, 3]
    sc = np.max(np.abs(y)) + 1
    assert np.max(np.abs(end_val[:-1] - c[1:, 0])) <= 1e-12 * sc                       # C0 at interior knots
    assert np.max(np.abs(end_val[-1] - y[-1])) <= 1e-12 * sc                            # interpolates last knot
    assert np.max(np.abs(end_d1[:-1] - c[1:, 1])) <= 1e-11 * sc / h.min()               # C1
    assert np.max(np.abs(end_d2[:-1] - 2 * c[1:, 2])) <= 1e-10 * sc / h.min() ** 2      # C2
    assert np.max(np.abs(c[0, 3] - c[1, 3])) <= 1e-10 * sc / h.min() ** 3               # not-a-knot at t_1
    assert np.max(np.abs(c[-1, 3] - c[-2, 3])) <= 1e-10 * sc / h.min() ** 3             # not-a-knot at t_{n-2}


# ---------------------------------------------------------------- P3: library special case
def test_p3_scipy_cubicspline():
    from scipy.interpolate import CubicSpline
    rng = np.random.default_rng(0)
    for n in (4, 5, 12, 100):
        t = np.sort(rng.uniform(0, 10, n)); t[0] = 0
        y = rng.normal(size=(n, 3))
        coef = oracle.spline_fit(t, y)
        cs = CubicSpline(t, y, bc_type="not-a-knot")
        for p in range(4):      # scipy c[3-p] multiplies dx^p
            ref = cs.c[3 - p]
            assert np.max(np.abs(coef[:, p, :] - ref)) <= 1e-11 * (np.max(np.abs(ref)) + 1), (n, p)


def test_spline_errors():
    with pytest.raises(ValueError):
        oracle.spline_fit(np.arange(3.0), np.zeros((3, 1)))
    with pytest.raises(ValueError):
        oracle.spline_fit(np.array([0.0, 1.0, 1.0, 2.0]), np.zeros((4, 1)))


# ---------------------------------------------------------------- P6: harmonics
def wigner_ylm(s, l, m, th, ph):
    """Independent formula: sY_lm = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi}, Wigner small-d by its
    explicit factorial sum (a different sum from the Goldberg form the oracle uses)."""
    f = math.factorial
    mp_, m_ = m, -s
    tot = 0.0
    for k in range(0, 2 * l + 1):
        a, b, c, d = l + m_ - k, k, mp_ - m_ + k, l - mp_ - k
        if min(a, b, c, d) < 0:
            continue
        tot += (-1) ** (mp_ - m_ + k) * math.cos(th / 2) ** (2 * l + m_ - mp_ - 2 * k) * math.sin(th / 2) ** (mp_ - m_ + 2 * k) \
            / (f(a) * f(b) * f(c) * f(d))
    dl = math.sqrt(f(l + mp_) * f(l - mp_) * f(l + m_) * f(l - m_)) * tot
    return (-1) ** s * math.sqrt((2 * l + 1) / (4 * math.pi)) * dl * np.exp(1j * m * ph)


def test_p6_ylm_closed_forms_l2():
    for th, ph in [(0.7, 1.1), (2.3, 4.0), (1e-3, 0.2), (math.pi - 1e-3, 5.0)]:
        c, s_ = math.cos(th), math.sin(th)
        cf = {2: math.sqrt(5 / (64 * math.pi)) * (1 + c) ** 2 * np.exp(2j * ph),
              1: math.sqrt(5 / (16 * math.pi)) * s_ * (1 + c) * np.exp(1j * ph),
              0: math.sqrt(15 / (32 * math.pi)) * s_ ** 2,
              -1: math.sqrt(5 / (16 * math.pi)) * s_ * (1 - c) * np.exp(-1j * ph),
              -2: math.sqrt(5 / (64 * math.pi)) * (1 - c) ** 2 * np.exp(-2j * ph)}
        for m, ref in cf.items():
            assert abs(oracle.ylm(2, m, th, ph) - ref) <= 1e-14, (th, ph, m)


def test_p6_ylm_wigner_cross_formula_and_symmetry():
    th, ph = 0.7, 1.1
    for l in range(2, 11):
        for m in range(-l, l + 1):
            y = oracle.ylm(l, m, th, ph)
            assert abs(y - wigner_ylm(-2, l, m, th, ph)) <= 1e-13, (l, m)
            # Y_{l,-m}(th, ph) = (-1)^l conj(Y_{l m}(pi - th, ph))   (s = -2)
            assert abs(oracle.ylm(l, -m, th, ph) - (-1) ** l * np.conj(oracle.ylm(l, m, math.pi - th, ph))) <= 1e-13
    with pytest.raises(ValueError):
        oracle.ylm(3, 4, th, ph)
    with pytest.raises(ValueError):
        oracle.ylm(1, 0, th, ph)


def test_p6_ylm_orthonormal_and_poles():
    x, w = np.polynomial.legendre.leggauss(40)
    ths = np.arccos(x); nph = 64; phs = 2 * math.pi * np.arange(nph) / nph
    modes = [(l, m) for l in range(2, 11) for m in range(-l, l + 1)]
    assert len(modes) == 117
    Y = np.array([[[oracle.ylm(l, m, t, p) for p in phs] for t in ths] for (l, m) in modes])
    G = np.einsum("atp,btp,t->ab", Y, Y.conj(), w) * (2 * math.pi / nph)
    assert np.max(np.abs(G - np.eye(len(modes)))) <= 1e-12
    for l in range(2, 11):
        for m in range(-l, l + 1):
            assert (abs(oracle.ylm(l, m, 0.0, 0.3)) > 1e-3) == (m == 2), (l, m)       # s=-2: only m=-s survives at theta=0
            assert (abs(oracle.ylm(l, m, math.pi, 0.3)) > 1e-3) == (m == -2), (l, m)


# ---------------------------------------------------------------- P11: index set (paper's numbers)
def test_p11_mode_grid_counts_match_paper():
    facts = paper_facts()
    l, m, n = synth.mode_grid()
    assert len(l) == facts["n_modes_schwarzschild"] == 3843
    assert l.min() == facts["l_min"] and l.max() == facts["l_max"] and np.abs(n).max() == facts["n_abs_max"]
    assert np.sum((l == 2) & (m == 2)) == facts["n_modes_22_family"] == 61
    assert np.sum(m == 0) == 549 and np.sum(m > 0) == 3294
    j = 61 * (l * (l + 1) // 2 - 3) + 61 * m + (n + 30)
    assert np.array_equal(j, np.arange(len(l)))
    assert np.all(m <= l) and np.all(m >= 0)


# ---------------------------------------------------------------- helpers for O4 pins
def fit_parts(w, s=0):
    yp, ym = oracle.ylm_modes(w.l, w.m, float(w.theta[s]), float(w.phi[s]))
    ca = oracle.spline_fit(w.t[s], np.ascontiguousarray(w.amp[s]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[s], w.phase[s])
    return yp, ym, ca, cp


def rel_l2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# ---------------------------------------------------------------- P4: closed form
@pytest.mark.parametrize("l,m,n,om_phi,om_r,tol", [(2, 2, 0, 3e-3, 2e-3, 1e-13), (3, 1, -2, 3e-3, 2e-3, 1e-13),
                                                  (5, 0, 4, 1e-3, 2.5e-3, 1e-13), (4, 3, 7, 20.0, 13.0, 1e-10)])
def test_p4_single_mode_closed_form(l, m, n, om_phi, om_r, tol):
    t = np.array([0.0, 700.0, 1500.0, 4000.0, 4100.0, 8000.0, 10000.0])
    a, chi, th, ph = 0.37, 0.9, 0.7, 1.1
    amp = np.full((len(t), 1), a * np.exp(1j * chi))
    phase = np.stack([om_phi * t, om_r * t], axis=1)
    yp = np.array([oracle.ylm(l, m, th, ph)]); ym = np.array([oracle.ylm(l, -m, th, ph)])
    ca = oracle.spline_fit(t, amp.view(np.float64)); cp = oracle.spline_fit_ext(t, phase)
    N, dt = 1000, 10.0
    h = oracle.sum_waveform(t, ca, cp, [l], [m], [n], None, yp, ym, 0.0, dt, N)
    ti = np.arange(N, dtype=np.longdouble) * dt
    om = np.longdouble(m) * np.longdouble(om_phi) + np.longdouble(n) * np.longdouble(om_r)
    e = (np.cos(om * ti) - 1j * np.sin(om * ti)).astype(np.complex128)
    ref = a * np.exp(1j * chi) * yp[0] * e
    if m > 0:
        ref = ref + (-1) ** l * a * np.exp(-1j * chi) * ym[0] * np.conj(e)
    assert rel_l2(h, ref) <= tol


# ---------------------------------------------------------------- P5: m -> -m symmetry, Eq. (9)
def test_p5_fold_equals_explicit_negative_m_sum():
    w = synth.random_problem(11, n_modes=14, n_samples=300)
    yp, ym, ca, cp = fit_parts(w)
    h_fold = oracle.sum_waveform(w.t[0], ca, cp, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, w.n_samples)
    # explicit list: every (l,m,n) plus, for m>0, (l,-m,-n) with amplitude (-1)^l conj(A) and harmonic Y_{l,-m}; no fold
    pos = w.m > 0
    l2 = np.concatenate([w.l, w.l[pos]]); m2 = np.concatenate([w.m, -w.m[pos]]); n2 = np.concatenate([w.n, -w.n[pos]])
    amp2 = np.concatenate([w.amp[0], ((-1.0) ** w.l[pos]) * np.conj(w.amp[0][:, pos])], axis=1)
    yp2 = np.concatenate([yp, ym[pos]])
    ca2 = oracle.spline_fit(w.t[0], np.ascontiguousarray(amp2).view(np.float64))
    h_exp = oracle.sum_waveform(w.t[0], ca2, cp, l2, m2, n2, None, yp2, None, w.t0, w.dt, w.n_samples, fold=False)
    assert rel_l2(h_fold, h_exp) <= 1e-13
    # and the fold really adds something (m>0 modes present)
    h_nofold = oracle.sum_waveform(w.t[0], ca, cp, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, w.n_samples, fold=False)
    assert rel_l2(h_nofold, h_fold) > 1e-3


# ---------------------------------------------------------------- P7: brute force with mpmath (config 0)
def test_p7_mpmath_bruteforce_config0():
    import mpmath as mp
    mp.mp.dps = 40
    w = synth.make_config(0)
    t = [mp.mpf(float(x)) for x in w.t[0]]
    nt = len(t)

    def mp_spline(y):
        """Dense solve of the 3-term not-a-knot system for the second-derivative-free (slope) form, in mpmath."""
        h = [t[i + 1] - t[i] for i in range(nt - 1)]; d = [(y[i + 1] - y[i]) / h[i] for i in range(nt - 1)]
        A = mp.zeros(nt, nt); b = mp.zeros(nt, 1)
        for i in range(1, nt - 1):
            A[i, i - 1], A[i, i], A[i, i + 1] = h[i], 2 * (h[i - 1] + h[i]), h[i - 1]
            b[i] = 3 * (h[i] * d[i - 1] + h[i - 1] * d[i])
        A[0, 0], A[0, 1], A[0, 2] = 1 / h[0] ** 2, 1 / h[0] ** 2 - 1 / h[1] ** 2, -1 / h[1] ** 2
        b[0] = 2 * d[0] / h[0] ** 2 - 2 * d[1] / h[1] ** 2
        A[nt - 1, nt - 3], A[nt - 1, nt - 2], A[nt - 1, nt - 1] = 1 / h[-2] ** 2, 1 / h[-2] ** 2 - 1 / h[-1] ** 2, -1 / h[-1] ** 2
        b[nt - 1] = 2 * d[-2] / h[-2] ** 2 - 2 * d[-1] / h[-1] ** 2
        s = mp.lu_solve(A, b)
        return [(y[i], s[i], (3 * d[i] - 2 * s[i] - s[i + 1]) / h[i], (s[i] + s[i + 1] - 2 * d[i]) / h[i] ** 2) for i in range(nt - 1)]

    def mp_ylm(l, m, th, ph):   # Wigner-d form in mpmath, s = -2
        s = -2; mp_, m_ = m, -s; tot = mp.mpf(0)
        for k in range(0, 2 * l + 1):
            a, b, c, d = l + m_ - k, k, mp_ - m_ + k, l - mp_ - k
            if min(a, b, c, d) < 0: continue
            tot += (-1) ** (mp_ - m_ + k) * mp.cos(th / 2) ** (2 * l + m_ - mp_ - 2 * k) * mp.sin(th / 2) ** (mp_ - m_ + 2 * k) \
                / (mp.factorial(a) * mp.factorial(b) * mp.factorial(c) * mp.factorial(d))
        dl = mp.sqrt(mp.factorial(l + mp_) * mp.factorial(l - mp_) * mp.factorial(l + m_) * mp.factorial(l - m_)) * tot
        return mp.sqrt((2 * l + 1) / (4 * mp.pi)) * dl * mp.expj(m * ph)

    th, ph = mp.mpf(float(w.theta[0])), mp.mpf(float(w.phi[0]))
    sp_phi = mp_spline([mp.mpf(float(x)) for x in w.phase[0, :, 0]])
    sp_r = mp_spline([mp.mpf(float(x)) for x in w.phase[0, :, 1]])
    sp_re = [mp_spline([mp.mpf(float(x)) for x in w.amp[0, :, j].real]) for j in range(w.n_modes)]
    sp_im = [mp_spline([mp.mpf(float(x)) for x in w.amp[0, :, j].imag]) for j in range(w.n_modes)]
    Yp = [mp_ylm(int(l), int(m), th, ph) for l, m in zip(w.l, w.m)]
    Ym = [mp_ylm(int(l), -int(m), th, ph) for l, m in zip(w.l, w.m)]
    idx = list(range(0, w.n_samples, 37)) + [1, w.n_samples - 1]

    def ev(c, dx): return c[0] + dx * (c[1] + dx * (c[2] + dx * c[3]))

    ref = []
    for i in idx:
        ti = mp.mpf(float(w.t0)) + i * mp.mpf(float(w.dt))
        k = max(kk for kk in range(nt - 1) if t[kk] <= ti)
        dx = ti - t[k]
        P, R = ev(sp_phi[k], dx), ev(sp_r[k], dx)
        hsum = mp.mpc(0)
        for j in range(w.n_modes):
            A = mp.mpc(ev(sp_re[j][k], dx), ev(sp_im[j][k], dx))
            W = A * mp.expj(-(int(w.m[j]) * P + int(w.n[j]) * R))
            hsum += Yp[j] * W
            if w.m[j] > 0:
                hsum += (-1) ** int(w.l[j]) * Ym[j] * mp.conj(W)
        ref.append(complex(hsum))
    ref = np.array(ref)
    h = oracle.waveform(w)[0]
    assert rel_l2(h[idx], ref) <= 1e-13


def test_p7_large_phase_sampled_against_mpmath():
    """Config-3-like phases (~1e6 rad) and high (m, n): the extended-precision phase path against 40-digit mpmath
    evaluation of the SAME extended-precision spline coefficients (pins the Horner + argument reduction, R13/R15)."""
    import mpmath as mp
    mp.mp.dps = 40
    w = synth.make_config(1, n_samples=64)
    t = w.t[0]
    phase = w.phase[0] * 6.0                # ~1.3e6 rad at the end
    cp = oracle.spline_fit_ext(t, phase)
    l, m, n = np.array([10], np.int32), np.array([10], np.int32), np.array([30], np.int32)
    amp = np.ones((len(t), 1), np.complex128)
    ca = oracle.spline_fit(t, amp.view(np.float64))
    yp = np.array([1.0 + 0j]); ym = np.array([0j])
    i0 = 3_100_000
    h = oracle.sum_waveform(t, ca, cp, l, m, n, None, yp, ym, 0.0, 10.0, 64, i0=i0, fold=False)
    ref = []
    for i in range(64):
        ti = (i0 + i) * 10.0
        k = int(np.searchsorted(t, ti, side="right") - 1)
        dx = mp.mpf(ti) - mp.mpf(float(t[k]))
        c = [[mp.mpf(float(cp[k, p, q])) + mp.mpf(float(cp[k, p, q] - np.longdouble(float(cp[k, p, q])))) for q in range(2)] for p in range(4)]
        P = c[0][0] + dx * (c[1][0] + dx * (c[2][0] + dx * c[3][0]))
        R = c[0][1] + dx * (c[1][1] + dx * (c[2][1] + dx * c[3][1]))
        ref.append(complex(mp.expj(-(10 * P + 30 * R))))
    assert np.max(np.abs(h - np.array(ref))) <= 2e-11     # 4e7 rad * 2^-64 ~ 2e-12 per op, a few ops


# ---------------------------------------------------------------- P8: selection
def brute_select(P, owner, eps, n_modes):
    """Definition by enumeration in exact rational arithmetic: per step, the shortest descending-power prefix
    whose dropped power is <= eps * total (ties -> lower entry index first); union of owners over steps."""
    keep = set()
    epsq = Fraction(eps)
    for row in P:
        order = sorted(range(len(row)), key=lambda e: (-row[e], e))
        fr = [Fraction(float(row[e])) for e in order]
        total = sum(fr)
        for L in range(1, len(order) + 1):
            if total - sum(fr[:L]) <= epsq * total:
                break
        keep |= {owner[e] for e in order[:L]}
    return np.array(sorted(keep), np.int32)


@pytest.mark.parametrize("seed", range(6))
def test_p8_selection_bruteforce_tiny(seed):
    rng = np.random.default_rng(seed)
    nm, nt = 7, 3
    m = rng.integers(0, 3, nm).astype(np.int32)
    amp = (rng.normal(size=(nt, nm)) + 1j * rng.normal(size=(nt, nm))) * 10.0 ** rng.uniform(-3, 0, (nt, nm))
    yp = rng.normal(size=nm) + 1j * rng.normal(size=nm); ym = rng.normal(size=nm) + 1j * rng.normal(size=nm)
    owner = list(range(nm)) + [j for j in range(nm) if m[j] > 0]
    P = np.concatenate([np.abs(amp) ** 2 * np.abs(yp) ** 2, (np.abs(amp) ** 2 * np.abs(ym) ** 2)[:, m > 0]], axis=1)
    for eps in (0.5, 1e-1, 1e-2, 1e-4, 1e-9):
        got, _ = oracle.select_modes(amp, m, yp, ym, eps)
        assert np.array_equal(got, brute_select(P, owner, eps, nm)), eps
        got2, _ = oracle.select_modes(amp, m, None, None, eps)          # bare |A|^2 variant, primaries only
        assert np.array_equal(got2, brute_select(np.abs(amp) ** 2, list(range(nm)), eps, nm)), eps


def test_p8_selection_invariants():
    w = synth.make_config(1, n_samples=16)
    yp, ym = oracle.ylm_modes(w.l, w.m, 0.7, 1.1)
    amp = w.amp[0][::9]                                   # 12 of the 100 steps keeps the test fast
    prev = None
    counts = []
    for eps in (1e-1, 1e-2, 1e-3, 1e-5):
        k, margin = oracle.select_modes(amp, w.m, yp, ym, eps)
        assert np.all(np.diff(k) > 0)
        if prev is not None:
            assert set(prev) <= set(k)                    # kept set grows as eps falls
        prev = k; counts.append(len(k))
        k2, _ = oracle.select_modes(3.7 * amp, w.m, yp, ym, eps)   # invariant under A -> cA
        assert np.array_equal(k, k2)
        # dropped power per step <= eps * total (extended precision)
        P = np.concatenate([np.abs(amp) ** 2 * np.abs(yp) ** 2, (np.abs(amp) ** 2 * np.abs(ym) ** 2)[:, w.m > 0]], axis=1).astype(np.longdouble)
        owner = np.concatenate([np.arange(w.n_modes), np.arange(w.n_modes)[w.m > 0]])
        kept_e = np.isin(owner, k)
        assert np.all(P[:, ~kept_e].sum(1) <= eps * P.sum(1) * (1 + 1e-12))
    assert counts == sorted(counts) and counts[0] < counts[-1]
    k_all, _ = oracle.select_modes(amp, w.m, yp, ym, 0.0)
    assert np.array_equal(k_all, np.arange(w.n_modes))    # eps <= 0 keeps everything (R6)
    k_one, _ = oracle.select_modes(amp, w.m, yp, ym, 1.0)  # eps >= 1: the per-step arg-max only
    P = np.concatenate([np.abs(amp) ** 2 * np.abs(yp) ** 2, (np.abs(amp) ** 2 * np.abs(ym) ** 2)[:, w.m > 0]], axis=1)
    owner = np.concatenate([np.arange(w.n_modes), np.arange(w.n_modes)[w.m > 0]])
    assert set(k_one) == set(owner[np.argmax(P, axis=1)])
    # relabelling modes permutes the result
    perm = np.random.default_rng(1).permutation(w.n_modes)
    k, _ = oracle.select_modes(amp, w.m, yp, ym, 1e-3)
    kp, _ = oracle.select_modes(amp[:, perm], w.m[perm], yp[perm], ym[perm], 1e-3)
    assert set(perm[kp]) == set(k)


def test_p8_ties_broken_by_entry_index():
    amp = np.ones((2, 5), np.complex128)                  # all powers equal
    m = np.zeros(5, np.int32)
    k, _ = oracle.select_modes(amp, m, None, None, 0.45)  # need > 55% of the power: 3 of 5 entries, the lowest indices
    assert list(k) == [0, 1, 2]


def brute_margin(P, owner, eps, n_modes):
    """The oracle's `margin` output by its definition, in exact rational arithmetic: for every mode the minimum, over the
    steps and over the mode's entries of rank r >= 1, of |C_{r-1} - (1 - eps) total| / total (C = inclusive cumulative sum in
    descending-power order, ties by entry index).  inf for a mode that is rank 0 in every step, and for eps <= 0."""
    out = [math.inf] * n_modes
    if eps <= 0:
        return out
    one_minus = 1 - Fraction(eps)
    for row in P:
        order = sorted(range(len(row)), key=lambda e: (-row[e], e))
        fr = [Fraction(float(row[e])) for e in order]
        total = sum(fr)
        c = Fraction(0)
        for r, e in enumerate(order):
            if r >= 1 and total > 0:
                d = abs(c - one_minus * total) / total
                out[owner[e]] = min(out[owner[e]], float(d))
            c += fr[r]
    return out


@pytest.mark.parametrize("seed", range(6))
def test_p8_margin_is_the_distance_to_the_threshold(seed):
    """`margin[j]` is what the GPU set-parity tests lean on (a kept-set difference is excused only inside the 1e-12 band), so it
    is pinned like the set itself: exact rationals on tiny rows, both power variants, five eps, plus eps <= 0 and a mode
    that is the strongest entry of every step (no rank >= 1 entry: inf)."""
    rng = np.random.default_rng(50 + seed)
    nm, nt = 7, 3
    m = rng.integers(0, 3, nm).astype(np.int32)
    amp = (rng.normal(size=(nt, nm)) + 1j * rng.normal(size=(nt, nm))) * 10.0 ** rng.uniform(-3, 0, (nt, nm))
    amp[:, 2] = 50.0                                        # mode 2 is rank 0 in every step ...
    m[2] = 0                                                # ... and has no mirror entry
    yp = rng.normal(size=nm) + 1j * rng.normal(size=nm); ym = rng.normal(size=nm) + 1j * rng.normal(size=nm)
    yp[2] = 1.0
    owner = list(range(nm)) + [j for j in range(nm) if m[j] > 0]
    P = np.concatenate([np.abs(amp) ** 2 * np.abs(yp) ** 2, (np.abs(amp) ** 2 * np.abs(ym) ** 2)[:, m > 0]], axis=1)
    for eps in (0.5, 1e-1, 1e-2, 1e-4, 1e-9):
        _, margin = oracle.select_modes(amp, m, yp, ym, eps)
        want = brute_margin(P, owner, eps, nm)
        assert margin[2] == math.inf and want[2] == math.inf
        for j in range(nm):
            if j != 2:
                assert abs(margin[j] - want[j]) <= 1e-15, (eps, j, margin[j], want[j])
        _, margin0 = oracle.select_modes(amp, m, None, None, eps)
        want0 = brute_margin(np.abs(amp) ** 2, list(range(nm)), eps, nm)
        assert all(abs(a - b) <= 1e-15 for a, b in zip(np.delete(margin0, 2), np.delete(want0, 2)))
    _, margin = oracle.select_modes(amp, m, yp, ym, 0.0)
    assert np.all(np.isinf(margin))


def test_p8_margin_of_a_constructed_threshold_hit():
    """A row built so that C_{r-1} equals (1 - eps) total up to rounding: the margin of the rank-r mode is ~1e-17, far
    inside the 1e-12 band, and every other mode is far outside it (the case the GPU band test is built on)."""
    p = np.array([0.5, 0.25, 0.125, 0.0625, 0.03125, 0.03125])            # total = 1 exactly; C = .5 .75 .875 .9375 ...
    amp = np.sqrt(p)[None, :].astype(np.complex128)
    m = np.zeros(6, np.int32)
    eps = 0.125                                                           # (1 - eps) total = 0.875 = C_2 exactly
    keep, margin = oracle.select_modes(amp, m, None, None, eps)
    want = brute_margin(np.abs(amp) ** 2, list(range(6)), eps, 6)
    assert abs(margin[3] - want[3]) <= 1e-15 and margin[3] <= 1e-15       # rank 3 sees C_2 = threshold
    assert list(keep) == [0, 1, 2] or list(keep) == [0, 1, 2, 3]          # C_2 < 0.875 decided by rounding of |a|^2
    assert all(margin[j] > 1e-3 for j in (1, 2, 4, 5))


def test_p8_mismatch_scales_like_eps_paper_fig3():
    """PAPER.md:300 (Fig. 3): mismatch ~1e-2 at eps=1e-1 falling as a power law.  On the synthetic model the
    kept-vs-all-modes mismatch must fall roughly linearly with eps (order-of-magnitude pin of O3 + O4 together)."""
    w = synth.make_config(1, n_samples=16)
    yp, ym, ca, cp = fit_parts(w)
    wins = [(i0, 40) for i0 in range(1000, 3_100_000, 100_000)]

    def wave(keep):
        return np.concatenate([oracle.sum_waveform(w.t[0], ca, cp, w.l, w.m, w.n, keep, yp, ym, 0.0, 10.0, nn, i0=i0) for i0, nn in wins])

    h_all = wave(None)
    mm = []
    for eps in (1e-1, 1e-2, 1e-3):
        k, _ = oracle.select_modes(w.amp[0], w.m, yp, ym, eps)
        h = wave(k)
        ov = np.real(np.vdot(h_all, h)) / math.sqrt(np.vdot(h, h).real * np.vdot(h_all, h_all).real)
        mm.append(1 - ov)
    facts = paper_facts()
    assert facts["eps_mismatch_at_1e-1"] / 30 < mm[0] < facts["eps_mismatch_at_1e-1"] * 30
    assert mm[0] > 3 * mm[1] > 9 * mm[2] > 0


# ---------------------------------------------------------------- P9 / P10
def test_p9_real_linearity():
    w = synth.random_problem(21, n_modes=9, n_samples=200)
    w2 = synth.random_problem(22, n_modes=9, n_samples=200)
    yp, ym, ca, cp = fit_parts(w)
    amp2 = w2.amp[0][:, : w.n_modes] if w2.n_modes >= w.n_modes else None
    assert amp2 is not None
    t = w.t[0]
    ca2 = oracle.spline_fit(t, np.ascontiguousarray(amp2).view(np.float64))
    al, be = 0.83, -1.7
    ca3 = oracle.spline_fit(t, np.ascontiguousarray(al * w.amp[0] + be * amp2).view(np.float64))
    f = lambda c: oracle.sum_waveform(t, c, cp, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, w.n_samples)
    assert rel_l2(f(ca3), al * f(ca) + be * f(ca2)) <= 1e-13


def test_p10_time_translation_and_batch_independence():
    w = synth.random_problem(31, n_src=3, n_modes=8, n_samples=150)
    h = oracle.waveform(w)
    assert h.shape == (3, 150)
    for s in range(3):
        ws = synth.Workload(w.name, w.t[s:s + 1], w.phase[s:s + 1], w.amp[s:s + 1], w.l, w.m, w.n, w.theta[s:s + 1],
                            w.phi[s:s + 1], w.t0, w.dt, w.n_samples, w.eps)
        assert np.array_equal(oracle.waveform(ws)[0], h[s])
    # power-of-two shift of every t_k and of t0 (dt a power of two so every t_i shifts exactly)
    wq = synth.random_problem(32, n_modes=8, n_samples=128, T=1024.0)
    tq = np.round(wq.t * 64) / 64
    yp, ym = oracle.ylm_modes(wq.l, wq.m, float(wq.theta[0]), float(wq.phi[0]))

    def run(shift):
        t = tq[0] + shift
        ca = oracle.spline_fit(t, np.ascontiguousarray(wq.amp[0]).view(np.float64))
        cp = oracle.spline_fit_ext(t, wq.phase[0])
        return oracle.sum_waveform(t, ca, cp, wq.l, wq.m, wq.n, None, yp, ym, shift, 8.0, 128)

    assert np.max(np.abs(run(0.0) - run(4096.0))) <= 1e-15 * np.max(np.abs(run(0.0)))


def test_o4_outside_range_and_knot_samples():
    w = synth.random_problem(41, n_modes=5, n_samples=64, T=640.0)
    yp, ym, ca, cp = fit_parts(w)
    t = w.t[0]
    h = oracle.sum_waveform(t, ca, cp, w.l, w.m, w.n, None, yp, ym, -50.0, 10.0, 80)
    ti = -50.0 + 10.0 * np.arange(80)
    assert np.all(h[ti < 0] == 0) and np.all(h[ti > 640.0] == 0) and np.all(h[(ti >= 0) & (ti <= 640)] != 0)   # R12
    # a sample exactly on the last knot uses the last segment; on an interior knot it equals the knot values
    hk = oracle.sum_waveform(t, ca, cp, w.l, w.m, w.n, None, yp, ym, float(t[3]), 1.0, 1)
    A = w.amp[0][3]; th = w.m * w.phase[0][3, 0] + w.n * w.phase[0][3, 1]
    W = A * np.exp(-1j * th)
    ref = np.sum(yp * W + np.where(w.m > 0, (-1.0) ** w.l * ym * np.conj(W), 0))
    assert abs(hk[0] - ref) <= 1e-13 * abs(ref)
    hl = oracle.sum_waveform(t, ca, cp, w.l, w.m, w.n, None, yp, ym, float(t[-1]), 1.0, 1)
    A = w.amp[0][-1]; th = w.m * w.phase[0][-1, 0] + w.n * w.phase[0][-1, 1]
    W = A * np.exp(-1j * th)
    ref = np.sum(yp * W + np.where(w.m > 0, (-1.0) ** w.l * ym * np.conj(W), 0))
    assert abs(hl[0] - ref) <= 1e-12 * abs(ref)


_SAN_WORKER = r"""
import sys
sys.path.insert(0, sys.argv[1])
import numpy as np
import oracle
oracle._SO = sys.argv[2]            # the sanitised build; oracle.build() finds it up to date and loads it
from paper_2104_04582_b200 import synth
oracle.set_threads(2)
w0 = synth.make_config(0)
h0 = oracle.waveform(w0)
assert np.all(np.isfinite(h0.view(np.float64)))
w1 = synth.make_config(1, n_samples=1500, t0=12_000_000.0)       # 3843 modes, selection at eps = 1e-5, 100 knots
h1, parts = oracle.waveform(w1, return_parts=True)
assert np.all(np.isfinite(h1.view(np.float64)))
yp, ym = oracle.ylm_modes(w1.l, w1.m, float(w1.theta[0]), float(w1.phi[0]))
for eps in (1e-2, 0.0, 1.0):
    keep, margin = oracle.select_modes(w1.amp[0], w1.m, yp, ym, eps)
    assert len(keep) >= 1
wk = synth.make_kerr(n_samples=200, n_t=12, l_max=3, k_max=2, n_max=2, t0=2_000_000.0)
ca = oracle.spline_fit(wk.t[0], np.ascontiguousarray(wk.amp[0]).view(np.float64))
cp = oracle.spline_fit_ext(wk.t[0], wk.phase[0])
ypk, ymk = oracle.ylm_modes(wk.l, wk.m, 0.8, 1.3)
hk = oracle.sum_waveform_kerr(wk.t[0], ca, cp, wk.l, wk.m, wk.k, wk.n, None, ypk, ymk, wk.t0, wk.dt, wk.n_samples)
assert np.all(np.isfinite(hk.view(np.float64)))
d = np.ones(64, np.complex128)
oracle.inner(d, d, 10.0); oracle.frame(0.3, 1.0, 1.2, 2.0)
print("sanitised oracle ok")
"""


def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the oracle built with -fsanitize=address,undefined and run on config 0, a config-1 slice with
    selection, the selection alone at three thresholds and a Kerr-shaped slice.  Any out-of-bounds access, use after free,
    signed overflow or misaligned access aborts the worker (halt_on_error, -fno-sanitize-recover)."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    so = str(tmp_path / "libfew_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-fopenmp", "-ffp-contract=off", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                           "-fno-omit-frame-pointer", "-shared", "-fPIC", "-std=c11", os.path.join(root, "oracle", "few_oracle.c"),
                           "-o", so, "-lm"])
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan.so not found next to gcc")
    script = tmp_path / "san_worker.py"
    script.write_text(_SAN_WORKER)
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    p = subprocess.run([sys.executable, str(script), root, so], capture_output=True, text=True, env=env, timeout=600)
    assert p.returncode == 0 and "sanitised oracle ok" in p.stdout, p.stdout[-2000:] + p.stderr[-4000:]
    assert "runtime error" not in p.stderr and "AddressSanitizer" not in p.stderr, p.stderr[-4000:]
