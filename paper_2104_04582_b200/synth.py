"""Seeded synthetic workloads shaped like the paper's (BASELINE.json `configs`).

This module serves BOTH the CUDA path and the CPU oracle (tests, bench).  It holds none of the
method's arithmetic: no spline, no Ylm, no selection, no summation.  It only draws the *inputs* of
the hot path -- the sparse trajectory times t_k, the phases Phi_phi(t_k), Phi_r(t_k) and the complex
mode amplitudes A_lmn(t_k) that the paper's trajectory and amplitude modules would hand over
("~100 time steps"; "two-dimensional array of individual complex mode
amplitudes"; PAPER.md:225 l in [2,10], m in [0,l], n in [-30,30] -> 3843 modes).

numpy only; imports neither the CUDA binding nor `oracle/`.
"""
from __future__ import annotations

import dataclasses
import numpy as np

MSUN_S = 4.925491025543576e-6  # G Msun / c^3 in seconds (BASELINE.json config 0 quotes M_s = 4.925 s at 1e6 Msun)
YEAR_S = 31_557_600.0          # Julian year; 3 155 760 samples at dt = 10 s (BASELINE.json config 1)
SEED_BASE = 2104045820
N_MIN, N_MAX, L_MIN, L_MAX = -30, 30, 2, 10


def mode_grid(l_max: int = L_MAX, n_max: int = N_MAX):
    """(l, m, n) int32 arrays of the Schwarzschild mode index set, m >= 0 only.

    Order: l slowest, then m, n fastest: j = 61*(l(l+1)/2 - 3) + 61*m + (n + 30) for the full grid.
    """
    ls, ms, ns = [], [], []
    for l in range(L_MIN, l_max + 1):
        for m in range(0, l + 1):
            for n in range(-n_max, n_max + 1):
                ls.append(l), ms.append(m), ns.append(n)
    return (np.asarray(ls, np.int32), np.asarray(ms, np.int32), np.asarray(ns, np.int32))


@dataclasses.dataclass
class Workload:
    """One batch of hot-path inputs.  Shapes: t [n_src, n_t]; phase [n_src, n_t, 2] (Phi_phi, Phi_r);
    amp [n_src, n_t, n_modes] complex128; l, m, n [n_modes] int32 (shared by the sources);
    theta, phi [n_src]; t0, dt, n_samples: dense output grid t_i = t0 + i*dt; eps: selection threshold
    (<= 0: keep all modes)."""
    name: str
    t: np.ndarray
    phase: np.ndarray
    amp: np.ndarray
    l: np.ndarray
    m: np.ndarray
    n: np.ndarray
    theta: np.ndarray
    phi: np.ndarray
    t0: float
    dt: float
    n_samples: int
    eps: float
    k: np.ndarray | None = None     # polar index per mode (Kerr-shaped workloads: phase then has 3 columns, Phi_phi, Phi_theta, Phi_r)
    n_t_src: np.ndarray | None = None   # ragged batches: knots per source, int32 [n_src]; rows beyond a source's count are padding (NaN)

    @property
    def n_src(self): return self.t.shape[0]
    @property
    def n_t(self): return self.t.shape[1]
    @property
    def n_modes(self): return self.l.shape[0]


def sparse_grid(T: float, n_t: int, uniform: bool) -> np.ndarray:
    """Sparse trajectory times.  Config 0 is uniform; configs 1-4 shrink the step linearly towards the
    end, t_k = T (1 - (1 - k/(n_t-1))^2), like an adaptive integrator approaching the separatrix
    (reading R17)."""
    x = np.arange(n_t, dtype=np.float64) / (n_t - 1)
    t = T * x if uniform else T * (1.0 - (1.0 - x) ** 2)
    t[0], t[-1] = 0.0, T
    return t


def _phases(t: np.ndarray, T: float, p0: float, p1: float, M_msun: float, sub: int = 256) -> np.ndarray:
    """Phi_phi, Phi_r at the sparse times by composite Simpson (= RK4, the rates depend on t only) with
    `sub` sub-steps per sparse interval; p(t) linear in t; Omega_phi = p^-1.5 / M_s,
    Omega_r = Omega_phi sqrt(1 - 6/p) (BASELINE.json config 0)."""
    Ms = M_msun * MSUN_S

    def omegas(tt):
        p = p0 + (p1 - p0) * (tt / T)
        of = p ** -1.5 / Ms
        return of, of * np.sqrt(1.0 - 6.0 / p)

    out = np.zeros((t.shape[0], 2))
    acc = np.zeros(2, dtype=np.longdouble)
    for k in range(t.shape[0] - 1):
        a, b = t[k], t[k + 1]
        h = (b - a) / sub
        x = a + h * np.arange(sub + 1)
        xm = x[:-1] + 0.5 * h
        fa, ra = omegas(x)
        fm, rm = omegas(xm)
        sf = (h / 6.0) * (fa[:-1] + 4.0 * fm + fa[1:])
        sr = (h / 6.0) * (ra[:-1] + 4.0 * rm + ra[1:])
        acc[0] += np.sum(sf.astype(np.longdouble))
        acc[1] += np.sum(sr.astype(np.longdouble))
        out[k + 1, 0], out[k + 1, 1] = float(acc[0]), float(acc[1])
    return out


def _amplitudes(rng, t, T, e_t, l, n, cfg0: bool) -> np.ndarray:
    """A_j(t_k) = |A|_j(t_k) (1 + 0.3 sin(2 pi f_j t_k / T + psi_j)) exp(i chi_j) (BASELINE.json configs 0, 1)."""
    nm = l.shape[0]
    if cfg0:
        base = 10.0 ** rng.uniform(-3.0, 0.0, nm)            # a ~ LogUniform(1e-3, 1)
    else:
        base = rng.lognormal(0.0, 0.5, nm)                   # LN_j
    f = rng.uniform(0.5, 2.0, nm)
    psi = rng.uniform(0.0, 2.0 * np.pi, nm)
    chi = rng.uniform(0.0, 2.0 * np.pi, nm)
    if cfg0:
        mag = np.broadcast_to(base, (t.shape[0], nm))
    else:
        n0 = np.rint(4.0 * e_t)[:, None]                     # round-half-even (reading R19)
        w = (3.0 + 10.0 * e_t)[:, None]
        mag = 10.0 ** (-(l[None, :].astype(np.float64) - 2.0)) * np.exp(-np.abs(n[None, :] - n0) / w) * base[None, :]
    mod = 1.0 + 0.3 * np.sin(2.0 * np.pi * f[None, :] * (t[:, None] / T) + psi[None, :])
    return (mag * mod) * np.exp(1j * chi)[None, :]


CFG0_MODES = [(2, 0, 0), (2, 1, 0), (2, 2, 0), (3, 0, 0), (3, 1, 0), (3, 2, 0), (3, 3, 0), (4, 4, 0)]  # DESIGN.md reading R16


def _one_source(rng, *, T, n_t, uniform, p0, p1, e0, e1, M, l, n, cfg0=False):
    t = sparse_grid(T, n_t, uniform)
    e_t = e0 + (e1 - e0) * (t / T)
    phase = _phases(t, T, p0, p1, M)
    amp = _amplitudes(rng, t, T, e_t, l, n, cfg0)
    return t, phase, amp


def make_config(config: int, *, n_samples: int | None = None, n_src: int | None = None,
                t0: float | None = None, eps: float | None = None) -> Workload:
    """Build BASELINE.json config 0..4.  `n_samples`, `n_src`, `t0`, `eps` override the config's values so
    tests can run the same trajectory on a short window (the sparse inputs never change with them)."""
    if config == 0:
        l, m, n = (np.asarray(x, np.int32) for x in zip(*CFG0_MODES))
        rng = np.random.Generator(np.random.PCG64(SEED_BASE + 0))
        t, ph, a = _one_source(rng, T=40960.0, n_t=20, uniform=True, p0=12.0, p1=10.0, e0=0.4, e1=0.35,
                               M=1e6, l=l, n=n, cfg0=True)
        w = Workload("config0_tiny", t[None], ph[None], a[None], l, m, n, np.array([0.7]), np.array([1.1]),
                     0.0, 10.0, 4096, 0.0)
    elif config in (1, 2):
        l, m, n = mode_grid()
        rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1))   # config 2 = config 1 inputs, eps = 0
        t, ph, a = _one_source(rng, T=YEAR_S, n_t=100, uniform=False, p0=14.0, p1=6.0 + 2 * 0.1 + 0.1,
                               e0=0.5, e1=0.1, M=1e6, l=l, n=n)
        w = Workload("config1_1yr_eps1e-5" if config == 1 else "config2_1yr_allmodes", t[None], ph[None], a[None],
                     l, m, n, np.array([0.7]), np.array([1.1]), 0.0, 10.0, 3_155_760, 1e-5 if config == 1 else 0.0)
    elif config == 3:
        l, m, n = mode_grid()
        ns = 64 if n_src is None else n_src
        ts, phs, amps, th, ph_ = [], [], [], [], []
        for s in range(ns):
            rng = np.random.Generator(np.random.PCG64(SEED_BASE + 3 + 1000 + s))
            p0 = rng.uniform(10.0, 16.0); e0 = rng.uniform(0.1, 0.6); M = 10.0 ** rng.uniform(5.0, 7.0)
            theta = rng.uniform(0.0, np.pi); phi = rng.uniform(0.0, 2.0 * np.pi)
            e1 = 0.5 * e0
            t, p, a = _one_source(rng, T=0.5 * YEAR_S, n_t=80, uniform=False, p0=p0, p1=6.0 + 2 * e1 + 0.1,
                                  e0=e0, e1=e1, M=M, l=l, n=n)
            ts.append(t), phs.append(p), amps.append(a), th.append(theta), ph_.append(phi)
        w = Workload("config3_batch64_halfyr", np.stack(ts), np.stack(phs), np.stack(amps), l, m, n,
                     np.asarray(th), np.asarray(ph_), 0.0, 15.0, 1_051_920, 1e-5)
    elif config == 4:
        l, m, n = mode_grid()
        rng = np.random.Generator(np.random.PCG64(SEED_BASE + 4))
        t, ph, a = _one_source(rng, T=4 * YEAR_S, n_t=300, uniform=False, p0=16.0, p1=6.0 + 2 * 0.05 + 0.1,
                               e0=0.7, e1=0.05, M=1e6, l=l, n=n)
        w = Workload("config4_4yr_sweep", t[None], ph[None], a[None], l, m, n, np.array([0.7]), np.array([1.1]),
                     0.0, 10.0, 12_623_040, 1e-5)
    else:
        raise ValueError(f"unknown config {config}")
    if n_samples is not None: w.n_samples = int(n_samples)
    if t0 is not None: w.t0 = float(t0)
    if eps is not None: w.eps = float(eps)
    return w


def make_ragged(counts=(40, 80, 137, 80, 40, 137), *, n_samples: int = 40_000, dt: float = 15.0, eps: float = 1e-5,
                seed: int = 0) -> Workload:
    """A ragged batch: sources drawn like config 3's (parameters uniform in the same ranges) but each with its own number of
    trajectory points and its own end time, as an adaptive integrator that stops at the separatrix hands them over
    ("~100" points).  Arrays are padded to the largest count; the padding is NaN so that any
    read of it shows up in the output.  Source s ends at T_s in [0.45, 1.05] x n_samples x dt: some end inside the output window
    (h = 0 from there on), some after it."""
    l, m, n = mode_grid()
    counts = np.asarray(counts, np.int32)
    n_src, n_max = len(counts), int(counts.max())
    t = np.full((n_src, n_max), np.nan)
    phase = np.full((n_src, n_max, 2), np.nan)
    amp = np.full((n_src, n_max, len(l)), np.nan + 1j * np.nan, dtype=np.complex128)
    th, ph_ = np.empty(n_src), np.empty(n_src)
    for s in range(n_src):
        rng = np.random.Generator(np.random.PCG64(SEED_BASE + 7000 + 100 * seed + s))
        p0 = rng.uniform(10.0, 16.0); e0 = rng.uniform(0.1, 0.6); M = 10.0 ** rng.uniform(5.0, 7.0)
        th[s] = rng.uniform(0.0, np.pi); ph_[s] = rng.uniform(0.0, 2.0 * np.pi)
        T = rng.uniform(0.45, 1.05) * n_samples * dt
        e1 = 0.5 * e0
        ts, p, a = _one_source(rng, T=T, n_t=int(counts[s]), uniform=False, p0=p0, p1=6.0 + 2 * e1 + 0.1, e0=e0, e1=e1, M=M, l=l, n=n)
        t[s, :counts[s]] = ts; phase[s, :counts[s]] = p; amp[s, :counts[s]] = a
    return Workload(f"ragged{n_src}", t, phase, amp, l, m, n, th, ph_, 0.0, dt, int(n_samples), eps, n_t_src=counts)


def source_of(w: Workload, s: int) -> Workload:
    """Source s of a batch as a one-source uniform workload with its own knot count (the padding cut off)."""
    c = int(w.n_t_src[s]) if w.n_t_src is not None else w.n_t
    return Workload(f"{w.name}[{s}]", w.t[s:s + 1, :c].copy(), w.phase[s:s + 1, :c].copy(), w.amp[s:s + 1, :c].copy(), w.l, w.m, w.n,
                    w.theta[s:s + 1].copy(), w.phi[s:s + 1].copy(), w.t0, w.dt, w.n_samples, w.eps, k=w.k)


def random_problem(seed: int, *, n_src=1, n_t=12, n_modes=10, l_max=5, n_max=3, T=1000.0, n_samples=257,
                   phase_scale=50.0) -> Workload:
    """Small random problem with a non-uniform grid and a random (l, m >= 0, n) list, for edge-case and
    property tests.  Amplitudes and phases are smooth random functions of t."""
    rng = np.random.Generator(np.random.PCG64(seed))
    allm = [(l, m, n) for l in range(2, l_max + 1) for m in range(0, l + 1) for n in range(-n_max, n_max + 1)]
    pick = rng.choice(len(allm), size=min(n_modes, len(allm)), replace=False)
    pick.sort()
    l, m, n = (np.asarray(x, np.int32) for x in zip(*[allm[i] for i in pick]))
    ts, phs, amps = [], [], []
    for _ in range(n_src):
        g = np.sort(rng.uniform(0.0, T, n_t)); g[0], g[-1] = 0.0, T
        x = g / T
        ph = np.stack([phase_scale * (x + 0.3 * x ** 2 + 0.05 * np.sin(3 * x)),
                       0.7 * phase_scale * (x + 0.2 * x ** 3)], axis=1)
        a = (rng.normal(size=(1, len(l))) + 1j * rng.normal(size=(1, len(l)))) * \
            (1.0 + 0.3 * np.sin(2 * np.pi * rng.uniform(0.5, 2, (1, len(l))) * x[:, None] + rng.uniform(0, 6.28, (1, len(l)))))
        ts.append(g), phs.append(ph), amps.append(a)
    return Workload(f"random{seed}", np.stack(ts), np.stack(phs), np.stack(amps), l, m, n,
                    rng.uniform(0.2, 2.9, n_src), rng.uniform(0, 6.28, n_src), 0.0, T / n_samples, n_samples, 0.0)


# ---------------------------------------------------------------------------------------------------------------
# Inputs of the SURVEY.md section 8(f) rows (still no method arithmetic: angles, a data stream, dense trajectories)
# ---------------------------------------------------------------------------------------------------------------
PAPER_ANGLES = (0.54, 5.36, 1.73, 3.20)   # (theta_S, phi_S, theta_K, phi_K): the one set the paper uses for all its tests


def sky_angles(n_src: int, seed: int = 0):
    """Detector-frame angles [n_src, 4] = (theta_S, phi_S, theta_K, phi_K) and mu/d_L [n_src].  Source 0 carries the paper's
    angles; the others are uniform on the two spheres ("chosen from a random uniform distribution across
    their domain").  mu/d_L ~ LogUniform(1e-2, 1) in the same arbitrary units as the amplitudes."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 500 + seed))
    sky = np.empty((n_src, 4))
    sky[:, 0] = np.arccos(rng.uniform(-1.0, 1.0, n_src)); sky[:, 1] = rng.uniform(0.0, 2.0 * np.pi, n_src)
    sky[:, 2] = np.arccos(rng.uniform(-1.0, 1.0, n_src)); sky[:, 3] = rng.uniform(0.0, 2.0 * np.pi, n_src)
    sky[0] = PAPER_ANGLES
    return sky, 10.0 ** rng.uniform(-2.0, 0.0, n_src)


def data_stream(shape, seed: int = 0, sigma: float = 1.0) -> np.ndarray:
    """White complex Gaussian noise (PSD = 1 up to a constant: the case PAPER.md:292 studies) standing in for the strain
    data d(t) of Eq. (15); tests add a signal to it."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 700 + seed))
    return sigma * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))


def dense_trajectory(n_samples: int, dt: float = 10.0, *, seed: int = 0, l_max: int = L_MAX, n_max: int = N_MAX,
                     p0: float = 14.0, p1: float | None = None, e0: float = 0.5, e1: float | None = None, M: float = 1e6,
                     T: float = YEAR_S, t_start: float = 0.0):
    """Dense inputs of the direct summation (amplitudes and phases "at each point in the dense trajectory",
    10 s steps, no interpolation): the config-1 source evaluated at t_i = t_start + i dt instead of at ~100 sparse points.
    p(t), e(t) linear in t over the year (a window of it if n_samples dt < T); Phi_phi, Phi_r are the closed-form integrals
    of Omega_phi = p^-1.5 / M_s and Omega_r = Omega_phi sqrt(1 - 6/p) for linear p(t); amplitudes by the config-1 model.
    -> (l, m, n, phase [N, 2] float64, amp [N, K] complex128)."""
    p1 = 6.0 + 2 * 0.1 + 0.1 if p1 is None else p1
    e1 = 0.1 if e1 is None else e1
    l, m, n = mode_grid(l_max, n_max)
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 900 + seed))
    t = t_start + dt * np.arange(n_samples, dtype=np.float64)
    Ms = M * MSUN_S
    slope = (p1 - p0) / T

    def F_phi(p):   # antiderivative of p^-1.5 in p
        return -2.0 / np.sqrt(p)

    def F_r(p):     # antiderivative of p^-2 sqrt(p - 6) in p
        return -np.sqrt(p - 6.0) / p + np.arctan(np.sqrt((p - 6.0) / 6.0)) / np.sqrt(6.0)

    p = (p0 + slope * t).astype(np.longdouble)
    phase = np.stack([(F_phi(p) - F_phi(np.longdouble(p0))) / (slope * Ms),
                      (F_r(p) - F_r(np.longdouble(p0))) / (slope * Ms)], axis=1).astype(np.float64)
    e_t = e0 + (e1 - e0) * (t / T)
    amp = _amplitudes(rng, t, T, e_t, l, n, cfg0=False)
    return l, m, n, phase, amp


# ---------------------------------------------------------------------------------------------------------------
# Kerr-shaped workload: polar index k and a third phase, ~10x the modes
# ---------------------------------------------------------------------------------------------------------------
def kerr_mode_grid(l_max: int = L_MAX, k_max: int = 5, n_max: int = N_MAX):
    """(l, m, k, n) int32 arrays, m >= 0 only: l slowest, then m, then k in [-k_max, k_max], n fastest.  Full grid:
    63 (l, m) x 11 x 61 = 42 273 modes, "roughly an order of magnitude" more than Schwarzschild's 3843."""
    ls, ms, ks, ns = [], [], [], []
    for l in range(L_MIN, l_max + 1):
        for m in range(0, l + 1):
            for k in range(-k_max, k_max + 1):
                for n in range(-n_max, n_max + 1):
                    ls.append(l), ms.append(m), ks.append(k), ns.append(n)
    return tuple(np.asarray(x, np.int32) for x in (ls, ms, ks, ns))


def make_kerr(*, n_samples: int = 3_155_760, n_t: int = 100, l_max: int = L_MAX, k_max: int = 5, n_max: int = N_MAX,
              eps: float = 1e-5, t0: float = 0.0, seed: int = 0) -> Workload:
    """Config-1 trajectory with a third, polar phase and the k index.  Nothing here is Kerr physics: the shapes are.
    Omega_theta = Omega_phi sqrt(1 - 3/p) lies between Omega_r and Omega_phi as the polar frequency does;
    |A_lmkn| = config-1 model x exp(-|k| / 1.5) (power concentrated at small |k|), each mode with its own seeded
    modulation and phase.  Phases by the same composite Simpson rule as the other configs."""
    l, m, k, n = kerr_mode_grid(l_max, k_max, n_max)
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 40 + seed))
    T, p0, p1, e0, e1, M = YEAR_S, 14.0, 6.0 + 2 * 0.1 + 0.1, 0.5, 0.1, 1e6
    t = sparse_grid(T, n_t, uniform=False)
    e_t = e0 + (e1 - e0) * (t / T)
    ph2 = _phases(t, T, p0, p1, M)
    Ms = M * MSUN_S
    # Phi_theta: Simpson with 256 sub-steps per interval, as _phases does for the other two
    pth = np.zeros(n_t)
    acc = np.longdouble(0)
    for q in range(n_t - 1):
        hh = (t[q + 1] - t[q]) / 256
        x = t[q] + hh * np.arange(257); xm = x[:-1] + 0.5 * hh
        f = lambda tt: (p0 + (p1 - p0) * tt / T) ** -1.5 / Ms * np.sqrt(1.0 - 3.0 / (p0 + (p1 - p0) * tt / T))
        fa, fm = f(x), f(xm)
        acc += np.sum(((hh / 6.0) * (fa[:-1] + 4.0 * fm + fa[1:])).astype(np.longdouble))
        pth[q + 1] = float(acc)
    phase = np.stack([ph2[:, 0], pth, ph2[:, 1]], axis=1)
    amp = _amplitudes(rng, t, T, e_t, l, n, cfg0=False) * np.exp(-np.abs(k) / 1.5)[None, :]
    return Workload(f"kerr_shaped_{len(l)}modes", t[None], phase[None], amp[None], l, m, n, np.array([0.7]), np.array([1.1]),
                    float(t0), 10.0, int(n_samples), float(eps), k=k)
