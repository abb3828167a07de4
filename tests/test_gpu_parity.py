"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (north_star): waveform rel-L2 <= 1e-10, mismatch <= 1e-12, kept sets identical except
modes whose cumulative power lies within 1e-12 (relative) of the threshold; spline coefficients 1e-12 scaled.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2104_04582_b200 import synth  # noqa: E402

REL_L2_TOL = 1e-10
MISMATCH_TOL = 1e-12
BAND = 1e-12


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "-m gpu tests need a GPU"
    from paper_2104_04582_b200 import api as a
    return a


def dev(a, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def mismatch(a, b):
    """1 - overlap (PSD = 1, time domain), computed as |a^ - b^|^2 / 2 to avoid 1 - x cancellation."""
    ah, bh = a / np.linalg.norm(a), b / np.linalg.norm(b)
    return 0.5 * float(np.linalg.norm(ah - bh) ** 2)


def dd_to_ext(c):
    return c[..., 0].astype(np.longdouble) + c[..., 1].astype(np.longdouble)


def gpu_inputs(w):
    return dict(t=dev(w.t), phase=dev(w.phase), amp=dev(w.amp), l=dev(w.l), m=dev(w.m), n=dev(w.n), theta=dev(w.theta),
                phi=dev(w.phi))


# ------------------------------------------------------------------------------------------- S0
def test_ylm_modes_vs_oracle(api):
    l, m, n = synth.mode_grid()
    theta = np.array([0.7, 2.54, 1e-3, math.pi - 1e-3, 1.2]); phi = np.array([1.1, 4.0, 0.3, 5.5, 0.0])
    yp, ym = api.few_ylm_modes(dev(theta), dev(phi), dev(l), dev(m))
    yp, ym = yp.cpu().numpy(), ym.cpu().numpy()
    for s in range(len(theta)):
        rp, rm = oracle.ylm_modes(l, m, theta[s], phi[s])
        assert np.max(np.abs(yp[s] - rp)) <= 1e-13 and np.max(np.abs(ym[s] - rm)) <= 1e-13
    for (ll, mm) in [(2, 2), (2, -1), (5, 3), (10, -10)]:
        assert abs(api.few_ylm(ll, mm, 0.7, 1.1) - oracle.ylm(ll, mm, 0.7, 1.1)) <= 1e-14
    with pytest.raises(api.FewError):
        api.few_ylm(3, 4, 0.7, 1.1)


# ------------------------------------------------------------------------------------------- S1
@pytest.mark.parametrize("n_t,n_sys,uniform", [(4, 1, True), (5, 33, False), (20, 18, True), (100, 257, False), (100, 7688, False),
                                              (300, 129, False), (736, 40, False), (430, 70, False)])
def test_spline_fit_vs_oracle(api, n_t, n_sys, uniform):
    rng = np.random.default_rng(n_t * 1000 + n_sys)
    n_src = 2
    t = np.stack([synth.sparse_grid(1000.0 * (s + 1), n_t, uniform) for s in range(n_src)])
    if not uniform:
        t[1] = np.sort(rng.uniform(0, 500.0, n_t)); t[1, 0] = 0
    y = rng.normal(size=(n_src, n_t, n_sys)) * 10.0 ** rng.uniform(-3, 1, (n_src, 1, n_sys))
    coef = api.few_spline_fit(dev(t), dev(y)).cpu().numpy()
    api.few_device_status()
    for s in range(n_src):
        ref = oracle.spline_fit(t[s], y[s])
        h = np.diff(t[s])[:, None]
        assert np.array_equal(coef[s][:, 0], y[s][:-1])                 # c0 is a bit copy
        # compare c_p h^p, i.e. each term's contribution at the end of its segment, against the size of the data.  Observed on
        # B200 (round 2): source 0 (the workloads' grid family: uniform / R17 shrinking steps) <= 4.1e-15
        # in every case; source 1 (random sorted knots, h_max/h_min 6 ... 1.1e4 with near-coincident knots, where both FP64
        # solves lose digits to conditioning) <= 5.8e-12.  Bars = ~10x those observations, flat (no scaling by h_max/h_min).
        bar = 5e-14 if s == 0 else 6e-11
        for p in (1, 2, 3):
            err = np.abs(coef[s][:, p] - ref[:, p]) * h ** p
            scale = np.max(np.abs(y[s]), axis=0)[None, :]
            obs = float(np.max(err / scale))
            print(f"S1 observed n_t={n_t} n_sys={n_sys} src={s} p={p} h_max/h_min={float(h.max() / h.min()):.3g}: max err/scale = {obs:.3e}")
            assert obs <= bar, (s, p, obs)


def test_spline_fit_dd_vs_oracle_ext(api):
    for cfg in (0, 1, 4):
        w = synth.make_config(cfg, n_samples=8)
        c = api.few_spline_fit_dd(dev(w.t), dev(w.phase)).cpu().numpy()
        api.few_device_status()
        ref = oracle.spline_fit_ext(w.t[0], w.phase[0])
        got = dd_to_ext(c[0])
        assert np.array_equal(c[0][:, 0, :, 0], w.phase[0][:-1]) and np.all(c[0][:, 0, :, 1] == 0)
        h = np.diff(w.t[0]).astype(np.longdouble)[:, None]
        for frac in (0.5, 1.0):          # phase reached inside / at the end of each segment
            x = frac * h
            pg = got[:, 0] + x * (got[:, 1] + x * (got[:, 2] + x * got[:, 3]))
            pr = ref[:, 0] + x * (ref[:, 1] + x * (ref[:, 2] + x * ref[:, 3]))
            assert float(np.max(np.abs(pg - pr))) <= 2e-12, (cfg, float(np.max(np.abs(pg - pr))))   # radians; x87 oracle ~1e-13


def test_spline_errors(api):
    t = dev(np.arange(3.0)[None]); y = dev(np.zeros((1, 3, 2)))
    with pytest.raises(api.FewError) as e:
        api.few_spline_fit(t, y)
    assert e.value.code == -2                                            # FEW_ERR_TOO_FEW_POINTS
    t = dev(np.array([[0.0, 1.0, 1.0, 2.0, 3.0]])); y = dev(np.zeros((1, 5, 2)))
    api.few_spline_fit(t, y)
    assert api.few_device_status(raise_on_error=False) == -3             # FEW_ERR_NOT_INCREASING
    assert api.few_device_status(raise_on_error=False) == 0              # cleared


# ------------------------------------------------------------------------------------------- S2
def check_keep(keep_gpu, nk_gpu, ref_keep, margin, n_modes, band=0.0):
    """Kept sets must be IDENTICAL (band = 0: the default, used for every BASELINE config and every other case whose
    margins are generic).  Only the constructed threshold-hit case passes band = BAND: there a mode whose cumulative power
    lies within 1e-12 (relative to the step's total) of the threshold may differ (north_star); `margin` is the oracle's pinned
    distance to the threshold (tests/test_oracle_pins.py::test_p8_margin_*).  Returns the modes that differ."""
    k = keep_gpu[: int(nk_gpu)]
    assert np.all(np.diff(k) > 0) and np.all(keep_gpu[int(nk_gpu):] == -1)
    diff = sorted(set(k.tolist()) ^ set(ref_keep.tolist()))
    bad = [j for j in diff if not (band > 0.0 and margin[j] <= band)]
    assert not bad, f"kept sets differ: {bad[:10]} ({len(k)} vs {len(ref_keep)}; margins {[margin[j] for j in bad[:10]]})"
    return diff


@pytest.mark.parametrize("cfg,eps", [(1, 1e-5), (1, 1e-2), (4, 1e-3), (1, 0.5)])
def test_select_modes_vs_oracle_configs(api, cfg, eps):
    w = synth.make_config(cfg, n_samples=8)
    g = gpu_inputs(w)
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    keep, nk = api.few_select_modes(g["amp"], g["m"], yp, ym, eps)
    api.few_device_status()
    ryp, rym = oracle.ylm_modes(w.l, w.m, float(w.theta[0]), float(w.phi[0]))
    # the harmonics differ in the last bits between the two sides; feed the oracle the GPU's so that powers are bit-equal
    ref, margin = oracle.select_modes(w.amp[0], w.m, yp[0].cpu().numpy(), ym[0].cpu().numpy(), eps)
    check_keep(keep[0].cpu().numpy(), nk[0].item(), ref, margin, w.n_modes)
    ref2, _ = oracle.select_modes(w.amp[0], w.m, ryp, rym, eps)
    assert abs(len(ref2) - len(ref)) <= 2


def test_select_modes_batch_and_variants(api):
    w = synth.make_config(3, n_src=5, n_samples=8)
    g = gpu_inputs(w)
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    keep, nk = api.few_select_modes(g["amp"], g["m"], yp, ym, 1e-5)
    keep0, nk0 = api.few_select_modes(g["amp"], g["m"], None, None, 1e-4)      # bare |A|^2 variant
    keepa, nka = api.few_select_modes(g["amp"], g["m"], yp, ym, 0.0)           # eps <= 0: all
    api.few_device_status()
    for s in range(w.n_src):
        ref, margin = oracle.select_modes(w.amp[s], w.m, yp[s].cpu().numpy(), ym[s].cpu().numpy(), 1e-5)
        check_keep(keep[s].cpu().numpy(), nk[s].item(), ref, margin, w.n_modes)
        ref, margin = oracle.select_modes(w.amp[s], w.m, None, None, 1e-4)
        check_keep(keep0[s].cpu().numpy(), nk0[s].item(), ref, margin, w.n_modes)
        assert nka[s].item() == w.n_modes and np.array_equal(keepa[s].cpu().numpy(), np.arange(w.n_modes))


def test_select_modes_tiny_and_ties(api):
    # all powers equal: ties must keep the lowest entry indices (R7)
    amp = np.ones((1, 2, 5), np.complex128); m = np.zeros(5, np.int32)
    keep, nk = api.few_select_modes(dev(amp), dev(m), None, None, 0.45)
    assert nk.item() == 3 and keep[0, :3].tolist() == [0, 1, 2]
    for seed in range(4):
        w = synth.random_problem(100 + seed, n_src=2, n_modes=11, n_t=6)
        g = gpu_inputs(w)
        yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
        for eps in (0.3, 1e-2, 1e-6):
            keep, nk = api.few_select_modes(g["amp"], g["m"], yp, ym, eps)
            for s in range(2):
                ref, margin = oracle.select_modes(w.amp[s], w.m, yp[s].cpu().numpy(), ym[s].cpu().numpy(), eps)
                check_keep(keep[s].cpu().numpy(), nk[s].item(), ref, margin, w.n_modes)


def test_select_modes_flat_and_mixed_rows(api):
    """Rows whose candidate list exceeds the fast kernel's capacity (flat spectra: every entry is above eps*total/(4 n)) go to
    the general kernel through the device-side row list; a batch mixes such a source with an ordinary one, and one source
    alternates flat and steep steps."""
    w = synth.make_config(3, n_src=3, n_samples=8)
    rng = np.random.default_rng(7)
    amp = w.amp.copy()
    flat = (rng.uniform(1.0, 2.0, amp[0].shape) * np.exp(1j * rng.uniform(0, 2 * np.pi, amp[0].shape)))
    amp[0] = flat * 1e-3
    amp[2, ::2] = flat[::2] * 1e-2                      # source 2: every other step flat
    g = gpu_inputs(w)
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    for eps in (1e-5, 1e-2):
        keep, nk = api.few_select_modes(dev(amp), g["m"], yp, ym, eps)
        api.few_device_status()
        for s in range(w.n_src):
            ref, margin = oracle.select_modes(amp[s], w.m, yp[s].cpu().numpy(), ym[s].cpu().numpy(), eps)
            check_keep(keep[s].cpu().numpy(), nk[s].item(), ref, margin, w.n_modes)
    assert nk[0].item() > 3000                             # the flat source keeps almost everything


def test_select_modes_constructed_threshold_hit_uses_the_band(api):
    """The one place the 1e-12 band (north_star) is allowed: eps is chosen so that, in step 0, the cumulative power in front
    of one entry equals (1 - eps) total up to the rounding of eps.  Whether that entry's mode is kept is decided by the
    summation order (oracle: sequential, extended; kernel: tree, FP64), so the two sets may differ by exactly that mode --
    and by nothing else."""
    from fractions import Fraction
    rng = np.random.default_rng(2104)
    n_modes, n_t = 600, 4
    amp = (rng.normal(size=(1, n_t, n_modes)) + 1j * rng.normal(size=(1, n_t, n_modes))) * 10.0 ** rng.uniform(-4, 0, (1, n_t, n_modes))
    m = np.zeros(n_modes, np.int32)
    p0 = amp[0, 0].real ** 2 + amp[0, 0].imag ** 2
    order = sorted(range(n_modes), key=lambda e: (-p0[e], e))
    fr = [Fraction(float(p0[e])) for e in order]
    total = sum(fr)
    r = 37                                                   # the entry of rank 37 sits exactly on the threshold
    eps = float(1 - sum(fr[:r]) / total)
    target = order[r]
    ref, margin = oracle.select_modes(amp[0], m, None, None, eps)
    assert margin[target] <= 1e-15                           # the construction worked (pinned margin)
    assert np.sum(margin <= BAND) == 1                       # and no other mode is anywhere near a threshold
    keep, nk = api.few_select_modes(dev(amp), dev(m), None, None, eps)
    api.few_device_status()
    diff = check_keep(keep[0].cpu().numpy(), nk[0].item(), ref, margin, n_modes, band=BAND)
    assert diff in ([], [target])


# ------------------------------------------------------------------------------------------- S3 and the whole path
def run_gpu_chain(api, w):
    g = gpu_inputs(w)
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32, device="cuda")
    nk = torch.empty((w.n_src,), dtype=torch.int32, device="cuda")
    h = api.few_waveform(g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt,
                         w.n_samples, keep_idx=keep, n_keep=nk)
    api.few_device_status()
    return h.cpu().numpy(), keep.cpu().numpy(), nk.cpu().numpy()


def oracle_with_gpu_keep(w, s, keep, windows):
    """Oracle waveform of source s restricted to a given kept set (so that a mode inside the 1e-12 band cannot
    masquerade as a summation error), on sample windows."""
    yp, ym = oracle.ylm_modes(w.l, w.m, float(w.theta[s]), float(w.phi[s]))
    ca = oracle.spline_fit(w.t[s], np.ascontiguousarray(w.amp[s]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[s], w.phase[s])
    return [oracle.sum_waveform(w.t[s], ca, cp, w.l, w.m, w.n, keep, yp, ym, w.t0, w.dt, nn, i0=i0) for i0, nn in windows]


def test_config0_whole_path(api):
    w = synth.make_config(0)
    h, keep, nk = run_gpu_chain(api, w)
    ref = oracle.waveform(w)
    assert nk[0] == 8
    assert rel_l2(h[0], ref[0]) <= REL_L2_TOL and mismatch(h[0], ref[0]) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - ref[0])) <= 1e-10 * np.max(np.abs(ref[0]))           # element by element


@pytest.mark.parametrize("cfg,n,t0", [(1, 70_000, 0.0), (1, 5_000, 31_500_000.0), (2, 3_000, 15_000_000.0), (4, 4_000, 126_200_000.0)])
def test_configs_window_whole_path(api, cfg, n, t0):
    """Configs 1/2/4 on a window that spans several tiles, a ragged tail and (first window) several sparse segments."""
    w = synth.make_config(cfg, n_samples=n, t0=t0)
    h, keep, nk = run_gpu_chain(api, w)
    ref, parts = oracle.waveform(w, return_parts=True)
    check_keep(keep[0], nk[0], parts[0]["keep_idx"], parts[0]["margin"], w.n_modes)
    ref_k = oracle_with_gpu_keep(w, 0, keep[0][: nk[0]], [(0, n)])[0]
    assert rel_l2(h[0], ref_k) <= REL_L2_TOL and mismatch(h[0], ref_k) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - ref_k)) <= 3e-10 * np.max(np.abs(ref_k))


def test_config3_batch_whole_path(api):
    w = synth.make_config(3, n_src=6, n_samples=3_000, t0=7_000_000.0)
    h, keep, nk = run_gpu_chain(api, w)
    for s in range(w.n_src):
        ref_k = oracle_with_gpu_keep(w, s, keep[s][: nk[s]], [(0, w.n_samples)])[0]
        assert rel_l2(h[s], ref_k) <= REL_L2_TOL, (s, rel_l2(h[s], ref_k))
        assert mismatch(h[s], ref_k) <= MISMATCH_TOL
    # per-source independence: source 2 alone gives the same bits
    w1 = synth.Workload(w.name, w.t[2:3], w.phase[2:3], w.amp[2:3], w.l, w.m, w.n, w.theta[2:3], w.phi[2:3], w.t0, w.dt,
                        w.n_samples, w.eps)
    h1, _, _ = run_gpu_chain(api, w1)
    assert np.array_equal(h1[0], h[2])


def test_layered_sum_with_oracle_coefficients(api):
    """GPU summation fed with the ORACLE's spline coefficients (phases split into hi + lo), all modes, no selection."""
    w = synth.make_config(1, n_samples=2_000, t0=20_000_000.0)
    yp, ym = oracle.ylm_modes(w.l, w.m, 0.7, 1.1)
    ca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[0], w.phase[0])
    hi = cp.astype(np.float64); lo = (cp - hi.astype(np.longdouble)).astype(np.float64)
    cdd = np.stack([hi, lo], axis=-1)
    g = gpu_inputs(w)
    h = api.few_sum_waveform(g["t"], dev(ca[None]), dev(cdd[None]), g["l"], g["m"], g["n"], None, None, dev(yp[None]), dev(ym[None]),
                             w.t0, w.dt, w.n_samples).cpu().numpy()
    ref = oracle.sum_waveform(w.t[0], ca, cp, w.l, w.m, w.n, None, yp, ym, w.t0, w.dt, w.n_samples)
    assert rel_l2(h[0], ref) <= REL_L2_TOL and mismatch(h[0], ref) <= MISMATCH_TOL


def test_sum_edge_cases(api):
    w = synth.random_problem(41, n_modes=9, n_samples=700, T=640.0, n_t=9)
    g = gpu_inputs(w)
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    ca = api.few_spline_fit(g["t"], g["amp"]); cp = api.few_spline_fit_dd(g["t"], g["phase"])
    oyp, oym = oracle.ylm_modes(w.l, w.m, float(w.theta[0]), float(w.phi[0]))
    oca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64)); ocp = oracle.spline_fit_ext(w.t[0], w.phase[0])

    def both(t0, dt, N, keep=None, scale=None):
        kd = nk = None
        if keep is not None:
            kk = np.full((1, w.n_modes), -1, np.int32); kk[0, : len(keep)] = keep
            kd, nk = dev(kk), dev(np.array([len(keep)], np.int32))
        h = api.few_sum_waveform(g["t"], ca, cp, g["l"], g["m"], g["n"], kd, nk, yp, ym, t0, dt, N,
                                 scale=None if scale is None else dev(np.array([scale]))).cpu().numpy()[0]
        ref = oracle.sum_waveform(w.t[0], oca, ocp, w.l, w.m, w.n, keep, oyp, oym, t0, dt, N, scale=1.0 if scale is None else scale)
        return h, ref

    h, ref = both(-50.0, 1.0, 800)                          # samples before t_0 and after t_last are exactly 0 (R12)
    ti = -50.0 + np.arange(800)
    assert np.all(h[(ti < 0) | (ti > 640.0)] == 0) and rel_l2(h, ref) <= REL_L2_TOL
    h, ref = both(float(w.t[0, 3]), 0.0625, 40)             # first sample exactly on an interior knot
    assert rel_l2(h, ref) <= REL_L2_TOL
    h, ref = both(float(w.t[0, -1]), 1.0, 3)                # first sample exactly on the last knot, rest outside
    assert h[1] == 0 and h[2] == 0 and abs(h[0] - ref[0]) <= 1e-10 * abs(ref[0])
    h, ref = both(0.0, 640.0 / 699, 700, keep=np.array([1, 4, 5], np.int32), scale=3.5e-3)   # sub-list + mu/dL scale
    assert rel_l2(h, ref) <= REL_L2_TOL
    h, ref = both(0.0, 1.0, 300, keep=np.array([], np.int32))                               # nothing kept -> zeros
    assert np.all(h == 0)
    h, ref = both(1000.0, 1.0, 300)                         # entirely outside
    assert np.all(h == 0)
    out = api.few_sum_waveform(g["t"], ca, cp, g["l"], g["m"], g["n"], None, None, yp, ym, 0.0, 1.0, 0)   # empty
    assert out.shape == (1, 0)
    api.few_device_status()


def test_bad_modes_reported(api):
    w = synth.random_problem(51, n_modes=6, n_samples=64)
    g = gpu_inputs(w)
    bad_m = w.m.copy(); bad_m[2] = w.l[2] + 1
    api.few_ylm_modes(g["theta"], g["phi"], g["l"], dev(bad_m))
    assert api.few_device_status(raise_on_error=False) == -4             # FEW_ERR_BAD_MODE
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    with pytest.raises(api.FewError) as e:                               # dt <= 0 is rejected on the host
        api.few_sum_waveform(g["t"], g["t"], g["t"], g["l"], g["m"], g["n"], None, None, yp, ym, 0.0, -1.0, 10)
    assert e.value.code == -1


def test_many_l_per_pair_and_n_gaps(api):
    """Mode lists outside the paper's grid: 15 distinct l for one (m, n), gaps in n, a single negative-n run."""
    rng = np.random.default_rng(7)
    modes = [(l, 0, 0) for l in range(2, 17)] + [(l, 3, n) for l in (3, 5, 9) for n in (-17, -4, 2, 11)] + [(6, 6, -2), (7, 5, 40)]
    l, m, n = (np.asarray(x, np.int32) for x in zip(*modes))
    n_t = 9
    t = np.sort(rng.uniform(0, 500.0, n_t)); t[0] = 0.0
    amp = rng.normal(size=(1, n_t, len(l))) + 1j * rng.normal(size=(1, n_t, len(l)))
    phase = np.stack([0.9 * t + 1e-3 * t ** 2, 0.4 * t + 2e-4 * t ** 2], axis=1)[None]
    w = synth.Workload("many_l", t[None], phase, amp, l, m, n, np.array([1.3]), np.array([0.4]), 3.0, 0.37, 1200, 0.0)
    h, keep, nk = run_gpu_chain(api, w)
    ref = oracle.waveform(w)
    assert nk[0] == len(l) and rel_l2(h[0], ref[0]) <= REL_L2_TOL and mismatch(h[0], ref[0]) <= MISMATCH_TOL


def wide_n_problem(seed, n_values, n_src=1, n_samples=900):
    """A mode list whose radial indices spread over many blocks of four: l = 2..4, m = 0..2, n in n_values."""
    rng = np.random.default_rng(seed)
    modes = [(l, m, n) for l in (2, 3, 4) for m in range(0, 3) for n in n_values]
    l, m, n = (np.asarray(x, np.int32) for x in zip(*modes))
    n_t = 12
    t = np.stack([np.sort(rng.uniform(0, 700.0, n_t)) for _ in range(n_src)]); t[:, 0] = 0.0
    amp = (rng.normal(size=(n_src, n_t, len(l))) + 1j * rng.normal(size=(n_src, n_t, len(l)))) * 10.0 ** rng.uniform(-2, 0, (n_src, 1, len(l)))
    phase = np.stack([0.31 * t + 2e-4 * t ** 2, 0.17 * t + 1e-4 * t ** 2], axis=2)
    return synth.Workload("wide_n", t, phase, amp, l, m, n, rng.uniform(0.3, 2.8, n_src), rng.uniform(0, 6.28, n_src), 1.5, 0.71, n_samples, 0.0)


def test_sum_recurrence_instantiation_more_than_8_nu_blocks(api):
    """Lists with more than 8 distinct blocks |n| >> 2 do not fit the tensor-memory table of the summation kernel and take its
    recurrence instantiation (rho^nu stepped in registers); 11 blocks here, with gaps, both signs and |n| up to 43."""
    w = wide_n_problem(11, [-43, -40, -33, -21, -12, -9, -2, 0, 1, 6, 14, 19, 25, 30, 36])
    assert len({abs(int(x)) // 4 for x in w.n}) > 8
    h, keep, nk = run_gpu_chain(api, w)
    ref = oracle.waveform(w)
    assert nk[0] == w.n_modes and rel_l2(h[0], ref[0]) <= REL_L2_TOL and mismatch(h[0], ref[0]) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - ref[0])) <= 1e-10 * np.max(np.abs(ref[0]))


def test_sum_batch_mixing_table_and_recurrence_sources(api):
    """One call, two kinds of kept lists: sources whose selection leaves <= 8 nu-blocks (table instantiation) and sources
    that keep a list with 12 (recurrence instantiation); each kernel takes its own tiles of the shared tile list."""
    w = wide_n_problem(12, list(range(-46, 47, 4)) + [1, 2, 3], n_src=4, n_samples=700)
    g = gpu_inputs(w)
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    ca = api.few_spline_fit(g["t"], g["amp"]); cp = api.few_spline_fit_dd(g["t"], g["phase"])
    narrow = np.flatnonzero(np.abs(w.n) <= 14).astype(np.int32)          # 4 blocks -> table mode
    keep = np.full((w.n_src, w.n_modes), -1, np.int32); nk = np.zeros(w.n_src, np.int32)
    for s in range(w.n_src):
        sel = narrow if s % 2 == 0 else np.arange(w.n_modes, dtype=np.int32)
        keep[s, : len(sel)] = sel; nk[s] = len(sel)
    h = api.few_sum_waveform(g["t"], ca, cp, g["l"], g["m"], g["n"], dev(keep), dev(nk), yp, ym, w.t0, w.dt, w.n_samples).cpu().numpy()
    api.few_device_status()
    for s in range(w.n_src):
        ref = oracle_with_gpu_keep(w, s, keep[s][: nk[s]], [(0, w.n_samples)])[0]
        assert rel_l2(h[s], ref) <= REL_L2_TOL and mismatch(h[s], ref) <= MISMATCH_TOL, s


@pytest.mark.parametrize("ms", [(0,), (2, 5), (0, 4)])
def test_sum_lists_of_m0_runs_only_and_without_m0(api, ms):
    """Runs with m = 0 accumulate the c half of a step in S and the s half in D (summed at the close); other runs keep S and D
    apart.  Lists made of m = 0 runs only, without any, and with an m increment above 1, long enough (8 nu-blocks per run) to
    cross the 16-step stages of the coefficient ring."""
    rng = np.random.default_rng(21 + sum(ms))
    modes = [(l, m, n) for m in ms for l in (max(2, m), max(2, m) + 1, max(2, m) + 3) for n in range(-31, 32, 3)]
    l, m, n = (np.asarray(x, np.int32) for x in zip(*modes))
    n_t = 10
    t = np.sort(rng.uniform(0, 900.0, n_t)); t[0] = 0.0
    amp = (rng.normal(size=(1, n_t, len(l))) + 1j * rng.normal(size=(1, n_t, len(l)))) * 10.0 ** rng.uniform(-2, 0, (1, 1, len(l)))
    phase = np.stack([0.23 * t + 1.5e-4 * t ** 2, 0.19 * t + 0.7e-4 * t ** 2], axis=1)[None]
    w = synth.Workload("m_runs", t[None], phase, amp, l, m, n, np.array([1.1]), np.array([5.0]), 2.0, 0.53, 1700, 0.0)
    h, keep, nk = run_gpu_chain(api, w)
    ref = oracle.waveform(w)
    assert nk[0] == w.n_modes and rel_l2(h[0], ref[0]) <= REL_L2_TOL and mismatch(h[0], ref[0]) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - ref[0])) <= 1e-10 * np.max(np.abs(ref[0]))


def test_sum_large_n_and_sparse_list_limit(api):
    """|n| up to FEW_MAX_ABS_N = 1023 (256 steps of the three-term recurrence: error <= 256^2 ulp) is summed; a list with
    fewer than 4 modes per step and more than 64 steps over n_modes / 4 does not fit the step capacity and is reported."""
    rng = np.random.default_rng(5)
    modes = [(2, 2, n) for n in (0, 1, 250, -640, 1023, -1023)] + [(3, 1, 512)]
    l, m, n = (np.asarray(x, np.int32) for x in zip(*modes))
    n_t = 8
    t = np.linspace(0.0, 64.0, n_t)
    amp = rng.normal(size=(1, n_t, len(l))) + 1j * rng.normal(size=(1, n_t, len(l)))
    phase = np.stack([0.05 * t + 1e-4 * t ** 2, 0.011 * t + 3e-5 * t ** 2], axis=1)[None]
    w = synth.Workload("large_n", t[None], phase, amp, l, m, n, np.array([0.9]), np.array([2.0]), 0.0, 0.05, 1200, 0.0)
    h, keep, nk = run_gpu_chain(api, w)
    ref = oracle.waveform(w)
    assert rel_l2(h[0], ref[0]) <= REL_L2_TOL and mismatch(h[0], ref[0]) <= MISMATCH_TOL
    # 400 modes, every one alone in its step (n = 4 j): 400 steps > 400 / 4 + 64
    modes = [(2, 0, 4 * j) for j in range(200)] + [(2, 1, 4 * j) for j in range(200)]
    l, m, n = (np.asarray(x, np.int32) for x in zip(*modes))
    amp = rng.normal(size=(1, n_t, len(l))) + 1j * rng.normal(size=(1, n_t, len(l)))
    w2 = synth.Workload("sparse", t[None], phase, amp, l, m, n, np.array([0.9]), np.array([2.0]), 0.0, 0.05, 64, 0.0)
    g = gpu_inputs(w2)
    api.few_waveform(g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], 0.0, w2.t0, w2.dt, w2.n_samples)
    assert api.few_device_status(raise_on_error=False) == -7            # FEW_ERR_LIMIT (FEW_DEV_SPARSE_LIST)
    assert api.few_device_status(raise_on_error=False) == 0


def test_step_bound_shrinks_the_workspace_and_keeps_the_bits(api):
    """few_set_max_steps (few.h): with the bound few_max_steps_for_modes gives for the grid (88) the workspace is a fraction of
    the default one and the waveform has the same bits; a bound the kept list exceeds is reported as FEW_ERR_LIMIT with every
    access still in bounds; a workspace sized for a smaller bound than the context's is refused; few_waveform_host bounds its own
    workspace from the host mode list and leaves the context's setting alone."""
    w = synth.make_config(3, n_src=3, n_samples=20_000)
    g = gpu_inputs(w)
    n_src, n_t, n_modes = w.amp.shape
    args = (g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt, w.n_samples)
    ref = api.few_waveform(*args)
    api.few_device_status()
    bound = api.few_max_steps_for_modes(torch.as_tensor(w.m), torch.as_tensor(w.n))
    assert bound == 88                                                    # 11 values of m x 8 blocks of four |n| (|n| <= 30)
    full = api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples)
    try:
        api.few_set_max_steps(bound)
        small = api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples)
        assert small == api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples, max_steps=bound) and small < 0.4 * full
        ws = torch.full((small,), 0xFF, dtype=torch.uint8, device="cuda")
        h = api.few_waveform(*args, workspace=ws)
        api.few_device_status()
        assert torch.equal(torch.view_as_real(h), torch.view_as_real(ref))
        cpu = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()      # noqa: E731
        hh = api.few_waveform_host(cpu(w.t), cpu(w.phase), cpu(w.amp), cpu(w.l), cpu(w.m), cpu(w.n), cpu(w.theta), cpu(w.phi),
                                   w.eps, w.t0, w.dt, w.n_samples)
        assert np.array_equal(hh.numpy().view(np.float64), ref.cpu().numpy().view(np.float64))
        # a workspace laid out for a smaller bound than the context holds is too small
        tiny = torch.empty(api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples, max_steps=8), dtype=torch.uint8, device="cuda")
        with pytest.raises(api.FewError) as e:
            api.few_waveform(*args, workspace=tiny)
        assert e.value.code == -5                                         # FEW_ERR_WORKSPACE
        # a bound below what the kept lists need (tens of steps per source): reported, nothing out of bounds
        api.few_set_max_steps(8)
        ws8 = torch.full((api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples),), 0xFF, dtype=torch.uint8, device="cuda")
        api.few_waveform(*args, workspace=ws8)
        torch.cuda.synchronize()
        assert api.few_device_status(raise_on_error=False) == -7          # FEW_ERR_LIMIT (FEW_DEV_SPARSE_LIST)
        # the host path computes its own bound (88 > 8 is not lower, so the caller's 8 stands and is reported the same way)
        with pytest.raises(api.FewError) as e:
            api.few_waveform_host(cpu(w.t), cpu(w.phase), cpu(w.amp), cpu(w.l), cpu(w.m), cpu(w.n), cpu(w.theta), cpu(w.phi),
                                  w.eps, w.t0, w.dt, w.n_samples)
        assert e.value.code == -7
    finally:
        api.few_set_max_steps(0)
    assert api.few_waveform_workspace(n_src, n_t, n_modes, w.n_samples) == full
    h = api.few_waveform(*args)
    api.few_device_status()
    assert torch.equal(torch.view_as_real(h), torch.view_as_real(ref))


@pytest.mark.parametrize("pinned_out", [True, False])
def test_whole_path_host_buffers(api, pinned_out):
    """few_waveform_host: pinned h is written by the summation kernel itself (mapped stores), pageable h by a copy."""
    w = synth.make_config(1, n_samples=4_000, t0=1_000_000.0)
    f = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    keep = torch.empty((1, w.n_modes), dtype=torch.int32).pin_memory(); nk = torch.empty((1,), dtype=torch.int32).pin_memory()
    out = torch.full((1, w.n_samples), float("nan"), dtype=torch.complex128)
    out = out.pin_memory() if pinned_out else out
    h = api.few_waveform_host(f(w.t), f(w.phase), f(w.amp), f(w.l), f(w.m), f(w.n), f(w.theta), f(w.phi), w.eps, w.t0, w.dt,
                              w.n_samples, out=out, keep_idx=keep, n_keep=nk).numpy()
    hd, keepd, nkd = run_gpu_chain(api, w)
    assert np.array_equal(h, hd) and nk[0].item() == nkd[0] and np.array_equal(keep.numpy(), keepd)
    ref_k = oracle_with_gpu_keep(w, 0, keepd[0][: nkd[0]], [(0, w.n_samples)])[0]
    assert rel_l2(h[0], ref_k) <= REL_L2_TOL


def test_host_buffers_batch_in_source_groups(api):
    """few_waveform_host cuts a batch into source groups (copy/compute overlap): results equal the one-shot device chain."""
    w = synth.make_config(3, n_src=11, n_samples=3_000, t0=2_000_000.0)
    f = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32).pin_memory(); nk = torch.empty((w.n_src,), dtype=torch.int32).pin_memory()
    h = api.few_waveform_host(f(w.t), f(w.phase), f(w.amp), f(w.l), f(w.m), f(w.n), f(w.theta), f(w.phi), w.eps, w.t0, w.dt,
                              w.n_samples, keep_idx=keep, n_keep=nk).numpy()
    hd, keepd, nkd = run_gpu_chain(api, w)
    assert np.array_equal(nk.numpy(), nkd) and np.array_equal(keep.numpy(), keepd) and np.array_equal(h, hd)


# ------------------------------------------------------------------------------------------- full size, sampled
@pytest.mark.parametrize("cfg", [1, 2])
def test_full_size_sampled_parity(api, cfg):
    """BASELINE configs 1 and 2 at full size in bench.py's launch configuration; the oracle recomputes sampled windows
    (first / last samples, segment boundaries, and a stride through the year)."""
    w = synth.make_config(cfg)
    h, keep, nk = run_gpu_chain(api, w)
    N = w.n_samples
    n_win = 256 if cfg == 1 else 48
    knots = [int(math.ceil(tk / w.dt)) for tk in w.t[0][[1, 37, 80, 98]]]
    windows = [(0, n_win), (N - n_win, n_win)] + [(max(i - n_win // 2, 0), n_win) for i in knots] + \
              [(i0, n_win) for i0 in range(99_991, N - n_win, N // 12)]
    refs = oracle_with_gpu_keep(w, 0, keep[0][: nk[0]], windows)
    got = np.concatenate([h[0][i0:i0 + nn] for i0, nn in windows]); ref = np.concatenate(refs)
    assert rel_l2(got, ref) <= REL_L2_TOL and mismatch(got, ref) <= MISMATCH_TOL
    assert np.all(np.isfinite(h.view(np.float64)))
    # property at any size: Parseval-like power check of the whole output against the kept modes' mean power is too loose;
    # instead every 4099th sample is recomputed one by one
    idx = np.arange(7, N, 4099 if cfg == 1 else 40_009)
    one = np.concatenate(oracle_with_gpu_keep(w, 0, keep[0][: nk[0]], [(int(i), 1) for i in idx]))
    assert rel_l2(h[0][idx], one) <= REL_L2_TOL


def test_sharded_calls_reassemble_bit_equal(api):
    """The property the multi-GPU split relies on: a waveform computed as two contiguous sample ranges
    (each call repeating S0-S2-S1 and passing t0 + i0 dt), and a batch computed as two source ranges, concatenate BIT-EQUAL to
    the unsharded call -- every sample's arithmetic depends on its own t_i only, whatever tile, warp or lane it lands in."""
    from paper_2104_04582_b200.shard import shard_samples, shard_sources, shard_t0
    w = synth.make_config(1)
    h, keep, nk = run_gpu_chain(api, w)
    parts = []
    for rank in range(2):
        i0, cnt = shard_samples(w.n_samples, rank, 2)
        ws = synth.Workload(w.name, w.t, w.phase, w.amp, w.l, w.m, w.n, w.theta, w.phi, shard_t0(w.t0, w.dt, i0), w.dt, cnt, w.eps)
        hs, ks, ns = run_gpu_chain(api, ws)
        assert np.array_equal(ks, keep) and np.array_equal(ns, nk)
        parts.append(hs[0])
    assert np.array_equal(np.concatenate(parts), h[0])
    # an odd split point (not a multiple of the tile) gives the same bits too
    i0 = 1_234_567
    wa = synth.Workload(w.name, w.t, w.phase, w.amp, w.l, w.m, w.n, w.theta, w.phi, w.t0, w.dt, i0, w.eps)
    wb = synth.Workload(w.name, w.t, w.phase, w.amp, w.l, w.m, w.n, w.theta, w.phi, shard_t0(w.t0, w.dt, i0), w.dt, w.n_samples - i0, w.eps)
    assert np.array_equal(np.concatenate([run_gpu_chain(api, wa)[0][0], run_gpu_chain(api, wb)[0][0]]), h[0])
    wb3 = synth.make_config(3, n_src=9, n_samples=5_000, t0=3_000_000.0)
    h3, _, _ = run_gpu_chain(api, wb3)
    for rank in range(2):
        s0, sc = shard_sources(wb3.n_src, rank, 2)
        wr = synth.Workload(wb3.name, wb3.t[s0:s0 + sc], wb3.phase[s0:s0 + sc], wb3.amp[s0:s0 + sc], wb3.l, wb3.m, wb3.n, wb3.theta[s0:s0 + sc],
                            wb3.phi[s0:s0 + sc], wb3.t0, wb3.dt, wb3.n_samples, wb3.eps)
        assert np.array_equal(run_gpu_chain(api, wr)[0], h3[s0:s0 + sc])


def knot_windows(w, s, knots, n_win):
    """Sample windows of n_win samples centred on the first dense sample at or after the given sparse knots of source s."""
    out = []
    for k in knots:
        i = int(math.ceil((w.t[s][k] - w.t0) / w.dt))
        out.append((min(max(i - n_win // 2, 0), w.n_samples - n_win), n_win))
    return out


def test_config3_full_size_sampled_parity_device_and_host_paths(api):
    """BASELINE config 3 exactly as bench.py times it: 64 sources x 1 051 920 samples, one few_waveform call, and the same
    through few_waveform_host (8 source groups, h stored by the kernel into a 1.08 GB pinned host buffer).  Kept sets of all
    64 sources must equal the oracle's; the waveform is recomputed by the oracle on windows at the first and last samples of
    every source and at segment boundaries, with the three sources whose phases end highest (59, 35, 9: 1.0-1.3e6 rad, the
    precision worst case of SURVEY H1) covered by several windows each including the end of the trajectory."""
    w = synth.make_config(3)
    assert w.n_src == 64 and w.n_samples == 1_051_920
    worst = [int(s) for s in np.argsort(-w.phase[:, -1, 0])[:3]]
    assert w.phase[worst[0], -1, 0] > 1.2e6
    g = gpu_inputs(w)
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32, device="cuda")
    nk = torch.empty((w.n_src,), dtype=torch.int32, device="cuda")
    h = api.few_waveform(g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt,
                         w.n_samples, keep_idx=keep, n_keep=nk)
    api.few_device_status()
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    yp, ym, keep_h, nk_h = yp.cpu().numpy(), ym.cpu().numpy(), keep.cpu().numpy(), nk.cpu().numpy()
    N = w.n_samples
    worst_err = 0.0
    for s in range(w.n_src):
        ref, margin = oracle.select_modes(w.amp[s], w.m, yp[s], ym[s], w.eps)      # the GPU's harmonics: bit-equal powers
        check_keep(keep_h[s], nk_h[s], ref, margin, w.n_modes)                   # identical, no band
        if s in worst:
            wins = [(0, 192), (N - 192, 192)] + knot_windows(w, s, [1, 2, 40, 77, 78], 192) + [(i0, 64) for i0 in range(50_021, N - 64, N // 9)]
        else:
            wins = [(0, 48), (N - 48, 48)] + knot_windows(w, s, [1 + s % 70, 78], 48)
        refs = np.concatenate(oracle_with_gpu_keep(w, s, keep_h[s][: nk_h[s]], wins))
        got = torch.cat([h[s, i0:i0 + nn] for i0, nn in wins]).cpu().numpy()
        e = rel_l2(got, refs)
        worst_err = max(worst_err, e)
        assert e <= REL_L2_TOL and mismatch(got, refs) <= MISMATCH_TOL, (s, e)
        assert np.max(np.abs(got - refs)) <= 3e-10 * np.max(np.abs(refs)), s
    print(f"config 3 full size: worst windowed rel-L2 over 64 sources {worst_err:.3e}; kept {int(nk_h.sum())}")
    assert bool(torch.isfinite(torch.view_as_real(h)).all())
    # host path: pinned inputs and a pinned 1.08 GB output written by the kernel's own stores
    f = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    keep2 = torch.empty((w.n_src, w.n_modes), dtype=torch.int32).pin_memory(); nk2 = torch.empty((w.n_src,), dtype=torch.int32).pin_memory()
    h_host = torch.full((w.n_src, N), float("nan"), dtype=torch.complex128).pin_memory()
    api.few_waveform_host(f(w.t), f(w.phase), f(w.amp), f(w.l), f(w.m), f(w.n), f(w.theta), f(w.phi), w.eps, w.t0, w.dt, N,
                          out=h_host, keep_idx=keep2, n_keep=nk2)
    assert np.array_equal(nk2.numpy(), nk_h) and np.array_equal(keep2.numpy(), keep_h)
    for s0 in range(0, w.n_src, 8):                       # bit-equal to the device-resident call, compared on the device
        assert torch.equal(h_host[s0:s0 + 8].cuda(), h[s0:s0 + 8]), s0


@pytest.mark.parametrize("eps", [1e-2, 1e-3, 1e-4, 1e-5, 0.0])
def test_config4_full_size_sampled_parity_eps_sweep(api, eps):
    """BASELINE config 4 at full size (12 623 040 samples, 300 knots: ~24.7 k tiles over 301 pseudo-segments) for every eps
    of the sweep bench.py times; windows include the first and last 256 samples and the knots 1, 150 and 298."""
    w = synth.make_config(4, eps=eps)
    assert w.n_samples == 12_623_040 and w.n_t == 300
    h, keep, nk = run_gpu_chain(api, w)
    yp, ym = api.few_ylm_modes(dev(w.theta), dev(w.phi), dev(w.l), dev(w.m))
    ref, margin = oracle.select_modes(w.amp[0], w.m, yp[0].cpu().numpy(), ym[0].cpu().numpy(), eps)
    check_keep(keep[0], nk[0], ref, margin, w.n_modes)
    N = w.n_samples
    n_win = 256 if eps > 0 else 64
    wins = [(0, n_win), (N - 256, 256)] + knot_windows(w, 0, [1, 150, 298], n_win) + [(i0, 32) for i0 in range(400_009, N - 32, N // 7)]
    refs = np.concatenate(oracle_with_gpu_keep(w, 0, keep[0][: nk[0]], wins))
    got = np.concatenate([h[0][i0:i0 + nn] for i0, nn in wins])
    assert rel_l2(got, refs) <= REL_L2_TOL and mismatch(got, refs) <= MISMATCH_TOL, (eps, rel_l2(got, refs))
    assert np.max(np.abs(got - refs)) <= 3e-10 * np.max(np.abs(refs))
    idx = np.arange(11, N, 250_007)
    one = np.concatenate(oracle_with_gpu_keep(w, 0, keep[0][: nk[0]], [(int(i), 1) for i in idx]))
    assert rel_l2(h[0][idx], one) <= REL_L2_TOL
    assert np.all(np.isfinite(h.view(np.float64)))
    print(f"config 4 eps={eps:g}: kept {int(nk[0])}, windowed rel-L2 {rel_l2(got, refs):.3e}")


def test_whole_path_under_cuda_graph_capture(api):
    """few_waveform enqueues everything on the caller's stream and two internal side streams forked and joined by events, never
    synchronises the host and allocates nothing: the call can be captured into a CUDA graph.  A replay on new input values gives
    the bits of the eager call."""
    w = synth.make_config(1)
    n = 40_000
    g = gpu_inputs(w)
    args = lambda amp: (g["t"], g["phase"], amp, g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0 + 3.0e6, w.dt, n)
    ws = torch.empty(api.few_waveform_workspace(w.n_src, w.n_t, w.n_modes, n), dtype=torch.uint8, device=g["t"].device)
    h_g = torch.zeros((w.n_src, n), dtype=torch.complex128, device=g["t"].device)
    amp_g = g["amp"].clone()
    api.few_profile_enable(False)
    api.few_waveform(*args(amp_g), out=h_g, workspace=ws)                 # warm-up outside the capture (attributes, lazy loading)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        api.few_waveform(*args(amp_g), out=h_g, workspace=ws)
    for scale in (1.0, 0.5):
        amp_g.copy_(g["amp"] * scale)
        h_g.zero_()
        graph.replay()
        torch.cuda.synchronize()
        h_e = api.few_waveform(*args(g["amp"] * scale))
        api.few_device_status()
        assert torch.equal(h_g, h_e), scale
    assert float(h_g.abs().max()) > 0.0


def test_fp64_peak_probe_runs(api):
    """The one measurement aid left in the ABI (the roofline denominator bench.py prints beside the nominal peak) launches,
    writes finite values and sustains a plausible FP64 rate; no throughput ordering is asserted."""
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device="cuda")
    api.few_fp64_peak_probe(148 * 8, 256, 500, sink); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); flops = api.few_fp64_peak_probe(148 * 8, 256, 5000, sink); b.record(); torch.cuda.synchronize()
    rate = flops / (a.elapsed_time(b) * 1e-3) / 1e12
    api.few_device_status()
    assert bool(torch.isfinite(sink).all()) and rate > 1.0, rate
