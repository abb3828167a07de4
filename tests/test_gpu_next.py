"""GPU parity of the SURVEY.md section 8(f) rows against the CPU oracle (through the C-ABI binding):
  NEXT-1  detector-frame transformation, fused into the summation (few_frame_constants, few_waveform_ssb) and as a pass
          (few_frame_rotate)
  NEXT-2  PSD = 1 inner products, fused into the summation kernel (few_sum_waveform_ex / few_waveform_ssb) and as a separate
          reduction (few_inner_products)
  NEXT-3  direct summation (few_sum_direct)
Bars: waveforms rel-L2 <= 1e-10 and mismatch <= 1e-12 (north_star); inner products within 1e-10 of 2 dt |d| |h| (the waveform
bar carried through Cauchy-Schwarz), in practice ~1e-14; constants 1e-14.
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
    ah, bh = a / np.linalg.norm(a), b / np.linalg.norm(b)
    return 0.5 * float(np.linalg.norm(ah - bh) ** 2)


# ------------------------------------------------------------------------------------------- NEXT-1
def test_frame_constants_vs_oracle(api):
    sky, mu = synth.sky_angles(40, seed=1)
    sky[1] = (1.0, 0.3, 1.0 + 1e-6, 0.3 + 1e-6)            # spin almost along the line of sight
    sky[2] = (1e-4, 2.0, math.pi - 1e-4, 5.0)              # both near the poles
    sky[3] = (0.9, 1.1, 0.9, 1.1)                          # exactly degenerate: N = D = 0 up to rounding of the products
    th, ph, f = api.few_frame_constants(dev(sky), dev(mu))
    th, ph, f = th.cpu().numpy(), ph.cpu().numpy(), f.cpu().numpy()
    for s in range(sky.shape[0]):
        rt, rp, rf = oracle.frame(*sky[s], mu[s])
        R = np.array([math.sin(sky[s, 0]) * math.cos(sky[s, 1]), math.sin(sky[s, 0]) * math.sin(sky[s, 1]), math.cos(sky[s, 0])])
        S = np.array([math.sin(sky[s, 2]) * math.cos(sky[s, 3]), math.sin(sky[s, 2]) * math.sin(sky[s, 3]), math.cos(sky[s, 2])])
        sin_rs = np.linalg.norm(np.cross(R, S))
        assert ph[s] == rp
        if s == 3:
            assert abs(abs(f[s]) - mu[s]) <= 1e-15          # direction of the factor is undefined; its modulus is not
            continue
        # theta from cos(theta) = -R.S: FP64 rounding of the dot product moves it by eps / sin(theta)
        assert abs(th[s] - rt) <= 4e-16 / max(sin_rs, 1e-8) + 4e-16, (s, th[s], rt)
        assert abs(f[s] - rf) <= 1e-15 * mu[s] / max(sin_rs, 1e-8) ** 2 + 4e-16 * mu[s], (s, f[s], rf)


def test_frame_rotate_vs_oracle(api):
    rng = np.random.default_rng(5)
    for n_src, N in [(1, 1), (3, 1000), (2, 70_001), (5, 4096)]:
        h = rng.normal(size=(n_src, N)) + 1j * rng.normal(size=(n_src, N))
        f = rng.normal(size=n_src) + 1j * rng.normal(size=n_src)
        out = api.few_frame_rotate(dev(h), dev(f)).cpu().numpy()
        for s in range(n_src):
            ref = oracle.frame_apply(h[s], complex(f[s]))
            assert np.max(np.abs(out[s] - ref)) <= 4e-16 * abs(f[s]) * np.max(np.abs(h[s]))
    hd = dev(h)
    api.few_frame_rotate(hd, dev(f), out=hd)               # in place
    assert np.array_equal(hd.cpu().numpy(), out)
    assert api.few_frame_rotate(dev(np.zeros((2, 0), np.complex128)), dev(f[:2])).shape == (2, 0)


def ssb_oracle(w, sky, mu, keep_by_src, windows=None):
    """Oracle chain in the detector frame: O5 -> O2 -> O1 -> O4 at (theta_src, phi_src) -> O5 apply, restricted to given kept sets."""
    out = []
    for s in range(w.n_src):
        th, ph, f = oracle.frame(*sky[s], mu[s] if mu is not None else 1.0)
        yp, ym = oracle.ylm_modes(w.l, w.m, th, ph)
        ca = oracle.spline_fit(w.t[s], np.ascontiguousarray(w.amp[s]).view(np.float64))
        cp = oracle.spline_fit_ext(w.t[s], w.phase[s])
        wins = windows if windows is not None else [(0, w.n_samples)]
        hs = [oracle.frame_apply(oracle.sum_waveform(w.t[s], ca, cp, w.l, w.m, w.n, keep_by_src[s], yp, ym, w.t0, w.dt, nn, i0=i0), f)
              for i0, nn in wins]
        out.append(np.concatenate(hs))
    return out


def run_ssb(api, w, sky, mu, d=None, want_h=True, want_inner=False):
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32, device="cuda")
    nk = torch.empty((w.n_src,), dtype=torch.int32, device="cuda")
    h, inner = api.few_waveform_ssb(dev(w.t), dev(w.phase), dev(w.amp), dev(w.l), dev(w.m), dev(w.n), dev(sky), w.eps, w.t0, w.dt,
                                    w.n_samples, mu_over_dl=None if mu is None else dev(mu), d=None if d is None else dev(d),
                                    want_inner=want_inner, want_h=want_h, keep_idx=keep, n_keep=nk)
    api.few_device_status()
    keep, nk = keep.cpu().numpy(), nk.cpu().numpy()
    return (None if h is None else h.cpu().numpy()), (None if inner is None else inner.cpu().numpy()), \
        [keep[s][: nk[s]] for s in range(w.n_src)]


def test_waveform_ssb_config0(api):
    w = synth.make_config(0)
    sky, mu = synth.sky_angles(1)
    h, _, keep = run_ssb(api, w, sky, mu)
    ref = ssb_oracle(w, sky, mu, keep)[0]
    assert len(keep[0]) == 8
    assert rel_l2(h[0], ref) <= REL_L2_TOL and mismatch(h[0], ref) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - ref)) <= 1e-10 * np.max(np.abs(ref))
    # fused == the separate pass over the source-frame waveform (what the paper's pipeline does)
    th, ph, f = api.few_frame_constants(dev(sky), dev(mu))
    h_src = api.few_waveform(dev(w.t), dev(w.phase), dev(w.amp), dev(w.l), dev(w.m), dev(w.n), th, ph, w.eps, w.t0, w.dt, w.n_samples)
    h2 = api.few_frame_rotate(h_src, f).cpu().numpy()
    assert rel_l2(h2[0], h[0]) <= 1e-13


@pytest.mark.parametrize("cfg,n,t0", [(1, 20_000, 0.0), (2, 3_000, 15_000_000.0)])
def test_waveform_ssb_windows(api, cfg, n, t0):
    w = synth.make_config(cfg, n_samples=n, t0=t0)
    sky, mu = synth.sky_angles(1)
    h, _, keep = run_ssb(api, w, sky, mu)
    ref = ssb_oracle(w, sky, mu, keep)[0]
    assert rel_l2(h[0], ref) <= REL_L2_TOL and mismatch(h[0], ref) <= MISMATCH_TOL
    # the kept set is the oracle's selection at the oracle's own viewing angles: identical (no band)
    th, ph, _ = oracle.frame(*sky[0])
    yp, ym = oracle.ylm_modes(w.l, w.m, th, ph)
    ref_keep, _ = oracle.select_modes(w.amp[0], w.m, yp, ym, w.eps)
    assert np.array_equal(np.asarray(ref_keep), np.asarray(keep[0])), np.setxor1d(ref_keep, keep[0])


def test_waveform_ssb_batch(api):
    w = synth.make_config(3, n_src=5, n_samples=2_500, t0=9_000_000.0)
    sky, mu = synth.sky_angles(5, seed=3)
    h, _, keep = run_ssb(api, w, sky, mu)
    ref = ssb_oracle(w, sky, mu, keep)
    for s in range(w.n_src):
        assert rel_l2(h[s], ref[s]) <= REL_L2_TOL, (s, rel_l2(h[s], ref[s]))
        assert mismatch(h[s], ref[s]) <= MISMATCH_TOL


# ------------------------------------------------------------------------------------------- NEXT-2
def inner_tol(d, h, dt):
    return 1e-10 * 2 * dt * np.linalg.norm(d) * np.linalg.norm(h)


def test_inner_products_standalone_vs_oracle(api):
    rng = np.random.default_rng(21)
    for n_src, N, dt in [(1, 1, 10.0), (2, 2047, 15.0), (3, 2048 * 3 + 5, 10.0), (1, 300_001, 5.0)]:
        d = rng.normal(size=(n_src, N)) + 1j * rng.normal(size=(n_src, N))
        h = rng.normal(size=(n_src, N)) + 1j * rng.normal(size=(n_src, N))
        got = api.few_inner_products(dev(d), dev(h), dt).cpu().numpy()
        got2 = api.few_inner_products(dev(d), dev(h), dt).cpu().numpy()
        assert np.array_equal(got, got2)                                   # fixed reduction order
        for s in range(n_src):
            ref = oracle.inner(d[s], h[s], dt)
            sc = 2 * dt * np.linalg.norm(d[s]) * np.linalg.norm(h[s])
            assert abs(got[s, 0] - ref[0]) <= 1e-14 * sc and abs(got[s, 1] - ref[1]) <= 1e-14 * sc
            assert abs(got[s, 2] - ref[2]) <= 1e-14 * ref[2]
    z = api.few_inner_products(dev(np.zeros((2, 0), np.complex128)), dev(np.zeros((2, 0), np.complex128)), 10.0).cpu().numpy()
    assert np.array_equal(z, np.zeros((2, 3)))


@pytest.mark.parametrize("cfg,n,t0", [(0, 4096, 0.0), (1, 30_000, 1_000_000.0), (0, 5000, -3000.0)])
def test_fused_inner_products_vs_oracle(api, cfg, n, t0):
    """<d|h> and <h|h> reduced inside the summation kernel, against O6 applied to the oracle's waveform.  The third case puts
    samples before t_0 and after t_last (h = 0 there, R12): they must contribute nothing."""
    w = synth.make_config(cfg, n_samples=n, t0=t0)
    sky, mu = synth.sky_angles(1)
    noise = synth.data_stream((1, n), seed=cfg)
    h_gpu, inner, keep = run_ssb(api, w, sky, mu, d=None, want_inner=True)
    ref = ssb_oracle(w, sky, mu, keep)[0]
    d = noise * (0.5 * np.std(ref.real)) + ref[None]                        # data = signal + noise
    h2, inner, keep2 = run_ssb(api, w, sky, mu, d=d)
    assert np.array_equal(h2, h_gpu) and all(np.array_equal(a, b) for a, b in zip(keep, keep2))
    r = oracle.inner(d[0], ref, w.dt)
    assert abs(inner[0, 0] - r[0]) <= inner_tol(d[0], ref, w.dt), (inner[0], r)
    assert abs(inner[0, 1] - r[1]) <= inner_tol(d[0], ref, w.dt)
    assert abs(inner[0, 2] - r[2]) <= 2e-10 * r[2]
    # in practice: rounding level
    assert abs(inner[0, 0] - r[0]) <= 1e-12 * 2 * w.dt * np.linalg.norm(d[0]) * np.linalg.norm(ref)
    # h never written: same three numbers, bit for bit; and the run is reproducible
    _, inner_only, _ = run_ssb(api, w, sky, mu, d=d, want_h=False)
    assert np.array_equal(inner_only, inner)
    # fused == separate reduction over the stored GPU waveform, to rounding
    sep = api.few_inner_products(dev(d), dev(h2), w.dt).cpu().numpy()
    assert np.max(np.abs(sep[0] - inner[0])) <= 1e-13 * 2 * w.dt * np.linalg.norm(d[0]) * np.linalg.norm(ref)
    # without data only <h|h> is formed
    _, hh_only, _ = run_ssb(api, w, sky, mu, d=None, want_inner=True, want_h=False)
    assert hh_only[0, 0] == 0.0 and hh_only[0, 1] == 0.0 and hh_only[0, 2] == inner[0, 2]
    # Eq. (15) and Eq. (17) from the three sums
    dd = oracle.inner(d[0], d[0], w.dt)[2]
    lnL = -0.5 * (dd - 2 * inner[0, 0] + inner[0, 2])
    lnL_ref = -0.5 * oracle.inner(d[0] - ref, d[0] - ref, w.dt)[2]
    assert abs(lnL - lnL_ref) <= 1e-9 * abs(lnL_ref)
    ov = inner[0, 0] / math.sqrt(dd * inner[0, 2])
    assert abs(ov - oracle.overlap(d[0], ref, w.dt)) <= 1e-12


def test_fused_inner_products_batch(api):
    w = synth.make_config(3, n_src=4, n_samples=3_000, t0=5_000_000.0)
    sky, mu = synth.sky_angles(4, seed=7)
    d = synth.data_stream((4, 3_000), seed=9)
    h, inner, keep = run_ssb(api, w, sky, mu, d=d)
    ref = ssb_oracle(w, sky, mu, keep)
    for s in range(4):
        r = oracle.inner(d[s], ref[s], w.dt)
        assert abs(inner[s, 0] - r[0]) <= inner_tol(d[s], ref[s], w.dt) and abs(inner[s, 2] - r[2]) <= 2e-10 * r[2]


# ------------------------------------------------------------------------------------------- NEXT-3
def direct_case(api, l, m, n, phase, amp, theta, phi, scale=None, factor=None):
    """amp [n_src, N, K], phase [n_src, N, 2] -> (gpu h, oracle h) per source."""
    n_src = amp.shape[0]
    yp, ym = api.few_ylm_modes(dev(theta), dev(phi), dev(l), dev(m))
    h = api.few_sum_direct(dev(amp), dev(phase), dev(l), dev(m), dev(n), yp, ym, scale=None if scale is None else dev(scale),
                           factor=None if factor is None else dev(factor)).cpu().numpy()
    api.few_device_status()
    refs = []
    for s in range(n_src):
        ryp, rym = oracle.ylm_modes(l, m, float(theta[s]), float(phi[s]))
        r = oracle.sum_direct(amp[s], phase[s], l, m, n, ryp, rym, scale=1.0 if scale is None else float(scale[s]))
        refs.append(r if factor is None else oracle.frame_apply(r, complex(factor[s])))
    return h, refs


@pytest.mark.parametrize("N,t_start", [(300, 0.0), (129, 25_000_000.0)])
def test_direct_full_grid_vs_oracle(api, N, t_start):
    """All 3843 modes of the Schwarzschild grid in natural order at dense samples (the slow model's summation);
    the second window sits late in the year where the phases are ~2e5 rad."""
    l, m, n, phase, amp = synth.dense_trajectory(N, t_start=t_start)
    h, refs = direct_case(api, l, m, n, phase[None], amp[None], np.array([0.7]), np.array([1.1]))
    assert rel_l2(h[0], refs[0]) <= REL_L2_TOL and mismatch(h[0], refs[0]) <= MISMATCH_TOL
    assert np.max(np.abs(h[0] - refs[0])) <= 1e-10 * np.max(np.abs(refs[0]))
    assert rel_l2(h[0], refs[0]) <= 1e-12                      # in practice: rounding level


@pytest.mark.parametrize("K,order", [(1, "natural"), (17, "natural"), (33, "reverse"), (200, "random"), (554, "gaps")])
def test_direct_mode_lists_and_ragged_chunks(api, K, order):
    """Ragged last chunk (K not a multiple of 16), descending and shuffled lists (every mode restarts E), lists with gaps in n."""
    l, m, n, phase, amp = synth.dense_trajectory(257, t_start=12_000_000.0, seed=K)
    rng = np.random.default_rng(K)
    if order == "gaps":
        idx = np.sort(rng.choice(len(l), K, replace=False))
    else:
        idx = np.arange(900, 900 + K)
        if order == "reverse": idx = idx[::-1]
        if order == "random": idx = rng.permutation(len(l))[:K]
    idx = np.ascontiguousarray(idx)
    h, refs = direct_case(api, l[idx], m[idx], n[idx], phase[None], np.ascontiguousarray(amp[:, idx])[None], np.array([2.1]),
                          np.array([4.0]))
    assert rel_l2(h[0], refs[0]) <= REL_L2_TOL and mismatch(h[0], refs[0]) <= MISMATCH_TOL
    assert rel_l2(h[0], refs[0]) <= 1e-12


def test_direct_batch_scale_factor_and_edges(api):
    n_src, N = 3, 130
    parts = [synth.dense_trajectory(N, seed=s, t_start=1e6 * s, l_max=4, n_max=5) for s in range(n_src)]
    l, m, n = parts[0][:3]
    phase = np.stack([p[3] for p in parts]); amp = np.stack([p[4] for p in parts])
    theta = np.array([0.3, 1.5, 3.0]); phi = np.array([0.0, 2.0, 5.0])
    scale = np.array([1.0, 0.25, 3.0]); factor = np.array([1j, -0.6 + 0.8j, 2.0 + 0j])
    h, refs = direct_case(api, l, m, n, phase, amp, theta, phi, scale=scale, factor=factor)
    for s in range(n_src):
        assert rel_l2(h[s], refs[s]) <= 1e-12
    # a single source gives the same bits as inside the batch
    h1, _ = direct_case(api, l, m, n, phase[1:2], amp[1:2], theta[1:2], phi[1:2], scale=scale[1:2], factor=factor[1:2])
    assert np.array_equal(h1[0], h[1])
    # empty output, bad modes
    yp, ym = api.few_ylm_modes(dev(theta), dev(phi), dev(l), dev(m))
    e = api.few_sum_direct(dev(np.zeros((3, 0, len(l)), np.complex128)), dev(np.zeros((3, 0, 2))), dev(l), dev(m), dev(n), yp, ym)
    assert e.shape == (3, 0)
    bad_m = m.copy(); bad_m[3] = -1
    api.few_sum_direct(dev(amp), dev(phase), dev(l), dev(bad_m), dev(n), yp, ym)
    assert api.few_device_status(raise_on_error=False) != 0


def test_direct_equals_interpolated_on_dense_spline_values(api):
    """Cross-check of the two summation modules on the GPU: the interpolated path's waveform equals the direct sum fed with the
    oracle's splines evaluated at every sample (amplitudes FP64, phases rounded to FP64: agreement to |m Phi| 2^-53)."""
    w = synth.make_config(0)
    h_int = api.few_waveform(dev(w.t), dev(w.phase), dev(w.amp), dev(w.l), dev(w.m), dev(w.n), dev(w.theta), dev(w.phi), 0.0, w.t0,
                             w.dt, 1500).cpu().numpy()[0]
    ca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[0], w.phase[0])
    ti = w.t0 + np.arange(1500) * w.dt
    k = np.clip(np.searchsorted(w.t[0], ti, side="right") - 1, 0, w.n_t - 2)
    dx = ti - w.t[0][k]
    c = ca[k]
    val = ((c[:, 3] * dx[:, None] + c[:, 2]) * dx[:, None] + c[:, 1]) * dx[:, None] + c[:, 0]
    A = np.ascontiguousarray(val[:, 0::2] + 1j * val[:, 1::2])
    dxl = dx.astype(np.longdouble)[:, None]; cpk = cp[k]
    ph = (((cpk[:, 3] * dxl + cpk[:, 2]) * dxl + cpk[:, 1]) * dxl + cpk[:, 0]).astype(np.float64)
    yp, ym = api.few_ylm_modes(dev(w.theta), dev(w.phi), dev(w.l), dev(w.m))
    h_dir = api.few_sum_direct(dev(A[None]), dev(ph[None]), dev(w.l), dev(w.m), dev(w.n), yp, ym).cpu().numpy()[0]
    assert rel_l2(h_dir, h_int) <= 1e-12


# ------------------------------------------------------------------------------------------- NEXT-4 (summation part)
def kerr_gpu_and_oracle(api, w, keep=None, theta=0.7, phi=1.1):
    """S0 + S1 (amplitudes FP64, three phases double-double) + Kerr-shaped S3 on the GPU; O2 + O1 + O8 on the CPU."""
    th, ph = dev(np.array([theta])), dev(np.array([phi]))
    yp, ym = api.few_ylm_modes(th, ph, dev(w.l), dev(w.m))
    coef = api.few_spline_fit(dev(w.t), dev(w.amp))
    cdd = api.few_spline_fit_dd(dev(w.t), dev(w.phase))
    assert cdd.shape[3] == 3
    kd = nk = None
    if keep is not None:
        pad = np.full((1, w.n_modes), -1, np.int32); pad[0, : len(keep)] = keep
        kd, nk = dev(pad), dev(np.array([len(keep)], np.int32))
    h, _ = api.few_sum_waveform_kerr(dev(w.t), coef, cdd, dev(w.l), dev(w.m), dev(w.k), dev(w.n), kd, nk, yp, ym, w.t0, w.dt, w.n_samples)
    api.few_device_status()
    ryp, rym = oracle.ylm_modes(w.l, w.m, theta, phi)
    ca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[0], w.phase[0])
    ref = oracle.sum_waveform_kerr(w.t[0], ca, cp, w.l, w.m, w.k, w.n, keep, ryp, rym, w.t0, w.dt, w.n_samples)
    return h.cpu().numpy()[0], ref


def test_kerr_sum_small_all_modes(api):
    w = synth.make_kerr(n_samples=3000, n_t=30, l_max=4, k_max=2, n_max=3, t0=20_000_000.0)
    h, ref = kerr_gpu_and_oracle(api, w)
    assert rel_l2(h, ref) <= REL_L2_TOL and mismatch(h, ref) <= MISMATCH_TOL
    assert np.max(np.abs(h - ref)) <= 1e-10 * np.max(np.abs(ref))


def test_kerr_sum_full_grid_sorted_in_workspace(api):
    """All 42 273 modes of the Kerr-shaped grid: the kept list (65 536 padded) exceeds the plan kernel's shared memory, so the
    ordering runs through the workspace; 7381 (m, k, n) runs of E."""
    w = synth.make_kerr(n_samples=700, t0=15_000_000.0)
    assert w.n_modes == 42273
    h, ref = kerr_gpu_and_oracle(api, w)
    assert rel_l2(h, ref) <= REL_L2_TOL and mismatch(h, ref) <= MISMATCH_TOL


@pytest.mark.parametrize("n_keep", [5000, 20000])
def test_kerr_sum_kept_subsets(api, n_keep):
    """Random kept subsets with gaps in k and n: 5000 sorts in shared memory, 20 000 (32 768 padded) through the workspace."""
    w = synth.make_kerr(n_samples=600, t0=3_000_000.0)
    keep = np.sort(np.random.default_rng(n_keep).choice(w.n_modes, n_keep, replace=False)).astype(np.int32)
    h, ref = kerr_gpu_and_oracle(api, w, keep=keep, theta=2.0, phi=5.0)
    assert rel_l2(h, ref) <= REL_L2_TOL and mismatch(h, ref) <= MISMATCH_TOL


def test_kerr_sum_reduces_to_schwarzschild_path(api):
    """n_phase = 2, k = NULL gives few_sum_waveform's bits; k = 0 with three phases gives the same waveform to rounding."""
    w = synth.make_config(1, n_samples=4000, t0=9_000_000.0)
    g = dict(t=dev(w.t), l=dev(w.l), m=dev(w.m), n=dev(w.n))
    yp, ym = api.few_ylm_modes(dev(w.theta), dev(w.phi), g["l"], g["m"])
    coef = api.few_spline_fit(g["t"], dev(w.amp))
    c2 = api.few_spline_fit_dd(g["t"], dev(w.phase))
    h_ref = api.few_sum_waveform(g["t"], coef, c2, g["l"], g["m"], g["n"], None, None, yp, ym, w.t0, w.dt, w.n_samples).cpu().numpy()
    h2, _ = api.few_sum_waveform_kerr(g["t"], coef, c2, g["l"], g["m"], None, g["n"], None, None, yp, ym, w.t0, w.dt, w.n_samples)
    assert np.array_equal(h2.cpu().numpy(), h_ref)
    ph3 = np.stack([w.phase[..., 0], 0.77 * w.phase[..., 0], w.phase[..., 1]], axis=-1)
    c3 = api.few_spline_fit_dd(g["t"], dev(ph3))
    k0 = dev(np.zeros(w.n_modes, np.int32))
    h3, _ = api.few_sum_waveform_kerr(g["t"], coef, c3, g["l"], g["m"], k0, g["n"], None, None, yp, ym, w.t0, w.dt, w.n_samples)
    assert rel_l2(h3.cpu().numpy()[0], h_ref[0]) <= 1e-13
    bad = np.zeros(w.n_modes, np.int32); bad[5] = 64
    api.few_sum_waveform_kerr(g["t"], coef, c3, g["l"], g["m"], dev(bad), g["n"], None, None, yp, ym, w.t0, w.dt, 16)
    assert api.few_device_status(raise_on_error=False) != 0


# ------------------------------------------------------------------------------------------- NEXT-4 (selection part)
def _check_keep(keep_gpu, nk_gpu, ref_keep, margin):
    k = keep_gpu[: int(nk_gpu)]
    assert np.all(np.diff(k) > 0) and np.all(keep_gpu[int(nk_gpu):] == -1)
    bad = sorted(set(k.tolist()) ^ set(ref_keep.tolist()))        # identical sets: no band (margins are generic here)
    assert not bad, f"kept sets differ: {bad[:10]} ({len(k)} vs {len(ref_keep)}; margins {[margin[j] for j in bad[:10]]})"


@pytest.mark.parametrize("eps", [1e-5, 1e-2, 0.7])
def test_kerr_select_rows_of_78507_entries_vs_oracle(api, eps):
    """Rows of the Kerr-shaped grid (42 273 modes + 36 234 mirrors) do not fit any block's registers: the streaming kernel
    recomputes the powers from the amplitudes on every pass of the selection."""
    w = synth.make_kerr(n_samples=8, n_t=24)
    yp, ym = api.few_ylm_modes(dev(w.theta), dev(w.phi), dev(w.l), dev(w.m))
    keep, nk = api.few_select_modes(dev(w.amp), dev(w.m), yp, ym, eps)
    api.few_device_status()
    ref, margin = oracle.select_modes(w.amp[0], w.m, yp[0].cpu().numpy(), ym[0].cpu().numpy(), eps)
    _check_keep(keep[0].cpu().numpy(), nk[0].item(), ref, margin)
    assert 0 < nk[0].item() < w.n_modes


def test_kerr_select_flat_rows_and_ties(api):
    """Equal powers on a long row: the threshold bucket holds far more entries than the fine step sorts, so the 63-step
    select and the 18-bit index select for ties run on streamed keys."""
    n_modes = 20000
    amp = np.ones((1, 3, n_modes), np.complex128)
    m = np.zeros(n_modes, np.int32)
    keep, nk = api.few_select_modes(dev(amp), dev(m), None, None, 0.25)
    api.few_device_status()
    assert nk.item() == 15000 and np.array_equal(keep[0, :15000].cpu().numpy(), np.arange(15000))
    rng = np.random.default_rng(3)
    amp = rng.uniform(1.0, 1.4, (1, 3, n_modes)) * np.exp(1j * rng.uniform(0, 6.28, (1, 3, n_modes)))
    m = rng.integers(0, 3, n_modes).astype(np.int32)
    keep, nk = api.few_select_modes(dev(amp), dev(m), None, None, 0.1)
    ref, margin = oracle.select_modes(amp[0], m, None, None, 0.1)
    _check_keep(keep[0].cpu().numpy(), nk[0].item(), ref, margin)


def test_kerr_whole_path_select_fit_sum(api):
    """S0 + S2 (streamed rows) + S1 + Kerr-shaped S3 chained on the device against O2 + O3 + O1 + O8."""
    w = synth.make_kerr(n_samples=500, n_t=24, t0=9_000_000.0)
    yp, ym = api.few_ylm_modes(dev(w.theta), dev(w.phi), dev(w.l), dev(w.m))
    keep, nk = api.few_select_modes(dev(w.amp), dev(w.m), yp, ym, 1e-4)
    coef = api.few_spline_fit(dev(w.t), dev(w.amp))
    cdd = api.few_spline_fit_dd(dev(w.t), dev(w.phase))
    h, _ = api.few_sum_waveform_kerr(dev(w.t), coef, cdd, dev(w.l), dev(w.m), dev(w.k), dev(w.n), keep, nk, yp, ym, w.t0, w.dt, w.n_samples)
    api.few_device_status()
    kept = keep[0, : nk[0].item()].cpu().numpy()
    ryp, rym = oracle.ylm_modes(w.l, w.m, float(w.theta[0]), float(w.phi[0]))
    ca = oracle.spline_fit(w.t[0], np.ascontiguousarray(w.amp[0]).view(np.float64))
    cp = oracle.spline_fit_ext(w.t[0], w.phase[0])
    ref = oracle.sum_waveform_kerr(w.t[0], ca, cp, w.l, w.m, w.k, w.n, kept, ryp, rym, w.t0, w.dt, w.n_samples)
    hh = h.cpu().numpy()[0]
    assert rel_l2(hh, ref) <= REL_L2_TOL and mismatch(hh, ref) <= MISMATCH_TOL
    # the single C call (few_waveform_kerr: fits on side streams, nothing read back) gives the same bits
    keep2 = torch.empty_like(keep); nk2 = torch.empty_like(nk)
    h2 = api.few_waveform_kerr(dev(w.t), dev(w.phase), dev(w.amp), dev(w.l), dev(w.m), dev(w.k), dev(w.n), dev(w.theta), dev(w.phi),
                               1e-4, w.t0, w.dt, w.n_samples, keep_idx=keep2, n_keep=nk2)
    api.few_device_status()
    assert torch.equal(keep2, keep) and torch.equal(nk2, nk) and torch.equal(h2, h)
