"""GPU parity of the ragged-batch entry points (include/few.h "Ragged batches"; adaptive trajectories give
every source its own number of sparse points and its own end time).  The oracle has no ragged mode: it is looped over the
sources, each cut to its own length (synth.source_of).  The padding of the batch arrays is NaN, so a read of it shows.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2104_04582_b200 import synth  # noqa: E402

REL_L2_TOL = 1e-10
MISMATCH_TOL = 1e-12
SENTINEL = 12345.0


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


def gpu_inputs(w):
    return dict(t=dev(w.t), phase=dev(w.phase), amp=dev(w.amp), l=dev(w.l), m=dev(w.m), n=dev(w.n), theta=dev(w.theta),
                phi=dev(w.phi), cnt=dev(w.n_t_src))


@pytest.fixture(scope="module")
def batch():
    return synth.make_ragged()          # counts 40, 80, 137, 80, 40, 137


def test_ragged_stages_vs_oracle(api, batch):
    """S1, S1 (double-double), S2 and S3 one by one, each against the oracle run on the source alone."""
    w = batch
    g = gpu_inputs(w)
    n_src, n_t, n_modes = w.amp.shape
    # ---- S1: rows of a source's own segments match, the rows of the padding keep the sentinel
    out = torch.full((n_src, n_t - 1, 4, 2 * n_modes), SENTINEL, dtype=torch.float64, device="cuda")
    coef = api.few_spline_fit_ragged(g["t"], g["amp"], g["cnt"], out=out)
    out_dd = torch.full((n_src, n_t - 1, 4, 2, 2), SENTINEL, dtype=torch.float64, device="cuda")
    coef_dd = api.few_spline_fit_dd_ragged(g["t"], g["phase"], g["cnt"], out=out_dd)
    api.few_device_status()
    c, cdd = coef.cpu().numpy(), coef_dd.cpu().numpy()
    for s in range(n_src):
        k = int(w.n_t_src[s])
        one = synth.source_of(w, s)
        y = np.ascontiguousarray(one.amp[0]).view(np.float64)
        ref = oracle.spline_fit(one.t[0], y)
        assert np.all(c[s, k - 1:] == SENTINEL) and np.all(cdd[s, k - 1:] == SENTINEL)
        assert np.all(np.isfinite(c[s, :k - 1])) and np.all(np.isfinite(cdd[s, :k - 1]))
        assert np.array_equal(c[s, :k - 1, 0], y[:-1])
        h = np.diff(one.t[0])[:, None]
        scale = np.max(np.abs(y), axis=0)[None, :]
        for p in (1, 2, 3):
            assert float(np.max(np.abs(c[s, :k - 1, p] - ref[:, p]) * h ** p / scale)) <= 5e-14      # the bar of test_gpu_parity S1
        ref_dd = oracle.spline_fit_ext(one.t[0], one.phase[0])
        got = cdd[s, :k - 1, ..., 0].astype(np.longdouble) + cdd[s, :k - 1, ..., 1].astype(np.longdouble)
        x = np.diff(one.t[0]).astype(np.longdouble)[:, None]
        pg = got[:, 0] + x * (got[:, 1] + x * (got[:, 2] + x * got[:, 3]))
        pr = ref_dd[:, 0] + x * (ref_dd[:, 1] + x * (ref_dd[:, 2] + x * ref_dd[:, 3]))
        assert float(np.max(np.abs(pg - pr))) <= 2e-12
    # ---- S2: the union runs over the source's own steps only; sets identical to the oracle's
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    for eps in (1e-5, 1e-2):
        keep, nk = api.few_select_modes_ragged(g["amp"], g["m"], yp, ym, g["cnt"], eps)
        api.few_device_status()
        for s in range(n_src):
            one = synth.source_of(w, s)
            ref, _ = oracle.select_modes(one.amp[0], w.m, yp[s].cpu().numpy(), ym[s].cpu().numpy(), eps)
            kk = keep[s].cpu().numpy()
            assert np.array_equal(kk[: nk[s].item()], ref) and np.all(kk[nk[s].item():] == -1)
    # ---- S3 on the coefficients above (their padding rows still hold the sentinel: never read)
    hh, _ = api.few_sum_waveform_ragged(g["t"], g["cnt"], coef, coef_dd, g["l"], g["m"], None, g["n"], keep, nk, yp, ym,
                                        w.t0, w.dt, w.n_samples)
    api.few_device_status()
    hh = hh.cpu().numpy()
    assert np.all(np.isfinite(hh.view(np.float64)))
    for s in range(n_src):
        one = synth.source_of(w, s)
        ryp, rym = oracle.ylm_modes(w.l, w.m, float(w.theta[s]), float(w.phi[s]))
        ca = oracle.spline_fit(one.t[0], np.ascontiguousarray(one.amp[0]).view(np.float64))
        cp = oracle.spline_fit_ext(one.t[0], one.phase[0])
        ref = oracle.sum_waveform(one.t[0], ca, cp, w.l, w.m, w.n, keep[s, : nk[s].item()].cpu().numpy(), ryp, rym, w.t0, w.dt,
                                  w.n_samples)
        assert rel_l2(hh[s], ref) <= REL_L2_TOL and mismatch(hh[s], ref) <= MISMATCH_TOL


def test_ragged_whole_path_vs_oracle(api, batch):
    w = batch
    g = gpu_inputs(w)
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32, device="cuda")
    nk = torch.empty((w.n_src,), dtype=torch.int32, device="cuda")
    h = api.few_waveform_ragged(g["t"], g["cnt"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0,
                                w.dt, w.n_samples, keep_idx=keep, n_keep=nk)
    api.few_device_status()
    h = h.cpu().numpy()
    assert np.all(np.isfinite(h.view(np.float64)))
    ends_inside = 0
    for s in range(w.n_src):
        one = synth.source_of(w, s)
        ref = oracle.waveform(one)[0]
        assert rel_l2(h[s], ref) <= REL_L2_TOL and mismatch(h[s], ref) <= MISMATCH_TOL, s
        assert np.max(np.abs(h[s] - ref)) <= 1e-10 * np.max(np.abs(ref))
        # after the source's last knot the waveform is exactly zero (R12), before it it is not
        i_end = int(np.floor((one.t[0, -1] - w.t0) / w.dt)) + 1
        if i_end < w.n_samples:
            ends_inside += 1
            assert np.all(h[s, i_end + 1:] == 0) and np.all(ref[i_end + 1:] == 0)
            assert np.any(h[s, i_end - 200:i_end - 1] != 0)
        # the same source as a uniform one-source call: the same bits (a source's tiles start at its own segment boundaries)
        g1 = {k: dev(getattr(one, k)) for k in ("t", "phase", "amp", "theta", "phi")}
        keep1 = torch.empty((1, w.n_modes), dtype=torch.int32, device="cuda")
        nk1 = torch.empty((1,), dtype=torch.int32, device="cuda")
        h1 = api.few_waveform(g1["t"], g1["phase"], g1["amp"], g["l"], g["m"], g["n"], g1["theta"], g1["phi"], w.eps, w.t0, w.dt,
                              w.n_samples, keep_idx=keep1, n_keep=nk1)
        assert nk1.item() == nk[s].item() and torch.equal(keep1[0], keep[s])
        assert np.array_equal(h1.cpu().numpy()[0].view(np.float64), h[s].view(np.float64))
    assert ends_inside >= 3                 # the batch does contain sources that end inside the window


def test_ragged_with_full_counts_is_the_uniform_call(api):
    w = synth.make_config(3, n_src=3, n_samples=20_000)
    g = {k: dev(getattr(w, k)) for k in ("t", "phase", "amp", "l", "m", "n", "theta", "phi")}
    cnt = dev(np.full(w.n_src, w.n_t, np.int32))
    a = api.few_waveform(g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt, w.n_samples)
    b = api.few_waveform_ragged(g["t"], cnt, g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt,
                                w.n_samples)
    api.few_device_status()
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))


def test_ragged_host_path_equals_device_path(api, batch):
    w = batch
    g = gpu_inputs(w)
    h = api.few_waveform_ragged(g["t"], g["cnt"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0,
                                w.dt, w.n_samples)
    api.few_device_status()
    cpu = lambda a, dt=None: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).pin_memory()      # noqa: E731
    keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32).pin_memory()
    nk = torch.empty((w.n_src,), dtype=torch.int32).pin_memory()
    hh = api.few_waveform_host_ragged(cpu(w.t), cpu(w.n_t_src), cpu(w.phase), cpu(w.amp), cpu(w.l), cpu(w.m), cpu(w.n), cpu(w.theta),
                                      cpu(w.phi), w.eps, w.t0, w.dt, w.n_samples, keep_idx=keep, n_keep=nk)
    assert np.array_equal(hh.numpy().view(np.float64), h.cpu().numpy().view(np.float64))
    assert int(nk.min()) > 0


@pytest.mark.parametrize("bad", [3, 138, -1])
def test_ragged_bad_count_is_reported(api, batch, bad):
    w = batch
    g = gpu_inputs(w)
    cnt = w.n_t_src.copy()
    cnt[1] = bad
    # The workspace starts as 0xFF bytes (NaN as doubles, -1 / huge as counts): whatever the kernels read must have been written
    # in this call.  few.h promises "outputs unspecified but in bounds" for a bad count: no fault, and here no NaN either, since
    # the bad source is treated as a 4-knot source by every kernel alike.
    n_src, n_t, n_modes = g["amp"].shape
    ws = torch.full((max(api.few_waveform_workspace(n_src, n_t, n_modes, 2_000), 256),), 0xFF, dtype=torch.uint8, device="cuda:0")
    h = api.few_waveform_ragged(g["t"], dev(cnt), g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt,
                                2_000, workspace=ws)
    torch.cuda.synchronize()                                                 # raises if a kernel faulted
    assert bool(torch.isfinite(torch.view_as_real(h)).all())
    assert api.few_device_status(raise_on_error=False) == -2                 # FEW_ERR_TOO_FEW_POINTS (FEW_DEV_BAD_COUNT)
    assert api.few_device_status(raise_on_error=False) == 0


def test_host_path_refuses_bad_arguments_before_copying(api, batch):
    """few_waveform_host(_ragged) checks what it can from the arguments alone -- the size limits and, since they are on the host,
    the per-source knot counts -- before it enqueues a single copy, so that a refused call leaves nothing in flight that still
    reads the caller's buffers.  The context stays usable afterwards."""
    w = batch
    cpu = lambda a, dt=None: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).pin_memory()      # noqa: E731
    args = [cpu(w.t), None, cpu(w.phase), cpu(w.amp), cpu(w.l), cpu(w.m), cpu(w.n), cpu(w.theta), cpu(w.phi), w.eps, w.t0, w.dt, 2_000]
    for bad in (3, 138, -1):
        cnt = w.n_t_src.copy()
        cnt[1] = bad
        args[1] = cpu(cnt)
        with pytest.raises(api.FewError) as e:
            api.few_waveform_host_ragged(*args)
        assert e.value.code == -2                                            # FEW_ERR_TOO_FEW_POINTS
    n_t = 737                                                                # FEW_MAX_NT_SPLINE + 1
    z = lambda *shape, dt=torch.float64: torch.zeros(shape, dtype=dt).pin_memory()                # noqa: E731
    with pytest.raises(api.FewError) as e:
        api.few_waveform_host(z(1, n_t), z(1, n_t, 2), z(1, n_t, 3, dt=torch.complex128), cpu(w.l[:3]), cpu(w.m[:3]), cpu(w.n[:3]),
                              z(1), z(1), 0.0, 0.0, 10.0, 100)
    assert e.value.code == -7                                                # FEW_ERR_LIMIT
    with pytest.raises(api.FewError) as e:                                   # dt = 0
        api.few_waveform_host_ragged(*(args[:1] + [cpu(w.n_t_src)] + args[2:11] + [0.0, 2_000]))
    assert e.value.code == -1
    assert api.few_device_status(raise_on_error=False) == 0                  # nothing ran, nothing was flagged
    args[1] = cpu(w.n_t_src)
    hh = api.few_waveform_host_ragged(*args)                                 # and the next good call is unaffected
    g = gpu_inputs(w)
    h = api.few_waveform_ragged(g["t"], g["cnt"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0,
                                w.dt, 2_000)
    assert np.array_equal(hh.numpy().view(np.float64), h.cpu().numpy().view(np.float64))
