"""few_inner_products_static: the inner products for callers that cannot allocate device memory.

Some users of the library may not call an allocator where they need <d|h> and <h|h>: host code in a region where the CUDA
runtime rejects allocation calls, a sampler that gave its whole device-memory budget to a pool it must not grow, a plug-in
handed device pointers by an application that owns the allocator.  few_inner_products is closed to them because it needs a
workspace.  few_inner_products_static takes only d, h and the output and keeps its partial sums in a 512 KB array compiled
into the library (include/few.h, FEW_INNER_STATIC_MAX_CHUNKS).  That array is shared by all calls and is never cleared, so the
thing to prove is that a call does not see what the call before it left behind.

The test therefore makes two calls in a row on one stream -- a large batch first, a smaller and differently shaped one second,
so the second call's slots all hold stale values from the first -- and compares each with few_inner_products on the same
inputs.  Same kernels, same reduction order: the results must be bit-equal, which is inside the 1e-14-of-scale bar that
test_gpu_next.py holds few_inner_products to against the oracle (that bar is asserted too).  It passes run alone in a fresh
process (the first call then does the per-device address look-up) and after the other GPU tests (the look-up may or may not
have happened; the array certainly holds nothing useful).  This file sorts last so that, under `pytest -x`, a failure here
cannot hide the parity tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

SCALE_TOL = 1e-14          # the bar of test_inner_products_standalone_vs_oracle, relative to 2 dt |d| |h|


@pytest.fixture(scope="module")
def api():
    assert torch.cuda.is_available(), "-m gpu tests need a GPU"
    from paper_2104_04582_b200 import api as a
    return a


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).to("cuda:0")


def series(rng, n_src, n):
    return rng.normal(size=(n_src, n)) + 1j * rng.normal(size=(n_src, n))


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(api):
    torch.cuda.set_device(0)
    rng = np.random.default_rng(2104)
    # (n_src, n_samples, dt): 3 x 150 chunks with a ragged last chunk, then 2 x 3 chunks (+1 sample) over the same slots
    cases = [(3, 2048 * 149 + 77, 10.0), (2, 2048 * 3 + 1, 15.0)]
    inputs = [(series(rng, s, n), series(rng, s, n), dt) for s, n, dt in cases]
    on_gpu = [(dev(d), dev(h)) for d, h, _ in inputs]
    outs = [torch.full((s, 3), float("nan"), dtype=torch.float64, device="cuda:0") for s, _, _ in cases]
    # everything the two calls need exists now; between here and the comparison nothing but the entry point under test runs
    api.few_inner_products_static(on_gpu[0][0], on_gpu[0][1], inputs[0][2], outs[0])
    api.few_inner_products_static(on_gpu[1][0], on_gpu[1][1], inputs[1][2], outs[1], use_context=False)   # ctx = NULL is allowed
    torch.cuda.synchronize()
    for (d, h, dt), (dg, hg), out in zip(inputs, on_gpu, outs):
        want = api.few_inner_products(dg, hg, dt).cpu().numpy()            # the existing path, workspace from torch
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got))
        for s in range(d.shape[0]):
            sc = 2 * dt * np.linalg.norm(d[s]) * np.linalg.norm(h[s])
            assert np.max(np.abs(got[s] - want[s])) <= SCALE_TOL * sc, (s, got[s], want[s])
        assert np.array_equal(got, want)                                    # in fact the same bits
    # the first case again, after the smaller one: still the same answer
    again = torch.empty_like(outs[0])
    api.few_inner_products_static(on_gpu[0][0], on_gpu[0][1], inputs[0][2], again)
    assert torch.equal(again, outs[0])


def test_static_scratch_rejects_what_does_not_fit(api):
    torch.cuda.set_device(0)
    out = torch.zeros((1, 3), dtype=torch.float64, device="cuda:0")
    # shapes only: the size check comes before anything touches the GPU, so the buffers can be tiny
    n_too_many = 2048 * api.INNER_STATIC_MAX_CHUNKS + 1                    # one chunk more than the array holds
    d = torch.zeros((1, 1), dtype=torch.complex128, device="cuda:0")        # never dereferenced
    with pytest.raises(api.FewError) as e:
        api._chk(api._lib.few_inner_products_static(None, d.data_ptr(), d.data_ptr(), 1, n_too_many, 10.0, out.data_ptr(), None),
                 "few_inner_products_static")
    assert e.value.code == -7 and "FEW_INNER_STATIC_MAX_CHUNKS" in str(e.value)
    with pytest.raises(api.FewError) as e:                                  # many sources of moderate length
        api._chk(api._lib.few_inner_products_static(None, d.data_ptr(), d.data_ptr(), 17, 2048 * 1024, 10.0, out.data_ptr(), None),
                 "few_inner_products_static")
    assert e.value.code == -7
    assert torch.count_nonzero(out).item() == 0                             # a rejected call writes nothing
    # exactly at the limit is accepted (16 sources x 1024 chunks); zeros in, zeros out
    n = 2048 * 1024
    z = torch.zeros((16, n), dtype=torch.complex128, device="cuda:0")
    o = torch.full((16, 3), float("nan"), dtype=torch.float64, device="cuda:0")
    api.few_inner_products_static(z, z, 10.0, o)
    assert torch.count_nonzero(o).item() == 0
