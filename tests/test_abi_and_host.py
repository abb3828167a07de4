"""No-GPU checks: the C-ABI library builds, loads and exports every symbol include/few.h declares; host-only entry points
behave; the sharding logic covers the work exactly; a world_size-2 gloo run reassembles sharded oracle waveforms."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2104_04582_b200 import build
    return ctypes.CDLL(build.build())


def declared_functions():
    src = open(os.path.join(ROOT, "include", "few.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(few_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert {"few_spline_fit", "few_select_modes", "few_sum_waveform", "few_waveform", "few_waveform_host"} <= set(names)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in few.h but not exported"
    from paper_2104_04582_b200 import api  # noqa: F401  (binding imports without a GPU)
    assert sorted(api.SYMBOLS) == names


def test_sass_is_sm100a(lib):
    from paper_2104_04582_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.SO], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out


def test_host_entry_points(lib):
    import oracle
    lib.few_ylm.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_double)]
    out = (ctypes.c_double * 2)()
    for l in range(2, 11):
        for m in range(-l, l + 1):
            assert lib.few_ylm(l, m, 0.7, 1.1, out) == 0
            assert abs(complex(out[0], out[1]) - oracle.ylm(l, m, 0.7, 1.1)) <= 1e-14
    assert lib.few_ylm(3, 4, 0.7, 1.1, out) == -4 and lib.few_ylm(1, 0, 0.7, 1.1, out) == -4
    lib.few_strerror.restype = ctypes.c_char_p
    assert b"TOO_FEW_POINTS" in lib.few_strerror(-2)
    assert lib.few_version() == 100
    lib.few_select_modes_workspace.restype = ctypes.c_size_t
    lib.few_sum_waveform_workspace.restype = ctypes.c_size_t
    lib.few_sum_waveform_workspace.argtypes = [ctypes.c_int] * 3 + [ctypes.c_longlong]
    assert lib.few_select_modes_workspace(1, 100, 3843) > 0
    assert lib.few_sum_waveform_workspace(1, 100, 3843, 1000) >= 99 * 3843 * 64


def test_step_bound_helper_and_workspace_queries(lib):
    """few_max_steps_for_modes counts the distinct (m, k, |n| >> 2) of a mode list; the *_workspace_ex queries shrink with the
    bound and fall back to the default for 0 or for a bound above it (host-only: no GPU needed)."""
    from paper_2104_04582_b200 import synth
    l, m, n = synth.mode_grid()
    i32p = ctypes.POINTER(ctypes.c_int)
    lib.few_max_steps_for_modes.argtypes = [i32p, i32p, i32p, ctypes.c_int]
    ptr = lambda a: np.ascontiguousarray(a, np.int32).ctypes.data_as(i32p)      # noqa: E731
    mm, nn = np.ascontiguousarray(m, np.int32), np.ascontiguousarray(n, np.int32)
    assert lib.few_max_steps_for_modes(ptr(mm), None, ptr(nn), len(mm)) == 88          # 11 m x 8 blocks of four |n|
    brute = len({(int(a), abs(int(b)) >> 2) for a, b in zip(mm, nn)})
    assert brute == 88
    k = np.arange(len(mm), dtype=np.int32) % 3 - 1                                     # a polar index multiplies the runs
    assert lib.few_max_steps_for_modes(ptr(mm), ptr(k), ptr(nn), len(mm)) == len({(int(a), int(c), abs(int(b)) >> 2) for a, b, c in zip(mm, nn, k)})
    assert lib.few_max_steps_for_modes(None, None, ptr(nn), len(mm)) == -1
    for name in ("few_sum_waveform_workspace_ex", "few_waveform_workspace_ex"):
        f = getattr(lib, name)
        f.restype, f.argtypes = ctypes.c_size_t, [ctypes.c_int] * 3 + [ctypes.c_longlong, ctypes.c_int]
        plain = getattr(lib, name[:-3])
        plain.restype, plain.argtypes = ctypes.c_size_t, [ctypes.c_int] * 3 + [ctypes.c_longlong]
        full = plain(64, 80, 3843, 1_051_920)
        assert f(64, 80, 3843, 1_051_920, 0) == full == f(64, 80, 3843, 1_051_920, 100_000)
        assert f(64, 80, 3843, 1_051_920, 88) < 0.35 * full
        assert f(64, 80, 3843, 1_051_920, 40) < f(64, 80, 3843, 1_051_920, 88)


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    ctx = ctypes.c_void_p()
    assert lib.few_create(ctypes.byref(ctx), 0) == -6           # FEW_ERR_CUDA: fails loudly, nothing to fall back to
    from paper_2104_04582_b200 import api
    with pytest.raises(RuntimeError):
        api.context()


def test_shard_ranges_cover_exactly():
    from paper_2104_04582_b200.shard import shard_range, shard_samples, shard_sources
    for n in (0, 1, 7, 64, 255, 256, 257, 3_155_760, 12_623_040):
        for world in (1, 2, 3, 4, 8):
            for align in (1, 256):
                pos = 0
                counts = []
                for r in range(world):
                    s, c = shard_range(n, r, world, align)
                    assert s == pos and c >= 0 and (s % align == 0 or c == 0)
                    pos += c; counts.append(c)
                assert pos == n
                assert max(counts) - min(counts) < 2 * align      # one unit of imbalance + the ragged last unit
    assert shard_sources(64, 3, 8) == (24, 8)
    assert shard_samples(3_155_760, 1, 2) == (1_577_984, 1_577_776)
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_2104_04582_b200 import synth
from paper_2104_04582_b200.shard import shard_samples, shard_sources, shard_t0
dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{sys.argv[2]}", rank=int(sys.argv[3]), world_size=2)
rank, world = dist.get_rank(), dist.get_world_size()
oracle.set_threads(2)
# (a) one waveform sharded by sample range: each rank sums its own range; rank 0 checks the gathered result
w = synth.make_config(0)
i0, cnt = shard_samples(w.n_samples, rank, world)
ws = synth.make_config(0, n_samples=cnt, t0=shard_t0(w.t0, w.dt, i0))
part = torch.from_numpy(np.ascontiguousarray(oracle.waveform(ws)[0]).view(np.float64).copy())
parts = [torch.empty(shard_samples(w.n_samples, r, world)[1] * 2, dtype=torch.float64) for r in range(world)]
dist.all_gather(parts, part) if len({p.numel() for p in parts}) == 1 else [dist.broadcast(parts[r] if r != rank else part, r) for r in range(world)]
parts[rank] = part
full = torch.cat(parts).numpy().view(np.complex128)
ref = oracle.waveform(w)[0]
assert np.array_equal(full, ref), "sample-sharded waveform differs from the unsharded one"
# (b) a batch sharded by source
wb = synth.random_problem(5, n_src=5, n_modes=6, n_samples=64)
s0, sc = shard_sources(wb.n_src, rank, world)
mine = synth.Workload(wb.name, wb.t[s0:s0+sc], wb.phase[s0:s0+sc], wb.amp[s0:s0+sc], wb.l, wb.m, wb.n, wb.theta[s0:s0+sc], wb.phi[s0:s0+sc], wb.t0, wb.dt, wb.n_samples, wb.eps)
hb = oracle.waveform(mine)
assert np.array_equal(hb, oracle.waveform(wb)[s0:s0+sc])
# (d) the split bench.py --gpus N runs on the GPU path (bench.shard_workload: config 3 by source, config 4 by time range), with
# the oracle standing in for few_waveform: the ranks' pieces reassemble to the unsharded result bit for bit
import bench
w3 = synth.random_problem(9, n_src=7, n_modes=5, n_samples=96)
mine = bench.shard_workload(w3, 3, rank, world)
s0, sc = shard_sources(w3.n_src, rank, world)
assert mine.n_src == sc and np.array_equal(mine.t, w3.t[s0:s0+sc]) and mine.n_samples == w3.n_samples
assert np.array_equal(oracle.waveform(mine), oracle.waveform(w3)[s0:s0+sc])
w4 = synth.make_config(0)
mine = bench.shard_workload(w4, 4, rank, world)
i0, cnt = shard_samples(w4.n_samples, rank, world)
assert mine.n_samples == cnt and mine.t0 == w4.t0 + i0 * w4.dt and mine.n_src == 1
assert np.array_equal(oracle.waveform(mine)[0], oracle.waveform(w4)[0][i0:i0+cnt])
assert bench.shard_workload(w4, 1, rank, world) is w4                     # configs 1, 2: replicas
lab3, sc3 = bench.parallelism_label(w3, 3, world); lab4, sc4 = bench.parallelism_label(w4, 4, world)
assert sc3 == sc4 == "strong" and "by source" in lab3 and "time range" in lab4
# (c) bench-style timing reduction: max over ranks
tmax = torch.tensor([float(rank + 1)]); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
assert tmax.item() == 2.0
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
'''


def test_gloo_world2_sharded_paths(tmp_path):
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"; script.write_text(_WORKER)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, str(port), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o


def test_bench_gpus_n_launches_its_own_ranks():
    """`python bench.py --gpus N` without torchrun starts N ranks itself (bench.self_launch): here through --dry-shard, the same
    launch, rendezvous, sharding and reductions with gloo and no GPU.  Two ranks are seen, one line is printed, the shares add up;
    a mismatch between --gpus and an existing WORLD_SIZE, or too few GPUs for a real run, is an error and not a silent 1-GPU run."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    bench = os.path.join(ROOT, "bench.py")
    for cfg, scaling in ((3, "strong"), (4, "strong"), (1, "weak")):
        p = subprocess.run([sys.executable, bench, "--gpus", "2", "--dry-shard", "--config", str(cfg)], capture_output=True, text=True,
                           env=env, timeout=240)
        assert p.returncode == 0, p.stderr
        lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
        assert len(lines) == 1, p.stdout
        d = json.loads(lines[0])
        assert d["n_gpus"] == 2 and d["ranks_seen"] == 2 and d["max_over_ranks"] == 2.0 and d["scaling"] == scaling
        total = sum(d["source_samples_per_rank"])
        assert total == (d["source_samples_total"] if scaling == "strong" else 2 * d["source_samples_total"])
    p = subprocess.run([sys.executable, bench, "--gpus", "4", "--dry-shard"], capture_output=True, text=True,
                       env=dict(env, WORLD_SIZE="2", RANK="0"), timeout=120)
    assert p.returncode != 0 and "WORLD_SIZE" in p.stderr
    import torch
    if torch.cuda.device_count() < 2:
        p = subprocess.run([sys.executable, bench, "--gpus", "2"], capture_output=True, text=True, env=env, timeout=240)
        assert p.returncode != 0 and "needs 2 CUDA devices" in p.stderr and p.stdout.strip() == ""
