"""Multi-GPU sharding of the hot path: the path partitions with NO data-path collective.

Every dense sample is independent given the (small) spline coefficients, and every source of a batch is independent
(PAPER.md:155-159 per-sample combine; PAPER.md:330, 386 many independent waveforms per MCMC step).  So ranks take
 - whole sources of a batch (`shard_sources`), or
 - contiguous sample ranges of one long waveform (`shard_samples`): each rank repeats the cheap S0-S2-S1 steps on the
   sparse inputs and sums only its own range [i0, i0 + n) by passing t0 + i0*dt as its t0.
Pure host logic (no kernels, no torch): `bench.py --gpus N --config 3|4` shards the GPU path with it (one process per GPU),
and `tests/test_abi_and_host.py` covers it with a world_size-2 gloo run on CPU.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int, align: int = 1) -> tuple[int, int]:
    """Contiguous block [start, start+count) of n items for `rank` of `world`; blocks are multiples of `align`
    (except the last), differ by at most one `align` unit, cover [0, n) exactly and are ordered by rank."""
    if not (0 <= rank < world) or n < 0 or align < 1:
        raise ValueError("need 0 <= rank < world, n >= 0, align >= 1")
    units = (n + align - 1) // align
    base, extra = divmod(units, world)
    u0 = rank * base + min(rank, extra)
    u1 = u0 + base + (1 if rank < extra else 0)
    start, stop = min(u0 * align, n), min(u1 * align, n)
    return start, stop - start


def shard_sources(n_src: int, rank: int, world: int) -> tuple[int, int]:
    return shard_range(n_src, rank, world)


def shard_samples(n_samples: int, rank: int, world: int, align: int = 256) -> tuple[int, int]:
    """Sample range of a rank.  Any split gives the same bits as the unsharded call (every sample's arithmetic depends on
    its own t_i only; the kernel re-clips its tiles to each call's range), so `align` is cosmetic: it keeps shard
    boundaries on multiples of 256 samples so that the ranks' stores start on 4 KB boundaries of h."""
    return shard_range(n_samples, rank, world, align)


def shard_t0(t0: float, dt: float, i0: int) -> float:
    """t0 of a sample shard.  Exact (hence bit-identical waveforms across world sizes) when t0 and dt are integers below
    2^53 / n_samples, which holds for every BASELINE config (t0 = 0, dt = 10 or 15 s)."""
    return t0 + float(i0) * dt
