"""Zone sharding for N > 1 GPUs: zones are independent,
so ranks take contiguous zone ranges with no data-path collective; only timings/counters are
reduced.  Pure index arithmetic -- no method arithmetic here."""
from __future__ import annotations


def shard_range(nz: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) of `nz` zones for `rank` of `world` (sizes differ by <= 1)."""
    if world < 1 or not (0 <= rank < world) or nz < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(nz, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_workload(rho, T, X, rank: int, world: int):
    """Slices of the SoA arrays (rho[nz], T[nz], X[N, nz]) owned by `rank`."""
    lo, hi = shard_range(rho.shape[0], rank, world)
    return rho[lo:hi], T[lo:hi], X[:, lo:hi], (lo, hi)
