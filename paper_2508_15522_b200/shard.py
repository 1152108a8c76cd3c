"""Host-side plumbing for running on N GPUs of one node: **replicas only** (SURVEY.md §8(e)).

Replicas and interpolation points are independent units and the coefficient store is replicated read-only on
every GPU, so the data path has no exchange step and no collective.  What crosses ranks is bookkeeping only: the timing (max over
ranks), the count of units processed, and the basin-energy histogram / minima count of the sampling run (a sum).  These helpers are
backend-agnostic (`nccl` on the GPU box, `gloo` in the CPU tests) and hold none of the method's arithmetic.
"""
import numpy as np


def replica_shard(n_total, world, rank):
    """Contiguous balanced split of n_total units over `world` ranks -> (first, count).  Strong-scaling form: the counts differ by at
    most one and add up to n_total."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard request (n_total=%r world=%r rank=%r)" % (n_total, world, rank))
    base, rem = divmod(n_total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def rank_seed(seed, rank, stream=0):
    """Seed of rank `rank`'s own batch in the weak-scaling run (every rank draws a different batch of the same size).  `stream`
    separates the uses (initial placement, velocities, restart generator)."""
    return int(seed) + 1000 * int(rank) + int(stream)


def _dist():
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized()) else None


def max_over_ranks(value, device="cpu"):
    """max over ranks of a python float (device-timed milliseconds); the identity on a single process."""
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(array, device="cpu"):
    """element-wise sum over ranks of a small int64 / float64 numpy array (histogram counts, units processed)."""
    a = np.ascontiguousarray(array)
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return a.copy()
    import torch
    t = torch.from_numpy(a.copy()).to(device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def basin_histogram(energies, e_lo, e_hi, bin_width=0.01):
    """Histogram of relaxed total energies (eV) in `bin_width` bins over [e_lo, e_hi) (config 2's report: 10 meV bins); energies
    outside fall into the first / last bin.  Pure counting: int64[n_bins]."""
    n_bins = max(1, int(np.ceil((e_hi - e_lo) / bin_width - 1e-9)))
    e = np.asarray(energies, np.float64)
    e = e[np.isfinite(e)]
    idx = np.clip(np.floor((e - e_lo) / bin_width).astype(np.int64), 0, n_bins - 1)
    return np.bincount(idx, minlength=n_bins).astype(np.int64)


def aggregate_throughput(units_this_rank, ms_this_rank, device="cpu"):
    """whole-job throughput = units all ranks processed / max-over-ranks time -> (units/s, ms)."""
    total = float(sum_over_ranks(np.array([float(units_this_rank)], np.float64), device)[0])
    ms = max_over_ranks(ms_this_rank, device)
    return total / (ms * 1e-3), ms
