"""Multi-GPU plumbing of bench.py (S 8(e)): the path shards by source -- every rank holds a replica of the operator and
solves its own sources; there is no data-path collective.  Only the timing is reduced (max over ranks)."""
import torch
import torch.distributed as dist


def source_offset(rank, n_rhs_per_rank):
    """Weak scaling: rank r solves sources [r * n, (r + 1) * n) of one global noise stream (noise_fill's rhs_offset)."""
    return rank * n_rhs_per_rank


def source_slices(n_total, world):
    """Strong-scaling split of n_total sources: contiguous, sizes differ by at most one; returns [(start, count)] per rank."""
    base, rem = divmod(n_total, world)
    out, s = [], 0
    for r in range(world):
        c = base + (1 if r < rem else 0)
        out.append((s, c))
        s += c
    return out


def max_over_ranks(x, device="cpu"):
    """Max of a python float over all ranks (identity without an initialised process group)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_seconds_per_source(ms_max, steps, n_rhs_per_rank, world):
    """value of bench.py: max-over-ranks time of `steps` steps divided by all sources solved by all ranks."""
    return ms_max * 1e-3 / (steps * n_rhs_per_rank * world)
