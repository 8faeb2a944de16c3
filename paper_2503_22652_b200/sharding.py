"""Host-side multi-GPU plumbing: the filter is column-separable (Algorithm 3 touches column j only
through eps_j and Lambda_k[j]), so ranks own disjoint column shards of the block and
need no data-path collective; only the timing (max over ranks) and the unit count are reduced."""


def column_shard(n_cols, rank, world):
    """[lo, hi) of the global columns owned by `rank`: contiguous, disjoint, covering, sizes differ by <= 1."""
    if world < 1 or not 0 <= rank < world or n_cols < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_cols, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_job(ms_local, units_local, group=None):
    """(max over ranks of the local time, sum over ranks of the local unit count) via torch.distributed.
    Works on any backend (NCCL on GPUs, gloo in the CPU tests); world size 1 needs no process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms_local), float(units_local)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), float(u.item())
