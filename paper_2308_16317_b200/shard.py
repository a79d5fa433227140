"""Multi-GPU plumbing: the batch shards by central atom, one process per GPU, no data-path collective
("The MPI ranks are evenly distributed on multiple GPUs").  Only the tiny
k x k outputs are (optionally) gathered, and timings are reduced with MAX over ranks."""
from __future__ import annotations


def shard_atoms(n_atoms_total: int, world: int, rank: int) -> range:
    """Contiguous slice of central atoms owned by `rank` (by atom first, so that each GPU keeps its
    energies together); sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(n_atoms_total, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def max_over_ranks(x: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_tau00(tau_local, counts: list[int]):
    """All-gather the per-rank tau00 blocks [b_r, k, k] into global batch order [sum b_r, k, k]
    (ranks own contiguous atom slices, so concatenation in rank order is batch order)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return tau_local
    k = tau_local.shape[-1]
    bmax = max(counts)
    pad = torch.zeros((bmax, k, k), dtype=tau_local.dtype, device=tau_local.device)
    pad[: tau_local.shape[0]] = tau_local
    real = torch.view_as_real(pad).contiguous()
    outs = [torch.empty_like(real) for _ in counts]
    dist.all_gather(outs, real)
    return torch.cat([torch.view_as_complex(o)[:c] for o, c in zip(outs, counts)], dim=0)
