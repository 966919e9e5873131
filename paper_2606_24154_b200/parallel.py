"""Multi-GPU plumbing: one process per GPU, torch.distributed.

The path shards over evaluation points (a7/a8) and over matrix columns (a3) with replicated element
tables and NO data-path collective; the LU does not shard (replicas only).  What is left for the host
side is: which slab of points a rank owns, the max-over-ranks of a device time, and — if the caller
wants the field on every rank — one all-gather of the outputs.  These helpers hold no arithmetic of the
method and work with any backend (nccl on GPUs, gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


def shard_bounds(m: int, world: int, rank: int):
    """Contiguous, balanced slab [start, stop) of m units for `rank`; the slabs tile [0, m) exactly."""
    base, extra = divmod(int(m), int(world))
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (a device-measured time); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_points(local: torch.Tensor, m: int) -> torch.Tensor:
    """All-gather of per-rank slabs along the LAST dimension (Phi: (m_local,), E: (3, m_local)) into the
    full (…, m) tensor on every rank.  Slabs are the ones of shard_bounds, so they may differ by one."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
    width = max(shard_bounds(m, world, r)[1] - shard_bounds(m, world, r)[0] for r in range(world))
    pad = torch.zeros(local.shape[:-1] + (width,), dtype=local.dtype, device=local.device)
    pad[..., : local.shape[-1]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = []
    for r in range(world):
        s, e = shard_bounds(m, world, r)
        out.append(parts[r][..., : e - s])
    return torch.cat(out, dim=-1)


def eval_sharded(nb, pts: torch.Tensor, gather: bool = True):
    """Strong-scaling evaluation: every rank holds the same solved context `nb` (replica) and evaluates its
    slab of the points; with gather=True every rank gets the full Phi (m) and E (3, m)."""
    m = pts.shape[1]
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    s, e = shard_bounds(m, world, rank)
    phi, E = nb.eval(pts[:, s:e].contiguous())
    if gather:
        return all_gather_points(phi, m), all_gather_points(E, m)
    return phi, E
