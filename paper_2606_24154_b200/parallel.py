"""Multi-GPU plumbing: one process per GPU, torch.distributed.

The path shards over evaluation points (a7/a8) and over matrix columns (a3) with replicated element
tables and NO data-path collective; the LU does not shard (replicas only).  What is left for the host
side is: which slab of points a rank owns, the max-over-ranks of a device time, — if the caller
wants the field on every rank — one all-gather of the outputs, and the per-step all-gather of the pushed charge
positions of the space-charge loop (c4_step_sharded).  These helpers hold no arithmetic of the
method and work with any backend (nccl on GPUs, gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


ALIGN = 128      # points per CTA of the evaluation kernels


def shard_bounds(m: int, world: int, rank: int, align: int = 1):
    """Contiguous, balanced slab [start, stop) of m units for `rank`; the slabs tile [0, m) exactly.  With align > 1 every
    boundary but the last is a multiple of `align`: the evaluation kernels decide their near/far branch per WARP, so only
    slabs cut at CTA boundaries (align = 128) give every point the warp it has in the unsharded launch, hence the same bits."""
    blocks = -(-int(m) // align)
    base, extra = divmod(blocks, int(world))
    start = (rank * base + min(rank, extra)) * align
    stop = start + (base + (1 if rank < extra else 0)) * align
    return min(start, int(m)), min(stop, int(m))


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (a device-measured time); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_points(local: torch.Tensor, m: int, align: int = 1) -> torch.Tensor:
    """All-gather of per-rank slabs along the LAST dimension (Phi: (m_local,), E: (3, m_local)) into the
    full (…, m) tensor on every rank.  Slabs are the ones of shard_bounds, so they may differ by one."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
    width = max(shard_bounds(m, world, r, align)[1] - shard_bounds(m, world, r, align)[0] for r in range(world))
    # a CPU-only backend (gloo: the multi-rank tests, also with the ranks' kernels on one shared GPU) gathers on the host
    via_host = local.is_cuda and dist.get_backend() == "gloo"
    src = local.cpu() if via_host else local
    pad = torch.zeros(src.shape[:-1] + (width,), dtype=src.dtype, device=src.device)
    pad[..., : src.shape[-1]] = src
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = []
    for r in range(world):
        s, e = shard_bounds(m, world, r, align)
        out.append(parts[r][..., : e - s])
    res = torch.cat(out, dim=-1)
    return res.to(local.device) if via_host else res


def c4_step_sharded(nb, pos: torch.Tensor, charge: torch.Tensor, mu_dt: float):
    """One step of the self-consistent space-charge loop (BASELINE configs[4]; Alg. 4) with the CHARGES
    sharded over the ranks: every rank holds the same solved context `nb` (replica: element tables,
    factors, all q charges) and the same positions `pos` (3, q);
      1. it evaluates E at ITS slab of the charges (from the panels and ALL charges) and pushes that slab,
      2. ONE all-gather of the pushed positions (24 q bytes in all) gives every rank the new cloud,
      3. every rank updates its replica: new charges -> right-hand side -> re-solve on the resident factors.
    Returns the new positions (3, q), identical on every rank.  No collective inside a kernel; the gather is the
    path's only exchange."""
    q = pos.shape[1]
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    s, e = shard_bounds(q, world, rank, ALIGN)
    mine = pos[:, s:e].contiguous()
    _, E = nb.eval(mine, want_phi=False)
    nb.push(mine, E, mu_dt)
    new_pos = all_gather_points(mine, q, ALIGN).contiguous()
    nb.add_space_charge(new_pos, charge, replace=True)
    nb.solve_resident()
    return new_pos


def eval_sharded(nb, pts: torch.Tensor, gather: bool = True):
    """Strong-scaling evaluation: every rank holds the same solved context `nb` (replica) and evaluates its
    slab of the points; with gather=True every rank gets the full Phi (m) and E (3, m).  With NEB_OPT_EVAL_SPLITS set
    to a fixed count the result is bit-identical to the unsharded evaluation (the partial sums then do not depend on
    how many points a call is given); with the default automatic split it agrees to rounding."""
    m = pts.shape[1]
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    s, e = shard_bounds(m, world, rank, ALIGN)
    phi, E = nb.eval(pts[:, s:e].contiguous())
    if gather:
        return all_gather_points(phi, m, ALIGN), all_gather_points(E, m, ALIGN)
    return phi, E
