"""Multi-GPU plumbing: one process per GPU, torch.distributed.

The path shards over evaluation points (a7/a8) and over matrix columns (a3) with replicated element
tables and NO data-path collective; the LU runs as replicas, or — for matrices beyond one GPU, SURVEY §8(f).4 —
block-cyclic over the ranks with the exchanges of DistSolver below.  What is left for the host
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
    if dist.get_backend() == "gloo":
        device = "cpu"                      # CPU-only backend (tests, rehearsals): reduce on the host
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


# ---------------------------------------------------------------------------------------------------------------
# Scale-out of the solve: 1-D block-cyclic LU over the ranks.  The library (neb_dist_* in include/neb.h)
# does the arithmetic; this class owns the buffers that travel and issues the exchanges between the library's steps.
# ---------------------------------------------------------------------------------------------------------------
DIST_BLOCK = 256


def dist_owner(g: int, world: int) -> int:
    """Rank that holds column block g (256 columns) of the block-cyclic matrix."""
    return g % world


def dist_local_blocks(n_blocks: int, world: int, rank: int):
    """Global indices of the column blocks a rank holds, in their local order."""
    return list(range(rank, n_blocks, world))


def _group():
    on = dist.is_available() and dist.is_initialized()
    return (dist.get_world_size(), dist.get_rank()) if on else (1, 0)


def _via_host(t: torch.Tensor) -> bool:
    return t.is_cuda and dist.get_backend() == "gloo"      # CPU-only backend (the tests): stage through the host


def _broadcast(t: torch.Tensor, src: int):
    world, rank = _group()
    if world == 1:
        return
    if _via_host(t):
        h = t.cpu()
        dist.broadcast(h, src)
        if rank != src:
            t.copy_(h)
    else:
        dist.broadcast(t, src)


def _all_reduce(t: torch.Tensor, op):
    world, _ = _group()
    if world == 1:
        return
    if _via_host(t):
        h = t.cpu()
        dist.all_reduce(h, op=op)
        t.copy_(h)
    else:
        dist.all_reduce(t, op=op)


class _HostStream:
    """Stream stand-in for a CPU device (the gloo test of the exchange protocol): everything is in order already."""
    cuda_stream = 0

    def wait_stream(self, other):
        pass

    def wait_event(self, ev):
        pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


class _HostEvent:
    def record(self, stream):
        pass


class DistSolver:
    """Assemble + LU + solve of ONE system spread over the ranks of the default process group (one process per GPU).

        nb = Neb(local_rank); ds = DistSolver(nb); ds.assemble(problem); ds.factor(); sigma = ds.solve()

    Every rank calls the same methods in the same order and ends with the same sigma and a context that evaluates
    fields as a replica (eval_sharded).  Exchanges per system: one MIN of the row scales (8 npad bytes), one broadcast
    per 256-column block ((npad - 256 g) x 2 KB + 1 KB of pivots; overlapped with the trailing update when
    lookahead is on), and per solve 2 npad/256 sums of 256 doubles plus one sum of the solution vector."""

    def __init__(self, nb, lookahead: bool = True):
        self.nb = nb
        self.world, self.rank = _group()
        self.lookahead = lookahead
        nb.dist_configure(self.rank, self.world)
        # a context is bound to a CUDA device; the CPU stand-in of the gloo test names its own
        self.dev = getattr(nb, "torch_device", None) or torch.device("cuda", nb.device)
        self.npad = 0

    def assemble(self, pr):
        nb = self.nb
        nb.assemble_problem(pr)
        self.npad = nb.dist_npad()
        self.n_blocks = self.npad // DIST_BLOCK
        f64 = dict(dtype=torch.float64, device=self.dev)
        scales = torch.empty(self.npad, **f64)
        nb.dist_row_scales(scales, False)
        _all_reduce(scales, dist.ReduceOp.MIN)              # 1 / (row maximum over ALL columns): reading S15
        nb.dist_row_scales(scales, True)
        self.panel = [torch.empty(self.npad * DIST_BLOCK, **f64) for _ in range(2)]
        self.piv = [torch.empty(DIST_BLOCK, dtype=torch.int32, device=self.dev) for _ in range(2)]
        self.y = torch.empty(self.npad, **f64)
        self.acc = torch.empty(self.npad, **f64)

    def factor(self):
        """The block loop.  Buffer b = g % 2 carries block g; with lookahead the owner of block g + 1 updates that block
        first, factors it on the side stream and the broadcast of g + 1 is issued there, beside the trailing update of g."""
        nb, world, rank, B = self.nb, self.world, self.rank, DIST_BLOCK
        main = torch.cuda.current_stream(self.dev) if self.dev.type == "cuda" else _HostStream()
        side = torch.cuda.Stream(self.dev, priority=-1) if (self.lookahead and self.dev.type == "cuda") else main
        new_event = torch.cuda.Event if self.dev.type == "cuda" else _HostEvent
        applied = [None, None]                              # event: the update that read buffer b has run (main stream)
        if dist_owner(0, world) == rank:
            side.wait_stream(main)
            nb.dist_factor_block(0, self.panel[0], self.piv[0], stream=side)
        for g in range(self.n_blocks):
            b = g % 2
            rows = self.npad - g * B
            if applied[b] is not None:                      # update g - 2 read this buffer: it must be done before the
                side.wait_event(applied[b])                 # broadcast of block g overwrites it
            with (torch.cuda.stream(side) if self.dev.type == "cuda" else _HostStream()):
                _broadcast(self.panel[b][: rows * B], dist_owner(g, world))
                _broadcast(self.piv[b], dist_owner(g, world))
            main.wait_stream(side)
            nxt = g + 1
            if nxt < self.n_blocks and dist_owner(nxt, world) == rank:
                nb.dist_apply_block(g, self.panel[b], self.piv[b], part=1)
                side.wait_stream(main)                      # block g + 1 is up to date, update g - 1 has released its buffer
                nb.dist_factor_block(nxt, self.panel[nxt % 2], self.piv[nxt % 2], stream=side)
                nb.dist_apply_block(g, self.panel[b], self.piv[b], part=2)
            else:
                nb.dist_apply_block(g, self.panel[b], self.piv[b], part=0)
            applied[b] = new_event()
            applied[b].record(main)
        main.wait_stream(side)
        flag = torch.tensor([nb.dist_finish_factor()], dtype=torch.int32, device=self.dev)
        _all_reduce(flag, dist.ReduceOp.MAX)
        if int(flag.item()):
            raise RuntimeError("NEB_ESINGULAR: zero or NaN pivot in the distributed factorisation")

    def solve(self, out=None):
        """Right-hand side (with the space charges the context holds) -> sigma (n) on every rank, on the resident factors."""
        nb, world, rank, B = self.nb, self.world, self.rank, DIST_BLOCK
        nb.dist_rhs(self.y)
        for upper in (False, True):
            self.acc.zero_()
            order = range(self.n_blocks - 1, -1, -1) if upper else range(self.n_blocks)
            for g in order:
                _all_reduce(self.acc[g * B:(g + 1) * B], dist.ReduceOp.SUM)
                nb.dist_tri_block(upper, g, self.y, self.acc)
        mine = (torch.arange(self.n_blocks, device=self.dev) % world == rank)[:, None]
        x = torch.where(mine, self.y.view(self.n_blocks, B), torch.zeros((), dtype=torch.float64, device=self.dev)).reshape(-1).contiguous()
        _all_reduce(x, dist.ReduceOp.SUM)
        if out is None:
            out = torch.empty(nb.n, dtype=torch.float64, device=self.dev)
        nb.dist_set_solution(x, out)
        return out
