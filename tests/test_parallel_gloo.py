"""Host-side multi-rank logic on CPU: world_size 2, gloo (shard over points, no data-path
collective; max-over-ranks timing; optional all-gather of the outputs)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_24154_b200 import parallel


def test_shard_bounds_tile_exactly():
    for m in (0, 1, 7, 100000, 100001):
        for world in (1, 2, 3, 8):
            b = [parallel.shard_bounds(m, world, r) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == m
            assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))
            sizes = [e - s for s, e in b]
            assert max(sizes) - min(sizes) <= 1
            a = [parallel.shard_bounds(m, world, r, align=128) for r in range(world)]
            assert a[0][0] == 0 and a[-1][1] == m and all(a[r][1] == a[r + 1][0] for r in range(world - 1))
            assert all(s % 128 == 0 or s == m for s, _ in a) and max(e - s for s, e in a) - min(e - s for s, e in a) <= 255


class _FakeNeb:
    """Stands in for a solved context: 'evaluates' a known function of the points on the CPU."""

    def eval(self, pts):
        return pts[0] * 2.0 + pts[2], torch.stack([pts[0], pts[1] * 3.0, -pts[2]])


class _FakeLoop:
    """A replica of the space-charge loop's state on the CPU: E = a known function of the point and of the whole cloud."""

    def __init__(self):
        self.cloud = None
        self.solves = 0

    def add_space_charge(self, pos, charge, replace=True):
        self.cloud = pos.clone()

    def eval(self, pts, want_phi=True):
        c = self.cloud.mean(dim=1, keepdim=True)              # depends on ALL charges, as the direct sum does
        return None, (pts - c) * 2.0

    def push(self, pos, E, mu_dt):
        pos += mu_dt * E
        return pos

    def solve_resident(self):
        self.solves += 1


def _worker(rank, world, port, m, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = torch.Generator().manual_seed(0)
        pts = torch.rand((3, m), generator=g, dtype=torch.float64)          # same points on every rank
        phi, E = parallel.eval_sharded(_FakeNeb(), pts, gather=True)
        ok = torch.equal(phi, pts[0] * 2.0 + pts[2]) and torch.equal(E, torch.stack([pts[0], pts[1] * 3.0, -pts[2]]))
        s, e = parallel.shard_bounds(m, world, rank, parallel.ALIGN)
        phi_l, _ = parallel.eval_sharded(_FakeNeb(), pts, gather=False)
        ok = ok and phi_l.shape[0] == e - s
        t = parallel.max_over_ranks(10.0 + rank)
        # the C4 step with the charges sharded: 3 steps equal the unsharded loop, on every rank
        pos = torch.rand((3, 1001), generator=g, dtype=torch.float64)
        ch = torch.ones(1001, dtype=torch.float64)
        loop, ref, pos_ref = _FakeLoop(), _FakeLoop(), pos.clone()
        loop.add_space_charge(pos, ch)
        ref.add_space_charge(pos_ref, ch)
        for _ in range(3):
            pos = parallel.c4_step_sharded(loop, pos, ch, 0.125)
            _, E = ref.eval(pos_ref)
            pos_ref = ref.push(pos_ref.clone(), E, 0.125)
            ref.add_space_charge(pos_ref, ch)
        ok = ok and torch.equal(pos, pos_ref) and loop.solves == 3 and torch.equal(loop.cloud, pos_ref)
        q.put((rank, bool(ok), t))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world, m = 2, 1001                                   # odd: slabs differ by one
    procs = [ctx.Process(target=_worker, args=(r, world, port, m, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [True, True]
    assert [r[2] for r in res] == [11.0, 11.0]           # max over ranks, identical everywhere


# ---------------------------------------------------------------------------------------------------------------
# Scale-out of the solve: the exchange protocol of parallel.DistSolver on CPU ranks.  _FakeDistNeb
# stands in for a context: it implements the contract of the neb_dist_* calls (include/neb.h) with plain torch CPU
# operations on ITS column blocks only, so that a wrong owner, buffer parity, look-ahead order or missing exchange in
# DistSolver gives a wrong sigma.  The truth is numpy.linalg.solve on the whole system.
# ---------------------------------------------------------------------------------------------------------------
class _FakeDistNeb:
    B = parallel.DIST_BLOCK
    torch_device = torch.device("cpu")
    device = 0

    def dist_configure(self, rank, world):
        self.rank, self.world = rank, world

    def assemble_problem(self, pr):
        A, b = pr                                              # the whole system is known to every rank (as the geometry is)
        self.n = A.shape[0]
        B = self.B
        self.npad = -(-self.n // B) * B
        full = torch.eye(self.npad, dtype=torch.float64)
        full[: self.n, : self.n] = A
        self.blocks = parallel.dist_local_blocks(self.npad // B, self.world, self.rank)
        self.K = torch.cat([full[:, g * B:(g + 1) * B] for g in self.blocks], dim=1).clone() if self.blocks else torch.zeros(self.npad, 0, dtype=torch.float64)
        self.b = torch.zeros(self.npad, dtype=torch.float64)
        self.b[: self.n] = b
        self.ipiv = torch.arange(self.npad, dtype=torch.int32)

    def dist_npad(self):
        return self.npad

    def _cols(self, g):
        lb = self.blocks.index(g)
        return slice(lb * self.B, (lb + 1) * self.B)

    def dist_row_scales(self, s, set_):
        if not set_:
            mx = self.K.abs().max(dim=1).values if self.K.shape[1] else torch.zeros(self.npad, dtype=torch.float64)
            s.copy_(torch.where(mx > 0, 1.0 / mx, torch.full_like(mx, float("inf"))))
        else:
            self.rscale = torch.where(torch.isinf(s), torch.ones_like(s), s).clone()
            self.K *= self.rscale[:, None]

    def _swap_rows(self, cols, k0, piv):
        for t, p in enumerate(piv.tolist()):
            if p != k0 + t:
                tmp = self.K[k0 + t, cols].clone()
                self.K[k0 + t, cols] = self.K[p, cols]
                self.K[p, cols] = tmp

    def dist_factor_block(self, g, panel, piv, stream=None):
        assert g % self.world == self.rank
        B, kb, cs = self.B, g * self.B, self._cols(g)
        blk = self.K[:, cs]
        for j in range(B):                                     # unblocked elimination with partial pivoting, rows kb..
            k = kb + j
            p = k + int(torch.argmax(blk[k:, j].abs()))
            self.ipiv[k] = p
            if p != k:
                blk[[k, p], :] = blk[[p, k], :]
            blk[k + 1:, j] /= blk[k, j]
            blk[k + 1:, j + 1:] -= torch.outer(blk[k + 1:, j], blk[k, j + 1:])
        rows = self.npad - kb
        panel[: rows * B].view(B, rows).copy_(blk[kb:, :].t())  # column-major (rows x 256)
        piv.copy_(self.ipiv[kb:kb + B])

    def dist_apply_block(self, g, panel, piv, part=0):
        B, kb = self.B, g * self.B
        rows = self.npad - kb
        P = panel[: rows * B].view(B, rows).t()                # (rows, 256): the factored block below row kb
        if part != 2:
            self.ipiv[kb:kb + B] = piv
        right = [h for h in self.blocks if h > g]
        nxt = [h for h in right if h == g + 1]
        if part == 1:
            right = nxt
        elif part == 2:
            right = [h for h in right if h != g + 1]
        for h in right:
            cs = self._cols(h)
            self._swap_rows(cs, kb, self.ipiv[kb:kb + B])
            L11 = torch.tril(P[:B, :], -1) + torch.eye(B, dtype=torch.float64)
            U12 = torch.linalg.solve_triangular(L11, self.K[kb:kb + B, cs], upper=False, unitriangular=True)
            self.K[kb:kb + B, cs] = U12
            self.K[kb + B:, cs] -= P[B:, :] @ U12
        if part != 1:
            for h in [h for h in self.blocks if h < g]:
                self._swap_rows(self._cols(h), kb, self.ipiv[kb:kb + B])

    def dist_finish_factor(self):
        perm = list(range(self.npad))
        for i, p in enumerate(self.ipiv.tolist()):
            perm[i], perm[p] = perm[p], perm[i]
        self.rowperm = torch.tensor(perm)
        return 0

    def dist_rhs(self, y):
        y.copy_((self.b * self.rscale)[self.rowperm])

    def dist_tri_block(self, upper, g, y, acc):
        if g % self.world != self.rank:
            return
        B, kb, cs = self.B, g * self.B, self._cols(g)
        T = self.K[kb:kb + B, cs]
        r = (y[kb:kb + B] - acc[kb:kb + B])[:, None]
        if upper:
            x = torch.linalg.solve_triangular(torch.triu(T), r, upper=True)[:, 0]
            acc[:kb] += self.K[:kb, cs] @ x
        else:
            x = torch.linalg.solve_triangular(torch.tril(T, -1) + torch.eye(B, dtype=torch.float64), r, upper=False, unitriangular=True)[:, 0]
            acc[kb + B:] += self.K[kb + B:, cs] @ x
        y[kb:kb + B] = x

    def dist_set_solution(self, x, out=None):
        out.copy_(x[: self.n])
        return out


def _dist_worker(rank, world, port, n, lookahead, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rs = np.random.RandomState(7)
        A = rs.normal(size=(n, n)) * np.exp(rs.uniform(-8, 8, size=(n, 1)))      # badly scaled rows: equilibration + pivoting
        b = rs.normal(size=n)
        nb = _FakeDistNeb()
        nb.n = n
        ds = parallel.DistSolver(nb, lookahead=lookahead)
        ds.assemble((torch.from_numpy(A), torch.from_numpy(b)))
        ds.factor()
        x = ds.solve().numpy()
        x2 = ds.solve().numpy()                                                    # a second solve on the resident factors
        ref = np.linalg.solve(A, b)
        err = np.max(np.abs(x - ref)) / np.max(np.abs(ref))
        q.put((rank, float(err), bool(np.array_equal(x, x2)), int(nb.K.shape[1])))
    finally:
        dist.destroy_process_group()


def _run_dist(world, n, lookahead):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_dist_worker, args=(r, world, port, n, lookahead, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return res


def test_dist_block_maps():
    for world in (1, 2, 3, 8):
        for nblk in (1, 2, 5, 16, 17):
            seen = []
            for r in range(world):
                mine = parallel.dist_local_blocks(nblk, world, r)
                assert all(parallel.dist_owner(g, world) == r for g in mine) and mine == sorted(mine)
                seen += mine
            assert sorted(seen) == list(range(nblk))                               # every block exactly once


def test_dist_solver_protocol_two_and_three_ranks():
    # 1100 -> npad 1280 = 5 blocks: ranks hold 3+2 (world 2) or 2+2+1 (world 3) blocks, the last block is mostly padding
    for world, lookahead in ((2, True), (3, True), (2, False)):
        res = _run_dist(world, 1100, lookahead)
        assert [r[0] for r in res] == list(range(world))
        assert all(r[1] < 1e-10 and r[2] for r in res), res
        assert sum(r[3] for r in res) == 1280                                      # the column blocks partition the matrix
