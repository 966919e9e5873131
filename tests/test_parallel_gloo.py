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
