"""One launch of each hot kernel on a named, seeded case — the command line Nsight Compute is pointed at.

    python -m paper_2606_24154_b200.profile_cases [case ...]        (no argument: every case)

Each case prints `case <name> kernel <kernel> units <pairs> ms <CUDA-event time of the stage>`; the units are the
(point, element copy) or (point, charge) pairs that ONE launch of the named kernel evaluates, so that per-pair
operation counts follow from ncu's per-launch `smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on.sum`
(SURVEY.md §8(d)(ii)).  bench.py reads the resulting table, profiles/r2_opcounts.md, for its roofline constants.

Cases (all through the C ABI; inputs from workloads/, seeded):
  eval_rect_uniform   C1 cube (6144 rectangles on uniform-axes windows), 1e5 points            -> eval_kernel
  eval_rect_single    the same with NEB_OPT_PAIR_STRIPS = 0 (every element on its own)         -> eval_kernel
  eval_images_single  eval_images with NEB_OPT_PAIR_STRIPS = 0                                 -> eval_kernel
  eval_tri_uniform    4096 equally oriented right triangles (uniform windows), 1e5 points      -> eval_kernel
  eval_rect_general   4096 randomly oriented rectangles (general windows), 1e5 points          -> eval_kernel
  eval_tri_general    4096 randomly oriented right triangles, 1e5 points                       -> eval_kernel
  eval_wire           4096 randomly oriented wires, 1e5 points                                 -> eval_kernel
  eval_images         C3-like: reduced double THGEM (d=20) with 5x5 copies, 2e4 points         -> eval_kernel
  eval_near           C1 cube, 1e5 points within 2 panel sizes of the surface (near branch)    -> eval_kernel
  assemble_c2         C2 at pitch divisor 30 (rectangles, triangles, dielectric rows)          -> assemble_kernel
  assemble_images     reduced double THGEM (d=20) with 5x5 copies                              -> assemble_kernel
  charges             1e5 points x 2e5 point charges                                           -> charge_kernel
  lines               1e5 points x the line charges of a voxelised 2e5-charge cloud            -> line_kernel
  lu_c1 / trisolve_c1 C1: factorisation and the two triangular solves                          -> panel/gemm/tri_wave
  max_n               (not in the default list) cube with 6 x 147^2 = 129654 panels, the largest mesh the panel cluster
                      takes (npad = 129664 of 130944): 134 GB matrix, whole step, stage times
"""
import sys

import numpy as np


def _sawtooth_triangles(n_side=64, side_mm=10.0):
    """n_side^2 right triangles with IDENTICAL axes (lower-left halves of a square grid): uniform windows."""
    from workloads import configs as W
    b = W._Builder()
    p = side_mm / n_side
    for i in range(n_side):
        for j in range(n_side):
            b.add(W.TRI, (-side_mm / 2 + i * p, -side_mm / 2 + j * p, 0.0), (p, 0, 0), (0, p, 0), (0, 0, 1),
                  bc_kind=W.DIRICHLET, bc_value=1.0)
    return b.finish("sawtooth")


def _points(seed, m, half_mm):
    from workloads import rng
    return np.stack([rng.uniform(seed, m, -half_mm, half_mm, offset=k * m) for k in range(3)]) * 1e-3


def run(cases):
    import torch
    from workloads import configs as W
    from . import Neb, binding as B

    def report(name, kernel, units, stage, nb):
        ms, launches = nb.stage_ms()[stage]
        print(f"case {name} kernel {kernel} units {units:d} ms {ms:.4f} launches {launches}", flush=True)

    def eval_case(name, pr, pts, sigma=None, pairs=1):
        nb = Neb()
        nb.set_option(B.NEB_OPT_PROFILE, 1)
        nb.set_option(B.NEB_OPT_PAIR_STRIPS, pairs)
        nb.assemble_problem(pr)
        nb.set_sigma(np.linspace(1e-8, 2e-8, pr.n) if sigma is None else sigma)
        d = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
        nb.eval(d)                                   # warm-up (untimed by the table: ncu sees both launches)
        nb.reset_stats()
        nb.eval(d)
        report(name, "eval_kernel", pts.shape[1] * pr.n * max(1, pr.n_img), "eval", nb)
        nb.close()

    m = 100_000
    for name in cases:
        if name in ("eval_rect_uniform", "eval_rect_single"):
            pr = W.cube()
            eval_case(name, pr, pr.points, pairs=int(name == "eval_rect_uniform"))
        elif name == "eval_tri_uniform":
            eval_case(name, _sawtooth_triangles(), _points(11, m, 15.0))
        elif name in ("eval_rect_general", "eval_tri_general", "eval_wire"):
            kind = {"eval_rect_general": W.RECT, "eval_tri_general": W.TRI, "eval_wire": W.WIRE}[name]
            pr = W.random_elements(4096, seed=12, kinds=(kind,), size_mm=(0.1, 0.3), box_mm=5.0)
            eval_case(name, pr, _points(13, m, 15.0))
        elif name in ("eval_images", "eval_images_single"):
            pr = W.double_thgem(d=20, n_plane=20, m_points=20_000)
            eval_case(name, pr, pr.points, pairs=int(name == "eval_images"))
        elif name == "eval_near":
            pr = W.cube()
            rs = np.random.RandomState(3)
            j = rs.randint(0, pr.n, m)
            c = pr.centroids()[:, j] + pr.normals()[:, j] * (rs.uniform(0.1, 2.0, m) * 0.3125e-3)
            eval_case(name, pr, c)
        elif name in ("assemble_c2", "assemble_images"):
            pr = W.thgem(d=30, n_plane=30, n_grid=2) if name == "assemble_c2" else W.double_thgem(d=20, n_plane=20, m_points=2)
            nb = Neb()
            nb.set_option(B.NEB_OPT_PROFILE, 1)
            nb.assemble_problem(pr)
            nb.reset_stats()
            nb.assemble_problem(pr)
            report(name, "assemble_kernel", pr.n * pr.n * max(1, pr.n_img), "assemble", nb)
            nb.close()
        elif name in ("charges", "lines"):
            pr = W.plate()
            q = 200_000
            rs = np.random.RandomState(4)
            pos = rs.normal(size=(3, q)) * 1e-3
            nb = Neb()
            nb.set_option(B.NEB_OPT_PROFILE, 1)
            nb.assemble_problem(pr)
            nb.set_sigma(np.zeros(pr.n))
            nb.add_space_charge(pos, np.full(q, W.Q_E))
            units = m * q
            if name == "lines":
                units = m * nb.voxelize_space_charge(np.full(3, -4e-3), np.full(3, 1e-4), np.full(3, 80, dtype=np.int32))
            d = torch.from_numpy(_points(14, m, 6.0)).cuda()
            nb.eval(d)
            nb.reset_stats()
            nb.eval(d)
            report(name, "charge_kernel" if name == "charges" else "line_kernel", units, "charges", nb)
            nb.close()
        elif name in ("lu_c1", "trisolve_c1"):
            pr = W.cube()
            nb = Neb()
            nb.set_option(B.NEB_OPT_PROFILE, 1)
            nb.assemble_problem(pr)
            nb.solve()
            nb.assemble_problem(pr)
            nb.reset_stats()
            nb.solve()
            report(name, "panel_stream_kernel+gemm_kernel" if name == "lu_c1" else "tri_wave_kernel", pr.n,
                   "lu" if name == "lu_c1" else "trisolve", nb)
            nb.close()
        elif name == "max_n":
            pr = W.cube(n_side=147, m_points=1000)
            nb = Neb()
            nb.set_option(B.NEB_OPT_PROFILE, 1)
            nb.assemble_problem(pr)
            sig = nb.solve()
            nb.eval(torch.from_numpy(pr.points).cuda())
            st = {k: round(v[0], 2) for k, v in nb.stage_ms().items() if v[0] > 0}
            cap = float(sig.sum() * (pr.meta["side"] / 147) ** 2 / (4 * np.pi * 8.8541878128e-12 * pr.meta["side"]))
            print(f"case max_n kernel all units {pr.n} stages_ms {st} lu_tflops {nb.counter(1) / st['lu'] * 1e-9:.2f} "
                  f"trisolve_gbs {8.0 * pr.n ** 2 / st['trisolve'] * 1e-6:.0f} capacitance/(4 pi eps0 a) {cap:.6f}", flush=True)
            nb.close()
        else:
            raise SystemExit(f"unknown case {name}")


ALL = ["eval_rect_uniform", "eval_rect_single", "eval_tri_uniform", "eval_rect_general", "eval_tri_general", "eval_wire", "eval_images",
       "eval_images_single", "eval_near", "assemble_c2", "assemble_images", "charges", "lines", "lu_c1", "trisolve_c1"]

if __name__ == "__main__":
    run(sys.argv[1:] or ALL)
