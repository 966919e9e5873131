#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

Workload (BASELINE.json configs[1], "C1"): conducting cube, 6 x 32 x 32 = 6144 rectangular panels at 1 V,
1e5 evaluation points uniform in the surrounding 3 cm cube (seed 1).  One STEP = one pass of the whole
hot path through the C ABI: neb_assemble (frame tables + 6144^2 fp64 influence matrix) -> neb_solve
(row scaling, blocked LU with DMMA trailing update, RHS, two triangular solves) -> neb_eval (Phi, E at the
1e5 points).  metric = element-point influence pairs/s: (N^2 + M N) pair evaluations per step divided by
the whole step time (LU and solves included in the time, not in the pair count).

  value : inputs already resident in HBM, outputs left in HBM
  e2e   : same step through the same public API with pinned HOST buffers (H2D of the geometry and the
          points, D2H of sigma, Phi and E inside the timed region)
  N > 1 : one process per GPU (torchrun); the LU does not shard (replicas), every rank
          factorises its replica and evaluates ITS OWN 1e5 points (seed 1 + rank): weak scaling, no
          data-path collective; time = max over ranks.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "element-point influence pairs/s (fp64)"
UNIT = "pairs/s"
# FP64 work of one (point, element copy) evaluation of (Phi', E') on the path that >99 % of the pairs of a field
# map take (uniform-axes window + warp-uniform far branch), counted in the SASS of
# eval_kernel<MathFast> (FMA = 2 flop): rectangle 101 DFMA + 32 DMUL + 14 DADD = 248 flop in 148 FP64-pipe
# instructions (general window: 279 flop / 167; near branch: +44 flop / +39); right triangle 199 flop (230 on a
# general window, less the same 31 flop of frame work); wire 139; point charge 30.  Windows that are not uniform
# do more work than counted here, so `achieved` is a lower bound on them.
FLOP_PER_PAIR = {"rect": 248.0, "tri": 199.0, "wire": 139.0, "charge": 30.0}
FP64_INSTR_PER_PAIR = {"rect": 148.0}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE eval_kernel launch on C1, from the ncu --set full capture
# summarised in profiles/r1_ncu_full_eval_assemble.md (3.285504 MB + 84.992 kB); algorithmic bytes of that launch:
# 2.4 MB of points in + 4 x 8 x 1e5 x n_split partial sums out, the 0.8 MB element table from L2
EVAL_TRAFFIC_C1_BYTES = 3285504 + 84992
L2_NOTE = "256 MiB buffer written between timed steps; the matrix exceeds L2"
WORKLOADS = {
    "C1": "C1 cube: N=6144 rect panels, M=100000 points (BASELINE configs[1])",
    "C2": "C2 THGEM cell: rectangles + right triangles, dielectric rows, 100^3 grid (BASELINE configs[2])",
    "C3": "C3 double THGEM: 5x5 image copies, points uniform in the cell (BASELINE configs[3])",
    "C4": "C4 space charge on the C3 geometry: per step E at the charges (panels + all other charges), push, "
          "RHS update, re-solve on the resident LU factors (BASELINE configs[4]); assembly + LU done once before",
}


def make_config(name, pr, m, q=0):
    cfg = {"workload": WORKLOADS[name], "n_elements": int(pr.n), "m_points": int(m), "image_copies": int(max(1, pr.n_img)),
           "step": "assemble+solve(LU)+eval" if name != "C4" else "eval(charges)+push+rhs+re-solve", "l2": L2_NOTE}
    if q:
        cfg["charges"] = int(q)
    return cfg


def load_problem(name, m_cap=None, seed_shift=0):
    from workloads import configs as W
    if name == "C1":
        return W.cube(seed=1 + seed_shift)
    if name == "C2":
        return W.thgem()
    if name == "C3":
        return W.double_thgem(m_points=m_cap or 10_000_000, seed=3 + seed_shift)
    if name == "C4":
        return W.space_charge(W.double_thgem(m_points=0), q_count=m_cap or 1_000_000, seed=4 + seed_shift)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """One long-running `nvidia-smi -lms 100` for the timed region (no per-sample process spawn)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self):
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", os.environ.get("LOCAL_RANK", "0")], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return []
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        rows = [[x.strip() for x in line.split(",")] for line in out.strip().splitlines()]
        return [r for r in rows if len(r) >= 6]


def _clocks_summary(samples):
    if not samples:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
    sm = sorted(int(s[0]) for s in samples if s[0].isdigit())
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    reasons = [n for k, n in enumerate(names) if any(s[2 + k].lower().startswith("active") for s in samples)]
    return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(samples[0][1]) if samples[0][1].isdigit() else None,
            "reasons": reasons}


def cpu_baseline_run(pr, n_rows=None, n_pts=None, with_lu=False):
    """The oracle as it stands (fp64 build, OpenMP on every host core): assembly rows 0..n_rows-1 and the first
    n_pts points (None = all); with_lu also factorises and solves, i.e. the whole step."""
    import oracle
    g = oracle.Geometry(pr)
    m = pr.points.shape[1]
    n_rows = pr.n if n_rows is None else min(n_rows, pr.n)
    n_pts = m if n_pts is None else min(n_pts, m)
    copies = max(1, pr.n_img)
    t0 = time.perf_counter()
    if with_lu:
        K = oracle.assemble(g, mode="f64")
        sig = oracle.solve(K, oracle.rhs(g, mode="f64"), mode="f64")
        n_rows = pr.n
    else:
        rows = np.repeat(np.arange(n_rows), pr.n)
        cols = np.tile(np.arange(pr.n), n_rows)
        sig = np.full(pr.n, 1e-8)
        oracle.matrix_entries(g, rows, cols, mode="f64")
    oracle.evaluate(g, sig, pr.points[:, :n_pts], mode="f64")
    dt = time.perf_counter() - t0
    pairs = copies * (n_rows * pr.n + n_pts * pr.n)
    what = (f"the whole step: assembly {pr.n}x{pr.n}, LU solve, eval at all {n_pts} points" if with_lu and n_pts == m else
            f"assembly rows 0..{n_rows - 1} ({n_rows}x{pr.n}x{copies} pairs) + eval of the first {n_pts} points "
            f"({n_pts}x{pr.n}x{copies} pairs)" + (", LU solve included" if with_lu else "; LU not sampled"))
    return {"value": pairs / dt, "unit": UNIT, "cores": oracle.threads("f64"), "kind": "oracle",
            "sample": what + "; fp64 build, gcc -O2 -fopenmp", "seconds": dt}


def run_reference(args):
    """Reference arm = the oracle (there is no reference code): rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pr = load_problem(args.workload, args.m_points)
    copies = max(1, pr.n_img)
    n_rows, n_pts = max(1, 1024 // copies), max(1, 20000 // copies)
    for _ in range(args.warmup):
        cpu_baseline_run(pr, max(1, n_rows // 32), max(1, n_pts // 100))
    t = []
    base = None
    for _ in range(args.steps):
        base = cpu_baseline_run(pr, n_rows, n_pts)
        t.append(base["seconds"])
    pairs = copies * (min(n_rows, pr.n) * pr.n + min(n_pts, pr.points.shape[1]) * pr.n)
    value = pairs * len(t) / sum(t)
    base["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(t) / len(t), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": make_config(args.workload, pr, pr.points.shape[1]), "cpu_baseline": base,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="C1", choices=sorted(WORKLOADS),
                    help="C1 is the bench line; C2..C4 are one-off full-size runs recorded under profiles/")
    ap.add_argument("--m-points", type=int, default=None, help="cap on the evaluation points (C3) / charges (C4)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "C1":
        args.warmup = max(args.warmup, 3)          # the bench line; C2..C4 one-off runs may use fewer (long steps)

    import torch
    import torch.distributed as dist
    import paper_2606_24154_b200 as P
    from paper_2606_24154_b200 import parallel
    from workloads import configs as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    name = args.workload
    pr = load_problem(name, args.m_points, seed_shift=rank)   # same geometry on every rank, its own points / charges
    is_c4 = name == "C4"
    pts_np = pr.charge_pos if is_c4 else pr.points
    n, m = pr.n, pts_np.shape[1]
    copies = max(1, pr.n_img)
    q = m if is_c4 else 0
    # pair evaluations per step (image copies count as pairs; C4: + charge-charge and charge-collocation pairs)
    pairs_step = copies * m * n + (q * q + n * q if is_c4 else copies * n * n)
    nb = P.Neb(local)

    def t_dev(a, dtype):
        return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dtype).to(dev)

    def pin(a):
        return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory()

    geo = dict(kind=(pr.kind, torch.int32), v0=(pr.v0, torch.float64), e1=(pr.e1, torch.float64), e2=(pr.e2, torch.float64),
               bc_kind=(pr.bc_kind, torch.int32), bc_value=(pr.bc_value, torch.float64), radius=(pr.radius, torch.float64),
               eps_plus=(pr.eps_plus, torch.float64), eps_minus=(pr.eps_minus, torch.float64),
               img_shift=(pr.img_shift, torch.float64))
    d = {k: t_dev(a, t) for k, (a, t) in geo.items()}
    h = {k: pin(None if a is None else np.asarray(a).astype(np.int32 if t == torch.int32 else np.float64))
         for k, (a, t) in geo.items()}
    d_pts = t_dev(pts_np, torch.float64)
    d_sig = torch.empty(n, dtype=torch.float64, device=dev)
    d_phi = torch.empty(m, dtype=torch.float64, device=dev)
    d_E = torch.empty((3, m), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    h_pts = pin(pts_np)
    h_sig = torch.empty(n, dtype=torch.float64).pin_memory()
    h_phi = torch.empty(m, dtype=torch.float64).pin_memory()
    h_E = torch.empty((3, m), dtype=torch.float64).pin_memory()

    def assemble_from(a):
        nb.assemble(a["kind"], a["v0"], a["e1"], a["e2"], a["bc_kind"], a["bc_value"], radius=a["radius"],
                    eps_plus=a["eps_plus"], eps_minus=a["eps_minus"], img_shift=a["img_shift"])

    if not is_c4:
        def step_resident():
            assemble_from(d)
            nb.solve(out=d_sig)
            nb.eval(d_pts, phi=d_phi, E=d_E)

        def step_e2e():
            assemble_from(h)
            nb.solve(out=h_sig)
            nb.eval(h_pts, phi=h_phi, E=h_E)

        h2d = sum(v.numel() * v.element_size() for v in h.values() if v is not None) + h_pts.numel() * 8
        d2h = (h_sig.numel() + h_phi.numel() + h_E.numel()) * 8
    else:
        # C4 (reading S22): geometry assembled and factorised ONCE, outside the timed steps; a step is one pass
        # of the self-consistent loop with all charges
        mu_dt = pr.meta["mu"] * pr.meta["dt"]
        d_ch = t_dev(pr.charge_q, torch.float64)
        h_ch = pin(pr.charge_q)
        assemble_from(d)
        nb.add_space_charge(d_pts, d_ch)
        nb.solve(out=d_sig)

        def step_resident():
            nb.eval(d_pts, E=d_E, want_phi=False)
            nb.push(d_pts, d_E, mu_dt)
            nb.add_space_charge(d_pts, d_ch, replace=True)
            nb.solve(out=d_sig)

        def step_e2e():
            nb.eval(h_pts, E=h_E, want_phi=False)
            nb.push(h_pts, h_E, mu_dt)
            nb.add_space_charge(h_pts, h_ch, replace=True)
            nb.solve(out=h_sig)

        h2d = (3 * m + 3 * m + 3 * m + 3 * m + m) * 8          # points for eval, pos+E for push, pos+q for the charges
        d2h = (3 * m + 3 * m + n) * 8                          # E, pushed positions, sigma

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        for e0, e1 in ev:
            flush.fill_(1)                          # L2 flush, outside the timed interval
            e0.record()
            fn()
            e1.record()
        barrier()
        ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
        return parallel.max_over_ranks(ms, dev)

    for _ in range(args.warmup):
        step_resident()
    torch.cuda.synchronize()
    sampler = ClockSampler()
    sampler.start()
    l0 = nb.launch_count()
    ms = timed(step_resident, args.steps)
    launches = nb.launch_count() - l0
    samples = sampler.stop()

    for _ in range(2):
        step_e2e()
    ms_e2e = timed(step_e2e, args.steps)

    # dominant kernel (a7 eval) alone: CUDA events on the launching stream around that kernel, averaged
    nb.set_option(P.binding.NEB_OPT_PROFILE, 1)
    nb.reset_stats()
    for _ in range(args.steps):
        flush.fill_(1)
        nb.eval(d_pts, phi=None if is_c4 else d_phi, E=d_E, want_phi=not is_c4)
    st = nb.stage_ms()
    eval_ms = st["eval"][0] / max(1, st["eval"][1])
    nb.reset_stats()
    flush.fill_(1)
    step_resident()
    stages = {k: round(v[0], 4) for k, v in nb.stage_ms().items()}
    # the trailing update alone is only timed without look-ahead (with it, it overlaps the next panel)
    nb.set_option(P.binding.NEB_OPT_LU_LOOKAHEAD, 0)
    nb.reset_stats()
    flush.fill_(1)
    step_resident()
    serial = nb.stage_ms()
    stages["lu_gemm"] = round(serial["lu_gemm"][0], 4)
    stages["lu_no_lookahead"] = round(serial["lu"][0], 4)
    nb.set_option(P.binding.NEB_OPT_LU_LOOKAHEAD, 1)
    nb.set_option(P.binding.NEB_OPT_PROFILE, 0)
    dfma_peak, dmma_peak = nb.fp64_peak(0), nb.fp64_peak(1)
    n_tri, n_wire = int(np.sum(pr.kind == 1)), int(np.sum(pr.kind == 2))
    flop_pair = (FLOP_PER_PAIR["rect"] * (n - n_tri - n_wire) + FLOP_PER_PAIR["tri"] * n_tri + FLOP_PER_PAIR["wire"] * n_wire) / n
    eval_pairs = copies * m * n
    achieved = flop_pair * eval_pairs / (eval_ms * 1e-3) * 1e-12
    lu_flop = 2.0 / 3.0 * n ** 3

    fastvol = None
    if name == "C2" and rank == 0:
        # the 100^3 field map of C2 as a FastVolume (same nodes as the eval points), then 1e7
        # trilinear lookups at seeded points inside it.  Bound by memory: 24 B of coordinates in, 32 B of results out
        # and 8 node records of 32 B per point (the 32 MB map stays in L2), reported against the measured HBM copy rate.
        from workloads import rng
        ng = int(round(m ** (1.0 / 3.0)))
        o = np.array([pr.points[0].min(), pr.points[1].min(), pr.points[2].min()])
        hh = (np.array([pr.points[0].max(), pr.points[1].max(), pr.points[2].max()]) - o) / (ng - 1)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        nb.fastvol_build(0, (ng, ng, ng), o, hh)
        ev1.record()
        torch.cuda.synchronize()
        build_ms = ev0.elapsed_time(ev1)
        ml = 10_000_000
        lp = torch.from_numpy(np.stack([o[k] + rng.uniform(7, ml, 0.0, 1.0, offset=k * ml) * hh[k] * (ng - 1) for k in range(3)])).to(dev)
        l_phi = torch.empty(ml, dtype=torch.float64, device=dev)
        l_E = torch.empty((3, ml), dtype=torch.float64, device=dev)
        for _ in range(3):
            nb.fastvol_eval(0, lp, phi=l_phi, E=l_E)
        t_l = []
        for _ in range(10):
            flush.fill_(1)
            ev0.record()
            nb.fastvol_eval(0, lp, phi=l_phi, E=l_E)
            ev1.record()
            torch.cuda.synchronize()
            t_l.append(ev0.elapsed_time(ev1))
        look_ms = sum(t_l) / len(t_l)
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            src = "MEASURED_PEAKS.json hbm_gbs (measured copy rate)"
        except Exception:
            hbm_peak, src = 6650.0, "fallback 6.65 TB/s of B200_PROFILING.md"
        gbs = ml * (24 + 32 + 8 * 32) / (look_ms * 1e-3) * 1e-9
        fastvol = {"grid": [ng, ng, ng], "build_ms": build_ms, "lookups": ml, "lookup_ms": look_ms,
                   "lookup_points_per_s": ml / (look_ms * 1e-3),
                   "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                                "bytes_per_point": 24 + 32 + 8 * 32, "peak_source": src,
                                "hbm_only_gbs": ml * (24 + 32) / (look_ms * 1e-3) * 1e-9,
                                "note": "algorithmic bytes incl. the 8 node records per point; the 32 MB map is served by "
                                        "L2, so only the 56 B/point of coordinates and results (hbm_only_gbs) cross HBM; "
                                        "ncu: the gather runs the L1/TEX pipe at 95 % of its peak "
                                        "(profiles/r1_ncu_full_lu_kernels.md)"}}
        del lp, l_phi, l_E

    adaptive = None
    if name == "C3" and rank == 0:
        # SURVEY 8(f).3, Adaptive Modelling (Table 2): the same field map with the periodic copies beyond
        # far_distance as point charges; time of the element kernel and the largest deviation from the exact map
        ex_phi, ex_E = d_phi.clone(), d_E.clone()
        adaptive = []
        for far_mm in (1.5, 0.9):
            nb.set_adaptive(far_mm * 1e-3)
            nb.set_option(P.binding.NEB_OPT_PROFILE, 1)
            nb.reset_stats()
            flush.fill_(1)
            nb.eval(d_pts, phi=d_phi, E=d_E)
            am_ms = nb.stage_ms()["eval"][0]
            nb.set_option(P.binding.NEB_OPT_PROFILE, 0)
            en = torch.linalg.vector_norm(ex_E, dim=0)
            adaptive.append({"far_distance_mm": far_mm,
                             "copies_simplified": int(np.sum(np.linalg.norm(pr.img_shift, axis=0) >= far_mm * 1e-3)),
                             "eval_kernel_ms": am_ms, "speedup_vs_exact": eval_ms / am_ms,
                             "max_err_phi_rel_to_max": float((d_phi - ex_phi).abs().max() / ex_phi.abs().max()),
                             "max_err_E_rel_to_max": float(torch.linalg.vector_norm(d_E - ex_E, dim=0).max() / en.max()),
                             "median_err_E_pointwise": float((torch.linalg.vector_norm(d_E - ex_E, dim=0) / en).median())})
        nb.set_adaptive(0.0)
        del ex_phi, ex_E

    voxelised = None
    if is_c4 and rank == 0:
        # SURVEY 8(f).2, Alg. 3: the same cloud as line charges (10 um voxels): time of the space-charge sums at the
        # charges' own positions and the deviation of E there from the point-charge sum (the paper leaves the accuracy
        # of the representation open; a charge sees its own voxel's line, so the near field differs)
        nb.set_option(P.binding.NEB_OPT_PROFILE, 1)
        nb.reset_stats()
        nb.add_space_charge(d_pts, d_ch, replace=True)
        nb.eval(d_pts, E=d_E, want_phi=False)
        pt_ms = nb.stage_ms()["charges"][0]
        E_pt = d_E.clone()
        # a 2 mm box of 200^3 voxels about the cloud's median (charges that were pushed far away count in border voxels)
        vox = np.full(3, 1e-5)
        dims = np.full(3, 200, dtype=np.int32)
        lo = d_pts.median(dim=1).values.cpu().numpy() - 0.5 * vox * dims
        nb.reset_stats()
        n_lines = nb.voxelize_space_charge(lo, vox, dims)
        vox_ms = nb.stage_ms()["charges"][0]
        nb.reset_stats()
        nb.eval(d_pts, E=d_E, want_phi=False)
        ln_ms = nb.stage_ms()["charges"][0]
        nb.set_option(P.binding.NEB_OPT_PROFILE, 0)
        en = torch.linalg.vector_norm(E_pt, dim=0)
        dev = torch.linalg.vector_norm(d_E - E_pt, dim=0) / en
        voxelised = {"voxel_um": 10.0, "grid": [int(v) for v in dims], "points": int(m), "lines": int(n_lines),
                     "voxelise_ms": vox_ms, "point_charge_sum_ms": pt_ms, "line_charge_sum_ms": ln_ms,
                     "median_dev_E_at_charges": float(dev.median()), "p99_dev_E_at_charges": float(dev.quantile(0.99))}
        nb.add_space_charge(d_pts, d_ch, replace=True)
        del E_pt

    if rank == 0:
        value = pairs_step * args.steps * world / (ms * 1e-3)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": make_config(name, pr, m, q),
            "e2e": {"value": pairs_step * args.steps * world / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": launches, "clocks": _clocks_summary(samples),
            "roofline": {"bound": "alu", "kernel": "eval_kernel<MathFast> (a7)", "achieved": achieved, "peak": dfma_peak,
                         "unit": "TFLOP/s", "frac": achieved / dfma_peak,
                         "traffic": EVAL_TRAFFIC_C1_BYTES if name == "C1" else None,
                         "peak_source": "neb_fp64_peak(0): DFMA-chain microbenchmark run in this process "
                                        "(nominal 148 SM x 64 DFMA/clk x 1.965 GHz = 37.2)",
                         "flop_per_pair": flop_pair, "kernel_ms": eval_ms,
                         "fp64_pipe_slot_frac": (FP64_INSTR_PER_PAIR["rect"] * eval_pairs / (eval_ms * 1e-3) / (0.5e12 * dfma_peak)
                                                 if n_tri + n_wire == 0 else None),
                         "pairs_per_s_kernel": eval_pairs / (eval_ms * 1e-3),
                         "field_map_points_per_s": m / (eval_ms * 1e-3)},
            "stages_ms": stages,
            "lu": {"tflops_whole_lu": lu_flop / (stages["lu"] * 1e-3) * 1e-12 if stages.get("lu") else None,
                   "tflops_trailing_update": lu_flop / (stages["lu_gemm"] * 1e-3) * 1e-12 if stages.get("lu_gemm") else None,
                   "dmma_peak_tflops": dmma_peak},
        }
        if fastvol:
            line["fastvol"] = fastvol
        if adaptive:
            line["adaptive_modelling"] = adaptive
        if voxelised:
            line["voxelised_space_charge"] = voxelised
        if not args.no_cpu_baseline and world == 1:
            if name == "C1":
                line["cpu_baseline"] = cpu_baseline_run(pr, with_lu=True)      # the whole C1 step, LU included
            elif not is_c4:
                per_unit = n * copies                                          # pairs per assembly row / per point
                line["cpu_baseline"] = cpu_baseline_run(pr, max(1, int(2e8 // per_unit)), max(1, int(1.8e9 // per_unit)))
        print(json.dumps(line), flush=True)
    nb.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
