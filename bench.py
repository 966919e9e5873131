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
# map take (warp-uniform far branch), counted in the SASS of eval_kernel<MathFast> (FMA = 2 flop):
# rectangle 113 DFMA + 38 DMUL + 15 DADD = 279 flop in 167 FP64-pipe instructions (the near branch: 323 flop,
# 206 instructions); right triangle 232 flop; wire 139; point charge 30
FLOP_PER_PAIR = {"rect": 279.0, "tri": 232.0, "wire": 139.0, "charge": 30.0}
FP64_INSTR_PER_PAIR = {"rect": 167.0}
CONFIG = {"workload": "C1 cube: N=6144 rect panels, M=100000 points (BASELINE configs[1])",
          "n_elements": 6144, "m_points": 100000, "step": "assemble+solve(LU)+eval",
          "l2": "256 MiB buffer written between timed steps; matrix (302 MB) exceeds L2"}


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


def cpu_baseline_run(pr, n_rows=1024, n_pts=20000):
    """The oracle as it stands (fp64 build, OpenMP on every host core) on a bounded sample of C1."""
    import oracle
    g = oracle.Geometry(pr)
    rows = np.repeat(np.arange(n_rows), pr.n)
    cols = np.tile(np.arange(pr.n), n_rows)
    sig = np.full(pr.n, 1e-8)
    t0 = time.perf_counter()
    oracle.matrix_entries(g, rows, cols, mode="f64")
    oracle.evaluate(g, sig, pr.points[:, :n_pts], mode="f64")
    dt = time.perf_counter() - t0
    pairs = n_rows * pr.n + n_pts * pr.n
    return {"value": pairs / dt, "unit": UNIT, "cores": oracle.threads("f64"), "kind": "oracle",
            "sample": f"assembly rows 0..{n_rows - 1} ({n_rows}x{pr.n} pairs) + eval of the first {n_pts} points "
                      f"({n_pts}x{pr.n} pairs) of C1, fp64 build, gcc -O2 -fopenmp; LU not sampled", "seconds": dt}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import configs as W
    pr = W.cube()
    n_rows, n_pts = 256, 4000
    for _ in range(args.warmup):
        cpu_baseline_run(pr, 32, 200)
    t = []
    base = None
    for _ in range(args.steps):
        base = cpu_baseline_run(pr, n_rows, n_pts)
        t.append(base["seconds"])
    pairs = n_rows * pr.n + n_pts * pr.n
    value = pairs * len(t) / sum(t)
    base["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(t) / len(t), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": CONFIG, "cpu_baseline": base,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

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

    pr = W.cube(seed=1 + rank)                     # same geometry on every rank, its own points
    n, m = pr.n, pr.points.shape[1]
    pairs_step = n * n + m * n
    nb = P.Neb(local)

    def t_dev(a, dtype):
        return torch.from_numpy(np.ascontiguousarray(a)).to(dtype).to(dev)

    d = dict(kind=t_dev(pr.kind, torch.int32), v0=t_dev(pr.v0, torch.float64), e1=t_dev(pr.e1, torch.float64),
             e2=t_dev(pr.e2, torch.float64), bc_kind=t_dev(pr.bc_kind, torch.int32), bc_value=t_dev(pr.bc_value, torch.float64))
    d_pts = t_dev(pr.points, torch.float64)
    d_sig = torch.empty(n, dtype=torch.float64, device=dev)
    d_phi = torch.empty(m, dtype=torch.float64, device=dev)
    d_E = torch.empty((3, m), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step_resident():
        nb.assemble(d["kind"], d["v0"], d["e1"], d["e2"], d["bc_kind"], d["bc_value"])
        nb.solve(out=d_sig)
        nb.eval(d_pts, phi=d_phi, E=d_E)

    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h = dict(kind=pin(pr.kind), v0=pin(pr.v0), e1=pin(pr.e1), e2=pin(pr.e2), bc_kind=pin(pr.bc_kind), bc_value=pin(pr.bc_value))
    h_pts = pin(pr.points)
    h_sig = torch.empty(n, dtype=torch.float64).pin_memory()
    h_phi = torch.empty(m, dtype=torch.float64).pin_memory()
    h_E = torch.empty((3, m), dtype=torch.float64).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in h.values()) + h_pts.numel() * 8
    d2h = (h_sig.numel() + h_phi.numel() + h_E.numel()) * 8

    def step_e2e():
        nb.assemble(h["kind"], h["v0"], h["e1"], h["e2"], h["bc_kind"], h["bc_value"])
        nb.solve(out=h_sig)
        nb.eval(h_pts, phi=h_phi, E=h_E)

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
        nb.eval(d_pts, phi=d_phi, E=d_E)
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
    flop_eval = FLOP_PER_PAIR["rect"] * m * n
    achieved = flop_eval / (eval_ms * 1e-3) * 1e-12
    lu_flop = 2.0 / 3.0 * n ** 3

    if rank == 0:
        value = pairs_step * args.steps * world / (ms * 1e-3)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": CONFIG,
            "e2e": {"value": pairs_step * args.steps * world / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": launches, "clocks": _clocks_summary(samples),
            "roofline": {"bound": "alu", "kernel": "eval_kernel<MathFast> (a7)", "achieved": achieved, "peak": dfma_peak,
                         "unit": "TFLOP/s", "frac": achieved / dfma_peak, "traffic": None,
                         "peak_source": "neb_fp64_peak(0): DFMA-chain microbenchmark run in this process "
                                        "(nominal 148 SM x 64 DFMA/clk x 1.965 GHz = 37.2)",
                         "flop_per_pair": FLOP_PER_PAIR["rect"], "kernel_ms": eval_ms,
                         "fp64_pipe_slot_frac": FP64_INSTR_PER_PAIR["rect"] * m * n / (eval_ms * 1e-3) / (0.5e12 * dfma_peak),
                         "pairs_per_s_kernel": m * n / (eval_ms * 1e-3),
                         "field_map_points_per_s": m / (eval_ms * 1e-3)},
            "stages_ms": stages,
            "lu": {"tflops_whole_lu": lu_flop / (stages["lu"] * 1e-3) * 1e-12 if stages.get("lu") else None,
                   "tflops_trailing_update": lu_flop / (stages["lu_gemm"] * 1e-3) * 1e-12 if stages.get("lu_gemm") else None,
                   "dmma_peak_tflops": dmma_peak},
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline_run(pr)
        print(json.dumps(line), flush=True)
    nb.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
