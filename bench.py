#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

Default workload (BASELINE.json configs[2], "C2"): THGEM-like unit cell, N = 19400 rectangles + right triangles, 4608
dielectric-interface rows, Phi and E on the 100^3 grid of the cell — the largest configuration whose
`--steps 20 --warmup 5` run, with the reference arm, fits the driver's budget.  One STEP = one pass of the whole hot path
through the C ABI: neb_assemble (frame tables + N^2 fp64 influence matrix) -> neb_solve (row scaling, blocked LU with
DMMA trailing update, RHS, two triangular solves) -> neb_eval (Phi, E at the M points).
metric = element-point influence pairs/s: copies x (N^2 + M N) pair evaluations per step divided by the whole step
time (LU and solves included in the time, not in the pair count).

  value : inputs already resident in HBM, outputs left in HBM
  e2e   : same step through the same public API with pinned HOST buffers (H2D of the geometry and the points, D2H of
          sigma, Phi and E inside the timed region)
  extra : (N = 1, default workload only; --no-extra skips) the two configurations that do not fit 25 steps:
          C3 — ONE full step (N = 49928 x 25 copies, 20 GB matrix, LU, all 1e7 points) and
          C4 — ALL 10 self-consistent steps with 1e6 charges on the resident C3 factors,
          each with its own stages_ms and roofline fractions.
  N > 1 : one process per GPU (torchrun); the LU does not shard (replicas), every rank factorises its
          replica and evaluates ITS OWN points: weak scaling, no data-path collective; time = max over ranks.

Roofline constants are not typed in: flop per pair and DRAM bytes per launch come from the ncu tables committed under
profiles/ (r2_opcounts.md: smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on per pair for every kernel path;
r2_bench_kernels.md: dram__bytes of the bench's own launches); peaks are measured in this process.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import re
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "element-point influence pairs/s (fp64)"
UNIT = "pairs/s"
DEFAULT_WORKLOAD = "C2"
# cases of profiles/r2_opcounts.md that count the same pairs with every element evaluated on its own (NEB_OPT_PAIR_STRIPS = 0)
ELEMENTWISE_CASE = {"eval_rect_uniform": "eval_rect_single", "eval_images": "eval_images_single"}
L2_NOTE = "256 MiB buffer written between timed steps; the matrix exceeds L2"
WORKLOADS = {
    "C1": "C1 cube: N=6144 rect panels, M=100000 points (BASELINE configs[1])",
    "C2": "C2 THGEM cell: N=19400 rectangles + right triangles, 4608 dielectric rows, 100^3 grid (BASELINE configs[2])",
    "C3": "C3 double THGEM: N=49928, 5x5 image copies, 1e7 points uniform in the cell (BASELINE configs[3])",
    "C4": "C4 space charge on the C3 geometry: per step E at the 1e6 charges (panels + all other charges), push, "
          "RHS update, re-solve on the resident LU factors (BASELINE configs[4]); assembly + LU done once before",
}


# ---------------------------------------------------------------------------------------------------------------
# constants from the committed ncu tables
# ---------------------------------------------------------------------------------------------------------------
def _md_table(path):
    """Rows of the first pipe table of a markdown file as dicts keyed by the header cells."""
    rows, hdr = [], None
    with open(path) as fh:
        for line in fh:
            if not line.startswith("|"):
                if hdr and rows:
                    break
                continue
            cells = [c.strip() for c in line.strip().strip("|").split("|")]
            if hdr is None:
                hdr = cells
            elif not all(re.fullmatch(r":?-+:?", c) for c in cells):
                rows.append(dict(zip(hdr, cells)))
    return rows


def load_opcounts():
    """case -> {dfma, dmul, dadd, flop, fp64_instr, dram} per pair / per launch (profiles/r2_opcounts.md)."""
    out = {}
    for r in _md_table(os.path.join(ROOT, "profiles", "r2_opcounts.md")):
        out[r["case"]] = dict(dfma=float(r["DFMA/pair"]), dmul=float(r["DMUL/pair"]), dadd=float(r["DADD/pair"]),
                              flop=2 * float(r["DFMA/pair"]) + float(r["DMUL/pair"]) + float(r["DADD/pair"]),
                              fp64_instr=float(r["FP64-pipe instr/pair"]))
    return out


def load_bench_traffic():
    """(workload, kernel) -> dram bytes per launch of the bench's own launch (profiles/r2_bench_kernels.md), if captured."""
    path = os.path.join(ROOT, "profiles", "r2_bench_kernels.md")
    out = {}
    if os.path.exists(path):
        for r in _md_table(path):
            out[(r["workload"], r["kernel"])] = float(r["dram read B"]) + float(r["dram write B"])
    return out


def flop_per_pair(pr, ops):
    """Counted flop of one (point, element copy) pair, averaged over the mesh: rectangles and right triangles on the
    path most of their pairs take (uniform-axes window, far branch; with image copies: the copy loop's count), wires
    on theirs.  Windows that are not uniform and near-branch pairs cost more than counted: a lower bound."""
    n_tri, n_wire = int(np.sum(pr.kind == 1)), int(np.sum(pr.kind == 2))
    rect = ops["eval_images" if pr.n_img > 1 else "eval_rect_uniform"]
    fl = (rect["flop"] * (pr.n - n_tri - n_wire) + ops["eval_tri_uniform"]["flop"] * n_tri + ops["eval_wire"]["flop"] * n_wire) / pr.n
    inst = (rect["fp64_instr"] * (pr.n - n_tri - n_wire) + ops["eval_tri_uniform"]["fp64_instr"] * n_tri
            + ops["eval_wire"]["fp64_instr"] * n_wire) / pr.n
    return fl, inst


# ---------------------------------------------------------------------------------------------------------------
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


# ---------------------------------------------------------------------------------------------------------------
# the CPU oracle as baseline / reference arm
# ---------------------------------------------------------------------------------------------------------------
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
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        # torchrun sets OMP_NUM_THREADS=1 for its workers; the one rank that runs the oracle gets the box's cores back
        # (read by the OpenMP runtime when the oracle's library is loaded, below)
        os.environ["OMP_NUM_THREADS"] = str(len(os.sched_getaffinity(0)))
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


# ---------------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------------
class Runner:
    """One workload on one GPU: device and pinned copies of the inputs, the step functions, and the measurements."""

    def __init__(self, name, pr, dev, P, ops, traffic, peaks, pinned=True):
        import torch
        self.torch, self.P, self.name, self.pr, self.dev = torch, P, name, pr, dev
        self.ops, self.traffic, self.peaks = ops, traffic, peaks
        self.is_c4 = name == "C4"
        self.pinned = pinned
        pts_np = pr.charge_pos if self.is_c4 else pr.points
        self.n, self.m = pr.n, pts_np.shape[1]
        self.copies = max(1, pr.n_img)
        self.q = self.m if self.is_c4 else 0
        # pair evaluations per step (image copies count as pairs; C4: + charge-charge and charge-collocation pairs)
        self.pairs_step = self.copies * self.m * self.n + (self.q * self.q + self.n * self.q if self.is_c4 else self.copies * self.n * self.n)
        self.nb = P.Neb(dev.index)
        geo = dict(kind=(pr.kind, torch.int32), v0=(pr.v0, torch.float64), e1=(pr.e1, torch.float64), e2=(pr.e2, torch.float64),
                   bc_kind=(pr.bc_kind, torch.int32), bc_value=(pr.bc_value, torch.float64), radius=(pr.radius, torch.float64),
                   eps_plus=(pr.eps_plus, torch.float64), eps_minus=(pr.eps_minus, torch.float64),
                   img_shift=(pr.img_shift, torch.float64))
        self.d = {k: self._dev(a, t) for k, (a, t) in geo.items()}
        self.h = {k: self._pin(None if a is None else np.asarray(a).astype(np.int32 if t == torch.int32 else np.float64))
                  for k, (a, t) in geo.items()}
        self.d_pts = self._dev(pts_np, torch.float64)
        self.h_pts = self._pin(pts_np)
        self.d_sig = torch.empty(self.n, dtype=torch.float64, device=dev)
        self.h_sig = torch.empty(self.n, dtype=torch.float64).pin_memory() if pinned else None
        self.d_phi = None if self.is_c4 else torch.empty(self.m, dtype=torch.float64, device=dev)
        self.h_phi = None if (self.is_c4 or not pinned) else torch.empty(self.m, dtype=torch.float64).pin_memory()
        self.d_E = torch.empty((3, self.m), dtype=torch.float64, device=dev)
        self.h_E = torch.empty((3, self.m), dtype=torch.float64).pin_memory() if pinned else None
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        if self.is_c4:
            self.mu_dt = pr.meta["mu"] * pr.meta["dt"]
            self.d_ch = self._dev(pr.charge_q, torch.float64)
            self.h_ch = self._pin(pr.charge_q)
            self.h2d = (3 * self.m + 3 * self.m + 3 * self.m + 3 * self.m + self.m) * 8    # eval points, pos+E for the push, pos+q
            self.d2h = (3 * self.m + 3 * self.m + self.n) * 8                              # E, pushed positions, sigma
        else:
            self.h2d = sum(v.numel() * v.element_size() for v in self.d.values() if v is not None) + 3 * self.m * 8
            self.d2h = (self.n + self.m + 3 * self.m) * 8

    def _dev(self, a, dtype):
        return None if a is None else self.torch.from_numpy(np.ascontiguousarray(a)).to(dtype).to(self.dev)

    def _pin(self, a):
        return None if (a is None or not self.pinned) else self.torch.from_numpy(np.ascontiguousarray(a)).pin_memory()

    def assemble_from(self, a):
        self.nb.assemble(a["kind"], a["v0"], a["e1"], a["e2"], a["bc_kind"], a["bc_value"], radius=a["radius"],
                         eps_plus=a["eps_plus"], eps_minus=a["eps_minus"], img_shift=a["img_shift"])

    def prepare_c4(self):
        """C4 (reading S22): geometry assembled and factorised ONCE, outside the timed steps."""
        self.assemble_from(self.d)
        self.nb.add_space_charge(self.d_pts, self.d_ch)
        self.nb.solve(out=self.d_sig)

    def step_resident(self):
        nb = self.nb
        if self.is_c4:
            nb.eval(self.d_pts, E=self.d_E, want_phi=False)
            nb.push(self.d_pts, self.d_E, self.mu_dt)
            nb.add_space_charge(self.d_pts, self.d_ch, replace=True)
            nb.solve(out=self.d_sig)
        else:
            self.assemble_from(self.d)
            nb.solve(out=self.d_sig)
            nb.eval(self.d_pts, phi=self.d_phi, E=self.d_E)

    def step_e2e(self):
        nb = self.nb
        if self.is_c4:
            nb.eval(self.h_pts, E=self.h_E, want_phi=False)
            nb.push(self.h_pts, self.h_E, self.mu_dt)
            nb.add_space_charge(self.h_pts, self.h_ch, replace=True)
            nb.solve(out=self.h_sig)
        else:
            self.assemble_from(self.h)
            nb.solve(out=self.h_sig)
            nb.eval(self.h_pts, phi=self.h_phi, E=self.h_E)

    def timed(self, fn, steps, barrier, max_over_ranks):
        torch = self.torch
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        per = []
        for e0, e1 in ev:
            self.flush.fill_(1)                     # L2 flush, outside the timed interval
            e0.record()
            fn()
            e1.record()
        barrier()
        per = [e0.elapsed_time(e1) for e0, e1 in ev]
        return max_over_ranks(sum(per)), per

    def staged(self, gathered_steps=0):
        """Per-stage CUDA-event times on the library's stream (per step) and the work counters: from one extra profiled
        step, or (gathered_steps > 0) from the stage timers that ran during that many timed steps."""
        nb, B = self.nb, self.P.binding
        if not gathered_steps:
            nb.set_option(B.NEB_OPT_PROFILE, 1)
            nb.reset_stats()
            self.flush.fill_(1)
            self.step_resident()
        st = nb.stage_ms()
        div = max(1, gathered_steps)
        stages = {k: round(v[0] / div, 4) for k, v in st.items()}
        launches = {k: int(round(v[1] / div)) for k, v in st.items()}
        counters = {"gemm_flop": nb.counter(0), "lu_flop": nb.counter(1), "matrix_bytes": nb.counter(2)}
        if not self.is_c4:
            # the trailing update alone is only timed without look-ahead (with it, it overlaps the next panels)
            nb.set_option(B.NEB_OPT_LU_LOOKAHEAD, 0)
            nb.reset_stats()
            self.flush.fill_(1)
            self.assemble_from(self.d)
            nb.solve(out=self.d_sig)
            serial = nb.stage_ms()
            stages["lu_gemm"] = round(serial["lu_gemm"][0], 4)
            stages["lu_no_lookahead"] = round(serial["lu"][0], 4)
            launches["lu_gemm"] = int(serial["lu_gemm"][1])
            nb.set_option(B.NEB_OPT_LU_LOOKAHEAD, 1)
        nb.set_option(B.NEB_OPT_PROFILE, 0)
        return stages, launches, counters

    def rooflines(self, stages, launches, counters):
        """Roofline objects of the kernels that carry the step, largest share of the step first."""
        pr, ops = self.pr, self.ops
        dfma, dmma = self.peaks["dfma"], self.peaks["dmma"]
        fl, inst = flop_per_pair(pr, ops)
        rect_key = "eval_images" if pr.n_img > 1 else "eval_rect_uniform"
        out = []
        eval_ms = stages["eval"] / max(1, launches["eval"])
        eval_pairs = self.copies * self.m * self.n
        ach = fl * eval_pairs / (eval_ms * 1e-3) * 1e-12
        out.append((stages["eval"], {
            "bound": "alu", "kernel": "eval_kernel<MathFast> (a7)", "achieved": ach, "peak": dfma, "unit": "TFLOP/s", "frac": ach / dfma,
            "traffic": self.traffic.get((self.name, "eval_kernel")), "kernel_ms": eval_ms, "flop_per_pair": fl,
            "fp64_instr_per_pair": inst, "fp64_pipe_slot_frac": inst * eval_pairs / (eval_ms * 1e-3) / (0.5e12 * dfma),
            "pairs_per_s_kernel": eval_pairs / (eval_ms * 1e-3), "field_map_points_per_s": self.m / (eval_ms * 1e-3),
            "frac_of_3operand_dfma_peak": ach / self.peaks["dfma3"],
            # the same pairs at the element-by-element operation count (strip pairs share an edge's two corner distances and
            # its logarithm: fewer executed flop for the same closed forms; profiles/r2_opcounts.md)
            "frac_elementwise": ach / dfma * ops[ELEMENTWISE_CASE[rect_key]]["flop"] / ops[rect_key]["flop"],
            "peak_source": "neb_fp64_peak(0): DFMA-chain microbenchmark run in this process (nominal 148 SM x 64 DFMA/clk x "
                           "2 x 1.965 GHz = 37.2); MEASURED_PEAKS.json has no FP64 entry",
            "constants_source": "profiles/r2_opcounts.md (ncu smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on per pair)"}))
        if stages.get("lu_gemm"):
            g_ms, g_n = stages["lu_gemm"], max(1, launches["lu_gemm"])
            ach = counters["gemm_flop"] / (g_ms * 1e-3) * 1e-12
            out.append((g_ms, {
                "bound": "tensor", "kernel": "gemm_kernel (a5 trailing update, FP64 DMMA mma.sync.m8n8k4)", "achieved": ach, "peak": dmma,
                "unit": "TFLOP/s", "frac": ach / dmma, "traffic": self.traffic.get((self.name, "gemm_kernel")),
                "kernel_ms": g_ms / g_n, "launches_per_step": g_n, "flop_per_step": counters["gemm_flop"],
                "peak_source": "neb_fp64_peak(1): mma.sync.m8n8k4.f64 register-only microbenchmark run in this process; "
                               "MEASURED_PEAKS.json holds bf16 only (its bf16 figure x the nominal 40/2250 FP64:bf16 tensor "
                               "ratio would give a LOWER peak: " + f"{self.peaks['dmma_from_bf16']:.1f})",
                "timed": "all launches of one factorisation without look-ahead (with it they overlap the panels)"}))
        if stages.get("charges"):
            c_ms = stages["charges"]                      # per step: E at the charges (m x q pairs) + the RHS update (n x q)
            pairs = self.m * self.q + self.n * self.q
            ach = ops["charges"]["flop"] * pairs / (c_ms * 1e-3) * 1e-12
            out.append((stages["charges"], {
                "bound": "alu", "kernel": "charge_kernel (a8)", "achieved": ach, "peak": dfma, "unit": "TFLOP/s", "frac": ach / dfma,
                "traffic": self.traffic.get((self.name, "charge_kernel")), "kernel_ms": c_ms, "flop_per_pair": ops["charges"]["flop"],
                "pairs_per_s_kernel": pairs / (c_ms * 1e-3), "frac_of_3operand_dfma_peak": ach / self.peaks["dfma3"],
                "fp64_pipe_slot_frac": ops["charges"]["fp64_instr"] * pairs / (c_ms * 1e-3) / (0.5e12 * dfma)}))
        if stages.get("assemble"):
            a_ms = stages["assemble"]
            pairs = self.copies * self.n * self.n
            afl = ops["assemble_images" if self.copies > 1 else "assemble_c2"]["flop"]
            ach = afl * pairs / (a_ms * 1e-3) * 1e-12
            out.append((a_ms, {
                "bound": "alu", "kernel": "assemble_kernel<MathFast> (a3)", "achieved": ach, "peak": dfma, "unit": "TFLOP/s",
                "frac": ach / dfma, "traffic": self.traffic.get((self.name, "assemble_kernel")), "kernel_ms": a_ms,
                "flop_per_pair": afl, "pairs_per_s_kernel": pairs / (a_ms * 1e-3),
                "matrix_write_gbs": counters["matrix_bytes"] / (a_ms * 1e-3) * 1e-9, "hbm_peak_gbs": self.peaks["hbm"]}))
        out.sort(key=lambda t: -t[0])
        step_ms = sum(v for k, v in stages.items() if k in ("geometry", "assemble", "equil", "lu", "rhs", "trisolve", "eval", "charges", "reduce"))
        for share_ms, r in out:
            r["share_of_step"] = share_ms / step_ms if step_ms else None
        return [r for _, r in out]

    def lu_summary(self, stages, counters):
        if not stages.get("lu"):
            return {"trisolve_ms": stages.get("trisolve"), "hbm_peak_gbs": self.peaks["hbm"],
                    "trisolve_gbs": 8.0 * self.n ** 2 / (stages["trisolve"] * 1e-3) * 1e-9 if stages.get("trisolve") else None}
        dmma = self.peaks["dmma"]
        whole = counters["lu_flop"] / (stages["lu"] * 1e-3) * 1e-12
        return {"tflops_whole_lu": whole, "whole_lu_frac_of_dmma_peak": whole / dmma,
                "tflops_trailing_update": counters["gemm_flop"] / (stages["lu_gemm"] * 1e-3) * 1e-12 if stages.get("lu_gemm") else None,
                "trailing_update_flop_share": counters["gemm_flop"] / counters["lu_flop"], "dmma_peak_tflops": dmma,
                "trisolve_gbs": 8.0 * self.n ** 2 / (stages["trisolve"] * 1e-3) * 1e-9 if stages.get("trisolve") else None,
                "hbm_peak_gbs": self.peaks["hbm"]}

    def close(self):
        self.nb.close()


def measure_peaks(P, local):
    nb = P.Neb(local)
    dfma, dmma, dfma3, dfma2c = nb.fp64_peak(0), nb.fp64_peak(1), nb.fp64_peak(2), nb.fp64_peak(3)
    nb.close()
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        hbm, src, bf16 = mp["hbm_gbs"], "MEASURED_PEAKS.json hbm_gbs (measured copy rate)", mp.get("bf16_tflops", 1590.0)
    except Exception:
        hbm, src, bf16 = 6650.0, "fallback 6.65 TB/s of B200_PROFILING.md", 1590.0
    return {"dfma": dfma, "dmma": dmma, "dfma3": dfma3, "dfma2c": dfma2c, "hbm": hbm, "hbm_source": src, "dmma_from_bf16": bf16 * 40.0 / 2250.0}


def extra_record(name, dev, P, ops, traffic, peaks, steps):
    """A full-size configuration that does not fit the 25-step line: `steps` timed steps after its own preparation."""
    import torch
    pr = load_problem(name)
    rn = Runner(name, pr, dev, P, ops, traffic, peaks, pinned=False)
    if rn.is_c4:
        rn.prepare_c4()
    ident = lambda x: x
    barrier = torch.cuda.synchronize
    # the stage timers run DURING the timed steps (an event pair per stage: microseconds against seconds per step)
    rn.nb.set_option(P.binding.NEB_OPT_PROFILE, 1)
    rn.nb.reset_stats()
    ms, per = rn.timed(rn.step_resident, steps, barrier, ident)
    stages, launches, counters = rn.staged(gathered_steps=steps)
    rec = {"config": make_config(name, pr, rn.m, rn.q), "steps": steps, "ms_per_step": ms / steps, "ms_each_step": [round(x, 2) for x in per],
           "value": rn.pairs_step * steps / (ms * 1e-3), "unit": UNIT, "stages_ms": stages,
           "rooflines": rn.rooflines(stages, launches, counters), "lu": rn.lu_summary(stages, counters)}
    rn.close()
    del rn
    torch.cuda.empty_cache()
    return rec


def dist_lu_record(dev, P):
    """SURVEY 8(f).4 on the one GPU at hand: the block-cyclic factorisation and solves of C2 driven by parallel.DistSolver
    with a single rank (every kernel of the distributed path runs; the broadcasts are no-ops), with and without
    look-ahead, beside which the single-GPU factorisation of the line can be read."""
    import torch
    from paper_2606_24154_b200 import parallel
    pr = load_problem("C2")
    out = {"workload": "C2", "n_elements": int(pr.n), "ranks": 1}
    for la in (True, False):
        nb = P.Neb(dev.index)
        ds = parallel.DistSolver(nb, lookahead=la)
        ds.assemble(pr)
        ds.factor()
        ds.solve()
        ds.assemble(pr)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        ds.factor()
        ev[1].record()
        ds.solve()
        ev[2].record()
        torch.cuda.synchronize()
        key = "lookahead" if la else "no_lookahead"
        out[f"factor_ms_{key}"] = ev[0].elapsed_time(ev[1])
        out[f"solve_ms_{key}"] = ev[1].elapsed_time(ev[2])
        out["lu_flop"] = nb.counter(1)
        nb.close()
    out["tflops_lookahead"] = out["lu_flop"] / (out["factor_ms_lookahead"] * 1e-3) * 1e-12
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS),
                    help="C2 is the bench line (with C3 and C4 as `extra` records); the others are one-off runs")
    ap.add_argument("--m-points", type=int, default=None, help="cap on the evaluation points (C3) / charges (C4)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the full-size C3 step and the 10 C4 steps")
    ap.add_argument("--set-option", action="append", default=[], metavar="ID=VALUE",
                    help="neb_set_option(ID, VALUE) on the bench context before the first step (A/B runs of a library option)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload in ("C1", "C2"):
        args.warmup = max(args.warmup, 3)          # the bench line; C3/C4 one-off runs may use fewer (long steps)

    import torch
    import torch.distributed as dist
    import paper_2606_24154_b200 as P
    from paper_2606_24154_b200 import parallel

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # NEB_BENCH_BACKEND=gloo: rehearsal of the multi-rank path on a box with fewer GPUs than ranks (the ranks then share
    # devices and the two collectives of this script, barrier and max, run on the host); never a measurement
    backend = os.environ.get("NEB_BENCH_BACKEND", "nccl")
    if backend != "nccl":
        local = local % max(1, torch.cuda.device_count())
    torch.cuda.set_device(local)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    dev = torch.device("cuda", local)
    ops, traffic = load_opcounts(), load_bench_traffic()
    peaks = measure_peaks(P, local)

    name = args.workload
    pr = load_problem(name, args.m_points, seed_shift=rank)   # same geometry on every rank, its own points / charges
    rn = Runner(name, pr, dev, P, ops, traffic, peaks)
    for kv in args.set_option:
        k, v = kv.split("=")
        rn.nb.set_option(int(k), int(v))
    if rn.is_c4:
        rn.prepare_c4()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    mx = lambda v: parallel.max_over_ranks(v, dev)
    for _ in range(args.warmup):
        rn.step_resident()
    torch.cuda.synchronize()
    sampler = ClockSampler()
    sampler.start()
    l0 = rn.nb.launch_count()
    ms, _ = rn.timed(rn.step_resident, args.steps, barrier, mx)
    launches = rn.nb.launch_count() - l0
    samples = sampler.stop()
    for _ in range(2):
        rn.step_e2e()
    ms_e2e, _ = rn.timed(rn.step_e2e, args.steps, barrier, mx)
    stages, st_launches, counters = rn.staged()
    roofs = rn.rooflines(stages, st_launches, counters)

    if rank == 0:
        line = {
            "metric": METRIC, "value": rn.pairs_step * args.steps * world / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": make_config(name, pr, rn.m, rn.q),
            **({"rehearsal": f"backend {backend}: ranks may share a GPU; not a measurement"} if backend != "nccl" else {}),
            "e2e": {"value": rn.pairs_step * args.steps * world / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": rn.h2d,
                    "d2h_bytes_per_step": rn.d2h, "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": launches, "clocks": _clocks_summary(samples),
            "roofline": roofs[0], "roofline_second": roofs[1] if len(roofs) > 1 else None, "rooflines_other": roofs[2:],
            "stages_ms": stages, "lu": rn.lu_summary(stages, counters),
            "peaks": {"fp64_dfma_tflops": peaks["dfma"], "fp64_dmma_tflops": peaks["dmma"], "fp64_dfma_3operand_tflops": peaks["dfma3"],
                      "fp64_dfma_2operand_const_tflops": peaks["dfma2c"],
                      "hbm_gbs": peaks["hbm"],
                      "hbm_source": peaks["hbm_source"]},
        }
        if not args.no_cpu_baseline and world == 1:
            if name == "C1":
                line["cpu_baseline"] = cpu_baseline_run(pr, with_lu=True)      # the whole C1 step, LU included
            elif not rn.is_c4:
                per_unit = rn.n * rn.copies                                    # pairs per assembly row / per point
                line["cpu_baseline"] = cpu_baseline_run(pr, max(1, int(2e8 // per_unit)), max(1, int(1.8e9 // per_unit)))
    rn.close()
    del rn
    torch.cuda.empty_cache()
    if rank == 0 and world == 1 and name == DEFAULT_WORKLOAD and not args.no_extra:
        line["extra"] = {"C3": extra_record("C3", dev, P, ops, traffic, peaks, steps=1),
                         "C4": extra_record("C4", dev, P, ops, traffic, peaks, steps=10),
                         "dist_lu_one_rank": dist_lu_record(dev, P)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
