#!/usr/bin/env python
"""bench.py -- BiCGSTAB iterations/s of the Poisson-Fermi hot path on BASELINE.json configs[3]
(256^3 fp64 channel grid), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 256] [--stencil onthefly|stored]
    python bench.py --impl reference ...      # the CPU oracle on the host cores (bounded sample)

One STEP = one pass of the whole hot path:
  rows L1-L2  pf_grid_create + pf_grid_set_workspace: eps scan, node classes, diagonal, (stored
              off-diagonals), fixed-charge deposition
  rows N1-N5  pf_solve_pf capped at one outer iteration with 25 fixed iterations per linear solve:
              initial guess, fused Fermi kernel, PF1, PF2, relaxation + max-norm (3 x 25 iterations)
  rows L3-L8  pf_solve_linear, tol = 0, 200 fixed Jacobi-BiCGSTAB iterations (configs[3] (ii))
value = BiCGSTAB iterations of the step (275) / step time, whole job.  Inputs are resident in HBM
for `value`; `e2e` repeats the step through the C ABI with HOST buffers (copies inside the timing).
Multi-GPU: the path does not shard (replicas only) -- every rank runs the same step.

Beside `value` the line carries, all measured in the same run (N = 1):
  roofline   the whole BiCGSTAB iteration (every kernel of the hot loop bracketed by CUDA events on the library's
             stream) against the measured HBM peak, per-kernel figures and the kernel furthest below its roofline
  variants   the same step with the stored-coefficient stencil (configs[3]'s comparison) and with the merged
             two-reduction solver (--solver merged) -- whichever is not the main configuration
  pf_solve   wall time and iteration counts of the full nonlinear PF solve of configs[2] (the metric's third part)
  cpu_baseline, e2e, clocks, gpu_launches as the contract says.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

LINEAR_ITERS = 200
PF_INNER_ITERS = 25
STEP_ITERS = LINEAR_ITERS + 3 * PF_INNER_ITERS
PROFILE_ITERS = 8       # iterations per linear solve whose three kernels are bracketed by CUDA events
                        # (launched one by one; the other iterations run as CUDA-graph replays)
METRIC = "bicgstab_iterations_per_s"
UNIT = "iterations/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", "--grid", dest="n", type=int, default=0, help="grid nodes per direction (default: 256 for configs[3], 512 for configs[4])")
    ap.add_argument("--workload", choices=["config3", "config4"], default="config3",
                    help="config3: the metric's 256^3 channel grid (default); config4: the 512^3 bandwidth stress "
                         "(100 fixed iterations + one PF pass, BASELINE.json configs[4])")
    ap.add_argument("--stencil", choices=["onthefly", "stored"], default="onthefly")
    ap.add_argument("--kernels", choices=["auto", "direct", "tiled"], default="auto")
    ap.add_argument("--launch-mode", choices=["auto", "loop", "chunks", "stream"], default="auto",
                    help="how the iterations reach the GPU (PF_OPT_GRAPH): auto = library default (device-side loop for "
                         "short solves, polled graph replays for long ones); loop = one graph per solve whose WHILE "
                         "node repeats the iterations on the device; chunks = graph replays of 16 iterations polled "
                         "by the host (ncu does not profile kernel nodes of graphs with conditional nodes: launch "
                         "lists are taken with this mode); stream = plain launches")
    ap.add_argument("--diag-from-code", type=int, choices=[0, 1, 2], default=None,
                    help="PF_OPT_DIAG_FROM_CODE of the timed steps (default: the library's own, 1): 0 the diagonal is read, "
                         "1 k1 takes it from the stencil codes, 2 k2 as well")
    ap.add_argument("--solver", choices=["table3", "merged"], default="table3",
                    help="table3: BiCGSTAB as Table 3 writes it, three kernels per iteration (the default, whose parity "
                         "reference is the oracle's Table 3); merged: the two-reduction recurrence (PF_OPT_SOLVER = 1, "
                         "reading M1), two kernels per iteration")
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-variants", action="store_true", help="skip the stored / merged variants of the step")
    ap.add_argument("--no-pf-solve", action="store_true", help="skip the full nonlinear PF solve of configs[2]")
    ap.add_argument("--ref-iters", type=int, default=4, help="oracle iterations per reference step")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_bytes_per_unknown(stored: bool, merged: bool = False) -> dict:
    """Algorithmic HBM bytes per unknown per launch: every input vector
    read once, every output written once, halos served on chip."""
    # k1 reads r, p, v, A0, r~ and writes p', v'; k2 reads r, v', A0 and writes t; k3 reads r, v', p', y, t, r~
    # and writes y, r; the on-the-fly variant adds a 2-byte stencil code per node to k1 and k2, the stored
    # variant six 8-byte off-diagonals.  The per-kernel events bracket iterations of the 200-iteration Poisson
    # solve only; there the on-the-fly k1 does not read A0 (it is a function of the code: PF_OPT_DIAG_FROM_CODE).
    # Merged solver (on-the-fly stencil; the events bracket its two kernels in the slots of k2 and k3): K2M reads r, v, A0,
    # r~ and the codes and writes t; K31 reads r, p, v, t, r~, y and the codes (the diagonal comes from them in a Poisson
    # solve) and writes r', p', v', y.
    if merged:
        return {"k2": (4 + 1) * 8 + 2, "k3": (6 + 4) * 8 + 2}
    if stored:
        return {"k1": (5 + 6 + 2) * 8, "k2": (3 + 6 + 1) * 8, "k3": (6 + 2) * 8}
    return {"k1": (4 + 2) * 8 + 2, "k2": (3 + 1) * 8 + 2, "k3": (6 + 2) * 8}


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores
# ---------------------------------------------------------------------------------------------------

def oracle_sample(w, iters: int):
    """Assembly + `iters` fixed Jacobi-BiCGSTAB iterations of the workload in the CPU oracle; seconds."""
    from oracle import pf_oracle as oracle
    import numpy as np
    rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges) if w.rhs is None else w.rhs
    t0 = time.perf_counter()
    out = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=0.0, maxit=iters)
    dt = time.perf_counter() - t0
    assert out["iters"] == iters and np.isfinite(out["relres"])
    return dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1711_04060_b200 import workloads as wl
    from oracle import pf_oracle as oracle
    oracle.build()
    w, _, wdesc = make_workload(args)
    args.n = w.nx
    for _ in range(args.warmup):
        oracle_sample(w, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample(w, args.ref_iters)
    dt = time.perf_counter() - t0
    value = args.steps * args.ref_iters / dt
    sample = (f"per step: DIA assembly + {args.ref_iters} fixed Jacobi-BiCGSTAB iterations of the {args.n}^3 "
              f"{args.workload} workload, single thread, g++ -O2")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wdesc, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# B200 arm
# ---------------------------------------------------------------------------------------------------

def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1711_04060_b200 import pf, workloads as wl

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU fallback")
    from paper_1711_04060_b200 import build as _build
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        _build.build()          # no-op when the in-tree library is up to date
    else:                       # the other ranks wait for rank 0's build
        t_wait = time.time()
        while _build._stale() and time.time() - t_wait < 600:
            time.sleep(1.0)
    pf.load()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w, lin_iters, wdesc = make_workload(args)
    args.n = w.nx
    step_iters = lin_iters + 3 * PF_INNER_ITERS
    sp = w.species
    n = w.n
    stencil = pf.STENCIL_STORED if args.stencil == "stored" else pf.STENCIL_ONTHEFLY
    kernels = {"auto": 0, "direct": 1, "tiled": 2}[args.kernels]
    rng = np.random.default_rng(3)
    rhs_np = rng.standard_normal(n) if w.rhs is None else w.rhs    # configs[3]: timing RHS, dense random
    eps_host = torch.tensor(w.eps).pin_memory()
    rhs_host = torch.tensor(rhs_np).pin_memory()
    x_host = torch.zeros(n, dtype=torch.float64).pin_memory()
    phi_host = torch.zeros(n, dtype=torch.float64).pin_memory()
    eps_dev = eps_host.cuda()
    # e2e: the eps map of the NEXT step is uploaded into the other of two device buffers while the current step's linear
    # solve runs (every step still uploads its own inputs inside the timed region; only the first upload is exposed)
    eps_bufs = [torch.empty_like(eps_dev), torch.empty_like(eps_dev)]
    eps_state = {"cur": 0, "ready": None}
    rhs_dev = rhs_host.cuda()
    x_dev = torch.zeros(n, dtype=torch.float64, device="cuda")
    phi_dev = torch.zeros(n, dtype=torch.float64, device="cuda")

    # workspace is allocated once, outside the timing: it is caller-owned scratch by the ABI
    def make_cfg(stencil_name: str, solver_name: str) -> dict:
        st = pf.STENCIL_STORED if stencil_name == "stored" else pf.STENCIL_ONTHEFLY
        probe = pf.pf_grid_create(w.nx, w.ny, w.nz, w.h, eps_dev, w.charges, w.bc_type, w.bc_value)
        pf.pf_grid_set_option(probe, pf.PF_OPT_STENCIL, st)
        wsp = torch.empty(pf.pf_grid_workspace_bytes(probe), dtype=torch.uint8, device="cuda")
        pf.pf_grid_destroy(probe)
        return dict(stencil=st, stencil_name=stencil_name, solver=1 if solver_name == "merged" else 0,
                    solver_name=solver_name, ws=wsp, prof={k: dict(ms=0.0, launches=0) for k in ("k1", "k2", "k3")})

    main_cfg = make_cfg(args.stencil, args.solver)
    side = torch.cuda.Stream()
    ws, prof_tot = main_cfg["ws"], main_cfg["prof"]

    def step(host_buffers: bool, profile: bool, cfg: dict = None):
        cfg = cfg or main_cfg
        ws, prof_tot = cfg["ws"], cfg["prof"]
        eps_in = eps_dev
        if host_buffers:
            eps_in = eps_bufs[eps_state["cur"]]
            if eps_state["ready"] is None:
                eps_in.copy_(eps_host, non_blocking=True)              # no step before this one: upload in line
            else:
                torch.cuda.current_stream().wait_event(eps_state["ready"])
        h = pf.pf_grid_create(w.nx, w.ny, w.nz, w.h, eps_in, w.charges, w.bc_type, w.bc_value)
        pf.pf_grid_set_option(h, pf.PF_OPT_STENCIL, cfg["stencil"])
        if kernels:
            pf.pf_grid_set_option(h, pf.PF_OPT_KERNELS, kernels)
        pf.pf_grid_set_option(h, pf.PF_OPT_GRAPH, {"auto": 3, "loop": 2, "chunks": 1, "stream": 0}[args.launch_mode])
        pf.pf_grid_set_option(h, pf.PF_OPT_SOLVER, cfg["solver"])
        if args.diag_from_code is not None:
            pf.pf_grid_set_option(h, pf.PF_OPT_DIAG_FROM_CODE, args.diag_from_code)
        pf.pf_grid_set_option(h, pf.PF_OPT_LINEAR_TOL, 0.0)
        pf.pf_grid_set_option(h, pf.PF_OPT_LINEAR_MAXIT, PF_INNER_ITERS)
        pf.pf_grid_set_option(h, pf.PF_OPT_MAX_OUTER, 1)
        pf.pf_grid_set_workspace(h, ws)                                            # rows L1, L2
        if host_buffers:
            # the upload of rhs and x0 runs on the grid's copy stream while the PF pass computes
            x_host.zero_()
            pf.pf_grid_stage_host(h, n, rhs_host, x_host)
        res = pf.pf_solve_pf(h, n, sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, phi_dev)  # N1-N5
        assert res["linear_iters"] == 3 * PF_INNER_ITERS, res
        if host_buffers:
            # ... and phi goes back to the host on a side stream while the linear solve runs
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                phi_host.copy_(phi_dev, non_blocking=True)
        if profile:      # the events bracket iterations of the long linear solve only (the PF pass runs unprofiled)
            pf.pf_grid_set_option(h, pf.PF_OPT_PROFILE, PROFILE_ITERS)
        if host_buffers:
            with torch.cuda.stream(side):                               # the next step's eps, behind the phi download
                eps_bufs[eps_state["cur"] ^ 1].copy_(eps_host, non_blocking=True)
                eps_state["ready"] = torch.cuda.Event()
                eps_state["ready"].record(side)
            eps_state["cur"] ^= 1
            out = pf.pf_solve_linear_host(h, n, rhs_host, x_host, 0.0, lin_iters, true_residual=False)
        else:
            x_dev.zero_()
            if cfg.get("solve_events") is not None:      # the linear solve alone between two CUDA events
                ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                ev[0].record()
            out = pf.pf_solve_linear(h, n, rhs_dev, x_dev, 0.0, lin_iters, true_residual=False)   # rows L3-L8
            if cfg.get("solve_events") is not None:
                ev[1].record()
                cfg["solve_events"].append(ev)
        assert out["iters"] == lin_iters, out
        if profile:
            p = pf.pf_grid_profile(h)
            for k in prof_tot:
                prof_tot[k]["ms"] += p[k]["ms"]
                prof_tot[k]["launches"] += p[k]["launches"]
            pf.pf_grid_set_option(h, pf.PF_OPT_PROFILE, 0)
        if host_buffers:
            side.synchronize()
            torch.cuda.current_stream().wait_stream(side)      # phi_dev is rewritten by the next step
        pf.pf_grid_destroy(h)
        return out

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, host_buffers, profile, cfg=None, sync=True):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if sync:
            barrier()
        else:
            torch.cuda.synchronize()
        e0.record()
        for _ in range(nsteps):
            step(host_buffers, profile, cfg)
        e1.record()
        if sync:
            barrier()
        else:
            torch.cuda.synchronize()
            return e0.elapsed_time(e1)
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item())

    for _ in range(max(args.warmup, 3)):
        step(False, False)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = pf.pf_launch_count()
    ms_total = timed(args.steps, False, True)
    launches = pf.pf_launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None

    e2e = None
    if not args.no_e2e:
        step(True, False)
        e2e_steps = max(1, min(args.steps, 3))
        ms_e2e = timed(e2e_steps, True, False)
        e2e = {"value": world * step_iters * e2e_steps / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": 8 * n * 3, "d2h_bytes_per_step": 8 * n * 2,
               "ms_per_step": ms_e2e / e2e_steps,
               "what": "eps, rhs, x0 host->device; x, phi device->host; C-ABI pf_grid_stage_host + pf_solve_linear_host: the "
                       "rhs/x0 upload overlaps the PF pass, the phi download and the next step's eps upload the linear solve; "
                       "the x download is exposed"}

    if rank == 0:
        peak, peak_src = measured_peak_gbs()

        def roofline_of(cfg: dict) -> dict:
            """Per-kernel and per-iteration roofline figures from the CUDA-event brackets of a configuration."""
            stored, merged = cfg["stencil_name"] == "stored", cfg["solver_name"] == "merged"
            bpu = kernel_bytes_per_unknown(stored, merged)
            names = {"k1": "k1 (p-update + matvec + r~.v)", "k2": "k2 (s-update + matvec + t.s, t.t)",
                     "k3": "k3 (x, r update + r~.r, r.r)"}
            tnames = {"k1": "k1", "k2": "k2", "k3": "k3"}
            if merged:
                names = {"k2": "K2M (s-update + matvec + t.s, t.t, r~.t)",
                         "k3": "K31 (x, r, p update + matvec + r~.v, r.r, r~.r)"}
                tnames = {"k2": "k2m", "k3": "k31"}
            # DRAM bytes per launch from the committed ncu --set full capture (profiles/traffic.csv); static, not
            # measured in this run: the csv names the capture and its commit
            tr, tr_src = {}, None
            try:
                with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
                    for row in f:
                        c = [x.strip() for x in row.split(",")]
                        if len(c) >= 5 and c[0] == cfg["stencil_name"] and c[1] == str(args.n):
                            tr[c[2]] = int(c[3]); tr_src = c[4]
            except (OSError, ValueError):
                pass
            per = {}
            for k in ("k1", "k2", "k3"):
                if cfg["prof"][k]["launches"] and k in bpu:
                    avg_ms = cfg["prof"][k]["ms"] / cfg["prof"][k]["launches"]
                    gbs = bpu[k] * n / (avg_ms * 1e-3) / 1e9
                    per[k] = {"name": names[k], "avg_ms": avg_ms, "launches": cfg["prof"][k]["launches"],
                              "bytes_per_unknown": bpu[k], "gbs": gbs, "frac": gbs / peak,
                              "traffic": tr.get(tnames[k])}
            if not per:
                return None
            iter_ms = sum(per[k]["avg_ms"] for k in per)
            iter_b = sum(per[k]["bytes_per_unknown"] for k in per)
            gbs = iter_b * n / (iter_ms * 1e-3) / 1e9
            worst = min(per, key=lambda k: per[k]["frac"])
            tsum = None if any(per[k]["traffic"] is None for k in per) else sum(per[k]["traffic"] for k in per)
            # headline: the whole iteration (every kernel of the hot loop, launched one by one between CUDA events), not
            # the kernel that happens to take longest; the kernel furthest below its roofline is named beside it
            return {"bound": "hbm", "kernel": "one BiCGSTAB iteration = " + " + ".join(per[k]["name"].split(" ")[0] for k in per),
                    "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                    "frac_of_nominal_8000": gbs / 8000.0, "traffic": tsum,
                    "traffic_source": (("static: " + tr_src + "; not measured in this run") if tsum is not None else None),
                    "peak_source": peak_src, "bytes_per_unknown": iter_b, "ms": iter_ms,
                    "iterations_per_s_linear_solve": 1e3 / iter_ms, "mupdates_per_s": n / iter_ms / 1e3,
                    "worst_kernel": {"kernel": per[worst]["name"], "frac": per[worst]["frac"], "gbs": per[worst]["gbs"]},
                    "per_kernel": per}

        roofline = roofline_of(main_cfg)
        # The same iteration as it runs in production: the whole linear solve of a step (initial residual + lin_iters
        # iterations as graph replays / a device-side loop + the closing x update) between two CUDA events, without the
        # per-kernel events of the profile, divided by the iterations.  Includes the gaps between kernels.
        if roofline is not None and world == 1:
            main_cfg["solve_events"] = []
            for _ in range(3):
                step(False, False)
            torch.cuda.synchronize()
            ms_solve = min(a.elapsed_time(b) for a, b in main_cfg["solve_events"]) / lin_iters
            main_cfg["solve_events"] = None
            gbs = roofline["bytes_per_unknown"] * n / (ms_solve * 1e-3) / 1e9
            roofline["in_solve"] = {"ms_per_iteration": ms_solve, "achieved": gbs, "frac": gbs / peak,
                                    "frac_of_nominal_8000": gbs / 8000.0, "iterations_per_s": 1e3 / ms_solve,
                                    "what": f"whole {lin_iters}-iteration pf_solve_linear between two CUDA events / {lin_iters} "
                                            "(best of 3 steps after the timed region; no per-kernel events)"}

        # configs[3] asks for the stored-coefficient stencil beside the on-the-fly one; SURVEY 8(f) #3 for the merged
        # recurrence beside Table 3: the same step, each variant with its own workspace, timed in this run
        variants = {}
        if not args.no_variants and world == 1:      # (replicas: rank 0 must not keep the other ranks waiting)
            for name, (st, so) in {"stored": ("stored", "table3"), "onthefly": ("onthefly", "table3"),
                                   "merged": ("onthefly", "merged")}.items():
                if (st, so) == (args.stencil, args.solver):
                    continue
                cfg = make_cfg(st, so)
                for _ in range(3):
                    step(False, False, cfg)
                vsteps = max(1, min(args.steps, 5))
                ms_v = timed(vsteps, False, True, cfg, sync=False)
                r = roofline_of(cfg)
                variants[name] = {"stencil": st, "solver": so, "value": step_iters * vsteps / (ms_v * 1e-3), "unit": UNIT,
                                  "steps": vsteps, "ms_per_step": ms_v / vsteps,
                                  "iteration": None if r is None else {k: r[k] for k in ("ms", "bytes_per_unknown", "achieved", "frac",
                                                                                         "iterations_per_s_linear_solve")},
                                  "per_kernel": None if r is None else {k: {kk: v[kk] for kk in ("name", "avg_ms", "bytes_per_unknown", "frac")}
                                                                        for k, v in r["per_kernel"].items()}}
                del cfg
                torch.cuda.empty_cache()

        # the metric's third part, "PF total solve time": the full nonlinear solve of configs[2] (128^3, +50 mV) to its
        # own tolerances (linear 1e-10, increment 1e-8), wall clock around pf_solve_pf, after one warm-up solve
        pf_solve = None
        if not args.no_pf_solve and world == 1:
            w2 = wl.config2(volt_mv=50.0)
            g2 = pf.Grid.from_workload(w2, options={pf.PF_OPT_SOLVER: main_cfg["solver"]})
            sp2 = w2.species
            g2.solve_pf(sp2.valence, sp2.bath_molar, sp2.radii, w2.l_c, w2.nonlinear_tol, want_conc=False)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            o2 = g2.solve_pf(sp2.valence, sp2.bath_molar, sp2.radii, w2.l_c, w2.nonlinear_tol, want_conc=False)
            torch.cuda.synchronize()
            dt2 = time.perf_counter() - t0
            g2.close()
            pf_solve = {"workload": "configs[2] channel 128^3, Na+/Ca2+/Cl-/water, +50 mV, linear tol 1e-10, increment tol 1e-8",
                        "seconds": dt2, "status": o2["status"], "outer_iterations": o2["outer_iters"],
                        "linear_iterations": o2["linear_iters"], "solver": args.solver,
                        "us_per_linear_iteration": 1e6 * dt2 / max(o2["linear_iters"], 1)}
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            from oracle import pf_oracle as oracle
            oracle.build()
            cpu_iters = 3 if args.n >= 512 else (12 if args.n >= 256 else 100)
            dt = oracle_sample(w, cpu_iters)
            cpu = {"value": cpu_iters / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "host_cores_available": os.cpu_count(),
                   "sample": f"DIA assembly + {cpu_iters} fixed Jacobi-BiCGSTAB iterations of the same {args.n}^3 "
                             f"workload ({dt:.1f} s), single thread, g++ -O2"}
        value = world * step_iters * args.steps / (ms_total * 1e-3)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{wdesc}; step = assembly + {lin_iters} fixed Jacobi-BiCGSTAB iterations + "
                                       f"one PF outer pass with 3x{PF_INNER_ITERS} inner iterations",
                           "stencil": args.stencil, "kernels": args.kernels, "launch_mode": args.launch_mode,
                           "solver": args.solver, "unknowns": n,
                           "iterations_per_step": step_iters, "parallelism": "replicas only" if world > 1 else "1 GPU",
                           "l2": "inputs larger than L2 (working set %.1f GB)" % (ws.numel() / 1e9)},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
                "variants": variants, "pf_solve": pf_solve,
                "paper_context": "paper: 22.8x linear-solver, 16.9x total speedup, GTX TITAN X vs Xeon E5-1650 "
                                 "(PAPER.md:305-311); other hardware, context only"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def make_workload(args):
    """(workload, linear iterations per step, description)."""
    from paper_1711_04060_b200 import workloads as wl
    if args.workload == "config4":
        n = args.n or 512
        return wl.config4(n=n), 100, (f"configs[4] bandwidth stress {n}^3 fp64 (random spheres eps 2/80, 30 % fill, seed 4, "
                                      f"Gaussian-smeared right-hand side), h=0.5 A")
    n = args.n or 256
    return wl.config3(n=n), LINEAR_ITERS, (f"configs[3] channel {n}^3 fp64 (slab 60 A, pore 8 A, 1536 charges, seed 3), "
                                           f"h=0.5 A")


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
