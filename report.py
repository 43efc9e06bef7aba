"""Report table of BASELINE.md section 4: one row per config x stencil variant, GPU next to the CPU oracle.

    python report.py [--out gpurun_out/report.md] [--skip-512]
    python report.py --launch-ab [--out gpurun_out/launch_ab.md]     (PF_OPT_GRAPH 0 / 1 / 2 / 3)
    python report.py --omega-sweep [--out gpurun_out/omega.md]       (omega_PF 0 .. 0.7 on configs[2]'s PF solve)

Needs a CUDA device (the GPU columns) and builds the oracle for the CPU columns; the oracle is only ever
run where it finishes in about a minute (full solves up to 64^3, a few iterations beyond).
A measurement script beside bench.py, not part of the product package: paper_1711_04060_b200/ never imports oracle/.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1711_04060_b200 import pf, workloads as wl  # noqa: E402

PEAK_NOMINAL = 8000.0


def measured_peak():
    import json
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0


def bytes_per_iter(stored: bool, merged: bool = False) -> int:
    # Poisson solves (all linear rows of the table): the on-the-fly k1 takes the diagonal from the stencil code
    # (50 + 34 + 64 B); PF1 / PF2 solves move 156 B; merged solver: K2M 42 + K31 82 B
    return 248 if stored else (124 if merged else 148)


def ncu_dram_bytes_per_iter(stencil_name: str, n: int, merged: bool):
    """Sum over the kernels of one iteration of the DRAM bytes per launch that the committed ncu --set full capture
    measured (profiles/traffic.csv); None where no capture exists for this stencil and size."""
    want = ("k2m", "k31") if merged else ("k1", "k2", "k3")
    got = {}
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in f:
                c = [x.strip() for x in row.split(",")]
                if len(c) >= 4 and c[0] == stencil_name and c[1] == str(n) and c[2] in want:
                    got[c[2]] = int(c[3])
    except (OSError, ValueError):
        return None
    return sum(got.values()) if len(got) == len(want) else None


def rel_l2(a, b):
    d = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / (d if d > 0 else 1.0))


def gpu_fixed_iterations(w, rhs, stencil, iters, solver=0):
    """ms per iteration of `iters` fixed iterations (second of two runs), whole-solve CUDA-event time."""
    g = pf.Grid.from_workload(w, stencil=stencil, options={pf.PF_OPT_SOLVER: solver})
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    rhs_d = torch.as_tensor(rhs, dtype=torch.float64).cuda()
    ms = None
    for _ in range(2):
        x.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        pf.pf_solve_linear(g.handle, w.n, rhs_d, x, 0.0, iters, true_residual=False)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / iters
    g.close()
    return ms


def linear_rows(name, w, rhs, oracle, oracle_full: bool, oracle_iters: int, peak):
    rows = []
    ref_t = None
    o_s_per_it = None
    if oracle_full:
        t0 = time.perf_counter()
        ref_t = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=1e-10)
        o_s_per_it = (time.perf_counter() - t0) / max(ref_t["iters"], 1)
    elif oracle_iters:
        t0 = time.perf_counter()
        oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=0.0, maxit=oracle_iters)
        o_s_per_it = (time.perf_counter() - t0) / oracle_iters
    ref_m = None
    if oracle_full:
        ref_m = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=1e-10,
                                    solver=oracle.SOLVER_MERGED)
    for stencil, solver, sname in ((pf.STENCIL_STORED, 0, "stored"), (pf.STENCIL_ONTHEFLY, 0, "on-the-fly"),
                                   (pf.STENCIL_ONTHEFLY, 1, "on-the-fly, merged solver")):
        g = pf.Grid.from_workload(w, stencil=stencil, options={pf.PF_OPT_SOLVER: solver})
        out = g.solve_linear(rhs, tol=1e-10)
        x = out["x"].cpu().numpy()
        g.close()
        ms = gpu_fixed_iterations(w, rhs, stencil, 200 if w.n >= 128 ** 3 else 400, solver)
        bpi = bytes_per_iter(stencil == pf.STENCIL_STORED, solver == 1)
        gbs = bpi * w.n / (ms * 1e-3) / 1e9
        nb = ncu_dram_bytes_per_iter("stored" if stencil == pf.STENCIL_STORED else "onthefly", w.nx, solver == 1)
        ref = ref_m if solver == 1 else ref_t
        rows.append(dict(config=name, N=w.n, variant=sname,
                         iters=f"{out['iters']} / {ref['iters'] if ref else 'n/a'}",
                         relres=f"{out['true_relres']:.2e}",
                         diff=f"{rel_l2(x, ref['x']):.1e}" if ref else "n/a",
                         ms=f"{ms:.4f}", its=f"{1e3 / ms:.0f}", mup=f"{w.n / ms / 1e3:.0f}", bpi=bpi,
                         gbs=f"{gbs:.0f}", ncu=f"{nb / (ms * 1e-3) / 1e9:.0f}" if nb else "n/a", p8=f"{100 * gbs / PEAK_NOMINAL:.0f} %", pm=f"{100 * gbs / peak:.0f} %",
                         osit=f"{o_s_per_it:.3f}" if o_s_per_it else "n/a", outer="-", pft="-"))
    return rows


def pf_row(name, w, oracle, oracle_full: bool):
    sp = w.species
    g = pf.Grid.from_workload(w)
    g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)   # warm-up
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    torch.cuda.synchronize()
    tg = time.perf_counter() - t0
    g.close()
    to, diff, oiters = None, "n/a", "n/a"
    if oracle_full:
        t0 = time.perf_counter()
        ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence,
                              sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, lin_tol=w.linear_tol, max_outer=1000)
        to = time.perf_counter() - t0
        diff = f"{rel_l2(out['phi'].cpu().numpy(), ref['phi']):.1e}"
        oiters = f"{ref['outer_iters']} ({ref['linear_iters']} lin.)"
    return dict(config=name, N=w.n, variant="PF (auto)", iters=f"{out['linear_iters']} lin. / {oiters}",
                relres="-", diff=diff, ms=f"{1e3 * tg / max(out['linear_iters'], 1):.4f}", its="-", mup="-", bpi="-",
                gbs="-", ncu="-", p8="-", pm="-", osit="-", outer=str(out["outer_iters"]),
                pft=f"{tg:.2f} s / {to:.0f} s" if to else f"{tg:.2f} s / n/a")


def launch_mode_ab(out_path):
    """PF_OPT_GRAPH 0 / 1 / 2 / 3 (stream launches and graph replays polled by the host, device-side loop, auto) side by side:
    whole-solve CUDA-event times of linear solves of configs 2 and 3 and wall time of config 2's PF solve, each the
    best of three, modes interleaved; checks that the three modes return the same bits."""
    lines = ["| workload | iterations | mode 0 (stream, polled) | mode 1 (graph chunks, polled) | mode 2 (device loop) | mode 3 (auto, default) | same bits |",
             "|---|---:|---:|---:|---:|---:|---|"]
    for name, w in (("config 2, 128^3", wl.config2()), ("config 2 at 192^3", wl.config2(n=192)),
                    ("config 3, 256^3", wl.config3())):
        rhs = torch.from_numpy(np.random.default_rng(3).standard_normal(w.n)).cuda()
        for tol, maxit in ((0.0, 200), (1e-10, 10000)):
            best, xs, its = {}, {}, {}
            for rep in range(3):
                for mode in (0, 1, 2, 3):
                    g = pf.Grid.from_workload(w, options={pf.PF_OPT_GRAPH: mode})
                    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
                    for _ in range(2):
                        x.zero_()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        torch.cuda.synchronize()
                        e0.record()
                        out = pf.pf_solve_linear(g.handle, w.n, rhs, x, tol, maxit, true_residual=False)
                        e1.record()
                        torch.cuda.synchronize()
                    best[mode] = min(best.get(mode, 1e30), e0.elapsed_time(e1))
                    xs[mode], its[mode] = x.clone(), out["iters"]
                    g.close()
            same = all(torch.equal(xs[0], xs[m]) and its[0] == its[m] for m in (1, 2, 3))
            lines.append(f"| {name}, linear, tol {tol:g} | {its[2]} | {best[0]:.2f} ms | {best[1]:.2f} ms | {best[2]:.2f} ms | {best[3]:.2f} ms | {same} |")
    w = wl.config2()
    sp = w.species
    best, phis, its = {}, {}, {}
    for rep in range(2):
        for mode in (0, 1, 2, 3):
            g = pf.Grid.from_workload(w, options={pf.PF_OPT_GRAPH: mode})
            g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)   # warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)
            torch.cuda.synchronize()
            best[mode] = min(best.get(mode, 1e30), time.perf_counter() - t0)
            phis[mode], its[mode] = out["phi"].clone(), (out["outer_iters"], out["linear_iters"])
            g.close()
    same = all(torch.equal(phis[0], phis[m]) and its[0] == its[m] for m in (1, 2, 3))
    lines.append(f"| config 2, 128^3, PF solve | {its[2][0]} outer, {its[2][1]} linear | {best[0]:.3f} s | {best[1]:.3f} s | {best[2]:.3f} s | {best[3]:.3f} s | {same} |")
    text = "\n".join(lines) + "\n"
    os.makedirs(os.path.dirname(out_path), exist_ok=True)
    with open(out_path, "w") as f:
        f.write(text)
    print(text)


def iteration_counts(out_path):
    """Iterations to 1e-10 of the linear solve of configs 0-3, direct and tiled kernels, Table 3 and merged solver, beside
    the oracle's (run where it finishes in a minute): the evidence behind the rounding contract of DESIGN.md section 4.
    Run once with the product library and once with a -DPF_EXPERIMENT_PLAIN_DOT build (PF_B200_LIB)."""
    from oracle import pf_oracle as oracle
    oracle.build()
    lines = [f"library: {pf.LIB_PATH}", "",
             "| config | solver | kernels | iterations GPU | iterations oracle | true rel. residual | rel. L2 diff vs oracle |",
             "|---|---|---|---:|---:|---:|---:|"]
    for name, w in (("0 (32^3)", wl.config0()), ("1 (64^3)", wl.config1()), ("2 (128^3)", wl.config2(volt_mv=50.0)),
                    ("3 (256^3)", wl.config3())):
        rhs = w.rhs if w.rhs is not None else oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
        for solver, sname in ((0, "Table 3"), (1, "merged")):
            ref = None
            if w.n <= 64 ** 3:
                ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=1e-10, solver=solver)
            for kern, kname in ((1, "direct"), (2, "tiled")):
                g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, kernels=kern, options={pf.PF_OPT_SOLVER: solver})
                out = g.solve_linear(rhs, tol=1e-10)
                g.close()
                lines.append(f"| {name} | {sname} | {kname} | {out['iters']} | {ref['iters'] if ref else 'n/a'} | "
                             f"{out['true_relres']:.2e} | " + (f"{rel_l2(out['x'].cpu().numpy(), ref['x']):.1e}" if ref else "n/a") + " |")
    text = "\n".join(lines) + "\n"
    os.makedirs(os.path.dirname(out_path), exist_ok=True)
    with open(out_path, "w") as f:
        f.write(text)
    print(text)


def omega_sweep(out_path):
    """omega_PF of Table 2 step 5 (PAPER.md:219 uses 0.3) on configs[2] (128^3, +50 mV): outer and linear iterations
    and wall time of the full nonlinear solve to BASELINE's tolerances, Table 3 and merged solver, plus the agreement
    of the converged potentials with the omega_PF = 0.3 result (the fixed point does not depend on the relaxation)."""
    w = wl.config2(volt_mv=50.0)
    sp = w.species
    lines = ["| omega_PF | solver | status | outer iterations | linear iterations | seconds | rel. L2 diff of phi vs omega_PF = 0.3 |",
             "|---:|---|---:|---:|---:|---:|---:|"]
    ref = {}
    for om in (0.3, 0.0, 0.1, 0.2, 0.4, 0.5, 0.6, 0.7):
        for solver, sname in ((0, "Table 3"), (1, "merged")):
            g = pf.Grid.from_workload(w, options={pf.PF_OPT_OMEGA_PF: om, pf.PF_OPT_SOLVER: solver, pf.PF_OPT_MAX_OUTER: 3000})
            g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)   # warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            g.close()
            phi = out["phi"].cpu().numpy()
            if om == 0.3:
                ref[solver] = phi
            lines.append(f"| {om:.1f} | {sname} | {out['status']} | {out['outer_iters']} | {out['linear_iters']} | {dt:.2f} | "
                         f"{rel_l2(phi, ref[solver]):.1e} |")
    lines[2:] = sorted(lines[2:], key=lambda l: (float(l.split('|')[1]), l.split('|')[2]))
    text = "\n".join(lines) + "\n"
    os.makedirs(os.path.dirname(out_path), exist_ok=True)
    with open(out_path, "w") as f:
        f.write(text)
    print(text)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "report.md"))
    ap.add_argument("--skip-512", action="store_true")
    ap.add_argument("--launch-ab", action="store_true", help="only the A/B table of the launch modes (PF_OPT_GRAPH)")
    ap.add_argument("--omega-sweep", action="store_true", help="only the omega_PF sweep of configs[2]'s PF solve")
    ap.add_argument("--iteration-counts", action="store_true",
                    help="only the iterations-to-tolerance table of configs 0-3 (both kernel families and solvers)")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise RuntimeError("report needs a CUDA device")
    pf.load()
    if args.launch_ab:
        launch_mode_ab(args.out)
        return
    if args.omega_sweep:
        omega_sweep(args.out)
        return
    if args.iteration_counts:
        iteration_counts(args.out)
        return
    from oracle import pf_oracle as oracle
    oracle.build()
    peak = measured_peak()
    rows = []
    w = wl.config0()
    rows += linear_rows("0 (32^3 channel)", w, oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges), oracle, True, 0, peak)
    rows.append(pf_row("0 (32^3 channel)", w, oracle, True))
    w = wl.config1()
    rows += linear_rows("1 (64^3 spheres)", w, w.rhs, oracle, True, 0, peak)
    w = wl.config2(volt_mv=50.0)
    rows += linear_rows("2 (128^3 channel, +50 mV)", w, oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges), oracle,
                        False, 20, peak)
    rows.append(pf_row("2 (128^3 channel, +50 mV)", w, oracle, False))
    w = wl.config3()
    rows += linear_rows("3 (256^3 channel)", w, oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges), oracle, False, 6,
                        peak)
    if not args.skip_512:
        w = wl.config4()
        rows += linear_rows("4 (512^3 spheres)", w, w.rhs, oracle, False, 0, peak)
    hdr = ["config", "N", "variant", "iters to 1e-10 (GPU / oracle)", "true rel. residual", "rel. L2 diff vs oracle",
           "ms/iter", "iterations/s", "Mupdates/s", "model B/unknown/iter", "effective GB/s (model)",
           "ncu DRAM GB/s (bytes of the committed capture / this time)", "% of 8.0 TB/s",
           f"% of {peak / 1e3:.2f} TB/s", "oracle s/iter (1 core)", "PF outer iters", "PF total time GPU / oracle"]
    keys = ["config", "N", "variant", "iters", "relres", "diff", "ms", "its", "mup", "bpi", "gbs", "ncu", "p8", "pm", "osit",
            "outer", "pft"]
    lines = ["| " + " | ".join(hdr) + " |", "|" + "---|" * len(hdr)]
    for r in rows:
        lines.append("| " + " | ".join(str(r[k]) for k in keys) + " |")
    text = "\n".join(lines) + "\n"
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    with open(args.out, "w") as f:
        f.write(text)
    print(text)


if __name__ == "__main__":
    main()
