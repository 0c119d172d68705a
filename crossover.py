"""Strategy crossover sweep (BASELINE.json configs[4]): VERTEX (both gather variants) against
every EDGE scatter variant, LJ at rho = 0.8 for N in {2^12 .. 2^22} x r_c in {1.5 .. 4.0} and the patchy potential of
config 4 at the same N, each under storage order NONE and HILBERT, seeded fcc + jitter positions, fp32.  One list
build per cell, then CUDA-event timed force evaluations (5 repeats, median; S:8(d) protocol).

    python crossover.py [--max-log2n 22] [--evals 10] [--melt-steps 0] [--rhos 0.1,0.3,0.5] [--orders none,hilbert] > table.md
    python bench.py --workload C5          # the same sweep as a bench.py mode: one JSON line with the table inside

`--rhos` replaces the densities of configs[4] (LJ 0.8, patchy 0.5) by a list applied to both potentials: the density
axis of the paper's Fig. 4 (P:119, S:8(f4)); `--melt-steps` thermalises every cell before timing.

Prints one JSON line per cell on stderr and a markdown table on stdout.  `x = entries/particle x flops per in-cutoff
pair` is the abscissa the paper's prediction is stated in (EDGE wins for few / complicated interactions).
"""
from __future__ import annotations

import argparse
import json
import statistics
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

VERTEX = ["smem", "l2"]
def _edge_variants():
    from paper_1401_4350_b200.binding import SCATTER
    return [v for v in ("red", "red_v4", "warp", "segmented", "cluster") if v in SCATTER]


EDGE = _edge_variants()
FLOPS_PER_PAIR = {"lj": 39.0, "patchy": 235.0,          # SURVEY 8(d) algorithmic work table
                  "patchy_pp": 260.0}                   # the paper's own model: core + 4 patch pairs (this build's count)


def time_calls(torch, fn, n, repeats=5):
    for _ in range(2):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(repeats):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b) * 1e3 / n)
    return statistics.median(ts)


def run_cell(torch, MDSystem, w, kind, evals, melt, rho, order="hilbert"):
    s = MDSystem.from_workload(w, device="cuda:0", order=order)
    vg = "smem" if order != "none" else "l2"
    s.build_cells(); s.build_verlet(); s.forces("vertex", vg)
    for k in range(0, melt, 100):                          # md_stats between chunks: the staged launch capacity follows
        s.integrate(w.dt, min(100, melt - k), "vertex", vg)   # the neighbourhoods while the lattice melts
        s.stats()
    if melt > 0:
        s.build_cells(); s.build_verlet()
    st = s.stats()
    E, nfull = st["n_edges"], st["n_full_entries"]
    out = {"kind": kind, "N": w.N, "rho": rho, "rcut": w.rcut, "order": order, "E": E, "entries_per_particle": nfull / w.N}
    for v in VERTEX:
        if v == "smem" and order == "none":
            out["vertex_smem"] = None              # the staged kernel needs cell-sorted storage
            continue
        out[f"vertex_{v}"] = time_calls(torch, lambda: s.forces("vertex", v), evals)
    for v in EDGE:
        n = max(2, evals // 4) if v == "red" else evals
        out[f"edge_{v}"] = time_calls(torch, lambda: s.forces("edge", v), n, repeats=3 if v == "red" else 5)
    m = max(1, min(12, s.max_neigh // 2))                  # the copies must fit in the per-edge scratch (sparse systems)
    out["vertex_n3"] = time_calls(torch, lambda: s.forces("vertex_n3", m), evals, repeats=3)   # P:71, beside the two contenders
    out["n3_copies"] = m
    s.close()
    bv = min((v for v in VERTEX if out[f"vertex_{v}"] is not None), key=lambda v: out[f"vertex_{v}"])
    be = min(EDGE, key=lambda v: out[f"edge_{v}"])
    out["best_vertex"], out["best_edge"] = bv, be
    out["t_vertex_over_t_edge"] = out[f"vertex_{bv}"] / out[f"edge_{be}"]
    out["x"] = out["entries_per_particle"] * FLOPS_PER_PAIR[kind]
    return out


def sweep(torch, MDSystem, log2ns, rcuts, rhos, orders, evals, melt, with_pp=True, log=sys.stderr):
    import workloads as W
    rows = []
    for lg in log2ns:
        N = 2 ** lg
        for order in orders:
            for rho in rhos:
                for rc in rcuts:
                    w = W.lj_fluid(N, rc, rho=rho or 0.8, seed=W.BASE_SEED + 5)
                    r = run_cell(torch, MDSystem, w, "lj", evals, melt, rho or 0.8, order)
                    print(json.dumps(r), file=log, flush=True)
                    rows.append(r)
                w = W.patchy_fluid(N, rho=rho or 0.5, seed=W.BASE_SEED + 5)
                r = run_cell(torch, MDSystem, w, "patchy", evals, melt, rho or 0.5, order)
                print(json.dumps(r), file=log, flush=True)
                rows.append(r)
            if with_pp:
                # the paper's own patchy model (S:8(f2), reading Q1; "mostly zero" interactions): bonded dimers on a lattice
                w = W.dimer_gas(N // 2, "patchy_pp", spacing=2.6)
                r = run_cell(torch, MDSystem, w, "patchy_pp", evals, 0, 2.0 / 2.6 ** 3, order)
                print(json.dumps(r), file=log, flush=True)
                rows.append(r)
    return rows


COLS = [f"vertex_{v}" for v in VERTEX] + [f"edge_{v}" for v in EDGE] + ["vertex_n3"]


def table(rows, out=sys.stdout):
    print("| potential | N | rho | r_c | order | entries/particle | E | " + " | ".join(c + " us" for c in COLS) +
          " | t_VERTEX / t_EDGE (best of each) | x |", file=out)
    print("|" + "---|" * (9 + len(COLS)), file=out)
    for r in rows:
        print(f"| {r['kind']} | 2^{r['N'].bit_length() - 1} | {r['rho']:.3g} | {r['rcut']} | {r['order']} | {r['entries_per_particle']:.1f} | {r['E']} | " +
              " | ".join("-" if r[c] is None else f"{r[c]:.1f}" for c in COLS) +
              f" | {r['t_vertex_over_t_edge']:.2f} ({r['best_vertex']} / {r['best_edge']}) | {r['x']:.0f} |", file=out)


def bench_mode(args):
    """`bench.py --workload C5`: the sweep of configs[4] as ONE JSON line (driver contract).  value = pair interactions/s
    of the best strategy summed over the cells (total pairs / total best time); the cells are in `cells`."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("the crossover sweep needs a CUDA device: the product path has no CPU fallback")
    from paper_1401_4350_b200 import MDSystem
    import bench
    log2ns = list(range(12, args.c5_max_log2n + 1, 2))
    rows = sweep(torch, MDSystem, log2ns, [1.5, 2.0, 2.5, 3.0, 4.0], [None], ["none", "hilbert"], max(3, min(args.steps, 10)), 0,
                 with_pp=False)
    pairs = sum(r["E"] for r in rows)
    t_best = sum(min(r[f"vertex_{r['best_vertex']}"], r[f"edge_{r['best_edge']}"]) for r in rows) * 1e-6
    line = {"metric": bench.metric_text("C5"), "value": pairs / t_best, "unit": bench.UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_best * 1e3 / max(1, len(rows)), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"C5: BASELINE.json configs[4], LJ rho=0.8 N=2^12..2^{args.c5_max_log2n} x rc in 1.5..4.0 + patchy, "
                                   "orders none and hilbert, fcc+jitter (lattice starts: no neighbour-count spread)"},
            "cells": rows}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--min-log2n", type=int, default=12)
    ap.add_argument("--max-log2n", type=int, default=22)
    ap.add_argument("--evals", type=int, default=10)
    ap.add_argument("--melt-steps", type=int, default=0)
    ap.add_argument("--rcuts", default="1.5,2.0,2.5,3.0,4.0")
    ap.add_argument("--rhos", default="", help="comma-separated densities for both potentials (default: LJ 0.8, patchy 0.5)")
    ap.add_argument("--orders", default="hilbert", help="comma-separated storage orders: none, cell, hilbert (Q19: none,hilbert)")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("the crossover sweep needs a CUDA device: the product path has no CPU fallback")
    from paper_1401_4350_b200 import MDSystem

    rhos = [float(x) for x in args.rhos.split(",")] if args.rhos else [None]
    rows = sweep(torch, MDSystem, range(args.min_log2n, args.max_log2n + 1, 2), [float(x) for x in args.rcuts.split(",")],
                 rhos, args.orders.split(","), args.evals, args.melt_steps)
    table(rows)


if __name__ == "__main__":
    main()
