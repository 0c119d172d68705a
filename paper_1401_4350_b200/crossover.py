"""Strategy crossover sweep (BASELINE.json configs[4]): VERTEX (both gather variants) against every EDGE
scatter variant, LJ at rho = 0.8 for N in {2^12 .. 2^22} x r_c in {1.5 .. 4.0} and the patchy potential of config 4 at
the same N, seeded fcc + jitter positions, fp32.  One list build, then CUDA-event timed force evaluations.

    python -m paper_1401_4350_b200.crossover [--max-log2n 22] [--evals 10] [--melt-steps 0] [--rhos 0.1,0.3,0.5] > table.md

`--rhos` replaces the densities of configs[4] (LJ 0.8, patchy 0.5) by a list applied to both potentials: the density
axis of the paper's Fig. 4 (P:119, S:8(f4)); `--melt-steps` thermalises every cell before timing.

Prints one JSON line per cell on stderr and a markdown table on stdout.  `x = entries/particle x flops per in-cutoff
pair` is the abscissa the paper's prediction is stated in (EDGE wins for few / complicated interactions).
"""
from __future__ import annotations

import argparse
import json
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

VERTEX = ["smem", "l2"]
EDGE = ["red", "red_v4", "warp", "segmented"]
FLOPS_PER_PAIR = {"lj": 39.0, "patchy": 235.0,          # SURVEY 8(d) algorithmic work table
                  "patchy_pp": 260.0}                   # the paper's own model: core + 4 patch pairs (this build's count)


def time_calls(torch, fn, n):
    for _ in range(2):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) * 1e3 / n


def run_cell(torch, MDSystem, w, kind, evals, melt, rho):
    s = MDSystem.from_workload(w, device="cuda:0", order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces("vertex", "smem")
    for k in range(0, melt, 100):                          # md_stats between chunks: the staged launch capacity follows
        s.integrate(w.dt, min(100, melt - k), "vertex", "smem")   # the neighbourhoods while the lattice melts
        s.stats()
    if melt > 0:
        s.build_cells(); s.build_verlet()
    st = s.stats()
    E, nfull = st["n_edges"], st["n_full_entries"]
    out = {"kind": kind, "N": w.N, "rho": rho, "rcut": w.rcut, "E": E, "entries_per_particle": nfull / w.N}
    for v in VERTEX:
        out[f"vertex_{v}"] = time_calls(torch, lambda: s.forces("vertex", v), evals)
    for v in EDGE:
        n = max(2, evals // 4) if v == "red" else evals
        out[f"edge_{v}"] = time_calls(torch, lambda: s.forces("edge", v), n)
    m = max(1, min(12, s.max_neigh // 2))                  # the copies must fit in the per-edge scratch (sparse systems)
    out["vertex_n3"] = time_calls(torch, lambda: s.forces("vertex_n3", m), evals)   # P:71, beside the two contenders
    out["n3_copies"] = m
    s.close()
    bv = min(VERTEX, key=lambda v: out[f"vertex_{v}"])
    be = min(EDGE, key=lambda v: out[f"edge_{v}"])
    out["best_vertex"], out["best_edge"] = bv, be
    out["t_vertex_over_t_edge"] = out[f"vertex_{bv}"] / out[f"edge_{be}"]
    out["x"] = out["entries_per_particle"] * FLOPS_PER_PAIR[kind]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--min-log2n", type=int, default=12)
    ap.add_argument("--max-log2n", type=int, default=22)
    ap.add_argument("--evals", type=int, default=10)
    ap.add_argument("--melt-steps", type=int, default=0)
    ap.add_argument("--rcuts", default="1.5,2.0,2.5,3.0,4.0")
    ap.add_argument("--rhos", default="", help="comma-separated densities for both potentials (default: LJ 0.8, patchy 0.5)")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("the crossover sweep needs a CUDA device: the product path has no CPU fallback")
    import workloads as W
    from paper_1401_4350_b200 import MDSystem

    rhos = [float(x) for x in args.rhos.split(",")] if args.rhos else [None]
    rows = []
    for lg in range(args.min_log2n, args.max_log2n + 1, 2):
        N = 2 ** lg
        for rho in rhos:
            for rc in [float(x) for x in args.rcuts.split(",")]:
                w = W.lj_fluid(N, rc, rho=rho or 0.8, seed=W.BASE_SEED + 5)
                r = run_cell(torch, MDSystem, w, "lj", args.evals, args.melt_steps, rho or 0.8)
                print(json.dumps(r), file=sys.stderr, flush=True)
                rows.append(r)
            w = W.patchy_fluid(N, rho=rho or 0.5, seed=W.BASE_SEED + 5)
            r = run_cell(torch, MDSystem, w, "patchy", args.evals, args.melt_steps, rho or 0.5)
            print(json.dumps(r), file=sys.stderr, flush=True)
            rows.append(r)
        # the paper's own patchy model (S:8(f2), reading Q1; "mostly zero" interactions): bonded dimers on a lattice
        w = W.dimer_gas(N // 2, "patchy_pp", spacing=2.6)
        r = run_cell(torch, MDSystem, w, "patchy_pp", args.evals, 0, 2.0 / 2.6 ** 3)
        print(json.dumps(r), file=sys.stderr, flush=True)
        rows.append(r)

    cols = [f"vertex_{v}" for v in VERTEX] + [f"edge_{v}" for v in EDGE] + ["vertex_n3"]
    print("| potential | N | rho | r_c | entries/particle | E | " + " | ".join(c + " us" for c in cols) +
          " | t_VERTEX / t_EDGE (best of each) | x |")
    print("|" + "---|" * (8 + len(cols)))
    for r in rows:
        print(f"| {r['kind']} | 2^{r['N'].bit_length() - 1} | {r['rho']:.3g} | {r['rcut']} | {r['entries_per_particle']:.1f} | {r['E']} | " +
              " | ".join(f"{r[c]:.1f}" for c in cols) +
              f" | {r['t_vertex_over_t_edge']:.2f} ({r['best_vertex']} / {r['best_edge']}) | {r['x']:.0f} |")


if __name__ == "__main__":
    main()
