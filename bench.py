#!/usr/bin/env python
"""bench.py -- pair interactions/s and us per force evaluation, VERTEX vs EDGE (BASELINE.json `metric`).

Workload (N = 1 GPU): BASELINE.json configs[1], Lennard-Jones fluid, N = 2^20, rho = 0.8, r_c = 2.5, skin 0.3
(`--workload C2b` for the r_c = 4.0 many-neighbour variant), seeded fcc + jitter, melted by an untimed
md_integrate run so that the timed state is the load-imbalanced fluid.

A timed "step" is one pass of the whole hot path: one md_integrate step (half kick, drift, skin check, device-side
cell + Verlet rebuild when the skin criterion fires, force evaluation, half kick); one md_energy closes the K
steps inside the timed region.  `value` = E (unordered Verlet pairs) x K / time.  The dominant kernel (the
force kernel) is timed alone with CUDA events for `force_eval` and `roofline`.

Multi-GPU: the path runs on one GPU (north_star) -> replicas only: every rank runs an independent system, no
data-path collective; value = pairs processed by all ranks / max-over-ranks time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np

METRIC = "pair interactions/s (Verlet pairs E per force evaluation / time), VERTEX vs EDGE, LJ N=2^20"
UNIT = "pair interactions/s"
EDGE_VARIANTS = ["red", "red_v4", "warp", "segmented"]
WORKLOAD_TEXT = {
    "C1": "BASELINE.json configs[0], LJ fluid N=2048 rho=0.8 rc=2.5 skin=0.3, fcc+jitter",
    "C2a": "BASELINE.json configs[1], LJ fluid N=2^20 rho=0.8 rc=2.5 skin=0.3, fcc+jitter",
    "C2b": "BASELINE.json configs[1] many-neighbour variant, LJ fluid N=2^20 rho=0.8 rc=4.0 skin=0.3, fcc+jitter",
    "C3": "BASELINE.json configs[2], bead-spring melt 4096 x 64, rho=0.85, FENE + WCA, skin=0.3, seeded walks + push-off",
    "C4": "BASELINE.json configs[3], patchy rigid bodies N=2^18 rho=0.5, WCA core + 4 tetrahedral patches, rc=1.5 skin=0.3",
}
VERTEX_VARIANTS = ["smem", "l2"]
NVT_N_NEWT, NVT_P = 20, 0.1     # thermostat leg (reading QT of P:53): refresh every 20 steps, 10 % of the particles


def workload(name: str):
    import workloads as W
    return W.config(name)


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def algorithmic_bytes(strategy: str, E: int, N: int, rigid: bool = False) -> float:
    """VERTEX 4(2E) + 4N + S_in N + S_out N; EDGE 8E + S_in N + 2 S_out N, with S_in = 16 (pos) [+16 quat]
    and S_out = 16 (force) [+16 torque]."""
    s_in = s_out = 32.0 if rigid else 16.0
    if strategy == "vertex":
        return 4.0 * 2 * E + 4.0 * N + s_in * N + s_out * N
    return 8.0 * E + s_in * N + 2 * s_out * N


def fp32_peak_tflops() -> float:
    """148 SMs x 128 FP32 lanes x 2 flops (FMA) x SM max clock (MEASURED_PEAKS.json, else 1965 MHz)."""
    p = ROOT / "MEASURED_PEAKS.json"
    mhz = float(json.loads(p.read_text()).get("sm_max_mhz", 1965.0)) if p.exists() else 1965.0
    return 148 * 128 * 2 * mhz * 1e6 / 1e12


def algorithmic_flops(strategy: str, E: int, rigid: bool, rcut: float, rv: float) -> float:
    """DESIGN.md 6 / SURVEY 8(d): LJ ~21 flops per visit + 18 inside the cutoff (in-cutoff share of a uniform fluid,
    (rc/rv)^3); patchy rigid bodies ~215 flops per visit.  VERTEX visits every pair twice, EDGE once."""
    visits = 2.0 * E if strategy == "vertex" else 1.0 * E
    per = 215.0 if rigid else 21.0 + 18.0 * (rcut / rv) ** 3
    return visits * per


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            out = self.proc.communicate(timeout=5)[0]
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def time_calls(torch, fn, n, warm=3):
    """Average device time of fn() in microseconds (CUDA events on the current stream = the library's stream)."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) * 1e3 / n


def cpu_baseline(w, seconds_hint=20.0):
    """The fp64 oracle, as it stands, timed on this box's host cores on a bounded sample of the workload:
    the same generator at N = 2^17 (same density, cutoff, skin -> same per-particle structure)."""
    import workloads as W
    from oracle import Oracle
    orc = Oracle()
    n_s = min(w.N, 2 ** 17)
    ws = W.lj_fluid(n_s, rcut=w.rcut, skin=w.skin, seed=W.BASE_SEED + 2)
    E_s = orc.pair_count(ws.pos, ws.box, ws.rcut, ws.skin)      # untimed: only to count the pairs credited
    orc.forces(ws.pos, ws.box, dict(ws.potential))               # warm (page in, thread pool)
    reps, t0 = 0, time.perf_counter()
    while True:
        orc.forces(ws.pos, ws.box, dict(ws.potential))
        reps += 1
        dt = time.perf_counter() - t0
        if dt > 0.5 * seconds_hint or reps >= 20:
            break
    t = dt / reps
    # the same oracle on ONE host core (the paper's "single CPU core" framing), two evaluations
    nthreads = orc.threads
    orc.set_threads(1)
    t1 = time.perf_counter()
    for _ in range(2):
        orc.forces(ws.pos, ws.box, dict(ws.potential))
    t1 = (time.perf_counter() - t1) / 2
    orc.set_threads(nthreads)
    return {"value": E_s / t, "unit": UNIT, "cores": nthreads, "kind": "oracle", "single_core_value": E_s / t1,
            "sample": f"oracle.forces (fp64 plain definition, OpenMP) on lj_fluid N={n_s} rc={w.rcut} (same generator, "
                      f"density and cutoffs as the bench workload), {reps} evaluations, E_sample={E_s}",
            "us_per_eval": t * 1e6}, orc


def run_reference(args):
    """--impl reference: the oracle on host cores, same metric / config; each step = one force evaluation on the
    bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads as W
    from oracle import Oracle
    orc = Oracle()
    wname = args.workload
    rcut = 4.0 if wname == "C2b" else 2.5
    n_s = 2 ** 17
    ws = W.lj_fluid(n_s, rcut=rcut, seed=W.BASE_SEED + 2)
    E_s = orc.pair_count(ws.pos, ws.box, ws.rcut, ws.skin)
    steps, warm = max(1, min(args.steps, 20)), max(1, min(args.warmup, 3))
    for _ in range(warm):
        orc.forces(ws.pos, ws.box, dict(ws.potential))
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.forces(ws.pos, ws.box, dict(ws.potential))
    t = (time.perf_counter() - t0) / steps
    val = E_s / t
    sample = f"oracle.forces on lj_fluid N={n_s} rc={rcut} (bounded sample of {wname}), E_sample={E_s}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{wname}: LJ fluid rho=0.8 rc={rcut} skin=0.3, oracle sample N={n_s}"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": orc.threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def aggregate(dist, torch, pairs_local: float, ms_local: float, device):
    """value = pairs of all ranks / max-over-ranks time (replicas only: the only collective is this report)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return pairs_local, ms_local
    t = torch.tensor([pairs_local], dtype=torch.float64, device=device)
    m = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    dist.all_reduce(m, op=dist.ReduceOp.MAX)
    return float(t.item()), float(m.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2a", choices=["C1", "C2a", "C2b", "C3", "C4"],
                    help="BASELINE.json config; the headline metric is quoted on C2a (default)")
    ap.add_argument("--strategy", default="vertex", choices=["vertex", "edge"])
    ap.add_argument("--scatter", default=None, choices=EDGE_VARIANTS + VERTEX_VARIANTS,
                    help="EDGE scatter variant (default warp) or VERTEX gather variant (default smem)")
    ap.add_argument("--order", default="hilbert", choices=["none", "cell", "hilbert"])
    ap.add_argument("--melt-steps", type=int, default=300)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=5)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.scatter is None:
        args.scatter = "smem" if args.strategy == "vertex" else "warp"
    if args.order == "none" and args.scatter == "smem":
        args.scatter = "l2"

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    from paper_1401_4350_b200 import MDSystem

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    K, Wm = args.steps, max(3, args.warmup)

    w = workload(args.workload)
    s = MDSystem.from_workload(w, device=str(dev), order=args.order)
    s.build_cells(); s.build_verlet(); s.forces(args.strategy, args.scatter)
    if args.melt_steps > 0:                       # untimed setup: melt the lattice (paper: thermalised states)
        for k in range(0, args.melt_steps, 100):  # md_stats between chunks lets the staged launch capacity follow the melt
            s.integrate(w.dt, min(100, args.melt_steps - k), args.strategy, args.scatter)
            s.stats()
    s.build_cells(); s.build_verlet(); s.forces(args.strategy, args.scatter)
    st0 = s.stats()
    E, N = st0["n_edges"], w.N

    # ---- whole-path steps: K x md_integrate(1 step) + one md_energy, device-resident state ----
    s.integrate(w.dt, Wm, args.strategy, args.scatter)
    stw = s.stats()
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = s.launch_count()
    torch.cuda.synchronize(dev)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    s.integrate(w.dt, K, args.strategy, args.scatter)
    e_tot = s.energy()                            # A9, synchronises: result read back by the host
    b.record()
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    ms_total = a.elapsed_time(b)
    launches = s.launch_count() - l0
    st1 = s.stats()
    E_run = 0.5 * (E + st1["n_edges"])
    pairs_all, ms_max = aggregate(dist, torch, E_run * K, ms_total, dev)
    value = pairs_all / (ms_max * 1e-3)

    # ---- dominant kernel alone: force evaluation, VERTEX and every EDGE variant (lists fixed, state in HBM) ----
    s.build_cells(); s.build_verlet()
    stf = s.stats()
    Ef = stf["n_edges"]
    fe = {}
    for gv in VERTEX_VARIANTS:
        if gv == "smem" and args.order == "none":
            continue
        t = time_calls(torch, lambda: s.forces("vertex", gv), 20)
        fe[f"vertex_{gv}"] = {"us": t, "pairs_per_s": Ef / (t * 1e-6)}
    for sc in EDGE_VARIANTS:
        t = time_calls(torch, lambda: s.forces("edge", sc), 10 if sc != "red" else 5)
        fe[f"edge_{sc}"] = {"us": t, "pairs_per_s": Ef / (t * 1e-6)}
    # S:8(f1): VERTEX with Newton's third law, m private force copies per particle (reported beside, not ranked)
    n3 = {}
    for m in (1, 4, 12):
        t = time_calls(torch, lambda: s.forces("vertex_n3", m), 10)
        n3[f"m{m}"] = {"us": t, "pairs_per_s": Ef / (t * 1e-6)}
    best_vertex = min((k for k in fe if k.startswith("vertex")), key=lambda k: fe[k]["us"])
    t_v = fe[best_vertex]["us"]
    clocks = sampler.stop()
    # S:8(f3): the same K steps in mixed precision (fp64 integration of the state, fp32 forces), reported beside
    s.set_precision("mixed")
    s.build_cells(); s.build_verlet(); s.forces(args.strategy, args.scatter)
    s.integrate(w.dt, Wm, args.strategy, args.scatter)
    torch.cuda.synchronize(dev)
    am, bm = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    am.record()
    s.integrate(w.dt, K, args.strategy, args.scatter)
    s.energy()
    bm.record()
    torch.cuda.synchronize(dev)
    ms_mixed = am.elapsed_time(bm) / K
    mixed = {"ms_per_step": ms_mixed, "cost_vs_fp32": ms_mixed / (ms_total / K), "paper": "10-40 % on C2070/K10/K20 (P:59)"}
    s.set_precision("f32")
    # S:8(f3): the same K steps under the thermostat of reading QT (NVT), reported beside; the target temperature
    # is the kinetic temperature the system has now, so the thermostat holds the state point instead of moving it
    s.build_cells(); s.build_verlet(); s.forces(args.strategy, args.scatter)
    T_now = 2.0 * s.energy()[1] / (3.0 * N)
    s.set_thermostat(T_now, NVT_N_NEWT, NVT_P, NVT_P if w.quat is not None else 0.0, 20140117)
    s.integrate(w.dt, Wm, args.strategy, args.scatter)
    torch.cuda.synchronize(dev)
    an, bn = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    an.record()
    s.integrate(w.dt, K, args.strategy, args.scatter)
    k_nvt = s.energy()[1]
    bn.record()
    torch.cuda.synchronize(dev)
    ms_nvt = an.elapsed_time(bn) / K
    s.set_thermostat(T_now, 0, 0.0, 0.0, 0)
    nvt = {"ms_per_step": ms_nvt, "cost_vs_nve": ms_nvt / (ms_total / K), "T_target": T_now, "T_after": 2.0 * k_nvt / (3.0 * N),
           "n_newt": NVT_N_NEWT, "p": NVT_P, "paper": "'does not significantly affect performances' (P:53)"}
    best_edge = min((k for k in fe if k.startswith("edge")), key=lambda k: fe[k]["us"])
    peak, peak_src = measured_peaks()
    dom = args.strategy
    t_dom = fe[f"{dom}_{args.scatter}"]["us"]
    rigid = w.quat is not None
    abytes = algorithmic_bytes(dom, Ef, N, rigid)
    achieved = abytes / (t_dom * 1e-6) / 1e9
    knames = {"smem": "k_vertex_lj_staged", "l2": "k_vertex_lj", "warp": "k_edge_warp", "red": "k_edge_red", "red_v4": "k_edge_red",
              "segmented": "k_edge_store+k_edge_segsum"}
    traffic = None
    tf = ROOT / "profiles" / "roofline_traffic.csv"     # dram bytes per launch from the committed ncu --set full capture
    if tf.exists():
        for ln in tf.read_text().splitlines()[1:]:
            f = ln.split(",")
            if len(f) >= 4 and f[0] == args.workload and f[1] == dom and f[2] == knames[args.scatter]:
                traffic = float(f[3])
    kname = knames[args.scatter]
    if rigid:
        kname = kname.replace("_lj", "_patchy")
    # B:5: the roofline is the SLOWER of the algorithmic bytes at HBM bandwidth and the FP32 flops at peak
    aflops = algorithmic_flops(dom, Ef, rigid, w.rcut, w.rcut + w.skin)
    fpeak = fp32_peak_tflops()
    t_hbm, t_alu = abytes / (peak * 1e9) * 1e6, aflops / (fpeak * 1e12) * 1e6
    if t_alu > t_hbm:
        ach = aflops / (t_dom * 1e-6) / 1e12
        roofline = {"bound": "alu", "kernel": kname, "achieved": ach, "peak": fpeak, "unit": "TFLOP/s", "frac": ach / fpeak,
                    "traffic": traffic, "algorithmic_flops_per_launch": aflops, "us_per_launch": t_dom,
                    "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x SM max clock (DESIGN.md 6)"}
    else:
        roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved,
                    "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                    "algorithmic_bytes_per_launch": abytes, "us_per_launch": t_dom, "peak_source": peak_src}
    roofline["t_bound_us"] = {"hbm": t_hbm, "fp32": t_alu}

    # ---- end to end through the C ABI with HOST buffers (md_step_host): H2D state, build, forces, 1 step, D2H ----
    e2e = None
    if rank == 0 or world > 1:
        pos_h = torch.from_numpy(s.in_id_order(s.pos)).pin_memory()
        vel_h = torch.from_numpy(s.in_id_order(s.vel)).pin_memory()
        f_h = torch.zeros_like(pos_h).pin_memory()
        rb = {}
        if rigid:                                 # rigid bodies: quaternions and angular momenta in, torques out as well
            rb = {"quat": torch.from_numpy(s.in_id_order(s.quat)).pin_memory(),
                  "angmom": torch.from_numpy(s.in_id_order(s.angmom)).pin_memory(),
                  "torque": torch.zeros_like(pos_h).pin_memory()}
        ne = max(1, args.e2e_steps)
        s.step_host(pos_h, vel_h, f_h, w.dt, 1, args.strategy, args.scatter, **rb)     # warm
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for _ in range(ne):
            s.step_host(pos_h, vel_h, f_h, w.dt, 1, args.strategy, args.scatter, **rb)
        t_e = (time.perf_counter() - t0) / ne
        Ee = s.stats()["n_edges"]
        pe_all, te_max = aggregate(dist, torch, float(Ee), t_e * 1e3, dev)
        e2e = {"value": pe_all / (te_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": (4 if rigid else 2) * 16 * N,
               "d2h_bytes_per_step": (6 if rigid else 3) * 16 * N, "ms_per_step": te_max,
               "what": "md_step_host: H2D pos+vel(+quat+angmom), cell+Verlet build, forces, 1 velocity-Verlet step, "
                       "D2H pos+vel+force(+quat+angmom+torque)"}

    if rank != 0:
        s.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline and world == 1 and args.workload in ("C2a", "C2b"):
        cpu, _ = cpu_baseline(w)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {WORKLOAD_TEXT[args.workload]}, relaxed by {args.melt_steps} untimed steps",
                   "N": N, "E": int(E_run), "strategy": args.strategy, "variant": args.scatter, "order": args.order,
                   "step": "md_integrate(1): kick, drift, skin check, device-side rebuild when triggered, forces, kick; "
                           "one md_energy per K steps",
                   "l2": (f"inputs larger than L2 (neighbour rows {4.0 * Ef / 1e6:.0f} MB streamed per evaluation; no flush needed)"
                          if 4.0 * Ef > 126e6 else
                          f"working set ({4.0 * Ef / 1e6:.0f} MB of neighbour rows) fits in the 126 MB L2: steady-state L2-resident "
                          "timing without a flush -- a secondary workload, the headline is C2a"),
                   "rebuilds_in_timed_region": st1["n_rebuilds"] - stw["n_rebuilds"],
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "force_eval": fe, "vertex_n3_eval": n3, "mixed_precision": mixed, "thermostat": nvt, "edge_vs_vertex": fe[best_vertex]["us"] / fe[best_edge]["us"], "best_edge": best_edge,
        "best_vertex": best_vertex,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "energy_total": sum(e_tot),
    }
    print(json.dumps(line))
    s.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
