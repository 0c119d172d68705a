#!/usr/bin/env python
"""bench.py -- pair interactions/s and us per force evaluation, VERTEX vs EDGE (BASELINE.json `metric`).

Workload (N = 1 GPU): BASELINE.json configs[1], Lennard-Jones fluid, N = 2^20, rho = 0.8, r_c = 2.5, skin 0.3
(`--workload C2b` for the r_c = 4.0 many-neighbour variant, C1 / C3 / C4 for the other configs, C5 for the strategy
crossover sweep of configs[4]), seeded fcc + jitter, melted by an untimed md_integrate run so that the timed state
is the load-imbalanced fluid.

A timed "step" is one pass of the whole hot path: one md_integrate step (half kick, drift, skin check, device-side
cell + Verlet rebuild when the skin criterion fires, force evaluation, half kick); one md_energy closes the K
steps inside the timed region.  `value` = E (unordered Verlet pairs) x K / time.  The same K steps are timed
for the other strategy too (`whole_step`).  The force kernels are timed alone with CUDA events, 5 repeats of >= 20
back-to-back calls, median and min (P:135, S:8(d)), for `force_eval` and `roofline`.

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

UNIT = "pair interactions/s"
def _edge_variants():
    from paper_1401_4350_b200.binding import SCATTER
    return [v for v in ("red", "red_v4", "warp", "segmented", "cluster") if v in SCATTER]


EDGE_VARIANTS = _edge_variants()
VERTEX_VARIANTS = ["smem", "l2"]
WORKLOAD_TEXT = {
    "C1": "BASELINE.json configs[0], LJ fluid N=2048 rho=0.8 rc=2.5 skin=0.3, fcc+jitter",
    "C2a": "BASELINE.json configs[1], LJ fluid N=2^20 rho=0.8 rc=2.5 skin=0.3, fcc+jitter",
    "C2b": "BASELINE.json configs[1] many-neighbour variant, LJ fluid N=2^20 rho=0.8 rc=4.0 skin=0.3, fcc+jitter",
    "C3": "BASELINE.json configs[2], bead-spring melt 4096 x 64, rho=0.85, FENE + WCA, skin=0.3, seeded walks + push-off",
    "C4": "BASELINE.json configs[3], patchy rigid bodies N=2^18 rho=0.5, WCA core + 4 tetrahedral patches, rc=1.5 skin=0.3",
}
METRIC_TEXT = {
    "C1": "LJ N=2048", "C2a": "LJ N=2^20", "C2b": "LJ N=2^20 rc=4.0", "C3": "bead-spring melt N=2^18",
    "C4": "patchy rigid bodies N=2^18", "C5": "strategy crossover sweep",
}
NVT_N_NEWT, NVT_P = 20, 0.1     # thermostat leg (reading QT of P:53): refresh every 20 steps, 10 % of the particles


def metric_text(workload: str) -> str:
    return f"pair interactions/s (Verlet pairs E per force evaluation / time), VERTEX vs EDGE, {METRIC_TEXT[workload]}"


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


def layout_bytes(strategy: str, variant: str, E: int, N: int, rigid: bool, units: int = 0) -> float:
    """Minimum bytes of the layout the kernel actually streams: the staged VERTEX rows hold 16-bit entries
    (2 B per visit), the cluster EDGE list one 8-byte unit per (cluster, j); everything else as algorithmic_bytes."""
    s_in = s_out = 32.0 if rigid else 16.0
    if strategy == "vertex" and variant == "smem":
        return 2.0 * 2 * E + 4.0 * N + s_in * N + s_out * N
    if strategy == "edge" and variant == "cluster":
        return 8.0 * units + s_in * N + 2 * s_out * N
    return algorithmic_bytes(strategy, E, N, rigid)


def fp32_nominal_tflops() -> float:
    """148 SMs x 128 FP32 lanes x 2 flops (FMA) x SM max clock (MEASURED_PEAKS.json, else 1965 MHz)."""
    p = ROOT / "MEASURED_PEAKS.json"
    mhz = float(json.loads(p.read_text()).get("sm_max_mhz", 1965.0)) if p.exists() else 1965.0
    return 148 * 128 * 2 * mhz * 1e6 / 1e12


def algorithmic_flops(strategy: str, E: int, E_in: int, rigid: bool) -> float:
    """LJ 21 flops per visit + 18 inside the cutoff (21 + 21 per EDGE pair); patchy rigid bodies 21 per
    visit + 194 inside the cutoff for VERTEX (215 per in-cutoff visit), 21 + 214 per EDGE pair (235 in-cutoff).
    VERTEX visits every pair twice, EDGE once.  E_in = listed pairs inside r_c (md_stats_ex, a device counter)."""
    if strategy == "vertex":
        return 2.0 * (21.0 * E + (194.0 if rigid else 18.0) * E_in)
    return 21.0 * E + (214.0 if rigid else 21.0) * E_in


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


def time_calls(torch, fn, n=20, warm=5, repeats=5):
    """S:8(d) timing protocol: CUDA events on the current stream (= the library's stream) around n back-to-back calls,
    `warm` warm-up calls, `repeats` repeats (the paper's count).  Returns (median, min) in microseconds per call."""
    for _ in range(warm):
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
    return statistics.median(ts), min(ts)


def time_steps(torch, s, w, K, Wm, strategy, variant, dev, dist=None):
    """K whole-path steps + one md_energy, device-resident state; returns (ms_total, E_run, launches, rebuilds, energies)."""
    s.build_cells(); s.build_verlet(); s.forces(strategy, variant)
    E0 = s.stats()["n_edges"]
    s.integrate(w.dt, Wm, strategy, variant)
    stw = s.stats()
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    l0 = s.launch_count()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    s.integrate(w.dt, K, strategy, variant)
    e_tot = s.energy()                            # A9, synchronises: result read back by the host
    b.record()
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    ms_total = a.elapsed_time(b)
    launches = s.launch_count() - l0
    st1 = s.stats()
    return ms_total, 0.5 * (E0 + st1["n_edges"]), launches, st1["n_rebuilds"] - stw["n_rebuilds"], e_tot


def in_situ_times(torch, s, w, strategy, variant, nsteps=10):
    """The force kernel timed INSIDE real steps (back-to-back calls on fixed lists are the warm best case):
    md_half_step(kick+drift) / md_forces / md_half_step(kick) with CUDA events around each call, `nsteps` steps right after
    a list build (no rebuild can fall due that soon), median per call in microseconds."""
    s.build_cells(); s.build_verlet(); s.forces(strategy, variant)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(nsteps)]
    for k in range(nsteps):
        ev[k][0].record(); s.half_step(w.dt, "kick_drift")
        ev[k][1].record(); s.forces(strategy, variant)
        ev[k][2].record(); s.half_step(w.dt, "kick")
        ev[k][3].record()
    torch.cuda.synchronize()
    med = lambda a, b: statistics.median(ev[k][a].elapsed_time(ev[k][b]) * 1e3 for k in range(2, nsteps))
    return {"kick_drift_us": med(0, 1), "force_us": med(1, 2), "kick_us": med(2, 3), "steps": nsteps - 2,
            "what": "CUDA events around md_half_step / md_forces / md_half_step inside consecutive real steps (plain launches)"}


def oracle_inputs(s, w):
    """The state the GPU holds, in original id order, as the oracle's input (identical input, S:8(d))."""
    pos = s.in_id_order(s.pos)
    quat = s.in_id_order(s.quat) if w.quat is not None else None
    return pos, quat


def cpu_baseline(w, pos, quat, E_gpu):
    """S:8(d) / P:91: the fp64 oracle, as it stands, on this box's host cores on the IDENTICAL input (the positions the
    GPU timed): (i) one thread over the half Verlet list with Newton's third law (O10), (ii) OpenMP over all cores with
    the plain per-particle definition (O1-O5).  Systems whose list exceeds 60 M pairs are sampled at N = 2^18 of the
    same generator (stated in `sample`)."""
    import workloads as W
    from oracle import Oracle
    orc = Oracle()
    sample = f"the bench input itself (N={w.N}, positions copied from the GPU after the melt)"
    box, pot = w.box, dict(w.potential)
    if E_gpu > 60e6:
        ws = W.lj_fluid(2 ** 18, rcut=w.rcut, skin=w.skin, seed=W.BASE_SEED + 2)
        pos, quat, box, pot = ws.pos, None, ws.box, dict(ws.potential)
        sample = f"lj_fluid N=2^18 rc={w.rcut} of the same generator (the full list has {E_gpu / 1e6:.0f} M pairs)"
    t0 = time.perf_counter()
    pairs = orc.pair_set(pos, box, w.rcut, w.skin)           # the oracle's own half list (timed separately)
    t_list = time.perf_counter() - t0
    E_s = int(pairs.shape[0])
    orc.forces(pos, box, pot, quat=quat)                     # warm (page in, thread pool)
    reps, t0 = 0, time.perf_counter()
    while True:
        orc.forces(pos, box, pot, quat=quat)
        reps += 1
        dt = time.perf_counter() - t0
        if dt > 8.0 or reps >= 10:
            break
    t_omp = dt / reps
    t0 = time.perf_counter()
    orc.forces_half(pos, box, pot, pairs, quat=quat)
    t_one = time.perf_counter() - t0
    return {"value": E_s / t_omp, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
            "sample": f"{sample}; oracle.forces (fp64 plain definition, OpenMP full lists), {reps} evaluations, E={E_s}",
            "us_per_eval": t_omp * 1e6,
            "single_core_half_list": {"value": E_s / t_one, "us_per_eval": t_one * 1e6, "cores": 1,
                                      "what": "oracle.forces_half (O10): one thread, half Verlet list, Newton's third law"},
            "list_build_s": t_list}


def run_reference(args):
    """--impl reference: the oracle on host cores on OUR arm's config -- the same workload at full size, melted by the
    same number of untimed steps (with the oracle's own integrator), W warm-up and K timed velocity-Verlet steps of
    oracle.integrate (O6/O7: force evaluation by the plain definition, OpenMP).  value = E x K / time like our arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import Oracle
    orc = Oracle()
    wname = args.workload if args.workload != "C5" else "C2a"
    w = workload(wname)
    pot = dict(w.potential)
    K, Wm = max(1, args.steps), max(0, args.warmup)
    pos, vel, quat, angmom = w.pos, w.vel, w.quat, w.angmom
    t_melt = time.perf_counter()
    for n in (args.melt_steps, Wm):                       # untimed: melt, then warm-up steps
        if n > 0:
            o = orc.integrate(pos, vel, w.box, pot, w.skin, w.dt, n, quat=quat, angmom=angmom)
            pos, vel = o["pos"], o["vel"]
            if quat is not None:
                quat, angmom = o["quat"], o["angmom"]
    t_melt = time.perf_counter() - t_melt
    pos32 = np.zeros((w.N, 4), dtype=np.float32)
    pos32[:, :3] = np.mod(pos[:, :3], w.box)
    E = orc.pair_count(pos32, w.box, w.rcut, w.skin)
    t0 = time.perf_counter()
    orc.integrate(pos, vel, w.box, pot, w.skin, w.dt, K, quat=quat, angmom=angmom)
    t = (time.perf_counter() - t0) / K
    val = E / t
    sample = (f"oracle.integrate (fp64 plain-definition forces, OpenMP) on the full workload N={w.N}, melted by "
              f"{args.melt_steps} + {Wm} untimed oracle steps ({t_melt:.0f} s), E={E}")
    line = {"impl": "reference", "metric": metric_text(args.workload), "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": K, "warmup": Wm, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{wname}: {WORKLOAD_TEXT[wname]}, relaxed by {args.melt_steps} untimed steps",
                       "N": w.N, "E": int(E)},
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


def roofline_for(strategy, variant, t_us, Ef, E_in, N, rigid, units, probes, workload_name):
    """B:5: the roofline is the SLOWER of the algorithmic bytes at the measured HBM bandwidth and the algorithmic FP32
    flops at peak.  The FP32 peak is the nominal one (conservative for `frac`); the measured FFMA / FFMA2 issue rates of
    this run (md_probe) are recorded beside it."""
    peak, peak_src = measured_peaks()
    abytes = algorithmic_bytes(strategy, Ef, N, rigid)
    aflops = algorithmic_flops(strategy, Ef, E_in, rigid)
    fpeak = fp32_nominal_tflops()
    t_hbm, t_alu = abytes / (peak * 1e9) * 1e6, aflops / (fpeak * 1e12) * 1e6
    knames = {"smem": "k_vertex_lj_staged", "l2": "k_vertex_lj", "warp": "k_edge_warp", "red": "k_edge_red",
              "red_v4": "k_edge_red", "segmented": "k_edge_store+k_edge_segsum", "cluster": "k_edge_cluster"}
    kname = knames[variant]
    if rigid:
        kname = kname.replace("_lj", "_patchy")
        if variant == "warp" and Ef < 28 * N:      # short rows of rigid bodies: the compacting walk (launch_edge, md_forces.cu)
            kname = "k_edge_warp_queue"
    traffic = None
    tf = ROOT / "profiles" / "roofline_traffic.csv"     # dram bytes per launch from the committed ncu --set full captures
    if tf.exists():
        for ln in tf.read_text().splitlines()[1:]:
            f = ln.split(",")
            if len(f) >= 4 and f[0] == workload_name and f[1] == strategy and f[2] == kname:
                traffic = float(f[3])
    if t_alu > t_hbm:
        ach = aflops / (t_us * 1e-6) / 1e12
        r = {"bound": "alu", "kernel": kname, "achieved": ach, "peak": fpeak, "unit": "TFLOP/s", "frac": ach / fpeak,
             "traffic": traffic, "algorithmic_flops_per_launch": aflops, "us_per_launch": t_us,
             "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x SM max clock (DESIGN.md 6); measured issue rates in fp32_measured"}
    else:
        ach = abytes / (t_us * 1e-6) / 1e9
        r = {"bound": "hbm", "kernel": kname, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
             "traffic": traffic, "algorithmic_bytes_per_launch": abytes, "us_per_launch": t_us, "peak_source": peak_src}
    r["t_bound_us"] = {"hbm": t_hbm, "fp32": t_alu}
    r["E_in"] = int(E_in)
    lb = layout_bytes(strategy, variant, Ef, N, rigid, units)
    r["vs_layout_bytes"] = {"bytes_per_launch": lb, "frac": lb / (t_us * 1e-6) / 1e9 / peak,
                            "note": "fraction of the HBM peak against the bytes of the layout the kernel streams (16-bit "
                                    "staged rows / 8-byte cluster units); `frac` above is against SURVEY 8(d)'s algorithmic bytes"}
    if traffic:
        r["dram_frac_measured"] = traffic / (t_us * 1e-6) / 1e9 / peak
    if probes:
        r["fp32_measured"] = probes
    return r


def run_dd(args):
    """--dd: ONE system of the workload's size split into slabs over the ranks (space decomposition, P:37-39, S:8(e) /
    S:8(f4); paper_1401_4350_b200/dd.py) instead of independent replicas -> "scaling": "strong".  A timed step = kick+drift,
    halo refresh (NCCL point-to-point), all-reduce of the skin flags, rebuild with migration when it trips, forces, kick."""
    import torch
    from paper_1401_4350_b200.dd import DDSimulation, DistTransport, Domain, LocalTransport, SlabPlan
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    w = workload(args.workload)
    plan = SlabPlan(w.box, world, w.rcut + w.skin)
    variant = args.scatter or ("smem" if args.strategy == "vertex" else "warp")
    d = Domain(rank, plan, w.N, w.rcut, w.skin, w.potential, w.max_neigh, device=str(dev), order=args.order,
               strategy=args.strategy, variant=variant)
    d.load_initial(w.pos, w.vel, w.quat, w.angmom)
    sim = DDSimulation([d], DistTransport(plan, dist, dev) if world > 1 else LocalTransport(plan))
    sim.rebuild()
    K, Wm = args.steps, max(3, args.warmup)
    sim.run(w.dt, args.melt_steps + Wm)
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    l0, r0 = d.sys.launch_count(), d.n_rebuilds
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    sim.run(w.dt, K)
    e = sim.energy()
    b.record()
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    ms = a.elapsed_time(b)
    E_loc = float(d.sys.stats()["n_edges"])                  # pairs of the local list (cross-face pairs are in two lists)
    n_loc = float(d.sys.N)
    if dist is not None:
        tt = torch.tensor([ms], dtype=torch.float64, device=dev); dist.all_reduce(tt, op=dist.ReduceOp.MAX); ms = float(tt.item())
        ee = torch.tensor(list(e) + [E_loc, n_loc], dtype=torch.float64, device=dev); dist.all_reduce(ee); e = ee[:3].tolist(); E_loc = float(ee[3]); n_loc = float(ee[4])
    if rank == 0:
        # credit the global system's pairs once: E_global ~ pairs of all local lists x N / (owned + ghosts)
        E = E_loc * w.N / n_loc
        print(json.dumps({"metric": metric_text(args.workload), "value": E * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
                          "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f32", "data": "synthetic",
                          "config": {"workload": f"{args.workload}: {WORKLOAD_TEXT[args.workload]}, relaxed by {args.melt_steps} untimed steps",
                                     "N": w.N, "E": int(E), "strategy": args.strategy, "variant": variant, "order": args.order,
                                     "parallelism": f"slab space decomposition over {world} rank(s), halo r_v, ghosts {n_loc / w.N - 1.0:.3f} x N",
                                     "rebuilds_in_timed_region": d.n_rebuilds - r0},
                          "gpu_launches": int(d.sys.launch_count() - l0), "energy_total": sum(e), "e2e": None, "roofline": None,
                          "cpu_baseline": None}))
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2a", choices=["C1", "C2a", "C2b", "C3", "C4", "C5"],
                    help="BASELINE.json config; the headline metric is quoted on C2a (default); C5 = crossover sweep")
    ap.add_argument("--strategy", default="vertex", choices=["vertex", "edge"])
    ap.add_argument("--scatter", default=None, choices=EDGE_VARIANTS + VERTEX_VARIANTS,
                    help="EDGE scatter variant (default: the fastest measured) or VERTEX gather variant (default smem)")
    ap.add_argument("--order", default="hilbert", choices=["none", "cell", "hilbert"])
    ap.add_argument("--melt-steps", type=int, default=300)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--c5-max-log2n", type=int, default=20, help="C5: largest N of the sweep (configs[4] goes to 22)")
    ap.add_argument("--no-graph", action="store_true",
                    help="md_set_option(MD_OPT_NO_GRAPH): plain kernel launches instead of CUDA graphs, so that ncu lists every kernel")
    ap.add_argument("--dd", action="store_true", help="slab space decomposition of ONE system over the ranks instead of replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "C5":
        import crossover
        return crossover.bench_mode(args)
    if args.dd:
        return run_dd(args)

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
    N = w.N
    rigid = w.quat is not None
    s = MDSystem.from_workload(w, device=str(dev), order=args.order)
    if args.no_graph:
        s.set_option("no_graph", 1)
    vgather = "smem" if args.order != "none" else "l2"
    s.build_cells(); s.build_verlet(); s.forces("vertex", vgather)
    if args.melt_steps > 0:                       # untimed setup: melt the lattice (paper: thermalised states)
        for k in range(0, args.melt_steps, 100):  # md_stats between chunks lets the staged launch capacity follow the melt
            s.integrate(w.dt, min(100, args.melt_steps - k), "vertex", vgather)
            s.stats()

    # ---- force evaluation alone, VERTEX and every EDGE variant (lists fixed, state in HBM), S:8(d) protocol ----
    s.build_cells(); s.build_verlet()
    stf = s.stats()
    Ef = stf["n_edges"]
    sampler = ClockSampler(local)
    sampler.start()
    fe = {}
    for gv in VERTEX_VARIANTS:
        if gv == "smem" and args.order == "none":
            continue
        med, mn = time_calls(torch, lambda: s.forces("vertex", gv), 20)
        fe[f"vertex_{gv}"] = {"us": med, "us_min": mn, "pairs_per_s": Ef / (med * 1e-6)}
    for sc in EDGE_VARIANTS:
        med, mn = time_calls(torch, lambda: s.forces("edge", sc), 20 if sc != "red" else 5, warm=3)
        fe[f"edge_{sc}"] = {"us": med, "us_min": mn, "pairs_per_s": Ef / (med * 1e-6)}
    # S:8(f1): VERTEX with Newton's third law, m private force copies per particle (reported beside, not ranked)
    n3 = {}
    for m in (1, 4, 12):
        if m * N > N * ((s.max_neigh + 3) // 4 * 4) // 2 + 64:
            continue
        med, mn = time_calls(torch, lambda: s.forces("vertex_n3", m), 10, warm=2, repeats=3)
        n3[f"m{m}"] = {"us": med, "us_min": mn, "pairs_per_s": Ef / (med * 1e-6)}
    best_vertex = min((k for k in fe if k.startswith("vertex")), key=lambda k: fe[k]["us"])
    best_edge = min((k for k in fe if k.startswith("edge")), key=lambda k: fe[k]["us"])
    # the whole-step EDGE leg runs the variant with the fastest force evaluation; within 5 % the cluster variant is
    # preferred because its list build is the cheaper one (0.97 ms against 1.8 ms for the explicit lists at C2a)
    edge_for_step = "edge_cluster" if "edge_cluster" in fe and fe["edge_cluster"]["us"] <= 1.05 * fe[best_edge]["us"] else best_edge
    sx = s.stats_ex()                              # E_in by a device counter (S:Q16), NS of the staged launch
    E_in, units = sx["n_in_cutoff"], sx["n_cluster_units"]
    probes = {"ffma_tflops": s.probe("ffma"), "ffma2_tflops": s.probe("ffma2"), "mufu_tops": s.probe("mufu"),
              "red_v4_scatter_gops": s.probe("red_v4_scatter"), "red_v4_coalesced_gops": s.probe("red_v4_coalesced"),
              "red_f32_scatter_gops": s.probe("red_f32_scatter"), "red_f32_coalesced_gops": s.probe("red_f32_coalesced"),
              "nominal_tflops": fp32_nominal_tflops()}
    if args.scatter is None:
        args.scatter = (vgather if args.strategy == "vertex" else edge_for_step[len("edge_"):])
    if args.order == "none" and args.scatter == "smem":
        args.scatter = "l2"
    other = ("edge", edge_for_step[len("edge_"):]) if args.strategy == "vertex" else ("vertex", vgather)
    rooflines = {}
    for strat, var in ((args.strategy, args.scatter), other):
        rooflines[f"{strat}_{var}"] = roofline_for(strat, var, fe[f"{strat}_{var}"]["us"], Ef, E_in, N, rigid, units,
                                                   probes, args.workload)
    roofline = rooflines[f"{args.strategy}_{args.scatter}"]
    roofline["threads_per_particle"] = sx["threads_per_particle"]
    situ = in_situ_times(torch, s, w, args.strategy, args.scatter)
    roofline["in_situ"] = dict(situ, frac=roofline["frac"] * roofline["us_per_launch"] / situ["force_us"])

    # ---- whole-path steps: K x md_integrate(1 step) + one md_energy, device-resident state; both strategies ----
    ms_total, E_run, launches, rebuilds, e_tot = time_steps(torch, s, w, K, Wm, args.strategy, args.scatter, dev, dist)
    pairs_all, ms_max = aggregate(dist, torch, E_run * K, ms_total, dev)
    value = pairs_all / (ms_max * 1e-3)
    ms_o, E_o, _, reb_o, _ = time_steps(torch, s, w, K, Wm, other[0], other[1], dev)
    whole = {f"{args.strategy}_{args.scatter}": {"ms_per_step": ms_total / K, "pairs_per_s": E_run * K / (ms_total * 1e-3),
                                                  "rebuilds": rebuilds},
             f"{other[0]}_{other[1]}": {"ms_per_step": ms_o / K, "pairs_per_s": E_o * K / (ms_o * 1e-3), "rebuilds": reb_o}}
    clocks = sampler.stop()

    # S:8(f3): the same K steps in mixed precision (fp64 integration of the state, fp32 forces), reported beside
    s.set_precision("mixed")
    ms_mixed = time_steps(torch, s, w, K, Wm, args.strategy, args.scatter, dev)[0] / K
    mixed = {"ms_per_step": ms_mixed, "cost_vs_fp32": ms_mixed / (ms_total / K), "paper": "10-40 % on C2070/K10/K20 (P:59)"}
    s.set_precision("f32")
    # S:8(f3): the same K steps under the thermostat of reading QT (NVT), reported beside; the target temperature
    # is the kinetic temperature the system has now, so the thermostat holds the state point instead of moving it
    s.build_cells(); s.build_verlet(); s.forces(args.strategy, args.scatter)
    T_now = 2.0 * s.energy()[1] / (3.0 * N)
    s.set_thermostat(T_now, NVT_N_NEWT, NVT_P, NVT_P if rigid else 0.0, 20140117)
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

    # ---- end to end through the C ABI with HOST buffers (md_step_host): H2D state, build, forces, 1 step, D2H ----
    pos_id, quat_id = oracle_inputs(s, w)         # the state the CPU baseline gets: identical input (S:8(d))
    e2e = None
    if rank == 0 or world > 1:
        pos_h = torch.from_numpy(pos_id.copy()).pin_memory()
        vel_h = torch.from_numpy(s.in_id_order(s.vel)).pin_memory()
        f_h = torch.zeros_like(pos_h).pin_memory()
        rb = {}
        if rigid:                                 # rigid bodies: quaternions and angular momenta in, torques out as well
            rb = {"quat": torch.from_numpy(quat_id.copy()).pin_memory(),
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
    if not args.no_cpu_baseline and world == 1:
        cpu = cpu_baseline(w, pos_id, quat_id, Ef)

    line = {
        "metric": metric_text(args.workload), "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
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
                   "timing": "force_eval: CUDA events, 5 warm-up calls, 5 repeats of 20 back-to-back calls, median (us) and min (us_min)",
                   "rebuilds_in_timed_region": rebuilds,
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "force_eval": fe, "whole_step": whole, "vertex_n3_eval": n3, "mixed_precision": mixed, "thermostat": nvt,
        "edge_vs_vertex": fe[best_vertex]["us"] / fe[best_edge]["us"], "best_edge": best_edge, "best_vertex": best_vertex,
        "roofline": roofline, "roofline_other_strategy": rooflines[f"{other[0]}_{other[1]}"],
        "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "energy_total": sum(e_tot),
    }
    print(json.dumps(line))
    s.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
