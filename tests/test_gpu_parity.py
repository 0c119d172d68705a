"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): pair sets bit-exact as sorted pair sets; forces and torques
|dF| <= 1e-4 max|F_oracle| + 1e-6 per component; energies 1e-5 relative."""
import numpy as np
import pytest

import workloads as W
from conftest import record_margin

pytestmark = pytest.mark.gpu

# (strategy, variant): VERTEX gather alternatives {l2, smem}, EDGE scatter alternatives {red, red_v4, warp, segmented};
# the shared-memory staged VERTEX variant needs cell-sorted storage (order != none)
# VERTEX with Newton's third law (S:8(f1)): the variant is m, the number of private force copies per particle
VARIANTS = [("vertex", "l2"), ("edge", "red"), ("edge", "red_v4"), ("edge", "warp"), ("edge", "segmented"),
            ("edge", "cluster"), ("vertex_n3", 1), ("vertex_n3", 12)]
STAGED = [("vertex", "smem")]


def variants(order):
    return (STAGED + VARIANTS) if order != "none" else VARIANTS
FTOL_REL, FTOL_ABS, ETOL = 1e-4, 1e-6, 1e-5


@pytest.fixture(scope="module")
def MD():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1401_4350_b200 import MDSystem
    return MDSystem


def sorted_pairs(p):
    return p[np.lexsort((p[:, 1], p[:, 0]))]


def assert_pairs(s, oracle, pos, box, rcut, skin):
    got = sorted_pairs(s.get_pairs())
    ref = oracle.pair_set(pos, box, rcut, skin)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    assert np.array_equal(got, ref)
    st = s.stats()
    assert st["n_edges"] == ref.shape[0] and st["n_full_entries"] == 2 * ref.shape[0]   # E = 1/2 sum |L_i|
    return ref.shape[0]


def assert_forces(s, o, rigid, label=("", "")):
    fmax = np.abs(o["F"]).max()
    F = s.in_id_order(s.force)
    tol = FTOL_REL * fmax + FTOL_ABS
    err = np.abs(F[:, :3] - o["F"]).max()
    record_margin(label[0], label[1], "F", err, tol)
    assert err <= tol
    # per-particle energies feed md_energy: compare the total to 1e-5 relative
    U, Kt, Kr = s.energy()
    Uo = o["pe"].sum()
    record_margin(label[0], label[1], "U", abs(U - Uo), ETOL * max(abs(Uo), abs(Uo) + Kt + Kr, 1e-30))
    assert abs(U - Uo) <= ETOL * max(abs(Uo), 1e-30) or abs(U - Uo) <= ETOL * (abs(Uo) + Kt + Kr)   # S:Q17
    if rigid:
        tmax = np.abs(o["T"]).max()
        T = s.in_id_order(s.torque)
        terr = np.abs(T[:, :3] - o["T"]).max()
        record_margin(label[0], label[1], "T", terr, FTOL_REL * tmax + FTOL_ABS)
        assert terr <= FTOL_REL * tmax + FTOL_ABS
    return F


CASES = {
    "C1_lj2048": lambda: W.config("C1"),
    "lj256_two_cells_per_axis": lambda: W.lj_fluid(256),
    "lj16384_rc4_many_neighbours": lambda: W.lj_fluid(2 ** 14, rcut=4.0),
    "lj4096_rc1.5_orthorhombic": lambda: W.lj_fluid(2 ** 12, rcut=1.5),
    "dimers_lj_ragged_N": lambda: W.dimer_gas(1001, "lj"),
    "dimers_fene": lambda: W.dimer_gas(4096, "fene_wca"),
    "dimers_patchy": lambda: W.dimer_gas(4096, "patchy"),
    "dimers_patchy_pp_paper_model": lambda: W.dimer_gas(4096, "patchy_pp"),   # S:8(f2), Eqs. (2)-(4) under reading Q1
    "polymer_64x64": lambda: W.polymer_melt(64, 64),
    "patchy4096": lambda: W.patchy_fluid(2 ** 12),
    "tiny_16": lambda: W.dimer_gas(8, "lj"),
}


@pytest.mark.parametrize("order", ["none", "cell", "hilbert"])
@pytest.mark.parametrize("case", list(CASES))
def test_step0_parity(MD, oracle, case, order):
    w = CASES[case]()
    s = MD.from_workload(w, order=order)
    s.build_cells(); s.build_verlet()
    assert_pairs(s, oracle, w.pos, w.box, w.rcut, w.skin)
    o = oracle.forces(w.pos, w.box, dict(w.potential), quat=w.quat)
    assert o["bad"] == 0
    results = {}
    from paper_1401_4350_b200 import MDError
    for strat, sc in variants(order):
        if strat == "vertex_n3" and sc * w.N > w.N * ((s.max_neigh + 3) // 4 * 4) // 2 + 64:
            with pytest.raises(MDError) as e:    # the m copies do not fit in the per-edge scratch: an error, not a clamp
                s.forces(strat, sc)
            assert e.value.code == -1
            continue
        s.forces(strat, sc)
        results[(strat, sc)] = assert_forces(s, o, w.quat is not None, (f"{case}/{order}", f"{strat}_{sc}"))
        if sc == "cluster":      # the unit list is a partition of the half list: sum of popcounts = E
            sx = s.stats_ex()
            assert sx["cluster_size"] == 16 and 0 < sx["n_cluster_units"] <= sx["n_edges"]
            assert sx["n_edges"] == oracle.pair_count(w.pos, w.box, w.rcut, w.skin)
            assert sx["n_in_cutoff"] == o["n_in_cut"]                      # E_in by the device counter (S:Q16)
    # the explicit global-slot lists (built on demand for the L2-gather variants) hold the same pair set
    assert_pairs(s, oracle, w.pos, w.box, w.rcut, w.skin)
    # P11: the strategies agree with each other within twice the oracle tolerance
    fmax = np.abs(o["F"]).max()
    ref = results[("vertex", "l2")]
    for k, F in results.items():
        assert np.abs(F[:, :3] - ref[:, :3]).max() <= 2 * (FTOL_REL * fmax + FTOL_ABS)
    # P7: Newton's third law survives fp32 accumulation
    N = w.N
    rms = np.sqrt((o["F"] ** 2).mean()) + 1e-30
    assert np.abs(ref[:, :3].astype(np.float64).sum(axis=0)).max() <= 1e-6 * N * rms + 1e-4
    s.close()


def test_ids_are_a_permutation_and_state_follows(MD):
    w = W.config("C1")
    s = MD.from_workload(w, order="hilbert")
    s.build_cells()
    ids = s.get_ids()
    assert np.array_equal(np.sort(ids), np.arange(w.N))
    assert not np.array_equal(ids, np.arange(w.N))
    assert np.array_equal(s.in_id_order(s.pos), w.pos)          # positions already in [0,L): wrap is the identity
    assert np.array_equal(s.in_id_order(s.vel), w.vel)
    s.close()


def test_vertex_and_segmented_are_bitwise_reproducible(MD):
    w = W.lj_fluid(2 ** 14)
    out = {}
    for rep in range(2):
        s = MD.from_workload(w, order="cell")
        s.build_cells(); s.build_verlet()
        for strat, sc in [("vertex", "l2"), ("vertex", "smem"), ("edge", "segmented")]:
            s.forces(strat, sc)
            F = s.in_id_order(s.force)
            if rep:
                assert np.array_equal(F, out[(strat, sc)])
            out[(strat, sc)] = F
        s.close()


def test_step_graph_equals_plain_launches(MD):
    """md_integrate replays CUDA graphs (rebuild inside a conditional node, 16 steps per launch, tails of 8, 4, 2, 1; the force
    kernel of an inner step carries the kicks and the drift of the next one unless MD_OPT_FUSE_STEPS is 0); with
    md_set_option(MD_OPT_NO_GRAPH, 1) it launches the plain kernels one by one.  VERTEX is deterministic, so all three give the
    same bits and the same number of device-side rebuilds; 37 steps exercise the multi-step graphs and the single-step tail."""
    w = W.lj_fluid(2 ** 14)
    out = []
    for no_graph, fuse in ((False, 1), (True, 1), (False, 0)):
        s = MD.from_workload(w, order="hilbert")
        s.set_option("no_graph", int(no_graph))
        s.set_option("fuse_steps", fuse)
        s.build_cells(); s.build_verlet(); s.forces("vertex", "smem")
        l0 = s.launch_count()
        s.integrate(w.dt, 37, "vertex", "smem")
        per_step = (s.launch_count() - l0) / 37
        out.append((s.in_id_order(s.pos), s.in_id_order(s.vel), s.stats()["n_rebuilds"], per_step))
        s.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert out[0][2] == out[1][2] and out[0][2] >= 1
    # graphs of 16, 8, 4, 2 steps: kick+drift once, then condition + forces per step (the force kernel of an inner step carries
    # the kicks and the drift of the next one), + the closing kick: 2 n + 2 kernels; a single step: 4.  37 = 2 x 16 + 4 + 1
    assert out[0][3] == (2 * 34 + 10 + 4) / 37 and out[1][3] > 4
    # separate kernels inside the graphs: kick+drift, condition, forces per step + the closing kick: 3 n + 1
    assert np.array_equal(out[0][0], out[2][0]) and np.array_equal(out[0][1], out[2][1]) and out[0][2] == out[2][2]
    assert out[2][3] == (2 * 49 + 13 + 4) / 37


def test_options_row_schedule_and_unknown(MD, oracle):
    """MD_OPT_ROW_SCHEDULE = 0 (Verlet rows in scan order instead of bank-column order: the measured alternative of
    DESIGN.md section 10) changes the order of the row entries only: same pair set, forces within tolerance."""
    from paper_1401_4350_b200 import MDError
    w = W.lj_fluid(2 ** 14)
    o = oracle.forces(w.pos, w.box, dict(w.potential))
    s = MD.from_workload(w, order="hilbert")
    for sched in (0, 1):
        s.set_option("row_schedule", sched)
        with pytest.raises(MDError) as e:
            s.forces("vertex", "smem")                   # the option invalidates the lists
        assert e.value.code == -2
        s.build_cells(); s.build_verlet()
        assert_pairs(s, oracle, s.in_id_order(s.pos), w.box, w.rcut, w.skin)
        s.forces("vertex", "smem")
        assert_forces(s, o, False, (f"lj16384 row_schedule={sched}", "vertex_smem"))
    with pytest.raises(MDError) as e:
        s.set_option(99, 1)
    assert e.value.code == -1
    with pytest.raises(MDError) as e:
        s.set_option("no_graph", -1)
    assert e.value.code == -1
    s.close()


def test_option_build_direct_same_rows(MD, oracle):
    """MD_OPT_BUILD_DIRECT: the dense-cell Verlet build emits its scheduled rows straight from the hit words of the
    transposed scan (1, default) or through column buckets in scratch memory (0).  Same pair set, and the SAME row order:
    the VERTEX forces agree bit for bit.  Run on a melted fluid (ragged cells) and at r_c = 4.0 (blocks whose own cells
    exceed one pass of hit words take the bucket form under either setting)."""
    for rcut, melt in ((2.5, 150), (4.0, 0)):
        w = W.lj_fluid(2 ** 14, rcut=rcut)
        s = MD.from_workload(w, order="hilbert")
        s.build_cells(); s.build_verlet(); s.forces("vertex", "smem")
        if melt:
            s.integrate(w.dt, melt, "vertex", "smem")
        out = []
        for direct in (1, 0, 1):
            s.set_option("build_direct", direct)
            s.build_cells(); s.build_verlet()
            if direct == 0:
                assert_pairs(s, oracle, s.in_id_order(s.pos), w.box, w.rcut, w.skin)
            s.forces("vertex", "smem")
            out.append((s.in_id_order(s.force).copy(), s.stats()["n_edges"]))
        assert out[0][1] == out[1][1] == out[2][1]
        assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][0], out[2][0])
        s.close()


def test_error_paths(MD):
    from paper_1401_4350_b200 import MDError
    w = W.config("C1")
    s = MD.from_workload(w)
    with pytest.raises(MDError) as e:
        s.forces("vertex")                      # forces before lists
    assert e.value.code == -2
    with pytest.raises(MDError) as e:
        s.build_verlet()                        # verlet before cells
    assert e.value.code == -2
    s.build_cells(); s.build_verlet()
    with pytest.raises(MDError) as e:
        s.integrate(0.002, 1)                   # integrate before forces
    assert e.value.code == -2
    with pytest.raises(MDError) as e:
        s.lib.md_forces(s.h, 7, 0) and None
        s._check(s.lib.md_forces(s.h, 7, 0))    # unknown strategy
    assert e.value.code == -1
    with pytest.raises(MDError) as e:
        s._check(s.lib.md_forces(s.h, 2, 65))   # VERTEX_N3: m out of range
    assert e.value.code == -1
    s.close()
    # capacity overflow is an error, never a silent truncation
    s = MD.from_workload(w, max_neigh=40)
    s.build_cells(); s.build_verlet()
    with pytest.raises(MDError) as e:
        s.stats()
    assert e.value.code == -3
    s.close()
    # ... and it is reported once: the handle works again after a rebind with data that fits
    good = W.lj_fluid(2048, rho=0.25)                        # ~23 neighbours inside r_v = 2.8
    s = MD.from_workload(good, max_neigh=40)
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    assert s.stats()["max_neigh_seen"] <= 40
    clumped = good.pos.copy()
    clumped[:, :3] *= 0.5                                    # the same particles in one octant: 8 x the density
    s.set_state(clumped, good.vel)
    s.build_cells()
    with pytest.raises(MDError) as e:
        s.build_verlet(); s.stats()
    assert e.value.code == -3
    with pytest.raises(MDError) as e:
        s.forces("vertex")                                   # the failed lists are not usable ...
    assert e.value.code == -2
    s.set_state(good.pos, good.vel)                          # ... and the error is not sticky
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    assert s.stats()["max_neigh_seen"] <= 40 and np.isfinite(s.energy()[0])
    s.close()
    # FENE bond stretched to R0
    d = W.dimer_gas(64, "fene_wca")
    d.pos[1, :3] = d.pos[0, :3] + np.array([1.6, 0, 0], dtype=np.float32)
    s = MD.from_workload(d)
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    with pytest.raises(MDError) as e:
        s.energy()
    assert e.value.code == -5
    s.close()


@pytest.mark.parametrize("strat,sc", [("vertex", "smem"), ("vertex", "l2"), ("edge", "warp"),
                                      ("edge", "segmented"), ("edge", "cluster"), ("vertex_n3", 12)])
def test_c1_trajectory_100_steps(MD, oracle, strat, sc):
    """C1 (BASELINE.json configs[0]): 100 velocity-Verlet steps at dt = 0.002; fp32 GPU state against the fp64
    oracle trajectory from the same fp32 input.  SURVEY 8(d): the two stay within the force tolerance for 100 steps."""
    w = W.config("C1")
    o = oracle.integrate(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, 100, every=100)
    s = MD.from_workload(w, order="cell")
    s.build_cells(); s.build_verlet(); s.forces(strat, sc)
    e0 = s.energy()
    assert abs(sum(e0) - o["e0"].sum()) <= ETOL * abs(o["e0"].sum())
    s.integrate(w.dt, 100, strat, sc)
    assert s.stats()["n_rebuilds"] >= 1                      # the skin criterion fired on the device
    fmax = np.abs(o["F"]).max()
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= FTOL_REL * fmax + FTOL_ABS
    x = s.in_id_order(s.pos)[:, :3].astype(np.float64)
    dx = x - o["pos"]
    dx -= w.box * np.round(dx / w.box)
    assert np.abs(dx).max() < 1e-4
    e1 = s.energy()
    assert abs(sum(e1) - o["energies"][-1].sum()) <= ETOL * abs(o["energies"][-1].sum())
    s.close()


@pytest.mark.parametrize("case,steps,strat,sc", [
    ("lj", 300, "vertex", "smem"), ("lj", 300, "vertex", "l2"), ("lj", 300, "edge", "red_v4"), 
    ("polymer", 200, "vertex", "smem"), ("polymer", 200, "edge", "warp"), 
    ("patchy", 300, "vertex", "smem"), ("patchy", 300, "vertex", "l2"), ("patchy", 300, "edge", "segmented"),
    ("lj", 300, "vertex_n3", 12), ("polymer", 200, "vertex_n3", 4), ("patchy", 300, "vertex_n3", 12),
    ("lj", 300, "edge", "cluster"), ("polymer", 200, "edge", "cluster"), ("patchy", 300, "edge", "cluster"),
    ])
def test_snapshot_parity_after_device_side_rebuilds(MD, oracle, case, steps, strat, sc):
    """Run md_integrate long enough for several skin-triggered rebuilds, then compare the forces the path holds
    (computed from lists rebuilt on the device) with the oracle's plain definition on the SAME positions, and the
    list of a fresh build with the oracle pair set (S:Q6: list parity on given positions, never along trajectories)."""
    w = {"lj": lambda: W.lj_fluid(2 ** 14), "polymer": lambda: W.polymer_melt(128, 64),
         "patchy": lambda: W.patchy_fluid(2 ** 12, T=1.0)}[case]()
    s = MD.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces(strat, sc)
    s.integrate(w.dt, steps, strat, sc)
    assert s.stats()["n_rebuilds"] >= 2
    pos = s.in_id_order(s.pos)
    quat = s.in_id_order(s.quat) if w.quat is not None else None
    o = oracle.forces(pos, w.box, dict(w.potential), quat=quat)
    assert_forces(s, o, quat is not None, (f"{case} after {steps} steps", f"{strat}_{sc}"))
    s.build_cells(); s.build_verlet()
    pos2 = s.in_id_order(s.pos)                               # wrapped by the build
    assert_pairs(s, oracle, pos2, w.box, w.rcut, w.skin)
    s.close()


def test_nve_drift_c1_10k_steps(MD):
    """P9 / north_star: NVE energy drift of C1 over 10^4 steps stays below 5e-5 relative."""
    w = W.config("C1")
    s = MD.from_workload(w, order="cell")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    e0 = sum(s.energy())
    worst = 0.0
    for _ in range(20):
        s.integrate(w.dt, 500, "vertex")
        worst = max(worst, abs(sum(s.energy()) - e0) / abs(e0))
    assert worst <= 5e-5
    st = s.stats()
    assert 300 <= st["n_rebuilds"] <= 600                     # a rebuild every ~25 steps
    v = s.vel.double().sum(dim=0).cpu().numpy()[:3]
    assert np.abs(v).max() < 1e-2                             # momentum stays ~0
    s.close()


def test_step_host_end_to_end(MD, oracle):
    import torch
    w = W.config("C1")
    s = MD.from_workload(w, order="hilbert")
    pos = torch.from_numpy(w.pos.copy()).pin_memory()
    vel = torch.from_numpy(w.vel.copy()).pin_memory()
    force = torch.zeros_like(pos).pin_memory()
    s.step_host(pos, vel, force, w.dt, 0, "vertex")
    o = oracle.forces(w.pos, w.box, dict(w.potential))
    assert np.abs(force.numpy()[:, :3] - o["F"]).max() <= FTOL_REL * np.abs(o["F"]).max() + FTOL_ABS
    assert np.array_equal(pos.numpy(), w.pos)
    s.step_host(pos, vel, force, w.dt, 10, "edge", "red_v4")
    o10 = oracle.integrate(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, 10)
    assert np.abs(force.numpy()[:, :3] - o10["F"]).max() <= FTOL_REL * np.abs(o10["F"]).max() + FTOL_ABS
    s.close()


def test_crossover_sweep_runs(capsys, monkeypatch):
    """The configs[4] sweep script: one small cell of the grid, every variant, a table on stdout."""
    import sys
    import crossover
    monkeypatch.setattr(sys, "argv", ["crossover", "--min-log2n", "12", "--max-log2n", "12", "--evals", "2", "--rcuts", "2.5",
                                      "--orders", "none,hilbert"])
    crossover.main()
    out = capsys.readouterr().out
    assert "| lj | 2^12 | 0.8 | 2.5 | hilbert |" in out and "| patchy | 2^12 | 0.5 | 1.5 | none |" in out and "| patchy_pp | 2^12 |" in out


# ---- mixed precision (S:8(f3)): fp64 integration of the state, fp32 forces ----
def test_mixed_precision_free_flight_matches_fp64_oracle(MD, oracle):
    """A dilute lattice (nearest neighbours beyond r_v, so every force is exactly zero) translating rigidly: the fp64
    state must follow the fp64 oracle and the closed form x0 + n dt v to rounding through ~20 device-side rebuilds
    (wrap in fp64, Hilbert reordering of the fp64 planes); the fp32 state of the default precision cannot."""
    w = W.lj_fluid(256, rho=0.03, jitter=0.0)
    w.vel[:, :3] = np.array([0.7, -0.3, 0.45], dtype=np.float32)
    nsteps = 2000
    o = oracle.integrate(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, nsteps)
    assert np.abs(o["F"]).max() == 0.0
    exact = w.pos[:, :3].astype(np.float64) + nsteps * w.dt * w.vel[:, :3].astype(np.float64)
    err = {}
    for prec in ("mixed", "f32"):
        s = MD.from_workload(w, order="hilbert")
        s.set_precision(prec)
        s.build_cells(); s.build_verlet(); s.forces("vertex")
        s.integrate(w.dt, nsteps, "vertex")
        assert s.stats()["n_rebuilds"] >= 10
        if prec == "mixed":
            x, v = s.state_f64()
            assert np.array_equal(v, w.vel[:, :3].astype(np.float64))
            x32 = s.in_id_order(s.pos)[:, :3]
            assert np.array_equal(x32, x.astype(np.float32))            # the fp32 arrays are the rounded fp64 state
        else:
            x = s.in_id_order(s.pos)[:, :3].astype(np.float64)
        for name, ref in (("oracle", o["pos"][:, :3]), ("closed_form", exact)):
            dx = x - ref
            dx -= w.box * np.round(dx / w.box)
            err[(prec, name)] = np.abs(dx).max()
        s.close()
    assert err[("mixed", "oracle")] < 1e-11 and err[("mixed", "closed_form")] < 1e-11
    assert err[("f32", "closed_form")] > 1e-8                            # what the mode is for


@pytest.mark.parametrize("strat,sc", [("vertex", "smem"), ("edge", "warp")])
def test_mixed_precision_c1_trajectory(MD, oracle, strat, sc):
    """C1, 100 steps: mixed precision stays within the tolerances of the fp32 trajectory test against the fp64 oracle."""
    w = W.config("C1")
    o = oracle.integrate(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, 100, every=100)
    s = MD.from_workload(w, order="cell")
    s.set_precision("mixed")
    s.build_cells(); s.build_verlet(); s.forces(strat, sc)
    s.integrate(w.dt, 100, strat, sc)
    assert s.stats()["n_rebuilds"] >= 1
    fmax = np.abs(o["F"]).max()
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= FTOL_REL * fmax + FTOL_ABS
    x, v = s.state_f64()
    dx = x - o["pos"][:, :3]
    dx -= w.box * np.round(dx / w.box)
    assert np.abs(dx).max() < 1e-4
    assert np.abs(v - o["vel"][:, :3]).max() < 1e-3
    e1 = s.energy()
    assert abs(sum(e1) - o["energies"][-1].sum()) <= ETOL * abs(o["energies"][-1].sum())
    s.close()


def test_mixed_precision_rigid_bodies_after_rebuilds(MD, oracle):
    """Patchy rigid bodies in mixed precision: after several device-side rebuilds the forces and torques the path holds
    equal the oracle's on the same positions and orientations, and the quaternions are still unit."""
    w = W.patchy_fluid(2 ** 12, T=1.0)
    s = MD.from_workload(w, order="hilbert")
    s.set_precision("mixed")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    s.integrate(w.dt, 300, "vertex")
    assert s.stats()["n_rebuilds"] >= 2
    pos, quat = s.in_id_order(s.pos), s.in_id_order(s.quat)
    assert np.abs(np.linalg.norm(quat.astype(np.float64), axis=1) - 1.0).max() < 1e-6
    o = oracle.forces(pos, w.box, dict(w.potential), quat=quat)
    assert_forces(s, o, True, ("patchy4096 mixed precision after 300 steps", "vertex_smem"))
    s.close()


def test_mixed_precision_nve_drift_c1(MD):
    """mixed precision 'improves stability': the C1 energy drift over 10^4 steps is bounded as in fp32."""
    w = W.config("C1")
    s = MD.from_workload(w, order="cell")
    s.set_precision("mixed")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    e0 = sum(s.energy())
    worst = 0.0
    for _ in range(20):
        s.integrate(w.dt, 500, "vertex")
        worst = max(worst, abs(sum(s.energy()) - e0) / abs(e0))
    print("mixed-precision C1 drift over 1e4 steps:", worst)
    assert worst <= 5e-5
    s.close()


def test_precision_errors(MD):
    from paper_1401_4350_b200 import MDError
    s = MD.from_workload(W.config("C1"))
    with pytest.raises(MDError) as e:
        s.set_precision(5)
    assert e.value.code == -1
    with pytest.raises(MDError) as e:
        s.state_f64()                          # default precision: no fp64 state
    assert e.value.code == -2
    s.close()


def test_patchy_pp_short_trajectory(MD, oracle):
    """The paper's own patchy model (S:8(f2)): bonded dimers released from rest, 100 rigid-body steps.  With a
    (sigma/r)^200 core a force follows a position error 200-fold, so the forces are compared on the positions and
    orientations the GPU holds (plain definition), the trajectory itself through positions and the conserved energy."""
    w = W.dimer_gas(512, "patchy_pp")
    o = oracle.integrate(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, 100, every=100, quat=w.quat, angmom=w.angmom)
    for strat, sc in (("vertex", "smem"), ("vertex", "l2"), ("edge", "red_v4"), ("edge", "segmented"), ("vertex_n3", 4)):
        s = MD.from_workload(w, order="hilbert")
        s.build_cells(); s.build_verlet(); s.forces(strat, sc)
        e0 = sum(s.energy())
        s.integrate(w.dt, 100, strat, sc)
        pos, quat = s.in_id_order(s.pos), s.in_id_order(s.quat)
        snap = oracle.forces(pos, w.box, dict(w.potential), quat=quat)
        assert_forces(s, snap, True, ("patchy_pp dimers after 100 steps", f"{strat}_{sc}"))
        dx = pos[:, :3].astype(np.float64) - o["pos"][:, :3]
        dx -= w.box * np.round(dx / w.box)
        assert np.abs(dx).max() < 1e-4
        e1 = sum(s.energy())                                  # U on these positions was compared inside assert_forces
        assert abs(e1 - e0) <= 2e-3 * abs(e0)                 # conserved along the stiff trajectory (dt = 0.002)
        assert abs(o["energies"][-1].sum() - o["e0"].sum()) <= 2e-3 * abs(o["e0"].sum())
        s.close()


@pytest.mark.parametrize("case", ["lj", "polymer", "patchy", "patchy_pp"])
def test_blocks_over_the_launch_capacity_take_the_unstaged_path(MD, oracle, case):
    """A block whose neighbourhood outgrew the staged launch capacity is computed from global memory through its
    segment table instead of failing the run: force every block onto that path (MD_OPT_STAGE_LIMIT) and compare with
    the oracle."""
    w = {"lj": lambda: W.lj_fluid(2 ** 13), "polymer": lambda: W.polymer_melt(64, 64),
         "patchy": lambda: W.patchy_fluid(2 ** 12, rho=0.9, jitter=0.1), "patchy_pp": lambda: W.dimer_gas(2048, "patchy_pp")}[case]()
    s = MD.from_workload(w, order="hilbert")
    s.set_option("stage_limit", 64)
    s.build_cells(); s.build_verlet(); s.forces("vertex", "smem")
    o = oracle.forces(w.pos, w.box, dict(w.potential), quat=w.quat)
    assert_forces(s, o, w.quat is not None, (f"{case} unstaged path", "vertex_smem"))
    s.integrate(w.dt, 20, "vertex", "smem")
    pos = s.in_id_order(s.pos)
    quat = s.in_id_order(s.quat) if w.quat is not None else None
    assert_forces(s, oracle.forces(pos, w.box, dict(w.potential), quat=quat), quat is not None, (f"{case} unstaged path after 20 steps", "vertex_smem"))
    s.close()


# ---- thermostat (S:8(f3); reading DESIGN.md QT, oracle O9) ----
@pytest.mark.parametrize("order", ["none", "hilbert"])
@pytest.mark.parametrize("prec", ["f32", "mixed"])
def test_thermostat_one_application_matches_oracle(MD, oracle, order, prec):
    """One application on rigid bodies over several blocks and a ragged tail: the SET of refreshed particles is the
    oracle's exactly (integer decision), untouched entries keep their bits, refreshed ones are the oracle's fp64 draws
    rounded to fp32 (fp64 copies: to 1e-13); independent of the storage order."""
    w = W.patchy_fluid(2 ** 12, T=0.15)
    T, pt, pr, seed, call = 0.4, 0.3, 0.6, (7 << 32) + 12345, 9
    s = MD.from_workload(w, order=order)
    s.set_precision(prec)
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    v_in, L_in = s.in_id_order(s.vel).copy(), s.in_id_order(s.angmom).copy()
    F_in = s.in_id_order(s.force).copy()
    ov, oL, nt, nr = oracle.thermostat(v_in[:, :3].astype(np.float64), dict(w.potential), T, pt, seed, call,
                                       angmom_d=L_in[:, :3].astype(np.float64), p_r=pr)
    s.thermostat(T, pt, pr, seed, call)
    v, L = s.in_id_order(s.vel), s.in_id_order(s.angmom)
    for got, before, ref, n in ((v, v_in, ov, nt), (L, L_in, oL, nr)):
        changed_ref = np.any(ref != before[:, :3].astype(np.float64), axis=1)
        changed = np.any(got[:, :3] != before[:, :3], axis=1)
        assert changed_ref.sum() == n and 0 < n < w.N
        assert np.array_equal(changed, changed_ref)
        assert np.array_equal(got[~changed], before[~changed])               # bits untouched, w component included
        assert np.array_equal(got[:, 3], before[:, 3])
        assert np.abs(got[:, :3] - ref).max() <= 2e-7 * np.abs(ref).max()
    assert np.array_equal(s.in_id_order(s.force), F_in)                       # forces untouched and still valid
    if prec == "mixed":
        _, v64 = s.state_f64()
        assert np.abs(v64 - ov).max() <= 1e-13
        assert np.array_equal(v64.astype(np.float32), v[:, :3])
    K = s.energy()[1]
    assert abs(K - 0.5 * (ov * ov).sum()) <= 1e-5 * K
    s.close()


def test_thermostat_p0_p1_and_small_sizes(MD, oracle):
    """p = 0 is the identity, p = 1 refreshes everything; N below one block, one block and a ragged tail."""
    for N in (32, 256, 500):
        w = W.lj_fluid(N, rho=0.03)
        s = MD.from_workload(w)
        v_in = s.in_id_order(s.vel).copy()
        s.thermostat(1.0, 0.0, 0.0, 3, 1)
        assert np.array_equal(s.in_id_order(s.vel), v_in)
        s.thermostat(1.3, 1.0, 0.0, 3, 1)
        ov, _, nt, _ = oracle.thermostat(v_in[:, :3], dict(w.potential), 1.3, 1.0, 3, 1)
        assert nt == w.N
        assert np.abs(s.in_id_order(s.vel)[:, :3] - ov).max() <= 2e-7 * np.abs(ov).max()
        s.close()


@pytest.mark.parametrize("strat,sc", [("vertex", "smem"), ("edge", "warp")])
def test_thermostat_nvt_trajectory_c1(MD, oracle, strat, sc):
    """C1, 60 steps with a refresh every 20 (three applications, one inside an 8-step graph chunk boundary): same
    tolerances as the NVE trajectory test, and the refreshed velocities of the LAST application are the oracle's."""
    w = W.config("C1")
    T, n_newt, pt, seed = 0.8, 20, 0.25, 424242
    o = oracle.integrate_nvt(w.pos, w.vel, w.box, dict(w.potential), w.skin, w.dt, 60, T=T, n_newt=n_newt, p_t=pt, seed=seed)
    s = MD.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces(strat, sc)
    s.set_thermostat(T, n_newt, pt, 0.0, seed)
    s.integrate(w.dt, 33, strat, sc)            # split across calls: the step count carries over
    s.integrate(w.dt, 27, strat, sc)
    fmax = np.abs(o["F"]).max()
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= FTOL_REL * fmax + FTOL_ABS
    x = s.in_id_order(s.pos)[:, :3].astype(np.float64)
    dx = x - o["pos"][:, :3]
    dx -= w.box * np.round(dx / w.box)
    assert np.abs(dx).max() < 1e-4
    v = s.in_id_order(s.vel)[:, :3]
    assert np.abs(v - o["vel"][:, :3]).max() < 1e-3
    # the particles refreshed by application 3 (after step 60) carry exactly the oracle's draw
    ov3, _, n3, _ = oracle.thermostat(np.zeros((w.N, 3)), dict(w.potential), T, pt, seed, 3)
    hit = np.any(ov3 != 0.0, axis=1)
    assert n3 == hit.sum() > 0
    assert np.abs(v[hit] - ov3[hit]).max() <= 2e-7 * np.abs(ov3).max()
    s.set_thermostat(T, 0, 0.0, 0.0, 0)         # off again: NVE
    e0 = sum(s.energy())
    s.integrate(w.dt, 40, strat, sc)
    assert abs(sum(s.energy()) - e0) <= 5e-5 * abs(e0)
    s.close()


def test_thermostat_relaxes_a_hot_fluid_and_errors(MD):
    from paper_1401_4350_b200 import MDError
    w = W.lj_fluid(2 ** 14, T=2.0)
    s = MD.from_workload(w, order="hilbert")
    with pytest.raises(MDError) as e:
        s.set_thermostat(-1.0, 10, 0.1)
    assert e.value.code == -1
    with pytest.raises(MDError) as e:
        s.thermostat(1.0, 1.5)
    assert e.value.code == -1
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    s.set_thermostat(1.0, 10, 0.2, 0.0, 11)
    s.integrate(w.dt, 1200, "vertex")
    temps = []
    for _ in range(10):
        s.integrate(w.dt, 20, "vertex")
        temps.append(2.0 * s.energy()[1] / (3.0 * w.N))
    assert abs(np.mean(temps) - 1.0) < 0.04
    s.close()
