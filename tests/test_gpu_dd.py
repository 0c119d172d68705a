"""Space decomposition on the GPU (P:37-39, S:8(e), S:8(f4)): the kernels md_dd_select / md_gather_ids / md_scatter_ids /
md_half_step / md_set_active / md_resize and the protocol of paper_1401_4350_b200/dd.py, with 2 and 3 slab domains
living in ONE process on ONE GPU (in-process transport; the domains run one after the other, nothing waits on a peer and
nothing is timed).  Checked against the oracle on the union of the domains and against the single-domain run."""
import numpy as np
import pytest

import workloads as W
from conftest import record_margin

pytestmark = pytest.mark.gpu

FTOL_REL, FTOL_ABS = 1e-4, 1e-6


def make_sim(w, nranks, strategy, variant, order="hilbert"):
    from paper_1401_4350_b200.dd import DDSimulation, Domain, LocalTransport, SlabPlan
    plan = SlabPlan(w.box, nranks, w.rcut + w.skin)
    doms = []
    for r in range(nranks):
        d = Domain(r, plan, w.N, w.rcut, w.skin, w.potential, w.max_neigh, order=order, strategy=strategy, variant=variant)
        d.load_initial(w.pos, w.vel, w.quat, w.angmom)
        doms.append(d)
    sim = DDSimulation(doms, LocalTransport(plan))
    sim.rebuild()
    return sim, plan


def test_select_gather_scatter_kernels():
    import torch
    from paper_1401_4350_b200 import MDSystem
    from paper_1401_4350_b200.binding import dd_select
    from paper_1401_4350_b200.dd import select_np
    w = W.lj_fluid(5000 if False else 2 ** 12, 2.5)
    pos = torch.from_numpy(w.pos).cuda()
    for lo, hi in ((0.0, 3.3), (2.5, 2.5), (4.0, 100.0), (-1.0, 0.0)):
        got = dd_select(pos, lo, hi).cpu().numpy()
        assert np.array_equal(got, select_np(w.pos[:, 0], lo, hi))            # stable, ascending, fp32 comparisons
    assert np.array_equal(dd_select(pos, 1.0, 2.0, axis=2).cpu().numpy(), select_np(w.pos[:, 2], 1.0, 2.0))
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    ids = torch.tensor([5, 17, 4095, 0, 2048], dtype=torch.int32, device="cuda")
    assert np.array_equal(s.gather_ids("pos", ids=ids).cpu().numpy(), w.pos[[5, 17, 4095, 0, 2048]])   # by ORIGINAL id, storage is Hilbert-ordered
    assert np.array_equal(s.gather_ids("vel", first_id=100, n=50).cpu().numpy(), w.vel[100:150])
    new = torch.from_numpy(w.pos[200:260] + np.float32(0.001)).cuda()
    s.scatter_ids("pos", 200, new)
    back = s.in_id_order(s.pos)
    assert np.array_equal(back[200:260], new.cpu().numpy()) and np.array_equal(back[:200], w.pos[:200])
    s.close()


def test_ghosts_are_neither_integrated_nor_counted():
    from paper_1401_4350_b200 import MDSystem
    w = W.config("C1")
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    e_all = s.energy()
    s.set_active(1500)
    e_act = s.energy()
    F = s.in_id_order(s.force)
    assert abs(e_act[0] - F[:1500, 3].astype(np.float64).sum()) < 1e-6 * abs(e_all[0])
    assert abs(e_act[1] - 0.5 * (w.vel[:1500, :3].astype(np.float64) ** 2).sum()) < 1e-6 * e_all[1]
    s.half_step(w.dt, "kick_drift")
    pos, vel = s.in_id_order(s.pos), s.in_id_order(s.vel)
    assert np.array_equal(pos[1500:], w.pos[1500:]) and np.array_equal(vel[1500:], w.vel[1500:])       # ghosts frozen
    assert not np.array_equal(pos[:1500], w.pos[:1500])
    s.forces("vertex"); s.half_step(w.dt, "kick")
    assert np.array_equal(s.in_id_order(s.vel)[1500:], w.vel[1500:])
    # md_half_step is md_integrate split in two: same bits as one md_integrate step when nobody is a ghost
    a = MDSystem.from_workload(w, order="hilbert"); b = MDSystem.from_workload(w, order="hilbert")
    for x in (a, b):
        x.build_cells(); x.build_verlet(); x.forces("vertex", "smem")
    a.integrate(w.dt, 1, "vertex", "smem")
    b.half_step(w.dt, "kick_drift"); b.forces("vertex", "smem"); b.half_step(w.dt, "kick")
    assert np.array_equal(a.in_id_order(a.pos), b.in_id_order(b.pos)) and np.array_equal(a.in_id_order(a.vel), b.in_id_order(b.vel))
    for x in (s, a, b):
        x.close()


@pytest.mark.parametrize("nranks,strategy,variant", [(2, "vertex", "smem"), (3, "vertex", "smem"), (3, "edge", "warp"), (2, "edge", "cluster")])
def test_lj_domains_match_the_oracle_and_the_single_domain(oracle, nranks, strategy, variant):
    from paper_1401_4350_b200 import MDSystem
    from paper_1401_4350_b200.dd import local_sets_np
    w = W.lj_fluid(2 ** 14, 2.5)                                     # cubic box 27.4 sigma: slabs of 13.7 / 9.1 >= 2 r_v
    sim, plan = make_sim(w, nranks, strategy, variant)
    # the local sets are the reference ones, ghosts in message order
    for r, d in sim.domains.items():
        own_ref, ghost_ref = local_sets_np(w.pos, plan, r)
        gid = d.sys.gather_ids("pos", first_id=0, n=d.sys.N).cpu().numpy()[:, 3].copy().view(np.int32)
        assert np.array_equal(gid[:d.n_own], own_ref) and np.array_equal(gid[d.n_own:], ghost_ref)
    # step 0: forces of the owned particles = the oracle's forces on the whole system
    o = oracle.forces(w.pos, w.box, dict(w.potential))
    F = sim.gather("force", w.N)
    assert not np.isnan(F).any()                                      # every particle is owned exactly once
    tol = FTOL_REL * np.abs(o["F"]).max() + FTOL_ABS
    err = np.abs(F[:, :3] - o["F"]).max()
    record_margin(f"dd {nranks} slabs lj N=2^14", f"{strategy}_{variant}", "F", err, tol)
    assert err <= tol
    U = sim.energy()[0]
    assert abs(U - o["pe"].sum()) <= 1e-5 * abs(o["pe"].sum())       # ghosts are left out of the sums: no double counting
    # 100 steps: rebuilds, migration across the faces, halo refresh every step
    own0 = {r: d.owned("pos")[0].copy() for r, d in sim.domains.items()}
    sim.run(w.dt, 100)
    assert all(d.n_rebuilds >= 3 for d in sim.domains.values())
    moved = sum(len(np.setxor1d(own0[r], d.owned("pos")[0])) for r, d in sim.domains.items())
    assert moved > 0                                                  # particles changed owner
    pos, F = sim.gather("pos", w.N), sim.gather("force", w.N)
    assert not np.isnan(pos).any()
    o = oracle.forces(pos, w.box, dict(w.potential))                 # snapshot parity on the positions the domains hold
    tol = FTOL_REL * np.abs(o["F"]).max() + FTOL_ABS
    err = np.abs(F[:, :3] - o["F"]).max()
    record_margin(f"dd {nranks} slabs lj N=2^14 after 100 steps", f"{strategy}_{variant}", "F", err, tol)
    assert err <= tol
    # the same trajectory as one domain (fp32 trajectories from one input stay together for 100 steps)
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet(); s.forces(strategy, variant)
    e0 = sum(s.energy())
    s.integrate(w.dt, 100, strategy, variant)
    x1 = s.in_id_order(s.pos)[:, :3].astype(np.float64)
    dx = pos[:, :3].astype(np.float64) - x1
    dx -= w.box * np.round(dx / w.box)
    assert np.abs(dx).max() < 1e-4
    assert abs(sum(sim.energy()) - e0) <= 5e-5 * abs(e0)             # NVE across the domains
    s.close(); sim.close()


def test_patchy_domains(oracle):
    """Rigid bodies: quaternions travel with the halo, angular momenta with the migrants."""
    w = W.patchy_fluid(2 ** 13, T=1.0)
    sim, plan = make_sim(w, 2, "vertex", "smem")
    sim.run(w.dt, 60)
    assert all(d.n_rebuilds >= 2 for d in sim.domains.values())
    pos, quat = sim.gather("pos", w.N), sim.gather("quat", w.N)
    F, T = sim.gather("force", w.N), sim.gather("torque", w.N)
    assert np.abs(np.linalg.norm(quat.astype(np.float64), axis=1) - 1.0).max() < 1e-5
    o = oracle.forces(pos, w.box, dict(w.potential), quat=quat)
    assert np.abs(F[:, :3] - o["F"]).max() <= FTOL_REL * np.abs(o["F"]).max() + FTOL_ABS
    assert np.abs(T[:, :3] - o["T"]).max() <= FTOL_REL * np.abs(o["T"]).max() + FTOL_ABS
    sim.close()


def _dd_worker(rank, world, port, out):
    import os
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    from paper_1401_4350_b200.dd import DDSimulation, DistTransport, Domain, SlabPlan
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.lj_fluid(2 ** 14, 2.5)
    plan = SlabPlan(w.box, world, w.rcut + w.skin)
    d = Domain(rank, plan, w.N, w.rcut, w.skin, w.potential, w.max_neigh, device="cuda:0", strategy="vertex", variant="smem")
    d.load_initial(w.pos, w.vel)
    sim = DDSimulation([d], DistTransport(plan, dist, torch.device("cuda:0"), stage_host=True))
    sim.rebuild()
    sim.run(w.dt, 60)
    np.save(out + f".pos.{rank}.npy", sim.gather("pos", w.N))
    np.save(out + f".force.{rank}.npy", sim.gather("force", w.N))
    np.save(out + f".e.{rank}.npy", np.array(list(sim.energy()) + [d.n_rebuilds, d.n_own]))
    sim.close()
    dist.barrier()
    dist.destroy_process_group()


def test_two_processes_over_torch_distributed(oracle, tmp_path):
    """The real multi-process path: two ranks, each with its own md_system and its own process, exchanging migrants and
    halos through torch.distributed (gloo, staged through host memory because both ranks share this one GPU; nothing
    is timed and no kernel waits on a peer -- the processes block on the host).  bench.py --dd is this with nccl."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "dd2")
    mp.spawn(_dd_worker, args=(2, port, out), nprocs=2, join=True)
    w = W.lj_fluid(2 ** 14, 2.5)
    pos = np.load(out + ".pos.0.npy"); F = np.load(out + ".force.0.npy")
    p1 = np.load(out + ".pos.1.npy"); F1 = np.load(out + ".force.1.npy")
    own0, own1 = ~np.isnan(pos[:, 0]), ~np.isnan(p1[:, 0])
    assert (own0 ^ own1).all()                                       # every particle owned by exactly one rank
    pos[own1] = p1[own1]; F[own1] = F1[own1]
    e0, e1 = np.load(out + ".e.0.npy"), np.load(out + ".e.1.npy")
    assert e0[3] >= 2 and e0[3] == e1[3] and e0[4] + e1[4] == w.N    # the ranks rebuilt together
    o = oracle.forces(pos, w.box, dict(w.potential))
    assert np.abs(F[:, :3] - o["F"]).max() <= FTOL_REL * np.abs(o["F"]).max() + FTOL_ABS
    assert abs((e0[0] + e1[0]) - o["pe"].sum()) <= 1e-5 * abs(o["pe"].sum())
