"""Parity at BASELINE.json's full size (configs[1]: LJ, N = 2^20, r_c = 2.5), in the launch configuration
bench.py times (order = hilbert, VERTEX and EDGE).  The oracle (OpenMP, cell-pruned plain definition) handles
the whole system in seconds, so every particle is compared, not a sample."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


def test_c2_full_size_parity(oracle):
    from paper_1401_4350_b200 import MDSystem
    w = W.config("C2a")
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet()
    got = s.get_pairs()
    got = got[np.lexsort((got[:, 1], got[:, 0]))]
    ref = oracle.pair_set(w.pos, w.box, w.rcut, w.skin)
    assert got.shape == ref.shape and np.array_equal(got, ref)
    o = oracle.forces(w.pos, w.box, dict(w.potential))
    fmax = np.abs(o["F"]).max()
    tol = 1e-4 * fmax + 1e-6
    for strat, sc in [("vertex", "smem"), ("vertex", "l2"), ("edge", "red_v4"), ("edge", "warp"),
                      ("edge", "segmented"), ("edge", "cluster"), ("vertex_n3", 12)]:
        s.forces(strat, sc)
        F = s.in_id_order(s.force)
        assert np.abs(F[:, :3] - o["F"]).max() <= tol, (strat, sc)
        U, Kt, _ = s.energy()
        assert abs(U - o["pe"].sum()) <= 1e-5 * abs(o["pe"].sum())
    # melted, load-imbalanced state: integrate, then snapshot parity on the positions the GPU holds
    s.forces("vertex")
    s.integrate(w.dt, 200, "vertex")
    pos = s.in_id_order(s.pos)
    o = oracle.forces(pos, w.box, dict(w.potential))
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= 1e-4 * np.abs(o["F"]).max() + 1e-6
    # the same in mixed precision: fp64 state through the device-side rebuilds, fp32 forces on its rounding
    s.set_precision("mixed")
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    s.integrate(w.dt, 100, "vertex")
    x64, _ = s.state_f64()
    pos = s.in_id_order(s.pos)
    assert np.array_equal(pos[:, :3], x64.astype(np.float32))
    o = oracle.forces(pos, w.box, dict(w.potential))
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= 1e-4 * np.abs(o["F"]).max() + 1e-6
    s.close()


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_c3_c4_full_size_parity(oracle, name):
    """configs[2] (polymer melt, 4096 x 64 beads) and configs[3] (patchy rigid bodies, N = 2^18) at full size, every
    particle compared: lattice / walk start, then the state after device-side rebuilds."""
    from paper_1401_4350_b200 import MDSystem
    w = W.config(name)
    rigid = w.quat is not None
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet()
    assert s.stats()["n_edges"] == oracle.pair_count(w.pos, w.box, w.rcut, w.skin)
    o = oracle.forces(w.pos, w.box, dict(w.potential), quat=w.quat)
    variants = [("vertex", "smem"), ("vertex", "l2"), ("edge", "red_v4"), ("edge", "warp"), ("edge", "segmented"), ("edge", "cluster"), ("vertex_n3", 4)]
    for strat, sc in variants:
        s.forces(strat, sc)
        F = s.in_id_order(s.force)
        assert np.abs(F[:, :3] - o["F"]).max() <= 1e-4 * np.abs(o["F"]).max() + 1e-6, (strat, sc)
        if rigid:
            T = s.in_id_order(s.torque)
            assert np.abs(T[:, :3] - o["T"]).max() <= 1e-4 * np.abs(o["T"]).max() + 1e-6, (strat, sc)
    s.forces("vertex")
    s.integrate(w.dt, 200, "vertex")
    assert s.stats()["n_rebuilds"] >= 1
    pos = s.in_id_order(s.pos)
    quat = s.in_id_order(s.quat) if rigid else None
    o = oracle.forces(pos, w.box, dict(w.potential), quat=quat)
    F = s.in_id_order(s.force)
    assert np.abs(F[:, :3] - o["F"]).max() <= 1e-4 * np.abs(o["F"]).max() + 1e-6
    if rigid:
        T = s.in_id_order(s.torque)
        assert np.abs(T[:, :3] - o["T"]).max() <= 1e-4 * np.abs(o["T"]).max() + 1e-6
    s.close()


def test_c2b_many_neighbours(oracle):
    """configs[1] many-neighbour variant (r_c = 4.0): full pair-count check and forces on the whole system."""
    from paper_1401_4350_b200 import MDSystem
    w = W.config("C2b")
    s = MDSystem.from_workload(w, order="hilbert")
    s.build_cells(); s.build_verlet()
    st = s.stats()
    o = oracle.forces(w.pos, w.box, dict(w.potential))
    for strat, sc in [("vertex", "smem"), ("vertex", "l2"), ("edge", "warp"), ("edge", "cluster")]:
        s.forces(strat, sc)
        F = s.in_id_order(s.force)
        assert np.abs(F[:, :3] - o["F"]).max() <= 1e-4 * np.abs(o["F"]).max() + 1e-6
    # E = 1/2 sum |L_i| must equal the oracle's pair count exactly (the sorted-set comparison at this
    # density and cutoff is done at N = 2^14 in test_step0_parity)
    assert st["n_edges"] == oracle.pair_count(w.pos, w.box, w.rcut, w.skin)
    s.close()


@pytest.mark.parametrize("name,prec", [("C2a", "f32"), ("C4", "mixed")])
def test_thermostat_full_size(oracle, name, prec):
    """The thermostat (reading QT) at full size in bench.py's configuration (Hilbert-ordered storage, so the
    id-keyed streams are read through a non-trivial permutation); O9 is O(N): every particle is compared."""
    from paper_1401_4350_b200 import MDSystem
    w = W.config(name)
    rigid = w.quat is not None
    s = MDSystem.from_workload(w, order="hilbert")
    s.set_precision(prec)
    s.build_cells(); s.build_verlet(); s.forces("vertex")
    assert not np.array_equal(s.get_ids(), np.arange(w.N))
    v0 = s.in_id_order(s.vel).copy()
    L0 = s.in_id_order(s.angmom).copy() if rigid else None
    T, pt, pr, seed, call = 0.7, 0.1, 0.1 if rigid else 0.0, (1 << 63) + 5, 4000000000
    s.thermostat(T, pt, pr, seed, call)
    ov, oL, nt, nr = oracle.thermostat(v0[:, :3].astype(np.float64), dict(w.potential), T, pt, seed, call,
                                       angmom_d=L0[:, :3].astype(np.float64) if rigid else None, p_r=pr)
    v1 = s.in_id_order(s.vel)
    hit = np.any(ov != v0[:, :3], axis=1)
    assert hit.sum() == nt and abs(nt - pt * w.N) < 5.0 * np.sqrt(w.N * pt * (1 - pt))
    assert np.array_equal(np.any(v1[:, :3] != v0[:, :3], axis=1), hit)
    assert np.array_equal(v1[~hit], v0[~hit])
    assert np.abs(v1[:, :3] - ov).max() <= 2e-7 * np.abs(ov).max()
    if rigid:
        L1 = s.in_id_order(s.angmom)
        hitr = np.any(oL != L0[:, :3], axis=1)
        assert hitr.sum() == nr > 0
        assert np.array_equal(np.any(L1[:, :3] != L0[:, :3], axis=1), hitr)
        assert np.abs(L1[:, :3] - oL).max() <= 2e-7 * np.abs(oL).max()
    if prec == "mixed":
        _, v64 = s.state_f64()
        assert np.abs(v64 - ov).max() <= 1e-13
    s.close()
