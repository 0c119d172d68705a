"""Pins of the fp64 oracle against things other than itself.

Closed forms, textbook lattice sums, brute force on small inputs, finite differences of the ENERGY
against the FORCE/TORQUE code, Newton-3 invariants, NVE drift, the free rotor, and the paper's one
numeric example (Fig. 1 thread counts).  CPU only.
"""
import math

import numpy as np
import pytest

import workloads as W
from conftest import read_kv, read_table

CF = read_kv("closed_forms.txt")
LJ25 = W.lj_potential(2.5)
LJ_UNSHIFTED = dict(W.lj_potential(2.5), shift_energy=0)
POLY = W.polymer_potential()
PATCHY = W.patchy_potential()
ID = (1.0, 0.0, 0.0, 0.0)


def quat_from_to(a, b):
    """Shortest-arc unit quaternion rotating unit vector a onto b."""
    a, b = np.asarray(a, float), np.asarray(b, float)
    c = np.cross(a, b)
    w = 1.0 + a @ b
    if w < 1e-12:  # antiparallel: rotate pi about any axis orthogonal to a
        ax = np.cross(a, [1.0, 0.0, 0.0])
        if np.linalg.norm(ax) < 1e-6:
            ax = np.cross(a, [0.0, 1.0, 0.0])
        ax /= np.linalg.norm(ax)
        return np.array([0.0, *ax])
    q = np.array([w, *c])
    return q / np.linalg.norm(q)


def rotate(q, v):
    w, x, y, z = q
    R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                  [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                  [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
    return R @ np.asarray(v, float)


def qmul(a, b):
    return np.array([a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3],
                     a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2],
                     a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1],
                     a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0]])


# ------------------------------------------------------------------ P1: LJ closed forms (Eq. 1)
def test_p1_lj_closed_forms(oracle):
    r0 = 2.0 ** (1.0 / 6.0)
    assert abs(r0 - CF["lj_zero_force_r"]) < 1e-14
    inside, V, Fj, _, _ = oracle.pair(LJ_UNSHIFTED, [r0, 0, 0])
    assert inside == 1
    assert abs(V + 1.0) < 1e-14                 # V = -eps at the minimum
    assert np.abs(Fj).max() < 1e-13             # zero force there
    _, V, Fj, _, _ = oracle.pair(LJ_UNSHIFTED, [1.0, 0, 0])
    assert abs(V - CF["lj_V_at_sigma"]) < 1e-14
    assert abs(Fj[0] - CF["lj_F_at_sigma"]) < 1e-12   # repulsive: force on j along +r_vec
    assert Fj[1] == 0 and Fj[2] == 0
    # attraction beyond the minimum: force on j points back towards i
    _, _, Fj, _, _ = oracle.pair(LJ_UNSHIFTED, [0, 1.5, 0])
    assert Fj[1] < 0
    # cut and shift: V(rc^-) -> 0, V_c value, force untouched by the shift, nothing beyond rc
    _, Vs, Fs, _, _ = oracle.pair(LJ25, [1.3, 0, 0])
    _, Vu, Fu, _, _ = oracle.pair(LJ_UNSHIFTED, [1.3, 0, 0])
    assert abs((Vu - Vs) - CF["lj_Vc_2p5"]) < 1e-12
    assert abs(4 * (2.5 ** -12 - 2.5 ** -6) - CF["lj_Vc_2p5"]) < 1e-12
    assert abs(4 * (4.0 ** -12 - 4.0 ** -6) - CF["lj_Vc_4p0"]) < 1e-14
    assert np.array_equal(Fs, Fu)
    _, V, _, _, _ = oracle.pair(LJ25, [2.5 * (1 - 1e-12), 0, 0])
    assert abs(V) < 1e-10
    inside, V, Fj, _, _ = oracle.pair(LJ25, [2.5, 0, 0])      # strict '<'
    assert inside == 0 and V == 0 and not Fj.any()


# ------------------------------------------------------------------ P2: WCA + FENE
def test_p2_wca_fene(oracle):
    rc = 2.0 ** (1.0 / 6.0)
    for r in (0.9, 1.0, 1.1):
        _, Vw, Fw, _, _ = oracle.pair(POLY, [0, 0, r])
        _, Vl, Fl, _, _ = oracle.pair(LJ_UNSHIFTED, [0, 0, r])
        assert abs(Vw - (Vl + 1.0)) < 1e-12          # WCA = LJ + eps inside the cut
        assert np.allclose(Fw, Fl, rtol=0, atol=1e-12)
    _, V, Fj, _, _ = oracle.pair(POLY, [rc * (1 - 1e-13), 0, 0])
    assert abs(V) < 1e-10 and np.abs(Fj).max() < 1e-9   # continuous at the cut
    assert oracle.pair(POLY, [rc * 1.0001, 0, 0])[0] == 0
    bad, V, Fj = oracle.bond(POLY, [0, 0, 0])
    assert bad == 0 and V == 0.0 and not Fj.any()         # U_b(0) = 0
    bad, _, Fb = oracle.bond(POLY, [0.97, 0, 0])
    assert abs(-Fb[0] - CF["fene_F_at_0p97"]) < 1e-8      # attractive: force on j towards i
    assert abs(30 * 0.97 / (1 - 0.97 ** 2 / 2.25) - CF["fene_F_at_0p97"]) < 1e-8
    _, _, Fw, _, _ = oracle.pair(POLY, [0.97, 0, 0])
    assert abs(Fw[0] - CF["wca_F_at_0p97"]) < 1e-8
    assert oracle.bond(POLY, [1.5, 0, 0])[0] == 1         # bond at R0 flagged
    # minimum of the bonded pair energy: bracket the zero of the total radial force by bisection
    def frad(r):
        return oracle.pair(POLY, [r, 0, 0])[2][0] + oracle.bond(POLY, [r, 0, 0])[2][0]
    lo, hi = 0.9, 1.05
    assert frad(lo) > 0 > frad(hi)
    for _ in range(100):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if frad(mid) > 0 else (lo, mid)
    rstar = 0.5 * (lo + hi)
    assert abs(rstar - CF["fene_wca_rstar"]) < 1e-10
    Ustar = oracle.pair(POLY, [rstar, 0, 0])[1] + oracle.bond(POLY, [rstar, 0, 0])[1]
    assert abs(Ustar - CF["fene_wca_Ustar"]) < 1e-9


# ------------------------------------------------------------------ P3/P4: patchy closed forms
def test_p3_patchy_aligned(oracle):
    b1 = W.TETRA[0]
    qi = quat_from_to(b1, [1, 0, 0])      # patch 1 of i points at j (+x)
    qj = quat_from_to(b1, [-1, 0, 0])     # patch 1 of j points at i (-x)
    e3 = math.exp(-(4.0 / 3.0) / 0.09)
    for tag, r in (("1p0", 1.0), ("1p05", 1.05), ("1p2", 1.2)):
        inside, V, Fj, ti, tj = oracle.pair(PATCHY, [r, 0, 0], qi, qj)
        assert inside == 1
        assert abs(V - CF[f"patchy_V_aligned_{tag}"]) < 5e-10
        assert abs(-Fj[0] - CF[f"patchy_Fix_aligned_{tag}"]) < 5e-8     # F_i = -F_j
        assert abs(Fj[1]) < 1e-9 and abs(Fj[2]) < 1e-9
        assert np.abs(ti).max() < 1e-9 and np.abs(tj).max() < 1e-9      # symmetric arrangement: no torque
    # the r = sigma value from its closed form (B:10): +1 (WCA core) - 5 (1 + 3 e^{-(4/3)/0.09})^2
    assert abs((1.0 - 5.0 * (1 + 3 * e3) ** 2) - CF["patchy_V_aligned_1p0"]) < 1e-11
    # truncation, not shift, at 1.5 sigma (S:Q15): eps_p G(1.5) A_i A_j jump
    assert abs(math.exp(-0.25 / 0.02) - CF["patchy_G_at_1p5"]) < 1e-14
    assert oracle.pair(PATCHY, [1.5, 0, 0], qi, qj)[0] == 0


def test_p4_patch_antialigned(oracle):
    one = dict(PATCHY, n_patches=1, patch_dir=W.TETRA[:1].copy())
    b1 = W.TETRA[0]
    q_anti = quat_from_to(b1, [-1, 0, 0])    # patch of i points AWAY from j: cos(theta_i) = -1
    q_to_i = quat_from_to(b1, [-1, 0, 0])    # patch of j points at i: cos(theta_j) = +1
    r = 1.2                                   # outside the WCA core, so V is the patch term alone
    _, V, _, _, _ = oracle.pair(one, [r, 0, 0], q_anti, q_to_i)
    G = math.exp(-(r - 1) ** 2 / 0.02)
    assert abs(math.exp(-2 / 0.09) - CF["patchy_single_anti"]) < 1e-18
    assert abs(V - (-5.0 * G * CF["patchy_single_anti"])) < 1e-15       # "vanishes": 2.2e-10 of the aligned term
    _, Val, _, _, _ = oracle.pair(one, [r, 0, 0], quat_from_to(b1, [1, 0, 0]), q_to_i)
    assert abs(Val - (-5.0 * G)) < 1e-12
    # with all 4 tetrahedral patches the sum does NOT vanish (S:P4): -9.10e-3 at r = sigma, core excluded
    _, V4, _, _, _ = oracle.pair(PATCHY, [1.0, 0, 0], q_anti, q_to_i)
    assert abs((V4 - 1.0) - CF["patchy_Vpp_anti_4patch"]) < 5e-6


# ------------------------------------------------------------------ finite differences: force/torque code vs energy code
def _fd_pair(oracle, pot, rvec, qi, qj, h=1e-6):
    rvec = np.asarray(rvec, float)
    g = np.zeros(3)
    for k in range(3):
        e = np.zeros(3)
        e[k] = h
        g[k] = (oracle.pair(pot, rvec + e, qi, qj)[1] - oracle.pair(pot, rvec - e, qi, qj)[1]) / (2 * h)
    ti, tj = np.zeros(3), np.zeros(3)
    for k in range(3):
        ax = np.zeros(3)
        ax[k] = 1.0
        dqp = np.array([math.cos(h / 2), *(math.sin(h / 2) * ax)])
        dqm = np.array([math.cos(h / 2), *(-math.sin(h / 2) * ax)])
        ti[k] = -(oracle.pair(pot, rvec, qmul(dqp, qi), qj)[1] - oracle.pair(pot, rvec, qmul(dqm, qi), qj)[1]) / (2 * h)
        tj[k] = -(oracle.pair(pot, rvec, qi, qmul(dqp, qj))[1] - oracle.pair(pot, rvec, qi, qmul(dqm, qj))[1]) / (2 * h)
    return -g, ti, tj      # F_j = -dV/dr_vec


def test_finite_difference_pairs(oracle):
    rng = np.random.default_rng(5)
    worst = 0.0
    for _ in range(200):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        r = rng.uniform(0.9, 1.45)
        qi = rng.normal(size=4)
        qi /= np.linalg.norm(qi)
        qj = rng.normal(size=4)
        qj /= np.linalg.norm(qj)
        if rng.random() < 0.5:    # make a strongly bonded geometry half of the time
            qi = qmul(quat_from_to(rotate(qi, W.TETRA[1]), d + 0.2 * rng.normal(size=3) * 0.3), qi)
            qi /= np.linalg.norm(qi)
            qj = qmul(quat_from_to(rotate(qj, W.TETRA[2]), -d), qj)
            qj /= np.linalg.norm(qj)
        _, V, Fj, ti, tj = oracle.pair(PATCHY, r * d, qi, qj)
        Fd, tid, tjd = _fd_pair(oracle, PATCHY, r * d, qi, qj)
        scale = max(1.0, np.abs(Fj).max(), np.abs(ti).max(), np.abs(tj).max())
        worst = max(worst, np.abs(Fj - Fd).max() / scale, np.abs(ti - tid).max() / scale, np.abs(tj - tjd).max() / scale)
        # pair invariant (S:P7): tau_i + tau_j + r_vec x F_j = 0
        inv = ti + tj + np.cross(r * d, Fj)
        assert np.abs(inv).max() < 1e-10 * scale
    assert worst < 2e-7
    for pot in (LJ25, POLY):
        for r in (0.95, 1.05, 1.1, 1.8, 2.4):
            rv = r * np.array([0.3, -0.5, 0.81])
            rv *= r / np.linalg.norm(rv)
            inside, V, Fj, _, _ = oracle.pair(pot, rv)
            if inside:
                Fd, _, _ = _fd_pair(oracle, pot, rv, ID, ID)
                assert np.abs(Fj - Fd).max() < 1e-6 * max(1.0, np.abs(Fj).max())
    for r in (0.8, 0.97, 1.3):
        rv = np.array([0.2, 0.4, -0.6])
        rv *= r / np.linalg.norm(rv)
        _, _, Fb = oracle.bond(POLY, rv)
        g = np.array([(oracle.bond(POLY, rv + e)[1] - oracle.bond(POLY, rv - e)[1]) / 2e-6
                      for e in np.eye(3) * 1e-6])
        assert np.abs(Fb + g).max() < 1e-6 * max(1.0, np.abs(Fb).max())


def _total_U(oracle, x, box, pot, q=None):
    return oracle.forces_d(x, box, pot, q)["pe"].sum()


@pytest.mark.parametrize("kind", ["lj", "fene_wca", "patchy"])
def test_finite_difference_system(oracle, kind):
    """F_i = -dU/dx_i and tau_i = -dU/d(rotation_i) for the whole periodic system (catches index/sign errors
    in the accumulation over neighbours, the minimum image and the bonded pass)."""
    rng = np.random.default_rng(11)
    if kind == "lj":
        w = W.lj_fluid(256, 2.5)
    elif kind == "patchy":
        w = W.patchy_fluid(256, rho=0.9, jitter=0.12)       # dense + jittered so that cores and patches act
    else:
        w = W.polymer_melt(8, 32, relax_iters=30)
    x = w.pos[:, :3].astype(np.float64)
    q = w.quat.astype(np.float64) if w.quat is not None else None
    if q is not None:
        q /= np.linalg.norm(q, axis=1, keepdims=True)
    f = oracle.forces_d(x, w.box, w.potential, q)
    assert f["bad"] == 0
    h = 1e-6
    scale = max(1.0, np.abs(f["F"]).max())
    for i in rng.choice(w.N, 6, replace=False):
        for k in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, k] += h
            xm[i, k] -= h
            fd = -(_total_U(oracle, xp, w.box, w.potential, q) - _total_U(oracle, xm, w.box, w.potential, q)) / (2 * h)
            assert abs(fd - f["F"][i, k]) < 2e-6 * scale
            if q is not None:
                ax = np.zeros(3)
                ax[k] = 1
                qp, qm = q.copy(), q.copy()
                qp[i] = qmul(np.array([math.cos(h / 2), *(math.sin(h / 2) * ax)]), q[i])
                qm[i] = qmul(np.array([math.cos(h / 2), *(-math.sin(h / 2) * ax)]), q[i])
                td = -(_total_U(oracle, x, w.box, w.potential, qp) - _total_U(oracle, x, w.box, w.potential, qm)) / (2 * h)
                assert abs(td - f["T"][i, k]) < 2e-6 * max(1.0, np.abs(f["T"]).max())


# ------------------------------------------------------------------ P5: perfect fcc lattice, textbook lattice sums
def _fcc_shells(a, rmax):
    m = int(math.ceil(2 * rmax / a)) + 1
    rng = np.arange(-m, m + 1)
    i, j, k = np.meshgrid(rng, rng, rng, indexing="ij")
    ok = ((i + j + k) % 2 == 0) & ~((i == 0) & (j == 0) & (k == 0))
    d2 = (i[ok] ** 2 + j[ok] ** 2 + k[ok] ** 2) * (a / 2) ** 2
    return np.sqrt(d2[d2 < rmax * rmax])


@pytest.mark.parametrize("row", read_table("fcc_lattice_sums.txt"))
def test_p5_fcc_lattice(oracle, row):
    rc, n_rc, n_rv, u_ref = row
    a = (4.0 / 0.8) ** (1.0 / 3.0)
    r = _fcc_shells(a, rc + 0.3)
    inside = r[r < rc]
    assert len(inside) == int(n_rc) and len(r) == int(n_rv)
    u = 0.5 * np.sum(4 * (inside ** -12 - inside ** -6) - 4 * (rc ** -12 - rc ** -6))
    assert abs(u - u_ref) < 5e-8                       # golden file (SURVEY used a 10-digit lattice constant) vs lattice sum
    # the oracle's pipeline (cells, minimum image, pair set, force sum) on an fp64 lattice
    shape = (6, 6, 6) if rc < 3.5 else (8, 8, 8)
    x = W.fcc_sites(shape, a)
    box = np.array(shape, float) * a
    N = x.shape[0]
    f = oracle.forces_d(x, box, W.lj_potential(rc))
    assert abs(f["pe"].sum() / N - u) < 1e-10
    assert np.abs(f["pe"] - u).max() < 1e-10           # every site equivalent
    assert np.abs(f["F"]).max() < 1e-10                # zero force by symmetry
    assert f["n_in_cut"] * 2 == N * int(n_rc)
    w = W.lj_fluid(4 * 8 ** 3, rc, jitter=0.0)         # the fp32-rounded lattice the GPU will see
    pairs = oracle.pair_set(w.pos, w.box, rc, 0.3)
    assert 2 * len(pairs) == w.N * int(n_rv)           # E = n_rv N / 2 exactly (e.g. 39 N at rc = 2.5)
    assert np.bincount(pairs.ravel(), minlength=w.N).tolist() == [int(n_rv)] * w.N


def test_p5_fcc_rho05(oracle):
    w = W.patchy_fluid(2048, jitter=0.0)
    pairs = oracle.pair_set(w.pos, w.box, 1.5, 0.3)
    assert len(pairs) == 6 * w.N                        # 12 neighbours at sqrt(2) sigma inside both 1.5 and 1.8
    f = oracle.forces(w.pos, w.box, w.potential, w.quat)
    assert f["n_in_cut"] == 6 * w.N


# ------------------------------------------------------------------ P6 / P8: brute force vs cells; list integer invariants
@pytest.mark.parametrize("gen", ["lj", "lj4", "poly", "patchy", "tiny"])
def test_p6_pair_set_brute_vs_cells(oracle, gen):
    if gen == "lj":
        w = W.lj_fluid(2048, 2.5)
    elif gen == "lj4":
        w = W.lj_fluid(2048, 4.0)         # 13.68/4.3 -> 3 cells per axis
    elif gen == "poly":
        w = W.polymer_melt(32, 64, relax_iters=20)
    elif gen == "patchy":
        w = W.patchy_fluid(4096)
    else:
        w = W.lj_fluid(256, 2.5)          # box 6.84: 2 cells per axis -> de-duplicated stencil (S:Q8)
    pb = oracle.pair_set(w.pos, w.box, w.rcut, w.skin, use_cells=False)
    pc = oracle.pair_set(w.pos, w.box, w.rcut, w.skin, use_cells=True)
    assert np.array_equal(pb, pc)
    assert (pc[:, 0] < pc[:, 1]).all()
    key = pc[:, 0].astype(np.int64) * w.N + pc[:, 1]
    assert (np.diff(key) > 0).all()                                      # sorted, no duplicates
    # independent numpy check of the predicate on a sample of ordered pairs (fp64, same op order)
    x = w.pos[:, :3].astype(np.float64)
    rng = np.random.default_rng(3)
    ii = rng.integers(0, w.N, 20000)
    jj = rng.integers(0, w.N, 20000)
    keep = ii < jj
    ii, jj = ii[keep], jj[keep]
    d = x[jj] - x[ii]
    d = np.where(d > 0.5 * w.box, d - w.box, np.where(d < -0.5 * w.box, d + w.box, d))
    inside = ((d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]) < (w.rcut + w.skin) ** 2
    have = np.isin(ii.astype(np.int64) * w.N + jj, key)
    assert np.array_equal(inside, have)
    # E = 1/2 sum_i |L_i|  ("sum of the number of neighbours of each particle divided by two")
    deg = np.bincount(pc.ravel(), minlength=w.N)
    assert deg.sum() == 2 * len(pc)


@pytest.mark.parametrize("gen", ["lj", "poly", "patchy"])
def test_p8_forces_brute_vs_cells(oracle, gen):
    if gen == "lj":
        w = W.lj_fluid(2048, 2.5)
    elif gen == "poly":
        w = W.polymer_melt(32, 64, relax_iters=20)
    else:
        w = W.patchy_fluid(2048, rho=0.9, jitter=0.1)
    a = oracle.forces(w.pos, w.box, w.potential, w.quat, use_cells=True)
    b = oracle.forces(w.pos, w.box, w.potential, w.quat, use_cells=False)
    s = max(1.0, np.abs(b["F"]).max())
    assert np.abs(a["F"] - b["F"]).max() < 1e-12 * s
    assert np.abs(a["pe"] - b["pe"]).max() < 1e-12 * max(1.0, np.abs(b["pe"]).max())
    assert a["n_in_cut"] == b["n_in_cut"]
    if w.quat is not None:
        assert np.abs(a["T"] - b["T"]).max() < 1e-12 * max(1.0, np.abs(b["T"]).max())


# ------------------------------------------------------------------ O10: the single-core half-list loop (S:8(d))
@pytest.mark.parametrize("gen", ["lj", "poly", "patchy"])
def test_o10_half_list_loop_equals_the_plain_definition(oracle, gen):
    """O10 walks the half Verlet list once with Newton's third law; the pins are the O(N^2) plain definition (no cells,
    no list), exact momentum conservation of a pairwise antisymmetric sum, and the fcc lattice sum (closed form)."""
    if gen == "lj":
        w = W.lj_fluid(2048, 2.5)
    elif gen == "poly":
        w = W.polymer_melt(32, 64, relax_iters=20)
    else:
        w = W.patchy_fluid(2048, rho=0.9, jitter=0.1)
    pairs = oracle.pair_set(w.pos, w.box, w.rcut, w.skin)
    h = oracle.forces_half(w.pos, w.box, w.potential, pairs, quat=w.quat)
    b = oracle.forces(w.pos, w.box, w.potential, w.quat, use_cells=False)
    s = max(1.0, np.abs(b["F"]).max())
    assert np.abs(h["F"] - b["F"]).max() < 1e-11 * s
    assert np.abs(h["pe"] - b["pe"]).max() < 1e-11 * max(1.0, np.abs(b["pe"]).max())
    assert h["n_in_cut"] == b["n_in_cut"] and h["bad"] == 0
    if w.quat is not None:
        assert np.abs(h["T"] - b["T"]).max() < 1e-11 * max(1.0, np.abs(b["T"]).max())
    assert np.abs(h["F"].sum(axis=0)).max() < 1e-9 * s                  # +f and -f of every pair are the same number
    # a dropped pair, a pair taken twice or a wrong sign changes these:
    half = oracle.forces_half(w.pos, w.box, w.potential, pairs[::2], quat=w.quat)
    assert np.abs(half["F"] - b["F"]).max() > 1e-3 * s


def test_o10_fcc_lattice_sum(oracle):
    rc, n_rc, n_rv, u_ref = [r for r in read_table("fcc_lattice_sums.txt") if r[0] == 2.5][0]
    w = W.lj_fluid(4 * 8 ** 3, rc, jitter=0.0)
    pairs = oracle.pair_set(w.pos, w.box, rc, 0.3)
    h = oracle.forces_half(w.pos, w.box, w.potential, pairs)
    assert abs(h["pe"].sum() / w.N - u_ref) < 2e-6                       # fp32-rounded lattice against the closed form
    assert 2 * h["n_in_cut"] == w.N * int(n_rc)
    assert np.abs(h["F"]).max() < 1e-4


# ------------------------------------------------------------------ P7: Newton's third law
@pytest.mark.parametrize("gen", ["lj", "poly", "patchy"])
def test_p7_newton3_invariants(oracle, gen):
    if gen == "lj":
        w = W.lj_fluid(2048, 2.5)
    elif gen == "poly":
        w = W.polymer_melt(32, 64, relax_iters=20)
    else:
        w = W.patchy_fluid(2048, rho=0.9, jitter=0.1)
    f = oracle.forces(w.pos, w.box, w.potential, w.quat)
    rms = math.sqrt((f["F"] ** 2).mean())
    assert np.abs(f["F"].sum(0)).max() < 1e-12 * w.N * rms
    if w.quat is not None:
        # sum_i tau_i + sum_pairs r_vec x F_j = 0 with pair-wise minimum-image r_vec (S:P7)
        x = w.pos[:, :3].astype(np.float64)
        q = w.quat.astype(np.float64)
        pairs = oracle.pair_set(w.pos, w.box, w.rcut, 0.0)
        acc = f["T"].sum(0)
        for i, j in pairs:
            d = x[j] - x[i]
            d = np.where(d > 0.5 * w.box, d - w.box, np.where(d < -0.5 * w.box, d + w.box, d))
            _, _, Fj, _, _ = oracle.pair(w.potential, d, q[i], q[j])
            acc = acc + np.cross(d, Fj)
        assert np.abs(acc).max() < 1e-9 * max(1.0, np.abs(f["T"]).sum())


# ------------------------------------------------------------------ P12: the paper's only numeric example (Fig. 1)
def test_p12_fig1_thread_counts(oracle):
    g = read_kv("fig1_thread_counts.txt")
    pos = np.array([[5, 5, 5], [5.9, 5, 5], [5, 5.9, 5], [5, 5, 5.9], [5.5, 5.5, 5.5]], dtype=np.float32)
    box = np.array([20.0, 20.0, 20.0])
    pairs = oracle.pair_set(pos, box, 2.5, 0.3)
    deg = np.bincount(pairs.ravel(), minlength=5)
    assert len(pos) == g["vertex_threads"]            # one thread per particle
    assert len(pairs) == g["edge_threads"]            # one thread per potentially interacting pair = C(5,2)
    assert deg.sum() // 2 == g["edge_threads"]        # "sum of the number of neighbours ... divided by two" P:63


# ------------------------------------------------------------------ P9: NVE drift, P10: free rotor
def test_p9_nve_drift_lj(oracle):
    w = W.config("C1")
    out = oracle.integrate(w.pos, w.vel, w.box, w.potential, w.skin, w.dt, 2000, every=20)
    e0 = out["e0"].sum()
    e = out["energies"].sum(1)
    assert np.abs(e - e0).max() / abs(e0) < 5e-5        # stated bound (S:P9), measured 3.6e-6 over 1e4 steps
    assert abs(e0 / w.N - (-4.38)) < 0.05               # E0/N ~ -4.38 (S:X3; seed-dependent at the 1e-2 level)
    assert 60 <= out["rebuilds"] <= 110                 # one rebuild every ~25 steps (S:X3: 19..29)
    p = out["vel"].sum(0) - w.vel[:, :3].astype(np.float64).sum(0)
    assert np.abs(p).max() < 1e-9                       # momentum conserved


def test_p9_nve_drift_patchy(oracle):
    w = W.patchy_fluid(256, jitter=0.05)
    out = oracle.integrate(w.pos, w.vel, w.box, w.potential, w.skin, w.dt, 2000, every=20, quat=w.quat, angmom=w.angmom)
    e0 = out["e0"].sum()
    e = out["energies"].sum(1)
    assert np.abs(e - e0).max() / w.N < 5e-4            # |dE|/N bound in eps (S:P9)
    assert np.abs(np.linalg.norm(out["quat"], axis=1) - 1).max() < 1e-12


def test_p9_nve_drift_polymer(oracle):
    w = W.polymer_melt(32, 64)
    out = oracle.integrate(w.pos, w.vel, w.box, w.potential, w.skin, w.dt, 1000, every=10)
    assert out["bad"] == 0
    e0 = out["e0"].sum()
    e = out["energies"].sum(1)
    assert np.abs(e - e0).max() / abs(e0) < 1e-3        # stated bound (S:P9)


def test_p10_free_rotor(oracle):
    w = W.dimer_gas(64, "patchy", spacing=6.0)
    x = w.pos.copy()
    x[1::2, :3] = x[0::2, :3] + np.float32(3.0)          # partners 5.2 sigma apart: no interaction at all
    rng = np.random.default_rng(2)
    L = np.zeros((w.N, 4), dtype=np.float32)
    L[:, :3] = rng.normal(size=(w.N, 3)) * 0.3
    dt, n = 0.002, 500
    out = oracle.integrate(x, w.vel, w.box, w.potential, w.skin, dt, n, quat=w.quat, angmom=L)
    assert np.array_equal(out["angmom"], L[:, :3].astype(np.float64))         # L constant
    assert np.abs(np.linalg.norm(out["quat"], axis=1) - 1).max() < 1e-12
    I = w.potential["inertia"]
    q0 = w.quat.astype(np.float64)
    q0 /= np.linalg.norm(q0, axis=1, keepdims=True)
    for i in range(0, w.N, 7):
        om = L[i, :3].astype(np.float64) / I
        ang = np.linalg.norm(om) * dt * n                                     # total rotation angle = |L| dt n / I
        dq = np.array([math.cos(ang / 2), *(math.sin(ang / 2) * om / np.linalg.norm(om))])
        want = qmul(dq, q0[i])
        got = out["quat"][i]
        assert min(np.abs(got - want).max(), np.abs(got + want).max()) < 1e-9


# ------------------------------------------------------------------ O8: the paper's own patchy model (S:8(f2), reading Q1)
PP = W.patchy_pp_potential()


def test_o8_patchy_pp_closed_forms(oracle):
    """Eqs. (3)-(4) P:103-113 for two particles on the x axis whose patches 0 face each other: the patch-patch distance
    is r - 1, so V = r^-200 - exp[-1/2 ((r - 1)/0.12)^10] and the force is its radial derivative; with the patch axes
    perpendicular to the bond every patch pair is beyond 0.18 sigma and only the core of Eq. (3) is left."""
    qi = quat_from_to([0, 0, 1], [1, 0, 0])
    qj = quat_from_to([0, 0, 1], [-1, 0, 0])
    for r in (1.0, 1.03, 1.12, 1.17):
        u = r - 1.0
        g = 0.5 * (u / 0.12) ** 10
        V_ref = r ** -200.0 - math.exp(-g)
        dVdr = -200.0 * r ** -201.0 + (math.exp(-g) * 10.0 * g / u if u > 0 else 0.0)
        inside, V, Fj, ti, tj = oracle.pair(PP, [r, 0, 0], qi, qj)
        assert inside
        assert abs(V - V_ref) < 1e-12 * max(1.0, abs(V_ref))
        assert abs(Fj[0] + dVdr) < 1e-9 * max(1.0, abs(dVdr)) and abs(Fj[1]) < 1e-12 and abs(Fj[2]) < 1e-12
        assert np.abs(ti).max() < 1e-12 and np.abs(tj).max() < 1e-12          # central geometry: no torque
    assert abs((1.12 ** -200.0 - math.exp(-0.5)) - oracle.pair(PP, [1.12, 0, 0], qi, qj)[1]) < 1e-12   # u = w: g = 1/2
    for r in (0.99, 1.05):
        inside, V, Fj, ti, tj = oracle.pair(PP, [r, 0, 0], ID, ID)            # patch axes along z, bond along x
        assert abs(V - r ** -200.0) < 1e-12 * r ** -200.0 and abs(Fj[0] - 200.0 * r ** -201.0) < 1e-9 * r ** -201.0 * 200
        assert np.abs(ti).max() == 0.0 and np.abs(tj).max() == 0.0
    assert not oracle.pair(PP, [1.18, 0, 0], qi, qj)[0]                       # strict centre cutoff 2 * 0.5 + 0.18
    # a patch pair just outside 0.18 sigma contributes nothing (truncated): tilt i's patch away
    tilt = quat_from_to([0, 0, 1], [math.cos(0.5), math.sin(0.5), 0.0])
    _, V, _, _, _ = oracle.pair(PP, [1.1, 0, 0], tilt, qj)
    pa = 0.5 * np.array([math.cos(0.5), math.sin(0.5), 0.0])
    d = np.array([1.1, 0, 0]) + np.array([-0.5, 0, 0]) - pa
    assert np.linalg.norm(d) > 0.18 and abs(V - 1.1 ** -200.0) < 1e-15


def test_o8_patchy_pp_finite_differences(oracle):
    """Force and both torques of O8 against central differences of its energy on bonded, tilted geometries, and the pair
    invariant tau_i + tau_j + r_vec x F_j = 0 (a wrong sign, a swapped patch or a dropped term fails one of them)."""
    rng = np.random.default_rng(8)
    worst, bonded = 0.0, 0
    for _ in range(200):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        r = rng.uniform(1.0, 1.15)
        def facing(target, patch):
            t = target + 0.12 * rng.normal(size=3)
            t /= np.linalg.norm(t)
            return quat_from_to(W.PP_DIRS[patch], t)
        qi, qj = facing(d, rng.integers(2)), facing(-d, rng.integers(2))
        _, V, Fj, ti, tj = oracle.pair(PP, r * d, qi, qj)
        bonded += V < r ** -200.0 - 1e-3
        Fd, tid, tjd = _fd_pair(oracle, PP, r * d, qi, qj, h=1e-7)
        scale = max(1.0, np.abs(Fj).max(), np.abs(ti).max(), np.abs(tj).max())
        worst = max(worst, np.abs(Fj - Fd).max() / scale, np.abs(ti - tid).max() / scale, np.abs(tj - tjd).max() / scale)
        assert np.abs(ti + tj + np.cross(r * d, Fj)).max() < 1e-10 * scale
    assert bonded > 60            # the sample does exercise the patch term
    assert worst < 5e-6


def test_o8_patchy_pp_system(oracle):
    """Whole periodic system of bonded dimers: cells vs brute force, zero net force, F_i = -dU/dx_i, tau_i = -dU/d(rot_i)."""
    w = W.dimer_gas(108, "patchy_pp")
    f = oracle.forces(w.pos, w.box, w.potential, w.quat)
    fb = oracle.forces(w.pos, w.box, w.potential, w.quat, use_cells=False)
    assert np.array_equal(f["F"], fb["F"]) or np.abs(f["F"] - fb["F"]).max() < 1e-10 * np.abs(f["F"]).max()
    assert f["n_in_cut"] == fb["n_in_cut"] and (f["pe"] < -0.05).sum() > 40
    assert np.abs(f["F"].sum(0)).max() < 1e-10 * np.abs(f["F"]).max()
    x = w.pos[:, :3].astype(np.float64)
    q = w.quat.astype(np.float64)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    fd = oracle.forces_d(x, w.box, w.potential, q)
    h = 1e-7
    bonded = np.nonzero(fd["pe"] < -0.05)[0]
    for i in bonded[:4]:
        for k in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, k] += h
            xm[i, k] -= h
            g = -(_total_U(oracle, xp, w.box, w.potential, q) - _total_U(oracle, xm, w.box, w.potential, q)) / (2 * h)
            assert abs(g - fd["F"][i, k]) < 5e-6 * max(1.0, np.abs(fd["F"]).max())
            ax = np.zeros(3)
            ax[k] = 1
            qp, qm = q.copy(), q.copy()
            qp[i] = qmul(np.array([math.cos(h / 2), *(math.sin(h / 2) * ax)]), q[i])
            qm[i] = qmul(np.array([math.cos(h / 2), *(-math.sin(h / 2) * ax)]), q[i])
            t = -(_total_U(oracle, x, w.box, w.potential, qp) - _total_U(oracle, x, w.box, w.potential, qm)) / (2 * h)
            assert abs(t - fd["T"][i, k]) < 5e-6 * max(1.0, np.abs(fd["T"]).max())


# ------------------------------------------------------------------ O9: thermostat (reading QT of P:53)
def test_o9_philox_known_answers(oracle):
    from conftest import GOLDEN
    rows = [ln.split() for ln in (GOLDEN / "philox4x32_10_kat.txt").read_text().splitlines()
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        assert [int(x) for x in oracle.philox(v[0:4], v[4:6])] == v[6:10]


def test_o9_p0_is_identity_p1_refreshes_everything(oracle):
    rng = np.random.default_rng(5)
    v = rng.normal(size=(1000, 3))
    L = rng.normal(size=(1000, 3))
    v0, L0, nt, nr = oracle.thermostat(v, PATCHY, 0.15, 0.0, 7, 1, angmom_d=L, p_r=0.0)
    assert nt == 0 and nr == 0 and np.array_equal(v0, v) and np.array_equal(L0, L)
    v1, L1, nt, nr = oracle.thermostat(v, PATCHY, 0.15, 1.0, 7, 1, angmom_d=L, p_r=1.0)
    assert nt == 1000 and nr == 1000
    assert not np.any(v1 == v) and not np.any(L1 == L)
    # the draw does not depend on the state it replaces, only on (id, call, seed)
    v2, L2, _, _ = oracle.thermostat(np.zeros_like(v), PATCHY, 0.15, 1.0, 7, 1, angmom_d=np.zeros_like(L), p_r=1.0)
    assert np.array_equal(v1, v2) and np.array_equal(L1, L2)
    v3, _, _, _ = oracle.thermostat(v, PATCHY, 0.15, 1.0, 7, 2, angmom_d=L, p_r=1.0)
    v4, _, _, _ = oracle.thermostat(v, PATCHY, 0.15, 1.0, 8, 1, angmom_d=L, p_r=1.0)
    assert not np.any(v3 == v1) and not np.any(v4 == v1)


def test_o9_maxwell_boltzmann_moments_and_ks(oracle):
    from scipy import stats
    N, T, mass, inertia = 200000, 1.7, 2.0, 0.1
    pot = dict(PATCHY, mass=mass, inertia=inertia)
    v, L, nt, nr = oracle.thermostat(np.zeros((N, 3)), pot, T, 1.0, 2024, 3, angmom_d=np.zeros((N, 3)), p_r=1.0)
    for a, var in ((v, T / mass), (L, T * inertia)):
        for k in range(3):
            x = a[:, k]
            assert abs(x.mean()) < 5.0 * math.sqrt(var / N)                 # 5 sigma of the sample mean
            assert abs(x.var() / var - 1.0) < 5.0 * math.sqrt(2.0 / N)      # 5 sigma of the sample variance
            assert abs(stats.kurtosis(x)) < 5.0 * math.sqrt(24.0 / N)
            assert stats.kstest(x / math.sqrt(var), "norm").pvalue > 1e-4
        c = np.corrcoef(a.T)
        assert np.abs(c - np.eye(3)).max() < 5.0 / math.sqrt(N)            # components independent
    assert np.abs(np.corrcoef(v[:, 0], L[:, 0])[0, 1]) < 5.0 / math.sqrt(N)  # streams independent
    # equipartition: 1/2 m <v^2> = 3/2 T, <L^2>/(2 I) = 3/2 T
    assert abs(0.5 * mass * (v * v).sum() / N / (1.5 * T) - 1.0) < 0.01
    assert abs((L * L).sum() / (2.0 * inertia) / N / (1.5 * T) - 1.0) < 0.01


def test_o9_refreshed_fraction_is_binomial(oracle):
    N = 200000
    for p in (0.02, 0.3, 0.75):
        v, _, nt, _ = oracle.thermostat(np.zeros((N, 3)), LJ25, 1.0, p, 99, 1)
        assert abs(nt - p * N) < 5.0 * math.sqrt(N * p * (1.0 - p))
        assert nt == int(np.count_nonzero(np.any(v != 0.0, axis=1)))


def test_o9_lj_fluid_relaxes_to_the_target_temperature(oracle):
    """A hot LJ fluid (T = 2) under the thermostat at T = 1 ends at kinetic temperature 1 (NVT)."""
    w = W.lj_fluid(500, T=2.0)
    out = oracle.integrate_nvt(w.pos, w.vel, w.box, w.potential, w.skin, w.dt, 1200, T=1.0, n_newt=10, p_t=0.2, seed=11)
    temps = out["temps"]
    assert temps[0] > 1.3
    assert abs(temps[-40:].mean() - 1.0) < 0.06
    assert out["bad"] == 0
