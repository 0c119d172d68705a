"""ctypes binding of oracle/md_oracle.c (fp64 CPU oracle; test infrastructure only).

`build()` compiles the C file with gcc (-O2 -ffp-contract=off -fopenmp) into oracle/libmd_oracle.so.
Nothing here touches CUDA or the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "md_oracle.c"
_LIB = _HERE / "libmd_oracle.so"

KINDS = {"lj": 0, "fene_wca": 1, "patchy": 2, "patchy_pp": 3}


class OrcPot(C.Structure):
    _fields_ = [
        ("kind", C.c_int),
        ("epsilon", C.c_double), ("sigma", C.c_double), ("mass", C.c_double),
        ("rcut", C.c_double),
        ("shift_energy", C.c_int),
        ("fene_K", C.c_double), ("fene_R0", C.c_double),
        ("chain_len", C.c_int),
        ("n_patches", C.c_int),
        ("patch_dir", (C.c_double * 3) * 8),
        ("eps_patch", C.c_double), ("patch_sigma_r", C.c_double), ("patch_sigma_ang", C.c_double),
        ("rcut_core", C.c_double),
        ("inertia", C.c_double),
        ("patch_radius", C.c_double), ("patch_exponent", C.c_double), ("core_exponent", C.c_double),
        ("rcut_patch", C.c_double),
    ]


def make_pot(d: dict) -> OrcPot:
    p = OrcPot()
    p.kind = KINDS[d["kind"]]
    p.epsilon = d.get("epsilon", 1.0)
    p.sigma = d.get("sigma", 1.0)
    p.mass = d.get("mass", 1.0)
    p.rcut = d["rcut"]
    p.shift_energy = int(d.get("shift_energy", 1))
    p.fene_K = d.get("fene_K", 30.0)
    p.fene_R0 = d.get("fene_R0", 1.5)
    p.chain_len = int(d.get("chain_len", 1))
    dirs = np.asarray(d.get("patch_dir", np.zeros((0, 3))), dtype=np.float64)
    p.n_patches = int(d.get("n_patches", dirs.shape[0]))
    for a in range(min(8, dirs.shape[0])):
        for k in range(3):
            p.patch_dir[a][k] = float(dirs[a, k])
    p.eps_patch = d.get("eps_patch", 0.0)
    p.patch_sigma_r = d.get("patch_sigma_r", 0.1)
    p.patch_sigma_ang = d.get("patch_sigma_ang", 0.3)
    p.rcut_core = d.get("rcut_core", 2.0 ** (1.0 / 6.0))
    p.inertia = d.get("inertia", 0.1)
    p.patch_radius = d.get("patch_radius", 0.5)
    p.patch_exponent = d.get("patch_exponent", 10.0)
    p.core_exponent = d.get("core_exponent", 200.0)
    p.rcut_patch = d.get("rcut_patch", 0.18)
    return p


def build(force: bool = False) -> Path:
    """Compile the oracle (gcc). Building the checker is not using it."""
    if force or (not _LIB.exists()) or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99",
               str(_SRC), "-o", str(_LIB), "-lm"]
        subprocess.check_call(cmd)
    return _LIB


_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def _d(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _f(a):
    return a.ctypes.data_as(_fp) if a is not None else None


class Oracle:
    """Thin numpy front-end. Positions are float32 [N,>=3] (only x,y,z are read), quats float32 [N,4]."""

    def __init__(self):
        self.lib = C.CDLL(str(build()))
        L = self.lib
        L.orc_num_threads.restype = C.c_int
        L.orc_pair_set.restype = C.c_int64
        L.orc_pair_set.argtypes = [C.c_int64, _fp, _dp, C.c_double, C.c_double, C.c_int, _ip, C.c_int64]
        L.orc_forces.restype = C.c_int
        L.orc_forces.argtypes = [C.c_int64, _fp, _fp, _dp, C.POINTER(OrcPot), C.c_int, _dp, _dp, _dp, _lp]
        L.orc_forces_half.restype = C.c_int
        L.orc_forces_half.argtypes = [C.c_int64, _fp, _fp, _dp, C.POINTER(OrcPot), _ip, C.c_int64, _dp, _dp, _dp, _lp]
        L.orc_forces_d.restype = C.c_int
        L.orc_forces_d.argtypes = [C.c_int64, _dp, _dp, _dp, C.POINTER(OrcPot), C.c_int, _dp, _dp, _dp, _lp]
        L.orc_pair.restype = C.c_int
        L.orc_pair.argtypes = [C.POINTER(OrcPot), _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_bond.restype = C.c_int
        L.orc_bond.argtypes = [C.POINTER(OrcPot), _dp, _dp, _dp]
        L.orc_energy_d.restype = None
        L.orc_energy_d.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, C.c_double, _dp, _dp, _dp]
        L.orc_integrate_d.restype = C.c_int
        L.orc_integrate_d.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, _dp, C.POINTER(OrcPot), C.c_double, C.c_double,
                                      C.c_int64, C.c_int64, _dp, _dp, _dp, _dp, _lp]
        L.orc_set_threads.argtypes = [C.c_int]
        _up = C.POINTER(C.c_uint32)
        L.orc_philox4x32_10.restype = None
        L.orc_philox4x32_10.argtypes = [_up, _up, _up]
        L.orc_thermostat_d.restype = C.c_int64
        L.orc_thermostat_d.argtypes = [C.c_int64, _dp, _dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                       C.c_uint64, C.c_uint32, _lp]

    @property
    def threads(self) -> int:
        return int(self.lib.orc_num_threads())

    def set_threads(self, n: int):
        self.lib.orc_set_threads(int(n))

    @staticmethod
    def _pos3(pos) -> np.ndarray:
        return np.ascontiguousarray(np.asarray(pos, dtype=np.float32)[:, :3])

    def pair_set(self, pos, box, rcut, skin, use_cells=True, cap=None) -> np.ndarray:
        """O0: sorted (i<j) pairs with d2 < (rcut+skin)^2, int32 [E,2]."""
        p3 = self._pos3(pos)
        N = p3.shape[0]
        box = np.ascontiguousarray(box, dtype=np.float64)
        if cap is None:
            cap = self.lib.orc_pair_set(N, _f(p3), _d(box), rcut, skin, int(use_cells), None, 0)
        out = np.empty((max(int(cap), 1), 2), dtype=np.int32)
        n = self.lib.orc_pair_set(N, _f(p3), _d(box), rcut, skin, int(use_cells), out.ctypes.data_as(_ip), int(cap))
        return out[:min(n, cap)]

    def pair_count(self, pos, box, rcut, skin, use_cells=True) -> int:
        """O0: number of pairs only (E = 1/2 sum |L_i|)."""
        p3 = self._pos3(pos)
        box = np.ascontiguousarray(box, dtype=np.float64)
        return int(self.lib.orc_pair_set(p3.shape[0], _f(p3), _d(box), rcut, skin, int(use_cells), None, 0))

    def forces(self, pos, box, pot, quat=None, use_cells=True):
        """O1-O5: returns dict(F [N,3], T [N,3] or None, pe [N], n_in_cut, bad) in fp64."""
        p3 = self._pos3(pos)
        N = p3.shape[0]
        box = np.ascontiguousarray(box, dtype=np.float64)
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        q4 = np.ascontiguousarray(quat, dtype=np.float32) if quat is not None else None
        F = np.zeros((N, 3))
        T = np.zeros((N, 3)) if quat is not None else None
        pe = np.zeros(N)
        nin = C.c_int64(0)
        bad = self.lib.orc_forces(N, _f(p3), _f(q4), _d(box), C.byref(op), int(use_cells), _d(F), _d(T), _d(pe),
                                  C.byref(nin))
        return dict(F=F, T=T, pe=pe, n_in_cut=int(nin.value), bad=int(bad))

    def forces_half(self, pos, box, pot, pairs, quat=None):
        """O10: the same sums by ONE thread over the half Verlet list `pairs` (int32 [E,2], i<j) with Newton's third
        law (S:8(d) single-core baseline).  Same return dict as forces()."""
        p3 = self._pos3(pos)
        N = p3.shape[0]
        box = np.ascontiguousarray(box, dtype=np.float64)
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        q4 = np.ascontiguousarray(quat, dtype=np.float32) if quat is not None else None
        pr = np.ascontiguousarray(pairs, dtype=np.int32)
        F = np.zeros((N, 3))
        T = np.zeros((N, 3)) if quat is not None else None
        pe = np.zeros(N)
        nin = C.c_int64(0)
        bad = self.lib.orc_forces_half(N, _f(p3), _f(q4), _d(box), C.byref(op), pr.ctypes.data_as(_ip), pr.shape[0],
                                       _d(F), _d(T), _d(pe), C.byref(nin))
        return dict(F=F, T=T, pe=pe, n_in_cut=int(nin.value), bad=int(bad))

    def forces_d(self, pos_d, box, pot, quat_d=None, use_cells=True):
        """Same on fp64 state (used by the finite-difference pins and the integrator tests)."""
        p3 = np.ascontiguousarray(pos_d, dtype=np.float64)
        N = p3.shape[0]
        box = np.ascontiguousarray(box, dtype=np.float64)
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        q4 = np.ascontiguousarray(quat_d, dtype=np.float64) if quat_d is not None else None
        F = np.zeros((N, 3))
        T = np.zeros((N, 3)) if quat_d is not None else None
        pe = np.zeros(N)
        nin = C.c_int64(0)
        bad = self.lib.orc_forces_d(N, _d(p3), _d(q4), _d(box), C.byref(op), int(use_cells), _d(F), _d(T), _d(pe),
                                    C.byref(nin))
        return dict(F=F, T=T, pe=pe, n_in_cut=int(nin.value), bad=int(bad))

    def pair(self, pot, rvec, qi=(1, 0, 0, 0), qj=(1, 0, 0, 0)):
        """One isolated pair: returns (inside, V, F_j, tau_i, tau_j)."""
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        rv = np.ascontiguousarray(rvec, dtype=np.float64)
        a = np.ascontiguousarray(qi, dtype=np.float64)
        b = np.ascontiguousarray(qj, dtype=np.float64)
        V = C.c_double(0)
        Fj, ti, tj = np.zeros(3), np.zeros(3), np.zeros(3)
        inside = self.lib.orc_pair(C.byref(op), _d(rv), _d(a), _d(b), C.byref(V), _d(Fj), _d(ti), _d(tj))
        return int(inside), V.value, Fj, ti, tj

    def bond(self, pot, rvec):
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        rv = np.ascontiguousarray(rvec, dtype=np.float64)
        V = C.c_double(0)
        Fj = np.zeros(3)
        bad = self.lib.orc_bond(C.byref(op), _d(rv), C.byref(V), _d(Fj))
        return int(bad), V.value, Fj

    def energy(self, pe, vel_d, pot, angmom_d=None):
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        v = np.ascontiguousarray(vel_d, dtype=np.float64)
        L = np.ascontiguousarray(angmom_d, dtype=np.float64) if angmom_d is not None else None
        U, Kt, Kr = C.c_double(0), C.c_double(0), C.c_double(0)
        self.lib.orc_energy_d(v.shape[0], _d(np.ascontiguousarray(pe, dtype=np.float64)), _d(v), _d(L),
                              op.mass, op.inertia, C.byref(U), C.byref(Kt), C.byref(Kr))
        return U.value, Kt.value, Kr.value

    def integrate(self, pos, vel, box, pot, skin, dt, nsteps, every=0, quat=None, angmom=None):
        """O6/O7 on fp64 copies of the fp32 inputs. Returns dict with final state, energies [k,3], rebuilds."""
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        x = np.ascontiguousarray(np.asarray(pos)[:, :3], dtype=np.float64).copy()
        v = np.ascontiguousarray(np.asarray(vel)[:, :3], dtype=np.float64).copy()
        N = x.shape[0]
        box = np.ascontiguousarray(box, dtype=np.float64)
        q = np.ascontiguousarray(quat, dtype=np.float64).copy() if quat is not None else None
        L = np.ascontiguousarray(np.asarray(angmom)[:, :3], dtype=np.float64).copy() if angmom is not None else None
        f0 = self.forces_d(x, box, op, q)
        F, pe = f0["F"], f0["pe"]
        T = f0["T"] if q is not None else None
        e0 = self.energy(pe, v, op, L)
        nrec = nsteps // every if every > 0 else 0
        en = np.zeros((max(nrec, 1), 3))
        nreb = C.c_int64(0)
        bad = self.lib.orc_integrate_d(N, _d(x), _d(v), _d(q), _d(L), _d(box), C.byref(op), skin, dt, nsteps, every,
                                       _d(F), _d(T), _d(pe), _d(en), C.byref(nreb))
        return dict(pos=x, vel=v, quat=q, angmom=L, F=F, T=T, pe=pe, e0=np.array(e0), energies=en[:nrec],
                    rebuilds=int(nreb.value), bad=int(bad | f0["bad"]))

    # ---- O9: thermostat (reading DESIGN.md QT of P:53; parity unpinned w.r.t. the paper's Ref. 27)
    def philox(self, ctr, key):
        """Philox4x32-10 block: ctr 4 x uint32, key 2 x uint32 -> 4 x uint32."""
        c = np.ascontiguousarray(ctr, dtype=np.uint32)
        k = np.ascontiguousarray(key, dtype=np.uint32)
        out = np.zeros(4, dtype=np.uint32)
        up = C.POINTER(C.c_uint32)
        self.lib.orc_philox4x32_10(c.ctypes.data_as(up), k.ctypes.data_as(up), out.ctypes.data_as(up))
        return out

    def thermostat(self, vel_d, pot, T, p_t, seed, call, angmom_d=None, p_r=0.0):
        """One application on fp64 copies (id order). Returns (vel, angmom, n_refreshed_trans, n_refreshed_rot)."""
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        v = np.ascontiguousarray(np.asarray(vel_d)[:, :3], dtype=np.float64).copy()
        L = np.ascontiguousarray(np.asarray(angmom_d)[:, :3], dtype=np.float64).copy() if angmom_d is not None else None
        nr = C.c_int64(0)
        nt = self.lib.orc_thermostat_d(v.shape[0], _d(v), _d(L), op.mass, op.inertia, float(T), float(p_t), float(p_r),
                                       int(seed), int(call), C.byref(nr))
        return v, L, int(nt), int(nr.value)

    def integrate_nvt(self, pos, vel, box, pot, skin, dt, nsteps, T, n_newt, p_t, seed, quat=None, angmom=None,
                      p_r=0.0, every=0):
        """O6/O7 with O9 applied after every n_newt-th step (call index = steps done / n_newt, counted from this
        call). Returns the dict of integrate() plus 'temps': kinetic temperature 2 K_t / (3 N) after each chunk."""
        op = pot if isinstance(pot, OrcPot) else make_pot(pot)
        x, v, q, L = pos, vel, quat, angmom
        done, temps, reb, out = 0, [], 0, None
        while done < nsteps:
            chunk = min(n_newt - done % n_newt, nsteps - done)
            out = self.integrate(x, v, box, op, skin, dt, chunk, quat=q, angmom=L)
            x, v, q, L = out["pos"], out["vel"], out["quat"], out["angmom"]
            reb += out["rebuilds"]
            done += chunk
            if done % n_newt == 0:
                v, L, _, _ = self.thermostat(v, op, T, p_t, seed, done // n_newt, angmom_d=L, p_r=p_r)
            temps.append(op.mass * float((v * v).sum()) / (3.0 * v.shape[0]))
        out = dict(out)
        out.update(vel=v, angmom=L, rebuilds=reb, temps=np.array(temps))
        return out


if __name__ == "__main__":
    print(build(force=True))
