"""Seeded synthetic input generators (BASELINE.json configs C1-C5).

This module serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_1401_4350_b200/``).  It holds none of the method's arithmetic: no pair
potential, no force, no neighbour predicate, no integrator.  It only draws numbers
from a counter-based generator and lays out particles (lattices, random walks,
a purely geometric overlap push-off for the polymer start).

All draws are made in fp64 from splitmix64 keyed on (seed, stream, index) and
rounded ONCE to fp32.  Box lengths are rounded to the nearest
fp32 value so that the GPU (float) and the oracle (double) see the same L (Q7).

State layout handed to both sides: float32 arrays of shape [N, 4]
  pos   = (x, y, z, 0)         vel    = (vx, vy, vz, 0)
  quat  = (w, x, y, z)         angmom = (Lx, Ly, Lz, 0)      (rigid bodies only)
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

BASE_SEED = 14014350  # seed_k = BASE_SEED + k for config k

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output step applied element-wise to uint64 counters."""
    with np.errstate(over="ignore"):
        z = (np.asarray(x, dtype=_U64) + _GOLD).astype(_U64)
        z = ((z ^ (z >> _U64(30))) * _M1).astype(_U64)
        z = ((z ^ (z >> _U64(27))) * _M2).astype(_U64)
        return z ^ (z >> _U64(31))


def uniform01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """n fp64 uniforms in [0,1): value k depends only on (seed, stream, offset+k)."""
    with np.errstate(over="ignore"):
        key = splitmix64(np.array([(seed * 0x100000001B3 + stream) & 0xFFFFFFFFFFFFFFFF], dtype=_U64))[0]
        idx = np.arange(offset, offset + n, dtype=_U64)
        bits = splitmix64(key + idx * _GOLD)
    return (bits >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, n: int) -> np.ndarray:
    """n fp64 standard normals (Box-Muller on two counter streams)."""
    u1 = uniform01(seed, stream, n)
    u2 = uniform01(seed, stream + 0x5bd1e995, n)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


def _f32_box(box) -> np.ndarray:
    return np.asarray(np.asarray(box, dtype=np.float32), dtype=np.float64)


def _wrap_to_f32(x: np.ndarray, box: np.ndarray) -> np.ndarray:
    """Wrap fp64 coordinates into [0, L) and round once to fp32 (exactly L -> 0, Q7)."""
    x = x - box * np.floor(x / box)
    xf = x.astype(np.float32)
    bf = box.astype(np.float32)
    xf = np.where(xf >= bf, np.float32(0.0), xf)
    xf = np.where(xf < 0, np.float32(0.0), xf)
    return xf


def _pad4(a3: np.ndarray) -> np.ndarray:
    out = np.zeros((a3.shape[0], 4), dtype=np.float32)
    out[:, :3] = a3
    return out


@dataclass
class Workload:
    """One synthetic input. Arrays are float32 [N,4]; `box` holds fp32-representable doubles."""
    name: str
    N: int
    box: np.ndarray
    pos: np.ndarray
    vel: np.ndarray
    rcut: float
    skin: float
    potential: dict
    dt: float
    quat: Optional[np.ndarray] = None
    angmom: Optional[np.ndarray] = None
    max_neigh: int = 0
    meta: dict = field(default_factory=dict)


# --------------------------------------------------------------------------------------
# fcc lattices (Q12: orthorhombic boxes of nx*ny*nz cubic cells, powers of two)
# --------------------------------------------------------------------------------------
FCC_SHAPES = {
    2 ** 8: (4, 4, 4), 2 ** 9: (4, 4, 8), 2 ** 10: (4, 8, 8),
    2 ** 11: (8, 8, 8), 2 ** 12: (8, 8, 16), 2 ** 13: (8, 16, 16), 2 ** 14: (16, 16, 16),
    2 ** 15: (16, 16, 32), 2 ** 16: (16, 32, 32), 2 ** 17: (32, 32, 32), 2 ** 18: (32, 32, 64),
    2 ** 19: (32, 64, 64), 2 ** 20: (64, 64, 64), 2 ** 21: (64, 64, 128), 2 ** 22: (64, 128, 128),
}


def fcc_shape(N: int):
    if N in FCC_SHAPES:
        return FCC_SHAPES[N]
    n = round((N / 4) ** (1.0 / 3.0))
    if 4 * n ** 3 == N:
        return (n, n, n)
    raise ValueError(f"no fcc shape for N={N}")


def fcc_sites(shape, a: float) -> np.ndarray:
    """fp64 site coordinates; order: cell (ix*ny+iy)*nz+iz, then basis (Q13)."""
    nx, ny, nz = shape
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], dtype=np.float64)
    return ((cells[:, None, :] + basis[None, :, :]) * a).reshape(-1, 3)


def neighbour_capacity(rho: float, rv: float) -> int:
    """max_neigh = ceil(1.35*rho*(4/3)*pi*rv^3) + 16, rounded up to a multiple of 8."""
    m = int(math.ceil(1.35 * rho * (4.0 / 3.0) * math.pi * rv ** 3)) + 16
    return (m + 7) // 8 * 8


def _velocities(seed: int, stream: int, N: int, T: float) -> np.ndarray:
    v = normal(seed, stream, 3 * N).reshape(N, 3) * math.sqrt(T)
    v -= v.mean(axis=0, keepdims=True)  # zero net momentum, no rescale (Q13)
    return v


def lj_potential(rcut: float) -> dict:
    return dict(kind="lj", epsilon=1.0, sigma=1.0, mass=1.0, shift_energy=1, rcut=rcut)


def lj_fluid(N: int, rcut: float = 2.5, skin: float = 0.3, rho: float = 0.8, T: float = 1.0,
             jitter: float = 0.05, seed: int = BASE_SEED + 1, dt: float = 0.002) -> Workload:
    """C1 / C2 / C5-LJ: fcc lattice + uniform jitter, Gaussian velocities (D1, D2a, D2b, D5)."""
    shape = fcc_shape(N)
    a = (4.0 / rho) ** (1.0 / 3.0)
    box = _f32_box([shape[0] * a, shape[1] * a, shape[2] * a])
    x = fcc_sites(shape, a)
    if jitter > 0:
        x = x + (uniform01(seed, 1, 3 * N).reshape(N, 3) * 2.0 - 1.0) * jitter
    pos = _pad4(_wrap_to_f32(x, box))
    vel = _pad4(_velocities(seed, 2, N, T).astype(np.float32))
    return Workload(name=f"lj_N{N}_rc{rcut}", N=N, box=box, pos=pos, vel=vel, rcut=rcut, skin=skin,
                    potential=lj_potential(rcut), dt=dt,
                    max_neigh=neighbour_capacity(rho, rcut + skin),
                    meta=dict(rho=rho, T=T, jitter=jitter, seed=seed, fcc_shape=shape, a=a))


# --------------------------------------------------------------------------------------
# C4 / D4: patchy rigid bodies
# --------------------------------------------------------------------------------------
TETRA = (np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64) / math.sqrt(3.0))


def patchy_potential() -> dict:
    return dict(kind="patchy", epsilon=1.0, sigma=1.0, mass=1.0, shift_energy=0, rcut=1.5,
                rcut_core=2.0 ** (1.0 / 6.0), n_patches=4, patch_dir=TETRA.copy(),
                eps_patch=5.0, patch_sigma_r=0.1, patch_sigma_ang=0.3, inertia=0.1)


PP_DIRS = np.array([[0.0, 0.0, 1.0], [0.0, 0.0, -1.0]])


def patchy_pp_potential() -> dict:
    """The paper's own patchy model under reading Q1: (sigma/r)^200 core, M = 2 antipodal
    patches at 0.5 sigma from the centre, -eps exp[-1/2 (r_pp / 0.12 sigma)^10] between patches closer than 0.18 sigma."""
    return dict(kind="patchy_pp", epsilon=1.0, sigma=1.0, mass=1.0, shift_energy=0, rcut=1.18, rcut_core=1.18,
                n_patches=2, patch_dir=PP_DIRS.copy(), eps_patch=1.0, patch_sigma_r=0.12, patch_sigma_ang=1.0,
                inertia=0.1, patch_radius=0.5, patch_exponent=10.0, core_exponent=200.0, rcut_patch=0.18)


def patchy_fluid(N: int = 2 ** 18, rho: float = 0.5, T: float = 0.15, skin: float = 0.3,
                 jitter: float = 0.05, seed: int = BASE_SEED + 4, dt: float = 0.002) -> Workload:
    pot = patchy_potential()
    shape = fcc_shape(N)
    a = (4.0 / rho) ** (1.0 / 3.0)
    box = _f32_box([shape[0] * a, shape[1] * a, shape[2] * a])
    x = fcc_sites(shape, a) + (uniform01(seed, 1, 3 * N).reshape(N, 3) * 2.0 - 1.0) * jitter
    pos = _pad4(_wrap_to_f32(x, box))
    vel = _pad4(_velocities(seed, 2, N, T).astype(np.float32))
    q = normal(seed, 3, 4 * N).reshape(N, 4)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    L = normal(seed, 4, 3 * N).reshape(N, 3) * math.sqrt(pot["inertia"] * T)
    return Workload(name=f"patchy_N{N}", N=N, box=box, pos=pos, vel=vel, rcut=pot["rcut"], skin=skin,
                    potential=pot, dt=dt, quat=q.astype(np.float32), angmom=_pad4(L.astype(np.float32)),
                    max_neigh=neighbour_capacity(rho, pot["rcut"] + skin),
                    meta=dict(rho=rho, T=T, jitter=jitter, seed=seed, fcc_shape=shape, a=a))


# --------------------------------------------------------------------------------------
# C3 / D3: bead-spring melt.  The start is purely geometric: chains grown bead by bead
# (all chains in lock-step) with rejection of close contacts, then a position-based
# push-off (overlapping pairs moved apart, long bonds pulled in).  No potential is
# evaluated here (DESIGN.md "input recipe" explains why this replaces SURVEY D3's
# energy descent: the generator must hold none of the method's arithmetic).
# --------------------------------------------------------------------------------------
def polymer_potential() -> dict:
    return dict(kind="fene_wca", epsilon=1.0, sigma=1.0, mass=1.0, shift_energy=1,
                rcut=2.0 ** (1.0 / 6.0), fene_K=30.0, fene_R0=1.5, chain_len=64)


def _unit_vectors(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    z = uniform01(seed, stream, n, offset) * 2.0 - 1.0
    phi = uniform01(seed, stream + 7919, n, offset) * 2.0 * math.pi
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def polymer_melt(n_chains: int = 4096, chain_len: int = 64, rho: float = 0.85, T: float = 1.0,
                 skin: float = 0.3, bond: float = 0.97, seed: int = BASE_SEED + 3, dt: float = 0.005,
                 d_min: float = 0.8, tries: int = 24, relax_iters: int = 60) -> Workload:
    from scipy.spatial import cKDTree

    N = n_chains * chain_len
    Lbox = (N / rho) ** (1.0 / 3.0)
    box = _f32_box([Lbox] * 3)
    L = box[0]
    x = np.zeros((n_chains, chain_len, 3), dtype=np.float64)
    x[:, 0, :] = uniform01(seed, 10, 3 * n_chains).reshape(n_chains, 3) * L
    draw = 0
    for b in range(1, chain_len):
        placed = (x[:, :b, :].reshape(-1, 3)) % L
        tree = cKDTree(placed, boxsize=L)
        todo = np.arange(n_chains)
        best = np.full(n_chains, -1.0)
        best_pos = np.zeros((n_chains, 3))
        for _ in range(tries):
            if todo.size == 0:
                break
            dirs = _unit_vectors(seed, 11 + b, todo.size, offset=draw)
            draw += todo.size
            cand = x[todo, b - 1, :] + bond * dirs
            # nearest placed bead other than the bonded predecessor (k=2: predecessor is at `bond`)
            dist, idx = tree.query(cand % L, k=3)
            pred_flat = todo * b + (b - 1)
            d = np.where(idx == pred_flat[:, None], np.inf, dist).min(axis=1)
            better = d > best[todo]
            best[todo[better]] = d[better]
            best_pos[todo[better]] = cand[better]
            todo = todo[d < d_min]
        x[:, b, :] = best_pos
    x = x.reshape(N, 3)

    # geometric push-off: separate pairs closer than d0, shorten bonds longer than bmax
    d0, bmax = 0.98, 1.15
    ids = np.arange(N)
    bi = ids[(ids + 1) % chain_len != 0]
    bj = bi + 1
    for _ in range(relax_iters):
        xw = x % L
        tree = cKDTree(xw, boxsize=L)
        pairs = tree.query_pairs(d0, output_type="ndarray")
        disp = np.zeros_like(x)
        if pairs.size:
            i, j = pairs[:, 0], pairs[:, 1]
            dv = xw[j] - xw[i]
            dv -= L * np.round(dv / L)
            r = np.linalg.norm(dv, axis=1)
            r = np.maximum(r, 1e-9)
            push = (0.5 * 0.5 * (d0 - r) / r)[:, None] * dv
            np.add.at(disp, j, push)
            np.add.at(disp, i, -push)
        dv = x[bj] - x[bi]
        r = np.linalg.norm(dv, axis=1)
        over = r > bmax
        pull = np.zeros_like(dv)
        pull[over] = (0.5 * 0.5 * (r[over] - bmax) / r[over])[:, None] * dv[over]
        np.add.at(disp, bi, pull)
        np.add.at(disp, bj, -pull)
        np.clip(disp, -0.05, 0.05, out=disp)
        x = x + disp
    pos = _pad4(_wrap_to_f32(x, box))
    vel = _pad4(_velocities(seed, 2, N, T).astype(np.float32))
    pot = polymer_potential()
    pot["chain_len"] = chain_len
    return Workload(name=f"polymer_N{N}", N=N, box=box, pos=pos, vel=vel, rcut=pot["rcut"], skin=skin,
                    potential=pot, dt=dt, max_neigh=32,
                    meta=dict(rho=rho, T=T, seed=seed, n_chains=n_chains, chain_len=chain_len))


# --------------------------------------------------------------------------------------
# D6: dimer gas (parity only) - isolated pairs sweeping every branch of the pair functions
# --------------------------------------------------------------------------------------
def dimer_gas(n_dimers: int = 4096, kind: str = "lj", seed: int = BASE_SEED + 6, spacing: float = 4.0) -> Workload:
    m = int(math.ceil(n_dimers ** (1.0 / 3.0)))
    box = _f32_box([m * spacing] * 3)
    g = np.stack(np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij"), axis=-1).reshape(-1, 3)
    centres = (g[:n_dimers].astype(np.float64) + 0.5) * spacing
    if kind == "lj":
        pot, lo, hi = lj_potential(2.5), 0.90, 1.05 * 2.5
    elif kind == "fene_wca":
        pot, lo, hi = polymer_potential(), 0.80, 1.40
        pot["chain_len"] = 2
    elif kind == "patchy":
        pot, lo, hi = patchy_potential(), 0.90, 1.05 * 1.5
    elif kind == "patchy_pp":
        pot, lo, hi = patchy_pp_potential(), 1.00, 1.14      # contact to just past the 0.18 sigma patch range
    else:
        raise ValueError(kind)
    sep = lo + (hi - lo) * uniform01(seed, 1, n_dimers)
    dirs = _unit_vectors(seed, 2, n_dimers)
    x = np.empty((2 * n_dimers, 3))
    x[0::2] = centres - 0.5 * sep[:, None] * dirs
    x[1::2] = centres + 0.5 * sep[:, None] * dirs
    N = 2 * n_dimers
    quat = angmom = None
    if kind in ("patchy", "patchy_pp"):
        q = normal(seed, 3, 4 * N).reshape(N, 4)
        q /= np.linalg.norm(q, axis=1, keepdims=True)
        # second half of the dimers: rotate each partner so that its patch 0 points within 30 deg
        # of the bond axis (towards the other partner) -> strong patch overlap is exercised.
        half = n_dimers // 2
        tgt = np.empty((N, 3))
        tgt[0::2] = dirs
        tgt[1::2] = -dirs
        tilt = _unit_vectors(seed, 5, N)
        ang = uniform01(seed, 6, N) * (math.pi / 6.0 if kind == "patchy" else math.pi / 18.0)
        perp = tilt - (tilt * tgt).sum(1, keepdims=True) * tgt
        perp /= np.maximum(np.linalg.norm(perp, axis=1, keepdims=True), 1e-12)
        want = np.cos(ang)[:, None] * tgt + np.sin(ang)[:, None] * perp   # desired space-frame patch 0
        b0 = TETRA[0] if kind == "patchy" else PP_DIRS[0]
        # shortest-arc quaternion taking b0 -> want
        c = np.cross(np.broadcast_to(b0, want.shape), want)
        w = 1.0 + (want * b0).sum(1)
        qa = np.concatenate([w[:, None], c], axis=1)
        qa /= np.maximum(np.linalg.norm(qa, axis=1, keepdims=True), 1e-12)
        sel = np.zeros(N, dtype=bool)
        sel[2 * half:] = True
        q[sel] = qa[sel]
        quat = q.astype(np.float32)
        angmom = np.zeros((N, 4), dtype=np.float32)
    pos = _pad4(_wrap_to_f32(x, box))
    vel = np.zeros((N, 4), dtype=np.float32)
    return Workload(name=f"dimers_{kind}_{n_dimers}", N=N, box=box, pos=pos, vel=vel, rcut=pot["rcut"], skin=0.3,
                    potential=pot, dt=0.002, quat=quat, angmom=angmom, max_neigh=16,
                    meta=dict(seed=seed, n_dimers=n_dimers, spacing=spacing))


def config(name: str, **kw) -> Workload:
    """Named BASELINE.json configs."""
    if name == "C1":
        return lj_fluid(2048, 2.5, seed=BASE_SEED + 1, **kw)
    if name == "C2a":
        return lj_fluid(2 ** 20, 2.5, seed=BASE_SEED + 2, **kw)
    if name == "C2b":
        return lj_fluid(2 ** 20, 4.0, seed=BASE_SEED + 2, **kw)
    if name == "C3":
        return polymer_melt(4096, 64, **kw)
    if name == "C4":
        return patchy_fluid(2 ** 18, **kw)
    raise ValueError(name)
