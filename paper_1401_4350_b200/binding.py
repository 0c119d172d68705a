"""ctypes binding of libmd_b200.so: argument marshalling only (same names as include/md_b200.h)."""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libmd_b200.so"

STRATEGY = {"vertex": 0, "edge": 1, "vertex_n3": 2}
SCATTER = {"red": 0, "red_v4": 1, "warp": 2, "segmented": 3, "cluster": 4}
GATHER = {"auto": 0, "l2": 1, "smem": 2}
ORDER = {"none": 0, "cell": 1, "hilbert": 2}
PRECISION = {"f32": 0, "mixed": 1}
ARRAY = {"pos": 0, "vel": 1, "force": 2, "quat": 3, "angmom": 4, "torque": 5}
STEP_PART = {"kick_drift": 0, "kick": 1}
OPTION = {"stage_limit": 0, "no_graph": 1, "debug": 2, "row_schedule": 3, "build_direct": 4, "fuse_steps": 5}
PROBE = {"ffma": 0, "ffma2": 1, "mufu": 2, "red_v4_scatter": 3, "red_f32_scatter": 4, "red_v4_coalesced": 5,
         "red_f32_coalesced": 6}
POT_KIND = {"lj": 0, "fene_wca": 1, "patchy": 2, "patchy_pp": 3}
STATUS = {0: "MD_OK", -1: "MD_ERR_INVALID", -2: "MD_ERR_STATE", -3: "MD_ERR_CAPACITY", -4: "MD_ERR_CUDA",
          -5: "MD_ERR_NUMERIC"}

# every symbol include/md_b200.h declares (checked by tests/test_abi.py against the header and the .so)
EXPORTED_SYMBOLS = ["md_workspace_bytes", "md_create", "md_bind_state", "md_set_order", "md_set_precision",
                    "md_get_state_double", "md_set_thermostat", "md_thermostat", "md_build_cells",
                    "md_build_verlet", "md_forces", "md_integrate", "md_energy", "md_stats", "md_stats_ex",
                    "md_set_option", "md_probe", "md_resize", "md_set_active", "md_half_step", "md_rebuild_flag",
                    "md_gather_ids", "md_scatter_ids", "md_dd_select", "md_energy_static", "md_get_pairs", "md_get_ids", "md_step_host", "md_launch_count",
                    "md_last_error", "md_destroy"]


class MDError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class MDPotential(C.Structure):
    _fields_ = [
        ("kind", C.c_int32),
        ("epsilon", C.c_float), ("sigma", C.c_float), ("mass", C.c_float),
        ("shift_energy", C.c_int32),
        ("fene_K", C.c_float), ("fene_R0", C.c_float),
        ("chain_len", C.c_int32),
        ("n_patches", C.c_int32),
        ("patch_dir", (C.c_float * 3) * 8),
        ("eps_patch", C.c_float), ("patch_sigma_r", C.c_float), ("patch_sigma_ang", C.c_float),
        ("rcut_core", C.c_float),
        ("inertia", C.c_float),
        ("patch_radius", C.c_float), ("patch_exponent", C.c_float), ("core_exponent", C.c_float),
        ("rcut_patch", C.c_float),
    ]


class MDStatsEx(C.Structure):
    _fields_ = [("n_edges", C.c_int64), ("n_full_entries", C.c_int64), ("n_rebuilds", C.c_int64),
                ("n_in_cutoff", C.c_int64), ("max_neigh_seen", C.c_int32), ("max_stage", C.c_int32),
                ("stage_launch", C.c_int32), ("threads_per_particle", C.c_int32), ("cluster_size", C.c_int32),
                ("pad0", C.c_int32), ("n_cluster_units", C.c_int64)]


def make_potential(d: dict) -> MDPotential:
    p = MDPotential()
    p.kind = POT_KIND[d["kind"]]
    p.epsilon = d.get("epsilon", 1.0)
    p.sigma = d.get("sigma", 1.0)
    p.mass = d.get("mass", 1.0)
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


def library_path() -> Path:
    return _LIB_PATH


_lib = None


def load_library() -> C.CDLL:
    """Load libmd_b200.so (built in-tree by paper_1401_4350_b200/build.py). Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_1401_4350_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(str(_LIB_PATH))
    dp3 = C.POINTER(C.c_double)
    vp = C.c_void_p
    L.md_workspace_bytes.restype = C.c_int
    L.md_workspace_bytes.argtypes = [C.c_int64, dp3, C.c_double, C.c_double, C.POINTER(MDPotential), C.c_int32,
                                     C.POINTER(C.c_size_t)]
    L.md_create.restype = C.c_int
    L.md_create.argtypes = [C.POINTER(vp), C.c_int64, dp3, C.c_double, C.c_double, C.POINTER(MDPotential), C.c_int32,
                            vp, C.c_size_t, vp]
    L.md_bind_state.restype = C.c_int
    L.md_bind_state.argtypes = [vp] * 7
    L.md_set_order.restype = C.c_int
    L.md_set_order.argtypes = [vp, C.c_int32]
    L.md_set_precision.restype = C.c_int
    L.md_set_precision.argtypes = [vp, C.c_int32]
    L.md_set_thermostat.restype = C.c_int
    L.md_set_thermostat.argtypes = [vp, C.c_double, C.c_int64, C.c_double, C.c_double, C.c_uint64]
    L.md_thermostat.restype = C.c_int
    L.md_thermostat.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_uint32]
    L.md_get_state_double.restype = C.c_int
    L.md_get_state_double.argtypes = [vp, vp, vp]
    for name in ("md_build_cells", "md_build_verlet"):
        getattr(L, name).restype = C.c_int
        getattr(L, name).argtypes = [vp]
    L.md_forces.restype = C.c_int
    L.md_forces.argtypes = [vp, C.c_int32, C.c_int32]
    L.md_integrate.restype = C.c_int
    L.md_integrate.argtypes = [vp, C.c_double, C.c_int64, C.c_int32, C.c_int32]
    L.md_energy.restype = C.c_int
    L.md_energy.argtypes = [vp, dp3, dp3, dp3]
    L.md_stats.restype = C.c_int
    L.md_stats.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_int64)]
    L.md_stats_ex.restype = C.c_int
    L.md_stats_ex.argtypes = [vp, C.POINTER(MDStatsEx), C.c_size_t]
    L.md_set_option.restype = C.c_int
    L.md_set_option.argtypes = [vp, C.c_int32, C.c_int64]
    L.md_probe.restype = C.c_int
    L.md_probe.argtypes = [vp, C.c_int32, dp3]
    L.md_resize.restype = C.c_int
    L.md_resize.argtypes = [vp, C.c_int64]
    L.md_set_active.restype = C.c_int
    L.md_set_active.argtypes = [vp, C.c_int64]
    L.md_half_step.restype = C.c_int
    L.md_half_step.argtypes = [vp, C.c_double, C.c_int32]
    L.md_rebuild_flag.restype = C.c_int
    L.md_rebuild_flag.argtypes = [vp, C.POINTER(C.c_int32)]
    L.md_gather_ids.restype = C.c_int
    L.md_gather_ids.argtypes = [vp, C.c_int32, vp, C.c_int64, C.c_int64, vp]
    L.md_scatter_ids.restype = C.c_int
    L.md_scatter_ids.argtypes = [vp, C.c_int32, C.c_int64, C.c_int64, vp]
    L.md_dd_select.restype = C.c_int
    L.md_dd_select.argtypes = [vp, C.c_int64, C.c_int32, C.c_double, C.c_double, vp, C.c_int64, C.POINTER(C.c_int64), vp,
                               C.c_size_t, vp]
    L.md_energy_static.restype = C.c_int
    L.md_energy_static.argtypes = [vp, vp, vp, C.c_int64, C.c_double, C.c_double, vp, vp, C.c_char_p, C.c_size_t]
    L.md_get_pairs.restype = C.c_int
    L.md_get_pairs.argtypes = [vp, C.POINTER(C.c_int32), C.c_int64, C.POINTER(C.c_int64)]
    L.md_get_ids.restype = C.c_int
    L.md_get_ids.argtypes = [vp, C.POINTER(C.c_int32)]
    L.md_step_host.restype = C.c_int
    L.md_step_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_double, C.c_int64, C.c_int32, C.c_int32]
    L.md_launch_count.restype = C.c_int64
    L.md_launch_count.argtypes = [vp]
    L.md_last_error.restype = C.c_char_p
    L.md_last_error.argtypes = [vp]
    L.md_destroy.restype = None
    L.md_destroy.argtypes = [vp]
    _lib = L
    return L


def variant_code(strategy: str, variant) -> int:
    """Third argument of md_forces / md_integrate / md_step_host: md_gather for VERTEX, md_scatter for EDGE, the number
    of force copies m for VERTEX_N3 (an int; anything else means the default)."""
    if strategy == "vertex":
        return GATHER.get(variant, 0)      # anything that is not a gather name means "auto"
    if strategy == "vertex_n3":
        return int(variant) if isinstance(variant, int) else 0
    return SCATTER[variant]


class MDSystem:
    """One system on one GPU. State lives in torch CUDA tensors ([N,4] float32) owned by this object and
    borrowed by the library; the workspace is one torch uint8 tensor."""

    def __init__(self, N: int, box, rcut: float, skin: float, potential: dict, max_neigh: int,
                 device: str = "cuda:0", order: str = "none", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1401_4350_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.N = int(N)
        self.box = np.ascontiguousarray(box, dtype=np.float64)
        self.rcut, self.skin = float(rcut), float(skin)
        self.pot = make_potential(potential)
        self.rigid = potential["kind"] in ("patchy", "patchy_pp")
        self.max_neigh = int(max_neigh)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        nbytes = C.c_size_t(0)
        boxp = self.box.ctypes.data_as(C.POINTER(C.c_double))
        rc = self.lib.md_workspace_bytes(self.N, boxp, self.rcut, self.skin, C.byref(self.pot), self.max_neigh,
                                         C.byref(nbytes))
        if rc != 0:
            raise MDError(rc, "md_workspace_bytes: invalid parameters")
        self.workspace_bytes = int(nbytes.value)
        self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        h = C.c_void_p(None)
        rc = self.lib.md_create(C.byref(h), self.N, boxp, self.rcut, self.skin, C.byref(self.pot), self.max_neigh,
                                C.c_void_p(self._ws_ptr), self.workspace_bytes, C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            raise MDError(rc, "md_create failed (invalid geometry / parameters)")
        self.h = h
        self.N_capacity = self.N
        z = lambda: torch.zeros((self.N, 4), dtype=torch.float32, device=self.device)
        self._full = {"pos": z(), "vel": z(), "force": z()}
        if self.rigid:
            self._full.update({"quat": z(), "angmom": z(), "torque": z()})
            self._full["quat"][:, 0] = 1.0
        self._views_and_bind()
        if order != "none":
            self.set_order(order)

    # ---- plumbing ----
    def _views_and_bind(self):
        """State tensors = the first N rows of the capacity tensors (md_resize keeps the base pointers)."""
        f = self._full
        self.pos, self.vel, self.force = f["pos"][:self.N], f["vel"][:self.N], f["force"][:self.N]
        self.quat = self.angmom = self.torque = None
        if self.rigid:
            self.quat, self.angmom, self.torque = f["quat"][:self.N], f["angmom"][:self.N], f["torque"][:self.N]
        self._check(self.lib.md_bind_state(self.h, *[C.c_void_p(x.data_ptr()) if x is not None else None for x in
                                                    (self.pos, self.vel, self.force, self.quat, self.angmom,
                                                     self.torque)]))

    def _check(self, rc: int):
        if rc != 0:
            raise MDError(rc, self.lib.md_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            self.torch.cuda.synchronize(self.device)
            self.lib.md_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @classmethod
    def from_workload(cls, w, device="cuda:0", order="none", max_neigh=None):
        s = cls(w.N, w.box, w.rcut, w.skin, w.potential, max_neigh or w.max_neigh, device=device, order=order)
        s.set_state(w.pos, w.vel, w.quat, w.angmom)
        return s

    def set_state(self, pos, vel=None, quat=None, angmom=None):
        """Upload state given in ORIGINAL id order (resets the slot map: call build_cells afterwards)."""
        t = self.torch
        up = lambda a: t.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(self.device)
        self.pos.copy_(up(pos))
        if vel is not None:
            self.vel.copy_(up(vel))
        if self.rigid and quat is not None:
            self.quat.copy_(up(quat))
        if self.rigid and angmom is not None:
            self.angmom.copy_(up(angmom))
        # a fresh bind resets the validity flags; slot map is identity only for a new handle or order none
        self._check(self.lib.md_bind_state(self.h, *[C.c_void_p(x.data_ptr()) if x is not None else None for x in
                                                    (self.pos, self.vel, self.force, self.quat, self.angmom,
                                                     self.torque)]))

    # ---- the C ABI, same names ----
    def set_order(self, order):
        self._check(self.lib.md_set_order(self.h, ORDER[order] if isinstance(order, str) else int(order)))

    def set_precision(self, precision):
        self._check(self.lib.md_set_precision(self.h, PRECISION[precision] if isinstance(precision, str) else int(precision)))

    def set_thermostat(self, T, n_newt, p_trans, p_rot=0.0, seed=0):
        """md_integrate applies the thermostat of reading QT after every n_newt-th step; n_newt = 0: off."""
        self._check(self.lib.md_set_thermostat(self.h, float(T), int(n_newt), float(p_trans), float(p_rot), int(seed)))

    def thermostat(self, T, p_trans, p_rot=0.0, seed=0, call=0):
        """One application of the thermostat (asynchronous)."""
        self._check(self.lib.md_thermostat(self.h, float(T), float(p_trans), float(p_rot), int(seed), int(call)))

    def state_f64(self):
        """(pos, vel) of MD_PREC_MIXED as float64 [N,3] arrays in original id order."""
        pos, vel = np.empty((self.N, 3), dtype=np.float64), np.empty((self.N, 3), dtype=np.float64)
        self._check(self.lib.md_get_state_double(self.h, C.c_void_p(pos.ctypes.data), C.c_void_p(vel.ctypes.data)))
        return pos, vel

    def build_cells(self):
        self._check(self.lib.md_build_cells(self.h))

    def build_verlet(self):
        self._check(self.lib.md_build_verlet(self.h))

    def forces(self, strategy="vertex", scatter="red_v4"):
        self._check(self.lib.md_forces(self.h, STRATEGY[strategy], variant_code(strategy, scatter)))

    def integrate(self, dt, nsteps, strategy="vertex", scatter="red_v4"):
        self._check(self.lib.md_integrate(self.h, float(dt), int(nsteps), STRATEGY[strategy],
                                            variant_code(strategy, scatter)))

    def energy(self):
        u, kt, kr = C.c_double(0), C.c_double(0), C.c_double(0)
        self._check(self.lib.md_energy(self.h, C.byref(u), C.byref(kt), C.byref(kr)))
        return u.value, kt.value, kr.value

    def stats(self):
        ne, nf, nr = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        mx = C.c_int32(0)
        self._check(self.lib.md_stats(self.h, C.byref(ne), C.byref(nf), C.byref(mx), C.byref(nr)))
        return dict(n_edges=ne.value, n_full_entries=nf.value, max_neigh_seen=mx.value, n_rebuilds=nr.value)

    def stats_ex(self):
        r = MDStatsEx()
        self._check(self.lib.md_stats_ex(self.h, C.byref(r), C.sizeof(r)))
        return {k: getattr(r, k) for k, _ in MDStatsEx._fields_ if k != "pad0"}

    def set_option(self, option, value):
        self._check(self.lib.md_set_option(self.h, OPTION[option] if isinstance(option, str) else int(option), int(value)))

    def probe(self, kind) -> float:
        """One machine ceiling measured on this device (md_probe_kind): TFLOP/s, Tops/s or G lane-operations/s."""
        v = C.c_double(0)
        self._check(self.lib.md_probe(self.h, PROBE[kind] if isinstance(kind, str) else int(kind), C.byref(v)))
        return v.value

    # ---- space decomposition support (md_b200.h "Space decomposition"; paper_1401_4350_b200/dd.py drives it) ----
    def resize(self, n: int):
        """md_resize + rebind: the state tensors become the first n rows of the capacity tensors (contents kept)."""
        self._check(self.lib.md_resize(self.h, int(n)))
        self.N = int(n)
        self._views_and_bind()

    def set_active(self, n_active: int):
        self._check(self.lib.md_set_active(self.h, int(n_active)))

    def half_step(self, dt, part):
        self._check(self.lib.md_half_step(self.h, float(dt), STEP_PART[part] if isinstance(part, str) else int(part)))

    def rebuild_flag(self) -> int:
        f = C.c_int32(0)
        self._check(self.lib.md_rebuild_flag(self.h, C.byref(f)))
        return int(f.value)

    def gather_ids(self, array, ids=None, first_id=0, n=None):
        """float32 [n,4] device tensor: array rows of the particles with ORIGINAL ids `ids` (int32 device tensor) or
        first_id .. first_id + n - 1."""
        t = self.torch
        n = int(ids.shape[0]) if ids is not None else int(n)
        out = t.empty((n, 4), dtype=t.float32, device=self.device)
        self._check(self.lib.md_gather_ids(self.h, ARRAY[array], C.c_void_p(ids.data_ptr()) if ids is not None and n > 0 else None,
                                           int(first_id), n, C.c_void_p(out.data_ptr()) if n > 0 else None))
        return out

    def scatter_ids(self, array, first_id, src):
        n = int(src.shape[0])
        src = src.contiguous()
        self._check(self.lib.md_scatter_ids(self.h, ARRAY[array], int(first_id), n, C.c_void_p(src.data_ptr()) if n > 0 else None))

    def get_pairs(self) -> np.ndarray:
        """Half list as ORIGINAL-id pairs (lo, hi), int32 [E,2], unsorted."""
        n = C.c_int64(0)
        self._check(self.lib.md_get_pairs(self.h, None, 0, C.byref(n)))
        out = np.empty((max(int(n.value), 1), 2), dtype=np.int32)
        self._check(self.lib.md_get_pairs(self.h, out.ctypes.data_as(C.POINTER(C.c_int32)), int(n.value), C.byref(n)))
        return out[:int(n.value)]

    def get_ids(self) -> np.ndarray:
        ids = np.empty(self.N, dtype=np.int32)
        self._check(self.lib.md_get_ids(self.h, ids.ctypes.data_as(C.POINTER(C.c_int32))))
        return ids

    def step_host(self, pos, vel, force, dt, nsteps, strategy="vertex", scatter="red_v4", quat=None, angmom=None,
                  torque=None):
        """End-to-end call on HOST (pinned or pageable) torch/numpy float32 [N,4] buffers, updated in place."""
        ptr = lambda a: None if a is None else C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
        self._check(self.lib.md_step_host(self.h, ptr(pos), ptr(vel), ptr(force), ptr(quat), ptr(angmom), ptr(torque),
                                          float(dt), int(nsteps), STRATEGY[strategy], variant_code(strategy, scatter)))

    def launch_count(self) -> int:
        return int(self.lib.md_launch_count(self.h))

    # ---- helpers (not part of the path) ----
    def in_id_order(self, tensor) -> np.ndarray:
        """Copy a state tensor to the host in ORIGINAL id order."""
        ids = self.get_ids()
        a = tensor.detach().cpu().numpy()
        out = np.empty_like(a)
        out[ids] = a
        return out


def dd_select(pos, lo: float, hi: float, axis: int = 0, stream=None):
    """md_dd_select: int32 device tensor of the indices i (ascending) with lo <= pos[i, axis] < hi (fp32 comparisons).
    pos: float32 [n,4] CUDA tensor."""
    import torch
    lib = load_library()
    n = int(pos.shape[0])
    pos = pos.contiguous()
    st = stream if stream is not None else torch.cuda.current_stream(pos.device)
    scratch = torch.empty(n // 1024 + 4, dtype=torch.int32, device=pos.device)
    out = torch.empty(max(n, 1), dtype=torch.int32, device=pos.device)
    cnt = C.c_int64(0)
    rc = lib.md_dd_select(C.c_void_p(pos.data_ptr()), n, int(axis), float(lo), float(hi), C.c_void_p(out.data_ptr()), n,
                          C.byref(cnt), C.c_void_p(scratch.data_ptr()), scratch.numel() * 4, C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise MDError(rc, "md_dd_select failed")
    return out[:int(cnt.value)]


ENERGY_STATIC_MAX_N = 16777216   # MD_ENERGY_STATIC_MAX_N


def energy_static(vel, force, out, angmom=None, mass: float = 1.0, inv_inertia: float = 0.0, stream=None):
    """md_energy_static: (U, K_t, K_r) of float32 [n,4] CUDA tensors into `out` (float64 [3] CUDA tensor, passed by the
    caller: this call allocates nothing on the device; its scratch is a static device array of the library).  Asynchronous
    on `stream` (default: torch's current stream of vel.device, which must be the current device).  Calls that overlap on
    the GPU race on the shared scratch."""
    import torch
    lib = load_library()
    for t in (vel, force) + ((angmom,) if angmom is not None else ()):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.dim() == 2 and t.shape[1] == 4):
            raise ValueError("energy_static: state arrays must be contiguous float32 [n,4] CUDA tensors")
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 3):
        raise ValueError("energy_static: out must be a contiguous float64 CUDA tensor of at least 3 elements")
    n = int(vel.shape[0])
    st = stream if stream is not None else torch.cuda.current_stream(vel.device)
    err = C.create_string_buffer(256)
    rc = lib.md_energy_static(C.c_void_p(vel.data_ptr()), C.c_void_p(force.data_ptr()),
                              C.c_void_p(angmom.data_ptr()) if angmom is not None else None, n, float(mass), float(inv_inertia),
                              C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream), err, 256)
    if rc != 0:
        raise MDError(rc, err.value.decode() or "md_energy_static failed")
    return out
