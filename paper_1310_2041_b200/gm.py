"""ctypes binding of include/gm.h -- argument marshalling only; every step of the path runs in the
CUDA kernels of libgm.so.  PyTorch supplies device memory (the workspace blob, device-side I/O
tensors) and the CUDA stream, nothing else.

Function names and argument order are those of include/gm.h; each wrapper raises GmError on a
non-zero status.  `System` bundles create + parameter calls for a workload description (any object
with the attributes of workloads.Workload; this module does not import it).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgm.so")

GM_OK = 0
GM_ERR_INVALID_ARG, GM_ERR_STATE, GM_ERR_CUDA, GM_ERR_WORKSPACE_TOO_SMALL = -1, -2, -3, -4
GM_ERR_BOX_TOO_SMALL, GM_ERR_NEIGHBOR_OVERFLOW, GM_ERR_BOND_OVERSTRETCH, GM_ERR_NONFINITE = -5, -6, -7, -8
GM_PAIR = {"none": 0, "lj": 1, "dpd": 2, "harmonic": 3, "gauss": 4, "table": 5}
GM_BOND = {"none": 0, "fene": 1, "harmonic": 2, "table": 3}
GM_INTEG = {"nve": 0, "langevin": 1, "gwvv": 2, "nose_hoover": 3, "andersen": 4, "berendsen": 5, "nph": 6, "npt": 7}
GM_ANGLE = {"none": 0, "harmonic": 1, "cosine": 2, "table": 3}
GM_FLAG_NO_GRAPH, GM_FLAG_NO_COND_NODES, GM_FLAG_STEP_SUBWARP, GM_FLAG_NO_WINDOWS = 1, 2, 4, 8

SYMBOLS = ["gm_query_workspace", "gm_create", "gm_destroy", "gm_set_pair_params", "gm_set_pair_table", "gm_fit_pair_table",
           "gm_set_bond_params", "gm_set_angle_params", "gm_set_dihedral_params", "gm_set_angles", "gm_set_dihedrals",
           "gm_set_particles", "gm_set_bonds", "gm_set_step", "gm_build_neighbors", "gm_compute_forces",
           "gm_step", "gm_step_timed", "gm_set_integrator", "gm_energies", "gm_get_particles", "gm_get_neighbors", "gm_get_stats",
           "gm_get_tuning", "gm_set_barostat", "gm_set_box_state", "gm_get_box", "gm_kinetic_static", "gm_set_bond_table", "gm_set_angle_table", "gm_set_dihedral_table",
           "gm_sfc_cell_order", "gm_last_error"]


class gm_config(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("device", C.c_int32), ("stream", C.c_void_p),
        ("n_particles", C.c_int64), ("n_types", C.c_int32), ("max_bonds_per_particle", C.c_int32),
        ("box", C.c_float * 3), ("r_cut_max", C.c_float), ("r_skin", C.c_float), ("dt", C.c_float),
        ("seed", C.c_uint64),
        ("pair_style", C.c_int32), ("bond_style", C.c_int32), ("integrator", C.c_int32),
        ("kT", C.c_float), ("gamma", C.c_float), ("lam", C.c_float),
        ("sfc_period", C.c_int32), ("nl_row_capacity", C.c_int32), ("flags", C.c_int32),
        ("x_cell_div", C.c_int32), ("nl_scan_trip", C.c_int32), ("step_shape", C.c_int32),
        ("table_points", C.c_int32), ("win_capacity", C.c_int32), ("tile_windows", C.c_int32),
        ("angle_style", C.c_int32), ("max_angles_per_particle", C.c_int32), ("max_dihedrals_per_particle", C.c_int32),
        ("bond_table_points", C.c_int32), ("angle_table_points", C.c_int32), ("dihedral_table_points", C.c_int32),
    ]


class GmError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"gm status {status}: {msg}")
        self.status = status


_lib = None


def lib():
    """Load libgm.so (no GPU needed to load; CUDA is initialised on the first device call)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1310_2041_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
        L.gm_query_workspace.argtypes = [C.POINTER(gm_config), C.POINTER(C.c_size_t)]
        L.gm_create.argtypes = [C.POINTER(gm_config), vp, C.c_size_t, C.POINTER(vp)]
        L.gm_destroy.argtypes = [vp]
        L.gm_set_pair_params.argtypes = [vp, i32, i32, vp, i32]
        L.gm_set_pair_table.argtypes = [vp, i32, i32, C.c_float, vp]
        L.gm_fit_pair_table.argtypes = [i32, C.c_double, vp, vp]
        L.gm_set_bond_params.argtypes = [vp, i32, C.c_float, C.c_float]
        L.gm_set_bond_table.argtypes = [vp, i32, C.c_float, vp]
        L.gm_set_angle_table.argtypes = [vp, i32, vp]
        L.gm_set_dihedral_table.argtypes = [vp, i32, vp]
        L.gm_set_angle_params.argtypes = [vp, i32, C.c_float, C.c_float]
        L.gm_set_dihedral_params.argtypes = [vp, i32, C.c_float, i32, C.c_float]
        L.gm_set_angles.argtypes = [vp, i64, vp, vp]
        L.gm_set_dihedrals.argtypes = [vp, i64, vp, vp]
        L.gm_set_particles.argtypes = [vp, vp, vp, vp, vp, i32]
        L.gm_set_bonds.argtypes = [vp, i64, vp, vp, i32]
        L.gm_set_step.argtypes = [vp, C.c_uint64]
        L.gm_build_neighbors.argtypes = [vp]
        L.gm_compute_forces.argtypes = [vp]
        L.gm_step.argtypes = [vp, i64]
        L.gm_step_timed.argtypes = [vp, i64, vp]
        L.gm_set_integrator.argtypes = [vp, i32, C.c_float, C.c_float]
        L.gm_energies.argtypes = [vp, vp]
        L.gm_set_barostat.argtypes = [vp, C.c_float, C.c_float]
        L.gm_set_box_state.argtypes = [vp, C.c_double, C.c_double]
        L.gm_get_box.argtypes = [vp, vp]
        L.gm_kinetic_static.argtypes = [vp, vp, i64, i32, vp, vp, C.c_char_p, C.c_size_t]
        L.gm_get_particles.argtypes = [vp, vp, vp, vp, i32]
        L.gm_get_neighbors.argtypes = [vp, vp, vp, i64, i32]
        L.gm_get_stats.argtypes = [vp, vp]
        L.gm_get_tuning.argtypes = [vp, vp]
        L.gm_sfc_cell_order.argtypes = [vp, vp]
        L.gm_last_error.argtypes = [vp]
        L.gm_last_error.restype = C.c_char_p
        for name in SYMBOLS[:-1]:
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(status: int, handle=None):
    if status != GM_OK:
        msg = lib().gm_last_error(handle).decode() if handle else "(no system)"
        raise GmError(status, msg)


def _ptr(a):
    """Pointer + residency of a numpy array (host) or torch tensor (host or device)."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data, False
    assert a.is_contiguous()
    return a.data_ptr(), a.is_cuda


def _same_side(*arrs) -> int:
    sides = {d for _, d in (_ptr(a) for a in arrs) if d is not None}
    if len(sides) > 1:
        raise ValueError("arrays of one call must all be host or all be device")
    return int(sides.pop()) if sides else 0


# ---- one function per entry of include/gm.h ----------------------------------------------------------
def gm_query_workspace(cfg: gm_config) -> int:
    out = C.c_size_t(0)
    _check(lib().gm_query_workspace(C.byref(cfg), C.byref(out)))
    return int(out.value)


def gm_create(cfg: gm_config, workspace) -> int:
    h = C.c_void_p(0)
    _check(lib().gm_create(C.byref(cfg), workspace.data_ptr(), workspace.numel() * workspace.element_size(), C.byref(h)))
    return h.value


def gm_destroy(h):
    _check(lib().gm_destroy(h))


def gm_set_pair_params(h, ti: int, tj: int, p):
    p = np.ascontiguousarray(p, dtype=np.float32)
    _check(lib().gm_set_pair_params(h, ti, tj, p.ctypes.data, p.size), h)


def gm_set_pair_table(h, ti: int, tj: int, interval: float, c4):
    c4 = np.ascontiguousarray(c4, dtype=np.float32)
    _check(lib().gm_set_pair_table(h, ti, tj, interval, c4.ctypes.data), h)


def gm_fit_pair_table(v, interval: float) -> np.ndarray:
    """Spline coefficients (Npoint, 4) float32 through the Npoint + 1 potential values v on the grid z = k * interval."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.zeros((len(v) - 1, 4), dtype=np.float32)
    _check(lib().gm_fit_pair_table(len(v) - 1, float(interval), v.ctypes.data, out.ctypes.data))
    return out


def gm_set_bond_params(h, btype: int, k: float, r0: float):
    _check(lib().gm_set_bond_params(h, btype, k, r0), h)


def gm_set_bond_table(h, btype: int, interval: float, c4):
    c4 = np.ascontiguousarray(c4, dtype=np.float32)
    _check(lib().gm_set_bond_table(h, btype, interval, c4.ctypes.data), h)


def gm_set_angle_table(h, atype: int, c4):
    c4 = np.ascontiguousarray(c4, dtype=np.float32)
    _check(lib().gm_set_angle_table(h, atype, c4.ctypes.data), h)


def gm_set_dihedral_table(h, dtype: int, c4):
    c4 = np.ascontiguousarray(c4, dtype=np.float32)
    _check(lib().gm_set_dihedral_table(h, dtype, c4.ctypes.data), h)


def gm_set_angle_params(h, atype: int, k: float, theta0: float):
    _check(lib().gm_set_angle_params(h, atype, k, theta0), h)


def gm_set_dihedral_params(h, dtype: int, k: float, n: int, delta: float):
    _check(lib().gm_set_dihedral_params(h, dtype, k, n, delta), h)


def gm_set_angles(h, tags3, atype=None):
    tags3 = np.ascontiguousarray(tags3, dtype=np.int32).reshape(-1, 3)
    atype = None if atype is None else np.ascontiguousarray(atype, dtype=np.int32)
    _check(lib().gm_set_angles(h, len(tags3), tags3.ctypes.data, None if atype is None else atype.ctypes.data), h)


def gm_set_dihedrals(h, tags4, dtype=None):
    tags4 = np.ascontiguousarray(tags4, dtype=np.int32).reshape(-1, 4)
    dtype = None if dtype is None else np.ascontiguousarray(dtype, dtype=np.int32)
    _check(lib().gm_set_dihedrals(h, len(tags4), tags4.ctypes.data, None if dtype is None else dtype.ctypes.data), h)


def gm_set_particles(h, pos3, vel3, type_, mass=None):
    dev = _same_side(pos3, vel3, type_, mass)
    _check(lib().gm_set_particles(h, _ptr(pos3)[0], _ptr(vel3)[0], _ptr(type_)[0], _ptr(mass)[0], dev), h)


def gm_set_bonds(h, tag_pairs2, btype=None):
    n = 0 if tag_pairs2 is None else int(tag_pairs2.shape[0])
    dev = _same_side(tag_pairs2, btype)
    _check(lib().gm_set_bonds(h, n, _ptr(tag_pairs2)[0], _ptr(btype)[0], dev), h)


def gm_set_step(h, step: int):
    _check(lib().gm_set_step(h, step), h)


def gm_build_neighbors(h):
    _check(lib().gm_build_neighbors(h), h)


def gm_compute_forces(h):
    _check(lib().gm_compute_forces(h), h)


def gm_step(h, n_steps: int):
    _check(lib().gm_step(h, n_steps), h)


def gm_step_timed(h, n_steps: int) -> np.ndarray:
    out = np.zeros(4, dtype=np.float64)
    _check(lib().gm_step_timed(h, n_steps, out.ctypes.data), h)
    return out


def gm_set_integrator(h, integrator: int, kT: float, gamma: float):
    _check(lib().gm_set_integrator(h, integrator, kT, gamma), h)


def gm_set_barostat(h, p_ext: float, piston_mass: float):
    _check(lib().gm_set_barostat(h, p_ext, piston_mass), h)


def gm_set_box_state(h, volume: float, piston_momentum: float):
    _check(lib().gm_set_box_state(h, volume, piston_momentum), h)


def gm_get_box(h) -> np.ndarray:
    out = np.zeros(8, dtype=np.float64)
    _check(lib().gm_get_box(h, out.ctypes.data), h)
    return out


GM_STATIC_MAX_BEADS = 8388608


def gm_kinetic_static(vel3, mass, out4, stream=None):
    """Kinetic energy and momentum of the beads (vel3: CUDA float32 (n, 3), mass: CUDA float32 (n,) or None) into out4 (CUDA
    float64 (4,)), asynchronously on `stream` (default: torch's current stream); allocates nothing (gm.h)."""
    import torch
    st = torch.cuda.current_stream(vel3.device) if stream is None else stream
    buf = C.create_string_buffer(256)
    r = lib().gm_kinetic_static(vel3.data_ptr(), mass.data_ptr() if mass is not None else None, int(vel3.shape[0]),
                                vel3.device.index or 0, st.cuda_stream, out4.data_ptr(), buf, 256)
    if r != GM_OK:
        raise GmError(r, buf.value.decode())


def gm_energies(h) -> np.ndarray:
    out = np.zeros(8, dtype=np.float64)
    _check(lib().gm_energies(h, out.ctypes.data), h)
    return out


def gm_get_particles(h, pos3=None, vel3=None, force3=None):
    dev = _same_side(pos3, vel3, force3)
    _check(lib().gm_get_particles(h, _ptr(pos3)[0], _ptr(vel3)[0], _ptr(force3)[0], dev), h)


def gm_get_neighbors(h, nn, nl_tags):
    dev = _same_side(nn, nl_tags)
    _check(lib().gm_get_neighbors(h, _ptr(nn)[0], _ptr(nl_tags)[0], int(nl_tags.shape[1]), dev), h)


def gm_get_stats(h, check: bool = True) -> dict:
    out = np.zeros(8, dtype=np.int64)
    st = lib().gm_get_stats(h, out.ctypes.data)
    if check:
        _check(st, h)
    keys = ["steps", "rebuilds", "reorders", "max_nn", "sum_nn", "dev_err", "nl_row_capacity", "n_cells"]
    d = dict(zip(keys, (int(x) for x in out)))
    d["status"] = st
    return d


def gm_get_tuning(h) -> dict:
    out = np.zeros(8, dtype=np.int64)
    _check(lib().gm_get_tuning(h, out.ctypes.data), h)
    keys = ["x_cell_div", "nl_scan_trip", "step_shape", "windows", "win_capacity", "tiles", "tiles_not_windowed",
            "nl_smem_bytes"]
    return dict(zip(keys, (int(x) for x in out)))


def gm_sfc_cell_order(nc) -> np.ndarray:
    nc = np.ascontiguousarray(nc, dtype=np.int32)
    out = np.zeros(int(nc[0]) * int(nc[1]) * int(nc[2]), dtype=np.uint32)
    _check(lib().gm_sfc_cell_order(nc.ctypes.data, out.ctypes.data))
    return out


# ---- convenience: one object per system ---------------------------------------------------------------
class System:
    """Create a gm_system for a workload description and keep its workspace alive.

    `w` needs: n, box, pos, vel, type, mass, bonds, bond_type, n_types, pair_style, pair, bond_style,
    bond, integrator, dt, kT, gamma, lam, r_skin, seed, sfc_period (see workloads.Workload).
    """

    def __init__(self, w, device: int = 0, flags: int = 0, nl_row_capacity: int = 0, sfc_period=None,
                 load: bool = True, tune: dict | None = None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1310_2041_b200 needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.w = w
        self.n = int(w.n)
        self.device = torch.device("cuda", device)
        cfg = gm_config()
        cfg.struct_size = C.sizeof(gm_config)
        cfg.device = device
        cfg.stream = torch.cuda.current_stream(self.device).cuda_stream
        cfg.n_particles = self.n
        cfg.n_types = int(w.n_types)
        bonds = np.ascontiguousarray(w.bonds, dtype=np.int32).reshape(-1, 2)
        self.bonds = bonds
        if len(bonds) and w.bond_style != "none":
            cfg.max_bonds_per_particle = int(np.bincount(bonds.ravel(), minlength=self.n).max())
        else:
            cfg.max_bonds_per_particle = 0
        for d in range(3):
            cfg.box[d] = float(w.box[d])
        pair = w.pair
        cfg.r_cut_max = float(np.max(pair["rc"])) if w.pair_style != "none" else 1.0
        cfg.table_points = int(pair["table"].shape[2]) if w.pair_style == "table" else 0
        cfg.r_skin = float(w.r_skin)
        cfg.dt = float(w.dt)
        cfg.seed = int(w.seed)
        cfg.pair_style = GM_PAIR[w.pair_style]
        cfg.bond_style = GM_BOND[w.bond_style] if cfg.max_bonds_per_particle else 0
        if cfg.bond_style == GM_BOND["table"]:
            cfg.bond_table_points = int(np.asarray(w.bond["table"]).shape[-2])
        cfg.integrator = GM_INTEG[w.integrator]
        cfg.kT, cfg.gamma, cfg.lam = float(w.kT), float(w.gamma), float(w.lam)
        cfg.sfc_period = int(w.sfc_period if sfc_period is None else sfc_period)
        cfg.nl_row_capacity = int(nl_row_capacity)
        cfg.flags = int(flags)
        topo = getattr(w, "topo", None) or {}
        ang = np.ascontiguousarray(topo.get("angles", np.zeros((0, 3))), np.int32).reshape(-1, 3)
        dih = np.ascontiguousarray(topo.get("dihedrals", np.zeros((0, 4))), np.int32).reshape(-1, 4)
        if len(ang):
            cfg.angle_style = GM_ANGLE[topo.get("angle_style", "harmonic")]
            cfg.max_angles_per_particle = int(np.bincount(ang.ravel(), minlength=self.n).max())
            if cfg.angle_style == GM_ANGLE["table"]:
                cfg.angle_table_points = int(np.asarray(topo["angle_table"]).shape[-2])
        if len(dih):
            cfg.max_dihedrals_per_particle = int(np.bincount(dih.ravel(), minlength=self.n).max())
            if topo.get("dihedral_table") is not None:
                cfg.dihedral_table_points = int(np.asarray(topo["dihedral_table"]).shape[-2])
        for k, v in (tune or {}).items():       # gm_config tuning overrides: x_cell_div, nl_scan_trip, step_shape
            setattr(cfg, k, int(v))
        self.cfg = cfg
        nbytes = gm_query_workspace(cfg)
        self.workspace_bytes = nbytes
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        self._ws_view = self.workspace[off:off + nbytes]
        self.h = gm_create(cfg, self._ws_view)
        nt = cfg.n_types
        for ti in range(nt):
            for tj in range(ti, nt):
                if w.pair_style == "lj":
                    gm_set_pair_params(self.h, ti, tj, [pair["eps"][ti][tj], pair["sigma"][ti][tj],
                                                        pair["rc"][ti][tj], 1.0 if pair.get("shift", True) else 0.0])
                elif w.pair_style in ("dpd", "harmonic"):
                    gm_set_pair_params(self.h, ti, tj, [pair["a"][ti][tj], pair["rc"][ti][tj]])
                elif w.pair_style == "gauss":
                    gm_set_pair_params(self.h, ti, tj, [pair["eps"][ti][tj], pair["sigma"][ti][tj],
                                                        pair["rc"][ti][tj], 1.0 if pair.get("shift", True) else 0.0])
                elif w.pair_style == "table":
                    gm_set_pair_table(self.h, ti, tj, float(pair["interval"]), pair["table"][ti][tj])
        if cfg.bond_style == GM_BOND["table"]:
            tb = np.asarray(w.bond["table"], np.float32)
            tb = tb.reshape(-1, tb.shape[-2], 4)
            for bt in range(len(tb)):
                gm_set_bond_table(self.h, bt, float(np.asarray(w.bond["interval"], np.float32).reshape(-1)[bt]), tb[bt])
        elif cfg.bond_style:
            for bt in range(len(w.bond["k"])):
                gm_set_bond_params(self.h, bt, float(w.bond["k"][bt]), float(w.bond["r0"][bt]))
        if len(ang):
            if cfg.angle_table_points:
                tb = np.asarray(topo["angle_table"], np.float32)
                for at, t4 in enumerate(tb.reshape(-1, tb.shape[-2], 4)):
                    gm_set_angle_table(self.h, at, t4)
            else:
                for at, (k, t0) in enumerate(zip(topo["angle_k"], topo["angle_t0"])):
                    gm_set_angle_params(self.h, at, float(np.float32(k)), float(np.float32(t0)))
            gm_set_angles(self.h, ang, topo.get("angle_type"))
        if len(dih):
            if cfg.dihedral_table_points:
                tb = np.asarray(topo["dihedral_table"], np.float32)
                for dt_, t4 in enumerate(tb.reshape(-1, tb.shape[-2], 4)):
                    gm_set_dihedral_table(self.h, dt_, t4)
            else:
                for dt_, (k, nn, dl) in enumerate(zip(topo["dihedral_k"], topo["dihedral_n"], topo["dihedral_delta"])):
                    gm_set_dihedral_params(self.h, dt_, float(np.float32(k)), int(nn), float(np.float32(dl)))
            gm_set_dihedrals(self.h, dih, topo.get("dihedral_type"))
        if w.integrator in ("nph", "npt"):
            gm_set_barostat(self.h, float(np.float32(getattr(w, "p_ext", 0.0))), float(np.float32(getattr(w, "piston_mass", 1.0))))
        if load:
            self.set_particles(w.pos, w.vel, w.type, w.mass)
            if cfg.max_bonds_per_particle:
                gm_set_bonds(self.h, bonds, np.ascontiguousarray(w.bond_type, dtype=np.int32))

    def close(self):
        if getattr(self, "h", None):
            gm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # thin forwards
    def set_particles(self, pos, vel, typ, mass=None):
        f32 = lambda a: None if a is None else (np.ascontiguousarray(a, dtype=np.float32) if isinstance(a, np.ndarray) else a)
        typ = np.ascontiguousarray(typ, dtype=np.int32) if isinstance(typ, np.ndarray) else typ
        gm_set_particles(self.h, f32(pos), f32(vel), typ, f32(mass))

    def build_neighbors(self):
        gm_build_neighbors(self.h)

    def compute_forces(self):
        gm_compute_forces(self.h)

    def step(self, n: int):
        gm_step(self.h, n)

    def step_timed(self, n: int) -> dict:
        t = gm_step_timed(self.h, n)
        return dict(force_ms=t[0], rebuild_ms=t[1], force_launches=int(t[2]), reorders=int(t[3]))

    def set_integrator(self, name: str, kT: float = 1.0, gamma: float = 0.0):
        gm_set_integrator(self.h, GM_INTEG[name], kT, gamma)

    def set_barostat(self, p_ext: float, piston_mass: float):
        gm_set_barostat(self.h, p_ext, piston_mass)

    def set_box_state(self, volume: float, piston_momentum: float = 0.0):
        gm_set_box_state(self.h, volume, piston_momentum)

    def box_state(self) -> dict:
        b = gm_get_box(self.h)
        return dict(box=b[0:3].copy(), volume=b[3], piston_momentum=b[4], pressure=b[5], virial=b[6], H=b[7])

    def energies(self) -> dict:
        e = gm_energies(self.h)
        return dict(ke=e[0], pe_pair=e[1], pe_bond=e[2], T=e[3], p=e[4:7].copy(), n_pairs=e[7],
                    etot=e[0] + e[1] + e[2])

    def get_particles(self, pos=True, vel=True, force=False):
        out = [np.empty((self.n, 3), np.float32) if f else None for f in (pos, vel, force)]
        gm_get_particles(self.h, *out)
        return out

    def neighbors(self):
        """(nn, nl_tags) on the host; nl_tags has max_nn columns."""
        gm_build_neighbors(self.h) if self.stats()["max_nn"] == 0 and self.stats()["rebuilds"] == 0 else None
        stride = max(1, self.stats()["max_nn"])
        nn = np.zeros(self.n, np.int32)
        nl = np.zeros((self.n, stride), np.int32)
        gm_get_neighbors(self.h, nn, nl)
        return nn, nl

    def tuning(self) -> dict:
        return gm_get_tuning(self.h)

    def stats(self, check: bool = True) -> dict:
        return gm_get_stats(self.h, check)

    def synchronize(self):
        self.torch.cuda.current_stream(self.device).synchronize()
