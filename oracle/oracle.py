"""ctypes binding of oracle/gm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It shares nothing with paper_1310_2041_b200/ (the CUDA path) and never imports it.
Observables that are plain post-processing (kinetic energy, momentum, chain Rg^2, bond lengths;
SURVEY.md 8(c) O8) are written here in numpy fp64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gm_oracle.c")
_LIB = os.path.join(_HERE, "libgm_oracle.so")

PAIR = {"none": 0, "lj": 1, "dpd": 2, "harmonic": 3, "gauss": 4, "table": 5}
BOND = {"none": 0, "fene": 1, "harmonic": 2, "table": 3}
INTEG = {"nve": 0, "langevin": 1, "gwvv": 2, "nose_hoover": 3, "andersen": 4, "berendsen": 5, "nph": 6, "npt": 7}
ORC_ERR_BOND_OVERSTRETCH = -7


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("n_types", C.c_int32), ("pair_style", C.c_int32),
        ("bond_style", C.c_int32), ("integrator", C.c_int32),
        ("box", C.c_double * 3),
        ("dt", C.c_double), ("kT", C.c_double), ("gamma", C.c_double), ("lam", C.c_double),
        ("seed", C.c_uint64),
        ("eps", C.c_void_p), ("sigma", C.c_void_p), ("rc", C.c_void_p), ("ushift", C.c_void_p),
        ("n_bonds", C.c_int64),
        ("bond_i", C.c_void_p), ("bond_j", C.c_void_p), ("bond_type", C.c_void_p),
        ("bond_k", C.c_void_p), ("bond_r0", C.c_void_p),
        ("type", C.c_void_p), ("mass", C.c_void_p),
        ("use_cells", C.c_int32), ("n_threads", C.c_int32),
        ("table", C.c_void_p), ("table_points", C.c_int32), ("table_interval", C.c_double),
        ("angle_style", C.c_int32), ("n_angles", C.c_int64),
        ("angle_i", C.c_void_p), ("angle_j", C.c_void_p), ("angle_k", C.c_void_p), ("angle_type", C.c_void_p),
        ("angle_kk", C.c_void_p), ("angle_t0", C.c_void_p),
        ("n_dihedrals", C.c_int64),
        ("dih_i", C.c_void_p), ("dih_j", C.c_void_p), ("dih_k", C.c_void_p), ("dih_l", C.c_void_p), ("dih_type", C.c_void_p),
        ("dih_kk", C.c_void_p), ("dih_delta", C.c_void_p), ("dih_n", C.c_void_p),
        ("thermo", C.c_void_p), ("baro", C.c_void_p),
        ("btable", C.c_void_p), ("btable_points", C.c_int32), ("btable_interval", C.c_void_p),
        ("atable", C.c_void_p), ("atable_points", C.c_int32), ("dtable", C.c_void_p), ("dtable_points", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_philox4x32_10.restype = None
        L.orc_u24.argtypes = [C.c_uint32]
        L.orc_u24.restype = C.c_double
        L.orc_pair_theta.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_int64]
        L.orc_pair_theta.restype = C.c_double
        L.orc_bead_xi.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_void_p]
        L.orc_bead_xi.restype = None
        L.orc_andersen_hit.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_double]
        L.orc_andersen_hit.restype = C.c_int
        L.orc_andersen_normals.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_void_p]
        L.orc_andersen_normals.restype = None
        L.orc_min_image.argtypes = [C.c_double, C.c_double]
        L.orc_min_image.restype = C.c_double
        L.orc_neighbor_pairs.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_double, C.c_int32,
                                         C.c_int64, C.c_void_p]
        L.orc_neighbor_pairs.restype = C.c_int64
        for name in ("orc_pair_bond_forces", "orc_compute_forces"):
            f = getattr(L, name)
            f.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
            f.restype = C.c_int
        L.orc_run.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64,
                              C.c_int64, C.c_void_p]
        L.orc_run.restype = C.c_int
        L.orc_num_threads.restype = C.c_int
        L.orc_virial.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p]
        L.orc_virial.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def u24(x: int) -> float:
    return float(lib().orc_u24(int(x) & 0xFFFFFFFF))


def pair_theta(seed: int, step: int, ti: int, tj: int) -> float:
    return float(lib().orc_pair_theta(seed, step, ti, tj))


def bead_xi(seed: int, step: int, tag: int) -> np.ndarray:
    out = np.zeros(3)
    lib().orc_bead_xi(seed, step, tag, _p(out))
    return out


def min_image(d: float, L: float) -> float:
    return float(lib().orc_min_image(d, L))


def neighbor_pairs(pos, box, r_list: float, use_cells: bool = False) -> np.ndarray:
    """Unique pairs (i<j) with min-image distance < r_list, sorted lexicographically; (P,2) int32."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[0]
    cap = max(1024, int(n * 8))
    while True:
        pairs = np.zeros((cap, 2), dtype=np.int32)
        cnt = int(lib().orc_neighbor_pairs(n, _p(pos), _p(box), float(r_list), int(use_cells), cap, _p(pairs)))
        if cnt <= cap:
            pairs = pairs[:cnt]
            break
        cap = cnt
    order = np.lexsort((pairs[:, 1], pairs[:, 0]))
    return pairs[order]


def spline_table(v, interval: float) -> np.ndarray:
    """Eq. (12): cubic spline through the potential values v[k] = V(z_k) on the grid z_k = k *
    interval of z = r^2, k = 0 .. Npoint (Npoint intervals).  Returns c[Npoint, 4] with V(z_k + d) = c0 + c1 d + c2 d^2
    + c3 d^3: c0 is the value at the grid point, c1..c3 make first and second derivative continuous across the grid
    points ("continuous up to second order").  The paper does not say how the spline ends: natural ends, V'' = 0 at
    z_0 and z_Npoint (reading c-24).  Plain tridiagonal solve for the second derivatives M_k (the textbook
    construction, ref. 41 of the paper), then c1 = (v[k+1] - v[k]) / h - h (2 M_k + M_{k+1}) / 6, c2 = M_k / 2,
    c3 = (M_{k+1} - M_k) / (6 h)."""
    v = np.asarray(v, np.float64)
    n = len(v) - 1
    h = float(interval)
    M = np.zeros(n + 1)
    if n >= 2:
        # h/6 M_{k-1} + 2h/3 M_k + h/6 M_{k+1} = (v[k+1] - 2 v[k] + v[k-1]) / h,  k = 1 .. n-1;  M_0 = M_n = 0
        a = np.full(n - 1, h / 6.0); b = np.full(n - 1, 2.0 * h / 3.0); c = np.full(n - 1, h / 6.0)
        d = (v[2:] - 2.0 * v[1:-1] + v[:-2]) / h
        for k in range(1, n - 1):               # forward elimination
            m = a[k] / b[k - 1]
            b[k] -= m * c[k - 1]
            d[k] -= m * d[k - 1]
        x = np.zeros(n - 1)
        x[-1] = d[-1] / b[-1]
        for k in range(n - 3, -1, -1):          # back substitution
            x[k] = (d[k] - c[k] * x[k + 1]) / b[k]
        M[1:n] = x
    out = np.zeros((n, 4))
    out[:, 0] = v[:-1]
    out[:, 1] = (v[1:] - v[:-1]) / h - h * (2.0 * M[:-1] + M[1:]) / 6.0
    out[:, 2] = 0.5 * M[:-1]
    out[:, 3] = (M[1:] - M[:-1]) / (6.0 * h)
    return out


def lj_ushift(eps, sigma, rc):
    """Energy shift of the 'shifted' LJ of the configs: U_shift = 4 eps [(s/rc)^12 - (s/rc)^6]
    (energy only, the force is untouched; reading c-9)."""
    eps = np.asarray(eps, np.float64)
    s = np.asarray(sigma, np.float64) / np.asarray(rc, np.float64)
    return 4.0 * eps * (s ** 12 - s ** 6)


class Oracle:
    """fp64 oracle over one system, in tag order.  Inputs are the workload's fp32 values promoted."""

    def __init__(self, w, use_cells: bool = True, n_threads: int = 0):
        self.w = w
        n = w.n
        self.n = n
        self.box = np.ascontiguousarray(w.box, dtype=np.float64)
        self.pos = np.ascontiguousarray(w.pos, dtype=np.float64).copy()
        self.vel = np.ascontiguousarray(w.vel, dtype=np.float64).copy()
        self.frc = np.zeros((n, 3))
        self.type = np.ascontiguousarray(w.type, dtype=np.int32)
        self.mass = np.ascontiguousarray(w.mass, dtype=np.float64)
        nt = w.n_types
        if w.pair_style == "lj":
            self.eps = np.ascontiguousarray(w.pair["eps"], np.float64).reshape(nt, nt)
            self.sigma = np.ascontiguousarray(w.pair["sigma"], np.float64).reshape(nt, nt)
            self.rc = np.ascontiguousarray(w.pair["rc"], np.float64).reshape(nt, nt)
            self.ushift = (lj_ushift(self.eps, self.sigma, self.rc) if w.pair.get("shift", True)
                           else np.zeros((nt, nt)))
        elif w.pair_style in ("dpd", "harmonic"):
            # DPD: a;  harmonic repulsion, Eq. (2): alpha
            self.eps = np.ascontiguousarray(w.pair["a"], np.float64).reshape(nt, nt)
            self.sigma = np.ones((nt, nt))
            self.rc = np.ascontiguousarray(w.pair["rc"], np.float64).reshape(nt, nt)
            self.ushift = np.zeros((nt, nt))
        elif w.pair_style == "gauss":
            # Eq. (3): eps exp(-r^2 / 2 sigma^2), cut at rc; shifted = minus its value at rc
            self.eps = np.ascontiguousarray(w.pair["eps"], np.float64).reshape(nt, nt)
            self.sigma = np.ascontiguousarray(w.pair["sigma"], np.float64).reshape(nt, nt)
            self.rc = np.ascontiguousarray(w.pair["rc"], np.float64).reshape(nt, nt)
            self.ushift = (self.eps * np.exp(-0.5 * (self.rc / self.sigma) ** 2) if w.pair.get("shift", True)
                           else np.zeros((nt, nt)))
        elif w.pair_style == "table":
            # the fp32 coefficients the GPU is given, promoted: table[ti, tj, point, 0..3]
            self.table = np.ascontiguousarray(w.pair["table"], np.float64).reshape(nt, nt, -1, 4)
            self.eps = np.zeros((nt, nt)); self.sigma = np.ones((nt, nt)); self.ushift = np.zeros((nt, nt))
            self.rc = np.ascontiguousarray(w.pair["rc"], np.float64).reshape(nt, nt)
        else:
            self.eps = np.zeros((nt, nt)); self.sigma = np.ones((nt, nt))
            self.rc = np.ones((nt, nt)); self.ushift = np.zeros((nt, nt))
        self.ushift = np.ascontiguousarray(self.ushift)
        b = np.ascontiguousarray(w.bonds, dtype=np.int32).reshape(-1, 2)
        self.bond_i = np.ascontiguousarray(b[:, 0])
        self.bond_j = np.ascontiguousarray(b[:, 1])
        self.bond_type = np.ascontiguousarray(w.bond_type, dtype=np.int32)
        self.bond_k = np.ascontiguousarray(w.bond.get("k", [0.0]), dtype=np.float64)
        self.bond_r0 = np.ascontiguousarray(w.bond.get("r0", [0.0]), dtype=np.float64)
        self.step = 0
        self.P = _Params()
        P = self.P
        P.n = n; P.n_types = nt
        P.pair_style = PAIR[w.pair_style]; P.bond_style = BOND[w.bond_style]
        P.integrator = INTEG[w.integrator]
        for d in range(3):
            P.box[d] = float(self.box[d])
        P.dt = float(np.float32(w.dt)); P.kT = float(np.float32(w.kT))
        P.gamma = float(np.float32(w.gamma)); P.lam = float(np.float32(w.lam))
        P.seed = int(w.seed)
        P.eps = _p(self.eps).value; P.sigma = _p(self.sigma).value
        P.rc = _p(self.rc).value; P.ushift = _p(self.ushift).value
        P.n_bonds = len(self.bond_i)
        P.bond_i = _p(self.bond_i).value; P.bond_j = _p(self.bond_j).value
        P.bond_type = _p(self.bond_type).value
        P.bond_k = _p(self.bond_k).value; P.bond_r0 = _p(self.bond_r0).value
        P.type = _p(self.type).value; P.mass = _p(self.mass).value
        P.use_cells = int(use_cells); P.n_threads = int(n_threads)
        # angles / dihedrals (optional attributes of the workload: w.topo = dict(angle_style, angles (n,3), angle_type,
        # angle_k, angle_t0, dihedrals (n,4), dihedral_type, dihedral_k, dihedral_n, dihedral_delta))
        topo = getattr(w, "topo", None) or {}
        ANG = {"none": 0, "harmonic": 1, "cosine": 2, "table": 3}
        self._ang = np.ascontiguousarray(topo.get("angles", np.zeros((0, 3))), np.int32).reshape(-1, 3)
        self._ang_cols = [np.ascontiguousarray(self._ang[:, c]) for c in range(3)]
        self._ang_type = np.ascontiguousarray(topo.get("angle_type", np.zeros(len(self._ang))), np.int32)
        self._ang_k = np.ascontiguousarray(topo.get("angle_k", [0.0]), np.float32).astype(np.float64)
        self._ang_t0 = np.ascontiguousarray(topo.get("angle_t0", [0.0]), np.float32).astype(np.float64)
        P.angle_style = ANG[topo.get("angle_style", "none")] if len(self._ang) else 0
        P.n_angles = len(self._ang)
        P.angle_i, P.angle_j, P.angle_k = (_p(c).value for c in self._ang_cols)
        P.angle_type = _p(self._ang_type).value
        P.angle_kk = _p(self._ang_k).value; P.angle_t0 = _p(self._ang_t0).value
        self._dih = np.ascontiguousarray(topo.get("dihedrals", np.zeros((0, 4))), np.int32).reshape(-1, 4)
        self._dih_cols = [np.ascontiguousarray(self._dih[:, c]) for c in range(4)]
        self._dih_type = np.ascontiguousarray(topo.get("dihedral_type", np.zeros(len(self._dih))), np.int32)
        self._dih_k = np.ascontiguousarray(topo.get("dihedral_k", [0.0]), np.float32).astype(np.float64)
        self._dih_delta = np.ascontiguousarray(topo.get("dihedral_delta", [0.0]), np.float32).astype(np.float64)
        self._dih_n = np.ascontiguousarray(topo.get("dihedral_n", [1]), np.int32)
        P.n_dihedrals = len(self._dih)
        P.dih_i, P.dih_j, P.dih_k, P.dih_l = (_p(c).value for c in self._dih_cols)
        P.dih_type = _p(self._dih_type).value
        P.dih_kk = _p(self._dih_k).value; P.dih_delta = _p(self._dih_delta).value; P.dih_n = _p(self._dih_n).value
        # tabulated angle / torsion potentials: topo["angle_table"] (n_types, Npoint, 4) on theta in [0, pi] with
        # angle_style "table"; topo["dihedral_table"] (n_types, Npoint, 4) on phi in [-pi, pi] replaces Eq. (10)
        if P.angle_style == 3:
            self._atable = np.ascontiguousarray(topo["angle_table"], np.float32).astype(np.float64)
            self._atable = self._atable.reshape(-1, self._atable.shape[-2], 4)
            P.atable = _p(self._atable).value; P.atable_points = int(self._atable.shape[1])
        if len(self._dih) and topo.get("dihedral_table") is not None:
            self._dtable = np.ascontiguousarray(topo["dihedral_table"], np.float32).astype(np.float64)
            self._dtable = self._dtable.reshape(-1, self._dtable.shape[-2], 4)
            P.dtable = _p(self._dtable).value; P.dtable_points = int(self._dtable.shape[1])
        self.thermo = np.zeros(4)       # [have half-step velocity, its kinetic energy, Nose-Hoover xi, -]
        P.thermo = _p(self.thermo).value
        # Andersen barostat (integrators "nph", "npt"): [P_ext, piston mass, piston momentum Pi, virial, virial valid]
        self.baro = np.zeros(5)
        self.baro[0] = float(np.float32(getattr(w, "p_ext", 0.0)))
        self.baro[1] = float(np.float32(getattr(w, "piston_mass", 1.0)))
        P.baro = _p(self.baro).value
        if w.bond_style == "table":
            # w.bond = dict(table=(n_bond_types, Npoint, 4) fp32 coefficients as the GPU gets them, interval=(n_bond_types,))
            self.btable = np.ascontiguousarray(w.bond["table"], np.float64)
            self.btable = self.btable.reshape(-1, self.btable.shape[-2], 4)
            self.btable_interval = np.ascontiguousarray(np.asarray(w.bond["interval"], np.float32).reshape(-1), np.float64)
            P.btable = _p(self.btable).value
            P.btable_points = int(self.btable.shape[1])
            P.btable_interval = _p(self.btable_interval).value
        if w.pair_style == "table":
            P.table = _p(self.table).value
            P.table_points = int(self.table.shape[2])
            P.table_interval = float(np.float32(w.pair["interval"]))
        self.last = np.zeros(3)     # pe_pair, pe_bond, n_pairs_in_rc of the last force call

    # -- forces ---------------------------------------------------------------------------------
    def pair_bond_forces(self, pos=None, vel=None, step=None):
        """F_c (+ DPD dissipative/random) at the given state; returns (F, pe_pair, pe_bond, n_pairs)."""
        pos = self.pos if pos is None else np.ascontiguousarray(pos, np.float64)
        vel = self.vel if vel is None else np.ascontiguousarray(vel, np.float64)
        step = self.step if step is None else step
        F = np.zeros((self.n, 3)); out = np.zeros(3)
        st = lib().orc_pair_bond_forces(C.byref(self.P), _p(pos), _p(vel), int(step), _p(F), _p(out))
        self.status = st
        return F, float(out[0]), float(out[1]), float(out[2])

    def compute_forces(self):
        """The integrator's force at the current state and time level (Langevin: incl. drag+noise)."""
        st = lib().orc_compute_forces(C.byref(self.P), _p(self.pos), _p(self.vel), int(self.step),
                                      _p(self.frc), _p(self.last))
        self.status = st
        return self.frc

    def run(self, n_steps: int):
        scratch = np.zeros(6 * self.n)
        st = lib().orc_run(C.byref(self.P), _p(self.pos), _p(self.vel), _p(self.frc), int(self.step),
                           int(n_steps), _p(scratch))
        self.step += int(n_steps)
        self.status = st
        for d in range(3):              # the barostat rescales the box
            self.box[d] = self.P.box[d]
        return st

    def set_box(self, box):
        """Change the box (the caller rescales positions); invalidates the stored virial."""
        for d in range(3):
            self.P.box[d] = float(box[d]); self.box[d] = float(box[d])
        self.baro[4] = 0.0

    def virial(self, pos=None) -> float:
        """W = sum of r_ij . F_ij over pairs and bonds at the given positions (orc_virial: the definition, O(N^2))."""
        pos = self.pos if pos is None else np.ascontiguousarray(pos, np.float64)
        out = np.zeros(1)
        self.status = lib().orc_virial(C.byref(self.P), _p(pos), _p(out))
        return float(out[0])

    def volume(self) -> float:
        return float(self.box[0] * self.box[1] * self.box[2])

    def pressure(self) -> float:
        """Instantaneous pressure (2 K + W) / (3 V) of the current state."""
        return (2.0 * self.kinetic() + self.virial()) / (3.0 * self.volume())

    def enthalpy_like(self) -> float:
        """Andersen's conserved H = K + U + P_ext V + Pi^2 / (2 M)."""
        a, b, _ = self.potential()
        return self.kinetic() + a + b + self.baro[0] * self.volume() + self.baro[2] ** 2 / (2.0 * self.baro[1])

    # -- observables (O8), plain numpy fp64 -------------------------------------------------------
    def kinetic(self) -> float:
        return 0.5 * float((self.mass[:, None] * self.vel ** 2).sum())

    def momentum(self) -> np.ndarray:
        return (self.mass[:, None] * self.vel).sum(axis=0)

    def temperature(self) -> float:
        return 2.0 * self.kinetic() / (3 * self.n - 3)

    def potential(self):
        """(pe_pair, pe_bond, n_pairs_in_rc) at the current positions (conservative part)."""
        _, a, b, c = self.pair_bond_forces()
        return a, b, c

    def neighbor_pairs(self, r_list: float, use_cells=None) -> np.ndarray:
        uc = bool(self.P.use_cells) if use_cells is None else use_cells
        return neighbor_pairs(self.pos, self.box, r_list, uc)


def bond_lengths(pos, box, bonds) -> np.ndarray:
    pos = np.asarray(pos, np.float64); box = np.asarray(box, np.float64)
    d = pos[bonds[:, 0]] - pos[bonds[:, 1]]
    d -= box * np.rint(d / box)
    return np.sqrt((d * d).sum(axis=1))


def chain_rg2(pos, box, chain_len: int) -> np.ndarray:
    """Per-chain squared radius of gyration by chain-walk unwrapping (sum of min-image bond
    vectors; bonds << L/2), chains = consecutive tags (O8)."""
    pos = np.asarray(pos, np.float64); box = np.asarray(box, np.float64)
    n = (pos.shape[0] // chain_len) * chain_len
    p = pos[:n].reshape(-1, chain_len, 3)
    d = p[:, 1:, :] - p[:, :-1, :]
    d -= box * np.rint(d / box)
    u = np.concatenate([np.zeros_like(p[:, :1, :]), np.cumsum(d, axis=1)], axis=1)
    u -= u.mean(axis=1, keepdims=True)
    return (u * u).sum(axis=2).mean(axis=1)
