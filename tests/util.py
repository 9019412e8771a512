"""Small helpers shared by the tests (no arithmetic of the method)."""
from __future__ import annotations

import numpy as np

from workloads import Workload


def custom(pos, box, vel=None, typ=None, bonds=None, pair_style="lj", eps=1.0, sigma=1.0, rc=2.5,
           shift=True, a=25.0, bond_style="none", k=30.0, r0=1.5, integrator="nve", dt=0.005,
           kT=1.0, gamma=0.0, lam=0.65, r_skin=0.4, seed=7, n_types=1, mass=None, table=None, interval=None,
           bond_table=None, bond_interval=None, bond_type=None) -> Workload:
    pos = np.asarray(pos, dtype=np.float32).reshape(-1, 3)
    n = pos.shape[0]
    box = np.asarray(box, dtype=np.float32).reshape(-1)
    if box.size == 1:
        box = np.repeat(box, 3)
    vel = np.zeros((n, 3), np.float32) if vel is None else np.asarray(vel, np.float32).reshape(n, 3)
    typ = np.zeros(n, np.int32) if typ is None else np.asarray(typ, np.int32)
    bonds = np.zeros((0, 2), np.int32) if bonds is None else np.asarray(bonds, np.int32).reshape(-1, 2)
    mass = np.ones(n, np.float32) if mass is None else np.asarray(mass, np.float32)

    def mat(x):
        x = np.asarray(x, np.float32)
        return np.broadcast_to(x, (n_types, n_types)).copy() if x.ndim == 0 else x.reshape(n_types, n_types).copy()

    if pair_style == "table":
        # table: (n_types, n_types, Npoint, 4) spline coefficients on a grid of z = r^2; the cutoff is "point < Npoint"
        tb = np.asarray(table, np.float32).reshape(n_types, n_types, -1, 4)
        iv = float(np.float32(interval))
        pair = dict(table=tb, interval=iv, rc=mat(np.sqrt(tb.shape[2] * iv)))
    elif pair_style in ("dpd", "harmonic"):
        pair = dict(a=mat(a), rc=mat(rc))
    else:
        pair = dict(eps=mat(eps), sigma=mat(sigma), rc=mat(rc), shift=shift)
    bond = dict(k=np.array([k], np.float32), r0=np.array([r0], np.float32))
    if bond_style == "table":
        # bond_table: (n_bond_types, Npoint, 4) spline coefficients on a grid of z = r^2, one interval per bond type
        bt = np.asarray(bond_table, np.float32)
        bt = bt.reshape(-1, bt.shape[-2], 4)
        bond = dict(table=bt, interval=np.asarray(bond_interval, np.float32).reshape(-1),
                    k=np.zeros(len(bt), np.float32), r0=np.zeros(len(bt), np.float32))
    return Workload(
        name="custom", box=box, pos=pos, vel=vel, type=typ, mass=mass, bonds=bonds,
        bond_type=np.zeros(len(bonds), np.int32) if bond_type is None else np.asarray(bond_type, np.int32),
        n_types=n_types, pair_style=pair_style, pair=pair, bond_style=bond_style, bond=bond,
        integrator=integrator, dt=dt, kT=kT, gamma=gamma, lam=lam, r_skin=r_skin, seed=seed,
    )


def pairs_to_set(pairs) -> set:
    return set(map(tuple, np.asarray(pairs).tolist()))
