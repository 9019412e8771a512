"""Pins of the oracle's tabulated angle and torsion potentials (Eq. (12) with x = theta, phi):

  * V = b theta (a spline with c2 = c3 = 0, exact): on a right angle the end beads feel b / |arm| perpendicular to their arm,
    in the plane, opening... closing the angle for b > 0 -- the closed form of F = -b grad(theta);
  * V = b phi: the end beads feel b / (distance from the j-k axis), perpendicular to the axis and to their radius;
    net force and net torque vanish;
  * finely tabulated Eq. (8) and Eq. (10) reproduce the analytic branches (themselves pinned in test_oracle_pins_topo.py)
    within the spline error on a melt;
  * force = -grad(energy) by central differences on the tabulated energy.
"""
from __future__ import annotations

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom
from workloads import make_config


def angle_table(fn, n_point):
    h = np.pi / n_point
    return orc.spline_table(fn(h * np.arange(n_point + 1)), h).astype(np.float32)


def dihedral_table(fn, n_point):
    h = 2.0 * np.pi / n_point
    return orc.spline_table(fn(-np.pi + h * np.arange(n_point + 1)), h).astype(np.float32)


def linear_table(b, x0, h, n_point):
    tb = np.zeros((n_point, 4), np.float32)
    tb[:, 0] = b * (x0 + h * np.arange(n_point))
    tb[:, 1] = b
    return tb


def test_linear_in_theta_on_a_right_angle():
    b, la, lb = 2.0, 1.25, 0.8
    pos = np.array([[la, 0.0, 0.0], [0.0, 0.0, 0.0], [0.0, lb, 0.0]])
    w = custom(pos, 12.0, pair_style="none")
    w.topo = dict(angle_style="table", angles=np.array([[0, 1, 2]]), angle_type=np.array([0]),
                  angle_table=linear_table(b, 0.0, np.pi / 256, 256)[None])
    f, _, u, _ = orc.Oracle(w, use_cells=False).pair_bond_forces()
    assert u == pytest.approx(b * np.pi / 2, rel=1e-6)
    np.testing.assert_allclose(f[0], [0.0, b / la, 0.0], atol=1e-9)          # closes the angle: toward the other arm
    np.testing.assert_allclose(f[2], [b / lb, 0.0, 0.0], atol=1e-9)
    np.testing.assert_allclose(f[1], -f[0] - f[2], atol=1e-12)


def test_linear_in_phi_end_beads_feel_b_over_their_distance_from_the_axis():
    b, d1, d2, phi0 = 1.5, 0.875, 1.25, 1.1               # (the workload stores fp32: tolerances 1e-6)
    pos = np.array([[d1, 0.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, 1.0], [d2 * np.cos(phi0), d2 * np.sin(phi0), 1.0]])
    w = custom(pos, 12.0, pair_style="none")
    w.topo = dict(dihedrals=np.array([[0, 1, 2, 3]]), dihedral_type=np.array([0]), dihedral_k=[0.0], dihedral_n=[1],
                  dihedral_delta=[0.0], dihedral_table=linear_table(b, -np.pi, 2 * np.pi / 256, 256)[None])
    o = orc.Oracle(w, use_cells=False)
    f, _, u, _ = o.pair_bond_forces()
    assert abs(u) == pytest.approx(b * phi0, rel=1e-6)                        # |phi| = phi0 (sign: reading c-27)
    assert np.linalg.norm(f[0]) == pytest.approx(b / d1, rel=1e-6)
    assert np.linalg.norm(f[3]) == pytest.approx(b / d2, rel=1e-6)
    assert abs(f[0][2]) < 1e-6 and abs(f[0][0]) < 1e-6                      # tangential: along y for a bead on the x axis
    radial = np.array([np.cos(phi0), np.sin(phi0), 0.0])
    assert abs(f[3] @ radial) < 1e-6 and abs(f[3][2]) < 1e-6
    # the two end beads are pushed so that |phi| shrinks (b > 0), i.e. toward each other's half plane
    assert np.sign(f[0][1]) == np.sign(pos[3][1]) and (f[3] @ np.array([-np.sin(phi0), np.cos(phi0), 0.0])) * pos[3][1] < 0
    np.testing.assert_allclose(f.sum(axis=0), 0.0, atol=1e-12)
    np.testing.assert_allclose(np.cross(o.pos, f).sum(axis=0), 0.0, atol=1e-12)


def melt_with_tables(n_point=2000):
    from tests.test_gpu_topo import with_topology
    w = with_topology(make_config("C1", scale=0.5), "harmonic")
    t = w.topo
    wt = with_topology(make_config("C1", scale=0.5), "harmonic")
    at = np.stack([angle_table(lambda th, k=k, t0=t0: k * (th - t0) ** 2, n_point)
                   for k, t0 in zip(t["angle_k"], t["angle_t0"])])
    dt = np.stack([dihedral_table(lambda ph, k=k, n=n, dl=dl: k * (1.0 + np.cos(n * ph - dl)), n_point)
                   for k, n, dl in zip(t["dihedral_k"], t["dihedral_n"], t["dihedral_delta"])])
    wt.topo = dict(t, angle_style="table", angle_table=at, dihedral_table=dt)
    return w, wt


def test_fine_tables_reproduce_eq8_and_eq10_on_a_melt():
    w, wt = melt_with_tables()
    for x in (w, wt):
        x.pair_style = "none"; x.bond_style = "none"
    rng = np.random.default_rng(2)
    jig = rng.normal(0, 0.08, w.pos.shape).astype(np.float32)                 # off the straight lattice chains
    w.pos = w.pos + jig; wt.pos = wt.pos + jig
    fa, _, ua, _ = orc.Oracle(w, use_cells=False).pair_bond_forces()
    ft, _, ut, _ = orc.Oracle(wt, use_cells=False).pair_bond_forces()
    frms = np.sqrt((fa ** 2).sum(axis=1).mean())
    assert frms > 1.0
    assert np.abs(fa - ft).max() < 2e-5 * frms
    assert ut == pytest.approx(ua, rel=1e-6)


def test_force_is_minus_gradient_of_the_tabulated_energy():
    _, wt = melt_with_tables(n_point=500)
    wt.pair_style = "none"; wt.bond_style = "none"
    rng = np.random.default_rng(4)
    wt.pos = wt.pos + rng.normal(0, 0.08, wt.pos.shape).astype(np.float32)
    o = orc.Oracle(wt, use_cells=False)
    f = o.pair_bond_forces()[0]
    h = 1e-6
    for i, d in ((0, 0), (5, 1), (11, 2), (57, 0), (140, 1)):
        p = o.pos.copy(); p[i, d] += h
        up = o.pair_bond_forces(pos=p)[2]
        p[i, d] -= 2 * h
        um = o.pair_bond_forces(pos=p)[2]
        assert -(up - um) / (2 * h) == pytest.approx(f[i, d], rel=1e-4, abs=1e-5)
