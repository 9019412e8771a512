"""Pins of the oracle's tabulated bond potential ("numerical ... bond ... potentials", Eqs. (11)-(12) with
x = z = r^2; reading c-32) against what the mathematics fixes:

  * V = a + b z is a cubic spline with c2 = c3 = 0, so the table is exact: F_i = -2 b r_ij, the force of the harmonic
    bond U = k r^2 (Eq. (7) with r0 = 0, itself pinned by its dimer frequency omega = 2 sqrt(k));
  * a finely tabulated U = k (r - r0)^2 oscillates at the textbook omega = 2 sqrt(k) (reduced mass 1/2);
  * force = -grad(energy) by central differences on a chain, and Newton's third law;
  * a bond stretched past the end of its table is reported, with no force from it;
  * the virial of tabulated bonds is minus the scaling derivative of their energy.
"""
from __future__ import annotations

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom


def table_of(fn, z_max, n_point):
    """spline coefficients of V(z) = fn(sqrt(z)) on n_point intervals of [0, z_max] (the oracle's own Eq. (12) fit)"""
    h = z_max / n_point
    z = h * np.arange(n_point + 1)
    return orc.spline_table(fn(np.sqrt(z)), h).astype(np.float32), np.float32(h)


def test_linear_in_z_table_is_the_r0_zero_harmonic_bond():
    k = 3.5
    n_point, h = 64, np.float32(0.125)
    tb = np.zeros((n_point, 4), np.float32)
    tb[:, 0] = 0.75 + k * h * np.arange(n_point)               # c0 = V(z_k), c1 = dV/dz = k (all exact in fp32)
    tb[:, 1] = k
    rng = np.random.default_rng(3)
    pos = rng.uniform(-1.0, 1.0, (8, 3))
    bonds = np.array([[0, 1], [1, 2], [2, 3], [4, 5], [5, 6], [6, 7], [7, 0]])
    wt = custom(pos, 12.0, bonds=bonds, pair_style="none", bond_style="table", bond_table=tb[None], bond_interval=[h])
    wh = custom(pos, 12.0, bonds=bonds, pair_style="none", bond_style="harmonic", k=k, r0=0.0)
    ft, _, ut, _ = orc.Oracle(wt, use_cells=False).pair_bond_forces()
    fh, _, uh, _ = orc.Oracle(wh, use_cells=False).pair_bond_forces()
    np.testing.assert_allclose(ft, fh, rtol=0, atol=1e-12)
    assert ut == pytest.approx(uh + 0.75 * len(bonds), abs=1e-10)


def test_tabulated_harmonic_dimer_oscillates_at_two_sqrt_k():
    k, r0 = 25.0, 1.0
    tb, h = table_of(lambda r: k * (r - r0) ** 2, 2.25, 4000)
    pos = np.array([[-0.53, 0.0, 0.0], [0.53, 0.0, 0.0]])
    w = custom(pos, 12.0, bonds=[[0, 1]], pair_style="none", bond_style="table", bond_table=tb[None], bond_interval=[h],
               dt=0.001)
    o = orc.Oracle(w, use_cells=False)
    o.compute_forces()
    xs = []
    for _ in range(1400):
        o.run(1)
        xs.append(o.pos[1, 0] - o.pos[0, 0] - r0)
    xs = np.array(xs)
    up = np.where((xs[:-1] < 0) & (xs[1:] >= 0))[0]
    t = (up + xs[up] / (xs[up] - xs[up + 1])) * float(np.float32(0.001))
    period = np.diff(t).mean()
    assert 2.0 * np.pi / period == pytest.approx(2.0 * np.sqrt(k), rel=2e-4)


def chain_workload(n=12, stretch=1.0):
    rng = np.random.default_rng(11)
    pos = np.cumsum(rng.normal(0, 0.55 * stretch, (n, 3)), axis=0)
    pos -= pos.mean(axis=0)
    k, R0 = 30.0, 1.5
    fene = lambda r: -0.5 * k * R0 * R0 * np.log(np.maximum(1.0 - (r / R0) ** 2, 1e-9))
    tb0, h0 = table_of(fene, 1.4 ** 2, 2000)
    tb1, h1 = table_of(lambda r: 7.0 * (r - 0.9) ** 2, 3.0 ** 2, 2000)
    bonds = np.stack([np.arange(n - 1), np.arange(1, n)], axis=1)
    return custom(pos, 30.0, bonds=bonds, bond_type=np.arange(n - 1) % 2, pair_style="none", bond_style="table",
                  bond_table=np.stack([tb0, tb1]), bond_interval=[h0, h1])


def test_force_is_minus_gradient_and_newton_and_virial():
    w = chain_workload(stretch=0.6)
    o = orc.Oracle(w, use_cells=False)
    f, _, u0, _ = o.pair_bond_forces()
    assert o.status == 0
    assert np.abs(f.sum(axis=0)).max() < 1e-10
    h = 1e-6
    for i, d in ((0, 0), (3, 1), (7, 2), (11, 0)):
        p = o.pos.copy(); p[i, d] += h
        up = o.pair_bond_forces(pos=p)[2]
        p[i, d] -= 2 * h
        um = o.pair_bond_forces(pos=p)[2]
        assert -(up - um) / (2 * h) == pytest.approx(f[i, d], rel=2e-5, abs=1e-6)
    W = o.virial()
    pos0, box0 = o.pos.copy(), o.box.copy()
    us = []
    for s in (1 + h, 1 - h):
        o.set_box(box0 * s)
        us.append(o.pair_bond_forces(pos=pos0 * s)[2])
    assert W == pytest.approx(-(us[0] - us[1]) / (2 * h), rel=1e-5)


def test_bond_past_the_end_of_its_table_is_reported_and_exerts_no_force():
    tb, h = table_of(lambda r: 5.0 * (r - 1.0) ** 2, 1.5 ** 2, 100)
    pos = np.array([[-0.8, 0.0, 0.0], [0.8, 0.0, 0.0], [0.8, 1.0, 0.0]])
    w = custom(pos, 12.0, bonds=[[0, 1], [1, 2]], pair_style="none", bond_style="table", bond_table=tb[None], bond_interval=[h])
    o = orc.Oracle(w, use_cells=False)
    f, _, u, _ = o.pair_bond_forces()
    assert o.status == orc.ORC_ERR_BOND_OVERSTRETCH
    assert np.abs(f[0]).max() == 0.0                           # bead 0 has only the over-long bond
    assert u == pytest.approx(0.0, abs=1e-6)                   # the other bond sits at its minimum r = 1
