"""Pins of the oracle's Eq. (2) / Eq. (3) pair potentials and of the tabulated (cubic-spline in z = r^2) pair
potential of Eqs. (11)-(12) / Algorithm 2.

Closed forms from tests/golden/closed_forms.txt, force = -grad(energy) by central differences, the spline fit against
scipy's natural cubic spline (a library routine), a tabulated Lennard-Jones against the analytic Eq. (1) within the
spline's error bound, the "point < Npoint" cutoff rule, and F = -2 r dV/dz on a potential that is linear in z.
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom
from workloads import make_random_box


def G(golden):
    return {r[0]: float(r[1]) for r in golden("closed_forms.txt")}


def dimer(r, **kw):
    w = custom([[-r / 2, 0, 0], [r / 2, 0, 0]], 20.0, **kw)
    o = orc.Oracle(w, use_cells=False)
    o.pos[:] = [[-r / 2, 0, 0], [r / 2, 0, 0]]
    return o


def fd_force_check(o, n_probe=6, h=1e-6, tol=1e-6):
    F, _, _, _ = o.pair_bond_forces()
    rng = np.random.default_rng(0)
    for i in rng.choice(o.n, n_probe, replace=False):
        for d in range(3):
            p = o.pos.copy(); p[i, d] += h
            up = o.pair_bond_forces(pos=p)[1]
            p[i, d] -= 2 * h
            um = o.pair_bond_forces(pos=p)[1]
            assert F[i, d] == pytest.approx(-(up - um) / (2 * h), abs=tol * max(1.0, np.abs(F).max()))


# ---- Eq. (2): harmonic repulsion -------------------------------------------------------------------------------
def test_harmonic_repulsion_closed_forms(golden):
    g = G(golden)
    o = dimer(1.0, pair_style="harmonic", a=3.0, rc=2.0)
    F, pe, _, npair = o.pair_bond_forces()
    assert npair == 1 and pe == pytest.approx(g["harm_u_at_half_rc"], abs=1e-14)
    assert F[0, 0] == pytest.approx(-g["harm_f_at_half_rc"], abs=1e-14)     # repulsive: bead 0 (at -x) pushed to -x
    assert F[1, 0] == pytest.approx(+g["harm_f_at_half_rc"], abs=1e-14)
    o = dimer(1e-9, pair_style="harmonic", a=3.0, rc=2.0)
    assert o.pair_bond_forces()[1] == pytest.approx(g["harm_u_at_zero"], rel=1e-8)   # alpha, not alpha / 2 (Eq. 13's form)
    o = dimer(2.0 * (1 - 1e-9), pair_style="harmonic", a=3.0, rc=2.0)        # continuous at the cutoff
    F, pe, _, npair = o.pair_bond_forces()
    assert npair == 1 and 0.0 <= pe < 1e-15 and np.abs(F).max() < 1e-8
    o = dimer(2.0 * (1 + 1e-9), pair_style="harmonic", a=3.0, rc=2.0)
    assert o.pair_bond_forces()[3] == 0


def test_harmonic_and_gauss_force_is_minus_gradient_and_third_law():
    for style, kw in (("harmonic", dict(a=25.0, rc=1.5)), ("gauss", dict(eps=3.0, sigma=0.7, rc=2.5))):
        w = make_random_box(300, (6.0, 7.0, 8.0), seed=11)
        w2 = custom(w.pos, w.box, pair_style=style, **kw)
        o = orc.Oracle(w2, use_cells=False)
        F = o.pair_bond_forces()[0]
        assert np.abs(F.sum(axis=0)).max() < 1e-10 and np.abs(F).max() > 1.0
        fd_force_check(o)
        oc = orc.Oracle(w2, use_cells=True)                                  # cell mode == all-pairs definition
        Fc, pec, _, nc = oc.pair_bond_forces()
        assert np.abs(Fc - F).max() < 1e-11 and nc == o.pair_bond_forces()[3]


# ---- Eq. (3): Gaussian repulsion -------------------------------------------------------------------------------
def test_gaussian_repulsion_closed_forms(golden):
    g = G(golden)
    o = dimer(0.8, pair_style="gauss", eps=2.0, sigma=0.8, rc=4.0, shift=False)
    o.sigma[:] = 0.8                                                         # exact fp64 sigma (the workload carries fp32)
    F, pe, _, npair = o.pair_bond_forces()
    assert npair == 1 and pe == pytest.approx(g["gauss_u_at_sigma"], rel=1e-14)
    assert F[1, 0] == pytest.approx(g["gauss_f_at_sigma"], rel=1e-14) and F[0, 0] == -F[1, 0]
    o = dimer(0.8, pair_style="gauss", eps=2.0, sigma=0.8, rc=4.0, shift=True)
    o.sigma[:] = 0.8; o.ushift[:] = 2.0 * math.exp(-0.5 * 25.0)              # shifted: minus U(r_cut), force untouched
    F2, pe2, _, _ = o.pair_bond_forces()
    assert pe2 == pytest.approx(g["gauss_u_at_sigma"] - 2.0 * math.exp(-12.5), rel=1e-14) and F2[1, 0] == F[1, 0]


# ---- Eqs. (11)-(12), Algorithm 2: tabulated pair potential -------------------------------------------------------
def test_spline_fit_matches_scipy_natural_cubic_spline():
    from scipy.interpolate import CubicSpline
    rng = np.random.default_rng(5)
    z = 0.01 * np.arange(401)
    v = np.cos(3.0 * z) * np.exp(-0.3 * z) + 0.05 * rng.normal(size=z.size).cumsum() * 0.01
    c = orc.spline_table(v, 0.01)
    cs = CubicSpline(z, v, bc_type="natural")
    # scipy stores the polynomial of interval k in descending powers of (z - z_k)
    assert np.allclose(c[:, 0], cs.c[3], rtol=0, atol=1e-13)
    assert np.allclose(c[:, 1], cs.c[2], rtol=1e-9, atol=1e-10)
    assert np.allclose(c[:, 2], cs.c[1], rtol=1e-8, atol=1e-8)
    assert np.allclose(c[:, 3], cs.c[0], rtol=1e-7, atol=1e-6)


def _lj_table(n_point, z_max, z_min):
    """U_LJ tabulated on a grid of z = r^2 (Eq. (1) in terms of z: 4 (z^-6 - z^-3)), flat below z_min (never reached)."""
    interval = z_max / n_point
    z = interval * np.arange(n_point + 1)
    zz = np.maximum(z, z_min)
    v = 4.0 * (zz ** -6 - zz ** -3)
    return orc.spline_table(v, interval), interval


def test_tabulated_lj_reproduces_analytic_lj_within_the_spline_error():
    # 4,000 grid points up to r_cut = 2.5 ("several thousands"): h = 1.5625e-3 in z.  Spline error of the
    # derivative ~ h^3 V(z) / 24; for r >= 0.9 (z >= 0.81) V = 4 (3024 z^-10 - 360 z^-7) < 1.0e5 -> < 1.6e-5 in
    # dV/dz, i.e. relative force error < 1e-4 at the steepest point and far less elsewhere.
    c, interval = _lj_table(4000, 6.25, 0.49)
    w = make_random_box(400, (8.0, 8.0, 8.0), seed=12, min_sep=0.9)
    wt = custom(w.pos, w.box, pair_style="table", table=c[None, None], interval=interval)
    wl = custom(w.pos, w.box, pair_style="lj", rc=2.5, shift=False)
    ot, ol = orc.Oracle(wt, use_cells=False), orc.Oracle(wl, use_cells=False)
    ot.table[:] = c; ot.P.table_interval = interval                       # exact fp64 table (the workload carries fp32)
    ol.rc[:] = 2.5
    Ft, pet, _, nt = ot.pair_bond_forces()
    Fl, pel, _, nl = ol.pair_bond_forces()
    assert nt == nl and nt > 1000
    assert np.abs(Ft - Fl).max() <= 1e-4 * np.abs(Fl).max()
    assert pet == pytest.approx(pel, rel=1e-6, abs=1e-6 * nt)
    fd_force_check(ot, tol=1e-5)
    # Newton's third law and the cell-list mode
    assert np.abs(Ft.sum(axis=0)).max() < 1e-9
    oc = orc.Oracle(wt, use_cells=True)
    oc.table[:] = c; oc.P.table_interval = interval
    assert np.abs(oc.pair_bond_forces()[0] - Ft).max() < 1e-11


def test_table_cutoff_is_point_less_than_npoint_and_force_is_minus_2r_dvdz():
    # V(z) = z (U = r^2): linear in z, reproduced exactly by the spline; Eq. (11): F_i = -2 r_ij dV/dz = -2 r_ij
    n_point, interval = 50, 0.08                                           # z_max = 4.0 -> r_cut = 2.0
    c = orc.spline_table(interval * np.arange(n_point + 1), interval)
    assert np.allclose(c[:, 1], 1.0) and np.abs(c[:, 2:]).max() < 1e-12
    for r, inside in ((1.3, True), (2.0 * (1 - 1e-9), True), (2.0 * (1 + 1e-9), False)):
        o = dimer(r, pair_style="table", table=c[None, None], interval=interval)
        o.table[:] = c; o.P.table_interval = interval
        F, pe, _, npair = o.pair_bond_forces()
        assert npair == (1 if inside else 0)
        if inside:
            assert pe == pytest.approx(r * r, rel=1e-12)
            assert F[0, 0] == pytest.approx(-2.0 * (-r), rel=1e-12)        # bead 0 at -r/2: r_01 = -r, F_0 = +2 r
            assert F[1, 0] == pytest.approx(-2.0 * r, rel=1e-12)
        else:
            assert pe == 0.0 and np.abs(F).max() == 0.0
