"""Pins of the oracle's Andersen barostat (NPH / NPT; PAPER.md:L133 names it, reading c-31) against what the
mathematics fixes -- none of them re-types the oracle's update formulas:

  * the virial is minus the derivative of the potential energy under a uniform scaling of coordinates and box
    (central differences of the oracle's own energies);
  * an ideal gas under the piston obeys the ODE  M V'' = 2 K0 (V0/V)^(2/3) / (3 V) - P_ext  (adiabatic K V^(2/3) = const):
    the oracle against scipy's integrator of that ODE, converging at second order in dt; and it stays at rest at the volume
    where 2 K / (3 V) = P_ext;
  * Andersen's H = K + U + P_ext V + Pi^2 / (2 M) is conserved, with a fluctuation that falls as dt^2;
  * the step is time-reversible;
  * with a huge piston mass it reduces to the oracle's NVE velocity-Verlet;
  * the time-averaged pressure of a long NPH run equals P_ext, and the NPT run also holds kT.
"""
from __future__ import annotations

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import oracle as orc
from workloads import make_config, make_random_box


def kg_small(integrator="nph", p_ext=5.0, piston_mass=0.01, dt=0.005):
    w = make_config("C1", scale=0.5)            # 200-bead WCA + FENE melt
    w.integrator = integrator
    w.dt = dt
    w.p_ext = p_ext
    w.piston_mass = piston_mass
    return w


def lj_small(integrator="nph", p_ext=0.5, piston_mass=0.002, dt=0.004, gamma=0.0, kT=1.2):
    w = make_config("F4LJ", n=216)              # LJ liquid of the paper's Fig. 4 recipe, 6^3 beads, r_c = 3.0
    w.integrator = integrator
    w.dt = dt
    w.p_ext = p_ext
    w.piston_mass = piston_mass
    w.gamma = gamma
    w.kT = kT
    return w


def test_virial_is_minus_the_scaling_derivative_of_the_energy():
    for w in (kg_small(), lj_small()):
        o = orc.Oracle(w, use_cells=False)
        W = o.virial()
        pos0, box0 = o.pos.copy(), o.box.copy()
        h = 1e-6            # small: with a larger step pairs cross the cutoff, where the truncated force jumps
        u = []
        for s in (1.0 + h, 1.0 - h):
            o.set_box(box0 * s)
            a, b, _ = o.pair_bond_forces(pos=pos0 * s)[1:]
            u.append(a + b)
        dU_dlns = (u[0] - u[1]) / (2.0 * h)
        assert abs(W + dU_dlns) <= 1e-7 * max(1.0, abs(W)), (W, dU_dlns)
        assert abs(W) > 1.0


def test_angle_and_dihedral_energies_are_scale_free():
    # orc_virial leaves angles and dihedrals out: their energy must not change when coordinates and box are scaled
    from tests.test_gpu_topo import with_topology
    w = with_topology(kg_small(), "harmonic")
    w.pair_style = "none"
    w.bond_style = "none"
    o = orc.Oracle(w, use_cells=False)
    u0 = o.pair_bond_forces()[2]
    assert abs(u0) > 1.0
    pos0, box0 = o.pos.copy(), o.box.copy()
    o.set_box(box0 * 1.07)
    assert o.pair_bond_forces(pos=pos0 * 1.07)[2] == pytest.approx(u0, rel=1e-12)
    assert o.virial(pos0 * 1.07) == 0.0


def ideal_gas(n=64, box=6.0, p_ext=0.7, piston_mass=0.02, dt=0.01):
    w = make_random_box(n, [box] * 3, seed=3)
    w.pair_style = "none"
    w.integrator = "nph"
    w.dt = dt
    w.p_ext = p_ext
    w.piston_mass = piston_mass
    return w


def test_ideal_gas_piston_follows_its_ode_at_second_order():
    t_end = 2.0
    errs = []
    for dt in (0.02, 0.01):
        w = ideal_gas(dt=dt)
        o = orc.Oracle(w)
        k0, v0 = o.kinetic(), o.volume()
        m, p = float(np.float32(w.piston_mass)), float(np.float32(w.p_ext))
        dt32 = float(np.float32(dt))
        n_steps = int(round(t_end / dt))
        o.compute_forces()
        o.run(n_steps)
        sol = solve_ivp(lambda t, y: [y[1], (2.0 * k0 * (v0 / y[0]) ** (2.0 / 3.0) / (3.0 * y[0]) - p) / m],
                        [0.0, n_steps * dt32], [v0, 0.0], rtol=1e-12, atol=1e-12)
        v_ref, vdot_ref = sol.y[0, -1], sol.y[1, -1]
        assert abs(v_ref - v0) > 0.05 * v0                       # the piston really moved
        errs.append(abs(o.volume() - v_ref))
        assert abs(o.volume() - v_ref) < 2e-3 * v0
        assert abs(o.baro[2] / m - vdot_ref) < 2e-3 * abs(v0)
        # adiabatic invariant of the ideal gas under the piston
        assert o.kinetic() * o.volume() ** (2.0 / 3.0) == pytest.approx(k0 * v0 ** (2.0 / 3.0), rel=1e-12)
    assert 3.0 < errs[0] / errs[1] < 5.0, errs                   # second order


def test_ideal_gas_rests_where_the_pressures_balance():
    w = ideal_gas()
    o = orc.Oracle(w)
    o.baro[0] = 2.0 * o.kinetic() / (3.0 * o.volume())
    v0 = o.volume()
    o.compute_forces()
    o.run(200)
    assert o.volume() == pytest.approx(v0, rel=1e-12)
    assert abs(o.baro[2]) < 1e-12


def test_conserved_quantity_fluctuation_falls_as_dt_squared():
    spans = []
    for dt in (0.004, 0.002):
        w = kg_small(dt=dt)
        o = orc.Oracle(w, use_cells=False)
        o.compute_forces()
        h = [o.enthalpy_like()]
        for _ in range(int(round(0.4 / dt)) // 10):
            o.run(10)
            h.append(o.enthalpy_like())
        h = np.array(h)
        spans.append(h.max() - h.min())
        assert abs(o.volume() / np.prod(w.box.astype(np.float64)) - 1.0) > 1e-3      # the box moved
        assert spans[-1] < 2e-3 * abs(o.kinetic())
    assert 2.5 < spans[0] / spans[1] < 6.0, spans


def test_time_reversal():
    w = lj_small()
    o = orc.Oracle(w, use_cells=False)
    pos0, vel0, box0 = o.pos.copy(), o.vel.copy(), o.box.copy()
    o.compute_forces()
    o.run(50)
    assert np.abs(o.box / box0 - 1.0).max() > 1e-4
    o.vel *= -1.0
    o.baro[2] *= -1.0
    o.run(50)
    d = o.pos - pos0
    d -= o.box * np.rint(d / o.box)
    assert np.abs(d).max() < 1e-9
    np.testing.assert_allclose(o.vel, -vel0, atol=1e-9)
    np.testing.assert_allclose(o.box, box0, rtol=1e-12)
    assert abs(o.baro[2]) < 1e-9


def test_infinite_piston_mass_is_velocity_verlet():
    w = kg_small(piston_mass=1e30)
    a = orc.Oracle(w, use_cells=False)
    w2 = kg_small()
    w2.integrator = "nve"
    b = orc.Oracle(w2, use_cells=False)
    for o in (a, b):
        o.compute_forces()
        o.run(40)
    np.testing.assert_allclose(a.pos, b.pos, atol=1e-12)
    np.testing.assert_allclose(a.vel, b.vel, atol=1e-12)


def test_mean_pressure_equals_the_external_pressure_and_npt_holds_kt():
    # NPH: the time average of (2K + W) / 3V over many piston periods is P_ext (virial theorem for the piston coordinate)
    w = lj_small(p_ext=1.0)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    o.run(500)
    ps = []
    for _ in range(300):
        o.run(10)
        ps.append(o.pressure())
    assert np.mean(ps) == pytest.approx(1.0, abs=0.06), np.mean(ps)
    # NPT: Andersen collisions at nu = 5 hold kT = 1.2 (temperature of the full-step velocities, 3N degrees of freedom)
    w = lj_small(integrator="npt", p_ext=1.0, gamma=5.0, kT=1.2)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    o.run(500)
    ts, ps = [], []
    for _ in range(300):
        o.run(10)
        ts.append(2.0 * o.kinetic() / (3 * o.n))
        ps.append(o.pressure())
    assert np.mean(ts) == pytest.approx(1.2, rel=0.03), np.mean(ts)
    assert np.mean(ps) == pytest.approx(1.0, abs=0.08), np.mean(ps)
