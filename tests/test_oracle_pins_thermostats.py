"""Pins of the oracle's NVT thermostats (PAPER.md:L133, L137 names Nose-Hoover, Andersen and Berendsen; the equations
are readings c-28..c-30 of DESIGN.md): closed forms on the ideal gas, where each scheme has one
-- Berendsen: the half-step temperature relaxes geometrically, (T - kT) <- (1 - gamma dt)(T - kT); Nose-Hoover: small
oscillations of (T, xi) at omega = sqrt(2) gamma; Andersen: collision frequency, Maxwell statistics, exact replacement --
and, on an interacting fluid, the run-averaged temperature and the conserved extended energy of Nose-Hoover."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom
from workloads import make_random_box, maxwell_velocities


def ideal_gas(n, kT0, integrator, gamma, kT, dt=0.005, seed=3):
    w = make_random_box(n, (12.0, 12.0, 12.0), seed=seed, kT=kT0)
    w.pair_style = "none"; w.integrator = integrator; w.gamma = gamma; w.kT = kT; w.dt = dt
    o = orc.Oracle(w, use_cells=False)
    o.P.dt = dt; o.P.gamma = gamma; o.P.kT = kT
    o.compute_forces()
    return o


def test_berendsen_ideal_gas_relaxes_geometrically():
    # lambda^2 = 1 + gamma dt (kT / T - 1)  =>  T' = T + gamma dt (kT - T): closed form of the recursion
    kT, g, dt, n = 1.0, 2.0, 0.005, 5000
    o = ideal_gas(n, 3.0, "berendsen", g, kT, dt)
    T0 = o.temperature()                                   # exactly 3.0 by construction (3N - 3 dof)
    o.run(1)                                               # first step: thermostat off, half-step velocity created
    assert 2.0 * o.thermo[1] / (3 * n - 3) == pytest.approx(T0, rel=1e-12)
    o.run(200)
    T_half = 2.0 * o.thermo[1] / (3 * n - 3)
    assert T_half == pytest.approx(kT + (T0 - kT) * (1.0 - g * dt) ** 200, rel=1e-10)
    assert o.temperature() == pytest.approx(T_half, rel=1e-12)      # no forces: full-step = half-step velocity


def test_nose_hoover_ideal_gas_small_oscillation_and_conserved_quantity():
    # ideal gas: dT/dt = -2 xi T, dxi/dt = gamma^2 (T / kT - 1): linearised around T = kT, omega = sqrt(2) gamma
    kT, g, dt, n = 1.0, 3.0, 0.002, 4000
    o = ideal_gas(n, 1.02, "nose_hoover", g, kT, dt)
    dof = 3 * n - 3
    xs, hs, eta = [], [], 0.0
    for _ in range(3000):
        o.run(1)
        xi = o.thermo[2]
        eta += xi * dt
        xs.append(xi)
        hs.append(o.thermo[1] + 0.5 * dof * kT / g ** 2 * xi ** 2 + dof * kT * eta)
    xs = np.array(xs)
    up = np.nonzero((xs[:-1] < 0) & (xs[1:] >= 0))[0]                  # upward zero crossings of xi
    period = np.diff(up).mean() * dt
    assert period == pytest.approx(2.0 * math.pi / (math.sqrt(2.0) * g), rel=0.01)
    hs = np.array(hs[10:])
    assert np.abs(hs - hs.mean()).max() <= 2e-4 * dof * kT            # extended energy (leapfrog: half-step KE, O(dt) offsets)


def test_andersen_statistics_and_exact_replacement():
    seed, nu_dt = 77, 0.05
    hits = sum(orc.lib().orc_andersen_hit(seed, 5, t, nu_dt) for t in range(40000))
    assert hits / 40000 == pytest.approx(math.floor(nu_dt * 2 ** 24) / 2 ** 24, abs=4 * math.sqrt(0.05 * 0.95 / 40000))
    g = np.zeros((20000, 3))
    for t in range(20000):
        out = np.zeros(3)
        orc.lib().orc_andersen_normals(seed, 9, t, out.ctypes.data)
        g[t] = out
    assert np.abs(g.mean(axis=0)).max() < 0.03 and np.abs(g.var(axis=0) - 1.0).max() < 0.04
    assert np.abs(np.corrcoef(g.T) - np.eye(3)).max() < 0.03
    assert ((g ** 4).mean() / 3.0) == pytest.approx(1.0, abs=0.06)       # Gaussian fourth moment
    # nu dt = 1: every bead is replaced in every kick: u = sqrt(kT / m) g(tag, step), whatever it was before
    o = ideal_gas(50, 2.0, "andersen", 200.0, 0.7, dt=0.005)
    o.mass[:] = np.linspace(0.5, 2.0, 50)
    o.run(3)                                               # kicks of time levels 0, 1, 2
    for t in (0, 7, 49):
        out = np.zeros(3)
        orc.lib().orc_andersen_normals(int(o.w.seed), 2, t, out.ctypes.data)
        assert np.allclose(o.vel[t], math.sqrt(0.7 / o.mass[t]) * out, rtol=1e-12)


@pytest.mark.parametrize("integrator,gamma", [("nose_hoover", 2.0), ("andersen", 5.0), ("berendsen", 2.0)])
def test_thermostats_hold_the_temperature_of_an_lj_fluid(integrator, gamma):
    rng = np.random.default_rng(2)
    n_side, rho = 9, 0.6
    L = (n_side ** 3 / rho) ** (1.0 / 3.0)
    g = (np.arange(n_side) + 0.5) * L / n_side - L / 2
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    vel = maxwell_velocities(rng, len(pos), 2.0, np.ones(len(pos), np.float32))     # starts hot
    w = custom(pos, L, vel=vel, pair_style="lj", rc=2.5, integrator=integrator, dt=0.004, kT=1.2, gamma=gamma)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    o.run(1500)
    Ts = []
    for _ in range(100):
        o.run(25)
        Ts.append(o.temperature())
    # 729 beads: one reading scatters by 3 %, the mean of 100 readings by < 0.5 %; Berendsen/NH half-step vs full-step
    # temperature differ by O(dt^2)
    assert np.mean(Ts) == pytest.approx(1.2, rel=0.02)
