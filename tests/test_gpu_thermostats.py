"""GPU-vs-oracle parity of the NVT thermostats (DESIGN.md readings
c-28..c-30): 10-step trajectories (the thermostat scale factors come from a global kinetic-energy sum, identical noise keys
for Andersen), the closed-form Berendsen relaxation on the ideal gas, and run-averaged temperatures."""
import numpy as np
import pytest

from oracle import oracle as orc
from tests.test_gpu_parity import trajectory_parity
from workloads import make_config, make_random_box

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1310_2041_b200 import gm as g
    g.lib()
    return g


@pytest.mark.parametrize("integrator,gamma", [("nose_hoover", 2.0), ("berendsen", 2.0), ("andersen", 10.0)])
def test_thermostat_trajectories_c1_and_c3_scaled(gm, integrator, gamma):
    for w in (make_config("C1"), make_config("C3", scale=0.3)):
        w.integrator = integrator; w.gamma = gamma; w.kT = 1.3; w.equil_steps = 0
        trajectory_parity(gm, w, n_steps=10)
        trajectory_parity(gm, w, n_steps=40, tol=2e-3)          # across rebuilds; fp32/fp64 paths have started to part


def test_berendsen_ideal_gas_closed_form_on_the_gpu(gm):
    # (T_half - kT) <- (1 - gamma dt)(T_half - kT) per step, exactly (tests/test_oracle_pins_thermostats.py)
    n, kT, g, dt = 20000, 1.0, 2.0, 0.005
    w = make_random_box(n, (30.0, 30.0, 30.0), seed=3, kT=3.0)
    w.pair_style = "none"; w.integrator = "berendsen"; w.gamma = g; w.kT = kT; w.dt = dt
    s = gm.System(w)
    s.step(201)                                                 # the first kick runs without the thermostat
    T = s.energies()["T"]
    assert T == pytest.approx(kT + (3.0 - kT) * (1.0 - g * dt) ** 200, rel=2e-5)
    s.close()


@pytest.mark.parametrize("integrator,gamma", [("nose_hoover", 2.0), ("berendsen", 2.0), ("andersen", 5.0)])
def test_thermostats_hold_the_temperature_c3_scaled(gm, integrator, gamma):
    w = make_config("C3", scale=0.3)                            # 27,000 beads
    w.integrator = integrator; w.gamma = gamma; w.kT = 1.2; w.equil_steps = 0
    s = gm.System(w)
    s.step(600)
    Tg = []
    for _ in range(20):                                         # the same window on both sides (the melt is still relaxing
        s.step(20)                                              # from its lattice start: compared like with like)
        Tg.append(s.energies()["T"])
    s.step(1000)
    Ts = []
    for _ in range(40):
        s.step(25)
        Ts.append(s.energies()["T"])
    s.close()
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    o.run(600)
    To = []
    for _ in range(20):
        o.run(20)
        To.append(o.temperature())
    assert np.mean(Tg) == pytest.approx(np.mean(To), rel=0.01)
    assert np.mean(Ts) == pytest.approx(1.2, rel=0.01)          # one reading of 27,000 beads scatters by 0.5 %
