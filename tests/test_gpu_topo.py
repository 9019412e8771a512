"""GPU-vs-oracle parity of angle and dihedral forces from per-particle tables (PAPER.md:L97,
Eqs. (8)-(10) L103-114): a bead-spring melt (config C1 and a scaled C3) with an angle on every consecutive bead triple
and a dihedral on every quadruple of each chain.  Same gates as everywhere: max |dF| <= 1e-4 F_rms, energies to 1e-5,
RMS position difference <= 1e-4 sigma after 10 steps, and a 40-step run across several rebuilds (the tables stay in tag
order while the beads are re-sorted)."""
import numpy as np
import pytest

from tests.test_gpu_parity import forces_parity, trajectory_parity
from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1310_2041_b200 import gm as g
    g.lib()
    return g


def with_topology(w, angle_style, dihedrals=True):
    n, L = w.n, w.chain_len
    k = np.arange(n)
    a0 = k[(k % L) <= L - 3]
    ang = np.stack([a0, a0 + 1, a0 + 2], axis=1)
    topo = dict(angle_style=angle_style, angles=ang, angle_type=(a0 % 2).astype(np.int32), angle_k=[3.0, 5.0],
                angle_t0=[2.0, 2.6])
    if dihedrals:
        d0 = k[(k % L) <= L - 4]
        topo.update(dihedrals=np.stack([d0, d0 + 1, d0 + 2, d0 + 3], axis=1), dihedral_type=(d0 % 2).astype(np.int32),
                    dihedral_k=[1.5, 0.7], dihedral_n=[1, 3], dihedral_delta=[0.4, -1.1])
    w.topo = topo
    return w


@pytest.mark.parametrize("style", ["harmonic", "cosine"])
def test_angles_and_dihedrals_forces_c1(gm, style):
    # the folded-lattice start has right angles and straight runs: theta = pi/2 and pi, phi = 0, +-pi/2, pi (jittered)
    forces_parity(gm, with_topology(make_config("C1"), style))
    forces_parity(gm, with_topology(make_config("C1"), style), steps_before=30)      # after the chains have moved


def trajectory_after(gm, w, steps_before, n_steps=10, tol=1e-4):
    """n_steps of both sides from the state the GPU reached after steps_before steps (full-step velocities handed to
    the oracle: for NVE the half-kick the library completes them with is the same arithmetic as the oracle's)."""
    from oracle import oracle as orc
    s = gm.System(w)
    o = orc.Oracle(w)
    s.step(steps_before)
    pos, vel, _ = s.get_particles(True, True, False)
    o.pos[:] = pos; o.vel[:] = vel; o.step = steps_before
    o.compute_forces()
    s.step(n_steps)
    o.run(n_steps)
    pos = s.get_particles(True, False, False)[0]
    d = pos.astype(np.float64) - o.pos
    d -= o.box * np.rint(d / o.box)
    rms = np.sqrt((d ** 2).sum(axis=1).mean())
    assert rms <= tol, f"RMS position difference after {n_steps} steps = {rms:.3e} sigma"
    s.close()


def test_angles_only_cosine_trajectory_and_rebuilds(gm):
    w = with_topology(make_config("C1"), "cosine", dihedrals=False)
    trajectory_parity(gm, w)
    forces_parity(gm, w, steps_before=40)


def test_angles_and_dihedrals_trajectory_c3_scaled(gm):
    w = with_topology(make_config("C3", scale=0.3), "harmonic")       # 27,000 beads, chains of 100
    w.integrator = "nve"; w.equil_steps = 0
    forces_parity(gm, w, steps_before=40)                             # several rebuilds (SFC sorts) in between
    # the folded-lattice start holds hundreds of nearly straight triples, where the dihedral force ~ 1 / sin(theta) is
    # ill-conditioned (an fp32 and an fp64 trajectory part within a few steps whatever the code): the 10-step gate is
    # taken from the state after 60 steps, when the angle terms have bent the chains
    trajectory_after(gm, w, 60)


# ---- tabulated angle and torsion potentials (Eq. (12) with x = theta, phi) -----------------------
def test_tabulated_angles_and_dihedrals_forces_and_trajectory(gm):
    from tests.test_oracle_pins_topotable import melt_with_tables
    w, wt = melt_with_tables(n_point=2000)                 # C1 scaled by 0.5 with Eq. (8) / Eq. (10) given as tables
    forces_parity(gm, wt, steps_before=25)
    trajectory_parity(gm, wt, n_steps=10)
    # against the analytic kernels on the same state: spline error of 2 000 intervals + fp32
    a, b = gm.System(w), gm.System(wt)
    a.step(25); b.step(25)
    fa = a.get_particles(False, False, True)[2]
    fb = b.get_particles(False, False, True)[2]
    frms = np.sqrt((fa.astype(np.float64) ** 2).sum(axis=1).mean())
    assert np.abs(fa - fb).max() <= 5e-3 * frms            # two fp32 trajectories of 25 steps apart + the spline
    ea, eb = a.energies(), b.energies()
    assert eb["pe_bond"] == pytest.approx(ea["pe_bond"], rel=1e-4)
    a.close(); b.close()
    # configuration errors
    c = gm.System(w)
    with pytest.raises(gm.GmError):
        gm.gm_set_angle_table(c.h, 0, np.zeros((16, 4), np.float32))
    with pytest.raises(gm.GmError):
        gm.gm_set_dihedral_table(c.h, 0, np.zeros((16, 4), np.float32))
    c.close()
