"""GPU-vs-oracle parity of the pair potentials beyond Lennard-Jones / DPD: harmonic
repulsion Eq. (2), Gaussian repulsion Eq. (3), the tabulated potential of Eqs. (11)-(12) /
Algorithm 2 (L118-129, L458), and the paper's own Fig. 4 benchmark liquids (L197).  Same gates as everywhere
(north_star): max |dF| <= 1e-4 F_rms on identical positions, RMS position difference <= 1e-4 sigma after 10 steps."""
import numpy as np
import pytest

from oracle import oracle as orc
from tests.test_gpu_parity import check_neighbor_sets, forces_parity, trajectory_parity
from tests.util import custom
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


def _soft_fluid(n, box, seed, n_types=2):
    w = make_random_box(n, box, seed=seed, n_types=n_types)
    w.pos[100:120] = w.pos[120:140]                       # coincident beads: r_ij = 0 (no force, finite energy)
    return w


def test_harmonic_repulsion_forces_and_trajectory(gm):
    b = _soft_fluid(6000, [12.0, 13.0, 14.0], 31)
    a = np.array([[25.0, 40.0], [40.0, 15.0]]); rc = np.array([[1.0, 1.2], [1.2, 0.9]])
    w = custom(b.pos, b.box, vel=b.vel, typ=b.type, pair_style="harmonic", a=a, rc=rc, dt=0.01, r_skin=0.3, n_types=2)
    forces_parity(gm, w)
    trajectory_parity(gm, w)


def test_gaussian_repulsion_forces_and_trajectory(gm):
    b = _soft_fluid(6000, [12.0, 13.0, 14.0], 32)
    eps = np.array([[3.0, 5.0], [5.0, 2.0]]); sig = np.array([[0.5, 0.6], [0.6, 0.7]]); rc = np.array([[1.5, 1.8], [1.8, 2.1]])
    for shift in (True, False):
        w = custom(b.pos, b.box, vel=b.vel, typ=b.type, pair_style="gauss", eps=eps, sigma=sig, rc=rc, shift=shift,
                   dt=0.01, r_skin=0.3, n_types=2)
        forces_parity(gm, w)
    trajectory_parity(gm, w)


def _lj_table(gm, n_point, r_cut, z_min, eps=1.0, sigma=1.0):
    """Lennard-Jones tabulated on a grid of z = r^2, fitted by the LIBRARY (gm_fit_pair_table); flat below z_min."""
    interval = r_cut * r_cut / n_point
    z = np.maximum(interval * np.arange(n_point + 1), z_min) / (sigma * sigma)
    return gm.gm_fit_pair_table(4.0 * eps * (z ** -6 - z ** -3), interval), float(np.float32(interval))


def test_tabulated_potential_matches_the_oracle_and_the_analytic_lj(gm):
    # one type, 4,000 grid points ("several thousands"), r_cut = 2.5; beads no closer than 0.9
    b = make_random_box(4000, [16.0, 17.0, 18.0], seed=33, min_sep=0.0)
    keep = np.ones(b.n, bool)                             # thin out close pairs (rejection on the oracle's pair list)
    for i, j in orc.neighbor_pairs(b.pos, b.box, 0.9, True):
        if keep[i] and keep[j]:
            keep[j] = False
    pos, vel = b.pos[keep], b.vel[keep]
    c, interval = _lj_table(gm, 4000, 2.5, 0.49)
    wt = custom(pos, b.box, vel=vel, pair_style="table", table=c[None, None], interval=interval, dt=0.002, r_skin=0.3)
    forces_parity(gm, wt)                                 # same fp32 coefficients on both sides
    trajectory_parity(gm, wt)
    # and against the analytic Eq. (1) on the GPU itself: the spline error bound of the pin (1e-4 of the largest force)
    s = gm.System(wt); s.compute_forces(); Ft = s.get_particles(False, False, True)[2]; s.close()
    wl = custom(pos, b.box, vel=vel, pair_style="lj", rc=2.5, shift=False, dt=0.002, r_skin=0.3)
    s = gm.System(wl); s.compute_forces(); Fl = s.get_particles(False, False, True)[2]; s.close()
    assert np.abs(Ft - Fl).max() <= 2e-4 * np.abs(Fl).max()


def test_tabulated_potential_two_types_neighbor_sets_and_forces(gm):
    b = make_random_box(5000, [14.0, 14.0, 15.0], seed=34, n_types=2)
    keep = np.ones(b.n, bool)
    for i, j in orc.neighbor_pairs(b.pos, b.box, 0.85, True):
        if keep[i] and keep[j]:
            keep[j] = False
    n_point = 2048
    c00, iv = _lj_table(gm, n_point, 2.0, 0.4)
    c01, _ = _lj_table(gm, n_point, 2.0, 0.4, eps=0.6, sigma=0.95)
    c11, _ = _lj_table(gm, n_point, 2.0, 0.4, eps=1.5, sigma=0.9)
    table = np.stack([np.stack([c00, c01]), np.stack([c01, c11])])
    w = custom(b.pos[keep], b.box, vel=b.vel[keep], typ=b.type[keep], pair_style="table", table=table, interval=iv,
               dt=0.002, r_skin=0.4, n_types=2)
    check_neighbor_sets(gm, w)
    forces_parity(gm, w)


def test_fig4_lj_liquid_scaled(gm):
    # the paper's LJ benchmark liquid (packing fraction 0.2, r_cut 3.0, dt 0.001), 30^3 = 27,000 beads
    w = make_config("F4LJ", n=27000)
    check_neighbor_sets(gm, w)
    forces_parity(gm, w, steps_before=20)
    trajectory_parity(gm, w)


def test_fig4_dpd_liquid_scaled(gm):
    # the paper's DPD benchmark liquid (rho 3, r_cut 1.0, dt 0.04), 30,000 beads, no bonds
    w = make_config("F4DPD", n=30000)
    check_neighbor_sets(gm, w)
    forces_parity(gm, w)          # at the start state: after steps the dissipative force sees v~, which the boundary does not return
    trajectory_parity(gm, w, n_steps=10)
