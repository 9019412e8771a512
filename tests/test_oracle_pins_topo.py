"""Pins of the oracle's angle potentials, Eqs. (8)-(9), and periodic dihedral, Eq. (10) (
SURVEY.md 8(f) row f2): closed-form energies on hand-placed beads (tests/golden/closed_forms.txt), force = -grad(energy)
by central differences, zero net force and zero net torque, invariance under rigid rotation and under the periodic
images, and the sign of the restoring force."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom


def G(golden):
    return {r[0]: float(r[1]) for r in golden("closed_forms.txt")}


def system(pos, topo, box=30.0):
    w = custom(pos, box, pair_style="none")
    w.topo = topo
    o = orc.Oracle(w, use_cells=False)
    o.pos[:] = np.asarray(pos, np.float64)
    return o


def bent(theta, l1=1.0, l2=1.3):
    """i - j - k with the angle theta at j (j at the origin, i on +x)."""
    return [[l1, 0, 0], [0, 0, 0], [l2 * math.cos(theta), l2 * math.sin(theta), 0]]


def torsion(phi):
    """i, j, k, l with j-k on the z axis and the dihedral phi (0 = cis)."""
    return [[1, 0, 0], [0, 0, 0], [0, 0, 1.2], [0.9 * math.cos(phi), 0.9 * math.sin(phi), 1.2]]


def test_angle_closed_forms(golden):
    g = G(golden)
    harm = dict(angle_style="harmonic", angles=[[0, 1, 2]], angle_k=[1.0], angle_t0=[math.pi])
    o = system(bent(math.pi / 2), harm); o._ang_t0[:] = math.pi
    assert o.pair_bond_forces()[2] == pytest.approx(g["angle_harm_u_90_vs_180"], rel=1e-14)
    o = system(bent(math.pi - 1e-7), harm); o._ang_t0[:] = math.pi         # straight chain: theta = pi, U -> 0
    assert o.pair_bond_forces()[2] < 1e-13
    cosn = dict(angle_style="cosine", angles=[[0, 1, 2]], angle_k=[1.0], angle_t0=[math.pi])
    o = system(bent(math.pi / 2), cosn); o._ang_t0[:] = math.pi
    assert o.pair_bond_forces()[2] == pytest.approx(g["angle_cos_u_90_vs_180"], rel=1e-14)
    cos2 = dict(angle_style="cosine", angles=[[0, 1, 2]], angle_k=[2.0], angle_t0=[2 * math.pi / 3])
    o = system(bent(math.pi / 3), cos2); o._ang_t0[:] = 2 * math.pi / 3
    assert o.pair_bond_forces()[2] == pytest.approx(g["angle_cos_u_60_vs_120"], rel=1e-13)
    # the force restores: at theta < theta0 bead k is pushed to larger angles (its tangential force is +theta direction)
    F = o.pair_bond_forces()[0]
    t_hat = np.array([-math.sin(math.pi / 3), math.cos(math.pi / 3), 0.0])
    assert F[2] @ t_hat > 0.1


def test_dihedral_closed_forms(golden):
    g = G(golden)
    d1 = dict(dihedrals=[[0, 1, 2, 3]], dihedral_k=[1.0], dihedral_n=[1], dihedral_delta=[0.0])
    assert system(torsion(0.0), d1).pair_bond_forces()[2] == pytest.approx(g["dihedral_u_cis_n1"], abs=1e-14)
    assert system(torsion(math.pi), d1).pair_bond_forces()[2] == pytest.approx(g["dihedral_u_trans_n1"], abs=1e-14)
    d3 = dict(dihedrals=[[0, 1, 2, 3]], dihedral_k=[3.0], dihedral_n=[3], dihedral_delta=[math.pi / 6])
    o = system(torsion(math.pi / 2), d3); o._dih_delta[:] = math.pi / 6
    assert o.pair_bond_forces()[2] == pytest.approx(g["dihedral_u_90_n3_d30"], rel=1e-13)
    # phi is odd under mirror reflection: U(phi; delta) = U(-phi; -delta)
    o2 = system(torsion(-math.pi / 2), dict(d3, dihedral_delta=[-math.pi / 6])); o2._dih_delta[:] = -math.pi / 6
    assert o2.pair_bond_forces()[2] == pytest.approx(g["dihedral_u_90_n3_d30"], rel=1e-13)


def _random_chain_topo(n, rng, angle_style):
    ang = np.array([[k, k + 1, k + 2] for k in range(n - 2)])
    dih = np.array([[k, k + 1, k + 2, k + 3] for k in range(n - 3)])
    return dict(angle_style=angle_style, angles=ang, angle_type=np.arange(len(ang)) % 2, angle_k=[3.0, 5.0],
                angle_t0=[2.0, 2.6], dihedrals=dih, dihedral_type=np.arange(len(dih)) % 2, dihedral_k=[1.5, 0.7],
                dihedral_n=[1, 3], dihedral_delta=[0.4, -1.1])


@pytest.mark.parametrize("style", ["harmonic", "cosine"])
def test_force_is_minus_gradient_net_force_and_torque_vanish(style):
    rng = np.random.default_rng(4)
    n = 24
    pos = np.cumsum(rng.normal(size=(n, 3)) * 0.6 + [0.5, 0, 0], axis=0)       # a kinked chain that leaves the box
    box = np.array([7.0, 8.0, 9.0])
    o = system(pos - box * np.floor(pos / box + 0.5), _random_chain_topo(n, rng, style), box=box)
    F, _, U, _ = o.pair_bond_forces()
    assert np.abs(F).max() > 0.5 and np.abs(F.sum(axis=0)).max() < 1e-11
    h = 1e-6
    for i in (0, 1, 5, 11, 22, 23):
        for d in range(3):
            p = o.pos.copy(); p[i, d] += h
            up = o.pair_bond_forces(pos=p)[2]
            p[i, d] -= 2 * h
            um = o.pair_bond_forces(pos=p)[2]
            assert F[i, d] == pytest.approx(-(up - um) / (2 * h), abs=2e-7 * max(1.0, np.abs(F).max()))
    # zero torque on the unwrapped chain, rotation invariance, periodic-image invariance
    o_un = system(pos, _random_chain_topo(n, rng, style), box=1000.0)
    Fu, _, Uu, _ = o_un.pair_bond_forces()
    assert Uu == pytest.approx(U, rel=1e-12) and np.abs(Fu - F).max() < 1e-10
    assert np.abs(np.cross(pos, Fu).sum(axis=0)).max() < 1e-9
    a = 0.7
    R = np.array([[math.cos(a), -math.sin(a), 0], [math.sin(a), math.cos(a), 0], [0, 0, 1.0]])
    o_rot = system(pos @ R.T, _random_chain_topo(n, rng, style), box=1000.0)
    Fr, _, Ur, _ = o_rot.pair_bond_forces()
    assert Ur == pytest.approx(Uu, rel=1e-12) and np.abs(Fr - Fu @ R.T).max() < 1e-10
