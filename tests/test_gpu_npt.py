"""f3, Andersen barostat on the GPU (NPH and NPT, reading c-31) against the fp64 oracle.

Tolerances: forces 1e-4 of the RMS force, positions after 10 steps 1e-4 sigma (the bars of the fixed-box tests), volume and
piston momentum 1e-5 relative; statistics (pressure, temperature, drift of Andersen's H) as stated per test.
"""
from __future__ import annotations

import numpy as np
import pytest

from oracle import oracle as orc
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


def with_barostat(w, integrator, p_ext, piston_mass, dt=None, gamma=None, kT=None):
    w.integrator = integrator
    w.p_ext = p_ext
    w.piston_mass = piston_mass
    if dt is not None:
        w.dt = dt
    if gamma is not None:
        w.gamma = gamma
    if kT is not None:
        w.kT = kT
    return w


def kg(scale, **kw):
    return with_barostat(make_config("C1", scale=scale), **kw)


def lj(n, **kw):
    return with_barostat(make_config("F4LJ", n=n), **kw)


def compare_state(s, o, tol_pos=1e-4, positions_only=False):
    pos, vel, frc = s.get_particles(True, True, True)
    b = s.box_state()
    np.testing.assert_allclose(b["box"], o.box, rtol=1e-5)
    d = pos.astype(np.float64) - o.pos
    d -= o.box * np.rint(d / o.box)
    rms = np.sqrt((d * d).sum(axis=1).mean())
    assert rms <= tol_pos, f"RMS position difference {rms:.3e}"
    assert b["volume"] == pytest.approx(o.volume(), rel=1e-5)
    if positions_only:
        return
    assert np.sqrt(((vel - o.vel) ** 2).sum(axis=1).mean()) <= 10 * tol_pos
    frms = np.sqrt((o.frc ** 2).sum(axis=1).mean())
    assert np.abs(frc - o.frc).max() <= 2e-3 * frms            # after chaotic amplification of 1e-4 position differences
    assert b["volume"] == pytest.approx(o.volume(), rel=1e-5)
    assert b["piston_momentum"] == pytest.approx(o.baro[2], rel=1e-3, abs=1e-4)
    assert b["virial"] == pytest.approx(o.virial(), rel=2e-3, abs=1e-2 * frms)
    assert b["pressure"] == pytest.approx(o.pressure(), rel=2e-3, abs=1e-3)


def test_forces_virial_and_energies_at_the_start(gm):
    for w in (kg(1.0, integrator="nph", p_ext=5.0, piston_mass=0.01), lj(1000, integrator="nph", p_ext=1.0, piston_mass=0.002)):
        s = gm.System(w)
        o = orc.Oracle(w, use_cells=True)
        o.compute_forces()
        pos, vel, frc = s.get_particles(True, True, True)
        np.testing.assert_array_equal(pos, w.pos)
        frms = np.sqrt((o.frc ** 2).sum(axis=1).mean())
        assert np.abs(frc - o.frc).max() <= 1e-4 * frms
        b = s.box_state()
        e = s.energies()
        pp, pb, _ = o.potential()
        assert b["virial"] == pytest.approx(o.virial(), rel=1e-5)
        assert b["pressure"] == pytest.approx(o.pressure(), rel=1e-5)
        assert e["ke"] == pytest.approx(o.kinetic(), rel=1e-6)
        assert e["pe_pair"] == pytest.approx(pp, rel=1e-5, abs=1e-3)
        assert e["pe_bond"] == pytest.approx(pb, rel=1e-5, abs=1e-3)
        assert b["H"] == pytest.approx(o.enthalpy_like(), rel=1e-5)
        assert b["volume"] == pytest.approx(o.volume(), rel=1e-7)
        s.close()


@pytest.mark.parametrize("integrator", ["nph", "npt"])
def test_trajectory_kg_melt(gm, integrator):
    w = kg(1.0, integrator=integrator, p_ext=5.0, piston_mass=0.01, gamma=2.0)
    s = gm.System(w)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    s.step(10)
    o.run(10)
    assert abs(o.volume() / float(np.prod(w.box.astype(np.float64))) - 1.0) > 1e-4       # the box moved
    compare_state(s, o)
    s.step(30)                  # spans neighbor rebuilds; chaos amplifies the round-off: statistics only
    o.run(30)
    b = s.box_state()
    assert b["volume"] == pytest.approx(o.volume(), rel=2e-3)
    assert s.stats()["rebuilds"] >= 2
    s.close()


def test_trajectory_lj_liquid_two_types_free_box(gm):
    w = lj(1000, integrator="nph", p_ext=0.3, piston_mass=0.002)
    w.n_types = 2                                   # two bead types with their own epsilon (the multi-type pair path)
    w.type = (np.arange(w.n) % 2).astype(np.int32)
    w.pair = dict(eps=np.array([[1.0, 0.8], [0.8, 1.2]], np.float32), sigma=np.ones((2, 2), np.float32),
                  rc=np.full((2, 2), 3.0, np.float32), shift=True)
    s = gm.System(w)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    s.step(10)
    o.run(10)
    compare_state(s, o)
    s.close()


def test_conserved_quantity_and_mean_pressure_long_run(gm):
    w = kg(2.0, integrator="nph", p_ext=5.0, piston_mass=1e-4)          # 17 560 beads, WCA + FENE
    s = gm.System(w)
    h0 = s.box_state()["H"]
    ke0 = s.energies()["ke"]
    s.step(500)
    ps, hs, vs = [], [], []
    for _ in range(150):
        s.step(20)
        b = s.box_state()
        ps.append(b["pressure"]); hs.append(b["H"]); vs.append(b["volume"])
    assert np.mean(ps) == pytest.approx(5.0, abs=0.1), np.mean(ps)
    # Andersen's H: no drift over the 3 000 sampled steps (spread below 1e-3 of the kinetic energy), and within 4e-3 of its
    # starting value (the lattice start, with its large first forces, shifts it once while the melt relaxes)
    assert max(hs) - min(hs) < 1e-3 * ke0, (h0, min(hs), max(hs))
    assert abs(np.mean(hs) - h0) < 4e-3 * ke0, (h0, np.mean(hs))
    assert np.std(vs) > 1e-4 * np.mean(vs)
    s.close()


def test_npt_holds_temperature_and_pressure(gm):
    w = kg(2.0, integrator="npt", p_ext=5.0, piston_mass=1e-4, gamma=5.0, kT=1.2)
    s = gm.System(w)
    s.step(600)
    ts, ps = [], []
    for _ in range(100):
        s.step(20)
        ts.append(s.energies()["T"]); ps.append(s.box_state()["pressure"])
    assert np.mean(ts) == pytest.approx(1.2, rel=0.02), np.mean(ts)
    assert np.mean(ps) == pytest.approx(5.0, abs=0.12), np.mean(ps)
    s.close()


def test_restart_from_box_state_and_errors(gm):
    w = kg(1.0, integrator="nph", p_ext=5.0, piston_mass=0.01)
    a = gm.System(w)
    a.step(24)
    pos, vel, _ = a.get_particles(True, True, False)
    ba = a.box_state()
    a.step(6)
    pa = a.get_particles(True, False, False)[0]
    # restart: same configuration, box state first, then the particles in the box of that volume
    b = gm.System(w, load=False)
    b.set_box_state(ba["volume"], ba["piston_momentum"])
    b.set_particles(pos, vel, w.type, w.mass)
    gm.gm_set_bonds(b.h, np.ascontiguousarray(w.bonds, np.int32), np.ascontiguousarray(w.bond_type, np.int32))
    bb = b.box_state()
    assert bb["volume"] == pytest.approx(ba["volume"], rel=1e-12)
    assert bb["pressure"] == pytest.approx(ba["pressure"], rel=1e-4)
    b.step(6)
    pb = b.get_particles(True, False, False)[0]
    d = pa - pb
    box = b.box_state()["box"]
    d -= box * np.rint(d / box)
    assert np.sqrt((d * d).sum(axis=1).mean()) < 1e-4
    with pytest.raises(gm.GmError):
        b.set_box_state(100.0, 0.0)                 # after gm_set_particles
    with pytest.raises(gm.GmError):
        b.set_integrator("nve")                     # a system under the barostat stays under it
    a.close(); b.close()
    # a window-staged system cannot be switched to the barostat
    w2 = make_config("C2", scale=0.5)
    c = gm.System(w2)
    if c.tuning()["windows"]:
        with pytest.raises(gm.GmError):
            c.set_integrator("nph")
    c.close()


def test_box_that_shrinks_past_the_list_radius_is_reported(gm):
    w = kg(1.0, integrator="nph", p_ext=400.0, piston_mass=0.0002)
    s = gm.System(w)
    with pytest.raises(gm.GmError):
        for _ in range(50):
            s.step(20)
            s.stats()
    s.close()


def test_trajectory_with_angles_and_dihedrals(gm):
    # angle and dihedral energies are scale-free: forces divide by the scale factor, the virial gets nothing from them
    from tests.test_gpu_topo import with_topology
    w = with_topology(kg(1.0, integrator="nph", p_ext=5.0, piston_mass=0.01), "cosine")
    s = gm.System(w)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    e = s.energies()
    pp, pb, _ = o.potential()
    assert e["pe_bond"] == pytest.approx(pb, rel=1e-5)
    assert s.box_state()["virial"] == pytest.approx(o.virial(), rel=1e-5)
    s.step(10)
    o.run(10)
    # the straight chains of the start make the dihedral forces ill-conditioned (as in test_gpu_topo): positions and box only
    compare_state(s, o, positions_only=True)
    s.close()
