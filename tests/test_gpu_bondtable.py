"""GPU-vs-oracle parity of tabulated bond potentials (SURVEY.md 8(f) row f1 "tabulated pair/bond potentials"; PAPER.md:L118,
Eqs. (11)-(12) in z = r^2; reading c-32).  Gates as everywhere: max |dF| <= 1e-4 F_rms, energies 1e-5, RMS position
difference <= 1e-4 sigma after 10 steps; plus: a table that is linear in z gives the r0 = 0 harmonic bond's forces to fp32
round-off, a bond past the end of its table is reported, and the barostat path takes the same tables."""
import numpy as np
import pytest

from oracle import oracle as orc
from tests.test_gpu_parity import forces_parity, trajectory_parity
from tests.test_oracle_pins_bondtable import table_of
from tests.util import custom
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


def kg_with_tabulated_fene(name="C1", scale=None, two_types=False):
    """the Kremer-Grest melt of the config with its FENE bonds given as a table (4 000 grid points up to r = 1.45)"""
    w = make_config(name, scale=scale)
    k, R0 = float(w.bond["k"][0]), float(w.bond["r0"][0])
    fene = lambda r: -0.5 * k * R0 * R0 * np.log(np.maximum(1.0 - (r / R0) ** 2, 1e-12))
    tb0, h0 = table_of(fene, 1.45 ** 2, 4000)
    tables, hs = [tb0], [h0]
    if two_types:                                   # every other bond a stiff harmonic spring of the same length scale
        tb1, h1 = table_of(lambda r: 40.0 * (r - 0.97) ** 2, 1.6 ** 2, 4000)
        tables.append(tb1); hs.append(h1)
        w.bond_type = (np.arange(len(w.bonds)) % 2).astype(np.int32)
    w.bond_style = "table"
    w.bond = dict(table=np.stack(tables), interval=np.array(hs, np.float32), k=np.zeros(len(hs), np.float32),
                  r0=np.zeros(len(hs), np.float32))
    return w


def test_forces_and_energies_c1_tabulated_fene(gm):
    forces_parity(gm, kg_with_tabulated_fene("C1"))
    forces_parity(gm, kg_with_tabulated_fene("C1", two_types=True), steps_before=25)


def test_tabulated_fene_reproduces_the_analytic_fene_forces(gm):
    w = make_config("C1")
    a = gm.System(w)
    fa = a.get_particles(False, False, True)[2]
    a.close()
    b = gm.System(kg_with_tabulated_fene("C1"))
    fb = b.get_particles(False, False, True)[2]
    b.close()
    frms = np.sqrt((fa.astype(np.float64) ** 2).sum(axis=1).mean())
    assert np.abs(fa - fb).max() <= 2e-4 * frms                # spline error of 4 000 intervals + fp32


def test_trajectories_c1_and_c3_scaled(gm):
    trajectory_parity(gm, kg_with_tabulated_fene("C1", two_types=True))
    trajectory_parity(gm, kg_with_tabulated_fene("C3", scale=0.3), n_steps=10)


def test_linear_in_z_table_is_the_r0_zero_harmonic_bond(gm):
    k, n_point, h = 3.5, 64, np.float32(0.125)
    tb = np.zeros((n_point, 4), np.float32)
    tb[:, 0] = 0.75 + k * h * np.arange(n_point)
    tb[:, 1] = k
    rng = np.random.default_rng(3)
    pos = np.cumsum(rng.normal(0.0, 0.6, (64, 3)), axis=0)      # a random-walk chain: bonds of ~1, the longest well below 2.8
    bonds = np.stack([np.arange(63), np.arange(1, 64)], axis=1)
    wt = custom(pos, 30.0, bonds=bonds, pair_style="none", bond_style="table", bond_table=tb[None], bond_interval=[h])
    wh = custom(pos, 30.0, bonds=bonds, pair_style="none", bond_style="harmonic", k=k, r0=0.0)
    ft = gm.System(wt).get_particles(False, False, True)[2]
    fh = gm.System(wh).get_particles(False, False, True)[2]
    np.testing.assert_allclose(ft, fh, rtol=2e-6, atol=2e-6)


def test_bond_past_its_table_is_reported(gm):
    tb, h = table_of(lambda r: 5.0 * (r - 1.0) ** 2, 1.5 ** 2, 100)
    pos = np.array([[-0.8, 0.0, 0.0], [0.8, 0.0, 0.0], [0.8, 1.0, 0.0], [3.0, 3.0, 3.0]])
    w = custom(pos, 12.0, bonds=[[0, 1], [1, 2]], pair_style="none", bond_style="table", bond_table=tb[None], bond_interval=[h])
    s = gm.System(w)
    with pytest.raises(gm.GmError) as e:
        s.get_particles(False, False, True)
    assert e.value.status == -7                                 # GM_ERR_BOND_OVERSTRETCH
    s.close()
    # configuration errors: a table for a system without GM_BOND_TABLE, parameters for one with it
    c = gm.System(make_config("C1"))
    with pytest.raises(gm.GmError):
        gm.gm_set_bond_table(c.h, 0, 0.1, np.zeros((8, 4), np.float32))
    c.close()
    d = gm.System(kg_with_tabulated_fene("C1"))
    with pytest.raises(gm.GmError):
        gm.gm_set_bond_params(d.h, 0, 30.0, 1.5)
    d.close()


def test_barostat_takes_tabulated_bonds(gm):
    w = kg_with_tabulated_fene("C1")
    w.integrator, w.p_ext, w.piston_mass = "nph", 5.0, 0.01
    s = gm.System(w)
    o = orc.Oracle(w, use_cells=True)
    o.compute_forces()
    b = s.box_state()
    assert b["virial"] == pytest.approx(o.virial(), rel=1e-5)
    assert b["pressure"] == pytest.approx(o.pressure(), rel=1e-5)
    s.step(10)
    o.run(10)
    pos = s.get_particles(True, False, False)[0]
    d = pos.astype(np.float64) - o.pos
    d -= o.box * np.rint(d / o.box)
    assert np.sqrt((d * d).sum(axis=1).mean()) <= 1e-4
    assert s.box_state()["volume"] == pytest.approx(o.volume(), rel=1e-5)
    s.close()
