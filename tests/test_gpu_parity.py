"""GPU-vs-oracle parity through the C ABI (run with -m gpu on a B200).

Gates (BASELINE.json north_star):
  * neighbor sets bit-exact, pairs within 1e-6 sigma of r_list excluded;
  * per-bead forces on identical positions: max|dF| <= 1e-4 F_rms;
  * RMS position difference after 10 steps <= 1e-4 sigma;
  * energies (fp32 terms, fp64 sums) to 1e-5 relative.
The oracle gets exactly the fp32 inputs the GPU holds, promoted to fp64.
"""
import numpy as np
import pytest

from oracle import oracle as orc
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


def r_list_of(w):
    rc = float(np.max(w.pair["rc"])) if w.pair_style != "none" else 1.0
    return float(np.float32(rc)) + float(np.float32(w.r_skin))


def gpu_pair_set(nn, nl):
    out = set()
    for i in range(len(nn)):
        for j in nl[i, :nn[i]]:
            out.add((i, int(j)))
    return out


def check_neighbor_sets(gm, w, use_cells=True, tune=None):
    s = gm.System(w, tune=tune)
    s.build_neighbors()
    nn, nl = s.neighbors()
    st = s.stats()
    assert st["max_nn"] == nn.max() and st["sum_nn"] == nn.sum()
    pos = s.get_particles(True, False, False)[0]
    np.testing.assert_array_equal(pos, w.pos)               # identical positions on both sides
    rl = r_list_of(w)
    inner = orc.neighbor_pairs(w.pos, w.box, rl - 1e-6, use_cells)
    outer = orc.neighbor_pairs(w.pos, w.box, rl + 1e-6, use_cells)
    # GPU list is FULL: (i,j) and (j,i) both present, no self, no duplicates
    n = w.n
    rows = np.repeat(np.arange(n), nn)
    cols = np.concatenate([nl[i, :nn[i]] for i in range(n)]) if nn.sum() else np.zeros(0, np.int32)
    assert (rows != cols).all()
    key = rows.astype(np.int64) * n + cols
    assert len(np.unique(key)) == len(key)
    keyT = cols.astype(np.int64) * n + rows
    assert np.array_equal(np.sort(key), np.sort(keyT))
    half = key[rows < cols]
    k_in = inner[:, 0].astype(np.int64) * n + inner[:, 1]
    k_out = outer[:, 0].astype(np.int64) * n + outer[:, 1]
    assert np.isin(k_in, half).all(), "GPU list misses a pair inside r_list - 1e-6"
    assert np.isin(half, k_out).all(), "GPU list holds a pair outside r_list + 1e-6"
    s.close()
    return len(half)


def test_neighbor_sets_c1(gm):
    assert check_neighbor_sets(gm, make_config("C1"), use_cells=False) > 10000


def test_neighbor_sets_c2_scaled(gm):
    check_neighbor_sets(gm, make_config("C2", scale=0.5))      # 20^3 = 8000 beads, r_list 2.8


def test_neighbor_sets_c3_scaled_and_c4_scaled(gm):
    check_neighbor_sets(gm, make_config("C3", scale=0.3))      # 30^3 lattice, 27000 beads
    check_neighbor_sets(gm, make_config("C4", scale=0.12))     # DPD, 12^3 box, 5184 beads, two types


def test_neighbor_sets_noncubic_random_with_beads_on_faces(gm):
    w = make_random_box(3000, [9.0, 13.5, 17.25], seed=5)
    w.pos[:50, 0] = -4.5                                       # exactly on the lower face
    w.pos[50:100, 1] = np.nextafter(np.float32(6.75), np.float32(0))   # last value below the upper face
    w.pos[100:120] = w.pos[120:140]                            # coincident beads
    check_neighbor_sets(gm, w, use_cells=False)


def forces_parity(gm, w, steps_before=0, tol=1e-4, tune=None):
    s = gm.System(w, tune=tune)
    o = orc.Oracle(w)
    if steps_before:
        s.step(steps_before)
        pos, vel, _ = s.get_particles(True, True, False)
        o.pos[:] = pos; o.vel[:] = vel; o.step = steps_before
    s.compute_forces()
    _, _, F = s.get_particles(False, False, True)
    Fo = o.compute_forces().copy()
    assert o.status == 0
    frms = np.sqrt((Fo ** 2).sum(axis=1).mean())
    err = np.abs(F - Fo).max()
    assert err <= tol * frms, f"max|dF| = {err:.3e} > {tol} * F_rms = {tol * frms:.3e}"
    e = s.energies()
    assert e["pe_pair"] == pytest.approx(o.last[0], rel=1e-5, abs=1e-5 * w.n)
    assert e["pe_bond"] == pytest.approx(o.last[1], rel=1e-5, abs=1e-5 * w.n)
    assert e["n_pairs"] == o.last[2]
    if not steps_before:
        assert e["ke"] == pytest.approx(o.kinetic(), rel=1e-6)
        assert np.allclose(e["p"], o.momentum(), atol=1e-3)
    s.close()
    return frms


@pytest.mark.parametrize("xdiv,trip", [(1, 4), (2, 8), (3, 4), (4, 8), (8, 4)])
def test_cell_refinement_and_scan_width_do_not_change_the_list_or_the_forces(gm, xdiv, trip):
    # a3: cells r_list / sx wide in x and 4 or 8 candidates per trip are exact accelerations (DESIGN.md c-12);
    # the overrides are gm_config fields.  Non-cubic box with beads on the faces, then C1 forces.
    tune = dict(x_cell_div=xdiv, nl_scan_trip=trip)
    w = make_random_box(3000, [9.0, 13.5, 17.25], seed=6)
    w.pos[:50, 0] = -4.5                                       # exactly on the lower face
    w.pos[50:100, 1] = np.nextafter(np.float32(6.75), np.float32(0))   # last value below the upper face
    w.pos[100:120] = w.pos[120:140]                            # coincident beads
    check_neighbor_sets(gm, w, use_cells=False, tune=tune)
    forces_parity(gm, make_config("C1"), steps_before=12, tune=tune)


def test_forces_dense_dpd_exercises_the_early_drain_of_the_compaction_column(gm):
    # a6: rho = 9 puts ~38 partners inside r_c = 1, more than the 28 the compaction column holds before it
    # is drained (pair_loop_dpd); 2 types, harmonic bonds, velocities set so the dissipative term is live
    rng = np.random.default_rng(21)
    box, n = 7.0, 3087
    pos = rng.uniform(-0.5 * box, 0.5 * box, (n, 3)).astype(np.float32)
    vel = rng.normal(0, 1, (n, 3)).astype(np.float32)
    typ = (np.arange(n) % 2).astype(np.int32)
    bonds = np.stack([np.arange(0, n - 1, 3), np.arange(1, n, 3)], axis=1)
    w = custom(pos, box, vel=vel, typ=typ, bonds=bonds, pair_style="dpd", a=np.array([[25.0, 40.0], [40.0, 25.0]]),
               rc=1.0, bond_style="harmonic", k=4.0, r0=0.0, integrator="gwvv", dt=0.04, gamma=4.5, r_skin=0.3,
               n_types=2)
    forces_parity(gm, w)


def test_forces_c1_wca_fene(gm):
    forces_parity(gm, make_config("C1"))


def test_forces_c1_after_steps(gm):
    forces_parity(gm, make_config("C1"), steps_before=37)


def test_forces_c2_scaled_lj25_langevin(gm):
    forces_parity(gm, make_config("C2", scale=0.5))           # includes drag + Philox per-bead noise


def test_forces_c4_scaled_dpd(gm):
    forces_parity(gm, make_config("C4", scale=0.12))          # dissipative + Philox pair noise, 2 types


def test_forces_c3_scaled(gm):
    forces_parity(gm, make_config("C3", scale=0.3))


def test_forces_multitype_lj_noncubic(gm):
    w = make_random_box(2500, [11.0, 14.0, 12.5], seed=11, n_types=3, min_sep=0.85)
    rng = np.random.default_rng(3)
    eps = rng.uniform(0.5, 1.5, (3, 3)); eps = ((eps + eps.T) / 2).astype(np.float32)
    sig = rng.uniform(0.9, 1.1, (3, 3)); sig = ((sig + sig.T) / 2).astype(np.float32)
    rc = rng.uniform(1.5, 2.5, (3, 3)); rc = ((rc + rc.T) / 2).astype(np.float32)
    w.pair = dict(eps=eps, sigma=sig, rc=rc, shift=True)
    forces_parity(gm, w)


def trajectory_parity(gm, w, n_steps=10, tol=1e-4, **kw):
    s = gm.System(w, **kw)
    o = orc.Oracle(w)
    o.compute_forces()
    s.step(n_steps)
    o.run(n_steps)
    pos, vel, _ = s.get_particles(True, True, False)
    d = pos.astype(np.float64) - o.pos
    d -= o.box * np.rint(d / o.box)
    rms = np.sqrt((d ** 2).sum(axis=1).mean())
    assert rms <= tol, f"RMS position difference after {n_steps} steps = {rms:.3e} sigma"
    dv = np.sqrt(((vel - o.vel) ** 2).sum(axis=1).mean())
    assert dv <= 20 * tol, f"RMS velocity difference {dv:.3e}"
    assert s.stats()["steps"] == n_steps
    s.close()
    return rms


def test_trajectory_c1_nve(gm):
    trajectory_parity(gm, make_config("C1"))


def test_trajectory_c2_scaled_langevin(gm):
    trajectory_parity(gm, make_config("C2", scale=0.5))


def test_trajectory_c4_scaled_dpd_gwvv(gm):
    trajectory_parity(gm, make_config("C4", scale=0.12))


def test_trajectory_c3_scaled_with_reorders(gm):
    trajectory_parity(gm, make_config("C3", scale=0.3), sfc_period=3)


def test_trajectory_c1_40_steps_spans_rebuilds(gm):
    w = make_config("C1")
    s = gm.System(w)
    o = orc.Oracle(w)
    o.compute_forces()
    s.step(40); o.run(40)
    pos = s.get_particles(True, False, False)[0]
    d = pos - o.pos; d -= o.box * np.rint(d / o.box)
    assert np.sqrt((d ** 2).sum(axis=1).mean()) < 5e-4
    assert s.stats()["rebuilds"] >= 2
    s.close()


def test_subwarp_step_variant_matches_oracle(gm):
    """GM_FLAG_STEP_SUBWARP: 8 lanes per bead with a shuffle reduction (long-list variant)."""
    trajectory_parity(gm, make_config("C2", scale=0.5), flags=gm.GM_FLAG_STEP_SUBWARP)
    trajectory_parity(gm, make_config("C4", scale=0.12), flags=gm.GM_FLAG_STEP_SUBWARP)
    trajectory_parity(gm, make_config("C1"), flags=gm.GM_FLAG_STEP_SUBWARP)


def test_launch_modes_are_bit_identical(gm):
    """Direct launches, graphs with early-exit gating and graphs with conditional nodes run the
    same kernels on the same data: trajectories agree bit for bit (and so does a repeated run)."""
    w = make_config("C1")
    outs = []
    for flags in (gm.GM_FLAG_NO_GRAPH, gm.GM_FLAG_NO_COND_NODES, 0, 0):
        s = gm.System(w, flags=flags)
        s.step(1); s.step(100); s.step(3)
        outs.append(s.get_particles(True, True, False))
        st = s.stats()
        assert st["steps"] == 104 and st["rebuilds"] >= 3
        s.close()
    for p, v, _ in outs[1:]:
        np.testing.assert_array_equal(p, outs[0][0])
        np.testing.assert_array_equal(v, outs[0][1])


def test_rebuild_rule_keeps_every_interacting_pair_listed(gm):
    """Reading c-11: whatever the rebuild schedule, every pair inside r_cut is in the list."""
    w = make_config("C1")
    s = gm.System(w)
    rc = float(np.max(w.pair["rc"]))
    for _ in range(6):
        s.step(17)
        pos = s.get_particles(True, False, False)[0]
        nn, nl = s.neighbors()
        need = orc.neighbor_pairs(pos, w.box, rc, use_cells=True)
        have = gpu_pair_set(nn, nl)
        assert all((int(a), int(b)) in have for a, b in need)
    s.close()


def test_free_flight_rebuilds_when_and_only_when_half_skin_is_crossed(gm):
    """P10: no forces -> r(t) = wrap(r0 + v t); the first rebuild after the initial build happens at
    the first step whose displacement exceeds skin/2."""
    n = 64
    rng = np.random.default_rng(1)
    pos = rng.uniform(-5, 5, (n, 3)).astype(np.float32)
    vel = np.zeros((n, 3), np.float32)
    vel[7] = [1.0, 0, 0]                                       # |v| dt = 0.01 per step; skin/2 = 0.2
    w = custom(pos, 10.0, vel=vel, eps=0.0, rc=1.0, r_skin=0.4, dt=0.01)
    s = gm.System(w)
    s.step(19)                                                 # displacement 0.19 < skin/2: only the initial build
    assert s.stats()["rebuilds"] == 1
    s.step(4)                                                  # 0.21 at level 21 -> rebuilt before its forces
    assert s.stats()["rebuilds"] == 2
    s.step(200)
    p = s.get_particles(True, False, False)[0]
    x = pos[7, 0] + 1.0 * 0.01 * 223
    x -= 10.0 * np.floor((x + 5.0) / 10.0)
    assert abs(p[7, 0] - x) < 1e-4
    np.testing.assert_array_equal(np.delete(p, 7, axis=0), np.delete(pos, 7, axis=0))
    s.close()


def test_edge_cases(gm):
    # one bead: empty rows, zero force
    w = custom([[0.1, 0.2, 0.3]], 10.0, vel=[[1, 0, 0]])
    s = gm.System(w)
    s.compute_forces(); s.step(5)
    p, v, f = s.get_particles(True, True, True)
    assert np.allclose(p, [[0.125, 0.2, 0.3]], atol=1e-6) and np.abs(f).max() == 0
    assert s.stats()["max_nn"] == 0
    s.close()
    # a bonded dimer across the periodic boundary (minimum image for pair and bond)
    rc = 2.0 ** (1.0 / 6.0)
    w = custom([[4.7, 0, 0], [-4.4, 0, 0]], 10.0, rc=rc, bond_style="fene", bonds=[[0, 1]])
    s = gm.System(w)
    s.compute_forces()
    f = s.get_particles(False, False, True)[2]
    o = orc.Oracle(w, use_cells=False)
    fo = o.compute_forces()
    assert np.abs(f - fo).max() < 1e-4 * np.abs(fo).max() and abs(f[0, 0] + f[1, 0]) < 1e-4
    s.close()
    # FENE over-stretch is latched and reported
    w = custom([[0, 0, 0], [1.6, 0, 0]], 10.0, rc=rc, bond_style="fene", bonds=[[0, 1]])
    s = gm.System(w)
    s.compute_forces()
    assert s.stats(check=False)["status"] == gm.GM_ERR_BOND_OVERSTRETCH
    s.close()
    # neighbor row overflow is latched and reported
    w = make_random_box(1500, [9.0, 9.0, 9.0], seed=2)              # ~ 210 neighbors per bead at r_list 2.9
    s = gm.System(w, nl_row_capacity=8)
    s.build_neighbors()
    assert s.stats(check=False)["status"] == gm.GM_ERR_NEIGHBOR_OVERFLOW
    s.close()
    # call order
    s = gm.System(make_config("C1"), load=False)
    with pytest.raises(gm.GmError) as e:
        s.step(1)
    assert e.value.status == gm.GM_ERR_STATE
    s.close()


def test_device_resident_io_matches_host_io(gm):
    import torch
    w = make_config("C1")
    s = gm.System(w, load=False)
    dev = s.device
    s.set_particles(torch.from_numpy(w.pos).to(dev), torch.from_numpy(w.vel).to(dev),
                    torch.from_numpy(w.type).to(dev), torch.from_numpy(w.mass).to(dev))
    gm.gm_set_bonds(s.h, torch.from_numpy(s.bonds).to(dev), None)
    s.step(25)
    p = torch.empty((w.n, 3), dtype=torch.float32, device=dev)
    v = torch.empty_like(p)
    gm.gm_get_particles(s.h, p, v, None)
    s2 = gm.System(w)
    s2.step(25)
    p2, v2, _ = s2.get_particles()
    np.testing.assert_array_equal(p.cpu().numpy(), p2)
    np.testing.assert_array_equal(v.cpu().numpy(), v2)
    s.close(); s2.close()
