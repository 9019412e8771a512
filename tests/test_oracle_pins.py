"""Pins of the fp64 oracle against what the paper and the mathematics fix.

None of these re-types an oracle formula and compares it with itself: they use closed-form values
(tests/golden/closed_forms.txt), published known answers (tests/golden/philox4x32_10_kat.txt),
force = -grad(energy) by central differences, all-pairs brute force versus the cell-list mode,
invariances, conservation laws and measured oscillation periods.
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from tests.util import custom
from workloads import make_config, make_random_box, maxwell_velocities


def G(golden):
    return {r[0]: float(r[1]) for r in golden("closed_forms.txt")}


def dimer(r, **kw):
    w = custom([[-r / 2, 0, 0], [r / 2, 0, 0]], 20.0, **kw)
    o = orc.Oracle(w, use_cells=False)
    o.pos[:] = [[-r / 2, 0, 0], [r / 2, 0, 0]]        # exact fp64 separation
    return o


# ---- P1: closed forms of Eq. (1) ------------------------------------------------
def test_lj_closed_forms(golden):
    g = G(golden)
    o = dimer(g["lj_zero_force_r"], rc=2.5, shift=False)
    F, pe, _, npair = o.pair_bond_forces()
    assert npair == 1
    assert np.abs(F).max() < 1e-12                       # zero-force point r = 2^(1/6) sigma
    assert pe == pytest.approx(g["lj_u_at_min"], abs=1e-14)
    o = dimer(1.0, rc=2.5, shift=False)
    F, pe, _, _ = o.pair_bond_forces()
    assert pe == pytest.approx(g["lj_u_at_sigma"], abs=1e-14)
    assert F[0, 0] == pytest.approx(-24.0, rel=1e-14)   # 24 eps (2 - 1)/r at r = sigma, pushes bead 0 to -x
    assert F[1, 0] == pytest.approx(+24.0, rel=1e-14)
    # shifted: U -> U - U(rc); at rc = 2.5 the shift is 4 (2.5^-12 - 2.5^-6)
    o = dimer(1.0, rc=2.5, shift=True)
    _, pe, _, _ = o.pair_bond_forces()
    assert pe == pytest.approx(-g["lj_ushift_rc2p5"], abs=1e-13)
    # WCA: r_c = 2^(1/6): shift is +eps and the shifted energy goes to 0+ at the cutoff
    rc = 2.0 ** (1.0 / 6.0)
    o = dimer(rc * (1 - 1e-9), rc=rc, shift=True)
    o.rc[:] = rc; o.ushift[:] = -1.0                      # exact fp64 cutoff (the workload carries fp32)
    _, pe, _, npair = o.pair_bond_forces()
    assert npair == 1 and 0.0 <= pe < 1e-12
    o = dimer(rc * (1 + 1e-9), rc=rc, shift=True)        # strict '<' at the cutoff (reading c-10)
    o.rc[:] = rc; o.ushift[:] = -1.0
    F, pe, _, npair = o.pair_bond_forces()
    assert npair == 0 and pe == 0.0 and np.abs(F).max() == 0.0
    # eps and sigma scale as the formula says: U(2^(1/6) s) = -eps for s = 1.3, eps = 0.7
    o = dimer(1.3 * g["lj_zero_force_r"], rc=5.0, shift=False, eps=0.7, sigma=1.3)
    F, pe, _, _ = o.pair_bond_forces()
    assert pe == pytest.approx(-0.7, rel=1e-6) and np.abs(F).max() < 1e-5   # eps, sigma are fp32 inputs


# ---- P2: FENE + WCA dimer (Kremer-Grest bond; reading c-8) ---------------------------------------
def test_fene_wca_dimer_closed_form(golden):
    g = G(golden)
    rc = 2.0 ** (1.0 / 6.0)
    o = dimer(g["fene_wca_rstar"], rc=rc, shift=True, bond_style="fene", k=30.0, r0=1.5, bonds=[[0, 1]])
    o.rc[:] = rc                                          # exact fp64 cutoff -> exact +1 shift
    o.ushift[:] = -1.0
    F, pe_pair, pe_bond, _ = o.pair_bond_forces()
    assert np.abs(F).max() < 1e-9                         # force root r*
    assert pe_pair + pe_bond == pytest.approx(g["fene_wca_u_rstar"], rel=1e-12)
    # pure FENE at r = 1: F = -k r / (1 - 1/2.25) = -54, attractive
    o = dimer(1.0, pair_style="none", bond_style="fene", k=30.0, r0=1.5, bonds=[[0, 1]])
    F, _, pe_bond, _ = o.pair_bond_forces()
    assert F[1, 0] == pytest.approx(-54.0, rel=1e-12) and F[0, 0] == pytest.approx(54.0, rel=1e-12)
    assert pe_bond == pytest.approx(-0.5 * 30 * 2.25 * math.log(1 - 1 / 2.25), rel=1e-12)
    # over-stretched bond is an error, not a number
    o = dimer(1.6, pair_style="none", bond_style="fene", k=30.0, r0=1.5, bonds=[[0, 1]])
    o.pair_bond_forces()
    assert o.status == orc.ORC_ERR_BOND_OVERSTRETCH


def test_fene_wca_dimer_period(golden):
    """O7 NVE: the measured small-amplitude period of the dimer is 2 pi / sqrt(U''(r*)/mu)."""
    g = G(golden)
    rc = 2.0 ** (1.0 / 6.0)
    r0 = g["fene_wca_rstar"] + 1e-3
    o = dimer(r0, rc=rc, shift=True, bond_style="fene", k=30.0, r0=1.5, bonds=[[0, 1]], dt=0.0005)
    o.compute_forces()
    seps = []
    for _ in range(1200):
        o.run(1)
        seps.append(o.pos[1, 0] - o.pos[0, 0] - g["fene_wca_rstar"])
    seps = np.array(seps)
    t = (np.arange(len(seps)) + 1) * o.P.dt
    # upward zero crossings, linearly interpolated
    idx = np.where((seps[:-1] < 0) & (seps[1:] >= 0))[0]
    tc = t[idx] - seps[idx] * (t[idx + 1] - t[idx]) / (seps[idx + 1] - seps[idx])
    period = np.diff(tc).mean()
    assert period == pytest.approx(g["fene_wca_period"], rel=2e-3)


# ---- P9: harmonic bond follows the paper's Eq. (7): U = k (r - r0)^2, no 1/2 -----------------------
def test_harmonic_dimer_frequency(golden):
    g = G(golden)
    o = dimer(0.5, pair_style="none", bond_style="harmonic", k=4.0, r0=0.0, bonds=[[0, 1]], dt=0.001)
    o.compute_forces()
    F = o.frc.copy()
    assert F[1, 0] == pytest.approx(-2 * 4.0 * 0.5, rel=1e-12)     # F = -2 k r
    sep = []
    for _ in range(4000):
        o.run(1)
        sep.append(o.pos[1, 0] - o.pos[0, 0])
    sep = np.array(sep)
    t = (np.arange(len(sep)) + 1) * o.P.dt
    idx = np.where((sep[:-1] < 0) & (sep[1:] >= 0))[0]
    tc = t[idx] - sep[idx] * (t[idx + 1] - t[idx]) / (sep[idx + 1] - sep[idx])
    omega = 2 * math.pi / np.diff(tc).mean()
    assert omega == pytest.approx(g["harmonic_dimer_omega"], rel=1e-3)   # 2.828 under the 1/2 k convention
    # r0 != 0: energy k (r - r0)^2 and restoring force -2k (r - r0)
    o = dimer(1.5, pair_style="none", bond_style="harmonic", k=3.0, r0=1.0, bonds=[[0, 1]])
    Fh, _, pe_bond, _ = o.pair_bond_forces()
    assert pe_bond == pytest.approx(3.0 * 0.25, rel=1e-12)
    assert Fh[1, 0] == pytest.approx(-2 * 3.0 * 0.5, rel=1e-12)


# ---- force = -grad(energy), for every potential on the path ---------------------------------------
def _fd_check(w, n_probe=6, h=1e-6, tol=2e-6):
    o = orc.Oracle(w, use_cells=False)
    F, _, _, _ = o.pair_bond_forces()
    rng = np.random.default_rng(5)
    scale = np.sqrt((F ** 2).sum(axis=1).mean())
    for i in rng.choice(w.n, size=n_probe, replace=False):
        for d in range(3):
            p = o.pos.copy(); p[i, d] += h
            _, a1, b1, _ = o.pair_bond_forces(pos=p)
            p[i, d] -= 2 * h
            _, a0, b0, _ = o.pair_bond_forces(pos=p)
            fd = -((a1 + b1) - (a0 + b0)) / (2 * h)
            assert abs(fd - F[i, d]) <= tol * max(scale, abs(F[i, d]))


def test_force_is_minus_gradient_kg():
    w = make_config("C1", scale=0.55)                     # 7^3 lattice, FENE + WCA, chains of 20
    _fd_check(w)
    w.pair["rc"][:] = 2.5                                 # full LJ, shifted
    _fd_check(w)


def test_force_is_minus_gradient_dpd_conservative_and_harmonic():
    w = make_config("C4", scale=0.06)                     # 6^3 box, rho = 3, A5B5 + harmonic bonds
    w.gamma = 0.0; w.kT = 0.0                             # conservative part only
    _fd_check(w, tol=5e-6)


# ---- P3: all pairs versus the oracle's cell-list mode ---------------------------------------------
@pytest.mark.parametrize("box", [(9.0, 9.0, 9.0), (7.6, 11.0, 14.5)])
def test_bruteforce_vs_cells(box):
    w = make_random_box(900, box, seed=3, n_types=2, min_sep=0.8)
    w.pair["eps"][:] = [[1.0, 0.6], [0.6, 1.4]]
    w.pair["sigma"][:] = [[1.0, 1.1], [1.1, 0.9]]
    w.pair["rc"][:] = [[2.5, 2.2], [2.2, 1.9]]
    # beads exactly on faces and corners of the box
    w.pos[0] = [-box[0] / 2, 0, 0]; w.pos[1] = [-box[0] / 2, -box[1] / 2, -box[2] / 2]
    w.pos[2] = [np.nextafter(np.float32(box[0] / 2), np.float32(0)), 0.3, -box[2] / 2]
    a = orc.Oracle(w, use_cells=False); b = orc.Oracle(w, use_cells=True)
    Fa, pa, _, na = a.pair_bond_forces(); Fb, pb, _, nb = b.pair_bond_forces()
    assert na == nb and na > 1000
    assert np.abs(Fa - Fb).max() <= 1e-12 * np.abs(Fa).max()
    assert pa == pytest.approx(pb, rel=1e-12)
    for r_list in (1.5225, 2.8):
        pa_ = a.neighbor_pairs(r_list, use_cells=False); pb_ = b.neighbor_pairs(r_list, use_cells=True)
        assert np.array_equal(pa_, pb_)
        # and against numpy's own all-pairs distance matrix
        d = w.pos.astype(np.float64)[:, None, :] - w.pos.astype(np.float64)[None, :, :]
        L = np.asarray(box); d -= L * np.rint(d / L)
        r2 = (d * d).sum(axis=2)
        iu = np.triu_indices(w.n, 1)
        assert int((r2[iu] < r_list * r_list).sum()) == len(pa_)


def test_bruteforce_vs_cells_kg_c1_and_dpd():
    w = make_config("C1")
    a = orc.Oracle(w, use_cells=False); b = orc.Oracle(w, use_cells=True)
    Fa = a.compute_forces().copy(); Fb = b.compute_forces().copy()
    assert np.abs(Fa - Fb).max() <= 1e-12 * np.abs(Fa).max()
    assert np.array_equal(a.neighbor_pairs(1.5225, False), b.neighbor_pairs(1.5225, True))
    w = make_config("C4", scale=0.07)
    a = orc.Oracle(w, use_cells=False); b = orc.Oracle(w, use_cells=True)
    Fa = a.compute_forces().copy(); Fb = b.compute_forces().copy()
    assert np.abs(Fa - Fb).max() <= 1e-12 * np.abs(Fa).max()


# ---- P4: invariants --------------------------------------------------------------------------------
@pytest.mark.parametrize("name,scale", [("C1", None), ("C2", 0.2), ("C4", 0.07)])
def test_newton_third_law_and_invariances(name, scale):
    w = make_config(name, scale=scale)
    w.integrator = "nve" if w.pair_style == "lj" else "gwvv"      # no per-bead Langevin noise here
    o = orc.Oracle(w)
    F, pe, pb, npair = o.pair_bond_forces()
    assert np.abs(F.sum(axis=0)).max() <= 1e-10 * np.abs(F).sum()   # zero net force (theta_ij = theta_ji for DPD)
    L = o.box
    # global translation + rewrap
    p2 = o.pos + np.array([0.37, -1.21, 2.6])
    p2 -= L * np.floor((p2 + L / 2) / L)
    F2, pe2, pb2, np2 = o.pair_bond_forces(pos=p2)
    assert np2 == npair
    assert np.abs(F2 - F).max() <= 1e-9 * np.abs(F).max()
    # shifting single beads by +-L in any direction changes nothing
    p3 = o.pos.copy(); p3[::7, 0] += L[0]; p3[1::5, 2] -= L[2]
    F3, _, _, _ = o.pair_bond_forces(pos=p3)
    assert np.abs(F3 - F).max() <= 1e-9 * np.abs(F).max()


def test_pairwise_antisymmetry_dpd_noise():
    # theta_ij = theta_ji, zero mean, unit variance, bounded by sqrt(3)
    assert orc.pair_theta(11, 5, 3, 9) == orc.pair_theta(11, 5, 9, 3)
    assert orc.pair_theta(11, 5, 3, 9) != orc.pair_theta(11, 6, 3, 9)
    assert orc.pair_theta(11, 5, 3, 9) != orc.pair_theta(12, 5, 3, 9)
    th = np.array([orc.pair_theta(42, s, i, i + 1 + (s % 3)) for s in range(200) for i in range(300)])
    assert abs(th.mean()) < 0.02 and abs(th.var() - 1.0) < 0.02 and np.abs(th).max() <= math.sqrt(3)
    xi = np.array([orc.bead_xi(42, s, i) for s in range(100) for i in range(200)])
    assert np.abs(xi.mean(axis=0)).max() < 0.02 and np.abs(xi.var(axis=0) - 1 / 3).max() < 0.01
    assert abs(np.corrcoef(xi.T)[0, 1]) < 0.03


def test_permutation_invariance():
    """Relabelling storage changes nothing for LJ (noise-free) forces."""
    w = make_config("C1")
    o = orc.Oracle(w)
    F, *_ = o.pair_bond_forces()
    perm = np.random.default_rng(0).permutation(w.n)
    inv = np.argsort(perm)
    w2 = make_config("C1")
    w2.pos = w.pos[perm]; w2.vel = w.vel[perm]; w2.bonds = inv[w.bonds].astype(np.int32)
    F2, *_ = orc.Oracle(w2).pair_bond_forces()
    assert np.abs(F2 - F[perm]).max() <= 1e-10 * np.abs(F).max()


# ---- P8: Philox4x32-10 -----------------------------------------------------------------------------
def _philox_bigint(ctr, key):
    """Independent restatement with Python big integers (SC'11: 10 rounds, key bumped between rounds)."""
    c, k = list(ctr), list(key)
    for r in range(10):
        if r:
            k = [(k[0] + 0x9E3779B9) % 2 ** 32, (k[1] + 0xBB67AE85) % 2 ** 32]
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 % 2 ** 32, (p0 >> 32) ^ c[3] ^ k[1], p0 % 2 ** 32]
    return c


def test_philox_known_answers(golden):
    rows = golden("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]
        assert _philox_bigint(v[0:4], v[4:6]) == v[6:10]
    rng = np.random.default_rng(1)
    for _ in range(200):
        v = [int(x) for x in rng.integers(0, 2 ** 32, size=6)]
        assert [int(x) for x in orc.philox4x32_10(v[:4], v[4:])] == _philox_bigint(v[:4], v[4:])


def test_u24_symmetric_variate_is_exact_in_fp32():
    # u = (k + 1/2) 2^-24 has 25 significant bits, but the variate the method uses, 2u - 1 =
    # (2k + 1 - 2^24) 2^-24, is an odd 24-bit integer over 2^24: the same real number in fp32 and fp64.
    for x in (0, 1, 255, 256, 0xFFFFFFFF, 0x80000000, 123456789):
        u = orc.u24(x)
        assert 0.0 < u < 1.0
        assert u == ((x >> 8) + 0.5) / 2 ** 24
        s = 2.0 * u - 1.0
        assert float(np.float32(s)) == s and s == (2 * (x >> 8) + 1 - 2 ** 24) / 2 ** 24
    # keying: counter = (min tag, max tag, step, 0), key = (seed lo, seed hi), first word -> theta
    seed, step, i, j = (5 << 32) | 77, 9, 12, 4
    w0 = _philox_bigint([4, 12, 9, 0], [77, 5])[0]
    assert orc.pair_theta(seed, step, i, j) == pytest.approx(math.sqrt(3) * (2 * ((w0 >> 8) + 0.5) / 2 ** 24 - 1), rel=1e-15)
    w = _philox_bigint([12, 0, 9, 1], [77, 5])
    assert np.allclose(orc.bead_xi(seed, step, 12), [2 * ((x >> 8) + 0.5) / 2 ** 24 - 1 for x in w[:3]], rtol=1e-15)


# ---- O1 / P10: geometry and free flight ------------------------------------------------------------
def test_min_image_and_free_flight():
    assert orc.min_image(4.9, 10.0) == pytest.approx(4.9)
    assert orc.min_image(5.1, 10.0) == pytest.approx(-4.9)
    assert orc.min_image(-5.1, 10.0) == pytest.approx(4.9)
    assert orc.min_image(14.9, 10.0) == pytest.approx(4.9)
    w = make_random_box(200, (6.0, 7.0, 8.0), seed=2)
    w.pair["eps"][:] = 0.0                                # no forces: r(t) = wrap(r0 + v t) exactly
    o = orc.Oracle(w)
    o.compute_forces()
    r0, v0 = o.pos.copy(), o.vel.copy()
    o.run(400)
    L = o.box
    exp = r0 + v0 * (400 * o.P.dt)
    exp -= L * np.floor((exp + L / 2) / L)
    d = o.pos - exp; d -= L * np.rint(d / L)
    assert np.abs(d).max() < 1e-11
    assert (o.pos >= -L / 2).all() and (o.pos < L / 2).all()
    assert np.array_equal(o.vel, v0)


# ---- P5 / P6: NVE velocity-Verlet ------------------------------------------------------------------
def _lj_liquid(n_side, rho, rc, dt, seed=4, shift=False):
    n = n_side ** 3
    L = (n / rho) ** (1 / 3)
    g = (np.indices((n_side,) * 3).reshape(3, -1).T + 0.5) * (L / n_side) - L / 2
    rng = np.random.default_rng(seed)
    w = custom(g + rng.uniform(-0.05, 0.05, g.shape), L, rc=rc, shift=shift, dt=dt)
    w.vel = maxwell_velocities(rng, n, 1.0, w.mass)
    return w


def _total_energy(o):
    pe, pb, _ = o.potential()
    return o.kinetic() + pe + pb


def test_nve_energy_error_scales_as_dt_squared_and_reverses():
    rms = {}
    for dt in (0.004, 0.002):
        w = _lj_liquid(6, 0.8, 2.5, dt, shift=True)
        o = orc.Oracle(w)
        o.compute_forces()
        o.run(int(round(1.0 / dt)))                       # melt the lattice a little: 1 tau
        es = []
        for _ in range(60):
            o.run(int(round(0.02 / dt)))
            es.append(_total_energy(o))
        es = np.array(es)
        rms[dt] = es.std() / abs(es.mean())
        assert abs(es[-1] - es[0]) / abs(es.mean()) < 2e-3     # no drift
    ratio = rms[0.004] / rms[0.002]
    assert 2.5 < ratio < 6.0                               # ~ 4: second-order integrator
    # P6 time reversal: n steps, v -> -v, n steps returns to the start (fp64 roundoff)
    w = _lj_liquid(5, 0.8, 2.5, 0.004, shift=True)
    o = orc.Oracle(w)
    r0, v0 = o.pos.copy(), o.vel.copy()
    o.compute_forces()
    o.run(100)
    o.vel *= -1.0
    o.run(100)
    d = o.pos - r0; d -= o.box * np.rint(d / o.box)
    assert np.abs(d).max() < 1e-9 and np.abs(o.vel + v0).max() < 1e-9


def test_nve_energy_rms_at_the_papers_level():
    """PAPER.md:L225-227 (Fig. 12): LJ liquid rho = 0.8, T = 1.0, l = 12, plain-cut r_cut = 3.4:
    relative RMS deviation of the total energy < 4e-5 for dt <= 0.004, sampled every 0.1 tau.
    Order-of-magnitude check on one short sample (the paper averages five 1000-tau runs)."""
    n_side = 11                                           # 1331 beads in l = 11.85 (rho = 0.8); paper: l = 12
    w = _lj_liquid(n_side, 0.8, 3.4, 0.004, shift=False)
    w.integrator = "langevin"; w.gamma = 1.0
    o = orc.Oracle(w)
    o.compute_forces()
    o.run(750)                                            # 3 tau of thermostatted equilibration
    w2 = custom(o.pos, w.box, vel=o.vel, rc=3.4, shift=False, dt=0.004)
    o2 = orc.Oracle(w2)
    o2.pos[:] = o.pos; o2.vel[:] = o.vel
    o2.compute_forces()
    es = []
    for _ in range(40):                                   # 4 tau sampled every 0.1 tau
        o2.run(25)
        es.append(_total_energy(o2))
    es = np.array(es)
    dE = es.std() / abs(es.mean())
    assert dE < 4e-5 * 3                                  # same order as the paper's SP/DP level
    assert 0.7 < o2.temperature() < 1.3


# ---- P7: thermostats -------------------------------------------------------------------------------
def test_langevin_ideal_gas_temperature_and_decay():
    w = make_random_box(40000, (20.0, 20.0, 20.0), seed=8, kT=1.0)
    w.pair_style = "none"                                 # ideal gas
    w.integrator = "langevin"; w.gamma = 1.0; w.kT = 1.0; w.dt = 0.005
    w.vel[:] = 0.0; w.vel[:, 0] = 2.0                      # cold start with a drift: <v_x> decays as exp(-gamma t)
    o = orc.Oracle(w)
    o.compute_forces()
    o.run(200)                                            # t = 1
    assert o.vel[:, 0].mean() == pytest.approx(2.0 * math.exp(-1.0), rel=0.02)   # O(gamma dt) scheme error 0.5 %
    Ts = []
    o.run(1400)
    for _ in range(20):
        o.run(50)
        Ts.append(o.temperature())
    assert np.mean(Ts) == pytest.approx(1.0, rel=0.02)


def test_dpd_temperature_and_momentum():
    w = make_config("C4", scale=0.07)                     # 7^3 box, ~1030 beads, rho = 3
    o = orc.Oracle(w)
    o.compute_forces()
    p0 = o.momentum().copy()
    Ts = []
    o.run(150)
    for _ in range(30):
        o.run(10)
        Ts.append(o.temperature())
    assert np.abs(o.momentum() - p0).max() < 1e-9         # pairwise noise conserves momentum exactly
    assert np.mean(Ts) == pytest.approx(1.0, rel=0.06)    # GW-VV at dt = 0.04, lambda = 0.65


def test_dpd_temperature_long_average():
    """Fluctuation-dissipation through <T> (sigma_R^2 = 2 gamma kT, reading c-3) on a longer average: 2,058 beads,
    220 readings over 2,200 steps after a 300-step transient.  One reading of N beads scatters by sqrt(2/3N) = 1.8 %;
    readings 10 steps apart are nearly independent (DPD velocity correlations die within ~0.3 tau = 8 steps), so the mean
    is good to ~0.15 %; the integrator's own offset at dt = 0.04, lambda = 0.65 stays below 1 %, so the window is
    1.5 % (was 6 %): a wrong noise amplitude (sigma_R^2 = gamma kT or 4 gamma kT) gives 0.5 or 2.0, a missing 1/sqrt(dt)
    gives 0.04, uniform noise without the sqrt(3) gives 1/3."""
    w = make_config("C4", scale=0.0882)                   # 8.82^3 box: 205 chains, 2,050 beads, rho = 3
    o = orc.Oracle(w, n_threads=4)
    o.compute_forces()
    o.run(300)
    Ts = []
    for _ in range(220):
        o.run(10)
        Ts.append(o.temperature())
    T = float(np.mean(Ts))
    assert T == pytest.approx(1.0, rel=0.015), T


# ---- GW-VV predictor/corrector (reading c-6) ------------------------------------------
def _dpd_conservative(seed, dt, integrator):
    """Soft-sphere fluid with the DPD conservative force only (gamma = 0, kT = 0): Hamiltonian."""
    w = make_random_box(600, (6.0, 6.0, 6.0), seed=seed, kT=1.0)
    w.pair_style = "dpd"; w.pair = dict(a=np.full((1, 1), 25.0, np.float32), rc=np.ones((1, 1), np.float32))
    w.integrator = integrator; w.gamma = 0.0; w.kT = 0.0; w.lam = 0.65; w.dt = dt
    o = orc.Oracle(w, use_cells=False)
    o.P.dt = dt                                           # exact fp64 time step
    return o


def test_gwvv_without_thermostat_is_velocity_verlet():
    """With gamma = 0 the force does not see v~, and GW-VV (r += dt v + dt^2/2 f; v += dt/2 (f + f')) IS velocity
    Verlet: the ORC_GWVV branch of orc_run must reproduce the ORC_NVE branch (pinned by P2, P5, P6) to fp64
    round-off.  A missing dt^2/2 f drift, v += dt f' or a corrector without the old force all break this."""
    a = _dpd_conservative(31, 0.01, "nve")
    b = _dpd_conservative(31, 0.01, "gwvv")
    a.compute_forces(); b.compute_forces()
    a.run(200); b.run(200)
    d = a.pos - b.pos; d -= a.box * np.rint(d / a.box)
    # round-off (1e-16) grows along the chaotic trajectory to ~3e-10 by t = 2; a wrong scheme differs by O(dt^2) = 1e-4
    assert np.abs(d).max() < 1e-8 and np.abs(a.vel - b.vel).max() < 1e-8
    assert np.abs(a.vel).max() > 0.5                      # the run did move


def test_gwvv_energy_error_is_second_order():
    """Same Hamiltonian system through the GW-VV branch: halving dt quarters the energy error."""
    def rms(dt, n):
        o = _dpd_conservative(32, dt, "gwvv")
        o.compute_forces()
        es = []
        for _ in range(n):
            o.run(1)
            es.append(o.kinetic() + o.potential()[0])
        es = np.array(es)
        return float(np.sqrt(np.mean((es - es.mean()) ** 2)))
    e1, e2 = rms(0.02, 100), rms(0.01, 200)
    assert 3.0 < e1 / e2 < 5.0, (e1, e2)


def test_gwvv_two_bead_step_depends_on_lambda(golden):
    """tests/golden/closed_forms.txt: one GW-VV step of two approaching beads under the dissipative force alone,
    worked by hand for lambda = 0.65.  Pins v~ = v + lambda dt f (lambda = 0.5 gives f' = -1.2448 instead of
    -1.2272), the dt^2/2 f drift and the dt/2 (f + f') corrector."""
    g = G(golden)

    def one_step(lam):
        w = custom([[-0.25, 0, 0], [0.25, 0, 0]], 20.0, vel=[[0.5, 0, 0], [-0.5, 0, 0]], pair_style="dpd", a=0.0,
                   rc=1.0, integrator="gwvv", dt=0.04, kT=0.0, gamma=4.5, lam=lam)
        o = orc.Oracle(w, use_cells=False)
        o.P.dt = 0.04; o.P.lam = lam                      # exact fp64 parameters (the workload carries fp32)
        o.compute_forces()
        assert o.frc[0, 0] == pytest.approx(-1.125, abs=1e-14) and o.frc[1, 0] == pytest.approx(1.125, abs=1e-14)
        o.run(1)
        return o
    o = one_step(0.65)
    assert o.frc[0, 0] == pytest.approx(g["gwvv_two_bead_f1"], abs=1e-11)
    assert o.frc[1, 0] == pytest.approx(-g["gwvv_two_bead_f1"], abs=1e-11)
    assert o.vel[0, 0] == pytest.approx(g["gwvv_two_bead_v1"], abs=1e-12)
    assert o.vel[1, 0] == pytest.approx(-g["gwvv_two_bead_v1"], abs=1e-12)
    assert o.pos[0, 0] == pytest.approx(g["gwvv_two_bead_x1"], abs=1e-14)
    assert np.abs(o.pos[:, 1:]).max() == 0.0 and np.abs(o.vel[:, 1:]).max() == 0.0
    o = one_step(0.5)                                     # the pin must tell lambda = 0.5 from 0.65
    assert abs(o.frc[0, 0] - g["gwvv_two_bead_f1"]) > 1e-2
    assert abs(o.vel[0, 0] - g["gwvv_two_bead_v1"]) > 1e-4


# ---- O8 observables ---------------------------------------------------------------------------------
def test_rod_radius_of_gyration_and_bond_lengths(golden):
    """chain_rg2 / bond_lengths on straight rods that cross the periodic faces: Rg^2 = (n^2 - 1) a^2 / 12."""
    g = G(golden)
    n, a, box = 10, 0.9, np.array([5.0, 6.0, 7.0])
    rng = np.random.default_rng(3)
    pos = []
    for _ in range(7):                                    # 7 rods, random origins and directions
        e = rng.normal(size=3); e /= np.linalg.norm(e)
        r0 = rng.uniform(-0.5, 0.5, 3) * box
        pos.append(r0 + a * np.arange(n)[:, None] * e)
    pos = np.concatenate(pos)
    pos -= box * np.floor(pos / box + 0.5)                # wrapped into the box: the rods are cut by the faces
    rg2 = orc.chain_rg2(pos, box, n)
    assert rg2.shape == (7,) and np.allclose(rg2, g["rod_rg2_n10_a0p9"], rtol=1e-12)
    bonds = np.array([[c * n + k, c * n + k + 1] for c in range(7) for k in range(n - 1)])
    assert np.allclose(orc.bond_lengths(pos, box, bonds), a, rtol=1e-12)
