"""Seeded synthetic melts shaped like the paper's benchmarks (BASELINE.json `configs`).

The paper (Fig. 4) measures a monomeric LJ liquid and a DPD liquid; no
dataset is published.  BASELINE.json names five synthetic bead-spring / DPD melts instead; this
module is their recipe.  Draw order is fixed: jitter -> velocities (DPD:
chain starts -> step directions -> velocities).  Everything is stored as fp32 (the oracle promotes
the same fp32 values to fp64).  No arithmetic of the method lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 13102041


@dataclass
class Workload:
    name: str
    box: np.ndarray            # (3,) float32, origin-centred cuboid edge lengths
    pos: np.ndarray            # (N,3) float32 in [-L/2, L/2)
    vel: np.ndarray            # (N,3) float32
    type: np.ndarray           # (N,) int32
    mass: np.ndarray           # (N,) float32
    bonds: np.ndarray          # (n_bonds,2) int32 tag pairs
    bond_type: np.ndarray      # (n_bonds,) int32
    n_types: int
    pair_style: str            # "lj" | "dpd" | "harmonic" | "gauss" | "table" | "none"
    pair: dict                 # lj / gauss: eps,sigma,rc (n_types x n_types float32), shift (bool); dpd / harmonic: a, rc;
                               # table: table (n_types, n_types, Npoint, 4) float32, interval, rc = sqrt(Npoint * interval)
    bond_style: str            # "fene" | "harmonic" | "none"
    bond: dict                 # k, r0 (per bond type, float32)   (FENE: r0 means R0)
    integrator: str            # "nve" | "langevin" | "gwvv"
    dt: float
    kT: float = 1.0
    gamma: float = 0.0
    lam: float = 0.65
    r_skin: float = 0.4
    seed: int = 0              # seed of the method's counter-based noise
    n_steps: int = 0           # run length the config names
    sfc_period: int = 500
    chain_len: int = 1
    equil_steps: int = 0       # Langevin equilibration the config names (C3)
    notes: dict = field(default_factory=dict)
    topo: dict = field(default_factory=dict)   # angles / dihedrals: see oracle.Oracle and gm.System (empty: none)

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])


def maxwell_velocities(rng: np.random.Generator, n: int, kT: float, mass: np.ndarray) -> np.ndarray:
    """Gaussian(0, kT/m) per component, zero net momentum, rescaled to exactly kT with 3N-3 dof
    (SURVEY.md §8(c) c-22).  fp64 inside, fp32 out."""
    m = mass.astype(np.float64)[:, None]
    v = rng.standard_normal((n, 3)) * np.sqrt(kT / m)
    p = (m * v).sum(axis=0) / m.sum()
    v -= p
    if n > 1:
        ke2 = float((m * v * v).sum())
        v *= np.sqrt((3 * n - 3) * kT / ke2)
    return v.astype(np.float32)


def _boustrophedon_sites(n_lat: int, n_beads: int) -> np.ndarray:
    """Integer lattice coordinates of sites 0..n_beads-1 on a 3-D boustrophedon path through an
    n_lat^3 simple-cubic lattice: consecutive sites are always lattice neighbors."""
    s = np.arange(n_beads, dtype=np.int64)
    g = s // n_lat                    # global row
    ixp = s % n_lat
    iyp = g % n_lat
    iz = g // n_lat
    ix = np.where(g % 2 == 1, n_lat - 1 - ixp, ixp)
    iy = np.where(iz % 2 == 1, n_lat - 1 - iyp, iyp)
    return np.stack([ix, iy, iz], axis=1)


def make_kg_melt(name: str, n_beads: int, chain_len: int, n_lat: int, box_l: float, seed: int,
                 rc: float, r_skin: float, integrator: str, gamma: float, n_steps: int,
                 sfc_period: int = 500, equil_steps: int = 0, jitter: float = 0.05) -> Workload:
    """Kremer-Grest melt: beads on the first n_beads sites of an n_lat^3 lattice along a
    boustrophedon, cut into consecutive chains; each site jittered uniform +-jitter."""
    rng = np.random.Generator(np.random.PCG64(seed))
    L = np.float32(box_l)
    a = float(L) / n_lat
    sites = _boustrophedon_sites(n_lat, n_beads)
    jit = rng.uniform(-jitter, jitter, size=(n_beads, 3))
    pos = (sites + 0.5) * a - 0.5 * float(L) + jit
    pos = pos.astype(np.float32)
    half = np.float32(0.5) * L
    # keep inside [-L/2, L/2) after fp32 rounding
    pos = np.where(pos >= half, pos - L, pos)
    pos = np.where(pos < -half, pos + L, pos).astype(np.float32)
    mass = np.ones(n_beads, dtype=np.float32)
    vel = maxwell_velocities(rng, n_beads, 1.0, mass)
    s = np.arange(n_beads - 1, dtype=np.int64)
    same_chain = (s // chain_len) == ((s + 1) // chain_len)
    bi = s[same_chain]
    bonds = np.stack([bi, bi + 1], axis=1).astype(np.int32)
    one = np.ones((1, 1), dtype=np.float32)
    return Workload(
        name=name, box=np.array([L, L, L], dtype=np.float32), pos=pos, vel=vel,
        type=np.zeros(n_beads, dtype=np.int32), mass=mass, bonds=bonds,
        bond_type=np.zeros(len(bonds), dtype=np.int32), n_types=1, pair_style="lj",
        pair=dict(eps=one.copy(), sigma=one.copy(), rc=one * np.float32(rc), shift=True),
        bond_style="fene", bond=dict(k=np.array([30.0], np.float32), r0=np.array([1.5], np.float32)),
        integrator=integrator, dt=0.005, kT=1.0, gamma=gamma, r_skin=r_skin, seed=seed,
        n_steps=n_steps, sfc_period=sfc_period, chain_len=chain_len, equil_steps=equil_steps,
    )


def make_dpd_diblock(name: str, n_chains: int, box_l: float, seed: int, n_steps: int,
                     r_skin: float = 0.4, chain_len: int = 10, n_a: int = 5, step_len: float = 0.9) -> Workload:
    """DPD A5B5 diblock melt: uniform random chain starts, random walk of step 0.9, wrapped."""
    rng = np.random.Generator(np.random.PCG64(seed))
    L = np.float32(box_l)
    Ld = float(L)
    starts = rng.uniform(-0.5 * Ld, 0.5 * Ld, size=(n_chains, 3))
    # uniform directions on the sphere: z uniform in [-1,1], phi uniform
    z = rng.uniform(-1.0, 1.0, size=(n_chains, chain_len - 1))
    phi = rng.uniform(0.0, 2.0 * np.pi, size=(n_chains, chain_len - 1))
    s = np.sqrt(1.0 - z * z)
    steps = step_len * np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=2)
    walk = np.concatenate([np.zeros((n_chains, 1, 3)), np.cumsum(steps, axis=1)], axis=1)
    pos = (starts[:, None, :] + walk).reshape(-1, 3)
    pos = pos - Ld * np.floor((pos + 0.5 * Ld) / Ld)
    pos = pos.astype(np.float32)
    half = np.float32(0.5) * L
    pos = np.where(pos >= half, pos - L, pos)
    pos = np.where(pos < -half, pos + L, pos).astype(np.float32)
    n = n_chains * chain_len
    mass = np.ones(n, dtype=np.float32)
    vel = maxwell_velocities(rng, n, 1.0, mass)
    k = np.arange(n, dtype=np.int64)
    typ = ((k % chain_len) >= n_a).astype(np.int32)
    bi = k[(k % chain_len) != chain_len - 1]
    bonds = np.stack([bi, bi + 1], axis=1).astype(np.int32)
    a = np.array([[25.0, 40.0], [40.0, 25.0]], dtype=np.float32)
    return Workload(
        name=name, box=np.array([L, L, L], dtype=np.float32), pos=pos, vel=vel, type=typ, mass=mass,
        bonds=bonds, bond_type=np.zeros(len(bonds), dtype=np.int32), n_types=2, pair_style="dpd",
        pair=dict(a=a, rc=np.ones((2, 2), dtype=np.float32)),
        bond_style="harmonic", bond=dict(k=np.array([4.0], np.float32), r0=np.array([0.0], np.float32)),
        integrator="gwvv", dt=0.04, kT=1.0, gamma=4.5, lam=0.65, r_skin=r_skin, seed=seed,
        n_steps=n_steps, sfc_period=500, chain_len=chain_len,
    )


def _kg_box(n: int, rho: float = 0.85) -> float:
    return (n / rho) ** (1.0 / 3.0)


WCA_RC = 2.0 ** (1.0 / 6.0)

# BASELINE.json `configs`, in order.  Index 0..4 = C1..C5.
CONFIGS = {
    "C1": dict(kind="kg", n=2_000, chain_len=20, n_lat=13, box=13.30, rc=WCA_RC, skin=0.4,
               integrator="nve", gamma=0.0, n_steps=1_000),
    "C2": dict(kind="kg", n=64_000, chain_len=64, n_lat=40, box=_kg_box(64_000), rc=2.5, skin=0.3,
               integrator="langevin", gamma=1.0, n_steps=10_000),
    "C3": dict(kind="kg", n=1_000_000, chain_len=100, n_lat=100, box=_kg_box(1_000_000), rc=WCA_RC,
               skin=0.4, integrator="nve", gamma=1.0, n_steps=10_000, sfc_period=500, equil_steps=1_000),
    "C4": dict(kind="dpd", n_chains=300_000, box=100.0, skin=0.6, n_steps=5_000),
    "C5": dict(kind="kg", n=8_000_000, chain_len=200, n_lat=200, box=_kg_box(8_000_000), rc=2.5,
               skin=0.3, integrator="nve", gamma=0.0, n_steps=2_000, sfc_period=200),
}


def make_lj_liquid(n_side: int, seed: int = BASE_SEED + 6, kT: float = 1.2) -> Workload:
    """The paper's own LJ benchmark liquid (Fig. 4): monomers, packing fraction 0.2
    (rho = 0.2 * 6 / pi = 0.38197 sigma^-3), dt = 0.001, r_cut = 3.0, no bonds.  N = n_side^3 beads on a simple-cubic
    lattice with +-0.1 a jitter.  The paper gives no temperature, ensemble or buffer: kT = 1.2 (one-phase fluid at this
    density), NVE, skin 0.4, plain cut with shifted energy (reading c-25)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_side ** 3
    rho = 0.2 * 6.0 / np.pi
    L = (n / rho) ** (1.0 / 3.0)
    a = L / n_side
    g = np.arange(n_side, dtype=np.float64)
    ix, iy, iz = np.meshgrid(g, g, g, indexing="ij")
    pos = (np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1) + 0.5) * a - 0.5 * L
    pos += rng.uniform(-0.1, 0.1, size=(n, 3)) * a
    pos = pos.astype(np.float32)
    mass = np.ones(n, dtype=np.float32)
    vel = maxwell_velocities(rng, n, kT, mass)
    one = np.ones((1, 1), dtype=np.float32)
    return Workload(
        name=f"F4LJ{n_side}", box=np.array([L, L, L], dtype=np.float32), pos=pos, vel=vel,
        type=np.zeros(n, np.int32), mass=mass, bonds=np.zeros((0, 2), np.int32), bond_type=np.zeros(0, np.int32),
        n_types=1, pair_style="lj", pair=dict(eps=one.copy(), sigma=one.copy(), rc=one * np.float32(3.0), shift=True),
        bond_style="none", bond=dict(k=np.zeros(1, np.float32), r0=np.zeros(1, np.float32)),
        integrator="nve", dt=0.001, kT=kT, gamma=0.0, r_skin=0.4, seed=seed, n_steps=10_000, sfc_period=500,
    )


def make_dpd_liquid(n: int, seed: int = BASE_SEED + 7) -> Workload:
    """The paper's own DPD benchmark liquid (Fig. 4): monomers at number density 3.0, dt = 0.04,
    r_cut = 1.0, no bonds, uniform random start.  a = 25, gamma = 4.5, kT = 1, GW-VV lambda = 0.65 as in config C4
    (the paper names none of them; reading c-25), skin 0.6."""
    rng = np.random.Generator(np.random.PCG64(seed))
    L = (n / 3.0) ** (1.0 / 3.0)
    pos = (rng.uniform(-0.5, 0.5, size=(n, 3)) * L).astype(np.float32)
    half = np.float32(0.5 * L)
    pos = np.where(pos >= half, pos - np.float32(L), pos).astype(np.float32)
    mass = np.ones(n, dtype=np.float32)
    vel = maxwell_velocities(rng, n, 1.0, mass)
    one = np.ones((1, 1), dtype=np.float32)
    return Workload(
        name=f"F4DPD{n}", box=np.array([L, L, L], dtype=np.float32), pos=pos, vel=vel,
        type=np.zeros(n, np.int32), mass=mass, bonds=np.zeros((0, 2), np.int32), bond_type=np.zeros(0, np.int32),
        n_types=1, pair_style="dpd", pair=dict(a=one * np.float32(25.0), rc=one.copy()),
        bond_style="none", bond=dict(k=np.zeros(1, np.float32), r0=np.zeros(1, np.float32)),
        integrator="gwvv", dt=0.04, kT=1.0, gamma=4.5, lam=0.65, r_skin=0.6, seed=seed, n_steps=5_000, sfc_period=500,
    )


def make_config(name: str, scale: float | None = None, n: int | None = None) -> Workload:
    """Build one of C1..C5, or the paper's Fig. 4 liquids "F4LJ" / "F4DPD" with about `n` beads (default 1,000,000).
    `scale` (tests only) shrinks a config to a geometrically similar smaller melt: KG lattice edge and DPD chain
    count are scaled, density and all parameters kept."""
    if name == "F4LJ":
        return make_lj_liquid(int(round((n or 1_000_000) ** (1.0 / 3.0))))
    if name == "F4DPD":
        return make_dpd_liquid(int(n or 1_000_000))
    c = dict(CONFIGS[name])
    seed = BASE_SEED + int(name[1])
    if c["kind"] == "kg":
        n, n_lat, box = c["n"], c["n_lat"], c["box"]
        if scale is not None:
            n_lat = max(4, int(round(n_lat * scale)))
            n = (n_lat ** 3 // c["chain_len"]) * c["chain_len"]
            box = c["box"] * n_lat / c["n_lat"]
        return make_kg_melt(name, n, c["chain_len"], n_lat, box, seed, c["rc"], c["skin"],
                            c["integrator"], c["gamma"], c["n_steps"],
                            sfc_period=c.get("sfc_period", 500), equil_steps=c.get("equil_steps", 0))
    n_chains, box = c["n_chains"], c["box"]
    if scale is not None:
        box = max(4.0, round(c["box"] * scale))
        n_chains = int(round(3.0 * box ** 3 / 10.0))
    return make_dpd_diblock(name, n_chains, box, seed, c["n_steps"], r_skin=c["skin"])


def make_random_box(n: int, box, seed: int, n_types: int = 1, min_sep: float = 0.0,
                    kT: float = 1.0) -> Workload:
    """Uniform random beads in a (possibly non-cubic) box, no bonds; for brute-force pins and
    edge-case tests.  With min_sep > 0 beads closer than min_sep to an earlier bead are re-drawn
    (simple rejection, small n only)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = np.asarray(box, dtype=np.float32).reshape(3)
    Ld = box.astype(np.float64)
    pos = rng.uniform(-0.5, 0.5, size=(n, 3)) * Ld
    if min_sep > 0.0:
        for i in range(1, n):
            for _ in range(1000):
                d = pos[:i] - pos[i]
                d -= Ld * np.rint(d / Ld)
                if (np.einsum("ij,ij->i", d, d) >= min_sep * min_sep).all():
                    break
                pos[i] = rng.uniform(-0.5, 0.5, size=3) * Ld
    pos = pos.astype(np.float32)
    half = np.float32(0.5) * box
    pos = np.where(pos >= half, pos - box, pos)
    pos = np.where(pos < -half, pos + box, pos).astype(np.float32)
    mass = np.ones(n, dtype=np.float32)
    vel = maxwell_velocities(rng, n, kT, mass)
    typ = (np.arange(n) % n_types).astype(np.int32)
    ones = np.ones((n_types, n_types), dtype=np.float32)
    return Workload(
        name=f"random{n}", box=box, pos=pos, vel=vel, type=typ, mass=mass,
        bonds=np.zeros((0, 2), np.int32), bond_type=np.zeros(0, np.int32), n_types=n_types,
        pair_style="lj", pair=dict(eps=ones.copy(), sigma=ones.copy(), rc=ones * np.float32(2.5), shift=True),
        bond_style="none", bond=dict(k=np.zeros(1, np.float32), r0=np.zeros(1, np.float32)),
        integrator="nve", dt=0.005, kT=kT, seed=seed,
    )
