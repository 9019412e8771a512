/*
 * gm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the short-range force pipeline of GALAMOST-style
 * coarse-grained polymer MD computes (arXiv 1310.2041, "PAPER.md").  It shares no code, header,
 * table or constant generator with the CUDA path under paper_1310_2041_b200/, and neither side
 * imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Nature of the result: cell list, Verlet list, skin and SFC order are exact
 * accelerations -- they never change the mathematical result -- so for neighbor sets and forces this
 * file is the plain definition (all-pairs O(N^2); an independent cell-list O(N) mode exists only so
 * that large systems finish, and is checked against the O(N^2) mode), and for trajectories it is the
 * integrator written out step by step.
 *
 * What follows the paper, and what the paper leaves to a stated reading:
 *   - neighbor set within r_cut + r_buffer, full list
 *   - minimum image in a cuboid periodic box                      PAPER.md:L133, Alg. 2 line 6 (L458)
 *   - Lennard-Jones, Eq. (1)
 *   - harmonic bond U = k (r - r0)^2, Eq. (7) (no 1/2)
 *   - bonds act from both ends, no exclusions
 *   - velocity-Verlet NVE / "BD" (Langevin) / GW-VV for DPD
 *   - harmonic repulsion Eq. (2), Gaussian repulsion Eq. (3)
 *   - tabulated pair potential: cubic spline in z = r^2, Eq. (12); F = -2 r dV/dz, Eq. (11);
 *     cutoff = "point < Npoint", Alg. 2 lines 8-12
 *   - tabulated angle and torsion potentials: Eq. (12) with x = theta on [0, pi] and x = phi on [-pi, pi]
 *     (L118, L127: "x corresponds to z, theta, and phi")
 *   - tabulated bond potential: the same spline in z = r^2 per bond type (L118: "numerical non-bonded,
 *     bond ... potentials"); a bond past the end of its table is an error (reading c-32)
 *   - angle potentials Eqs. (8), (9) and the periodic dihedral Eq. (10), each interaction
 *     stored under every member with its position
 *     (theta = angle at the middle bead between the two bonds, pi for a straight chain; phi = 0
 *     for cis, pi for trans: DESIGN.md readings c-26, c-27)
 *   - NVT by Nose-Hoover, Andersen or Berendsen thermostat: named only
 *     (leapfrog forms with the temperature of the half-step velocities; readings c-28..c-30)
 *   - NPH / NPT by the Andersen barostat: named only
 *     (Andersen 1980's extended Hamiltonian with the volume as a coordinate, integrated by a symmetric
 *     splitting; NPT adds Andersen's stochastic collisions; reading c-31)
 *   - FENE, WCA, the DPD force law, Philox: not in PAPER.md; readings c-3..c-8:
 *     Kremer-Grest FENE, Groot-Warren DPD with uniform unit-variance noise, Philox4x32-10
 *     (Salmon et al., SC'11) keyed (seed; min tag, max tag, step, stream).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms of Eq. (1) and FENE+WCA, force =
 * -grad(energy) by central differences, O(N^2) vs cell mode, Newton's third law / zero net force,
 * translation / image / permutation invariance, NVE conservation ~ dt^2 and time reversal, harmonic
 * dimer frequency (omega = 2 sqrt(k) under Eq. (7)), free flight, Philox known answers, thermostat
 * temperatures.  Unpinned: equilibrium <Rg^2> of the melts in absolute terms ("parity unpinned";
 * compared GPU-vs-oracle only).
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_PAIR_NONE = 0, ORC_PAIR_LJ = 1, ORC_PAIR_DPD = 2, ORC_PAIR_HARMONIC = 3, ORC_PAIR_GAUSS = 4, ORC_PAIR_TABLE = 5 };
enum { ORC_BOND_NONE = 0, ORC_BOND_FENE = 1, ORC_BOND_HARMONIC = 2, ORC_BOND_TABLE = 3 };
enum { ORC_NVE = 0, ORC_LANGEVIN = 1, ORC_GWVV = 2, ORC_NOSE_HOOVER = 3, ORC_ANDERSEN = 4, ORC_BERENDSEN = 5,
       ORC_NPH = 6, ORC_NPT = 7 };
enum { ORC_OK = 0, ORC_ERR_BOND_OVERSTRETCH = -7, ORC_ERR_ARG = -1 };

typedef struct {
    int64_t n;              /* beads */
    int32_t n_types;
    int32_t pair_style;
    int32_t bond_style;
    int32_t integrator;
    double box[3];          /* origin-centred cuboid: x in [-L/2, L/2) */
    double dt, kT, gamma, lambda;
    uint64_t seed;
    const double *eps;      /* [n_types^2]  LJ epsilon | DPD a           */
    const double *sigma;    /* [n_types^2]  LJ sigma   | unused          */
    const double *rc;       /* [n_types^2]  cutoff                        */
    const double *ushift;   /* [n_types^2]  LJ energy shift (0 = plain cut) */
    int64_t n_bonds;
    const int32_t *bond_i, *bond_j, *bond_type;
    const double *bond_k, *bond_r0;     /* per bond type; FENE: r0 is R0 */
    const int32_t *type;    /* [n] */
    const double *mass;     /* [n] */
    int32_t use_cells;      /* 0: all pairs O(N^2) (the definition); 1: cell-list O(N) */
    int32_t n_threads;      /* OpenMP threads for the per-bead loops; <=0: library default */
    /* ORC_PAIR_TABLE (Eqs. 11-12, Alg. 2): cubic-spline coefficients on a grid of z = r^2,       */
    /* table[((ti * n_types + tj) * table_points + point) * 4 + {0,1,2,3}] = c0, c1, c2, c3       */
    const double *table;
    int32_t table_points;   /* Npoint: a pair interacts iff int(r^2 / interval) < Npoint */
    double table_interval;
    /* Angles (i, j, k), j the middle bead, and dihedrals (i, j, k, l)      PAPER.md:L97, Eqs. (8)-(10) L103-114 */
    int32_t angle_style;    /* 0 none, 1 Eq. (8) k (theta - theta0)^2, 2 Eq. (9) k (cos theta - cos theta0)^2 */
    int64_t n_angles;
    const int32_t *angle_i, *angle_j, *angle_k, *angle_type;
    const double *angle_kk, *angle_t0;      /* per angle type */
    int64_t n_dihedrals;    /* Eq. (10): k [1 + cos(n phi - delta)] */
    const int32_t *dih_i, *dih_j, *dih_k, *dih_l, *dih_type;
    const double *dih_kk, *dih_delta;       /* per dihedral type */
    const int32_t *dih_n;
    /* NVT thermostats (equations: DESIGN.md readings c-28..c-30), leapfrog form.  `gamma` is the
       coupling rate: Nose-Hoover 1/tau, Berendsen 1/tau_T, Andersen collision frequency nu.  thermo[0] = 1 once a
       half-step velocity exists, thermo[1] = its kinetic energy sum 1/2 m u^2, thermo[2] = Nose-Hoover xi.           */
    double *thermo;
    /* Andersen barostat (reading c-31): baro[0] = P_ext, baro[1] = piston mass M, baro[2] = piston
       momentum Pi = M dV/dt, baro[3] = virial W = sum over pairs and bonds of r_ij . F_ij at the current positions,
       baro[4] = 1 once baro[3] is valid.  The volume is box[0] box[1] box[2]: orc_run rescales box[] in place.       */
    double *baro;
    /* ORC_BOND_TABLE: "numerical ... bond ... potentials" as cubic splines on a grid of z = r^2, Eq. (12),
       F = -2 r dV/dz, Eq. (11): btable[(bond_type * btable_points + point) * 4 + {0,1,2,3}] = c0..c3 with one grid interval
       per bond type.  A bond stretched past its table (point >= btable_points) has no defined energy: reported as
       ORC_ERR_BOND_OVERSTRETCH, no force (reading c-32).                                                    */
    const double *btable;
    int32_t btable_points;
    const double *btable_interval;      /* per bond type */
    /* angle_style 3 / dtable_points > 0: "numerical ... angle, and torsion potentials", Eq. (12) with
       x = theta on [0, pi] (interval pi / atable_points) and x = phi on [-pi, pi] (interval 2 pi / dtable_points,
       grid point k at -pi + k interval); atable[(angle_type * atable_points + point) * 4 + {0..3}], dtable likewise.   */
    const double *atable;
    int32_t atable_points;
    const double *dtable;
    int32_t dtable_points;
} orc_params;

/* ------------------------------------------------------------------------------------------ */
/* O6. Philox4x32-10 exactly as published (Salmon, Moraes, Dror, Shaw, SC'11).                  */
void orc_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;      /* multipliers */
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;      /* Weyl key increments */
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Uniform in (0,1) from the top 24 bits of a word, u = (k + 1/2) 2^-24.  The method only uses the
   symmetric variate 2u - 1 = (2k + 1 - 2^24) 2^-24, which is exact in fp32 as well as fp64. */
double orc_u24(uint32_t x) { return ((double)(x >> 8) + 0.5) * (1.0 / 16777216.0); }

/* counter = (A, B, step low 32, stream); key = (seed low 32, seed high 32) */
static void noise_words(uint64_t seed, uint32_t a, uint32_t b, uint64_t step, uint32_t stream, uint32_t out[4])
{
    uint32_t ctr[4] = { a, b, (uint32_t)(step & 0xFFFFFFFFu), stream };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    orc_philox4x32_10(ctr, key, out);
}

/* DPD pair noise theta_ij = theta_ji: uniform, zero mean, unit variance (reading c-4). */
double orc_pair_theta(uint64_t seed, uint64_t step, int64_t tag_i, int64_t tag_j)
{
    uint32_t lo = (uint32_t)(tag_i < tag_j ? tag_i : tag_j);
    uint32_t hi = (uint32_t)(tag_i < tag_j ? tag_j : tag_i);
    uint32_t w[4];
    noise_words(seed, lo, hi, step, 0u, w);
    return sqrt(3.0) * (2.0 * orc_u24(w[0]) - 1.0);
}

/* Langevin per-bead noise xi in (-1,1)^3, variance 1/3 per component. */
void orc_bead_xi(uint64_t seed, uint64_t step, int64_t tag, double xi[3])
{
    uint32_t w[4];
    noise_words(seed, (uint32_t)tag, 0u, step, 1u, w);
    xi[0] = 2.0 * orc_u24(w[0]) - 1.0;
    xi[1] = 2.0 * orc_u24(w[1]) - 1.0;
    xi[2] = 2.0 * orc_u24(w[2]) - 1.0;
}

/* ------------------------------------------------------------------------------------------ */
/* O1. Geometry.                                                                                */
double orc_min_image(double d, double L) { return d - L * nearbyint(d / L); }

static double wrap1(double x, double L)
{
    /* one conditional add/subtract per component: a step never moves a bead by a box length */
    if (x >= 0.5 * L) x -= L;
    else if (x < -0.5 * L) x += L;
    return x;
}

/* ------------------------------------------------------------------------------------------ */
/* The oracle's own cell list (used only when use_cells = 1): n_d = floor(L_d / r), w_d = L_d / n_d. */
typedef struct {
    int nc[3];
    int64_t *start;     /* [ncells+1] */
    int64_t *item;      /* [n] bead ids grouped by cell */
    int ok;             /* 0: fewer than 3 cells in some dimension -> caller must use all pairs */
} orc_cells;

static int cell_coord(double x, double L, int nc)
{
    double u = (x + 0.5 * L) / L;
    u -= floor(u);                          /* beads given outside the box land in their image's cell */
    int c = (int)floor(u * nc);
    if (c < 0) c = 0;
    if (c >= nc) c = nc - 1;
    return c;
}

static void cells_build(orc_cells *cl, int64_t n, const double *pos, const double box[3], double r)
{
    cl->ok = 1;
    for (int d = 0; d < 3; ++d) {
        cl->nc[d] = (int)floor(box[d] / r);
        if (cl->nc[d] < 3) cl->ok = 0;
    }
    cl->start = NULL; cl->item = NULL;
    if (!cl->ok) return;
    int64_t ncells = (int64_t)cl->nc[0] * cl->nc[1] * cl->nc[2];
    cl->start = (int64_t *)calloc((size_t)ncells + 1, sizeof(int64_t));
    cl->item = (int64_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int64_t));
    int64_t *cid = (int64_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) {
        int cx = cell_coord(pos[3 * i + 0], box[0], cl->nc[0]);
        int cy = cell_coord(pos[3 * i + 1], box[1], cl->nc[1]);
        int cz = cell_coord(pos[3 * i + 2], box[2], cl->nc[2]);
        cid[i] = ((int64_t)cz * cl->nc[1] + cy) * cl->nc[0] + cx;
        cl->start[cid[i] + 1] += 1;
    }
    for (int64_t c = 0; c < ncells; ++c) cl->start[c + 1] += cl->start[c];
    int64_t *fill = (int64_t *)calloc((size_t)ncells, sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = cid[i];
        cl->item[cl->start[c] + fill[c]] = i;
        fill[c] += 1;
    }
    free(fill); free(cid);
}

static void cells_free(orc_cells *cl) { free(cl->start); free(cl->item); }

/* ------------------------------------------------------------------------------------------ */
/* O2. Neighbor set S = {(i,j), i<j : |minimg(r_i - r_j)|^2 < r_list^2}.        */
/* Returns the number of pairs; writes at most cap of them as (i,j) with i<j.                   */
int64_t orc_neighbor_pairs(int64_t n, const double *pos, const double box[3], double r_list,
                           int32_t use_cells, int64_t cap, int32_t *pairs)
{
    const double r2l = r_list * r_list;
    int64_t cnt = 0;
    orc_cells cl; cl.ok = 0; cl.start = NULL; cl.item = NULL;
    if (use_cells) cells_build(&cl, n, pos, box, r_list);
    if (!use_cells || !cl.ok) {
        for (int64_t i = 0; i < n; ++i)
            for (int64_t j = i + 1; j < n; ++j) {
                double dx = orc_min_image(pos[3 * i + 0] - pos[3 * j + 0], box[0]);
                double dy = orc_min_image(pos[3 * i + 1] - pos[3 * j + 1], box[1]);
                double dz = orc_min_image(pos[3 * i + 2] - pos[3 * j + 2], box[2]);
                if (dx * dx + dy * dy + dz * dz < r2l) {
                    if (cnt < cap) { pairs[2 * cnt] = (int32_t)i; pairs[2 * cnt + 1] = (int32_t)j; }
                    ++cnt;
                }
            }
        if (use_cells) cells_free(&cl);
        return cnt;
    }
    for (int64_t i = 0; i < n; ++i) {
        int cx = cell_coord(pos[3 * i + 0], box[0], cl.nc[0]);
        int cy = cell_coord(pos[3 * i + 1], box[1], cl.nc[1]);
        int cz = cell_coord(pos[3 * i + 2], box[2], cl.nc[2]);
        for (int oz = -1; oz <= 1; ++oz) for (int oy = -1; oy <= 1; ++oy) for (int ox = -1; ox <= 1; ++ox) {
            int ax = (cx + ox + cl.nc[0]) % cl.nc[0];
            int ay = (cy + oy + cl.nc[1]) % cl.nc[1];
            int az = (cz + oz + cl.nc[2]) % cl.nc[2];
            int64_t c = ((int64_t)az * cl.nc[1] + ay) * cl.nc[0] + ax;
            for (int64_t s = cl.start[c]; s < cl.start[c + 1]; ++s) {
                int64_t j = cl.item[s];
                if (j <= i) continue;
                double dx = orc_min_image(pos[3 * i + 0] - pos[3 * j + 0], box[0]);
                double dy = orc_min_image(pos[3 * i + 1] - pos[3 * j + 1], box[1]);
                double dz = orc_min_image(pos[3 * i + 2] - pos[3 * j + 2], box[2]);
                if (dx * dx + dy * dy + dz * dz < r2l) {
                    if (cnt < cap) { pairs[2 * cnt] = (int32_t)i; pairs[2 * cnt + 1] = (int32_t)j; }
                    ++cnt;
                }
            }
        }
    }
    cells_free(&cl);
    return cnt;
}

/* Andersen thermostat (reading c-29): bead `tag` collides with the heat bath in the kick of time level `step` iff
   the top 24 bits of Philox(tag, 0, step, stream 3) word 0 are < floor(nu dt 2^24); its new velocity components are
   sqrt(kT/m) times three standard normals by Box-Muller from the four words of stream 2:
   g0 = sqrt(-2 ln u0) cos(2 pi u1), g1 = sqrt(-2 ln u0) sin(2 pi u1), g2 = sqrt(-2 ln u2) cos(2 pi u3). */
int orc_andersen_hit(uint64_t seed, uint64_t step, int64_t tag, double nu_dt)
{
    uint32_t w[4];
    noise_words(seed, (uint32_t)tag, 0u, step, 3u, w);
    double thr = floor(nu_dt * 16777216.0);
    return (double)(w[0] >> 8) < thr;
}

void orc_andersen_normals(uint64_t seed, uint64_t step, int64_t tag, double g[3])
{
    uint32_t w[4];
    noise_words(seed, (uint32_t)tag, 0u, step, 2u, w);
    const double two_pi = 6.283185307179586476925286766559;
    double r0 = sqrt(-2.0 * log(orc_u24(w[0]))), r2 = sqrt(-2.0 * log(orc_u24(w[2])));
    g[0] = r0 * cos(two_pi * orc_u24(w[1]));
    g[1] = r0 * sin(two_pi * orc_u24(w[1]));
    g[2] = r2 * cos(two_pi * orc_u24(w[3]));
}

/* ------------------------------------------------------------------------------------------ */
/* O3 + O5. Contribution of bead j to the force on bead i.                                      */
/* vel is the velocity the DPD dissipative term sees (v-tilde in GW-VV); unused for LJ.         */
/* Adds to f[3]; adds the FULL pair energy to *u (the caller halves the double count).          */
/* Returns 1 if the pair is inside its cutoff.                                                  */
static int pair_term(const orc_params *p, const double *pos, const double *vel, uint64_t step,
                     int64_t i, int64_t j, double f[3], double *u)
{
    double dx = orc_min_image(pos[3 * i + 0] - pos[3 * j + 0], p->box[0]);
    double dy = orc_min_image(pos[3 * i + 1] - pos[3 * j + 1], p->box[1]);
    double dz = orc_min_image(pos[3 * i + 2] - pos[3 * j + 2], p->box[2]);
    double r2 = dx * dx + dy * dy + dz * dz;
    int t = p->type[i] * p->n_types + p->type[j];
    if (p->pair_style == ORC_PAIR_TABLE) {
        /* Alg. 2 lines 8-12: point = int(dr^2 / interval); if point < Npoint: delta = dr^2 -
           point * interval; Eq. (12): V = c0 + c1 d + c2 d^2 + c3 d^3; Eq. (11): F = -2 r dV/dz */
        long point = (long)(r2 / p->table_interval);
        if (!(point < p->table_points)) return 0;
        const double *c = p->table + ((size_t)t * p->table_points + point) * 4;
        double d = r2 - (double)point * p->table_interval;
        double dvdz = c[1] + 2.0 * c[2] * d + 3.0 * c[3] * d * d;
        double fs = -2.0 * dvdz;
        f[0] += fs * dx; f[1] += fs * dy; f[2] += fs * dz;
        *u += c[0] + c[1] * d + c[2] * d * d + c[3] * d * d * d;
        return 1;
    }
    double rc = p->rc[t];
    if (!(r2 < rc * rc)) return 0;
    if (p->pair_style == ORC_PAIR_HARMONIC) {
        /* Eq. (2): U = alpha (1 - r/r_cut)^2 (no 1/2);  F_i = -dU/dr e = (2 alpha / r_cut) (1 - r/r_cut) e */
        double a = p->eps[t];
        double r = sqrt(r2);
        double w = 1.0 - r / rc;
        *u += a * w * w;
        if (r > 0.0) {
            double fs = 2.0 * a / rc * w / r;
            f[0] += fs * dx; f[1] += fs * dy; f[2] += fs * dz;
        }
        return 1;
    }
    if (p->pair_style == ORC_PAIR_GAUSS) {
        /* Eq. (3): U = eps exp(-1/2 (r/sigma)^2);  F_i = (eps / sigma^2) exp(-1/2 (r/sigma)^2) r_ij;
           truncated at r_cut, energy shifted by U(r_cut) when asked (as for LJ, reading c-9) */
        double e = p->eps[t], sig = p->sigma[t];
        double g = e * exp(-0.5 * r2 / (sig * sig));
        double fs = g / (sig * sig);
        f[0] += fs * dx; f[1] += fs * dy; f[2] += fs * dz;
        *u += g - p->ushift[t];
        return 1;
    }
    if (p->pair_style == ORC_PAIR_LJ) {
        /* Eq. (1): U = 4 eps [(s/r)^12 - (s/r)^6];  F_i = 24 eps / r^2 [2 (s/r)^12 - (s/r)^6] r_ij */
        double eps = p->eps[t], sig = p->sigma[t];
        double s2 = sig * sig / r2;
        double s6 = s2 * s2 * s2;
        double s12 = s6 * s6;
        double fs = 24.0 * eps / r2 * (2.0 * s12 - s6);
        f[0] += fs * dx; f[1] += fs * dy; f[2] += fs * dz;
        *u += 4.0 * eps * (s12 - s6) - p->ushift[t];
        return 1;
    }
    if (p->pair_style == ORC_PAIR_DPD) {
        /* Groot-Warren (reading c-3): F_ij = [a w - gamma w^2 (e.v_ij) + sigma_R w theta / sqrt(dt)] e */
        if (r2 < 1e-12) return 1;   /* e undefined */
        double r = sqrt(r2);
        double w = 1.0 - r / rc;
        double ex = dx / r, ey = dy / r, ez = dz / r;
        double dvx = vel[3 * i + 0] - vel[3 * j + 0];
        double dvy = vel[3 * i + 1] - vel[3 * j + 1];
        double dvz = vel[3 * i + 2] - vel[3 * j + 2];
        double edv = ex * dvx + ey * dvy + ez * dvz;
        double sigma_r = sqrt(2.0 * p->gamma * p->kT);
        double theta = orc_pair_theta(p->seed, step, i, j);
        double a = p->eps[t];
        double fs = a * w - p->gamma * w * w * edv + sigma_r * w * theta / sqrt(p->dt);
        f[0] += fs * ex; f[1] += fs * ey; f[2] += fs * ez;
        *u += 0.5 * a * rc * w * w;
        return 1;
    }
    return 0;
}

static double max_cutoff(const orc_params *p)
{
    double r = 0.0;
    for (int t = 0; t < p->n_types * p->n_types; ++t) if (p->rc[t] > r) r = p->rc[t];
    return r;
}

/* O3-O5. Conservative (+ DPD dissipative/random) forces at positions pos.                      */
/* out[0] = pair energy, out[1] = bond energy, out[2] = number of unique pairs inside r_c.      */
int orc_pair_bond_forces(const orc_params *p, const double *pos, const double *vel, uint64_t step,
                         double *frc, double out[3])
{
    const int64_t n = p->n;
    double pe_pair = 0.0, n_in = 0.0;
    orc_cells cl; cl.ok = 0; cl.start = NULL; cl.item = NULL;
    int have_pairs = (p->pair_style != ORC_PAIR_NONE);
    if (have_pairs && p->use_cells) cells_build(&cl, n, pos, p->box, max_cutoff(p));
#ifdef _OPENMP
    if (p->n_threads > 0) omp_set_num_threads(p->n_threads);
#endif
    if (!have_pairs) {
        memset(frc, 0, (size_t)(3 * n) * sizeof(double));
    } else if (!p->use_cells || !cl.ok) {
#pragma omp parallel for schedule(static) reduction(+ : pe_pair, n_in)
        for (int64_t i = 0; i < n; ++i) {
            double f[3] = { 0, 0, 0 }, u = 0.0;
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                n_in += pair_term(p, pos, vel, step, i, j, f, &u);
            }
            frc[3 * i] = f[0]; frc[3 * i + 1] = f[1]; frc[3 * i + 2] = f[2];
            pe_pair += 0.5 * u;
        }
    } else {
#pragma omp parallel for schedule(static) reduction(+ : pe_pair, n_in)
        for (int64_t i = 0; i < n; ++i) {
            double f[3] = { 0, 0, 0 }, u = 0.0;
            int cx = cell_coord(pos[3 * i + 0], p->box[0], cl.nc[0]);
            int cy = cell_coord(pos[3 * i + 1], p->box[1], cl.nc[1]);
            int cz = cell_coord(pos[3 * i + 2], p->box[2], cl.nc[2]);
            for (int oz = -1; oz <= 1; ++oz) for (int oy = -1; oy <= 1; ++oy) for (int ox = -1; ox <= 1; ++ox) {
                int ax = (cx + ox + cl.nc[0]) % cl.nc[0];
                int ay = (cy + oy + cl.nc[1]) % cl.nc[1];
                int az = (cz + oz + cl.nc[2]) % cl.nc[2];
                int64_t c = ((int64_t)az * cl.nc[1] + ay) * cl.nc[0] + ax;
                for (int64_t s = cl.start[c]; s < cl.start[c + 1]; ++s) {
                    int64_t j = cl.item[s];
                    if (j == i) continue;
                    n_in += pair_term(p, pos, vel, step, i, j, f, &u);
                }
            }
            frc[3 * i] = f[0]; frc[3 * i + 1] = f[1]; frc[3 * i + 2] = f[2];
            pe_pair += 0.5 * u;
        }
    }
    if (have_pairs && p->use_cells) cells_free(&cl);

    /* O4. Bonds: each bond (i,j) once, acting on both ends (the GPU evaluates it from both ends,
       PAPER.md:L97; the sum is the same). */
    double pe_bond = 0.0;
    int status = ORC_OK;
    if (p->bond_style != ORC_BOND_NONE) {
        for (int64_t b = 0; b < p->n_bonds; ++b) {
            int64_t i = p->bond_i[b], j = p->bond_j[b];
            double k = p->bond_k[p->bond_type[b]], r0 = p->bond_r0[p->bond_type[b]];
            double dx = orc_min_image(pos[3 * i + 0] - pos[3 * j + 0], p->box[0]);
            double dy = orc_min_image(pos[3 * i + 1] - pos[3 * j + 1], p->box[1]);
            double dz = orc_min_image(pos[3 * i + 2] - pos[3 * j + 2], p->box[2]);
            double r2 = dx * dx + dy * dy + dz * dz;
            double fs;
            if (p->bond_style == ORC_BOND_FENE) {
                /* U = -1/2 k R0^2 ln(1 - r^2/R0^2);  F_i = -k r_ij / (1 - r^2/R0^2)   (reading c-8) */
                double q = 1.0 - r2 / (r0 * r0);
                if (!(q > 0.0)) { status = ORC_ERR_BOND_OVERSTRETCH; continue; }
                fs = -k / q;
                pe_bond += -0.5 * k * r0 * r0 * log(q);
            } else if (p->bond_style == ORC_BOND_TABLE) {
                /* Eqs. (11)-(12) with x = z = r^2: point = int(z / interval); delta = z - point * interval */
                double h = p->btable_interval[p->bond_type[b]];
                long point = (long)(r2 / h);
                if (!(point < p->btable_points)) { status = ORC_ERR_BOND_OVERSTRETCH; continue; }
                const double *c = p->btable + ((size_t)p->bond_type[b] * p->btable_points + point) * 4;
                double d = r2 - (double)point * h;
                fs = -2.0 * (c[1] + 2.0 * c[2] * d + 3.0 * c[3] * d * d);
                pe_bond += c[0] + c[1] * d + c[2] * d * d + c[3] * d * d * d;
            } else {
                /* Eq. (7): U = k (r - r0)^2;  F_i = -2 k (1 - r0/r) r_ij */
                double r = sqrt(r2);
                if (r0 == 0.0) fs = -2.0 * k;
                else fs = (r > 0.0) ? -2.0 * k * (1.0 - r0 / r) : 0.0;
                pe_bond += k * (r - r0) * (r - r0);
            }
            frc[3 * i] += fs * dx; frc[3 * i + 1] += fs * dy; frc[3 * i + 2] += fs * dz;
            frc[3 * j] -= fs * dx; frc[3 * j + 1] -= fs * dy; frc[3 * j + 2] -= fs * dz;
        }
    }
    /* Angles, Eqs. (8)-(9): a = r_i - r_j, b = r_k - r_j (minimum image), cos(theta) = a.b / |a||b|.
       d cos(theta) / d r_i = (b^ - cos(theta) a^) / |a|, d/d r_k = (a^ - cos(theta) b^) / |b|, and the middle bead takes
       minus their sum.  Each angle once, acting on its three beads (the GPU evaluates it three times, L97).      */
    if (p->angle_style != 0) {
        for (int64_t q = 0; q < p->n_angles; ++q) {
            int64_t i = p->angle_i[q], j = p->angle_j[q], k = p->angle_k[q];
            double kk = p->angle_kk[p->angle_type[q]], t0 = p->angle_t0[p->angle_type[q]];
            double a[3], b[3];
            for (int d = 0; d < 3; ++d) {
                a[d] = orc_min_image(pos[3 * i + d] - pos[3 * j + d], p->box[d]);
                b[d] = orc_min_image(pos[3 * k + d] - pos[3 * j + d], p->box[d]);
            }
            double la = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
            double lb = sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
            double c = (a[0] * b[0] + a[1] * b[1] + a[2] * b[2]) / (la * lb);
            if (c > 1.0) c = 1.0;
            if (c < -1.0) c = -1.0;
            double dudc;                                  /* dU / d cos(theta) */
            if (p->angle_style == 1) {
                /* Eq. (8): U = k (theta - theta0)^2;  dU/dcos = dU/dtheta * (-1 / sin(theta)) */
                double th = acos(c), sn = sqrt(1.0 - c * c);
                if (sn < 1e-12) sn = 1e-12;
                pe_bond += kk * (th - t0) * (th - t0);
                dudc = -2.0 * kk * (th - t0) / sn;
            } else if (p->angle_style == 3) {
                /* Eq. (12) with x = theta: point = int(theta / h), delta = theta - point h; dU/dcos = -U'(theta) / sin */
                double th = acos(c), sn = sqrt(1.0 - c * c);
                if (sn < 1e-12) sn = 1e-12;
                double h = M_PI / p->atable_points;
                long point = (long)(th / h);
                if (point > p->atable_points - 1) point = p->atable_points - 1;
                const double *cf = p->atable + ((size_t)p->angle_type[q] * p->atable_points + point) * 4;
                double d = th - (double)point * h;
                pe_bond += cf[0] + cf[1] * d + cf[2] * d * d + cf[3] * d * d * d;
                dudc = -(cf[1] + 2.0 * cf[2] * d + 3.0 * cf[3] * d * d) / sn;
            } else {
                /* Eq. (9): U = k (cos(theta) - cos(theta0))^2 */
                double dc = c - cos(t0);
                pe_bond += kk * dc * dc;
                dudc = 2.0 * kk * dc;
            }
            for (int d = 0; d < 3; ++d) {
                double fi = -dudc * (b[d] / lb - c * a[d] / la) / la;
                double fk = -dudc * (a[d] / la - c * b[d] / lb) / lb;
                frc[3 * i + d] += fi; frc[3 * k + d] += fk; frc[3 * j + d] -= fi + fk;
            }
        }
    }
    /* Dihedrals, Eq. (10): b1 = r_j - r_i, b2 = r_k - r_j, b3 = r_l - r_k, n1 = b1 x b2, n2 = b2 x b3,
       phi = atan2(|b2| b1.n2, n1.n2) (0 = cis, pi = trans).  d phi / d r_i = -|b2| n1 / |n1|^2, d phi / d r_l = |b2| n2 / |n2|^2,
       d phi / d r_j = -(1 + b1.b2 / |b2|^2) dphi/dr_i + (b3.b2 / |b2|^2) dphi/dr_l, d phi / d r_k = -(1 + b3.b2 / |b2|^2) dphi/dr_l
       + (b1.b2 / |b2|^2) dphi/dr_i  (the textbook form, e.g. Blondel and Karplus 1996; pinned by central differences).  */
    for (int64_t q = 0; q < p->n_dihedrals; ++q) {
        int64_t m[4] = { p->dih_i[q], p->dih_j[q], p->dih_k[q], p->dih_l[q] };
        double kk = p->dih_kk[p->dih_type[q]], dl = p->dih_delta[p->dih_type[q]];
        int nn = p->dih_n[p->dih_type[q]];
        double b1[3], b2[3], b3[3], n1[3], n2[3];
        for (int d = 0; d < 3; ++d) {
            b1[d] = orc_min_image(pos[3 * m[1] + d] - pos[3 * m[0] + d], p->box[d]);
            b2[d] = orc_min_image(pos[3 * m[2] + d] - pos[3 * m[1] + d], p->box[d]);
            b3[d] = orc_min_image(pos[3 * m[3] + d] - pos[3 * m[2] + d], p->box[d]);
        }
        n1[0] = b1[1] * b2[2] - b1[2] * b2[1]; n1[1] = b1[2] * b2[0] - b1[0] * b2[2]; n1[2] = b1[0] * b2[1] - b1[1] * b2[0];
        n2[0] = b2[1] * b3[2] - b2[2] * b3[1]; n2[1] = b2[2] * b3[0] - b2[0] * b3[2]; n2[2] = b2[0] * b3[1] - b2[1] * b3[0];
        double l2 = sqrt(b2[0] * b2[0] + b2[1] * b2[1] + b2[2] * b2[2]);
        double n1s = n1[0] * n1[0] + n1[1] * n1[1] + n1[2] * n1[2];
        double n2s = n2[0] * n2[0] + n2[1] * n2[1] + n2[2] * n2[2];
        if (n1s < 1e-24 || n2s < 1e-24) continue;     /* three beads in line: phi undefined, no force */
        double phi = atan2(l2 * (b1[0] * n2[0] + b1[1] * n2[1] + b1[2] * n2[2]), n1[0] * n2[0] + n1[1] * n2[1] + n1[2] * n2[2]);
        double dudphi;
        if (p->dtable_points > 0) {
            /* Eq. (12) with x = phi: grid point k at -pi + k h, h = 2 pi / Npoint */
            double h = 2.0 * M_PI / p->dtable_points, x = phi + M_PI;
            long point = (long)(x / h);
            if (point < 0) point = 0;
            if (point > p->dtable_points - 1) point = p->dtable_points - 1;
            const double *cf = p->dtable + ((size_t)p->dih_type[q] * p->dtable_points + point) * 4;
            double d = x - (double)point * h;
            pe_bond += cf[0] + cf[1] * d + cf[2] * d * d + cf[3] * d * d * d;
            dudphi = cf[1] + 2.0 * cf[2] * d + 3.0 * cf[3] * d * d;
        } else {
            pe_bond += kk * (1.0 + cos(nn * phi - dl));
            dudphi = -kk * nn * sin(nn * phi - dl);
        }
        double s12 = (b1[0] * b2[0] + b1[1] * b2[1] + b1[2] * b2[2]) / (l2 * l2);
        double s32 = (b3[0] * b2[0] + b3[1] * b2[1] + b3[2] * b2[2]) / (l2 * l2);
        for (int d = 0; d < 3; ++d) {
            double gi = -l2 * n1[d] / n1s, gl = l2 * n2[d] / n2s;
            double gj = -(1.0 + s12) * gi + s32 * gl, gk = -(1.0 + s32) * gl + s12 * gi;
            frc[3 * m[0] + d] -= dudphi * gi; frc[3 * m[1] + d] -= dudphi * gj;
            frc[3 * m[2] + d] -= dudphi * gk; frc[3 * m[3] + d] -= dudphi * gl;
        }
    }
    if (out) { out[0] = pe_pair; out[1] = pe_bond; out[2] = 0.5 * n_in; }
    return status;
}

/* The virial W = sum over interacting pairs and bonds of r_ij . F_ij (F_ij: force on i from j, r_ij the minimum-image
 * displacement; each pair once), written out as that definition: all pairs, O(N^2).  Angle and dihedral energies do not
 * change under a uniform scaling of the coordinates, so they add nothing.  With it the instantaneous pressure is
 * P = (2 K + W) / (3 V)  (Andersen 1980, Eq. 3.4c; PAPER.md:L133 names the barostat only).                       */
int orc_virial(const orc_params *p, const double *pos, double *w_out)
{
    const int64_t n = p->n;
    double w = 0.0;
    int status = ORC_OK;
    if (p->pair_style != ORC_PAIR_NONE) {
#pragma omp parallel for schedule(static) reduction(+ : w)
        for (int64_t i = 0; i < n; ++i)
            for (int64_t j = i + 1; j < n; ++j) {
                double f[3] = { 0, 0, 0 }, u = 0.0;
                if (!pair_term(p, pos, pos, 0, i, j, f, &u)) continue;
                for (int d = 0; d < 3; ++d)
                    w += f[d] * orc_min_image(pos[3 * i + d] - pos[3 * j + d], p->box[d]);
            }
    }
    if (p->bond_style != ORC_BOND_NONE) {
        for (int64_t b = 0; b < p->n_bonds; ++b) {
            int64_t i = p->bond_i[b], j = p->bond_j[b];
            double k = p->bond_k[p->bond_type[b]], r0 = p->bond_r0[p->bond_type[b]];
            double r2 = 0.0;
            for (int d = 0; d < 3; ++d) {
                double x = orc_min_image(pos[3 * i + d] - pos[3 * j + d], p->box[d]);
                r2 += x * x;
            }
            if (p->bond_style == ORC_BOND_FENE) {
                double q = 1.0 - r2 / (r0 * r0);                     /* F_ij = -k r_ij / q */
                if (!(q > 0.0)) { status = ORC_ERR_BOND_OVERSTRETCH; continue; }
                w += -k / q * r2;
            } else if (p->bond_style == ORC_BOND_TABLE) {
                double h = p->btable_interval[p->bond_type[b]];           /* F_ij = -2 dV/dz r_ij */
                long point = (long)(r2 / h);
                if (!(point < p->btable_points)) { status = ORC_ERR_BOND_OVERSTRETCH; continue; }
                const double *c = p->btable + ((size_t)p->bond_type[b] * p->btable_points + point) * 4;
                double d = r2 - (double)point * h;
                w += -2.0 * (c[1] + 2.0 * c[2] * d + 3.0 * c[3] * d * d) * r2;
            } else {
                double r = sqrt(r2);                                 /* F_ij = -2 k (r - r0) r_ij / r */
                w += -2.0 * k * (r - r0) * r;
            }
        }
    }
    *w_out = w;
    return status;
}

/* The force the integrator uses at time level `step` (O7):
 *   NVE, GW-VV : F(pos [, vel])
 *   Langevin   : F_c(pos) - gamma m v + sqrt(6 gamma m kT / dt) xi(tag, step)   (reading c-7)
 * vel is v (initial call), v' (Langevin half-step velocity) or v-tilde (GW-VV).              */
int orc_compute_forces(const orc_params *p, const double *pos, const double *vel, uint64_t step,
                       double *frc, double out[3])
{
    int status = orc_pair_bond_forces(p, pos, vel, step, frc, out);
    if (p->integrator == ORC_LANGEVIN) {
        for (int64_t i = 0; i < p->n; ++i) {
            double xi[3], m = p->mass[i];
            orc_bead_xi(p->seed, step, i, xi);
            double amp = sqrt(6.0 * p->gamma * m * p->kT / p->dt);
            for (int d = 0; d < 3; ++d)
                frc[3 * i + d] += -p->gamma * m * vel[3 * i + d] + amp * xi[d];
        }
    }
    return status;
}

/* O7. n_steps of the integrator, starting at time level step0 with frc = orc_compute_forces(step0). */
/* scratch: 6n doubles (GW-VV: v-tilde and the old acceleration).                                  */
int orc_run(orc_params *p, double *pos, double *vel, double *frc, uint64_t step0, int64_t n_steps,
            double *scratch)
{
    const int64_t n = p->n;
    const double dt = p->dt;
    int status = ORC_OK;
    for (int64_t s = 0; s < n_steps; ++s) {
        uint64_t step = step0 + (uint64_t)s + 1;    /* time level of the new force */
        if (p->integrator >= ORC_NOSE_HOOVER && p->integrator <= ORC_BERENDSEN) {
            /* Leapfrog with a thermostat on the half-step velocity u (vel holds the full-step v^m = u^{m-1/2} + dt/2 a^m
               between steps; a = frc / m is a^m).  First step after a (re)start: u^{1/2} = v^0 + dt/2 a^0, thermostat off.
                 Berendsen (c-30):   lambda = sqrt(1 + dt gamma (kT / T_half - 1));  u' = lambda (u + dt a)
                 Nose-Hoover (c-28): xi += dt gamma^2 (T_half / kT - 1);  u' = [u (1 - dt xi / 2) + dt a] / (1 + dt xi / 2)
                 Andersen (c-29):    u' = u + kick a, then beads hit by the bath draw u' = sqrt(kT/m) g
               with T_half = 2 K_half / (3N - 3) the temperature of the previous half-step velocities; then
               r += dt u';  a = F(r) / m;  v = u' + dt/2 a.                                                           */
            const double dof = n > 1 ? 3.0 * n - 3.0 : 3.0;
            const int have = p->thermo[0] != 0.0;
            double sa = 1.0, sb = 1.0;              /* u' = sa u + sb kick a */
            if (have && p->integrator == ORC_BERENDSEN) {
                double t_half = 2.0 * p->thermo[1] / dof;
                sa = sb = sqrt(1.0 + dt * p->gamma * (p->kT / t_half - 1.0));
            } else if (have && p->integrator == ORC_NOSE_HOOVER) {
                double t_half = 2.0 * p->thermo[1] / dof;
                p->thermo[2] += dt * p->gamma * p->gamma * (t_half / p->kT - 1.0);
                double h = 0.5 * dt * p->thermo[2];
                sa = (1.0 - h) / (1.0 + h); sb = 1.0 / (1.0 + h);
            }
            const double kick = have ? dt : 0.5 * dt;
            double k_half = 0.0;
            for (int64_t i = 0; i < n; ++i) {
                double a[3], u[3], m = p->mass[i];
                for (int d = 0; d < 3; ++d) {
                    a[d] = frc[3 * i + d] / m;
                    double u_old = have ? vel[3 * i + d] - 0.5 * dt * a[d] : vel[3 * i + d];
                    u[d] = sa * u_old + sb * kick * a[d];
                }
                if (p->integrator == ORC_ANDERSEN && orc_andersen_hit(p->seed, step - 1, i, p->gamma * dt)) {
                    double g[3];
                    orc_andersen_normals(p->seed, step - 1, i, g);
                    for (int d = 0; d < 3; ++d) u[d] = sqrt(p->kT / m) * g[d];
                }
                for (int d = 0; d < 3; ++d) {
                    vel[3 * i + d] = u[d];
                    pos[3 * i + d] = wrap1(pos[3 * i + d] + dt * u[d], p->box[d]);
                    k_half += 0.5 * m * u[d] * u[d];
                }
            }
            p->thermo[0] = 1.0; p->thermo[1] = k_half;
            int st = orc_compute_forces(p, pos, vel, step, frc, NULL);
            if (st != ORC_OK) status = st;
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d)
                    vel[3 * i + d] += 0.5 * dt * frc[3 * i + d] / p->mass[i];
        } else if (p->integrator == ORC_NPH || p->integrator == ORC_NPT) {
            /* Andersen barostat (PAPER.md:L133 names it; reading c-31).  Andersen 1980, Eq. 3.2: scaled coordinates
               rho_i = r_i / V^(1/3) with momenta pi_i, the volume V with momentum Pi, and
                   H = sum pi_i^2 / (2 m_i V^(2/3)) + U(V^(1/3) rho) + Pi^2 / (2 M) + P_ext V.
               The physical velocity is v_i = pi_i / (m_i V^(1/3)).  H = H_kin(pi, V) + H_pot(rho, V) + H_pis(Pi), and each
               part alone is solved exactly:
                 H_pot for t:  pi_i += t V^(1/3) F_i  (v_i += t F_i / m_i),   Pi += t (W / (3 V) - P_ext)
                 H_kin for t:  rho_i += t pi_i / (m_i V^(2/3))  (r_i += t v_i),   Pi += t 2 K / (3 V),  K = sum m v^2 / 2
                 H_pis for t:  V += t Pi / M  at fixed rho, pi:  r_i *= mu, v_i /= mu, box *= mu, mu = (V'/V)^(1/3)
               One step is the symmetric product  pot(dt/2) kin(dt/2) pis(dt) kin(dt/2) pot(dt/2): time-reversible and
               second order, velocity-Verlet when M is infinite.  NPT (Andersen's own constant-T proposal, his section
               IV): after the second kin part every bead is hit by the bath with probability nu dt and then draws
               v = sqrt(kT/m) g, with the draws of the NVT Andersen thermostat (c-29).                                  */
            double *b = p->baro;
            if (b[4] == 0.0) { orc_virial(p, pos, &b[3]); b[4] = 1.0; }
            double V = p->box[0] * p->box[1] * p->box[2];
            double K = 0.0;
            b[2] += 0.5 * dt * (b[3] / (3.0 * V) - b[0]);
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d) {
                    vel[3 * i + d] += 0.5 * dt * frc[3 * i + d] / p->mass[i];
                    pos[3 * i + d] += 0.5 * dt * vel[3 * i + d];
                    K += 0.5 * p->mass[i] * vel[3 * i + d] * vel[3 * i + d];
                }
            b[2] += 0.5 * dt * 2.0 * K / (3.0 * V);
            double Vn = V + dt * b[2] / b[1];
            if (!(Vn > 0.0)) return ORC_ERR_ARG;
            double mu = cbrt(Vn / V);
            for (int d = 0; d < 3; ++d) p->box[d] *= mu;
            K = 0.0;
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d) {
                    vel[3 * i + d] /= mu;
                    pos[3 * i + d] = pos[3 * i + d] * mu + 0.5 * dt * vel[3 * i + d];
                    K += 0.5 * p->mass[i] * vel[3 * i + d] * vel[3 * i + d];
                }
            b[2] += 0.5 * dt * 2.0 * K / (3.0 * Vn);
            for (int64_t i = 0; i < n; ++i) {
                for (int d = 0; d < 3; ++d) pos[3 * i + d] = wrap1(pos[3 * i + d], p->box[d]);
                if (p->integrator == ORC_NPT && orc_andersen_hit(p->seed, step - 1, i, p->gamma * dt)) {
                    double g[3];
                    orc_andersen_normals(p->seed, step - 1, i, g);
                    for (int d = 0; d < 3; ++d) vel[3 * i + d] = sqrt(p->kT / p->mass[i]) * g[d];
                }
            }
            int st = orc_compute_forces(p, pos, vel, step, frc, NULL);
            if (st != ORC_OK) status = st;
            st = orc_virial(p, pos, &b[3]);
            if (st != ORC_OK) status = st;
            b[2] += 0.5 * dt * (b[3] / (3.0 * Vn) - b[0]);
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d)
                    vel[3 * i + d] += 0.5 * dt * frc[3 * i + d] / p->mass[i];
        } else if (p->integrator == ORC_NVE || p->integrator == ORC_LANGEVIN) {
            /* v' = v + dt/2 a;  r = r + dt v';  wrap;  a = F(r)/m;  v = v' + dt/2 a */
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d) {
                    vel[3 * i + d] += 0.5 * dt * frc[3 * i + d] / p->mass[i];
                    pos[3 * i + d] = wrap1(pos[3 * i + d] + dt * vel[3 * i + d], p->box[d]);
                }
            int st = orc_compute_forces(p, pos, vel, step, frc, NULL);   /* Langevin drag sees v' */
            if (st != ORC_OK) status = st;
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d)
                    vel[3 * i + d] += 0.5 * dt * frc[3 * i + d] / p->mass[i];
        } else {
            /* GW-VV: r += dt v + dt^2/2 f;  v~ = v + lambda dt f;  f' = F(r, v~);  v += dt/2 (f + f') */
            double *vt = scratch, *f_old = scratch + 3 * n;
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d) {
                    double f = frc[3 * i + d] / p->mass[i];
                    pos[3 * i + d] = wrap1(pos[3 * i + d] + dt * vel[3 * i + d] + 0.5 * dt * dt * f, p->box[d]);
                    vt[3 * i + d] = vel[3 * i + d] + p->lambda * dt * f;
                    f_old[3 * i + d] = f;
                }
            int st = orc_compute_forces(p, pos, vt, step, frc, NULL);
            if (st != ORC_OK) status = st;
            for (int64_t i = 0; i < n; ++i)
                for (int d = 0; d < 3; ++d)
                    vel[3 * i + d] += 0.5 * dt * (f_old[3 * i + d] + frc[3 * i + d] / p->mass[i]);
        }
    }
    return status;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
