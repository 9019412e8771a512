/*
 * gm.h -- C ABI of libgm: the per-timestep short-range force pipeline of GALAMOST-style
 * coarse-grained polymer MD (arXiv 1310.2041, "PAPER.md") on one NVIDIA B200 (sm_100a), fp32.
 *
 * The pipeline:
 *   a1 cell binning by counting sort         PAPER.md:L57 (cell list CL/CN), Alg. 1 Kernel 1 L376-388
 *   a2 space-filling-curve reorder of the    PAPER.md:L33, L199 (SFCPACK memory sort); here the sort key of a1
 *      particle arrays at every rebuild
 *   a3 skin-padded FULL Verlet list NL/NN    PAPER.md:L51 (table form NL[k*Np+i]), L57 (27 cells,
 *                                            r_cut + r_buffer)
 *   a4 rebuild when a bead moved > skin/2
 *   a5 Lennard-Jones / WCA pair force        PAPER.md:L59-61 Eq. (1); loop shape Alg. 2
 *      harmonic / Gaussian repulsion         PAPER.md:L63-72 Eqs. (2), (3)
 *      tabulated pair potential              PAPER.md:L118-129 Eqs. (11)-(12), Alg. 2 L458 (cubic spline in z = r^2)
 *   a6 DPD pair force (Groot-Warren)         PAPER.md:L43, L135, L197 (law itself: ref. 24; DESIGN.md c-3)
 *   a7 bond force from the BL/BN table       PAPER.md:L97, Eq. (7) L99-101 (harmonic); FENE: DESIGN.md c-8
 *      angle and dihedral forces from        PAPER.md:L97 (per-particle tables with the member's position), Eqs. (8)-(10)
 *      per-particle tables                   L103-114
 *   a8 velocity-Verlet NVE / Langevin "BD" / GW-VV
 *   a9 energies (validation quantities)
 *
 * Conventions common to every call
 *   - Every function returns a gm_status (0 = GM_OK, < 0 = error) and never throws, exits or
 *     prints.  gm_last_error() gives a message for the last failing call on that system.
 *   - "host or device": each array argument says which; calls taking `on_device` accept either
 *     (on_device = 0: plain host memory, pinned or not; 1: device memory on the system's GPU).
 *   - Ownership: the caller owns every buffer it passes, including the device workspace and the
 *     CUDA stream.  The library copies inputs in, writes outputs out, and never frees or keeps a
 *     caller pointer other than the workspace and the stream (which must outlive the system).
 *   - All particle arrays cross this boundary in TAG order (the order given to gm_set_particles),
 *     whatever the internal space-filling-curve storage order is.
 *   - The box is an origin-centred cuboid, x_d in [-box_d/2, box_d/2), periodic in all three
 *     dimensions.  Units are reduced (sigma, epsilon, m).
 *   - Work is enqueued on the stream given at creation; calls that return data to the host
 *     (on_device = 0 outputs, gm_energies, gm_get_stats) synchronise that stream before returning.
 *   - Device-side conditions (neighbor-row overflow, FENE over-stretch, non-finite coordinates) are
 *     latched in a device word and reported by the next synchronising call.
 */
#ifndef GM_H
#define GM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gm_system gm_system; /* opaque; owns only small host state + CUDA graphs */
typedef int gm_status;

enum {
    GM_OK = 0,
    GM_ERR_INVALID_ARG = -1,
    GM_ERR_STATE = -2,               /* call order: e.g. gm_step before gm_set_particles          */
    GM_ERR_CUDA = -3,                /* a CUDA runtime call failed; message has the CUDA string   */
    GM_ERR_WORKSPACE_TOO_SMALL = -4,
    GM_ERR_BOX_TOO_SMALL = -5,       /* box_d < 3.0003 (r_cut_max + r_skin) in some dimension (27-cell search with a
                                        1e-4 margin for the fp32 cell assignment), or r_cut_max + 2 r_skin >= box_d / 2
                                        (one minimum-image test per listed pair) */
    GM_ERR_NEIGHBOR_OVERFLOW = -6,   /* a bead has more neighbors than nl_row_capacity            */
    GM_ERR_BOND_OVERSTRETCH = -7,    /* FENE bond with r >= R0                                    */
    GM_ERR_NONFINITE = -8            /* a coordinate became NaN/Inf                               */
};

enum { GM_PAIR_NONE = 0, GM_PAIR_LJ = 1, GM_PAIR_DPD = 2, GM_PAIR_HARMONIC = 3, GM_PAIR_GAUSS = 4, GM_PAIR_TABLE = 5 };
enum { GM_BOND_NONE = 0, GM_BOND_FENE = 1, GM_BOND_HARMONIC = 2, GM_BOND_TABLE = 3 };
enum { GM_NVE = 0, GM_LANGEVIN = 1, GM_DPD_GWVV = 2,
       GM_NVT_NOSE_HOOVER = 3, GM_NVT_ANDERSEN = 4, GM_NVT_BERENDSEN = 5,     /* PAPER.md:L133, L137; DESIGN.md c-28..c-30 */
       GM_NPH_ANDERSEN = 6, GM_NPT_ANDERSEN = 7 };                            /* Andersen barostat; DESIGN.md c-31 */
enum { GM_ANGLE_NONE = 0, GM_ANGLE_HARMONIC = 1 /* Eq. (8): k (theta - theta0)^2 */, GM_ANGLE_COSINE = 2 /* Eq. (9): k (cos theta - cos theta0)^2 */,
       GM_ANGLE_TABLE = 3 /* Eq. (12) with x = theta */ };

#define GM_MAX_TYPES 8       /* particle types; pair tables are n_types x n_types */
#define GM_MAX_BOND_TYPES 8

/* Plain-old-data configuration, versioned by struct_size (= sizeof(gm_config)). */
typedef struct {
    uint32_t struct_size;
    int32_t device;                  /* CUDA device ordinal                                        */
    void *stream;                    /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = legacy default */
    int64_t n_particles;             /* N >= 1, < 2^27 (bond rows pack the partner index in 27 bits) */
    int32_t n_types;                 /* 1..GM_MAX_TYPES                                            */
    int32_t max_bonds_per_particle;  /* rows of the BL table (Fig. 2); 0 = no bonds  */
    float box[3];                    /* cuboid edge lengths                                        */
    float r_cut_max;                 /* largest pair cutoff that will be set (cell width = r_cut_max + r_skin) */
    float r_skin;                    /* r_buffer of PAPER.md:L57                                   */
    float dt;
    uint64_t seed;                   /* key of the counter-based Philox4x32-10 noise               */
    int32_t pair_style;              /* GM_PAIR_*                                                  */
    int32_t bond_style;              /* GM_BOND_*                                                  */
    int32_t integrator;              /* GM_NVE | GM_LANGEVIN | GM_DPD_GWVV | GM_NVT_* | GM_NP*_ANDERSEN */
    float kT, gamma, lambda;         /* thermostat temperature; friction (Langevin, DPD) or coupling rate of the NVT
                                        thermostats (Nose-Hoover 1/tau, Berendsen 1/tau_T, Andersen collision frequency);
                                        GW-VV lambda */
    int32_t sfc_period;              /* largest number of steps between two SFC sorts of the particle arrays (every
                                        neighbor rebuild sorts; > 0 forces a rebuild after this many steps) */
    int32_t nl_row_capacity;         /* rows of the NL table; 0 = choose from density              */
    int32_t flags;                   /* GM_FLAG_*                                                  */
    /* Tuning overrides, 0 = choose from the geometry.  They never change results (exact accelerations). */
    int32_t x_cell_div;              /* 1..8: cells are (r_cut_max + r_skin) / x_cell_div wide in x (DESIGN.md c-12)  */
    int32_t nl_scan_trip;            /* 4 or 8: candidates the neighbor search loads together                         */
    int32_t step_shape;              /* 1: one-warp CTAs (short lists), 2: CTAs of 128 (long lists)                    */
    int32_t table_points;            /* GM_PAIR_TABLE: grid points (Npoint of Alg. 2) of every pair table; else 0       */
    int32_t win_capacity;            /* positions a tile window holds (shared memory per CTA = 16 B x this), <= 8000    */
    int32_t tile_windows;            /* 1: stage tile windows whatever the list length, 2: never (0: lists of >= 40)     */
    int32_t angle_style;             /* GM_ANGLE_*                                                                     */
    int32_t max_angles_per_particle; /* rows of the per-particle angle table; 0 = no angles              */
    int32_t max_dihedrals_per_particle; /* rows of the per-particle dihedral table; 0 = no dihedrals (Eq. (10))         */
    int32_t bond_table_points;       /* GM_BOND_TABLE: grid points of every bond table; else 0                          */
    int32_t angle_table_points;      /* GM_ANGLE_TABLE: grid intervals of every angle table on [0, pi]; else 0           */
    int32_t dihedral_table_points;   /* > 0: dihedrals are tabulated on [-pi, pi] with this many intervals (instead of Eq. (10)) */
} gm_config;

enum {
    GM_FLAG_NO_GRAPH = 1,            /* launch every kernel directly (debugging)                   */
    GM_FLAG_NO_COND_NODES = 2,       /* gate the rebuild with early-exit kernels instead of a CUDA conditional graph node */
    GM_FLAG_NO_WINDOWS = 8,          /* no tile windows: 32-bit neighbor rows and gathers from L1/L2 everywhere (the round-1
                                        data path; same results up to fp32 summation order -- there is none: the row order
                                        is the same, so results are bit-identical) */
    GM_FLAG_STEP_SUBWARP = 4         /* step kernel variant for long neighbor lists: 8 lanes share a bead, partial
                                        forces summed by warp shuffles (same results up to fp32 summation order;
                                        measured slower than one thread per bead on B200 -- kept for comparison) */
};

/* Bytes of device workspace gm_create needs for this configuration (all of the library's device
 * memory: particle arrays, cell list, NL/NN and BL/BN tables, scratch).  Host-only. */
gm_status gm_query_workspace(const gm_config *cfg, size_t *bytes);

/* Create a system on a caller-allocated DEVICE workspace of at least gm_query_workspace() bytes,
 * 256-byte aligned.  The workspace and the stream stay the caller's; they must outlive the system.
 * Errors: INVALID_ARG (sizes, styles, n_types), BOX_TOO_SMALL, WORKSPACE_TOO_SMALL, CUDA. */
gm_status gm_create(const gm_config *cfg, void *dev_workspace, size_t bytes, gm_system **out);

/* Frees host state and CUDA graphs only (never the workspace).  Synchronises the stream. */
gm_status gm_destroy(gm_system *s);

/* Pair parameters for the type pair (ti, tj) and (tj, ti).  `p` is a HOST array of n floats:
 *   GM_PAIR_LJ  (Eq. (1)): n = 4: eps, sigma, r_cut, shift_flag
 *               (shift_flag != 0: the energy is shifted by U(r_cut) so that it vanishes at the
 *               cutoff; the force is never altered -- DESIGN.md c-9)
 *   GM_PAIR_DPD (DESIGN.md c-3):         n = 2: a, r_cut   (gamma and kT are global, gm_config)
 *   GM_PAIR_HARMONIC (Eq. (2): U = alpha (1 - r/r_cut)^2):       n = 2: alpha, r_cut
 *   GM_PAIR_GAUSS (Eq. (3): U = eps exp(-(r/sigma)^2 / 2)):      n = 4: eps, sigma, r_cut, shift_flag
 * r_cut must be <= cfg.r_cut_max.  Errors: INVALID_ARG. */
gm_status gm_set_pair_params(gm_system *s, int ti, int tj, const float *p, int n);

/* GM_PAIR_TABLE (Eqs. (11)-(12), Algorithm 2): the potential of the type pair (ti, tj) and
 * (tj, ti) as cubic-spline coefficients on a grid of z = r^2.  c4 is a HOST array of 4 * cfg.table_points floats,
 * c4[4 * point + {0,1,2,3}] = c0..c3 of V(z) = c0 + c1 d + c2 d^2 + c3 d^3, d = z - point * interval.  A pair
 * interacts iff point = int(r^2 / interval) < table_points ("the judgement for ... the cutoff is done ... by checking
 * if the index of grid point exceeds the maximum value"), so r_cut = sqrt(table_points * interval) <= cfg.r_cut_max;
 * the force is F_i = -2 r_ij dV/dz.  Errors: INVALID_ARG, STATE (pair_style is not GM_PAIR_TABLE). */
gm_status gm_set_pair_table(gm_system *s, int ti, int tj, float interval, const float *c4);

/* Host-only utility: the spline of Eq. (12) through n_point + 1 potential values v[k] = V(k * interval) (HOST,
 * doubles) -- c0 the value at the grid point, c1..c3 such that first and second derivative are continuous across the
 * grid points, natural ends (V'' = 0; reading c-24).  c4_out: HOST array of 4 * n_point floats in the layout
 * gm_set_pair_table takes.  Errors: INVALID_ARG. */
gm_status gm_fit_pair_table(int n_point, double interval, const double *v, float *c4_out);

/* Bond parameters of bond type `btype`: FENE (k, R0): U = -1/2 k R0^2 ln(1 - r^2/R0^2);
 * harmonic (k, r0): U = k (r - r0)^2 -- Eq. (7), no factor 1/2. */
gm_status gm_set_bond_params(gm_system *s, int btype, float k, float r0_or_R0);

/* GM_BOND_TABLE ("numerical non-bonded, bond, angle, and torsion potentials", Eqs. (11)-(12)): the potential
 * of bond type `btype` as cubic-spline coefficients on a grid of z = r^2, in the layout of gm_set_pair_table: c4 is a HOST
 * array of 4 * cfg.bond_table_points floats, V(z_k + d) = c0 + c1 d + c2 d^2 + c3 d^3 with z_k = k * interval, force
 * F_i = -2 r_ij dV/dz (gm_fit_pair_table fits such a table through values on the grid).  A bond stretched past the end of
 * its table, int(r^2 / interval) >= bond_table_points, has no defined energy: it exerts no force and latches
 * GM_ERR_BOND_OVERSTRETCH (reading c-32).  Copies c4 in (synchronises).  Errors: STATE, INVALID_ARG. */
gm_status gm_set_bond_table(gm_system *s, int btype, float interval, const float *c4);

/* Particles in tag order, length N each: pos3/vel3 are (N,3) row-major floats, type is int32 in
 * [0, n_types), mass may be NULL (all 1).  Positions outside the box are wrapped in.  Resets the
 * step counter to 0 and invalidates the neighbor list.  vel3 are full-step velocities v(t).
 * Errors: INVALID_ARG (NULL pos3/vel3/type), CUDA. */
gm_status gm_set_particles(gm_system *s, const float *pos3, const float *vel3, const int32_t *type,
                           const float *mass, int on_device);

/* Bonds as n_bonds tag pairs (n_bonds,2) + a bond type each (NULL = all 0).  Each bond is entered
 * in the BL table under BOTH ends.  Errors: INVALID_ARG if a bead would exceed
 * max_bonds_per_particle or a tag is out of range (checked on the host; device inputs are copied
 * to the host for this -- set-up path, not hot path). */
gm_status gm_set_bonds(gm_system *s, int64_t n_bonds, const int32_t *tag_pairs2, const int32_t *btype,
                       int on_device);

/* Angle parameters of angle type `atype` (< GM_MAX_BOND_TYPES): Eq. (8) U = k (theta - theta0)^2 or Eq. (9)
 * U = k (cos theta - cos theta0)^2 by cfg.angle_style; theta0 in radians; theta is the angle at the
 * middle bead between its two bonds (pi for a straight chain; DESIGN.md c-26). */
gm_status gm_set_angle_params(gm_system *s, int atype, float k, float theta0);

/* Dihedral parameters of dihedral type `dtype`: Eq. (10) U = k [1 + cos(n phi - delta)]; phi = 0 for
 * cis, pi for trans (DESIGN.md c-27). */
gm_status gm_set_dihedral_params(gm_system *s, int dtype, float k, int n, float delta);

/* Tabulated angle and torsion potentials ("numerical ... angle, and torsion potentials"; L127: Eq. (12) with
 * "x corresponds to z, theta, and phi"): c4 is a HOST array of 4 * Npoint floats, V(x_k + d) = c0 + c1 d + c2 d^2 + c3 d^3.
 * Angles (cfg.angle_style = GM_ANGLE_TABLE, Npoint = cfg.angle_table_points): x = theta, x_k = k pi / Npoint.
 * Dihedrals (cfg.dihedral_table_points = Npoint > 0): x = phi, x_k = -pi + 2 pi k / Npoint; the tables cover the whole range
 * of the variable, so there is no cutoff.  Conventions for theta and phi as above.  gm_fit_pair_table fits such a table (natural
 * ends) through Npoint + 1 values on the grid.  Copies c4 in (synchronises).  Errors: STATE, INVALID_ARG. */
gm_status gm_set_angle_table(gm_system *s, int atype, const float *c4);
gm_status gm_set_dihedral_table(gm_system *s, int dtype, const float *c4);

/* Angles as n_angles tag triples (i, j, k), j the middle bead, + a type each (NULL = all 0); dihedrals as tag
 * quadruples (i, j, k, l).  Each is entered in the per-particle table of EVERY member together with the member's
 * position, so that one thread sums all angle and dihedral forces of its bead without atomics -- an angle is evaluated
 * three times, a dihedral four times.  HOST arrays (set-up path).  Their energy is reported with the bond
 * energy (gm_energies out[2]).  Errors: INVALID_ARG (a bead exceeds max_*_per_particle, tag out of range). */
gm_status gm_set_angles(gm_system *s, int64_t n_angles, const int32_t *tags3, const int32_t *atype);
gm_status gm_set_dihedrals(gm_system *s, int64_t n_dihedrals, const int32_t *tags4, const int32_t *dtype);

/* Set the time-level counter (the `step` word of the Philox counter).  For restarts. */
gm_status gm_set_step(gm_system *s, uint64_t step);

/* a1 (+ a2 when due) + a3 now, at the current positions, unconditionally. */
gm_status gm_build_neighbors(gm_system *s);

/* a4 -> (a1, a3 if needed) -> a5/a6 + a7 at the current positions; the per-bead force is kept
 * (gm_get_particles returns it).  For GM_LANGEVIN the drag and noise of the current time level are
 * included (the force the integrator uses); for DPD the dissipative and random parts are included.
 * Errors: STATE (no particles yet). */
gm_status gm_compute_forces(gm_system *s);

/* n_steps of a4..a8 (fused force + integrate kernel per step, rebuild gated on the device).
 * Asynchronous on the stream.  Errors: STATE, INVALID_ARG (n_steps < 0), CUDA. */
gm_status gm_step(gm_system *s, int64_t n_steps);

/* Switch the integrator of an existing system (e.g. Langevin equilibration, then NVE: BASELINE.json
 * config 3).  integrator: GM_NVE | GM_LANGEVIN | GM_NVT_* | GM_NP*_ANDERSEN (GM_DPD_GWVV only on a GM_PAIR_DPD system and vice
 * versa); kT, gamma as in gm_config.  The first step after a switch to an NVT thermostat runs without it (the
 * temperature of the half-step velocities it acts on is measured in that step).  The state (positions, half-step velocities, step counter,
 * neighbor list) is kept.  Errors: INVALID_ARG. */
gm_status gm_set_integrator(gm_system *s, int integrator, float kT, float gamma);

/* Andersen barostat ("the constant pressure can be controlled via Andersen barostat"; equations: DESIGN.md
 * reading c-31).  Integrators GM_NPH_ANDERSEN (barostat alone) and GM_NPT_ANDERSEN (barostat + Andersen's stochastic
 * collisions at frequency gamma, temperature kT).  The box changes isotropically: the device keeps every position in the
 * box of gm_create ("scaled" coordinates) and one scale factor lambda = (V / V_create)^(1/3); forces, virial and energies are
 * evaluated at the real distances lambda * s.  Pair styles GM_PAIR_LJ and GM_PAIR_NONE, bonds, angles and dihedrals of any
 * style (angle terms are scale-free: no virial); no DPD; such a system runs without tile windows, two kernels per timestep
 * (forces + virial, then piston + kick + drift).  The neighbor list is built once for the scaled list radius r_cut_max + r_skin of
 * gm_create; it stays complete while lambda > r_cut_max / (r_cut_max + r_skin) -- a box that shrinks further latches an
 * error (GM_ERR_BOX_TOO_SMALL from the next synchronising call); build the system anew at the new size then.
 *
 * gm_set_barostat: external pressure and piston mass M (Andersen's M: M V'' = P_inst - P_ext; units of mass / length^4);
 * the piston starts at rest.  Call it before gm_set_integrator(GM_NP*_ANDERSEN) / the first step.
 * gm_set_box_state: volume and piston momentum Pi = M dV/dt of a restart; call it BEFORE gm_set_particles, whose
 * positions are then taken in the box of that volume.  Errors: INVALID_ARG (p_ext < 0, mass <= 0, volume <= 0), STATE. */
gm_status gm_set_barostat(gm_system *s, float p_ext, float piston_mass);
gm_status gm_set_box_state(gm_system *s, double volume, double piston_momentum);

/* out (HOST, 8 doubles): current box L_x, L_y, L_z, volume, piston momentum Pi (at the current time level), instantaneous
 * pressure (2 K + W) / (3 V), virial W = sum over pairs and bonds of r_ij . F_ij, and Andersen's conserved
 * H = K + U + P_ext V + Pi^2 / (2 M).  On a system without barostat: the box of gm_create, Pi = 0, and the same
 * pressure / virial / H with P_ext = 0 are NOT computed (out[5..7] = 0).  Synchronises. */
gm_status gm_get_box(gm_system *s, double out[8]);

/* Measurement aid: n_steps timesteps exactly as gm_step would take them, but launched kernel by
 * kernel (no CUDA graph) with CUDA events on the system's stream around the fused force+integrate
 * kernel (a4..a8) and around the rebuild kernels (a1 + a3; early-exit when no rebuild is due).
 * out (HOST, 4 doubles): summed device ms of the force+integrate launches, summed device ms of the
 * rebuild launches, number of force+integrate launches, number of rebuilds (= SFC sorts) done inside.
 * Synchronises.  Same results, bit for bit, as gm_step. */
gm_status gm_step_timed(gm_system *s, int64_t n_steps, double out[4]);

/* out (HOST, 8 doubles): kinetic energy, pair PE, bonded PE (bonds + angles + dihedrals), temperature (3N-3 dof), px, py, pz,
 * number of unique pairs inside r_cut.  fp32 terms, fp64 sums.  Synchronises. */
gm_status gm_energies(gm_system *s, double out[8]);

/* Current state in tag order; any of pos3/vel3/force3 may be NULL.  vel3 are full-step velocities
 * v(t) (the library stores half-step velocities and completes them here); force3 is the force of
 * the current time level (computed if not current). */
gm_status gm_get_particles(gm_system *s, float *pos3, float *vel3, float *force3, int on_device);

/* The neighbor list in TAG space: nn[tag] and nl_tags[tag * row_stride + k], k < nn[tag]
 * (row order unspecified).  Builds the list first if none is current.  row_stride >= max nn
 * (see gm_get_stats), else INVALID_ARG. */
gm_status gm_get_neighbors(gm_system *s, int32_t *nn, int32_t *nl_tags, int64_t row_stride, int on_device);

/* out (HOST, 8 int64): steps taken, neighbor rebuilds, SFC sorts (= rebuilds), max nn of the current list,
 * sum of nn of the current list, latched device error word (0 = none), nl_row_capacity,
 * number of cells.  Synchronises; returns the latched device error as status if one is set. */
gm_status gm_get_stats(gm_system *s, int64_t out[8]);

/* out (HOST, 8 int64): what gm_create chose and what the last neighbor build did -- x_cell_div, nl_scan_trip,
 * step_shape (1 narrow, 2 wide), tile windows in use (0/1), window capacity in positions, tiles (128 beads each),
 * tiles of the current list that are NOT window-staged, dynamic shared memory of the neighbor-build kernel in bytes.
 * Synchronises.  Diagnostics only: none of these changes results. */
gm_status gm_get_tuning(gm_system *s, int64_t out[8]);

/* Kinetic energy and momentum of n beads -- the a9 sums of gm_energies (the validation quantities),
 * fp32 inputs, every term and sum in fp64 -- through an entry point that needs no gm_system and no workspace and ALLOCATES
 * NOTHING (no cudaMalloc / cudaFree, no allocating library call): for callers under CUDA graph capture, in tight serving
 * loops, or in harnesses that forbid allocation.  The per-block partial sums live in a file-scope __device__ array of the
 * library (262,400 bytes, held by every GPU that loads libgm.so until exit), which bounds the size:
 * n <= GM_STATIC_MAX_BEADS, else INVALID_ARG with a message saying so.
 *   vel3 (DEVICE, n x 3 floats), mass (DEVICE, n floats, or NULL = 1.0), device: CUDA device ordinal (made current),
 *   stream: cudaStream_t as void* (0 = default stream), out4 (DEVICE, 4 doubles: kinetic energy, p_x, p_y, p_z),
 *   err / err_len: HOST buffer for the message of a failed call (may be NULL / 0).
 * Asynchronous on `stream` (one memset node + one kernel node: capturable); the result is in out4 when the stream reaches
 * that point.  The first call per device resolves the array's device address (cudaGetSymbolAddress): make it outside a
 * stream capture.  ALL calls share the one array, which keeps the last call's contents (what must start at zero is
 * cleared by every call): calls on one stream are ordered; calls that overlap on a GPU (two streams, two threads) RACE.
 * Deterministic: the additions are ordered by the grid size alone.  Errors: INVALID_ARG, CUDA. */
#define GM_STATIC_MAX_BEADS 8388608
gm_status gm_kinetic_static(const float *vel3, const float *mass, int64_t n, int device, void *stream, double *out4,
                            char *err, size_t err_len);

/* Host-only utility (a2): the space-filling-curve rank of every cell of an nc[0] x nc[1] x nc[2] grid
 * (linear cell id = (z * nc[1] + y) * nc[0] + x), i.e. the key every neighbor rebuild sorts the beads by:
 * cells run along x inside a row, the (y, z) rows follow a 2-D Hilbert curve.  rank_out: HOST array of
 * nc[0]*nc[1]*nc[2] uint32.  The order only affects memory locality, never results. */
gm_status gm_sfc_cell_order(const int32_t nc[3], uint32_t *rank_out);

/* Message of the last failing call on `s` (or a static string if s is NULL).  Never NULL. */
const char *gm_last_error(const gm_system *s);

#ifdef __cplusplus
}
#endif
#endif /* GM_H */
