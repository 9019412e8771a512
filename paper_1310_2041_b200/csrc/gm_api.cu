// gm_api.cu -- the C ABI of include/gm.h: host-side state, workspace layout, the step scheduler
// (CUDA graphs with the rebuild inside a conditional node) and marshalling.  All device work is in
// gm_sort.cu / gm_nlist.cu / gm_force.cu / gm_io.cu; there is no CPU fallback for any of it.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <new>
#include <vector>

#include "gm_internal.cuh"
#include "gm_npt.cuh"

// Timesteps per graph launch (even): a launch costs ~7 us of device time (the one gate kernel of its first timestep and the
// gap to the next graph), so long runs go in graphs of 64 (measured against 16: C3 70.18 -> 69.85, C1 17.75 -> 17.33 us per
// timestep), what is left in graphs of 16, then of 2
#define GM_GRAPH_STEPS 64
#define GM_GRAPH_STEPS_MID 16

struct gm_system {
    gm_config cfg;
    GmParams P;
    GmDev D;
    cudaStream_t st, cap_st, cap_st2;
    GmFork fk;                     // side branch of the rebuild (gm_launch_nl_build)
    int cur;                       // which pos/vt buffer holds the current time level
    bool have_particles, lagged, nl_valid, force_current, bonds_dirty, pair_set_any;
    uint64_t step;
    bool use_graph, use_cond;
    cudaGraphExec_t exec_big, exec_mid, exec_two;
    // Andersen barostat (gm_npt.cuh): host copies of what gm_set_barostat / gm_set_box_state last set
    double npt_vol0, npt_V, npt_Pi, npt_p_ext, npt_mass;
    char err[512];
};

static const char *k_null_msg = "gm: null system";

static gm_status fail(gm_system *s, gm_status code, const char *fmt, const char *arg = "")
{
    if (s) snprintf(s->err, sizeof(s->err), fmt, arg);
    return code;
}

#define CU(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) return fail(s, GM_ERR_CUDA, "CUDA: %s", cudaGetErrorString(e_)); \
    } while (0)

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

static bool is_npt(const gm_system *s) { return s->P.integrator == GM_NPH_ANDERSEN || s->P.integrator == GM_NPT_ANDERSEN; }

// ---- geometry and constants derived from the configuration ----------------------------------------
static gm_status derive(const gm_config *c, GmParams *P)
{
    memset(P, 0, sizeof(*P));
    if (!c || c->struct_size != sizeof(gm_config)) return GM_ERR_INVALID_ARG;
    if (c->n_particles < 1 || c->n_particles >= (1ll << 27)) return GM_ERR_INVALID_ARG;
    if (c->n_types < 1 || c->n_types > GM_MAX_TYPES) return GM_ERR_INVALID_ARG;
    if (c->max_bonds_per_particle < 0 || c->max_bonds_per_particle > 16) return GM_ERR_INVALID_ARG;
    if (c->pair_style < GM_PAIR_NONE || c->pair_style > GM_PAIR_TABLE) return GM_ERR_INVALID_ARG;
    if (c->table_points < 0 || c->table_points > (1 << 20) || ((c->pair_style == GM_PAIR_TABLE) != (c->table_points > 0)))
        return GM_ERR_INVALID_ARG;
    if (c->bond_style < GM_BOND_NONE || c->bond_style > GM_BOND_TABLE) return GM_ERR_INVALID_ARG;
    if (c->bond_table_points < 0 || c->bond_table_points > (1 << 20) || ((c->bond_style == GM_BOND_TABLE) != (c->bond_table_points > 0)))
        return GM_ERR_INVALID_ARG;
    if (c->integrator < GM_NVE || c->integrator > GM_NPT_ANDERSEN) return GM_ERR_INVALID_ARG;
    if ((c->integrator == GM_DPD_GWVV) != (c->pair_style == GM_PAIR_DPD)) return GM_ERR_INVALID_ARG;
    const bool npt = c->integrator == GM_NPH_ANDERSEN || c->integrator == GM_NPT_ANDERSEN;
    if (npt && ((c->pair_style != GM_PAIR_LJ && c->pair_style != GM_PAIR_NONE) || (c->flags & GM_FLAG_STEP_SUBWARP)))
        return GM_ERR_INVALID_ARG;
    if (!(c->r_cut_max > 0.f) || !(c->r_skin >= 0.f) || !(c->dt > 0.f)) return GM_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d) if (!(c->box[d] > 0.f)) return GM_ERR_INVALID_ARG;
    if (c->x_cell_div < 0 || c->x_cell_div > 8 || (c->nl_scan_trip != 0 && c->nl_scan_trip != 4 && c->nl_scan_trip != 8) ||
        c->step_shape < 0 || c->step_shape > 2 || c->win_capacity < 0 || c->win_capacity > 8000 || c->tile_windows < 0 || c->tile_windows > 2 ||
        c->angle_style < GM_ANGLE_NONE || c->angle_style > GM_ANGLE_TABLE || c->max_angles_per_particle < 0 ||
        c->angle_table_points < 0 || c->angle_table_points > (1 << 20) || ((c->angle_style == GM_ANGLE_TABLE) != (c->angle_table_points > 0)) ||
        c->dihedral_table_points < 0 || c->dihedral_table_points > (1 << 20) ||
        (c->dihedral_table_points > 0 && c->max_dihedrals_per_particle == 0) ||
        c->max_angles_per_particle > 64 || c->max_dihedrals_per_particle < 0 || c->max_dihedrals_per_particle > 64 ||
        (c->max_angles_per_particle > 0 && c->angle_style == GM_ANGLE_NONE))
        return GM_ERR_INVALID_ARG;
    P->n = (int)c->n_particles;
    P->ns = (P->n + 8 + GM_PAD - 1) / GM_PAD * GM_PAD;     // slots n .. n+7 (at least): far-away pad beads
    P->sfc_period = c->sfc_period;
    P->n_types = c->n_types;
    P->max_bonds = c->max_bonds_per_particle;
    const double r_list = (double)c->r_cut_max + (double)c->r_skin;
    double vol = 1.0;
    for (int d = 0; d < 3; ++d) {
        P->box[d] = c->box[d];
        P->half[d] = 0.5f * c->box[d];
        // cell width >= r_list with a 1e-4 relative margin for the fp32 cell assignment (reading c-12)
        P->nc[d] = (int)std::floor((double)c->box[d] / (r_list * 1.0001));
        if (P->nc[d] < 3) return GM_ERR_BOX_TOO_SMALL;
        // one |a - b| > L/2 test per listed pair (gm_min_image_signed) and the plain differences of the search
        // pick the right image only while r_list + r_skin < L/2 (a listed pair drifts by at most r_skin)
        if (!(r_list + (double)c->r_skin < 0.5 * (double)c->box[d])) return GM_ERR_BOX_TOO_SMALL;
        if (P->nc[d] > 1024) P->nc[d] = 1024;
        vol *= c->box[d];
    }
    // x only: cells r_list / sx wide, searched sx to either side (the run of a (y, z) row shrinks from 3 to
    // 2 + 1/sx list radii); sx grows with the number of beads per r_list^3 cell
    {
        const double per_cell = (double)P->n / ((double)P->nc[0] * P->nc[1] * P->nc[2]);
        int sx = per_cell >= 6.0 ? 4 : (per_cell >= 2.0 ? 3 : (per_cell >= 1.0 ? 2 : 1));   // measured: C3 3, C2/C4/C5 4
        if (c->x_cell_div > 0) sx = c->x_cell_div;
        P->sx = sx;
        // mean candidates per run of a (y, z) row: (2 sx + 1) cells of per_cell / sx beads
        P->nl_trip = per_cell * (2.0 * sx + 1.0) / sx >= 16.0 ? 8 : 4;
        if (c->nl_scan_trip > 0) P->nl_trip = c->nl_scan_trip;
        if (sx > 1) {
            P->nc[0] = (int)std::floor((double)c->box[0] * sx / (r_list * 1.0001));
            if (P->nc[0] > 4096) { P->sx = 1; P->nc[0] = 1024; }
        }
    }
    // sparse boxes: no more cells than a few per bead (wider cells stay correct)
    while ((long long)P->nc[0] * P->nc[1] * P->nc[2] > 8ll * P->n + 64) {
        int d = 0;
        if (P->nc[1] > P->nc[d]) d = 1;
        if (P->nc[2] > P->nc[d]) d = 2;
        if (P->nc[d] <= 3 * (d == 0 ? P->sx : 1)) break;
        P->nc[d] -= 1;
    }
    P->n_cells = P->nc[0] * P->nc[1] * P->nc[2];
    for (int d = 0; d < 3; ++d) P->inv_w[d] = (float)((double)P->nc[d] / (double)c->box[d]);
    P->r_list2 = (float)(r_list * r_list);
    P->half_skin2 = (float)(0.25 * (double)c->r_skin * (double)c->r_skin);
    P->edge_margin = (float)(r_list + (double)c->r_skin);
    P->dt = c->dt; P->kT = c->kT; P->gamma = c->gamma; P->lambda = c->lambda;
    P->sigma_r_sqrt_inv_dt = (float)std::sqrt(2.0 * (double)c->gamma * (double)c->kT / (double)c->dt);
    P->lang_amp2 = (float)(6.0 * (double)c->gamma * (double)c->kT / (double)c->dt);
    P->seed_lo = (uint32_t)(c->seed & 0xFFFFFFFFu);
    P->seed_hi = (uint32_t)(c->seed >> 32);
    P->pair_style = c->pair_style; P->bond_style = c->bond_style; P->integrator = c->integrator;
    int cap = c->nl_row_capacity;
    if (cap <= 0) {
        double nbar = (double)P->n / vol * (4.0 / 3.0) * 3.14159265358979323846 * r_list * r_list * r_list;
        cap = (int)(2.0 * nbar) + 48;     // random-walk DPD starts (C4) reach ~3x the mean in places
    }
    {
        const double nbar = (double)P->n / vol * (4.0 / 3.0) * 3.14159265358979323846 * r_list * r_list * r_list;
        // measured: C1/C3 (n_l 13) narrow; C5 (78, 8M beads) wide; C2 (78, 64k beads: less than one wave) narrow
        P->step_wide = (nbar >= 40.0 && P->n > 262144) ? 1 : 0;
        if (c->step_shape > 0) P->step_wide = c->step_shape == 2;
    }
    if ((long long)cap > (long long)P->n) cap = std::max(1, P->n - 1 + (P->n == 1));
    cap = (cap + 7) / 8 * 8;
    P->nl_cap = cap;
    // lanes per bead of the step kernel: 8 lanes sharing a bead (shuffle reduction) measured SLOWER than one
    // thread per bead on every config, so it is opt-in
    P->angle_style = c->angle_style; P->max_angles = c->max_angles_per_particle; P->max_dihedrals = c->max_dihedrals_per_particle;
    P->step_subw = ((c->flags & GM_FLAG_STEP_SUBWARP) && P->max_angles + P->max_dihedrals == 0 && c->integrator <= GM_DPD_GWVV) ? 8 : 1;
    P->capq = cap / 4;
    P->minq = std::min(4, P->capq);
    // tile windows (gm_nlist.cu): every pair style but DPD (which also gathers velocities), one thread per bead.  A window holds the hulls of the x runs
    // of a tile's 128 beads in 9 (y, z) rows: 9 (128 + (2 sx + 1) beads-per-x-cell) positions for a tile inside one row;
    // tiles at a row end hold two partial hulls plus the wrapped pieces -- 1.25 x + 64 covers nearly all of them, the
    // rest keep the gather path.
    {
        const double per_xcell = (double)P->n / ((double)P->nc[0] * P->nc[1] * P->nc[2]);
        const double est = 9.0 * ((double)GM_TILE + (2.0 * P->sx + 1.0) * per_xcell);
        int wc = (int)(1.25 * est) + 64;
        wc = (wc + 7) / 8 * 8;
        if (c->win_capacity > 0) wc = (c->win_capacity + 7) / 8 * 8;
        // Measured (same-box A/B against the gather path): windows pay for long lists -- C5 (n_l 92) 2148 ->
        // 1970 us per timestep, C2 (88) 37.2 -> 34.5 -- and cost a little for short ones (C3, n_l 13.5: the step kernel
        // gains 0.3 us, the rebuild loses 3), so they are chosen by the estimated list length; tile_windows overrides.
        const double nbar_w = (double)P->n / vol * (4.0 / 3.0) * 3.14159265358979323846 * r_list * r_list * r_list;
        const bool can = c->pair_style != GM_PAIR_NONE && c->pair_style != GM_PAIR_DPD && P->step_subw == 1 &&
                         !(c->flags & GM_FLAG_NO_WINDOWS) && wc <= 8000 && !npt;      // the barostat path reads 32-bit rows
        P->use_win = (can && c->tile_windows != 2 && (c->tile_windows == 1 || nbar_w >= 40.0)) ? 1 : 0;
        if (P->n <= 4096 && P->use_win) wc = std::max(wc, (P->n + 7) / 8 * 8);
        P->win_cap = P->use_win ? wc : 0;
    }
    if (!gm_nl_capacity_ok(*P)) return GM_ERR_INVALID_ARG;
    P->table_points = c->table_points;      // (memset above: every pair coefficient starts at 0 = no interaction)
    P->bond_table_points = c->bond_table_points;
    P->angle_table_points = c->angle_table_points; P->dihedral_table_points = c->dihedral_table_points;
    return GM_OK;
}

// ---- workspace layout: one pass with base == nullptr sizes it, a second pass assigns pointers ------
static size_t carve(const GmParams &P, const gm_config &c, char *base, GmDev *D)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> char * {
        char *p = base ? base + off : nullptr;
        off += align_up(bytes);
        return p;
    };
    const size_t n = (size_t)P.ns;      // padded: whole tiles of GM_PAD beads can be bulk-copied
    GmDev d;
    memset(&d, 0, sizeof(d));
    d.ctl = (GmCtl *)take(sizeof(GmCtl));
    d.pos[0] = (float4 *)take(n * 16); d.pos[1] = (float4 *)take(n * 16);
    d.ref = (float4 *)take(n * 16);
    d.vel = (float4 *)take(n * 16); d.svel = (float4 *)take(n * 16);
    if (c.pair_style == GM_PAIR_DPD) {
        d.vt[0] = (float4 *)take(n * 16); d.vt[1] = (float4 *)take(n * 16); d.svt = (float4 *)take(n * 16);
    }
    d.frc = (float4 *)take(n * 16);
    if (P.table_points > 0) d.table = (float4 *)take((size_t)P.n_types * P.n_types * P.table_points * 16);
    if (P.bond_table_points > 0) d.btable = (float4 *)take((size_t)GM_MAX_BOND_TYPES * P.bond_table_points * 16);
    if (P.angle_table_points > 0) d.atable = (float4 *)take((size_t)GM_MAX_BOND_TYPES * P.angle_table_points * 16);
    if (P.dihedral_table_points > 0) d.dtable = (float4 *)take((size_t)GM_MAX_BOND_TYPES * P.dihedral_table_points * 16);
    if (P.max_angles + P.max_dihedrals > 0) d.ftopo = (float4 *)take(n * 16);
    if (P.max_angles > 0) d.at = (int4 *)take(n * 16 * (size_t)P.max_angles);
    if (P.max_dihedrals > 0) d.dt = (int4 *)take(n * 16 * (size_t)P.max_dihedrals);
    d.tag[0] = (int *)take(n * 4); d.tag[1] = (int *)take(n * 4); d.rtag = (int *)take(n * 4);
    d.nn = (int *)take(n * 4);
    d.nnw = (int *)take(n / 32 * 4);
    d.nl = (int4 *)take(n * 4 * (size_t)P.nl_cap);
    if (P.max_bonds > 0) {
        const size_t bb = n * 4 * (size_t)P.max_bonds;
        d.bl = (int *)take(bb); d.blt[0] = (int *)take(bb); d.blt[1] = (int *)take(bb); d.bl_tag = (int *)take(bb);
    }
    if (P.use_win) d.wdesc = (int4 *)take((n / GM_TILE + 1) * (size_t)GM_WD_STRIDE * sizeof(int4));
    d.key = (int *)take(n * 4); d.rank = (int *)take(n * 4); d.sorted = (int *)take(n * 4);
    d.cstart = (int *)take(((size_t)P.n_cells + 1 + 4) * 4);
    d.ccount = (int *)take(((size_t)P.n_cells + 1 + 4) * 4);
    size_t per = (size_t)GM_SCAN_BLOCK * GM_SCAN_ITEMS;
    d.scan_sums = (int *)take((((size_t)P.n_cells + 1 + per - 1) / per + 1) * 4);
    d.row_rank = (uint32_t *)take((size_t)P.nc[1] * P.nc[2] * 4);
    d.stage = (float *)take(n * 4 * 11);
    d.esum = (double *)take((((size_t)GM_ESUM_BLOCKS + 1) * 8 + GM_NPT_DOUBLES) * sizeof(double));     // + GmNpt (gm_npt.cuh)
    if (D) *D = d;
    return off;
}

// ---- a2: the space-filling curve the beads are sorted along ------------------------------------------
// Cells run along x inside a row (so the x-neighbors of a cell are its memory neighbors and the 27-cell
// search reads 9 contiguous runs); the (y, z) rows follow a 2-D Hilbert curve, so the 8 neighbor rows
// of a row are close in memory too.  Hilbert index in Skilling's transpose form (J. Skilling,
// "Programming the Hilbert curve", AIP Conf. Proc. 707, 2004), restated for ND dimensions: axes ->
// transposed index in place, then the bits are interleaved.
template <int ND>
static uint64_t hilbert_index(const uint32_t *axes, int bits)
{
    uint32_t X[ND];
    for (int i = 0; i < ND; ++i) X[i] = axes[i];
    const uint32_t M = 1u << (bits - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
        const uint32_t Pm = Q - 1;
        for (int i = 0; i < ND; ++i) {
            if (X[i] & Q) X[0] ^= Pm;
            else { uint32_t t = (X[0] ^ X[i]) & Pm; X[0] ^= t; X[i] ^= t; }
        }
    }
    for (int i = 1; i < ND; ++i) X[i] ^= X[i - 1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1) if (X[ND - 1] & Q) t ^= Q - 1;
    for (int i = 0; i < ND; ++i) X[i] ^= t;
    uint64_t h = 0;
    for (int b = bits - 1; b >= 0; --b)
        for (int i = 0; i < ND; ++i) h = (h << 1) | ((X[i] >> b) & 1u);
    return h;
}

// rank of every (y, z) row of cells along the 2-D Hilbert curve (row id = z * ncy + y)
static void sfc_row_order(int ncy, int ncz, std::vector<uint32_t> &row_rank)
{
    int mx = std::max(ncy, ncz);
    int bits = 1;
    while ((1 << bits) < mx) ++bits;
    const size_t nrow = (size_t)ncy * ncz;
    std::vector<std::pair<uint64_t, uint32_t>> v(nrow);
    for (int z = 0; z < ncz; ++z)
        for (int y = 0; y < ncy; ++y) {
            const uint32_t ax[2] = { (uint32_t)y, (uint32_t)z };
            v[(size_t)z * ncy + y] = std::make_pair(hilbert_index<2>(ax, bits), (uint32_t)(z * ncy + y));
        }
    std::sort(v.begin(), v.end());
    row_rank.resize(nrow);
    for (size_t r = 0; r < nrow; ++r) row_rank[v[r].second] = (uint32_t)r;
}

extern "C" gm_status gm_sfc_cell_order(const int32_t nc[3], uint32_t *rank_out)
{
    if (!nc || !rank_out || nc[0] < 1 || nc[1] < 1 || nc[2] < 1) return GM_ERR_INVALID_ARG;
    std::vector<uint32_t> rr;
    sfc_row_order(nc[1], nc[2], rr);
    for (int z = 0; z < nc[2]; ++z)
        for (int y = 0; y < nc[1]; ++y)
            for (int x = 0; x < nc[0]; ++x)
                rank_out[((size_t)z * nc[1] + y) * nc[0] + x] = rr[(size_t)z * nc[1] + y] * (uint32_t)nc[0] + (uint32_t)x;
    return GM_OK;
}

// ---- create / destroy -----------------------------------------------------------------------------
extern "C" gm_status gm_query_workspace(const gm_config *cfg, size_t *bytes)
{
    GmParams P;
    gm_status r = derive(cfg, &P);
    if (r != GM_OK) return r;
    if (!bytes) return GM_ERR_INVALID_ARG;
    *bytes = carve(P, *cfg, nullptr, nullptr);
    return GM_OK;
}

static void drop_graphs(gm_system *s)
{
    if (s->exec_big) { cudaGraphExecDestroy(s->exec_big); s->exec_big = nullptr; }
    if (s->exec_mid) { cudaGraphExecDestroy(s->exec_mid); s->exec_mid = nullptr; }
    if (s->exec_two) { cudaGraphExecDestroy(s->exec_two); s->exec_two = nullptr; }
}

extern "C" gm_status gm_create(const gm_config *cfg, void *dev_workspace, size_t bytes, gm_system **out)
{
    if (!out) return GM_ERR_INVALID_ARG;
    *out = nullptr;
    GmParams P;
    gm_status r = derive(cfg, &P);
    if (r != GM_OK) return r;
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255)) return GM_ERR_INVALID_ARG;
    if (bytes < carve(P, *cfg, nullptr, nullptr)) return GM_ERR_WORKSPACE_TOO_SMALL;
    gm_system *s = new (std::nothrow) gm_system;
    if (!s) return GM_ERR_INVALID_ARG;
    memset(s, 0, sizeof(*s));
    s->cfg = *cfg;
    s->P = P;
    carve(P, *cfg, (char *)dev_workspace, &s->D);
    s->P.table = s->D.table;
    s->P.btable = s->D.btable;
    s->P.atable = s->D.atable; s->P.dtable = s->D.dtable;
    s->st = (cudaStream_t)cfg->stream;
    s->use_graph = !(cfg->flags & GM_FLAG_NO_GRAPH);
    s->use_cond = !(cfg->flags & GM_FLAG_NO_COND_NODES);
    s->err[0] = 0;
    cudaError_t e = cudaSetDevice(cfg->device);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->cap_st, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->cap_st2, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->fk.side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->fk.fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->fk.join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = gm_nl_prepare(P);
    if (e == cudaSuccess) {
        std::vector<uint32_t> rr;
        sfc_row_order(P.nc[1], P.nc[2], rr);
        e = cudaMemcpyAsync(s->D.row_rank, rr.data(), rr.size() * 4, cudaMemcpyHostToDevice, s->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->st);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(s->D.ccount, 0, ((size_t)P.n_cells + 1 + 4) * 4, s->st);
    if (e == cudaSuccess && P.max_bonds > 0) {
        const size_t bb = (size_t)P.ns * 4 * (size_t)P.max_bonds;       // -1 everywhere: no bonds
        e = cudaMemsetAsync(s->D.bl, 0xFF, bb, s->st);
        if (e == cudaSuccess) e = cudaMemsetAsync(s->D.blt[0], 0xFF, bb, s->st);
        if (e == cudaSuccess) e = cudaMemsetAsync(s->D.blt[1], 0xFF, bb, s->st);
        if (e == cudaSuccess) e = cudaMemsetAsync(s->D.bl_tag, 0xFF, bb, s->st);
    }
    if (e == cudaSuccess && P.max_angles + P.max_dihedrals > 0) e = cudaMemsetAsync(s->D.ftopo, 0, (size_t)P.ns * 16, s->st);
    if (e == cudaSuccess && P.max_angles > 0) e = cudaMemsetAsync(s->D.at, 0xFF, (size_t)P.ns * 16 * P.max_angles, s->st);
    if (e == cudaSuccess && P.max_dihedrals > 0) e = cudaMemsetAsync(s->D.dt, 0xFF, (size_t)P.ns * 16 * P.max_dihedrals, s->st);
    if (e == cudaSuccess) {
        gm_launch_init_pad(P, s->D, s->st);
        gm_launch_set_ctl(s->D, 0, 1, 0, s->st);
        s->npt_vol0 = (double)cfg->box[0] * (double)cfg->box[1] * (double)cfg->box[2];
        s->npt_V = s->npt_vol0; s->npt_Pi = 0.0; s->npt_p_ext = 0.0; s->npt_mass = 1.0;
        gm_launch_npt_init(s->D, 0, s->npt_vol0, s->npt_V, s->npt_Pi, s->npt_p_ext, s->npt_mass, s->st);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (s->cap_st) cudaStreamDestroy(s->cap_st);
        if (s->cap_st2) cudaStreamDestroy(s->cap_st2);
        if (s->fk.side) cudaStreamDestroy(s->fk.side);
        if (s->fk.fork) cudaEventDestroy(s->fk.fork);
        if (s->fk.join) cudaEventDestroy(s->fk.join);
        delete s;
        return GM_ERR_CUDA;
    }
    s->bonds_dirty = true;
    *out = s;
    return GM_OK;
}

extern "C" gm_status gm_destroy(gm_system *s)
{
    if (!s) return GM_ERR_INVALID_ARG;
    cudaSetDevice(s->cfg.device);
    cudaStreamSynchronize(s->st);
    drop_graphs(s);
    cudaStreamDestroy(s->cap_st);
    cudaStreamDestroy(s->cap_st2);
    cudaStreamDestroy(s->fk.side);
    cudaEventDestroy(s->fk.fork);
    cudaEventDestroy(s->fk.join);
    delete s;
    return GM_OK;
}

extern "C" const char *gm_last_error(const gm_system *s) { return s ? s->err : k_null_msg; }

// ---- parameters -------------------------------------------------------------------------------------
extern "C" gm_status gm_set_pair_params(gm_system *s, int ti, int tj, const float *p, int n)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!p || ti < 0 || tj < 0 || ti >= s->P.n_types || tj >= s->P.n_types)
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: bad type index or NULL%s");
    GmPair c;
    memset(&c, 0, sizeof(c));
    if (s->P.pair_style == GM_PAIR_LJ) {
        if (n != 4) return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: LJ takes eps, sigma, r_cut, shift%s");
        double eps = p[0], sig = p[1], rc = p[2];
        if (!(rc > 0.0) || rc > (double)s->cfg.r_cut_max * (1.0 + 1e-6))
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: r_cut outside (0, r_cut_max]%s");
        double s6 = std::pow(sig, 6.0), s12 = s6 * s6;
        double q6 = std::pow(sig / rc, 6.0);
        c.c0 = (float)(rc * rc);
        c.c1 = (float)(48.0 * eps * s12);
        c.c2 = (float)(24.0 * eps * s6);
        c.c3 = (p[3] != 0.f) ? (float)(4.0 * eps * (q6 * q6 - q6)) : 0.f;
    } else if (s->P.pair_style == GM_PAIR_DPD) {
        if (n != 2) return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: DPD takes a, r_cut%s");
        double rc = p[1];
        if (!(rc > 0.0) || rc > (double)s->cfg.r_cut_max * (1.0 + 1e-6))
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: r_cut outside (0, r_cut_max]%s");
        c.c0 = (float)(rc * rc); c.c1 = p[0]; c.c2 = (float)(1.0 / rc); c.c3 = p[1];
    } else if (s->P.pair_style == GM_PAIR_HARMONIC) {
        if (n != 2) return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: harmonic repulsion takes alpha, r_cut%s");
        double rc = p[1];
        if (!(rc > 0.0) || rc > (double)s->cfg.r_cut_max * (1.0 + 1e-6))
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: r_cut outside (0, r_cut_max]%s");
        c.c0 = (float)(rc * rc); c.c1 = (float)(2.0 * (double)p[0] / rc); c.c2 = (float)(1.0 / rc); c.c3 = p[0];
    } else if (s->P.pair_style == GM_PAIR_GAUSS) {
        if (n != 4) return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: Gaussian repulsion takes eps, sigma, r_cut, shift%s");
        double eps = p[0], sig = p[1], rc = p[2];
        if (!(rc > 0.0) || rc > (double)s->cfg.r_cut_max * (1.0 + 1e-6) || !(sig > 0.0))
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_params: r_cut outside (0, r_cut_max] or sigma <= 0%s");
        c.c0 = (float)(rc * rc); c.c1 = (float)(eps / (sig * sig)); c.c2 = (float)(-0.5 / (sig * sig));
        c.c3 = (p[3] != 0.f) ? (float)(eps * std::exp(-0.5 * rc * rc / (sig * sig))) : 0.f;
        c.c4 = p[0];
    } else if (s->P.pair_style == GM_PAIR_TABLE) {
        return fail(s, GM_ERR_STATE, "gm_set_pair_params: tables are set with gm_set_pair_table%s");
    } else {
        return fail(s, GM_ERR_STATE, "gm_set_pair_params: pair_style is GM_PAIR_NONE%s");
    }
    s->P.pair[ti * s->P.n_types + tj] = c;
    s->P.pair[tj * s->P.n_types + ti] = c;
    s->force_current = false;
    drop_graphs(s);     // kernel parameters are baked into the graphs
    return GM_OK;
}

extern "C" gm_status gm_set_pair_table(gm_system *s, int ti, int tj, float interval, const float *c4)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (s->P.pair_style != GM_PAIR_TABLE) return fail(s, GM_ERR_STATE, "gm_set_pair_table: pair_style is not GM_PAIR_TABLE%s");
    if (!c4 || ti < 0 || tj < 0 || ti >= s->P.n_types || tj >= s->P.n_types || !(interval > 0.f))
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_table: bad type index, interval or NULL%s");
    const int np = s->P.table_points;
    const double zc = (double)np * (double)interval;
    if (std::sqrt(zc) > (double)s->cfg.r_cut_max * (1.0 + 1e-6))
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_pair_table: sqrt(table_points * interval) exceeds r_cut_max%s");
    CU(cudaSetDevice(s->cfg.device));
    const int pairs[2] = { ti * s->P.n_types + tj, tj * s->P.n_types + ti };
    for (int q = 0; q < (ti == tj ? 1 : 2); ++q) {
        CU(cudaMemcpyAsync(s->D.table + (size_t)pairs[q] * np, c4, (size_t)np * 16, cudaMemcpyHostToDevice, s->st));
        GmPair c;
        memset(&c, 0, sizeof(c));
        c.c0 = (float)zc; c.c1 = (float)(1.0 / (double)interval); c.c2 = interval;
        const int off = pairs[q] * np;
        memcpy(&c.c4, &off, sizeof(int));
        s->P.pair[pairs[q]] = c;
    }
    CU(cudaStreamSynchronize(s->st));              // the caller may reuse c4 at once
    s->force_current = false;
    drop_graphs(s);
    return GM_OK;
}

// Eq. (12): natural cubic spline through v[k] = V(k * interval), k = 0 .. n_point (Thomas algorithm for the second
// derivatives m_k; m_0 = m_n = 0), as coefficients of powers of d = z - z_k.
extern "C" gm_status gm_fit_pair_table(int n_point, double interval, const double *v, float *c4_out)
{
    if (n_point < 1 || !(interval > 0.0) || !v || !c4_out) return GM_ERR_INVALID_ARG;
    const int n = n_point;
    const double h = interval;
    std::vector<double> m((size_t)n + 1, 0.0);
    if (n >= 2) {
        // m_{k-1} + 4 m_k + m_{k+1} = 6 (v_{k+1} - 2 v_k + v_{k-1}) / h^2, k = 1 .. n-1
        std::vector<double> cp((size_t)n, 0.0), dp((size_t)n, 0.0);
        for (int k = 1; k < n; ++k) {
            const double rhs = 6.0 * (v[k + 1] - 2.0 * v[k] + v[k - 1]) / (h * h);
            const double den = 4.0 - cp[k - 1];
            cp[k] = 1.0 / den;
            dp[k] = (rhs - dp[k - 1]) / den;
        }
        for (int k = n - 1; k >= 1; --k) m[k] = dp[k] - cp[k] * m[k + 1];
    }
    for (int k = 0; k < n; ++k) {
        c4_out[4 * k + 0] = (float)v[k];
        c4_out[4 * k + 1] = (float)((v[k + 1] - v[k]) / h - h * (2.0 * m[k] + m[k + 1]) / 6.0);
        c4_out[4 * k + 2] = (float)(0.5 * m[k]);
        c4_out[4 * k + 3] = (float)((m[k + 1] - m[k]) / (6.0 * h));
    }
    return GM_OK;
}

extern "C" gm_status gm_set_bond_params(gm_system *s, int btype, float k, float r0)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (btype < 0 || btype >= GM_MAX_BOND_TYPES) return fail(s, GM_ERR_INVALID_ARG, "gm_set_bond_params: bad bond type%s");
    if (s->P.bond_style == GM_BOND_TABLE) return fail(s, GM_ERR_STATE, "gm_set_bond_params: tables are set with gm_set_bond_table%s");
    if (s->P.bond_style == GM_BOND_FENE && !(r0 > 0.f)) return fail(s, GM_ERR_INVALID_ARG, "gm_set_bond_params: FENE needs R0 > 0%s");
    s->P.bond_k[btype] = k;
    s->P.bond_r0[btype] = r0;
    s->P.bond_c[btype] = (r0 != 0.f) ? (float)(1.0 / ((double)r0 * (double)r0)) : 0.f;
    s->force_current = false;
    drop_graphs(s);
    return GM_OK;
}

extern "C" gm_status gm_set_bond_table(gm_system *s, int btype, float interval, const float *c4)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (s->P.bond_style != GM_BOND_TABLE) return fail(s, GM_ERR_STATE, "gm_set_bond_table: bond_style is not GM_BOND_TABLE%s");
    if (!c4 || btype < 0 || btype >= GM_MAX_BOND_TYPES || !(interval > 0.f))
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_bond_table: bad bond type, interval or NULL%s");
    CU(cudaSetDevice(s->cfg.device));
    const int np = s->P.bond_table_points;
    CU(cudaMemcpyAsync(s->D.btable + (size_t)btype * np, c4, (size_t)np * 16, cudaMemcpyHostToDevice, s->st));
    CU(cudaStreamSynchronize(s->st));              // the caller may reuse c4 at once
    s->P.bond_k[btype] = (float)(1.0 / (double)interval);
    s->P.bond_r0[btype] = interval;
    s->P.bond_c[btype] = 0.f;
    s->force_current = false;
    drop_graphs(s);
    return GM_OK;
}

extern "C" gm_status gm_set_angle_params(gm_system *s, int atype, float k, float theta0)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (atype < 0 || atype >= GM_MAX_BOND_TYPES) return fail(s, GM_ERR_INVALID_ARG, "gm_set_angle_params: bad angle type%s");
    s->P.angle_k[atype] = k; s->P.angle_t0[atype] = theta0; s->P.angle_c0[atype] = (float)std::cos((double)theta0);
    s->force_current = false;
    drop_graphs(s);
    return GM_OK;
}

extern "C" gm_status gm_set_dihedral_params(gm_system *s, int dtype, float k, int n, float delta)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (dtype < 0 || dtype >= GM_MAX_BOND_TYPES) return fail(s, GM_ERR_INVALID_ARG, "gm_set_dihedral_params: bad dihedral type%s");
    s->P.dih_k[dtype] = k; s->P.dih_n[dtype] = n; s->P.dih_delta[dtype] = delta;
    s->force_current = false;
    drop_graphs(s);
    return GM_OK;
}

static gm_status set_topo_table(gm_system *s, int type, const float *c4, float4 *dst, int np, const char *who)
{
    if (np <= 0) return fail(s, GM_ERR_STATE, "%s: the system was not created with such tables", who);
    if (!c4 || type < 0 || type >= GM_MAX_BOND_TYPES) return fail(s, GM_ERR_INVALID_ARG, "%s: bad type or NULL", who);
    CU(cudaSetDevice(s->cfg.device));
    CU(cudaMemcpyAsync(dst + (size_t)type * np, c4, (size_t)np * 16, cudaMemcpyHostToDevice, s->st));
    CU(cudaStreamSynchronize(s->st));              // the caller may reuse c4 at once
    s->force_current = false;
    return GM_OK;
}

extern "C" gm_status gm_set_angle_table(gm_system *s, int atype, const float *c4)
{
    if (!s) return GM_ERR_INVALID_ARG;
    return set_topo_table(s, atype, c4, s->D.atable, s->P.angle_table_points, "gm_set_angle_table");
}

extern "C" gm_status gm_set_dihedral_table(gm_system *s, int dtype, const float *c4)
{
    if (!s) return GM_ERR_INVALID_ARG;
    return set_topo_table(s, dtype, c4, s->D.dtable, s->P.dihedral_table_points, "gm_set_dihedral_table");
}

// Per-particle angle / dihedral tables: every interaction under every member, with the member's
// position.  NM = members per interaction (3 or 4); entry of the member at position p: the other members in order,
// then (angles) p and the type, (dihedrals) p | type << 2.
template <int NM>
static gm_status set_topology(gm_system *s, int64_t count, const int32_t *tags, const int32_t *type, int max_rows, int4 *table,
                              const char *who)
{
    if (count < 0 || (count > 0 && !tags)) return fail(s, GM_ERR_INVALID_ARG, "%s: bad arguments", who);
    if (max_rows <= 0) {
        if (count == 0) return GM_OK;
        return fail(s, GM_ERR_INVALID_ARG, "%s: the per-particle table has no rows (max_*_per_particle is 0)", who);
    }
    CU(cudaSetDevice(s->cfg.device));
    const size_t n = (size_t)s->P.n, ns = (size_t)s->P.ns;
    std::vector<int32_t> rows(n, 0);
    std::vector<int4> tb(ns * (size_t)max_rows, make_int4(-1, -1, -1, -1));
    for (int64_t q = 0; q < count; ++q) {
        const int32_t *m = tags + NM * q;
        const int32_t ty = type ? type[q] : 0;
        if (ty < 0 || ty >= GM_MAX_BOND_TYPES) return fail(s, GM_ERR_INVALID_ARG, "%s: type out of range", who);
        for (int a = 0; a < NM; ++a) {
            if (m[a] < 0 || (size_t)m[a] >= n) return fail(s, GM_ERR_INVALID_ARG, "%s: tag out of range", who);
            for (int b = 0; b < a; ++b) if (m[a] == m[b]) return fail(s, GM_ERR_INVALID_ARG, "%s: a bead appears twice", who);
        }
        for (int p = 0; p < NM; ++p) {
            const int32_t own = m[p];
            if (rows[own] >= max_rows) return fail(s, GM_ERR_INVALID_ARG, "%s: a bead exceeds max_*_per_particle", who);
            int32_t o[3] = { -1, -1, -1 };
            for (int a = 0, c = 0; a < NM; ++a) if (a != p) o[c++] = m[a];
            int4 e;
            if (NM == 3) e = make_int4(o[0], o[1], p, ty);
            else e = make_int4(o[0], o[1], o[2], p | (ty << 2));
            tb[(size_t)rows[own] * ns + own] = e;
            rows[own] += 1;
        }
    }
    CU(cudaMemcpyAsync(table, tb.data(), tb.size() * sizeof(int4), cudaMemcpyHostToDevice, s->st));
    CU(cudaStreamSynchronize(s->st));
    s->force_current = false;
    return GM_OK;
}

extern "C" gm_status gm_set_angles(gm_system *s, int64_t n_angles, const int32_t *tags3, const int32_t *atype)
{
    if (!s) return GM_ERR_INVALID_ARG;
    return set_topology<3>(s, n_angles, tags3, atype, s->P.max_angles, s->D.at, "gm_set_angles");
}

extern "C" gm_status gm_set_dihedrals(gm_system *s, int64_t n_dihedrals, const int32_t *tags4, const int32_t *dtype)
{
    if (!s) return GM_ERR_INVALID_ARG;
    return set_topology<4>(s, n_dihedrals, tags4, dtype, s->P.max_dihedrals, s->D.dt, "gm_set_dihedrals");
}

// ---- particles and bonds ----------------------------------------------------------------------------
extern "C" gm_status gm_set_particles(gm_system *s, const float *pos3, const float *vel3, const int32_t *type,
                                      const float *mass, int on_device)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!pos3 || !vel3 || !type) return fail(s, GM_ERR_INVALID_ARG, "gm_set_particles: NULL array%s");
    CU(cudaSetDevice(s->cfg.device));
    const size_t n = (size_t)s->P.n;
    const float *dp = pos3, *dv = vel3, *dm = mass;
    const int *dt = type;
    if (!on_device) {
        float *st = s->D.stage;
        CU(cudaMemcpyAsync(st, pos3, n * 12, cudaMemcpyHostToDevice, s->st));
        CU(cudaMemcpyAsync(st + 3 * n, vel3, n * 12, cudaMemcpyHostToDevice, s->st));
        CU(cudaMemcpyAsync(st + 9 * n, type, n * 4, cudaMemcpyHostToDevice, s->st));
        if (mass) CU(cudaMemcpyAsync(st + 10 * n, mass, n * 4, cudaMemcpyHostToDevice, s->st));
        dp = st; dv = st + 3 * n; dt = (const int *)(st + 9 * n); dm = mass ? st + 10 * n : nullptr;
        CU(cudaStreamSynchronize(s->st));      // "copies inputs in": the caller may reuse (pinned) buffers at once
    }
    // Andersen barostat (gm_npt.cuh): the arrays hold s = r / lambda and c = lambda v; the box of gm_set_box_state applies
    const double lam = std::cbrt(s->npt_V / s->npt_vol0);
    if (lam != 1.0) {
        float *st = s->D.stage;
        if (on_device) {
            CU(cudaMemcpyAsync(st, pos3, n * 12, cudaMemcpyDeviceToDevice, s->st));
            CU(cudaMemcpyAsync(st + 3 * n, vel3, n * 12, cudaMemcpyDeviceToDevice, s->st));
            dp = st; dv = st + 3 * n;
        }
        gm_launch_scale3(st, 3 * n, (float)(1.0 / lam), s->st);
        gm_launch_scale3(st + 3 * n, 3 * n, (float)lam, s->st);
    }
    s->cur = 0;
    gm_launch_npt_init(s->D, 0, s->npt_vol0, s->npt_V, s->npt_Pi, s->npt_p_ext, s->npt_mass, s->st);
    gm_launch_set_ctl(s->D, 0, 1, 0, s->st);             // clears the latched device errors: before the pack
    gm_launch_pack(s->P, s->D, 0, dp, dv, dt, dm, s->st);
    CU(cudaGetLastError());
    s->step = 0;
    s->have_particles = true;
    s->lagged = false;
    s->nl_valid = false;
    s->force_current = false;
    s->bonds_dirty = true;
    return GM_OK;
}

extern "C" gm_status gm_set_bonds(gm_system *s, int64_t n_bonds, const int32_t *tag_pairs2, const int32_t *btype,
                                  int on_device)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (n_bonds < 0 || (n_bonds > 0 && !tag_pairs2)) return fail(s, GM_ERR_INVALID_ARG, "gm_set_bonds: bad arguments%s");
    if (s->P.max_bonds <= 0) {
        if (n_bonds == 0) return GM_OK;
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_bonds: max_bonds_per_particle is 0%s");
    }
    CU(cudaSetDevice(s->cfg.device));
    std::vector<int32_t> hp, ht;
    const int32_t *pp = tag_pairs2, *tt = btype;
    if (on_device && n_bonds > 0) {
        hp.resize((size_t)n_bonds * 2);
        CU(cudaMemcpyAsync(hp.data(), tag_pairs2, hp.size() * 4, cudaMemcpyDeviceToHost, s->st));
        if (btype) { ht.resize((size_t)n_bonds); CU(cudaMemcpyAsync(ht.data(), btype, ht.size() * 4, cudaMemcpyDeviceToHost, s->st)); }
        CU(cudaStreamSynchronize(s->st));
        pp = hp.data(); tt = btype ? ht.data() : nullptr;
    }
    const size_t n = (size_t)s->P.n, ns = (size_t)s->P.ns;
    const int mb = s->P.max_bonds;
    std::vector<int32_t> bn(n, 0), bl(ns * (size_t)mb, -1);
    for (int64_t b = 0; b < n_bonds; ++b) {
        int32_t i = pp[2 * b], j = pp[2 * b + 1];
        int32_t t = tt ? tt[b] : 0;
        if (i < 0 || j < 0 || (size_t)i >= n || (size_t)j >= n || i == j || t < 0 || t >= GM_MAX_BOND_TYPES)
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_bonds: tag or bond type out of range%s");
        if (bn[i] >= mb || bn[j] >= mb)
            return fail(s, GM_ERR_INVALID_ARG, "gm_set_bonds: a bead exceeds max_bonds_per_particle%s");
        bl[(size_t)bn[i] * ns + i] = j | (t << GM_BOND_SHIFT); bn[i] += 1;   // stored under both ends
        bl[(size_t)bn[j] * ns + j] = i | (t << GM_BOND_SHIFT); bn[j] += 1;
    }
    CU(cudaMemcpyAsync(s->D.bl_tag, bl.data(), ns * 4 * (size_t)mb, cudaMemcpyHostToDevice, s->st));
    CU(cudaStreamSynchronize(s->st));      // the host vectors go out of scope
    s->bonds_dirty = true;
    s->force_current = false;
    return GM_OK;
}

extern "C" gm_status gm_set_step(gm_system *s, uint64_t step)
{
    if (!s) return GM_ERR_INVALID_ARG;
    CU(cudaSetDevice(s->cfg.device));
    gm_launch_set_ctl(s->D, step, 0, s->cur, s->st);
    CU(cudaGetLastError());
    s->step = step;
    s->nl_valid = false;       // `need` was reset: rebuild before the next force evaluation
    s->force_current = false;
    return GM_OK;
}

// ---- rebuild scheduling -------------------------------------------------------------------------------
// gate kernel (decides on the device, publishes ctl->go) -> a1 + a2 (sort) -> a3 (NL build)
static void enqueue_rebuild(gm_system *s, int gate, cudaStream_t st)
{
    gm_launch_gate(s->D, gate, s->cur, 0ull, 0, st);
    gm_launch_sort(s->P, s->D, s->cur, st);
    gm_launch_nl_build(s->P, s->D, st, &s->fk);
}

// Make the NL usable for a force evaluation at the current time level, outside the graphs.
static gm_status ensure_list(gm_system *s)
{
    const bool forced = !s->nl_valid;
    if (s->bonds_dirty) { gm_launch_bonds_from_master(s->P, s->D, s->st); s->bonds_dirty = false; }
    enqueue_rebuild(s, forced ? 0 : 1, s->st);
    if (forced) s->force_current = false;
    s->nl_valid = true;
    CU(cudaGetLastError());
    return GM_OK;
}

static void kicks(const gm_system *s, float *kick, float *kick_vt)
{
    const float dt = s->P.dt;
    *kick = s->lagged ? dt : 0.5f * dt;
    if (s->P.integrator == GM_DPD_GWVV) *kick_vt = s->lagged ? (0.5f + s->P.lambda) * dt : s->P.lambda * dt;
    else *kick_vt = *kick;
}

static void enqueue_step_kernel(gm_system *s, bool lagged, cudaStream_t st)
{
    bool keep = s->lagged;
    s->lagged = lagged;
    float kick, kick_vt;
    kicks(s, &kick, &kick_vt);
    s->lagged = keep;
    if (is_npt(s)) {         // Andersen barostat: forces + virial, then piston + kick + drift (gm_npt.cu)
        gm_launch_npt_force(s->P, s->D, s->cur, 0, st);
        gm_launch_npt_update(s->P, s->D, s->cur, kick, st);
    } else
        gm_launch_force(s->P, s->D, GM_MODE_STEP, s->cur, kick, kick_vt, 0, st);
    s->cur ^= 1;
}

// Capture `nsteps` (even) steps starting from buffer 0 into an executable graph.  Each step is:
// gate -> IF(rebuild due){a1, a3} -> fused force + integrate kernel.  Without conditional nodes the
// rebuild kernels are launched every step and return at once when no rebuild is due.
static gm_status capture_graph(gm_system *s, int nsteps, cudaGraphExec_t *exec)
{
    const int cur0 = s->cur;
    cudaGraph_t graph = nullptr;
    s->cur = 0;
    cudaError_t e = cudaStreamBeginCapture(s->cap_st, cudaStreamCaptureModeRelaxed);
    bool ok = (e == cudaSuccess);
    // one conditional handle per timestep (default 0 at every graph launch): timestep 0 is gated by a one-thread kernel
    // that reads ctl->need; the step kernel of timestep k - 1 raises the handle of timestep k itself
    std::vector<cudaGraphConditionalHandle> hs((size_t)nsteps);
    if (ok && s->use_cond) {
        cudaStreamCaptureStatus status;
        cudaGraph_t g = nullptr;
        ok = cudaStreamGetCaptureInfo(s->cap_st, &status, nullptr, &g, nullptr, nullptr) == cudaSuccess;
        for (int k = 0; ok && k < nsteps; ++k)
            ok = cudaGraphConditionalHandleCreate(&hs[k], g, 0, cudaGraphCondAssignDefault) == cudaSuccess;
    }
    for (int k = 0; ok && k < nsteps; ++k) {
        if (s->use_cond) {
            cudaStreamCaptureStatus status;
            cudaGraph_t g = nullptr;
            const cudaGraphNode_t *deps = nullptr;
            size_t ndeps = 0;
            const cudaGraphConditionalHandle h = hs[k];
            if (k == 0) gm_launch_gate(s->D, 1, s->cur, (unsigned long long)h, 1, s->cap_st);
            ok = ok && cudaStreamGetCaptureInfo(s->cap_st, &status, nullptr, &g, &deps, &ndeps) == cudaSuccess;
            cudaGraphNodeParams np = {};
            np.type = cudaGraphNodeTypeConditional;
            np.conditional.handle = h;
            np.conditional.type = cudaGraphCondTypeIf;
            np.conditional.size = 1;
            cudaGraphNode_t node = nullptr;
            ok = ok && cudaGraphAddNode(&node, g, deps, ndeps, &np) == cudaSuccess;
            if (ok) {
                cudaGraph_t body = np.conditional.phGraph_out[0];
                ok = cudaStreamBeginCaptureToGraph(s->cap_st2, body, nullptr, nullptr, 0,
                                                   cudaStreamCaptureModeRelaxed) == cudaSuccess;
                if (ok) {
                    // the body of a gate-less timestep starts with the gate's bookkeeping (ctl->go, rebuild counter)
                    if (k > 0) gm_launch_gate(s->D, 1, s->cur, 0ull, 0, s->cap_st2);
                    gm_launch_sort(s->P, s->D, s->cur, s->cap_st2);
                    gm_launch_nl_build(s->P, s->D, s->cap_st2, &s->fk);
                    cudaGraph_t tmp = nullptr;
                    ok = cudaStreamEndCapture(s->cap_st2, &tmp) == cudaSuccess;
                }
                ok = ok && cudaStreamUpdateCaptureDependencies(s->cap_st, &node, 1,
                                                               cudaStreamSetCaptureDependencies) == cudaSuccess;
            }
        } else {
            enqueue_rebuild(s, 1, s->cap_st);
        }
        if (ok) {
            s->D.next_cond = (s->use_cond && k + 1 < nsteps) ? (unsigned long long)hs[k + 1] : 0ull;
            enqueue_step_kernel(s, true, s->cap_st);
            s->D.next_cond = 0ull;
        }
    }
    e = cudaStreamEndCapture(s->cap_st, &graph);
    ok = ok && e == cudaSuccess && graph != nullptr;
    if (ok) ok = cudaGraphInstantiate(exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    s->cur = cur0;
    if (!ok) {
        cudaGetLastError();
        *exec = nullptr;
        return GM_ERR_CUDA;
    }
    return GM_OK;
}

static gm_status get_graph(gm_system *s, int nsteps, cudaGraphExec_t *slot)
{
    if (*slot) return GM_OK;
    gm_status r = capture_graph(s, nsteps, slot);
    if (r != GM_OK && s->use_cond) {      // conditional nodes unavailable: fall back to early-exit gating
        s->use_cond = false;
        r = capture_graph(s, nsteps, slot);
    }
    if (r != GM_OK) return fail(s, GM_ERR_CUDA, "CUDA graph capture failed%s");
    return GM_OK;
}

extern "C" gm_status gm_build_neighbors(gm_system *s)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_build_neighbors: no particles set%s");
    CU(cudaSetDevice(s->cfg.device));
    s->nl_valid = false;
    return ensure_list(s);
}

extern "C" gm_status gm_compute_forces(gm_system *s)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_compute_forces: no particles set%s");
    CU(cudaSetDevice(s->cfg.device));
    gm_status r = ensure_list(s);
    if (r != GM_OK) return r;
    if (is_npt(s)) gm_launch_npt_force(s->P, s->D, s->cur, 1, s->st);
    else gm_launch_force(s->P, s->D, GM_MODE_FORCES, s->cur, 0.f, 0.f, 0, s->st);
    CU(cudaGetLastError());
    s->force_current = true;
    return GM_OK;
}

struct StepTiming {
    std::vector<cudaEvent_t> ev;     // 3 per step: before rebuild, before force, after force
};

static gm_status step_impl(gm_system *s, int64_t n_steps, StepTiming *tm)
{
    if (n_steps > 0 && (!s->nl_valid || s->bonds_dirty)) {
        gm_status r = ensure_list(s);
        if (r != GM_OK) return r;
    }
    int64_t done = 0;
    while (done < n_steps) {
        const int64_t rem = n_steps - done;
        if (!tm && s->use_graph && s->lagged && s->cur == 0 && rem >= 2) {
            cudaGraphExec_t *slot = rem >= GM_GRAPH_STEPS ? &s->exec_big : (rem >= GM_GRAPH_STEPS_MID ? &s->exec_mid : &s->exec_two);
            const int ns = rem >= GM_GRAPH_STEPS ? GM_GRAPH_STEPS : (rem >= GM_GRAPH_STEPS_MID ? GM_GRAPH_STEPS_MID : 2);
            gm_status r = get_graph(s, ns, slot);
            if (r != GM_OK) return r;
            CU(cudaGraphLaunch(*slot, s->st));
            done += ns;
            s->step += (uint64_t)ns;
        } else {
            cudaEvent_t e[3] = { nullptr, nullptr, nullptr };
            if (tm) {
                for (int q = 0; q < 3; ++q) { CU(cudaEventCreate(&e[q])); tm->ev.push_back(e[q]); }
                CU(cudaEventRecord(e[0], s->st));
            }
            enqueue_rebuild(s, 1, s->st);
            if (tm) CU(cudaEventRecord(e[1], s->st));
            enqueue_step_kernel(s, s->lagged, s->st);
            if (tm) CU(cudaEventRecord(e[2], s->st));
            s->lagged = true;
            done += 1;
            s->step += 1;
        }
    }
    CU(cudaGetLastError());
    if (n_steps > 0) s->force_current = false;
    return GM_OK;
}

extern "C" gm_status gm_step(gm_system *s, int64_t n_steps)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_step: no particles set%s");
    if (n_steps < 0) return fail(s, GM_ERR_INVALID_ARG, "gm_step: n_steps < 0%s");
    CU(cudaSetDevice(s->cfg.device));
    return step_impl(s, n_steps, nullptr);
}

extern "C" gm_status gm_step_timed(gm_system *s, int64_t n_steps, double out[4])
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_step_timed: no particles set%s");
    if (n_steps < 0 || n_steps > 100000 || !out) return fail(s, GM_ERR_INVALID_ARG, "gm_step_timed: bad arguments%s");
    CU(cudaSetDevice(s->cfg.device));
    StepTiming tm;
    GmCtl c0, c1;
    CU(cudaMemcpyAsync(&c0, s->D.ctl, sizeof(c0), cudaMemcpyDeviceToHost, s->st));
    CU(cudaStreamSynchronize(s->st));
    gm_status r = step_impl(s, n_steps, &tm);
    if (cudaMemcpyAsync(&c1, s->D.ctl, sizeof(c1), cudaMemcpyDeviceToHost, s->st) != cudaSuccess) c1 = c0;
    cudaError_t e = cudaStreamSynchronize(s->st);
    double t_force = 0.0, t_rebuild = 0.0;
    for (size_t k = 0; k + 2 < tm.ev.size() + 0 && e == cudaSuccess; k += 3) {
        float a = 0.f, b = 0.f;
        e = cudaEventElapsedTime(&a, tm.ev[k], tm.ev[k + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&b, tm.ev[k + 1], tm.ev[k + 2]);
        t_rebuild += a; t_force += b;
    }
    for (cudaEvent_t ev : tm.ev) cudaEventDestroy(ev);
    if (r != GM_OK) return r;
    if (e != cudaSuccess) return fail(s, GM_ERR_CUDA, "CUDA: %s", cudaGetErrorString(e));
    out[0] = t_force; out[1] = t_rebuild; out[2] = (double)(tm.ev.size() / 3); out[3] = (double)(c1.n_rebuilds - c0.n_rebuilds);
    return GM_OK;
}

extern "C" gm_status gm_set_integrator(gm_system *s, int integrator, float kT, float gamma)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (integrator < GM_NVE || integrator > GM_NPT_ANDERSEN)
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_integrator: unknown integrator%s");
    const bool to_npt = integrator == GM_NPH_ANDERSEN || integrator == GM_NPT_ANDERSEN;
    if (to_npt && (s->P.use_win || s->P.step_subw != 1 || (s->P.pair_style != GM_PAIR_LJ && s->P.pair_style != GM_PAIR_NONE)))
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_integrator: the barostat needs GM_PAIR_LJ or GM_PAIR_NONE "
                                           "and a system without tile windows (GM_FLAG_NO_WINDOWS, or created with an NP* integrator)%s");
    if (!to_npt && is_npt(s))
        return fail(s, GM_ERR_STATE, "gm_set_integrator: a system under the barostat stays under it (its box has changed)%s");
    if (integrator >= GM_NVT_NOSE_HOOVER && s->P.step_subw != 1)
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_integrator: the NVT thermostats do not run on the sub-warp step kernel%s");
    if ((integrator == GM_DPD_GWVV) != (s->P.pair_style == GM_PAIR_DPD))
        return fail(s, GM_ERR_INVALID_ARG, "gm_set_integrator: GM_DPD_GWVV goes with GM_PAIR_DPD only%s");
    if (!(kT >= 0.f) || !(gamma >= 0.f)) return fail(s, GM_ERR_INVALID_ARG, "gm_set_integrator: kT, gamma must be >= 0%s");
    s->cfg.integrator = integrator; s->cfg.kT = kT; s->cfg.gamma = gamma;
    s->P.integrator = integrator; s->P.kT = kT; s->P.gamma = gamma;
    s->P.sigma_r_sqrt_inv_dt = (float)std::sqrt(2.0 * (double)gamma * (double)kT / (double)s->P.dt);
    s->P.lang_amp2 = (float)(6.0 * (double)gamma * (double)kT / (double)s->P.dt);
    s->force_current = false;
    drop_graphs(s);
    CU(cudaSetDevice(s->cfg.device));
    gm_launch_thermo_reset(s->D, s->cur, s->st);
    CU(cudaGetLastError());
    return GM_OK;
}

// ---- results ----------------------------------------------------------------------------------------
static gm_status dev_error(gm_system *s, const GmCtl &c)
{
    if (c.err & GM_DEV_ERR_BAD_INPUT) return fail(s, GM_ERR_INVALID_ARG, "gm_set_particles: a type outside [0, n_types) or a mass <= 0%s");
    if (c.err & GM_DEV_ERR_BOX) return fail(s, GM_ERR_BOX_TOO_SMALL, "the barostat shrank the box below what the neighbor list of gm_create covers%s");
    if (c.err & GM_DEV_ERR_WINDOW) return fail(s, GM_ERR_CUDA, "a tile window copy did not complete (internal error)%s");
    if (c.err & GM_DEV_ERR_NONFINITE) return fail(s, GM_ERR_NONFINITE, "a coordinate became non-finite%s");
    if (c.err & GM_DEV_ERR_OVERSTRETCH) return fail(s, GM_ERR_BOND_OVERSTRETCH, "a FENE bond reached r >= R0%s");
    if (c.err & GM_DEV_ERR_OVERFLOW) return fail(s, GM_ERR_NEIGHBOR_OVERFLOW, "a neighbor row exceeded nl_row_capacity%s");
    return GM_OK;
}

static gm_status sync_and_check(gm_system *s, GmCtl *out = nullptr)
{
    GmCtl c;
    CU(cudaMemcpyAsync(&c, s->D.ctl, sizeof(c), cudaMemcpyDeviceToHost, s->st));
    CU(cudaStreamSynchronize(s->st));
    if (out) *out = c;
    return dev_error(s, c);
}

// Andersen barostat: one force evaluation at the current time level outside the time stepping, and what follows from its
// sums -- the kinetic energy of the full-step velocities v = (c + h lambda F / m) / lambda, h = dt/2 once a half-step
// velocity is stored, and the piston momentum completed by the same half kick
struct NptProbe { double K, pe_pair, pe_bond, W, V, Pi, lam, P_inst, H; };

static gm_status npt_probe(gm_system *s, NptProbe *o)
{
    gm_status r = ensure_list(s);
    if (r != GM_OK) return r;
    gm_launch_npt_force(s->P, s->D, s->cur, 1, s->st);
    CU(cudaGetLastError());
    s->force_current = true;
    GmNpt h;
    CU(cudaMemcpyAsync(&h, gm_npt_state(s->D), sizeof(h), cudaMemcpyDeviceToHost, s->st));
    r = sync_and_check(s);
    double sm[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
    for (int c = 0; c < GM_NPT_SLOTS; ++c)
        for (int q = 0; q < 8; ++q) sm[q] += h.sum[2][c][q];
    const double lam = h.lam[s->cur], V = h.V[s->cur], hk = s->lagged ? 0.5 * (double)s->P.dt : 0.0;
    const double S = sm[1] + 2.0 * hk * lam * sm[2] + hk * hk * lam * lam * sm[3];
    o->K = S / (2.0 * lam * lam);
    o->pe_pair = sm[4]; o->pe_bond = sm[5]; o->W = sm[0]; o->V = V; o->lam = lam;
    o->Pi = h.Pi[s->cur] + hk * (sm[0] / (3.0 * V) - h.p_ext);
    o->P_inst = (2.0 * o->K + o->W) / (3.0 * V);
    o->H = o->K + o->pe_pair + o->pe_bond + h.p_ext * V + o->Pi * o->Pi / (2.0 * h.mass);
    return r;
}

extern "C" gm_status gm_set_barostat(gm_system *s, float p_ext, float piston_mass)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!(p_ext >= 0.f) || !(piston_mass > 0.f)) return fail(s, GM_ERR_INVALID_ARG, "gm_set_barostat: p_ext >= 0 and piston_mass > 0%s");
    if (s->have_particles && s->step > 0 && is_npt(s))
        return fail(s, GM_ERR_STATE, "gm_set_barostat: call it before the first step under the barostat%s");
    CU(cudaSetDevice(s->cfg.device));
    s->npt_p_ext = (double)p_ext; s->npt_mass = (double)piston_mass;
    gm_launch_npt_init(s->D, s->cur, s->npt_vol0, s->npt_V, s->npt_Pi, s->npt_p_ext, s->npt_mass, s->st);
    CU(cudaGetLastError());
    return GM_OK;
}

extern "C" gm_status gm_set_box_state(gm_system *s, double volume, double piston_momentum)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!(volume > 0.0) || !std::isfinite(piston_momentum)) return fail(s, GM_ERR_INVALID_ARG, "gm_set_box_state: volume > 0%s");
    if (s->have_particles) return fail(s, GM_ERR_STATE, "gm_set_box_state: call it before gm_set_particles%s");
    CU(cudaSetDevice(s->cfg.device));
    s->npt_V = volume; s->npt_Pi = piston_momentum;
    gm_launch_npt_init(s->D, s->cur, s->npt_vol0, s->npt_V, s->npt_Pi, s->npt_p_ext, s->npt_mass, s->st);
    CU(cudaGetLastError());
    return GM_OK;
}

extern "C" gm_status gm_get_box(gm_system *s, double out[8])
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!out) return fail(s, GM_ERR_INVALID_ARG, "gm_get_box: NULL out%s");
    CU(cudaSetDevice(s->cfg.device));
    for (int q = 0; q < 8; ++q) out[q] = 0.0;
    if (!is_npt(s) || !s->have_particles) {
        const double lam = std::cbrt(s->npt_V / s->npt_vol0);
        for (int d = 0; d < 3; ++d) out[d] = lam * (double)s->cfg.box[d];
        out[3] = s->npt_V; out[4] = s->npt_Pi;
        return GM_OK;
    }
    NptProbe q;
    gm_status r = npt_probe(s, &q);
    for (int d = 0; d < 3; ++d) out[d] = q.lam * (double)s->cfg.box[d];
    out[3] = q.V; out[4] = q.Pi; out[5] = q.P_inst; out[6] = q.W; out[7] = q.H;
    return r;
}

extern "C" gm_status gm_energies(gm_system *s, double out[8])
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!out) return fail(s, GM_ERR_INVALID_ARG, "gm_energies: NULL out%s");
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_energies: no particles set%s");
    CU(cudaSetDevice(s->cfg.device));
    if (is_npt(s)) {
        NptProbe q;
        gm_status rq = npt_probe(s, &q);
        const double dofq = s->P.n > 1 ? 3.0 * s->P.n - 3.0 : 3.0;
        out[0] = q.K; out[1] = q.pe_pair; out[2] = q.pe_bond; out[3] = 2.0 * q.K / dofq;
        out[4] = out[5] = out[6] = out[7] = 0.0;
        return rq;
    }
    gm_status r = ensure_list(s);
    if (r != GM_OK) return r;
    gm_launch_force(s->P, s->D, GM_MODE_ENERGY, s->cur, 0.f, 0.f, s->lagged ? 1 : 0, s->st);
    CU(cudaGetLastError());
    double h[8];
    CU(cudaMemcpyAsync(h, s->D.esum + (size_t)GM_ESUM_BLOCKS * 8, sizeof(h), cudaMemcpyDeviceToHost, s->st));
    r = sync_and_check(s);
    const double dof = s->P.n > 1 ? 3.0 * s->P.n - 3.0 : 3.0;
    out[0] = h[0]; out[1] = h[1]; out[2] = h[2];
    out[3] = 2.0 * h[0] / dof;
    out[4] = h[3]; out[5] = h[4]; out[6] = h[5]; out[7] = h[6];
    return r;
}

extern "C" gm_status gm_get_particles(gm_system *s, float *pos3, float *vel3, float *force3, int on_device)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_get_particles: no particles set%s");
    CU(cudaSetDevice(s->cfg.device));
    if ((force3 || (vel3 && s->lagged)) && !s->force_current) {
        gm_status r = gm_compute_forces(s);
        if (r != GM_OK) return r;
    }
    const size_t n = (size_t)s->P.n;
    float *st = s->D.stage;
    float *dp = pos3, *dv = vel3, *df = force3;
    if (!on_device) {
        dp = pos3 ? st : nullptr; dv = vel3 ? st + 3 * n : nullptr; df = force3 ? st + 6 * n : nullptr;
    }
    if (is_npt(s)) {
        if (!s->force_current) {           // the real-unit output needs the forces of this time level in any case
            gm_status r = gm_compute_forces(s);
            if (r != GM_OK) return r;
        }
        gm_launch_npt_unpack(s->P, s->D, s->cur, dp, dv, df, s->lagged ? 1 : 0, s->st);
    } else
        gm_launch_unpack(s->P, s->D, s->cur, dp, dv, df, s->lagged ? 1 : 0, s->st);
    CU(cudaGetLastError());
    if (!on_device) {
        if (pos3) CU(cudaMemcpyAsync(pos3, dp, n * 12, cudaMemcpyDeviceToHost, s->st));
        if (vel3) CU(cudaMemcpyAsync(vel3, dv, n * 12, cudaMemcpyDeviceToHost, s->st));
        if (force3) CU(cudaMemcpyAsync(force3, df, n * 12, cudaMemcpyDeviceToHost, s->st));
        return sync_and_check(s);
    }
    return GM_OK;
}

extern "C" gm_status gm_get_neighbors(gm_system *s, int32_t *nn, int32_t *nl_tags, int64_t row_stride, int on_device)
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!s->have_particles) return fail(s, GM_ERR_STATE, "gm_get_neighbors: no particles set%s");
    if (!nn || !nl_tags || row_stride < 1) return fail(s, GM_ERR_INVALID_ARG, "gm_get_neighbors: bad arguments%s");
    CU(cudaSetDevice(s->cfg.device));
    {   // gated rebuild: a no-op when the list is current at this time level (a4)
        gm_status r = ensure_list(s);
        if (r != GM_OK) return r;
    }
    GmCtl c;
    gm_status r = sync_and_check(s, &c);
    if (r != GM_OK) return r;
    if (row_stride < c.max_nn) return fail(s, GM_ERR_INVALID_ARG, "gm_get_neighbors: row_stride < max nn%s");
    const int n = s->P.n;
    if (on_device) {
        gm_launch_unpack_neighbors(s->P, s->D, nn, nl_tags, row_stride, 0, n, s->st);
        CU(cudaGetLastError());
        return GM_OK;
    }
    // host output: tag ranges that fit the I/O staging area of the workspace (11 ns floats), one range at a time
    int *st = reinterpret_cast<int *>(s->D.stage);
    const long long rows_fit = (long long)((size_t)s->P.ns * 11 / (size_t)(row_stride + 1));
    if (rows_fit < 1) return fail(s, GM_ERR_INVALID_ARG, "gm_get_neighbors: row_stride too large for the staging area%s");
    for (long long t0 = 0; t0 < n; t0 += rows_fit) {
        const int t1 = (int)std::min<long long>(n, t0 + rows_fit);
        const size_t m = (size_t)(t1 - t0);
        gm_launch_unpack_neighbors(s->P, s->D, st, st + m, row_stride, (int)t0, t1, s->st);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(nn + t0, st, m * 4, cudaMemcpyDeviceToHost, s->st));
        CU(cudaMemcpyAsync(nl_tags + t0 * row_stride, st + m, m * 4 * (size_t)row_stride, cudaMemcpyDeviceToHost, s->st));
        CU(cudaStreamSynchronize(s->st));
    }
    return GM_OK;
}

extern "C" gm_status gm_get_tuning(gm_system *s, int64_t out[8])
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!out) return fail(s, GM_ERR_INVALID_ARG, "gm_get_tuning: NULL out%s");
    CU(cudaSetDevice(s->cfg.device));
    GmCtl c;
    gm_status r = sync_and_check(s, &c);
    if (r == GM_ERR_CUDA) return r;
    out[0] = s->P.sx; out[1] = s->P.nl_trip; out[2] = s->P.step_wide ? 2 : 1; out[3] = s->P.use_win;
    out[4] = s->P.win_cap; out[5] = (s->P.n + GM_TILE - 1) / GM_TILE;
    out[6] = s->P.use_win ? c.n_glob_tiles : out[5];
    out[7] = gm_nl_smem_bytes(s->P);
    return GM_OK;
}

extern "C" gm_status gm_get_stats(gm_system *s, int64_t out[8])
{
    if (!s) return GM_ERR_INVALID_ARG;
    if (!out) return fail(s, GM_ERR_INVALID_ARG, "gm_get_stats: NULL out%s");
    CU(cudaSetDevice(s->cfg.device));
    GmCtl c;
    gm_status r = sync_and_check(s, &c);
    if (r == GM_ERR_CUDA) return r;
    out[0] = (int64_t)s->step;
    out[1] = (int64_t)c.n_rebuilds;
    out[2] = (int64_t)c.n_rebuilds;      // every rebuild sorts along the SFC
    out[3] = c.max_nn;
    out[4] = (int64_t)c.sum_nn;
    out[5] = c.err;
    out[6] = s->P.nl_cap;
    out[7] = s->P.n_cells;
    return r;
}
