// gm_internal.cuh -- shared declarations of libgm's CUDA path (sm_100a).  Nothing here is used by,
// or derived from, the CPU oracle under oracle/.
//
// Device data layout.  STORAGE order is the cell order of the last
// neighbor-list rebuild: every rebuild counting-sorts the beads by cell (a1) along the space-filling
// curve (a2) and moves all per-bead state, so bead s of cell c sits at s in [cstart[c], cstart[c+1]).
//   pos[2]  float4[ns]  x, y, z, type (int bits)          ping-pong by time-level parity
//   ref     float4[ns]  pos at the last rebuild, sorted    = the cell list CL in CSR form,
//                                                          the displacement reference (a4), and the
//                                                          position source of the step right after a rebuild
//   vel     float4[ns]  u_x, u_y, u_z, mass               u = half-step velocity; updated in place
//   svel    float4[ns]  vel permuted by the last rebuild  (source of the step right after a rebuild)
//   vt[2]   float4[ns]  v~_x, v~_y, v~_z, tag (int bits)  DPD only: the velocity the dissipative force sees
//   svt     float4[ns]  vt permuted by the last rebuild
//   frc     float4[ns]  F_x, F_y, F_z, per-bead PE        materialised only by gm_compute_forces
//   tag[2]  int[ns]     tag of the bead in each slot      double-buffered by rebuild parity (n_rebuilds & 1)
//   rtag    int[ns]     slot of each tag
//   nl      int4[n_tiles * capq * 32]  NL in tiles of 32 beads: entries 4q..4q+3 of bead (tile, lane)
//                       are the int4 at (tile * capq + q) * 32 + lane; slots past NN hold the index n
//                       (a far-away pad bead).  PAPER.md:L51, Fig. 1 (table form NL[k*Np+i], re-tiled)
//                       Window-staged tiles (wdesc header mode 1) hold 16-bit offsets into the tile's position window
//                       instead, eight per uint4 ("oct"), oct o of bead (tile, lane) at (tile * capq + o) * 32 + lane;
//                       unused slots hold 0, the window's pad bead.
//   wdesc   int4[n_tiles * GM_WD_STRIDE]  tile window descriptors: [k] = (first slot, window offset, length,
//                       n_ranges | mode << 8 | window length << 16) of range k < n_ranges; mode 0: [0] = 0
//   nn      int[ns]     NN[i];   nnw int[ns/32]: max NN per tile
//   blt[2]  int[mb*ns]  BL in TAG space, storage order: blt[k*ns + i] = partner tag | btype << 28, -1 = none
//   bl      int[mb*ns]  BL in index space: bl[k*ns + i] = j | btype << 28, -1 = none   PAPER.md:L97, Fig. 2
//   cstart  int[n_cells + 1]   replaces CN: cell c holds slots [cstart[c], cstart[c+1])
//   ccount  int[n_cells + 1]   histogram scratch (left zeroed by the scan)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gm.h"

#define GM_PAD 256               // per-bead arrays are allocated (and table rows strided) in multiples of this
#define GM_BOND_SHIFT 28
#define GM_BOND_LOCAL (1 << 27)  // BL entry: the partner index is an offset into the tile's position window
#define GM_BOND_MASK ((1 << 27) - 1)
#define GM_TILE 128              // beads per tile of the window-staged path: one CTA of k_nl_build and of the force kernels
#define GM_WD_STRIDE 40          // int4 entries per tile window descriptor, one per range
#define GM_WD_MAXR 40
#define GM_WIN_SLOTS 54          // window range slots of a tile: 2 row groups x 9 (y, z) rows x {A, B_lo, B_hi}
#define GM_NEVER (~0ull)

// latched device error bits (GmCtl::err)
enum { GM_DEV_ERR_OVERFLOW = 1, GM_DEV_ERR_OVERSTRETCH = 2, GM_DEV_ERR_NONFINITE = 4, GM_DEV_ERR_BAD_INPUT = 8, GM_DEV_ERR_WINDOW = 16 };

// Small device control block (one per system).
struct GmCtl {
    unsigned long long step[2];    // time level m, indexed by the parity of the current position buffer
    unsigned long long need;       // time level at which the NL must be rebuilt before forces (a4)
    unsigned long long rebuilt_at; // time level of the last rebuild: while == step, ref/svel/svt are current
    unsigned long long n_rebuilds; // its low bit selects the current tag[] / blt[] buffers
    unsigned long long sum_nn;
    int max_nn;
    int err;
    int go;                        // decision of the last k_gate: the rebuild chain runs iff != 0
    int n_glob_tiles;              // tiles of the current list that are NOT window-staged (32-bit rows, gathers from HBM/L2)
    // NVT thermostats (Nose-Hoover, Berendsen): sum of m u^2 over the half-step velocities written by the step kernel of
    // time level m goes to ke2[(m + 1) % 3]; that kernel reads ke2[m % 3] and clears ke2[(m + 2) % 3]; xi likewise
    double ke2[3];
    double xi[3];
    unsigned long long thermo_start;   // time level of the first kick after a (re)start: the thermostat acts from the next
};

// Per-type-pair coefficients.  LJ:       c0 = r_c^2, c1 = 48 eps sigma^12, c2 = 24 eps sigma^6, c3 = U_shift.
//                              DPD:      c0 = r_c^2, c1 = a, c2 = 1/r_c, c3 = r_c.
//                              harmonic: c0 = r_c^2, c1 = 2 alpha / r_c, c2 = 1/r_c, c3 = alpha           (Eq. 2)
//                              Gauss:    c0 = r_c^2, c1 = eps / sigma^2, c2 = -1/(2 sigma^2), c3 = U_shift, c4 = eps   (Eq. 3)
//                              table:    c0 = Npoint * interval (z at the cutoff), c1 = 1 / interval, c2 = interval,
//                                        c4 = index of the pair's first grid point in GmParams::table (int bits)   (Eqs. 11-12)
struct GmPair { float c0, c1, c2, c3, c4, c5, c6, c7; };

// Constants of one system, passed to kernels by value (constant bank).
struct GmParams {
    int n, n_types, max_bonds, nl_cap;
    int ns;                        // padded bead count: n + 8 rounded up to GM_PAD (slots n.. are far-away pad beads)
    int capq;                      // nl_cap / 4: int4 quads per NL row
    int minq;                      // quads of every row that are always written (padded): min(4, capq)
    int nc[3], n_cells;
    int nl_trip;                   // candidates the NL build loads together: 4 (short runs) or 8
    int sx;                        // cells are r_list / sx wide in x: the search reaches sx cells to either side
    int step_wide;                 // step kernel shape: 0 = one-warp CTAs (short lists), 1 = CTAs of 128 (long lists)
    int step_subw;                 // lanes per bead of the step kernel: 1 (short lists), 4 or 8 (long lists)
    int sfc_period;                // a rebuild (= SFC sort) is forced after this many steps without one; <= 0: never
    int use_win;                   // 1: tiles are window-staged where they can be (16-bit window-local NL rows)
    int win_cap;                   // positions a tile window holds at most (the shared-memory budget per warp)
    float box[3], half[3], inv_w[3];
    float r_list2, half_skin2;
    float edge_margin;             // r_list + r_skin: beads further than this from every face need no image test
    float dt, kT, gamma, lambda;
    float sigma_r_sqrt_inv_dt;     // sqrt(2 gamma kT / dt)             (DPD random force amplitude)
    float lang_amp2;               // 6 gamma kT / dt                   (Langevin: amp/m = sqrt(lang_amp2 / m))
    uint32_t seed_lo, seed_hi;
    int pair_style, bond_style, integrator;
    GmPair pair[GM_MAX_TYPES * GM_MAX_TYPES];
    float bond_k[GM_MAX_BOND_TYPES], bond_r0[GM_MAX_BOND_TYPES];
    float bond_c[GM_MAX_BOND_TYPES];   // FENE: 1 / R0^2
    int angle_style, max_angles, max_dihedrals;   // per-particle angle / dihedral tables (gm_topo.cu); has_topo = either > 0
    float angle_k[GM_MAX_BOND_TYPES], angle_t0[GM_MAX_BOND_TYPES], angle_c0[GM_MAX_BOND_TYPES];   // c0 = cos(theta0)
    float dih_k[GM_MAX_BOND_TYPES], dih_delta[GM_MAX_BOND_TYPES];
    int dih_n[GM_MAX_BOND_TYPES];
    const float4 *table;               // GM_PAIR_TABLE: (c0, c1, c2, c3) per grid point, n_types^2 tables of table_points
    int table_points;
    // GM_BOND_TABLE: (c0, c1, c2, c3) per grid point of z = r^2, GM_MAX_BOND_TYPES tables of bond_table_points;
    // bond_k[t] = 1 / interval, bond_r0[t] = interval of bond type t
    const float4 *btable;
    int bond_table_points;
    // GM_ANGLE_TABLE / tabulated dihedrals: (c0..c3) per grid interval of theta in [0, pi] / phi in [-pi, pi]
    const float4 *atable, *dtable;
    int angle_table_points, dihedral_table_points;
};

// Device pointers.
struct GmDev {
    float4 *pos[2];
    float4 *ref;
    float4 *vel, *svel;
    float4 *vt[2], *svt;
    float4 *frc;
    float4 *table;           // GM_PAIR_TABLE: spline coefficients, [n_types^2][table_points]
    float4 *btable;          // GM_BOND_TABLE: spline coefficients, [GM_MAX_BOND_TYPES][bond_table_points]
    float4 *atable, *dtable; // tabulated angle / dihedral potentials, [GM_MAX_BOND_TYPES][points]
    float4 *ftopo;           // angle + dihedral force (x, y, z) and energy share (w) of every bead, storage order
    int4 *at;                // angle table in TAG order: at[k * ns + tag] = (tag a, tag b, own position 0/1/2, type); x < 0: none
    int4 *dt;                // dihedral table in TAG order: dt[k * ns + tag] = (tag a, tag b, tag c, own position | type << 2)
    int *tag[2], *rtag;
    int *nn, *nnw;
    int4 *nl;
    int *bl;                 // index space
    int *blt[2];             // tag space, storage order
    int *bl_tag;             // tag space master copy in TAG order (bl_tag[k*ns + tag]), from gm_set_bonds
    int4 *wdesc;             // [n_tiles * GM_WD_STRIDE] tile window descriptors (see gm_nlist.cu)
    int *key, *rank, *sorted;
    int *cstart, *ccount;
    int *scan_sums;          // per scan block
    uint32_t *row_rank;      // SFC rank of each (y, z) row of cells
    float *stage;            // 11 ns floats: I/O staging (pos3, vel3, force3, type, mass)
    double *esum;            // [GM_ESUM_BLOCKS * 8] partials, then [8] totals at the end
    GmCtl *ctl;
    // Conditional-graph handle of the NEXT timestep's rebuild node (0 = none): inside a step graph the step kernel that
    // sees a displacement beyond skin/2 raises it itself, so only the first timestep of a graph needs a gate kernel
    unsigned long long next_cond;
};

#define GM_ESUM_BLOCKS 1184      // 8 x 148: grid of the energy reduction
#define GM_SCAN_BLOCK 1024
#define GM_SCAN_ITEMS 4          // per thread

enum { GM_MODE_STEP = 0, GM_MODE_FORCES = 1, GM_MODE_ENERGY = 2 };

// ---- launch wrappers (each enqueues on `st`; `gate` != 0: run only if ctl->need == ctl->step[parity];
//      a rebuild is always skipped when the list is already current, ctl->rebuilt_at == ctl->step[parity]) ----
void gm_launch_gate(const GmDev &D, int gate, int parity, unsigned long long cond_handle, int use_handle,
                    cudaStream_t st);                                                  // decides, publishes ctl->go
void gm_launch_sort(const GmParams &P, const GmDev &D, int parity, cudaStream_t st);    // a1 + a2 (if ctl->go)
// A side stream and two events (no timing) of one system: work that only the step kernel waits for (the BL remap of systems
// without tile windows) runs beside the neighbor build -- as a parallel branch when the launches are being captured
struct GmFork {
    cudaStream_t side;
    cudaEvent_t fork, join;
};
void gm_launch_nl_build(const GmParams &P, const GmDev &D, cudaStream_t st, const GmFork *fk = nullptr);   // a3 (if ctl->go)
int gm_nl_capacity_ok(const GmParams &P);
int gm_nl_smem_bytes(const GmParams &P);
cudaError_t gm_nl_prepare(const GmParams &P);      // opt-in shared-memory sizes of the kernels that stage windows
void gm_launch_bonds_from_master(const GmParams &P, const GmDev &D, cudaStream_t st);
void gm_launch_force(const GmParams &P, const GmDev &D, int mode, int parity, float kick, float kick_vt,
                     int lagged, cudaStream_t st);
void gm_launch_pack(const GmParams &P, const GmDev &D, int cur, const float *pos3, const float *vel3,
                    const int *type, const float *mass, cudaStream_t st);
void gm_launch_unpack(const GmParams &P, const GmDev &D, int cur, float *pos3, float *vel3, float *force3,
                      int lagged, cudaStream_t st);
void gm_launch_unpack_neighbors(const GmParams &P, const GmDev &D, int *nn_out, int *nl_out, long long stride,
                                int t0, int t1, cudaStream_t st);
void gm_launch_topo(const GmParams &P, const GmDev &D, int parity, cudaStream_t st);     // angle + dihedral forces -> D.ftopo
void gm_launch_thermo_reset(const GmDev &D, int parity, cudaStream_t st);
void gm_launch_set_ctl(const GmDev &D, unsigned long long step, int reset_all, int parity, cudaStream_t st);
void gm_launch_init_pad(const GmParams &P, const GmDev &D, cudaStream_t st);

// ---- device helpers ---------------------------------------------------------------------------------
#ifdef __CUDACC__
// Does the rebuild run now?  gate = 0: forced (unless the list is already current at this time level).
__device__ __forceinline__ bool gm_rebuild_off(const GmCtl *ctl, int gate, int parity)
{
    const unsigned long long m = ctl->step[parity];
    return ctl->rebuilt_at == m || (gate && ctl->need != m);
}

// Where the current time level lives: right after a rebuild (ctl->rebuilt_at == step) the sorted copies
// written by the sort are current; otherwise the ping-pong buffers of this parity.
struct Src {
    const float4 *__restrict__ pos;
    const float4 *__restrict__ vel;
    const float4 *__restrict__ vt;
    const int *__restrict__ tag;
};

__device__ __forceinline__ Src current_src(const GmDev &D, int parity, unsigned long long step)
{
    const bool fresh = D.ctl->rebuilt_at == step;
    Src s;
    s.pos = fresh ? D.ref : D.pos[parity];
    s.vel = fresh ? D.svel : D.vel;
    s.vt = fresh ? D.svt : D.vt[parity];
    s.tag = D.tag[D.ctl->n_rebuilds & 1ull];
    return s;
}

// Minimum image of a - b in a periodic box (PAPER.md: Alg. 2 line 6, L458).  A direct a - b is exact
// (Sterbenz) or rounded to half an ulp of the SMALL result when the pair does not cross the box; a
// pair across the boundary has |a - b| ~ L, where the subtraction would round at ulp(L) -- so those
// are taken relative to the two faces, (a -+ L/2) - (b +- L/2), which is again exact for any pair
// closer than L/3.
__device__ __forceinline__ float gm_min_image(float a, float b, float half)
{
    float d = a - b;
    if (d > half) d = (a - half) - (b + half);
    else if (d < -half) d = (a + half) - (b - half);
    return d;
}

// Minimum image for a bead whose own coordinate a is known: with hs = copysign(L/2, a) a partner across
// the boundary can only lie on the far side of that face (a >= 0: a - b > L/2 only), so one magnitude
// test selects between the plain difference and the face-relative one (a - hs) - (b + hs).
__device__ __forceinline__ float gm_min_image_signed(float a, float a_minus_hs, float hs, float b, float half)
{
    const float t = a - b;
    const float d2 = a_minus_hs - (b + hs);
    return fabsf(t) > half ? d2 : t;
}

// Streaming loads: not kept in L1, and (with an evict-first policy) first out of L2, so that the
// arrays that are re-read every step (positions, velocities, reference positions) stay L2-resident.
__device__ __forceinline__ uint64_t gm_policy_evict_first()
{
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

__device__ __forceinline__ int4 gm_ld_stream(const int4 *ptr, uint64_t pol)
{
    int4 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0, %1, %2, %3}, [%4], %5;"
        : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(ptr), "l"(pol));
    return v;
}

__device__ __forceinline__ float4 gm_ld_nol1(const float4 *ptr)
{
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(ptr));
    return v;
}

// ---- mbarrier + 1-D bulk copy (TMA engine: global -> shared without LSU wavefronts) ----------------------------
__device__ __forceinline__ void gm_mbar_init(uint32_t mbar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(mbar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void gm_mbar_expect_tx(uint32_t mbar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mbar), "r"(bytes) : "memory");
}

// bytes > 0, multiple of 16; dst and src 16-byte aligned
__device__ __forceinline__ void gm_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}

// try_wait with a suspend-time hint: the warp sleeps in hardware until the phase completes (or the hint, 1 ms, runs
// out) instead of burning issue slots in a polling loop.  Returns false if the phase did not complete within ~4 s
// (a byte-count mismatch would otherwise hang the GPU); the caller latches GM_DEV_ERR_WINDOW and carries on.
__device__ __forceinline__ bool gm_mbar_wait(uint32_t mbar, uint32_t parity)
{
    uint32_t ok;
    int polls = 0;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(mbar), "r"(parity), "r"(1000000u) : "memory");
    } while (!ok && ++polls < 4096);
    return ok != 0;
}

__device__ __forceinline__ float4 gm_lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

__device__ __forceinline__ float gm_wrap(float x, float half, float L)
{
    if (x >= half) x -= L;
    else if (x < -half) x += L;
    return x;
}

__device__ __forceinline__ int gm_cell_coord(float x, float half, float inv_w, int nc)
{
    int c = (int)((x + half) * inv_w);
    return min(max(c, 0), nc - 1);
}

__device__ __forceinline__ float gm_rcp(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the publication: ten rounds of
// two 32x32->64 multiplies with the key bumped by the Weyl constants between rounds.
__device__ __forceinline__ uint4 gm_philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// Symmetric uniform variate in (-1, 1) from the top 24 bits: 2u - 1 with u = (k + 1/2) 2^-24,
// i.e. (2k + 1 - 2^24) 2^-24 -- an odd integer below 2^24 in magnitude, exact in fp32.
__device__ __forceinline__ float gm_sym24(uint32_t x)
{
    int k = (int)(x >> 8);
    return (float)(2 * k + 1 - 16777216) * (1.0f / 16777216.0f);
}
#endif
