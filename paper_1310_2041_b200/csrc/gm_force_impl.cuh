// gm_force.cu -- a4..a9: pair + bond forces from the NL/BL tables, fused with the integrator and the
// displacement test.
//
//   a5  Lennard-Jones, Eq. (1); gather loop over row i of NL with minimum image and a
//       cutoff test as in Alg. 2, L458.  One thread owns bead i and sums all of its forces
//       ("one thread calculates and sums all non-bonded forces of a particle"), so a pair
//       is evaluated from both sides and no atomics are needed.
//   a6  DPD (Groot-Warren; reading c-3) with one Philox4x32-10 draw per pair keyed
//       (seed; min tag, max tag, step, 0) so that theta_ij = theta_ji without communication.
//   a7  bonds from BL, each bond evaluated from both ends; harmonic Eq. (7),
//       FENE (reading c-8).
//   a8  velocity-Verlet NVE / Langevin ("BD") / GW-VV in kick-drift form: the kernel
//       at time level m computes a(r^m), then u^{m} = u^{m-1} + kick a, r^{m+1} = r^m + dt u^m, where u
//       is the half-step velocity v^{m-1/2} (kick = dt), or the full-step v^m right after
//       gm_set_particles (kick = dt/2).  The force never leaves registers.
//   a4  displacement test |r^{m+1} - r_ref| > skin/2 -> ctl->need = m + 1.
//   a9  energies: fp32 terms, fp64 sums, fixed-order two-stage reduction.
//
// Memory plan of the step kernel: per bead it streams pos, vel, ref (48 B in), pos,
// vel (32 B out), NN (4 B), its NL quads (16 B per 4 list entries, 512-byte coalesced per warp) and its BL
// column; neighbor positions are 16-byte gathers that hit L1/L2 because storage order is cell order.
// The gather loop is software-pipelined: the index quads of the next batch and all position gathers
// of this batch are in flight before the first force term is evaluated.
#pragma once
#include <cooperative_groups.h>
#include <cooperative_groups/reduce.h>

#include "gm_internal.cuh"

#define FORCE_BLOCK 128          // = GM_TILE: a CTA of k_force / k_energy owns one tile
#ifndef STEP_BLOCK
#define STEP_BLOCK 32            // beads per CTA of the short-list step kernel: one warp
#endif
#ifndef STEP_MINB
#define STEP_MINB 32             // resident CTAs per SM of the short-list step kernel (<= 64 registers, 32 warps)
#endif
#ifndef WIDE_BLOCK
#define WIDE_BLOCK 128           // long lists and DPD: CTAs of 128 beads,
#define WIDE_MINB 7              //   7 resident per SM (72 registers)
#endif
#ifndef WIDE_NQ
#define WIDE_NQ 2                //   gather batches of two quads
#endif
#ifndef WINS_MINB
#define WINS_MINB 8              // short lists on window-staged systems: CTAs of GM_TILE beads, 8 resident per SM
#endif
static_assert(WIDE_BLOCK == GM_TILE && FORCE_BLOCK == GM_TILE, "a CTA of the window-staged force kernels owns one tile");
#ifndef SUB_BLOCK
#define SUB_BLOCK 128            // threads per CTA of the sub-warp step kernel
#endif
#ifndef GM_LJ_NQ
#define GM_LJ_NQ 1               // quads (of 4 list entries) per batch of the LJ gather loop
#endif

// a4: the list must be rebuilt before the forces of time level step + 1.  Inside a step graph the conditional node of the
// next timestep is switched on right here (GmDev::next_cond); otherwise the next gate kernel reads ctl->need.
__device__ __forceinline__ void raise_rebuild(const GmDev &D, unsigned long long step)
{
    D.ctl->need = step + 1;
    if (D.next_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)D.next_cond, 1u);
}

struct BeadForce {
    float fx, fy, fz;
    float pe_pair, pe_bond;   // this bead's half share
    float cnt;                // partners inside r_cut
};

// One list entry of the pair loop (Alg. 2: displacement, cutoff test, accumulate).  The LJ term is
// branch-free (out-of-range entries, and the far-away pad bead, select 0).
struct Own {                 // per-bead constants of the pair loop
    float4 p;                // position, type
    float ax, ay, az;        // p - hs          (MI path only)
    float hx, hy, hz;        // copysign(L/2, p)
    float4 vt;               // DPD: v~, tag
    int t;                   // type
};

template <int PAIR, bool NT1, bool ENERGY, bool MI>
__device__ __forceinline__ void pair_term(const GmParams &P, const Own &me, const float4 pj, const float4 vtj,
                                          const GmPair p0, uint32_t step, float &fx, float &fy, float &fz,
                                          float &pe, float &cnt)
{
    const float4 pi = me.p;
    const float4 vti = me.vt;
    const int ti = me.t;
    float dx, dy, dz;
    if (MI) {
        dx = gm_min_image_signed(pi.x, me.ax, me.hx, pj.x, P.half[0]);
        dy = gm_min_image_signed(pi.y, me.ay, me.hy, pj.y, P.half[1]);
        dz = gm_min_image_signed(pi.z, me.az, me.hz, pj.z, P.half[2]);
    } else {
        dx = pi.x - pj.x; dy = pi.y - pj.y; dz = pi.z - pj.z;
    }
    const float r2 = dx * dx + dy * dy + dz * dz;
    GmPair c = p0;
    if (!NT1) c = P.pair[ti * P.n_types + __float_as_int(pj.w)];
    if (PAIR == GM_PAIR_LJ) {
        // F_i = 24 eps / r^2 [2 (s/r)^12 - (s/r)^6] r_ij = r^-2 r^-6 (48 eps s^12 r^-6 - 24 eps s^6) r_ij
        const bool in = r2 < c.c0;
        const float r2i = gm_rcp(r2);
        const float r6i = r2i * r2i * r2i;
        const float fs = in ? r2i * r6i * (c.c1 * r6i - c.c2) : 0.0f;
        fx += fs * dx; fy += fs * dy; fz += fs * dz;
        if (ENERGY) {
            pe += in ? r6i * (c.c1 * (1.0f / 12.0f) * r6i - c.c2 * (1.0f / 6.0f)) - c.c3 : 0.0f;
            cnt += in ? 1.0f : 0.0f;
        }
    } else if (PAIR == GM_PAIR_HARMONIC) {
        // Eq. (2): U = alpha (1 - r/r_c)^2;  F_i = (2 alpha / r_c) (1 - r/r_c) r_ij / r
        const bool in = r2 < c.c0;
        const float ri = rsqrtf(fmaxf(r2, 1e-30f));          // coincident beads: r_ij = 0, no force (as the oracle)
        const float w = 1.0f - r2 * ri * c.c2;
        const float fs = in ? c.c1 * w * ri : 0.0f;
        fx += fs * dx; fy += fs * dy; fz += fs * dz;
        if (ENERGY) {
            pe += in ? c.c3 * w * w : 0.0f;
            cnt += in ? 1.0f : 0.0f;
        }
    } else if (PAIR == GM_PAIR_GAUSS) {
        // Eq. (3): U = eps exp(-r^2 / 2 sigma^2);  F_i = (eps / sigma^2) exp(-r^2 / 2 sigma^2) r_ij
        const bool in = r2 < c.c0;
        const float g = __expf(c.c2 * fminf(r2, c.c0));
        const float fs = in ? c.c1 * g : 0.0f;
        fx += fs * dx; fy += fs * dy; fz += fs * dz;
        if (ENERGY) {
            pe += in ? c.c4 * g - c.c3 : 0.0f;
            cnt += in ? 1.0f : 0.0f;
        }
    } else if (PAIR == GM_PAIR_TABLE) {
        // Algorithm 2 lines 8-12: point = int(dr^2 / interval); if point < Npoint: delta = dr^2 - point *
        // interval; Eq. (12) V = c0 + c1 d + c2 d^2 + c3 d^3; Eq. (11) F_i = -2 r_ij dV/dz.  The coefficients come
        // through the read-only path (L1/L2-resident: the paper's texture fetch of line 10).
        if (r2 < c.c0) {
            const int point = min((int)(r2 * c.c1), P.table_points - 1);
            const float4 k = __ldg(P.table + __float_as_int(c.c4) + point);
            const float d = r2 - (float)point * c.c2;
            const float fs = -2.0f * (k.y + d * (2.0f * k.z + 3.0f * k.w * d));
            fx += fs * dx; fy += fs * dy; fz += fs * dz;
            if (ENERGY) {
                pe += k.x + d * (k.y + d * (k.z + d * k.w));
                cnt += 1.0f;
            }
        }
    } else if (PAIR == GM_PAIR_DPD) {
        if (r2 < c.c0) {
            if (ENERGY) cnt += 1.0f;
            if (r2 >= 1e-12f) {
                // F_ij = [a w - gamma w^2 (e.v_ij) + sigma_R w theta / sqrt(dt)] e,  w = 1 - r/r_c
                const float ri = rsqrtf(r2);
                const float r = r2 * ri;
                const float w = 1.0f - r * c.c2;
                const float edv = (dx * (vti.x - vtj.x) + dy * (vti.y - vtj.y) + dz * (vti.z - vtj.z)) * ri;
                const uint32_t ta = (uint32_t)__float_as_int(vti.w), tb = (uint32_t)__float_as_int(vtj.w);
                const uint4 rn = gm_philox4x32_10(make_uint4(min(ta, tb), max(ta, tb), step, 0u),
                                                  make_uint2(P.seed_lo, P.seed_hi));
                const float theta = 1.7320508075688772f * gm_sym24(rn.x);
                const float fs = (c.c1 * w - P.gamma * w * w * edv + P.sigma_r_sqrt_inv_dt * w * theta) * ri;
                fx += fs * dx; fy += fs * dy; fz += fs * dz;
                if (ENERGY) pe += 0.5f * c.c1 * c.c3 * w * w;
            }
        }
    }
}

__device__ __forceinline__ int quad_get(const int4 &e, int u)
{
    return u == 0 ? e.x : (u == 1 ? e.y : (u == 2 ? e.z : e.w));
}

#define GM_PRE 4      // quads of a row loaded before NN is known (GmParams::minq = min(GM_PRE, capq))

__device__ __forceinline__ const int4 *nl_row(const GmParams &P, const GmDev &D, int i)
{
    return D.nl + ((size_t)(i >> 5) * P.capq) * 32 + (i & 31);
}

// The head of row i, issued together with the other streaming loads of the bead (always written by the build and
// padded, so it does not depend on NN).  The first two int4 are needed whatever the tile's format is (quads 0-1 of
// a 32-bit row, octs 0-1 of a 16-bit row); quads 2-3 of a 32-bit row follow once the format is known (at once on
// systems without tile windows).
template <bool WINS>
__device__ __forceinline__ void nl_preload(const GmParams &P, const int4 *__restrict__ t, uint64_t pol,
                                           int4 (&pre)[GM_PRE])
{
    const int4 pad = make_int4(P.n, P.n, P.n, P.n);
#pragma unroll
    for (int u = 0; u < GM_PRE; ++u)
        pre[u] = (u < P.minq && (u < 2 || !WINS || !P.use_win)) ? gm_ld_stream(t + u * 32, pol) : pad;
}

__device__ __forceinline__ void nl_preload_rest(const GmParams &P, const int4 *__restrict__ t, uint64_t pol,
                                                int4 (&pre)[GM_PRE])
{
#pragma unroll
    for (int u = 2; u < GM_PRE; ++u)
        if (u < P.minq) pre[u] = gm_ld_stream(t + u * 32, pol);
}

// Gather loop over row i of NL (Alg. 2), NQ quads (4 NQ list entries) per batch:
// first the preloaded quads, then a software-pipelined loop over the rest of the row.
template <int PAIR, bool NT1, bool ENERGY, bool MI, int NQL>
__device__ __forceinline__ void pair_loop(const GmParams &P, const Src &S, const int4 *__restrict__ t,
                                          uint64_t pol, const int4 (&pre)[GM_PRE], const int nn, const Own &me,
                                          unsigned long long step, BeadForce &o)
{
    constexpr int NQ = (PAIR == GM_PAIR_DPD) ? 1 : NQL;
    const int nq = (nn + 3) >> 2;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, cnt = 0.f;
    const GmPair p0 = P.pair[0];
    const int4 pad = make_int4(P.n, P.n, P.n, P.n);
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    int4 en[NQ];
#pragma unroll
    for (int u = 0; u < NQ; ++u) en[u] = (GM_PRE + u < nq) ? gm_ld_stream(t + (GM_PRE + u) * 32, pol) : pad;
#pragma unroll
    for (int b = 0; b < GM_PRE; b += NQ) {
        if (b < nq) {
            float4 pj[4 * NQ], vj[4 * NQ];
#pragma unroll
            for (int u = 0; u < 4 * NQ; ++u) pj[u] = __ldg(S.pos + quad_get(pre[b + (u >> 2)], u & 3));
            if (PAIR == GM_PAIR_DPD) {
#pragma unroll
                for (int u = 0; u < 4 * NQ; ++u) vj[u] = __ldg(S.vt + quad_get(pre[b + (u >> 2)], u & 3));
            }
#pragma unroll
            for (int u = 0; u < 4 * NQ; ++u)
                pair_term<PAIR, NT1, ENERGY, MI>(P, me, pj[u], PAIR == GM_PAIR_DPD ? vj[u] : zero4, p0,
                                                 (uint32_t)step, fx, fy, fz, pe, cnt);
        }
    }
    for (int q = GM_PRE; q < nq; q += NQ) {
        float4 pj[4 * NQ], vj[4 * NQ];
#pragma unroll
        for (int u = 0; u < 4 * NQ; ++u) pj[u] = __ldg(S.pos + quad_get(en[u >> 2], u & 3));
        if (PAIR == GM_PAIR_DPD) {
#pragma unroll
            for (int u = 0; u < 4 * NQ; ++u) vj[u] = __ldg(S.vt + quad_get(en[u >> 2], u & 3));
        }
#pragma unroll
        for (int u = 0; u < NQ; ++u) en[u] = (q + NQ + u < nq) ? gm_ld_stream(t + (q + NQ + u) * 32, pol) : pad;
#pragma unroll
        for (int u = 0; u < 4 * NQ; ++u)
            pair_term<PAIR, NT1, ENERGY, MI>(P, me, pj[u], PAIR == GM_PAIR_DPD ? vj[u] : zero4, p0,
                                             (uint32_t)step, fx, fy, fz, pe, cnt);
    }
    o.fx += fx; o.fy += fy; o.fz += fz;
    o.pe_pair = 0.5f * pe;
    o.cnt = cnt;
}

// ---- window-staged tiles (gm_nlist.cu "tile windows") -------------------------------------------------------------
// The positions a tile's NL rows refer to are a few contiguous ranges of the position array (the same ranges at every
// step until the next rebuild, because storage order is fixed in between).  The warp copies them into shared memory
// with cp.async.bulk (TMA engine: no LSU wavefronts, no registers, completion on an mbarrier) while its lanes request
// their own streams; the NL rows hold 16-bit window offsets, and every neighbor "gather" is an LDS.128.
// shared memory of one CTA (= one tile of GM_TILE beads) of a force kernel: the window (pad bead + win_cap positions)
// and its mbarrier
__host__ __device__ __forceinline__ int gm_win_bytes(const GmParams &P) { return P.use_win ? (P.win_cap + 2) * 16 : 0; }

struct Tile {
    uint32_t win;            // shared-memory byte address of window position 0 (the far-away pad bead)
    uint32_t mbar;
    int staged;              // 1: window-staged tile (16-bit rows), copies in flight; 0: 32-bit rows, gathers
    uint32_t parity;         // mbarrier phase to wait for
};

#define GM_WD_FIRST 12       // descriptor entries fetched before the range count is known (a tile inside one row has 9-10)

// Step 1, with the bead's other streaming loads: the header word of the tile's window descriptor (every thread; one
// broadcast load) and, in warp 0, this lane's range.
__device__ __forceinline__ int4 tile_desc(const GmParams &P, const GmDev &D, int tile)
{
    int4 d = make_int4(0, 0, 0, 0);
    if (!P.use_win) return d;
    const int4 *__restrict__ wd = D.wdesc + (size_t)tile * GM_WD_STRIDE;
    if (threadIdx.x < GM_WD_FIRST) d = __ldg(wd + threadIdx.x);
    d.w = __ldg(&wd[0].w);                   // entries past the tile's range count are stale: the header is entry 0's
    return d;
}

// Step 2 (all threads of the CTA that owns `tile`; one block-level barrier inside): thread 0 arms the mbarrier, the
// lanes of warp 0 issue one bulk copy per range.  smem: the CTA's window area (pad bead + win_cap positions) + mbarrier.
__device__ __forceinline__ Tile tile_stage(const GmParams &P, const GmDev &D, const Src &S, int tile, int4 d, char *smem,
                                           uint32_t parity, bool first)
{
    Tile T;
    T.win = (uint32_t)__cvta_generic_to_shared(smem);
    T.mbar = T.win + (uint32_t)(P.win_cap + 1) * 16u;
    T.staged = 0;
    T.parity = parity;
    if (!P.use_win) return T;
    const int hdr = d.w;                     // the same word in every entry of the descriptor
    if (first) {
        if (threadIdx.x == 0) {
            gm_mbar_init(T.mbar, 1);
            *reinterpret_cast<float4 *>(smem) = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        }
        __syncthreads();
    }
    if (!(hdr & 0x100)) return T;
    T.staged = 1;
    if (threadIdx.x >= 32) return T;
    const int lane = threadIdx.x;
    const int nr = hdr & 0xff;
    if (lane == 0) gm_mbar_expect_tx(T.mbar, (uint32_t)(hdr >> 16) * 16u);
    __syncwarp();
    const int4 *__restrict__ wd = D.wdesc + (size_t)tile * GM_WD_STRIDE;
    if (lane >= GM_WD_FIRST && lane < nr) d = __ldg(wd + lane);
    if (lane < nr) gm_bulk_g2s(T.win + (uint32_t)d.y * 16u, S.pos + d.x, (uint32_t)d.z * 16u, T.mbar);
    if (lane + 32 < nr) {
        const int4 e = __ldg(wd + lane + 32);
        gm_bulk_g2s(T.win + (uint32_t)e.y * 16u, S.pos + e.x, (uint32_t)e.z * 16u, T.mbar);
    }
    return T;
}

// Gather loop over row i of a window-staged tile: eight 16-bit window offsets per int4 ("oct"), the first GM_PRE_W
// octs preloaded; unused slots hold offset 0, the pad bead.
#define GM_PRE_W 2
template <int PAIR, bool NT1, bool ENERGY, bool MI>
__device__ __forceinline__ void pair_loop_win(const GmParams &P, const Tile &T, const int4 *__restrict__ t,
                                              uint64_t pol, const int4 (&pre)[GM_PRE], const int nn, const Own &me,
                                              BeadForce &o)
{
    const int no = (nn + 7) >> 3;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, cnt = 0.f;
    const GmPair p0 = P.pair[0];
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const int4 none = make_int4(0, 0, 0, 0);
    const uint32_t win = T.win;
    auto half_oct = [&](const uint32_t a, const uint32_t b) {
        float4 pj[4];
        pj[0] = gm_lds128(win + ((a & 0xffffu) << 4));
        pj[1] = gm_lds128(win + ((a >> 16) << 4));
        pj[2] = gm_lds128(win + ((b & 0xffffu) << 4));
        pj[3] = gm_lds128(win + ((b >> 16) << 4));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            pair_term<PAIR, NT1, ENERGY, MI>(P, me, pj[u], zero4, p0, 0u, fx, fy, fz, pe, cnt);
    };
    int4 en = (GM_PRE_W < no) ? gm_ld_stream(t + GM_PRE_W * 32, pol) : none;
#pragma unroll
    for (int b = 0; b < GM_PRE_W; ++b)
        if (b < no) {
            half_oct((uint32_t)pre[b].x, (uint32_t)pre[b].y);
            half_oct((uint32_t)pre[b].z, (uint32_t)pre[b].w);
        }
    for (int q = GM_PRE_W; q < no; ++q) {
        const int4 e = en;
        en = (q + 1 < no) ? gm_ld_stream(t + (q + 1) * 32, pol) : none;
        half_oct((uint32_t)e.x, (uint32_t)e.y);
        half_oct((uint32_t)e.z, (uint32_t)e.w);
    }
    o.fx += fx; o.fy += fy; o.fz += fz;
    o.pe_pair = 0.5f * pe;
    o.cnt = cnt;
}

// DPD gather loop with per-lane compaction (a6).  A list slot costs ~12 instructions to test against r_c but
// ~100 to evaluate (ten Philox rounds), and only ~37 % of the slots of a skin-padded list are inside r_c (C4):
// evaluated slot by slot, a warp pays the Philox rounds for a slot whenever ANY of its lanes is in range, i.e.
// always.  So pass 1 walks the row, tests r^2 and appends the in-range partner indices to a lane-private
// shared-memory column; pass 2 evaluates two compacted partners per trip -- the warp makes max-over-lanes
// (in-range count) / 2 trips instead of NN / 1.  The column holds GM_CPT_ROWS entries; it is drained early if
// it could overflow.  col: this thread's column, entries `stride` (= blockDim.x) ints apart.
#define GM_CPT_ROWS 32
// the compaction columns of a CTA of NT threads (DPD kernels only); entry k of thread t is gm_cpt[k * NT + t]
#define GM_CPT_DECL(PAIR, NT) __shared__ int gm_cpt[(PAIR) == GM_PAIR_DPD ? GM_CPT_ROWS * (NT) : 1]
template <bool NT1, bool ENERGY, bool MI>
__device__ __forceinline__ void pair_loop_dpd(const GmParams &P, const Src &S, const int4 *__restrict__ t,
                                              uint64_t pol, const int4 (&pre)[GM_PRE], const int nn, const Own &me,
                                              unsigned long long step, BeadForce &o, int *__restrict__ col)
{
    const int stride = (int)blockDim.x;
    const int nq = (nn + 3) >> 2;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, cnt = 0.f;
    const GmPair p0 = P.pair[0];
    int k = 0;
    auto scan_quad = [&](const int4 e) {
        float4 pj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) pj[u] = __ldg(S.pos + quad_get(e, u));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float dx, dy, dz;
            if (MI) {
                dx = gm_min_image_signed(me.p.x, me.ax, me.hx, pj[u].x, P.half[0]);
                dy = gm_min_image_signed(me.p.y, me.ay, me.hy, pj[u].y, P.half[1]);
                dz = gm_min_image_signed(me.p.z, me.az, me.hz, pj[u].z, P.half[2]);
            } else {
                dx = me.p.x - pj[u].x; dy = me.p.y - pj[u].y; dz = me.p.z - pj[u].z;
            }
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float cut = NT1 ? p0.c0 : P.pair[me.t * P.n_types + __float_as_int(pj[u].w)].c0;
            col[k * stride] = quad_get(e, u);       // kept only if in range
            k += (r2 < cut) ? 1 : 0;
        }
    };
    auto drain = [&]() {
        for (int c = 0; c < k; c += 2) {
            const int j0 = col[c * stride];
            const int j1 = (c + 1 < k) ? col[(c + 1) * stride] : P.n;     // the far-away pad bead
            const float4 q0 = __ldg(S.pos + j0), q1 = __ldg(S.pos + j1);
            const float4 w0 = __ldg(S.vt + j0), w1 = __ldg(S.vt + j1);
            pair_term<GM_PAIR_DPD, NT1, ENERGY, MI>(P, me, q0, w0, p0, (uint32_t)step, fx, fy, fz, pe, cnt);
            pair_term<GM_PAIR_DPD, NT1, ENERGY, MI>(P, me, q1, w1, p0, (uint32_t)step, fx, fy, fz, pe, cnt);
        }
        k = 0;
    };
    const int4 pad = make_int4(P.n, P.n, P.n, P.n);
    int4 en = (GM_PRE < nq) ? gm_ld_stream(t + GM_PRE * 32, pol) : pad;
#pragma unroll
    for (int b = 0; b < GM_PRE; ++b)
        if (b < nq) scan_quad(pre[b]);
    for (int q = GM_PRE; q < nq; ++q) {
        const int4 e = en;
        en = (q + 1 < nq) ? gm_ld_stream(t + (q + 1) * 32, pol) : pad;
        if (k > GM_CPT_ROWS - 4) drain();
        scan_quad(e);
    }
    drain();
    o.fx += fx; o.fy += fy; o.fz += fz;
    o.pe_pair = 0.5f * pe;
    o.cnt = cnt;
}

// Bond partners of bead i from column i of BL (Fig. 2), two at a time; -1 = no bond.
template <int BOND>
__device__ __forceinline__ void bond_head(const GmParams &P, const GmDev &D, int i, int (&be)[2])
{
    be[0] = be[1] = -1;
    if (BOND == GM_BOND_NONE) return;
#pragma unroll
    for (int u = 0; u < 2; ++u)
        if (u < P.max_bonds) be[u] = __ldg(D.bl + i + (size_t)u * P.ns);
}

// be: rows 0 and 1 of column i (bond_head, requested with the bead's other streams)
template <int BOND, bool ENERGY, bool WINS>
__device__ __forceinline__ void bond_loop(const GmParams &P, const GmDev &D, const Src &S, int i, const float4 pi,
                                          const int (&be)[2], const Tile &T, BeadForce &o)
{
    if (BOND == GM_BOND_NONE) return;
    float pe = 0.f;
    const size_t n = (size_t)P.ns;
    const int *__restrict__ bl = D.bl + i;
    for (int k = 0; k < P.max_bonds; k += 2) {
        int e[2];
        float4 pj[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) e[u] = (k == 0) ? be[u] : ((k + u < P.max_bonds) ? __ldg(bl + (size_t)(k + u) * n) : -1);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            // a partner inside the tile's window is a window offset (GM_BOND_LOCAL, set by k_nl_build), else a bead index
            if (e[u] < 0) pj[u] = pi;
            else if (WINS && (e[u] & GM_BOND_LOCAL)) pj[u] = gm_lds128(T.win + ((uint32_t)(e[u] & 0xffff) << 4));
            else pj[u] = __ldg(S.pos + (e[u] & GM_BOND_MASK));
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (e[u] < 0) continue;
            const int bt = (unsigned)e[u] >> GM_BOND_SHIFT;
            const float dx = gm_min_image(pi.x, pj[u].x, P.half[0]);
            const float dy = gm_min_image(pi.y, pj[u].y, P.half[1]);
            const float dz = gm_min_image(pi.z, pj[u].z, P.half[2]);
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float kb = P.bond_k[bt], r0 = P.bond_r0[bt];
            float fs;
            if (BOND == GM_BOND_FENE) {
                // U = -1/2 k R0^2 ln(1 - r^2/R0^2);  F_i = -k r_ij / (1 - r^2/R0^2)
                const float q = 1.0f - r2 * P.bond_c[bt];
                if (!(q > 0.0f)) { atomicOr(&D.ctl->err, GM_DEV_ERR_OVERSTRETCH); continue; }
                fs = -kb * gm_rcp(q);
                if (ENERGY) pe += -0.5f * kb * r0 * r0 * logf(q);
            } else if (BOND == GM_BOND_TABLE) {
                // Eqs. (11)-(12) in z = r^2: kb = 1 / interval, r0 = interval of this bond type
                const int point = (int)(r2 * kb);
                if (!(point < P.bond_table_points)) { atomicOr(&D.ctl->err, GM_DEV_ERR_OVERSTRETCH); continue; }
                const float4 c = __ldg(P.btable + bt * P.bond_table_points + point);
                const float d = r2 - (float)point * r0;
                fs = -2.0f * (c.y + d * (2.0f * c.z + 3.0f * c.w * d));
                if (ENERGY) pe += c.x + d * (c.y + d * (c.z + d * c.w));
            } else {
                // Eq. (7): U = k (r - r0)^2;  F_i = -2 k (1 - r0/r) r_ij
                if (r0 == 0.0f) {
                    fs = -2.0f * kb;
                    if (ENERGY) pe += kb * r2;
                } else {
                    const float r = sqrtf(r2);
                    fs = (r > 0.0f) ? -2.0f * kb * (1.0f - r0 / r) : 0.0f;
                    if (ENERGY) pe += kb * (r - r0) * (r - r0);
                }
            }
            o.fx += fs * dx; o.fy += fs * dy; o.fz += fs * dz;
        }
    }
    o.pe_bond = 0.5f * pe;
}

// Force on bead i at time level `step`, conservative + (DPD) dissipative/random.  vti: own v~ and tag.
// pre / nn: the preloaded head of row i and NN[i].
template <int PAIR, bool NT1, int BOND, bool ENERGY, int NQL, bool WINS>
__device__ __forceinline__ BeadForce bead_force(const GmParams &P, const GmDev &D, const Src &S, int i,
                                                const float4 pi, const float4 vti, const int4 *__restrict__ t,
                                                uint64_t pol, const int4 (&pre)[GM_PRE], const int nn,
                                                unsigned long long step, int *__restrict__ col, const Tile &T,
                                                const int (&be)[2], const bool valid)
{
    BeadForce o;
    o.fx = o.fy = o.fz = o.pe_pair = o.pe_bond = o.cnt = 0.f;
    if (WINS && T.staged && !gm_mbar_wait(T.mbar, T.parity)) atomicOr(&D.ctl->err, GM_DEV_ERR_WINDOW);   // the window has landed
    bond_loop<BOND, ENERGY, WINS>(P, D, S, i, pi, be, T, o);
    if (PAIR != GM_PAIR_NONE) {
        Own me;
        me.p = pi; me.vt = vti; me.t = __float_as_int(pi.w);
        me.hx = copysignf(P.half[0], pi.x); me.hy = copysignf(P.half[1], pi.y); me.hz = copysignf(P.half[2], pi.z);
        me.ax = pi.x - me.hx; me.ay = pi.y - me.hy; me.az = pi.z - me.hz;
        // A bead further than r_list + skin from every face cannot have a listed partner across the
        // boundary (both moved < skin/2 since the build): plain differences, no image test.  Decided per
        // warp so that a warp runs one of the two loops, not both.
        const float m = P.edge_margin;
        const bool interior = !valid || (fabsf(pi.x) < P.half[0] - m && fabsf(pi.y) < P.half[1] - m &&
                                         fabsf(pi.z) < P.half[2] - m);
        if (PAIR == GM_PAIR_DPD) {
            if (__all_sync(__activemask(), interior)) pair_loop_dpd<NT1, ENERGY, false>(P, S, t, pol, pre, nn, me, step, o, col);
            else pair_loop_dpd<NT1, ENERGY, true>(P, S, t, pol, pre, nn, me, step, o, col);
        } else if (WINS && T.staged) {
            if (__all_sync(__activemask(), interior)) pair_loop_win<PAIR, NT1, ENERGY, false>(P, T, t, pol, pre, nn, me, o);
            else pair_loop_win<PAIR, NT1, ENERGY, true>(P, T, t, pol, pre, nn, me, o);
        } else if (__all_sync(__activemask(), interior)) pair_loop<PAIR, NT1, ENERGY, false, NQL>(P, S, t, pol, pre, nn, me, step, o);
        else pair_loop<PAIR, NT1, ENERGY, true, NQL>(P, S, t, pol, pre, nn, me, step, o);
    }
    return o;
}

// a7: the angle + dihedral force of bead i (gm_topo.cu ran just before) and its share of their energy
__device__ __forceinline__ void topo_add(const GmParams &P, const GmDev &D, int i, BeadForce &f)
{
    if (P.max_angles + P.max_dihedrals > 0) {
        const float4 ft = D.ftopo[i];
        f.fx += ft.x; f.fy += ft.y; f.fz += ft.z;
        f.pe_bond += ft.w;
    }
}

// Acceleration the integrator uses: F/m, plus Langevin drag on the stored velocity and the per-bead
// noise of this time level (reading c-7): a = F/m - gamma u + sqrt(6 gamma kT / (dt m)) xi.
__device__ __forceinline__ float3 bead_accel(const GmParams &P, const Src &S, int i, const BeadForce &f,
                                             const float4 u, unsigned long long step)
{
    const float im = 1.0f / u.w;
    float3 a = make_float3(f.fx * im, f.fy * im, f.fz * im);
    if (P.integrator == GM_LANGEVIN) {
        const uint4 rn = gm_philox4x32_10(make_uint4((uint32_t)S.tag[i], 0u, (uint32_t)step, 1u),
                                          make_uint2(P.seed_lo, P.seed_hi));
        const float amp = sqrtf(P.lang_amp2 * im);
        a.x += -P.gamma * u.x + amp * gm_sym24(rn.x);
        a.y += -P.gamma * u.y + amp * gm_sym24(rn.y);
        a.z += -P.gamma * u.z + amp * gm_sym24(rn.z);
    }
    return a;
}

// ---- NVT thermostats in leapfrog form (readings c-28..c-30) ----------------------------
// u' = sa u + sb kick a with (sa, sb) from the temperature T_half of the half-step velocities the previous step wrote:
//   Berendsen:   lambda = sqrt(1 + dt gamma (kT / T_half - 1)), sa = sb = lambda
//   Nose-Hoover: xi += dt gamma^2 (T_half / kT - 1), h = dt xi / 2, sa = (1 - h) / (1 + h), sb = 1 / (1 + h)
// Every thread derives the same pair from the control block (a few flops on uniform values); thread 0 of block 0 stores
// the new xi and clears the accumulator of the step after next (three-slot rotation: no slot is read and written in one
// launch).  The first kick after a (re)start runs without the thermostat.
struct Thermo { float sa, sb; bool on; };

__device__ __forceinline__ Thermo thermo_begin(const GmParams &P, const GmDev &D, unsigned long long step, float kick)
{
    Thermo T;
    T.sa = 1.0f; T.sb = 1.0f; T.on = false;
    if (P.integrator != GM_NVT_NOSE_HOOVER && P.integrator != GM_NVT_BERENDSEN) return T;
    T.on = true;
    GmCtl *c = D.ctl;
    const int r = (int)(step % 3ull), w = (int)((step + 1ull) % 3ull), z = (int)((step + 2ull) % 3ull);
    const bool active = step > c->thermo_start;
    double xi = c->xi[r];
    if (active) {
        const double dof = P.n > 1 ? 3.0 * P.n - 3.0 : 3.0;
        const double t_half = c->ke2[r] / dof;
        if (P.integrator == GM_NVT_BERENDSEN) {
            const double lam = sqrt(1.0 + (double)P.dt * P.gamma * ((double)P.kT / t_half - 1.0));
            T.sa = T.sb = (float)lam;
        } else {
            xi += (double)P.dt * P.gamma * P.gamma * (t_half / (double)P.kT - 1.0);
            const double h = 0.5 * (double)P.dt * xi;
            T.sa = (float)((1.0 - h) / (1.0 + h)); T.sb = (float)(1.0 / (1.0 + h));
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { c->xi[w] = xi; c->ke2[z] = 0.0; }
    (void)kick;
    return T;
}

// sum of m u'^2 over the lanes that hold a bead -> the accumulator the next step reads (one double atomic per warp)
__device__ __forceinline__ void thermo_accumulate(const GmDev &D, unsigned long long step, float m_u2)
{
    namespace cg = cooperative_groups;
    const cg::coalesced_group g = cg::coalesced_threads();
    const float sum = cg::reduce(g, m_u2, cg::plus<float>());
    if (g.thread_rank() == 0) atomicAdd(&D.ctl->ke2[(int)((step + 1ull) % 3ull)], (double)sum);
}

// Andersen thermostat (c-29): the bead collides with the heat bath in this kick iff the top 24 bits of Philox(tag, 0,
// step, 3) word 0 are below floor(nu dt 2^24); its new velocity is sqrt(kT / m) times three Box-Muller normals from the
// words of Philox(tag, 0, step, 2).
__device__ __forceinline__ void andersen_collide(const GmParams &P, const Src &S, int i, unsigned long long step, float mass,
                                                 float &ux, float &uy, float &uz)
{
    const uint32_t tag = (uint32_t)S.tag[i];
    const uint2 key = make_uint2(P.seed_lo, P.seed_hi);
    const uint4 d = gm_philox4x32_10(make_uint4(tag, 0u, (uint32_t)step, 3u), key);
    const float thr = floorf(P.gamma * P.dt * 16777216.0f);
    if ((float)(d.x >> 8) < thr) {
        const uint4 w = gm_philox4x32_10(make_uint4(tag, 0u, (uint32_t)step, 2u), key);
        const float u0 = ((float)(w.x >> 8) + 0.5f) * (1.0f / 16777216.0f), u1 = ((float)(w.y >> 8) + 0.5f) * (1.0f / 16777216.0f);
        const float u2 = ((float)(w.z >> 8) + 0.5f) * (1.0f / 16777216.0f), u3 = ((float)(w.w >> 8) + 0.5f) * (1.0f / 16777216.0f);
        const float r0 = sqrtf(-2.0f * logf(u0)), r2 = sqrtf(-2.0f * logf(u2));
        float s1, c1, s3, c3;
        sincospif(2.0f * u1, &s1, &c1);
        sincospif(2.0f * u3, &s3, &c3);
        const float a = sqrtf(P.kT / mass);
        ux = a * r0 * c1; uy = a * r0 * s1; uz = a * r2 * c3;
    }
}

// ---- the per-step work of one bead (MODE_STEP) / its materialised force (MODE_FORCES) -----------------
// Called by all threads of the CTA (window staging is a block-collective step); threads past the last bead
// (valid = false) work on the pad slots (far away, NN = 0, no bonds) and store nothing.
template <int PAIR, bool NT1, int BOND, int MODE, int NQL, bool WINS>
__device__ __forceinline__ void bead_step(const GmParams &P, const GmDev &D, const Src &S, const int i, const bool valid,
                                          const unsigned long long step, const int parity, const float kick,
                                          const float kick_vt, int *__restrict__ col, char *wsm)
{
    // every stream of this bead is requested before anything is used; the tile's window descriptor first (the bulk
    // copies wait for it)
    int4 wd = make_int4(0, 0, 0, 0);
    if (WINS) wd = tile_desc(P, D, blockIdx.x);
    const uint64_t pol = gm_policy_evict_first();
    const int4 *__restrict__ t = nl_row(P, D, i);
    int4 pre[GM_PRE];
    if (PAIR != GM_PAIR_NONE) nl_preload<WINS>(P, t, pol, pre);
    const float4 pi = S.pos[i];
    const int nn = (PAIR != GM_PAIR_NONE) ? D.nn[i] : 0;
    const float4 u = gm_ld_nol1(S.vel + i);
    float4 rf = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == GM_MODE_STEP) rf = gm_ld_nol1(D.ref + i);
    float4 vti = make_float4(0.f, 0.f, 0.f, 0.f);
    if (PAIR == GM_PAIR_DPD) vti = S.vt[i];
    int be[2];
    bond_head<BOND>(P, D, i, be);
    // the window's ranges are known: the copies go out while the streams above are in flight
    Tile T;
    T.win = 0; T.mbar = 0; T.staged = 0; T.parity = 0;
    if (WINS) T = tile_stage(P, D, S, blockIdx.x, wd, wsm, 0u, true);
    if (WINS && PAIR != GM_PAIR_NONE && P.use_win && !T.staged) nl_preload_rest(P, t, pol, pre);
    BeadForce f = bead_force<PAIR, NT1, BOND, MODE == GM_MODE_FORCES, NQL, WINS>(P, D, S, i, pi, vti, t, pol, pre, nn, step, col, T, be, valid);
    if (!valid) return;
    topo_add(P, D, i, f);
    const float3 a = bead_accel(P, S, i, f, u, step);
    if (MODE == GM_MODE_FORCES) {
        D.frc[i] = make_float4(a.x * u.w, a.y * u.w, a.z * u.w, f.pe_pair + f.pe_bond);
        return;
    }
    // a8: kick, drift, wrap
    if (PAIR == GM_PAIR_DPD)
        D.vt[parity ^ 1][i] = make_float4(u.x + kick_vt * a.x, u.y + kick_vt * a.y, u.z + kick_vt * a.z, vti.w);
    float ux = u.x + kick * a.x, uy = u.y + kick * a.y, uz = u.z + kick * a.z;
    if (P.integrator >= GM_NVT_NOSE_HOOVER) {
        const Thermo th = thermo_begin(P, D, step, kick);
        if (th.on) {
            ux = th.sa * u.x + th.sb * kick * a.x; uy = th.sa * u.y + th.sb * kick * a.y; uz = th.sa * u.z + th.sb * kick * a.z;
            thermo_accumulate(D, step, u.w * (ux * ux + uy * uy + uz * uz));
        } else {
            andersen_collide(P, S, i, step, u.w, ux, uy, uz);
        }
    }
    D.vel[i] = make_float4(ux, uy, uz, u.w);
    // positions are NOT wrapped here: between two rebuilds a bead may sit up to skin/2 outside the box (the
    // sort wraps it back), so that every listed pair keeps the periodic image it had at the build
    const float x = pi.x + P.dt * ux, y = pi.y + P.dt * uy, z = pi.z + P.dt * uz;
    D.pos[parity ^ 1][i] = make_float4(x, y, z, pi.w);
    // a4: displacement since the last NL build (ref holds the wrapped position the bead had then)
    const float dx = x - rf.x, dy = y - rf.y, dz = z - rf.z;
    if (!(dx * dx + dy * dy + dz * dz <= P.half_skin2)) raise_rebuild(D, step);
}

// gm_compute_forces: one block per 128 beads.
template <int PAIR, bool NT1, int BOND>
__global__ void __launch_bounds__(FORCE_BLOCK)
k_force(const __grid_constant__ GmParams P, GmDev D, int parity)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    GM_CPT_DECL(PAIR, FORCE_BLOCK);
    extern __shared__ __align__(16) char gm_win_smem[];
    bead_step<PAIR, NT1, BOND, GM_MODE_FORCES, GM_LJ_NQ, PAIR != GM_PAIR_DPD && PAIR != GM_PAIR_NONE>(P, D, S, i, i < P.n, step, parity, 0.f, 0.f, gm_cpt + threadIdx.x,
                                                        gm_win_smem);
}

// The step kernel (a4..a8).  A CTA owns BLOCK consecutive beads: storage order is cell order along the curve,
// so neighboring CTAs work side by side on a few adjacent (y, z) rows of cells and share the neighbor positions
// they gather through the SM's L1.  Two shapes, chosen by the mean list length (GmParams::step_wide):
//   short lists (C1/C3, n_l ~ 13): CTAs of ONE warp, 32 resident per SM (<= 64 registers), gather batches of one
//     quad -- a warp's slot is free the moment it is done instead of waiting for the slowest of four
//     (measured on C3: 48.2 -> 42.8 us);
//   long lists (C2/C5, n_l ~ 90) and DPD: CTAs of 128, 7 resident per SM, batches of two quads.
template <int PAIR, bool NT1, int BOND, int BLOCK, int MINB, int NQL, bool WINS>
__global__ void __launch_bounds__(BLOCK, MINB)
k_step(const __grid_constant__ GmParams P, GmDev D, int parity, float kick, float kick_vt)
{
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        D.ctl->step[parity ^ 1] = step + 1;
        // a2: at most sfc_period steps between two sorts
        if (P.sfc_period > 0 && D.ctl->rebuilt_at != GM_NEVER &&
            step + 1 - D.ctl->rebuilt_at >= (unsigned long long)P.sfc_period)
            raise_rebuild(D, step);
    }
    const int i = blockIdx.x * BLOCK + threadIdx.x;
    GM_CPT_DECL(PAIR, BLOCK);
    extern __shared__ __align__(16) char gm_win_smem[];
    // window-staged systems run CTAs of GM_TILE beads (one tile each); every thread takes part in the staging
    if (WINS || i < P.n)
        bead_step<PAIR, NT1, BOND, GM_MODE_STEP, NQL, WINS>(P, D, S, i, i < P.n, step, parity, kick, kick_vt, gm_cpt + threadIdx.x,
                                                            gm_win_smem);
}

// The step kernel for LONG neighbor lists (n_l of 80-100: LJ with r_c = 2.5, configs C2/C5): SUBW lanes share
// one bead.  Lane `sub` of the group walks quads sub, sub + SUBW, ... of the bead's NL row (two quads, eight
// gathers, in flight per iteration), the partial forces are summed with xor-shuffles inside the group, and
// lane 0 of the group adds the bonds and integrates.  With one thread per bead a 64,000-bead system is
// 2,000 warps -- half a wave on 148 SMs, each thread walking ~90 dependent gathers; with 8 lanes per bead it is
// 16,000 warps of ~11 gathers per lane.  Still no atomics: a bead's force is owned by one group.
template <int PAIR, bool NT1, int BOND, int SUBW>
__global__ void __launch_bounds__(SUB_BLOCK)
k_step_sub(const __grid_constant__ GmParams P, GmDev D, int parity, float kick, float kick_vt)
{
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        D.ctl->step[parity ^ 1] = step + 1;
        if (P.sfc_period > 0 && D.ctl->rebuilt_at != GM_NEVER &&
            step + 1 - D.ctl->rebuilt_at >= (unsigned long long)P.sfc_period)
            raise_rebuild(D, step);
    }
    const long long gt = (long long)blockIdx.x * SUB_BLOCK + threadIdx.x;
    const int i = (int)(gt / SUBW), sub = (int)(gt % SUBW);
    const bool valid = i < P.n;
    const int ic = valid ? i : 0;                       // idle groups shadow bead 0 and write nothing
    const uint64_t pol = gm_policy_evict_first();
    const int4 *__restrict__ t = nl_row(P, D, ic);
    const float4 pi = S.pos[ic];
    const int nq = valid ? (D.nn[ic] + 3) >> 2 : 0;
    float4 vti = make_float4(0.f, 0.f, 0.f, 0.f);
    if (PAIR == GM_PAIR_DPD) vti = S.vt[ic];
    Own me;
    me.p = pi; me.vt = vti; me.t = __float_as_int(pi.w);
    me.hx = copysignf(P.half[0], pi.x); me.hy = copysignf(P.half[1], pi.y); me.hz = copysignf(P.half[2], pi.z);
    me.ax = pi.x - me.hx; me.ay = pi.y - me.hy; me.az = pi.z - me.hz;
    const GmPair p0 = P.pair[0];
    const int4 pad = make_int4(P.n, P.n, P.n, P.n);
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, cnt = 0.f;
    if (PAIR != GM_PAIR_NONE) {
        int4 ea = (sub < nq) ? gm_ld_stream(t + sub * 32, pol) : pad;
        int4 eb = (sub + SUBW < nq) ? gm_ld_stream(t + (sub + SUBW) * 32, pol) : pad;
        for (int q = sub; q < nq; q += 2 * SUBW) {
            float4 pj[8], vj[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) pj[u] = __ldg(S.pos + quad_get(u < 4 ? ea : eb, u & 3));
            if (PAIR == GM_PAIR_DPD) {
#pragma unroll
                for (int u = 0; u < 8; ++u) vj[u] = __ldg(S.vt + quad_get(u < 4 ? ea : eb, u & 3));
            }
            ea = (q + 2 * SUBW < nq) ? gm_ld_stream(t + (q + 2 * SUBW) * 32, pol) : pad;
            eb = (q + 3 * SUBW < nq) ? gm_ld_stream(t + (q + 3 * SUBW) * 32, pol) : pad;
#pragma unroll
            for (int u = 0; u < 8; ++u)
                pair_term<PAIR, NT1, false, true>(P, me, pj[u], PAIR == GM_PAIR_DPD ? vj[u] : zero4, p0,
                                                  (uint32_t)step, fx, fy, fz, pe, cnt);
        }
    }
#pragma unroll
    for (int o = SUBW >> 1; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
    }
    if (!valid || sub != 0) return;
    BeadForce f;
    f.fx = 0.f; f.fy = 0.f; f.fz = 0.f; f.pe_pair = 0.f; f.pe_bond = 0.f; f.cnt = 0.f;
    Tile T;
    T.win = 0; T.mbar = 0; T.staged = 0; T.parity = 0;     // GM_FLAG_STEP_SUBWARP systems keep 32-bit rows everywhere
    int be[2];
    bond_head<BOND>(P, D, i, be);
    bond_loop<BOND, false, false>(P, D, S, i, pi, be, T, f);
    f.fx += fx; f.fy += fy; f.fz += fz;
    const float4 u = gm_ld_nol1(S.vel + i);
    const float4 rf = gm_ld_nol1(D.ref + i);
    const float3 a = bead_accel(P, S, i, f, u, step);
    if (PAIR == GM_PAIR_DPD)
        D.vt[parity ^ 1][i] = make_float4(u.x + kick_vt * a.x, u.y + kick_vt * a.y, u.z + kick_vt * a.z, vti.w);
    const float ux = u.x + kick * a.x, uy = u.y + kick * a.y, uz = u.z + kick * a.z;
    D.vel[i] = make_float4(ux, uy, uz, u.w);
    const float x = pi.x + P.dt * ux, y = pi.y + P.dt * uy, z = pi.z + P.dt * uz;
    D.pos[parity ^ 1][i] = make_float4(x, y, z, pi.w);
    const float dx = x - rf.x, dy = y - rf.y, dz = z - rf.z;
    if (!(dx * dx + dy * dy + dz * dz <= P.half_skin2)) raise_rebuild(D, step);
}

// ---- a9 energies: grid-stride, fp64 accumulation, per-block partials in fixed order ----------------
template <int PAIR, bool NT1, int BOND>
__global__ void __launch_bounds__(FORCE_BLOCK)
k_energy(const __grid_constant__ GmParams P, GmDev D, int parity, int lagged)
{
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    GM_CPT_DECL(PAIR, FORCE_BLOCK);
    double acc[7] = { 0, 0, 0, 0, 0, 0, 0 };   // ke, pe_pair, pe_bond, px, py, pz, pairs
    extern __shared__ __align__(16) char gm_win_smem[];
    char *wsm = gm_win_smem;
    uint32_t phase = 0;
    bool armed = false;                                     // the CTA's mbarrier is initialised
    // a CTA takes tiles blockIdx, blockIdx + gridDim, ...: the trip count is CTA-uniform (window staging is a
    // block-collective step)
    for (int base = blockIdx.x * FORCE_BLOCK; base < P.n; base += gridDim.x * FORCE_BLOCK) {
        const int i = base + threadIdx.x;
        __syncthreads();                                    // every thread is done with the previous window
        const bool valid = i < P.n;
        const uint64_t pol = gm_policy_evict_first();
        const int4 *__restrict__ t = nl_row(P, D, i);
        int4 pre[GM_PRE];
        if (PAIR != GM_PAIR_NONE) nl_preload<true>(P, t, pol, pre);
        const float4 pi = S.pos[i];
        const int nn = (PAIR != GM_PAIR_NONE) ? D.nn[i] : 0;
        float4 vti = make_float4(0.f, 0.f, 0.f, 0.f);
        if (PAIR == GM_PAIR_DPD) vti = S.vt[i];
        int be[2];
        bond_head<BOND>(P, D, i, be);
        const Tile T = tile_stage(P, D, S, base / GM_TILE, tile_desc(P, D, base / GM_TILE), wsm, phase, !armed);
        armed = true;
        if (T.staged) phase ^= 1u;                          // the mbarrier completes one phase per staged tile
        if (PAIR != GM_PAIR_NONE && P.use_win && !T.staged) nl_preload_rest(P, t, pol, pre);
        BeadForce f = bead_force<PAIR, NT1, BOND, true, GM_LJ_NQ, PAIR != GM_PAIR_DPD && PAIR != GM_PAIR_NONE>(P, D, S, i, pi, vti, t, pol, pre, nn, step, gm_cpt + threadIdx.x, T, be, valid);
        if (!valid) continue;
        topo_add(P, D, i, f);
        const float4 u = S.vel[i];
        float vx = u.x, vy = u.y, vz = u.z;
        if (lagged) {   // complete the half-step velocity: v^m = u^{m-1} + dt/2 a^m
            const float3 a = bead_accel(P, S, i, f, u, step);
            vx += 0.5f * P.dt * a.x; vy += 0.5f * P.dt * a.y; vz += 0.5f * P.dt * a.z;
        }
        acc[0] += 0.5 * (double)u.w * ((double)vx * vx + (double)vy * vy + (double)vz * vz);
        acc[1] += (double)f.pe_pair;
        acc[2] += (double)f.pe_bond;
        acc[3] += (double)u.w * vx; acc[4] += (double)u.w * vy; acc[5] += (double)u.w * vz;
        acc[6] += 0.5 * (double)f.cnt;
    }
    __shared__ double sh[FORCE_BLOCK / 32][7];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 7; ++q) {
        double v = acc[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) sh[wid][q] = v;
    }
    __syncthreads();
    if (threadIdx.x < 7) {
        double v = 0.0;
        for (int w = 0; w < FORCE_BLOCK / 32; ++w) v += sh[w][threadIdx.x];
        D.esum[(size_t)blockIdx.x * 8 + threadIdx.x] = v;
    }
}

// Second stage: warp q sums quantity q over the block partials -- lane l takes blocks l, l + 32, ... in
// order, then a fixed xor-shuffle tree: the order of the additions depends on nothing but n_blocks.
static __global__ void __launch_bounds__(7 * 32) k_energy_final(GmDev D, int n_blocks)
{
    const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double v = 0.0;
    for (int b = lane; b < n_blocks; b += 32) v += D.esum[(size_t)b * 8 + q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) D.esum[(size_t)GM_ESUM_BLOCKS * 8 + q] = v;
}

// Kernels that stage tile windows take their shared memory at launch; above 48 KB per CTA that needs an opt-in, set
// once per instantiation and size.
template <typename K>
static void allow_smem(K kernel, int bytes)
{
    if (bytes > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <int PAIR, bool NT1, int BOND>
static void launch_force_t(const GmParams &P, const GmDev &D, int mode, int parity, float kick, float kick_vt,
                           int lagged, cudaStream_t st)
{
    int nb = (P.n + FORCE_BLOCK - 1) / FORCE_BLOCK;
    const int wb = gm_win_bytes(P);
    if (mode == GM_MODE_STEP) {
        if (P.step_subw == 8 && (PAIR == GM_PAIR_LJ || PAIR == GM_PAIR_DPD)) {
            if constexpr (PAIR == GM_PAIR_LJ || PAIR == GM_PAIR_DPD) {
                const long long nt = (long long)P.n * 8;
                k_step_sub<PAIR, NT1, BOND, 8><<<(unsigned)((nt + SUB_BLOCK - 1) / SUB_BLOCK), SUB_BLOCK, 0, st>>>(
                    P, D, parity, kick, kick_vt);
            }
        } else if (P.step_wide || PAIR == GM_PAIR_DPD) {
            constexpr bool CANWIN = PAIR != GM_PAIR_DPD && PAIR != GM_PAIR_NONE;
            if (CANWIN && P.use_win) {
                if constexpr (CANWIN) {
                    allow_smem(k_step<PAIR, NT1, BOND, WIDE_BLOCK, WIDE_MINB, WIDE_NQ, true>, wb);
                    k_step<PAIR, NT1, BOND, WIDE_BLOCK, WIDE_MINB, WIDE_NQ, true><<<(P.n + WIDE_BLOCK - 1) / WIDE_BLOCK, WIDE_BLOCK, wb, st>>>(
                        P, D, parity, kick, kick_vt);
                }
            } else
                k_step<PAIR, NT1, BOND, WIDE_BLOCK, WIDE_MINB, WIDE_NQ, false><<<(P.n + WIDE_BLOCK - 1) / WIDE_BLOCK, WIDE_BLOCK, 0, st>>>(
                    P, D, parity, kick, kick_vt);
        } else if constexpr (PAIR != GM_PAIR_DPD) {
            if (P.use_win && PAIR != GM_PAIR_NONE) {        // short lists, window-staged: CTAs of one tile, 8 resident per SM (<= 64 registers)
                if constexpr (PAIR != GM_PAIR_NONE) {
                    allow_smem(k_step<PAIR, NT1, BOND, GM_TILE, WINS_MINB, GM_LJ_NQ, true>, wb);
                    k_step<PAIR, NT1, BOND, GM_TILE, WINS_MINB, GM_LJ_NQ, true><<<(P.n + GM_TILE - 1) / GM_TILE, GM_TILE, wb, st>>>(
                        P, D, parity, kick, kick_vt);
                }
            } else
                k_step<PAIR, NT1, BOND, STEP_BLOCK, STEP_MINB, GM_LJ_NQ, false><<<(P.n + STEP_BLOCK - 1) / STEP_BLOCK, STEP_BLOCK, 0, st>>>(
                    P, D, parity, kick, kick_vt);
        }
    } else if (mode == GM_MODE_FORCES) {
        allow_smem(k_force<PAIR, NT1, BOND>, wb);
        k_force<PAIR, NT1, BOND><<<nb, FORCE_BLOCK, wb, st>>>(P, D, parity);
    } else {
        int g = nb < GM_ESUM_BLOCKS ? nb : GM_ESUM_BLOCKS;
        allow_smem(k_energy<PAIR, NT1, BOND>, wb);
        k_energy<PAIR, NT1, BOND><<<g, FORCE_BLOCK, wb, st>>>(P, D, parity, lagged);
        k_energy_final<<<1, 7 * 32, 0, st>>>(D, g);
    }
}

template <int PAIR, bool NT1>
static void launch_force_b(const GmParams &P, const GmDev &D, int mode, int parity, float kick, float kick_vt,
                           int lagged, cudaStream_t st)
{
    const int bond = (P.max_bonds > 0) ? P.bond_style : GM_BOND_NONE;
    if (bond == GM_BOND_FENE) launch_force_t<PAIR, NT1, GM_BOND_FENE>(P, D, mode, parity, kick, kick_vt, lagged, st);
    else if (bond == GM_BOND_TABLE) launch_force_t<PAIR, NT1, GM_BOND_TABLE>(P, D, mode, parity, kick, kick_vt, lagged, st);
    else if (bond == GM_BOND_HARMONIC)
        launch_force_t<PAIR, NT1, GM_BOND_HARMONIC>(P, D, mode, parity, kick, kick_vt, lagged, st);
    else launch_force_t<PAIR, NT1, GM_BOND_NONE>(P, D, mode, parity, kick, kick_vt, lagged, st);
}

// One translation unit per pair style (they compile in parallel): gm_force.cu (none, LJ), gm_force_dpd.cu,
// gm_force_soft.cu (harmonic and Gaussian repulsion), gm_force_table.cu.
#define GM_DEFINE_PAIR_LAUNCH(NAME, PAIR)                                                                            \
    void NAME(const GmParams &P, const GmDev &D, int mode, int parity, float kick, float kick_vt, int lagged,       \
              cudaStream_t st)                                                                                      \
    {                                                                                                               \
        if (P.n_types == 1) launch_force_b<PAIR, true>(P, D, mode, parity, kick, kick_vt, lagged, st);             \
        else launch_force_b<PAIR, false>(P, D, mode, parity, kick, kick_vt, lagged, st);                            \
    }
