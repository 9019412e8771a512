// gm_nlist.cu -- a3: skin-padded FULL Verlet neighbor list from the 27 surrounding cells
// ("searching neighboring particles from the surrounding 27 cells (including the cell
// that the target particle resides in)", all neighbors "within a distance that is the sum of the
// cutoff ... r_cut, and the buffer distance, r_buffer"; table form NL[k*Np + i], NN[i]: L51, Fig. 1).
//
// Runs right after the sort of gm_sort.cu, so bead index == slot in the cell-sorted array `ref`: one
// thread per bead, a warp owns 32 consecutive beads (a few adjacent cells of one x row), its lanes
// read the same or adjacent candidates at every iteration and run nearly equal trip counts.  Cells run
// along x inside a row, so the x-adjacent cells of one (y, z) row are one contiguous run of
// ref[]: nine runs per bead instead of 27 cells (more where the row wraps around the box).  Cells are
// r_list wide in y and z but r_list / sx in x (GmParams::sx): a run then spans (2 + 1/sx) r_list instead
// of 3 r_list -- fewer candidates per bead at no extra runs.
//
// Hits are staged in a small lane-private shared-memory ring (NL_STAGE entries per lane, column l of
// [NL_STAGE][32]: conflict-free and private to the lane, so no synchronisation); candidates are scanned
// four at a time, and after each four every lane that holds 16 or more staged entries writes four whole
// int4 quads of its NL row (gm_internal.cuh: entries 4q..4q+3 of a bead are one int4; the 32 int4 of a
// quad are contiguous, so a warp stores 512-byte lines).  The ring keeps shared memory at 20 KB per CTA
// whatever the row capacity (window systems add their set-up scratch and, for dense cells, the union scan's buffers),
// which leaves the rest of the SM's 228 KB to L1 for the candidate loads.
#include "gm_internal.cuh"

#ifndef NL_MINB_WIN
#define NL_MINB_WIN 6          // resident CTAs per SM the window-system build is compiled for (77 registers, no spills; 8 -> 64 registers with spills measured 1 % slower on C2 / C5)
#endif
#define NL_STAGE 32          // ring entries per lane of the kernels that scan 8 candidates per trip (power of two)
// Ring entries per lane by trip width: a lane flushes half a ring when that much is staged, so the ring must hold
// (half - 1) + TRIP entries.  A ring of 16 would do for TRIP = 4 (8 KB per CTA instead of 16), but it flushes twice as
// often: measured on C3 70.35 against 69.87 us per timestep with the ring of 32 (same box) -- 32 for both.
#ifndef NL_STAGE4
#define NL_STAGE4 32
#endif
#define NL_STAGE_OF(TRIP) ((TRIP) == 4 ? NL_STAGE4 : 32)
#ifndef NL_COOP
#define NL_COOP 1            // dense cells: warps of one piece scan the union of their lanes' runs together (nl_scan_warp)
#endif
#ifndef NL_WARPS
#define NL_WARPS 4
#endif
static_assert(NL_WARPS * 32 == GM_TILE, "one CTA of k_nl_build owns one tile");

// ---- tile windows -----------------------------------------------------------------------------------------------
// A tile = the GM_TILE = 128 consecutive beads of one CTA.  Storage order is cell order, so the candidates of ALL beads of a
// tile lie in a few contiguous ranges of the position array: for each of the 9 (y, z) rows around the tile's row the
// hull of the beads' x runs ("A"), plus, for beads within sx cells of an x face, the cells at the other end of the
// row ("B_lo": beads at the low face see the high end, "B_hi": the reverse); a tile that straddles a row end has two
// row groups, each with its own 27 range slots.  The concatenation of the non-empty ranges is the tile's WINDOW.
// k_nl_build writes the window's descriptor (D.wdesc) and the NL row of a bead as 16-bit offsets into the window;
// the force kernels (gm_force.cu) bulk-copy the window of the CURRENT positions into shared memory each step
// (cp.async.bulk, TMA engine: no LSU wavefronts; storage order is fixed until the next rebuild) and turn the neighbor
// gathers into LDS.128.  Window offset 0 is a far-away pad bead.
// A system of at most win_cap beads takes the whole position array as the window of every tile (one range).
// Tiles whose window does not fit (more than GM_WD_MAXR ranges, more than GmParams::win_cap positions, more than two
// rows of cells) keep 32-bit rows and the gather path (mode 0).
// The build itself keeps reading its candidates through L1 (79 % hits; a shared-memory copy of the window cost more
// in occupancy than the remaining misses do -- profiles/r02_windows.md).
struct NlWin {
    const int4 *rng;         // [GM_WIN_SLOTS] (first slot, window offset, length, row base r0 * ncx) per range slot
    int group;               // row group of this lane's bead (0 or 1)
    int whole;               // the window is the whole position array (small systems): offset = bead slot + 1
};

struct NlRow {
    int *ring;               // this lane's column of the ring: ring[(k & (NL_STAGE-1)) * 32]
    uint32_t lb;             // shared-memory byte address of ring[0] (the warp's ring is 4 KB-aligned)
    int4 *tile;              // this lane's int4 column of its NL tile: tile[q * 32]
    int k;                   // hits so far
    int flushed;             // entries already written to the tile (multiple of 16)
    int cap;
};

__device__ __forceinline__ uint32_t nl_pack2(int lo, int hi) { return (uint32_t)lo | ((uint32_t)hi << 16); }

// write entries [flushed, flushed + STAGE / 2) of the row from the ring to the tile: quads of 32-bit bead indices, or
// (W16) octs of 16-bit window offsets
template <int STAGE, bool W16>
__device__ __forceinline__ void nl_flush_half(NlRow &r)
{
    constexpr int H = STAGE / 2;
    if (r.flushed + H <= r.cap) {
        if (W16) {
#pragma unroll
            for (int o = 0; o < H / 8; ++o) {
                const int e = r.flushed + 8 * o;
                int v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) v[u] = r.ring[((e + u) & (STAGE - 1)) * 32];
                r.tile[(e >> 3) * 32] = make_int4((int)nl_pack2(v[0], v[1]), (int)nl_pack2(v[2], v[3]),
                                                  (int)nl_pack2(v[4], v[5]), (int)nl_pack2(v[6], v[7]));
            }
        } else {
#pragma unroll
            for (int q = 0; q < H / 4; ++q) {
                const int e = r.flushed + 4 * q;
                r.tile[(e >> 2) * 32] = make_int4(r.ring[((e + 0) & (STAGE - 1)) * 32], r.ring[((e + 1) & (STAGE - 1)) * 32],
                                                  r.ring[((e + 2) & (STAGE - 1)) * 32], r.ring[((e + 3) & (STAGE - 1)) * 32]);
            }
        }
    }
    r.flushed += H;
}

// Append candidate s to the lane's ring column if it is inside the run (u < left), inside r_list and
// (SELF) not bead i: ring[(k & (NL_STAGE-1)) * 32] = s; k += 1, with k kept as the byte offset kb = 128 k.
// The address is (kb & mask) | lb, one LOP3 (the warp's ring is 4 KB-aligned, so the two terms share no
// bits); store and increment are predicated on the hit (written in PTX: the compiler otherwise builds the
// increment from three selects).
template <bool SELF, int STAGE>
__device__ __forceinline__ void nl_append(uint32_t &kb, uint32_t lb, float r2, float r_list2, int left, int u,
                                          int s, int i)
{
    if (SELF)
        asm volatile("{\n\t.reg .pred v, p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %7, %8, 0xEA;\n\t"
                     "setp.gt.s32 v, %3, %4;\n\tsetp.lt.and.f32 p, %1, %2, v;\n\t"
                     "setp.ne.and.s32 p, %5, %6, p;\n\t@p st.shared.b32 [t], %5;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(left), "r"(u), "r"(s), "r"(i),
                       "n"((STAGE - 1) * 128), "r"(lb) : "memory");
    else
        asm volatile("{\n\t.reg .pred v, p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %7, %8, 0xEA;\n\t"
                     "setp.gt.s32 v, %3, %4;\n\tsetp.lt.and.f32 p, %1, %2, v;\n\t"
                     "@p st.shared.b32 [t], %5;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(left), "r"(u), "r"(s), "r"(i),
                       "n"((STAGE - 1) * 128), "r"(lb) : "memory");
}

// One run of candidates ref[s0 .. s1) against bead i, TRIP at a time, every one predicated on s < s1 (the
// runs of C3 hold ~7 candidates: no remainder loop, and the lanes of a warp make ceil(len / TRIP) trips).
// The entry appended for candidate s is s + delta: the bead index (delta = 0), or (W16) its offset in the tile's window.
// SHIFT: the run lies across a periodic face in some dimension; the displacement is then taken relative to
// the two faces, (a -+ L/2) - (b +- L/2) (see gm_min_image), with the bead side (ax, ay, az) prepared once
// per run and the candidate side b + (hx, hy, hz) per candidate.  SELF: the run holds bead i itself.
template <int TRIP, bool SHIFT, bool SELF, bool W16>
__device__ __forceinline__ void nl_scan_run(const float4 *__restrict__ ref, int s0, int s1, int delta, int i, float ax,
                                            float ay, float az, float hx, float hy, float hz, float r_list2,
                                            NlRow &r)
{
    constexpr int STAGE = NL_STAGE_OF(TRIP);
    uint32_t kb = (uint32_t)r.k * 128u;
    const int ie = i + delta;
    for (int s = s0; s < s1; s += TRIP) {
        // loads past the end of the run stay inside the array (per-bead arrays carry >= 8 pad slots after
        // bead n - 1, GmParams::ns); what they return is masked by the `left` test
        float4 q[TRIP];
#pragma unroll
        for (int u = 0; u < TRIP; ++u) q[u] = __ldg(ref + s + u);
        const int left = s1 - s;
        const int se = s + delta;
#pragma unroll
        for (int u = 0; u < TRIP; ++u) {
            float dx, dy, dz;
            if (SHIFT) { dx = ax - (q[u].x + hx); dy = ay - (q[u].y + hy); dz = az - (q[u].z + hz); }
            else { dx = ax - q[u].x; dy = ay - q[u].y; dz = az - q[u].z; }
            const float r2 = dx * dx + dy * dy + dz * dz;
            nl_append<SELF, STAGE>(kb, r.lb, r2, r_list2, left, u, se + u, ie);
        }
        // at most TRIP new entries per trip: flush as soon as half a ring is staged
        r.k = (int)(kb >> 7);
        if (r.k - r.flushed >= STAGE / 2) nl_flush_half<STAGE, W16>(r);
    }
}

// ---- warp-cooperative scan (dense cells: TRIP == 8) ----------------------------------------------------------------
// With several beads per cell the 32 beads of a warp sit in a handful of x-adjacent cells of ONE row, and their runs in
// each of the nine neighbor rows overlap almost entirely: the union of the 32 runs is 1.7 x one run on C5.  Per-lane
// scanning reads that union 32 times through the L1 data pipe (each LDG.128 of 32 slightly shifted addresses takes ~6
// wavefronts; the pipe was at 89 % on C5).  Here the warp loads the union once, 32 candidates per coalesced LDG.128, into
// a small shared-memory buffer, and every lane tests every candidate of the union from a broadcast LDS.128 (one wavefront
// per candidate per warp).  A candidate outside the lane's own run is more than r_list away in x (sx cells), so the
// distance test alone decides and the row comes out identical, entry for entry, to the per-lane scan.  All lanes run the
// same trips, so the flush is taken together too.  Warps that are not of one piece (a lane near a periodic face, two
// rows, pad lanes) keep the per-lane scan.
template <bool SELF>
__device__ __forceinline__ void nl_append_all(uint32_t &kb, uint32_t lb, float r2, float r_list2, int s, int i)
{
    if (SELF)
        asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %5, %6, 0xEA;\n\t"
                     "setp.lt.f32 p, %1, %2;\n\t"
                     "setp.ne.and.s32 p, %3, %4, p;\n\t@p st.shared.b32 [t], %3;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(s), "r"(i), "n"((NL_STAGE - 1) * 128), "r"(lb) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %5, %6, 0xEA;\n\t"
                     "setp.lt.f32 p, %1, %2;\n\t"
                     "@p st.shared.b32 [t], %3;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(s), "r"(i), "n"((NL_STAGE - 1) * 128), "r"(lb) : "memory");
}

// write entries [flushed, flushed + 8) of the row from the ring to the tile: one oct of window offsets or two quads
template <bool W16>
__device__ __forceinline__ void nl_flush8(NlRow &r)
{
    if (r.flushed + 8 <= r.cap) {
        const int e = r.flushed;
        int v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = r.ring[((e + u) & (NL_STAGE - 1)) * 32];
        if (W16) {
            r.tile[(e >> 3) * 32] = make_int4((int)nl_pack2(v[0], v[1]), (int)nl_pack2(v[2], v[3]),
                                              (int)nl_pack2(v[4], v[5]), (int)nl_pack2(v[6], v[7]));
        } else {
            r.tile[(e >> 2) * 32] = make_int4(v[0], v[1], v[2], v[3]);
            r.tile[((e >> 2) + 1) * 32] = make_int4(v[4], v[5], v[6], v[7]);
        }
    }
    r.flushed += 8;
}

// one row run of the union [u0, u1) against the warp's 32 beads; buf: the warp's [2][32] candidate buffer, b: the
// half to fill next
template <bool SELF, bool W16>
__device__ __forceinline__ void nl_union_run(const float4 *__restrict__ ref, int u0, int u1, int delta, int i, const float4 pi,
                                             float r_list2, NlRow &r, uint32_t &kb, float4 *buf, int &b)
{
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int ie = i + delta;
    if (u0 >= u1) return;
    float4 qn = __ldg(ref + (u0 + lane < u1 ? u0 + lane : u0));
    for (int base = u0; base < u1; base += 32) {
        const int cnt = min(32, u1 - base);
        float4 *cb = buf + b * 32;
        cb[lane] = lane < cnt ? qn : make_float4(1e18f, 1e18f, 1e18f, 0.f);      // the tail of the chunk: far away
        __syncwarp();
        // the next chunk's candidates are in flight while this one is tested.  One __syncwarp per chunk is enough:
        // half b is written again two chunks on, behind the barrier of the chunk in between
        if (base + 32 < u1) qn = __ldg(ref + (base + 32 + lane < u1 ? base + 32 + lane : base + 32));
        for (int j = 0; j < cnt; j += 8) {
            float4 q[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) q[u] = cb[j + u];
            const int se = base + j + delta;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float dx = pi.x - q[u].x, dy = pi.y - q[u].y, dz = pi.z - q[u].z;
                const float r2 = dx * dx + dy * dy + dz * dz;
                nl_append_all<SELF>(kb, r.lb, r2, r_list2, se + u, ie);
            }
            // fewer than 16 entries are staged before a trip and at most 8 arrive: when any lane reaches 16, every lane
            // holding a whole oct writes it, which leaves all lanes below 16 again (ring of 32)
            r.k = (int)(kb >> 7);
            if (__any_sync(full, r.k - r.flushed >= 16)) {
                if (r.k - r.flushed >= 8) nl_flush8<W16>(r);
            }
        }
        b ^= 1;
    }
}

// the nine runs of a warp of one piece: all 32 lanes hold beads of row (cy, cz), cells cx_lo .. cx_hi, none within
// sx cells of an x face or in a boundary row (so no periodic shifts and no wrapped pieces)
template <bool WIN>
__device__ __forceinline__ void nl_scan_warp(const GmParams &P, const GmDev &D, int i, const float4 pi, int cx_lo, int cx_hi,
                                             int cy, int cz, const NlWin &W, NlRow &row, float4 *buf)
{
    const float4 *__restrict__ ref = D.ref;
    const int *__restrict__ cstart = D.cstart;
    const uint32_t *__restrict__ rr = D.row_rank;
    const int ncx = P.nc[0], ncy = P.nc[1];
    const float rl2 = P.r_list2;
    const int c0 = cx_lo - P.sx, c1 = cx_hi + P.sx + 1;
    uint32_t kb = (uint32_t)row.k * 128u;
    int b = 0;
#pragma unroll 1
    for (int run = 0; run < 9; ++run) {
        const int oz = run / 3 - 1, oy = run - 3 * (run / 3) - 1;
        const int slot = W.group * 27 + run * 3;
        const int r0 = (WIN && !W.whole) ? W.rng[slot].w : (int)__ldg(rr + (cz + oz) * ncy + cy + oy) * ncx;
        const int u0 = __ldg(cstart + r0 + c0), u1 = __ldg(cstart + r0 + c1);
        int delta = 0;
        if (WIN) {
            const int4 g = W.rng[slot];
            delta = g.y - g.x;
        }
        if (run == 4) nl_union_run<true, WIN>(ref, u0, u1, delta, i, pi, rl2, row, kb, buf, b);
        else nl_union_run<false, WIN>(ref, u0, u1, delta, i, pi, rl2, row, kb, buf, b);
    }
    row.k = (int)(kb >> 7);
}

// Window set-up of a tile (all threads of the CTA; block-level barriers inside): range slots -> rng[], descriptor ->
// D.wdesc.  Returns 1 if the tile is window-staged (16-bit rows), 0 if it keeps 32-bit rows and the gather path.
// Descriptor: int4 per non-empty range k = 0 .. nr-1: (first slot, window offset, length, nr | mode << 8 | total << 16);
// a tile in mode 0 has entry 0 = (0, 0, 0, 0).
// cell: [GM_TILE] scratch, rng: [GM_WIN_SLOTS], sh_mode: one int -- all shared by the CTA.
__device__ __forceinline__ int nl_window(const GmParams &P, const GmDev &D, int tile, bool valid, int cx, int cy, int cz,
                                         int4 *rng, int4 *cell, int *sh_mode, int *group_out)
{
    const unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31;
    const int ncx = P.nc[0], ncy = P.nc[1], ncz = P.nc[2], sx = P.sx;
    int4 *__restrict__ wd = D.wdesc + (size_t)tile * GM_WD_STRIDE;
    *group_out = 0;
    if (P.n <= P.win_cap) {                  // small system: one range, the whole array
        if (tid == 0) wd[0] = make_int4(0, 1, P.n, 1 | (1 << 8) | (P.n << 16));
        if (tid < GM_WIN_SLOTS) rng[tid] = make_int4(0, 1, P.n, 0);
        __syncthreads();
        return 1;
    }
    const int rowid = valid ? cz * ncy + cy : -1;
    cell[tid] = make_int4(cx, cy, cz, rowid);
    const int nv = __syncthreads_count(valid);                         // valid beads are threads 0 .. nv - 1, nv >= 1
    const int4 ca = cell[0], cb = cell[nv - 1];
    const int ok = __syncthreads_and(!valid || rowid == ca.w || rowid == cb.w);
    const int n_a = __syncthreads_count(valid && rowid == ca.w);       // beads of row group 0 (keys ascend: group 0 first)
    const int ngroups = n_a < nv ? 2 : 1;
    *group_out = (valid && rowid != ca.w) ? 1 : 0;
    if (tid < 32) {
        // hull of each group in x cells: its first and last bead (cx ascends inside a group)
        const int f0 = ca.x, l0 = cell[n_a - 1].x, f1 = cell[n_a < nv ? n_a : 0].x, l1 = cb.x;
        const int y0 = ca.y, z0 = ca.z, y1 = cb.y, z1 = cb.z;
        int st_[2], off_[2], len_[2], k_[2];
        int total = 0, nr = 0;
#pragma unroll
        for (int round = 0; round < 2; ++round) {
            const int q = round * 32 + lane;
            int start = 0, len = 0, r0 = 0;
            const int g = q / 27, rem = q - 27 * g, run = rem / 3, piece = rem - 3 * run;
            if (q < GM_WIN_SLOTS && g < ngroups) {
                const int f = g ? f1 : f0, l = g ? l1 : l0;
                int y = (g ? y1 : y0) + (run - 3 * (run / 3)) - 1, z = (g ? z1 : z0) + run / 3 - 1;
                y += (y < 0) ? ncy : 0; y -= (y >= ncy) ? ncy : 0;
                z += (z < 0) ? ncz : 0; z -= (z >= ncz) ? ncz : 0;
                r0 = (int)__ldg(D.row_rank + z * ncy + y) * ncx;
                int c0 = 0, c1 = -1;
                if (piece == 0) { c0 = max(f - sx, 0); c1 = min(l + sx, ncx - 1); }
                else if (piece == 1) { if (f < sx) { c0 = ncx - (sx - f); c1 = ncx - 1; } }
                else { if (l + sx > ncx - 1) { c0 = 0; c1 = l + sx - ncx; } }
                if (c1 >= c0) { start = __ldg(D.cstart + r0 + c0); len = __ldg(D.cstart + r0 + c1 + 1) - start; }
            }
            int incl = len;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(full, incl, o);
                if (lane >= o) incl += t;
            }
            const unsigned ne = __ballot_sync(full, len > 0);
            st_[round] = start; len_[round] = len;
            off_[round] = 1 + total + incl - len;                         // window offset 0 is the pad bead
            k_[round] = nr + __popc(ne & ((1u << lane) - 1u));            // rank among the non-empty ranges
            if (q < GM_WIN_SLOTS) rng[q] = make_int4(start, off_[round], len, r0);
            total += __shfl_sync(full, incl, 31);
            nr += __popc(ne);
        }
        const int mode = (ok && nr <= GM_WD_MAXR && total <= P.win_cap) ? 1 : 0;
        if (mode) {
            const int hdr = nr | (1 << 8) | (total << 16);
#pragma unroll
            for (int round = 0; round < 2; ++round)
                if (len_[round] > 0) wd[k_[round]] = make_int4(st_[round], off_[round], len_[round], hdr);
        } else if (lane == 0) {
            wd[0] = make_int4(0, 0, 0, 0);
            atomicAdd(&D.ctl->n_glob_tiles, 1);
        }
        if (lane == 0) *sh_mode = mode;
    }
    __syncthreads();
    return *sh_mode;
}

// The nine (or, at the x faces, eighteen) runs of bead i.  WIN: the entries written are window offsets.
template <int TRIP, bool WIN>
__device__ __forceinline__ void nl_scan_bead(const GmParams &P, const GmDev &D, int i, const float4 pi, int cx, int cy,
                                             int cz, const NlWin &W, NlRow &row)
{
    const float4 *__restrict__ ref = D.ref;
    const int *__restrict__ cstart = D.cstart;
    const uint32_t *__restrict__ rr = D.row_rank;
    const int ncx = P.nc[0], ncy = P.nc[1], ncz = P.nc[2];
    const float rl2 = P.r_list2;
    // x pieces of a row: cells [xa0, xa1] are contiguous in ref (cells are r_list / sx wide in x, so the
    // run reaches sx cells to either side); a bead within sx cells of a face also sees the cells
    // [xb0, xb1] on the other side of the box
    const int sx = P.sx;
    const int xa0 = max(cx - sx, 0), xa1 = min(cx + sx, ncx - 1);
    const int xb0 = (cx < sx) ? ncx - (sx - cx) : 0;
    const int xb1 = (cx < sx) ? ncx - 1 : cx + sx - ncx;
    const bool has_xb = cx < sx || cx + sx > ncx - 1;
    const float hxb = (cx < sx) ? -P.half[0] : P.half[0];       // candidate side of the wrapped x piece
    const int pb = (cx < sx) ? 1 : 2;                           // window piece of the wrapped cells: B_lo or B_hi
    const bool inner = cx >= sx && cx + sx <= ncx - 1 && cy > 0 && cy < ncy - 1 && cz > 0 && cz < ncz - 1;
    // bounds of the piece [c0, c1] of row r0 (bead slots) and, for WIN, d: window offset = bead slot + d
    auto bounds = [&](int r0, int c0, int c1, int slot, int &s0, int &s1, int &d) {
        s0 = __ldg(cstart + r0 + c0); s1 = __ldg(cstart + r0 + c1 + 1); d = 0;
        if (WIN) {
            const int4 g = W.rng[slot];
            d = g.y - g.x;
        }
    };
    if (inner) {
#pragma unroll 1
        for (int run = 0; run < 9; ++run) {
            const int oz = run / 3 - 1, oy = run - 3 * (run / 3) - 1;
            const int slot = W.group * 27 + run * 3;
            const int r0 = (WIN && !W.whole) ? W.rng[slot].w : (int)__ldg(rr + (cz + oz) * ncy + cy + oy) * ncx;
            int s0, s1, is;
            bounds(r0, xa0, xa1, slot, s0, s1, is);
            if (run == 4)
                nl_scan_run<TRIP, false, true, WIN>(ref, s0, s1, is, i, pi.x, pi.y, pi.z, 0.f, 0.f, 0.f, rl2, row);
            else
                nl_scan_run<TRIP, false, false, WIN>(ref, s0, s1, is, i, pi.x, pi.y, pi.z, 0.f, 0.f, 0.f, rl2, row);
        }
    } else {
#pragma unroll 1
        for (int run = 0; run < 9; ++run) {
            const int oz = run / 3 - 1, oy = run - 3 * (run / 3) - 1;
            int z = cz + oz, y = cy + oy;
            float az = pi.z, hz = 0.f, ay = pi.y, hy = 0.f;
            if (z < 0) { z += ncz; az = pi.z + P.half[2]; hz = -P.half[2]; }
            else if (z >= ncz) { z -= ncz; az = pi.z - P.half[2]; hz = P.half[2]; }
            if (y < 0) { y += ncy; ay = pi.y + P.half[1]; hy = -P.half[1]; }
            else if (y >= ncy) { y -= ncy; ay = pi.y - P.half[1]; hy = P.half[1]; }
            const int slot = W.group * 27 + run * 3;
            const int r0 = (WIN && !W.whole) ? W.rng[slot].w : (int)__ldg(rr + z * ncy + y) * ncx;
            int s0, s1, is;
            bounds(r0, xa0, xa1, slot, s0, s1, is);
            nl_scan_run<TRIP, true, true, WIN>(ref, s0, s1, is, i, pi.x, ay, az, 0.f, hy, hz, rl2, row);
            if (has_xb) {
                bounds(r0, xb0, xb1, slot + pb, s0, s1, is);
                nl_scan_run<TRIP, true, true, WIN>(ref, s0, s1, is, i, pi.x - hxb, ay, az, hxb, hy, hz, rl2, row);
            }
        }
    }
}

// TRIP: candidates loaded together (4: runs of ~10 candidates, C1/C3; 8: runs of 20 and more, C2/C4/C5)
// WINS: the system uses tile windows (GmParams::use_win) -- compiled apart so that systems without them (DPD) run the
// plain kernel (56 registers, 9 CTAs per SM)
template <int TRIP, bool WINS>
__global__ void __launch_bounds__(NL_WARPS * 32, WINS ? NL_MINB_WIN : 9)
k_nl_build(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // shared memory: [NL_WARPS][STAGE][32] ring ints, a warp's ring (STAGE * 128 bytes: 2 or 4 KB) aligned by hand to its
    // size in the shared window (nl_append ORs the entry offset into the lane's base address; the launch asks for that
    // much slack), then the range slots of the CTA's tile window and the scratch of its set-up
    constexpr int STAGE = NL_STAGE_OF(TRIP);
    constexpr uint32_t RALIGN = STAGE * 128u;
    extern __shared__ int nl_smem_raw[];
    const uint32_t raw = (uint32_t)__cvta_generic_to_shared(nl_smem_raw);
    int *nl_ring = nl_smem_raw + (((raw + RALIGN - 1u) & ~(RALIGN - 1u)) - raw) / 4;
    // behind the rings, window systems only: [GM_WIN_SLOTS] range slots, cell[GM_TILE], mode, then (TRIP == 8) the candidate
    // buffers [NL_WARPS][2][32] of the union scan
    int4 *rng = reinterpret_cast<int4 *>(nl_ring + NL_WARPS * STAGE * 32);
    int4 *cell = rng + GM_WIN_SLOTS;
    int *sh_mode = reinterpret_cast<int *>(cell + GM_TILE);
    float4 *ubuf = reinterpret_cast<float4 *>(cell + GM_TILE + 1) + wid * 64;
    NlWin W;
    W.rng = rng;
    W.group = 0;
    W.whole = WINS && P.n <= P.win_cap;
    NlRow row;
    row.ring = nl_ring + wid * (STAGE * 32) + lane;
    row.lb = (uint32_t)__cvta_generic_to_shared(row.ring);
    row.tile = D.nl + ((size_t)(i >> 5) * P.capq) * 32 + lane;
    row.k = 0; row.flushed = 0; row.cap = P.nl_cap;
    const int cap = P.nl_cap;
    const bool valid = i < P.n;
    float4 pi = make_float4(0.f, 0.f, 0.f, 0.f);
    int cx = 0, cy = 0, cz = 0;
    if (valid) {
        pi = D.ref[i];
        cx = gm_cell_coord(pi.x, P.half[0], P.inv_w[0], P.nc[0]);
        cy = gm_cell_coord(pi.y, P.half[1], P.inv_w[1], P.nc[1]);
        cz = gm_cell_coord(pi.z, P.half[2], P.inv_w[2], P.nc[2]);
    }
    int mode = 0;
    if (WINS && (int)(blockIdx.x * blockDim.x) < P.n)           // CTA-uniform: the tile holds at least one bead
        mode = nl_window(P, D, blockIdx.x, valid, cx, cy, cz, rng, cell, sh_mode, &W.group);
    bool scanned = false;
    if (TRIP == 8 && WINS && NL_COOP) {      // measured: C5 1 928 -> 1 899 us per timestep; the DPD melt C4 (no windows) lost 1.7 % at 7 CTAs per SM and 0.4 % at 9, and keeps the per-lane scan
        const unsigned full = 0xffffffffu;
        const int cy0 = __shfl_sync(full, cy, 0), cz0 = __shfl_sync(full, cz, 0);
        const bool inner = valid && cx >= P.sx && cx + P.sx <= P.nc[0] - 1 && cy > 0 && cy < P.nc[1] - 1 && cz > 0 && cz < P.nc[2] - 1;
        if (__all_sync(full, inner && cy == cy0 && cz == cz0)) {
            const int cx_lo = __reduce_min_sync(full, cx), cx_hi = __reduce_max_sync(full, cx);
            if (WINS && mode) nl_scan_warp<true>(P, D, i, pi, cx_lo, cx_hi, cy, cz, W, row, ubuf);
            else nl_scan_warp<false>(P, D, i, pi, cx_lo, cx_hi, cy, cz, W, row, ubuf);
            scanned = true;
        }
    }
    if (valid && !scanned) {
        if (WINS && mode) nl_scan_bead<TRIP, true>(P, D, i, pi, cx, cy, cz, W, row);
        else nl_scan_bead<TRIP, false>(P, D, i, pi, cx, cy, cz, W, row);
    }
    if (valid && row.k > cap) atomicOr(&D.ctl->err, GM_DEV_ERR_OVERFLOW);
    // the tail of the row: whole quads (octs), at least minq quads in all (the force kernel loads those before
    // it knows NN), padded with the far-away bead (index n; window offset 0)
    const int kc = min(row.k, cap);
    if (WINS && mode) {
        const int no = max((kc + 7) >> 3, P.minq >> 1);
        for (int e = max(kc, row.flushed); e < 8 * no; ++e) row.ring[(e & (STAGE - 1)) * 32] = 0;
        for (int o = row.flushed >> 3; o < no; ++o) {
            const int e = 8 * o;
            int v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = row.ring[((e + u) & (STAGE - 1)) * 32];
            row.tile[o * 32] = make_int4((int)nl_pack2(v[0], v[1]), (int)nl_pack2(v[2], v[3]),
                                         (int)nl_pack2(v[4], v[5]), (int)nl_pack2(v[6], v[7]));
        }
    } else {
        const int nq = max((kc + 3) >> 2, P.minq);
        for (int e = max(kc, row.flushed); e < 4 * nq; ++e) row.ring[(e & (STAGE - 1)) * 32] = P.n;
        for (int q = row.flushed >> 2; q < nq; ++q) {
            const int e = 4 * q;
            row.tile[q * 32] = make_int4(row.ring[((e + 0) & (STAGE - 1)) * 32], row.ring[((e + 1) & (STAGE - 1)) * 32],
                                         row.ring[((e + 2) & (STAGE - 1)) * 32], row.ring[((e + 3) & (STAGE - 1)) * 32]);
        }
    }
    if (i < P.ns) D.nn[i] = kc;
    const int m = __reduce_max_sync(0xffffffffu, kc);
    const unsigned int sum = __reduce_add_sync(0xffffffffu, (unsigned int)kc);
    if (lane == 0) {
        D.nnw[i >> 5] = m;
        if (sum > 0) {
            atomicMax(&D.ctl->max_nn, m);
            atomicAdd(&D.ctl->sum_nn, (unsigned long long)sum);
        }
    }
}

// a7 set-up: BL of every slot in index space from its tag-space row (the sort moved the beads).  A kernel of
// its own (full occupancy, a dozen registers): at the end of k_nl_build the dependent blt -> rtag -> store chain
// kept every warp's slot for two more memory latencies.  Runs after k_nl_build: a partner that lies inside the
// window of the bead's tile is stored as a window offset (GM_BOND_LOCAL) and read from shared memory by the force
// kernels; the others keep their bead index and are gathered.
__global__ void __launch_bounds__(256)
k_bl_remap(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const int sel = (int)(D.ctl->n_rebuilds & 1ull);
    const size_t ns = (size_t)P.ns;
    const int4 *__restrict__ wd = D.wdesc + (size_t)(i / GM_TILE) * GM_WD_STRIDE;
    const int hdr = P.use_win ? __ldg(&wd[0].w) : 0;
    const int nr = (hdr & 0x100) ? (hdr & 0xff) : 0;
    for (int b = 0; b < P.max_bonds; ++b) {
        const int e = D.blt[sel][b * ns + i];
        int out = -1;
        if (e >= 0) {
            const int j = D.rtag[e & GM_BOND_MASK];
            out = j | (e & ~(GM_BOND_MASK | GM_BOND_LOCAL));
            // the tile's ranges four at a time (independent loads; entries past nr are stale but inside the
            // descriptor's GM_WD_STRIDE slots and masked)
            for (int r = 0; r < nr; r += 4) {
                int4 g[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) g[u] = __ldg(wd + r + u);
                int off = -1;
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (r + u < nr && (unsigned)(j - g[u].x) < (unsigned)g[u].z) off = g[u].y + j - g[u].x;
                if (off >= 0) {
                    out = off | GM_BOND_LOCAL | (e & ~(GM_BOND_MASK | GM_BOND_LOCAL));
                    break;
                }
            }
        }
        D.bl[b * ns + i] = out;
    }
}

int gm_nl_capacity_ok(const GmParams &P) { return P.nl_cap >= 8 && P.nl_cap % 8 == 0; }

// dynamic shared memory of k_nl_build: the rings (+ one warp's ring of alignment slack), then what the variant needs
int gm_nl_smem_bytes(const GmParams &P)
{
    const int stage = NL_STAGE_OF(P.nl_trip);
    int b = NL_WARPS * stage * 32 * 4 + stage * 128;
    if (P.use_win) b += (GM_WIN_SLOTS + GM_TILE + 1) * 16 + (P.nl_trip == 8 ? NL_WARPS * 64 * 16 : 0);
    return b;
}

cudaError_t gm_nl_prepare(const GmParams &P)
{
    (void)P;            // 23 KB of dynamic shared memory: below the 48 KB that need an opt-in
    return cudaSuccess;
}

void gm_launch_nl_build(const GmParams &P, const GmDev &D, cudaStream_t st, const GmFork *fk)
{
    const int threads = NL_WARPS * 32;
    const int smem = gm_nl_smem_bytes(P);
    const int nb = (P.ns + threads - 1) / threads;
    // BL remap: needs the window descriptors of this build on window-staged systems, so it follows the build there;
    // otherwise it goes first (the order measured best in round 1)
    // Without windows the remap needs only the sort (rtag, blt) and only the step kernel needs its result: it runs on the
    // side stream, in the shadow of the build (C3: 13 of 118 us), and joins afterwards
    bool forked = false;
    if (P.max_bonds > 0 && !P.use_win) {
        if (fk && fk->side && cudaEventRecord(fk->fork, st) == cudaSuccess &&
            cudaStreamWaitEvent(fk->side, fk->fork, 0) == cudaSuccess) {
            k_bl_remap<<<(P.n + 255) / 256, 256, 0, fk->side>>>(P, D);
            forked = true;
        } else {
            k_bl_remap<<<(P.n + 255) / 256, 256, 0, st>>>(P, D);
        }
    }
    if (P.use_win) {
        if (P.nl_trip == 8) k_nl_build<8, true><<<nb, threads, smem, st>>>(P, D);
        else k_nl_build<4, true><<<nb, threads, smem, st>>>(P, D);
    } else {
        if (P.nl_trip == 8) k_nl_build<8, false><<<nb, threads, smem, st>>>(P, D);
        else k_nl_build<4, false><<<nb, threads, smem, st>>>(P, D);
    }
    if (forked) {
        cudaEventRecord(fk->join, fk->side);
        cudaStreamWaitEvent(st, fk->join, 0);
    }
    if (P.max_bonds > 0 && P.use_win) k_bl_remap<<<(P.n + 255) / 256, 256, 0, st>>>(P, D);
}

// Neighbor list in tag space for the boundary (gm_get_neighbors), tags [t0, t1): nn_out[tag - t0],
// nl_out[(tag - t0) * stride + k].  One thread per tag.
__global__ void __launch_bounds__(256)
k_unpack_neighbors(const __grid_constant__ GmParams P, GmDev D, int *__restrict__ nn_out,
                   int *__restrict__ nl_out, long long stride, int t0, int t1)
{
    const int t = t0 + blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= t1) return;
    const int *__restrict__ tag = D.tag[D.ctl->n_rebuilds & 1ull];
    const int i = D.rtag[t];
    const int nn = D.nn[i];
    nn_out[t - t0] = nn;
    const int *__restrict__ tile = reinterpret_cast<const int *>(D.nl + ((size_t)(i >> 5) * P.capq) * 32 + (i & 31));
    const int4 *__restrict__ wd = D.wdesc + (size_t)(i / GM_TILE) * GM_WD_STRIDE;
    const int hdr = P.use_win ? wd[0].w : 0;
    if (hdr & 0x100) {
        // window-staged tile: 16-bit window offsets, eight per int4; offset -> range -> bead index
        const int nr = hdr & 0xff;
        const unsigned short *__restrict__ t16 = reinterpret_cast<const unsigned short *>(tile);
        for (int k = 0; k < nn && k < stride; ++k) {
            const int off = t16[(k >> 3) * 256 + (k & 7)];
            int r = 0;
            while (r + 1 < nr && wd[r + 1].y <= off) ++r;
            nl_out[(long long)(t - t0) * stride + k] = tag[wd[r].x + off - wd[r].y];
        }
        return;
    }
    for (int k = 0; k < nn && k < stride; ++k)
        nl_out[(long long)(t - t0) * stride + k] = tag[tile[(k >> 2) * 128 + (k & 3)]];
}

void gm_launch_unpack_neighbors(const GmParams &P, const GmDev &D, int *nn_out, int *nl_out, long long stride,
                                int t0, int t1, cudaStream_t st)
{
    if (t1 <= t0) return;
    k_unpack_neighbors<<<(t1 - t0 + 255) / 256, 256, 0, st>>>(P, D, nn_out, nl_out, stride, t0, t1);
}
