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
// whatever the row capacity, which leaves the rest of the SM's 228 KB to L1 for the candidate loads.
#include "gm_internal.cuh"

#define NL_STAGE 32          // ring entries per lane (power of two, >= 16 + 4)
#ifndef NL_WARPS
#define NL_WARPS 4
#endif

struct NlRow {
    int *ring;               // this lane's column of the ring: ring[(k & (NL_STAGE-1)) * 32]
    uint32_t lb;             // shared-memory byte address of ring[0] (the warp's ring is 4 KB-aligned)
    int4 *tile;              // this lane's int4 column of its NL tile: tile[q * 32]
    int k;                   // hits so far
    int flushed;             // entries already written to the tile (multiple of 16)
    int cap;
};

// write entries [flushed, flushed + 16) of the row (whole quads) from the ring to the tile
__device__ __forceinline__ void nl_flush16(NlRow &r)
{
    if (r.flushed + 16 <= r.cap) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int e = r.flushed + 4 * q;
            r.tile[(e >> 2) * 32] = make_int4(r.ring[((e + 0) & (NL_STAGE - 1)) * 32], r.ring[((e + 1) & (NL_STAGE - 1)) * 32],
                                              r.ring[((e + 2) & (NL_STAGE - 1)) * 32], r.ring[((e + 3) & (NL_STAGE - 1)) * 32]);
        }
    }
    r.flushed += 16;
}

// Append candidate slot s to the lane's ring column if it is inside the run (u < left), inside r_list and
// (SELF) not bead i: ring[(k & (NL_STAGE-1)) * 32] = s; k += 1, with k kept as the byte offset kb = 128 k.
// The address is (kb & mask) | lb, one LOP3 (the warp's ring is 4 KB-aligned, so the two terms share no
// bits); store and increment are predicated on the hit (written in PTX: the compiler otherwise builds the
// increment from three selects).
template <bool SELF>
__device__ __forceinline__ void nl_append(uint32_t &kb, uint32_t lb, float r2, float r_list2, int left, int u,
                                          int s, int i)
{
    if (SELF)
        asm volatile("{\n\t.reg .pred v, p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %7, %8, 0xEA;\n\t"
                     "setp.gt.s32 v, %3, %4;\n\tsetp.lt.and.f32 p, %1, %2, v;\n\t"
                     "setp.ne.and.s32 p, %5, %6, p;\n\t@p st.shared.b32 [t], %5;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(left), "r"(u), "r"(s), "r"(i),
                       "n"((NL_STAGE - 1) * 128), "r"(lb) : "memory");
    else
        asm volatile("{\n\t.reg .pred v, p;\n\t.reg .b32 t;\n\tlop3.b32 t, %0, %7, %8, 0xEA;\n\t"
                     "setp.gt.s32 v, %3, %4;\n\tsetp.lt.and.f32 p, %1, %2, v;\n\t"
                     "@p st.shared.b32 [t], %5;\n\t@p add.u32 %0, %0, 128;\n\t}"
                     : "+r"(kb) : "f"(r2), "f"(r_list2), "r"(left), "r"(u), "r"(s), "r"(i),
                       "n"((NL_STAGE - 1) * 128), "r"(lb) : "memory");
}

// One run of candidates ref[s0 .. s1) against bead i, four at a time, every one predicated on s < s1 (the
// runs of C3 hold ~9 candidates: no remainder loop, and the lanes of a warp make ceil(len / 4) trips).
// SHIFT: the run lies across a periodic face in some dimension; the displacement is then taken relative to
// the two faces, (a -+ L/2) - (b +- L/2) (see gm_min_image), with the bead side (ax, ay, az) prepared once
// per run and the candidate side b + (hx, hy, hz) per candidate.  SELF: the run holds bead i itself.
template <int TRIP, bool SHIFT, bool SELF>
__device__ __forceinline__ void nl_scan_run(const float4 *__restrict__ ref, int s0, int s1, int i, float ax,
                                            float ay, float az, float hx, float hy, float hz, float r_list2,
                                            NlRow &r)
{
    uint32_t kb = (uint32_t)r.k * 128u;
    for (int s = s0; s < s1; s += TRIP) {
        // loads past the end of the run stay inside the array (per-bead arrays carry >= 8 pad slots after
        // bead n - 1, GmParams::ns); what they return is masked by the `left` test
        float4 q[TRIP];
#pragma unroll
        for (int u = 0; u < TRIP; ++u) q[u] = __ldg(ref + s + u);
        const int left = s1 - s;
#pragma unroll
        for (int u = 0; u < TRIP; ++u) {
            float dx, dy, dz;
            if (SHIFT) { dx = ax - (q[u].x + hx); dy = ay - (q[u].y + hy); dz = az - (q[u].z + hz); }
            else { dx = ax - q[u].x; dy = ay - q[u].y; dz = az - q[u].z; }
            const float r2 = dx * dx + dy * dy + dz * dz;
            nl_append<SELF>(kb, r.lb, r2, r_list2, left, u, s + u, i);
        }
        // at most TRIP <= 8 new entries per trip: flush as soon as 16 are staged (ring of 32)
        r.k = (int)(kb >> 7);
        if (r.k - r.flushed >= 16) nl_flush16(r);
    }
}

// TRIP: candidates loaded together (4: runs of ~10 candidates, C1/C3; 8: runs of 20 and more, C2/C4/C5)
template <int TRIP>
__global__ void __launch_bounds__(NL_WARPS * 32)
k_nl_build(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // [NL_WARPS][NL_STAGE][32] ints, 4 KB per warp, aligned by hand to 4 KB in the shared window (nl_ring_put
    // ORs the entry offset into the lane's base address); the launch asks for 4 KB of slack
    extern __shared__ int nl_ring_raw[];
    const uint32_t raw = (uint32_t)__cvta_generic_to_shared(nl_ring_raw);
    int *nl_ring = nl_ring_raw + (((raw + 4095u) & ~4095u) - raw) / 4;
    NlRow row;
    row.ring = nl_ring + wid * (NL_STAGE * 32) + lane;
    row.lb = (uint32_t)__cvta_generic_to_shared(row.ring);
    row.tile = D.nl + ((size_t)(i >> 5) * P.capq) * 32 + lane;
    row.k = 0; row.flushed = 0; row.cap = P.nl_cap;
    const int cap = P.nl_cap;
    if (i < P.n) {
        const float4 *__restrict__ ref = D.ref;
        const int *__restrict__ cstart = D.cstart;
        const uint32_t *__restrict__ rr = D.row_rank;
        const float4 pi = ref[i];
        const int cx = gm_cell_coord(pi.x, P.half[0], P.inv_w[0], P.nc[0]);
        const int cy = gm_cell_coord(pi.y, P.half[1], P.inv_w[1], P.nc[1]);
        const int cz = gm_cell_coord(pi.z, P.half[2], P.inv_w[2], P.nc[2]);
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
        const bool inner = cx >= sx && cx + sx <= ncx - 1 && cy > 0 && cy < ncy - 1 && cz > 0 && cz < ncz - 1;
        if (inner) {
            for (int oz = -1; oz <= 1; ++oz)
                for (int oy = -1; oy <= 1; ++oy) {
                    const int r0 = (int)__ldg(rr + (cz + oz) * ncy + cy + oy) * ncx;
                    if (oz == 0 && oy == 0)
                        nl_scan_run<TRIP, false, true>(ref, __ldg(cstart + r0 + xa0), __ldg(cstart + r0 + xa1 + 1), i, pi.x,
                                                 pi.y, pi.z, 0.f, 0.f, 0.f, rl2, row);
                    else
                        nl_scan_run<TRIP, false, false>(ref, __ldg(cstart + r0 + xa0), __ldg(cstart + r0 + xa1 + 1), i, pi.x,
                                                  pi.y, pi.z, 0.f, 0.f, 0.f, rl2, row);
                }
        } else {
            for (int oz = -1; oz <= 1; ++oz) {
                int z = cz + oz;
                float az = pi.z, hz = 0.f;
                if (z < 0) { z += ncz; az = pi.z + P.half[2]; hz = -P.half[2]; }
                else if (z >= ncz) { z -= ncz; az = pi.z - P.half[2]; hz = P.half[2]; }
                for (int oy = -1; oy <= 1; ++oy) {
                    int y = cy + oy;
                    float ay = pi.y, hy = 0.f;
                    if (y < 0) { y += ncy; ay = pi.y + P.half[1]; hy = -P.half[1]; }
                    else if (y >= ncy) { y -= ncy; ay = pi.y - P.half[1]; hy = P.half[1]; }
                    const int r0 = (int)__ldg(rr + z * ncy + y) * ncx;
                    nl_scan_run<TRIP, true, true>(ref, __ldg(cstart + r0 + xa0), __ldg(cstart + r0 + xa1 + 1), i, pi.x, ay, az,
                                      0.f, hy, hz, rl2, row);
                    if (has_xb)
                        nl_scan_run<TRIP, true, true>(ref, __ldg(cstart + r0 + xb0), __ldg(cstart + r0 + xb1 + 1), i, pi.x - hxb,
                                          ay, az, hxb, hy, hz, rl2, row);
                }
            }
        }
        if (row.k > cap) atomicOr(&D.ctl->err, GM_DEV_ERR_OVERFLOW);
    }
    // the tail of the row: whole quads, at least minq of them in all (the force kernel loads those before
    // it knows NN), padded with the far-away bead
    const int kc = min(row.k, cap);
    const int nq = max((kc + 3) >> 2, P.minq);
    for (int e = max(kc, row.flushed); e < 4 * nq; ++e) row.ring[(e & (NL_STAGE - 1)) * 32] = P.n;
    for (int q = row.flushed >> 2; q < nq; ++q) {
        const int e = 4 * q;
        row.tile[q * 32] = make_int4(row.ring[((e + 0) & (NL_STAGE - 1)) * 32], row.ring[((e + 1) & (NL_STAGE - 1)) * 32],
                                     row.ring[((e + 2) & (NL_STAGE - 1)) * 32], row.ring[((e + 3) & (NL_STAGE - 1)) * 32]);
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
// kept every warp's slot for two more memory latencies.
__global__ void __launch_bounds__(256)
k_bl_remap(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const int sel = (int)(D.ctl->n_rebuilds & 1ull);
    const size_t ns = (size_t)P.ns;
    for (int b = 0; b < P.max_bonds; ++b) {
        const int e = D.blt[sel][b * ns + i];
        D.bl[b * ns + i] = e < 0 ? -1 : (D.rtag[e & GM_BOND_MASK] | (e & ~GM_BOND_MASK));
    }
}

int gm_nl_capacity_ok(const GmParams &P) { return P.nl_cap >= 8 && P.nl_cap % 4 == 0; }

void gm_launch_nl_build(const GmParams &P, const GmDev &D, cudaStream_t st)
{
    const int threads = NL_WARPS * 32;
    if (P.max_bonds > 0) k_bl_remap<<<(P.n + 255) / 256, 256, 0, st>>>(P, D);
    const int smem = NL_WARPS * NL_STAGE * 32 * 4 + 4096;
    if (P.nl_trip == 8) k_nl_build<8><<<(P.ns + threads - 1) / threads, threads, smem, st>>>(P, D);
    else k_nl_build<4><<<(P.ns + threads - 1) / threads, threads, smem, st>>>(P, D);
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
    for (int k = 0; k < nn && k < stride; ++k)
        nl_out[(long long)(t - t0) * stride + k] = tag[tile[(k >> 2) * 128 + (k & 3)]];
}

void gm_launch_unpack_neighbors(const GmParams &P, const GmDev &D, int *nn_out, int *nl_out, long long stride,
                                int t0, int t1, cudaStream_t st)
{
    if (t1 <= t0) return;
    k_unpack_neighbors<<<(t1 - t0 + 255) / 256, 256, 0, st>>>(P, D, nn_out, nl_out, stride, t0, t1);
}
