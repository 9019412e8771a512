// gm_nlist.cu -- a3: skin-padded FULL Verlet neighbor list from the 27 surrounding cells
// ("searching neighboring particles from the surrounding 27 cells (including the cell
// that the target particle resides in)", all neighbors "within a distance that is the sum of the
// cutoff ... r_cut, and the buffer distance, r_buffer"; table form NL[k*Np + i], NN[i]: L51, Fig. 1).
//
// One thread per bead, in storage (SFC) order so a warp's beads sit in a handful of adjacent cells
// and share their candidate segments through L1.  The cell list is CSR over x-fastest linear cell
// ids, so the three x-adjacent cells of one (y, z) row form one contiguous segment of cpos[]: nine
// segments per bead instead of 27 (two extra pieces where the row wraps around the box).
#include "gm_internal.cuh"

#define NL_BLOCK 128

// One row piece: candidates cpos[s0 .. s1) against bead i.  SHIFT: the piece lies across a periodic face
// in some dimension; the displacement is then taken relative to the two faces, (a -+ L/2) - (b +- L/2)
// (see gm_min_image), with the bead side (ax, ay, az) prepared once per piece and the candidate side
// b + (hx, hy, hz) per candidate -- no branches in the loop.
template <bool SHIFT>
__device__ __forceinline__ int nl_scan_piece(const float4 *__restrict__ cpos, int s0, int s1, int i, float ax,
                                             float ay, float az, float hx, float hy, float hz, float r_list2,
                                             int k, int cap, int *__restrict__ col, size_t col_stride)
{
#pragma unroll 4
    for (int s = s0; s < s1; ++s) {
        const float4 q = cpos[s];
        float dx, dy, dz;
        if (SHIFT) { dx = ax - (q.x + hx); dy = ay - (q.y + hy); dz = az - (q.z + hz); }
        else { dx = ax - q.x; dy = ay - q.y; dz = az - q.z; }
        const float r2 = dx * dx + dy * dy + dz * dz;
        const int j = __float_as_int(q.w);
        if (r2 < r_list2 && j != i) {
            if (k < cap) col[(size_t)k * col_stride] = j;
            ++k;
        }
    }
    return k;
}

// Thread s owns the bead in slot s of the cell-sorted array cpos[] (not storage bead s): the 32 beads
// of a warp then sit in a few consecutive cells of one x row, so at every loop iteration the lanes read
// the same or adjacent candidates (few L1 wavefronts per request) and run nearly equal trip counts.
__global__ void __launch_bounds__(NL_BLOCK)
k_nl_build(const __grid_constant__ GmParams P, GmDev D, int gate, int parity)
{
    if (gate && D.ctl->need != D.ctl->step[parity]) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t ns = (size_t)P.ns;
    const int cap = P.nl_cap;
    int k = 0;
    if (s < P.n) {
        const float4 *__restrict__ cpos = D.cpos;
        const int *__restrict__ cstart = D.cstart;
        const float4 pi = cpos[s];
        const int i = __float_as_int(pi.w);
        int *__restrict__ col = D.nl + i;
        const int cx = gm_cell_coord(pi.x, P.half[0], P.inv_w[0], P.nc[0]);
        const int cy = gm_cell_coord(pi.y, P.half[1], P.inv_w[1], P.nc[1]);
        const int cz = gm_cell_coord(pi.z, P.half[2], P.inv_w[2], P.nc[2]);
        const int ncx = P.nc[0], ncy = P.nc[1], ncz = P.nc[2];
        const float rl2 = P.r_list2;
        // x pieces of a row: cells [xa0, xa1] are contiguous in cpos; a bead in an edge column also
        // sees the single cell xb on the other side of the box
        const int xa0 = max(cx - 1, 0), xa1 = min(cx + 1, ncx - 1);
        const int xb = (cx == 0) ? ncx - 1 : ((cx == ncx - 1) ? 0 : -1);
        const float hxb = (cx == 0) ? -P.half[0] : P.half[0];       // candidate side of the wrapped x piece
        const bool inner = cx > 0 && cx < ncx - 1 && cy > 0 && cy < ncy - 1 && cz > 0 && cz < ncz - 1;
        if (inner) {
            for (int oz = -1; oz <= 1; ++oz)
                for (int oy = -1; oy <= 1; ++oy) {
                    const int row = ((cz + oz) * ncy + cy + oy) * ncx;
                    k = nl_scan_piece<false>(cpos, cstart[row + xa0], cstart[row + xa1 + 1], i, pi.x, pi.y, pi.z,
                                             0.f, 0.f, 0.f, rl2, k, cap, col, ns);
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
                    const int row = (z * ncy + y) * ncx;
                    k = nl_scan_piece<true>(cpos, cstart[row + xa0], cstart[row + xa1 + 1], i, pi.x, ay, az,
                                            0.f, hy, hz, rl2, k, cap, col, ns);
                    if (xb >= 0)
                        k = nl_scan_piece<true>(cpos, cstart[row + xb], cstart[row + xb + 1], i, pi.x - hxb, ay, az,
                                                hxb, hy, hz, rl2, k, cap, col, ns);
                }
            }
        }
        const int kc = min(k, cap);
        D.nn[i] = kc;
        D.ref[i] = make_float4(pi.x, pi.y, pi.z, 0.f);
        atomicMax(&D.nnw[i >> 5], kc);     // tile height for the step kernel's bulk loads (cleared in k_sort_clear)
        if (k > cap) atomicOr(&D.ctl->err, GM_DEV_ERR_OVERFLOW);
    }
    const int kc = min(k, cap);
    const int m = __reduce_max_sync(0xffffffffu, kc);
    const unsigned int sum = __reduce_add_sync(0xffffffffu, (unsigned int)kc);
    if ((threadIdx.x & 31) == 0 && sum > 0) {
        atomicMax(&D.ctl->max_nn, m);
        atomicAdd(&D.ctl->sum_nn, (unsigned long long)sum);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) D.ctl->built = 1;
}

void gm_launch_nl_build(const GmParams &P, const GmDev &D, const float4 *pos, int gate, int parity,
                        cudaStream_t st)
{
    (void)pos;
    k_nl_build<<<(P.n + NL_BLOCK - 1) / NL_BLOCK, NL_BLOCK, 0, st>>>(P, D, gate, parity);
}

// Neighbor list in tag space for the boundary (gm_get_neighbors): nn_out[tag], nl_out[tag*stride + k].
__global__ void __launch_bounds__(256)
k_unpack_neighbors(GmParams P, GmDev D, int *__restrict__ nn_out, int *__restrict__ nl_out, long long stride)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    int t = D.tag[i];
    int nn = D.nn[i];
    nn_out[t] = nn;
    for (int k = 0; k < nn && k < stride; ++k)
        nl_out[(long long)t * stride + k] = D.tag[D.nl[(size_t)k * P.ns + i]];
}

void gm_launch_unpack_neighbors(const GmParams &P, const GmDev &D, int *nn_out, int *nl_out, long long stride,
                                cudaStream_t st)
{
    k_unpack_neighbors<<<(P.n + 255) / 256, 256, 0, st>>>(P, D, nn_out, nl_out, stride);
}
