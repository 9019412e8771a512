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

__global__ void __launch_bounds__(NL_BLOCK)
k_nl_build(const __grid_constant__ GmParams P, GmDev D, const float4 *__restrict__ pos, int gate, int parity)
{
    if (gate && D.ctl->need != D.ctl->step[parity]) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int k = 0;
    if (i < P.n) {
        const float4 pi = pos[i];
        const int cx = gm_cell_coord(pi.x, P.half[0], P.inv_w[0], P.nc[0]);
        const int cy = gm_cell_coord(pi.y, P.half[1], P.inv_w[1], P.nc[1]);
        const int cz = gm_cell_coord(pi.z, P.half[2], P.inv_w[2], P.nc[2]);
        const int ncx = P.nc[0], ncy = P.nc[1], ncz = P.nc[2];
        const float4 *__restrict__ cpos = D.cpos;
        const int *__restrict__ cstart = D.cstart;
        int *__restrict__ nl = D.nl + i;
        const size_t n = (size_t)P.n;
        const int cap = P.nl_cap;
        // x pieces of a row: [x0, x1] contiguous, plus a wrapped single cell when cx is at an edge
        int xa0 = max(cx - 1, 0), xa1 = min(cx + 1, ncx - 1);
        int xb = (cx == 0) ? ncx - 1 : ((cx == ncx - 1) ? 0 : -1);
        for (int oz = -1; oz <= 1; ++oz) {
            int z = cz + oz;
            z = (z < 0) ? z + ncz : ((z >= ncz) ? z - ncz : z);
            for (int oy = -1; oy <= 1; ++oy) {
                int y = cy + oy;
                y = (y < 0) ? y + ncy : ((y >= ncy) ? y - ncy : y);
                int row = (z * ncy + y) * ncx;
#pragma unroll 1
                for (int piece = 0; piece < 2; ++piece) {
                    int s0, s1;
                    if (piece == 0) { s0 = cstart[row + xa0]; s1 = cstart[row + xa1 + 1]; }
                    else {
                        if (xb < 0) break;
                        s0 = cstart[row + xb]; s1 = cstart[row + xb + 1];
                    }
                    for (int s = s0; s < s1; ++s) {
                        float4 q = cpos[s];
                        int j = __float_as_int(q.w);
                        float dx = gm_min_image(pi.x, q.x, P.half[0]);
                        float dy = gm_min_image(pi.y, q.y, P.half[1]);
                        float dz = gm_min_image(pi.z, q.z, P.half[2]);
                        float r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 < P.r_list2 && j != i) {
                            if (k < cap) nl[(size_t)k * n] = j;
                            ++k;
                        }
                    }
                }
            }
        }
        D.nn[i] = min(k, cap);
        D.ref[i] = pi;
        if (k > cap) atomicOr(&D.ctl->err, GM_DEV_ERR_OVERFLOW);
    }
    // list statistics (off the force path): max and sum of NN
    int m = k;
    unsigned int sum = (unsigned int)k;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
    }
    if ((threadIdx.x & 31) == 0 && sum > 0) {
        atomicMax(&D.ctl->max_nn, m);
        atomicAdd(&D.ctl->sum_nn, (unsigned long long)sum);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) D.ctl->built = 1;
}

void gm_launch_nl_build(const GmParams &P, const GmDev &D, const float4 *pos, int gate, int parity,
                        cudaStream_t st)
{
    k_nl_build<<<(P.n + NL_BLOCK - 1) / NL_BLOCK, NL_BLOCK, 0, st>>>(P, D, pos, gate, parity);
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
        nl_out[(long long)t * stride + k] = D.tag[D.nl[(size_t)k * P.n + i]];
}

void gm_launch_unpack_neighbors(const GmParams &P, const GmDev &D, int *nn_out, int *nl_out, long long stride,
                                cudaStream_t st)
{
    k_unpack_neighbors<<<(P.n + 255) / 256, 256, 0, st>>>(P, D, nn_out, nl_out, stride);
}
