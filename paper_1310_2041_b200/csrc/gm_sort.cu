// gm_sort.cu -- a1 cell binning by counting sort, a2 SFC reorder (PAPER.md:L57,
// Alg. 1 Kernel 1 L376-388 for what a cell list holds; L33/L199 for the memory sort).
//
// The paper claims a slot per particle with atomicInc into a fixed-slot CL table.  Here the cell
// list is CSR: key -> histogram -> exclusive scan -> scatter, then every cell's segment is sorted by
// storage index so that the result (and with it the NL row order and every fp32 sum downstream)
// is the same on every run, whatever order the histogram atomics were served in.
//
// One counting sort serves both uses:
//   use_sfc_rank = 0: key = linear cell id (x fastest)  -> cstart[], cpos[]   (a1, every rebuild)
//   use_sfc_rank = 1: key = Hilbert rank of that cell   -> permutation sorted[] (a2, every sfc_period)
#include "gm_internal.cuh"

#define SORT_BLOCK 256

__device__ __forceinline__ bool gm_gated_off(const GmCtl *ctl, int gate, int parity)
{
    return gate && ctl->need != ctl->step[parity];
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_sort_clear(GmParams P, GmDev D, int use_sfc_rank, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    int stride = gridDim.x * blockDim.x;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c <= P.n_cells; c += stride) D.cstart[c] = 0;
    if (!use_sfc_rank)
        for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < P.ns / 32; c += stride) D.nnw[c] = 0;
    if (!use_sfc_rank && blockIdx.x == 0 && threadIdx.x == 0) {
        D.ctl->n_rebuilds += 1;
        D.ctl->max_nn = 0;
        D.ctl->sum_nn = 0;
    }
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_sort_keys(GmParams P, GmDev D, const float4 *__restrict__ pos, int use_sfc_rank, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    float4 p = pos[i];
    int key = 0;
    if (isfinite(p.x) && isfinite(p.y) && isfinite(p.z)) {
        int cx = gm_cell_coord(p.x, P.half[0], P.inv_w[0], P.nc[0]);
        int cy = gm_cell_coord(p.y, P.half[1], P.inv_w[1], P.nc[1]);
        int cz = gm_cell_coord(p.z, P.half[2], P.inv_w[2], P.nc[2]);
        key = (cz * P.nc[1] + cy) * P.nc[0] + cx;
        if (use_sfc_rank) key = (int)D.cell_rank[key];
    } else {
        atomicOr(&D.ctl->err, GM_DEV_ERR_NONFINITE);
    }
    D.key[i] = key;
    D.rank[i] = atomicAdd(&D.cstart[key], 1);     // arrival order; made canonical in k_cell_finish
}

// ---- exclusive scan of cstart[0 .. n_cells] (n_cells + 1 entries, the last count is 0) ----------
__device__ __forceinline__ int block_exclusive_scan(int v, int *total)
{
    __shared__ int warp_sums[32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int nw = blockDim.x >> 5;
        int w = lane < nw ? warp_sums[lane] : 0;
        int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        warp_sums[lane] = wi - w;            // exclusive warp offsets
        if (lane == 31) *total = wi;
    }
    __syncthreads();
    int r = warp_sums[wid] + incl - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(GM_SCAN_BLOCK)
k_scan_local(GmParams P, GmDev D, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    __shared__ int total;
    int n = P.n_cells + 1;
    int base = (blockIdx.x * GM_SCAN_BLOCK + threadIdx.x) * GM_SCAN_ITEMS;
    int v[GM_SCAN_ITEMS], s = 0;
#pragma unroll
    for (int q = 0; q < GM_SCAN_ITEMS; ++q) {
        v[q] = (base + q < n) ? D.cstart[base + q] : 0;
        s += v[q];
    }
    int off = block_exclusive_scan(s, &total);
#pragma unroll
    for (int q = 0; q < GM_SCAN_ITEMS; ++q) {
        if (base + q < n) D.cstart[base + q] = off;
        off += v[q];
    }
    if (threadIdx.x == 0) D.scan_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(GM_SCAN_BLOCK)
k_scan_sums(GmParams P, GmDev D, int n_blocks, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    __shared__ int total;
    int carry = 0;
    for (int b0 = 0; b0 < n_blocks; b0 += GM_SCAN_BLOCK) {
        int idx = b0 + threadIdx.x;
        int v = idx < n_blocks ? D.scan_sums[idx] : 0;
        int off = block_exclusive_scan(v, &total);
        if (idx < n_blocks) D.scan_sums[idx] = carry + off;
        carry += total;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(GM_SCAN_BLOCK)
k_scan_add(GmParams P, GmDev D, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    int n = P.n_cells + 1;
    int add = D.scan_sums[blockIdx.x];
    int base = (blockIdx.x * GM_SCAN_BLOCK + threadIdx.x) * GM_SCAN_ITEMS;
#pragma unroll
    for (int q = 0; q < GM_SCAN_ITEMS; ++q)
        if (base + q < n) D.cstart[base + q] += add;
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_sort_scatter(GmParams P, GmDev D, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    D.sorted[D.cstart[D.key[i]] + D.rank[i]] = i;
}

// One thread per key: put the segment into ascending storage-index order (segments are a handful
// of beads: 3 to 19 per cell in the five configs), then, for the cell list, gather the coordinates.
__global__ void __launch_bounds__(SORT_BLOCK)
k_cell_finish(GmParams P, GmDev D, const float4 *__restrict__ pos, int write_cpos, int gate, int parity)
{
    if (gm_gated_off(D.ctl, gate, parity)) return;
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.n_cells) return;
    int b = D.cstart[c], e = D.cstart[c + 1];
    for (int s = b + 1; s < e; ++s) {
        int v = D.sorted[s];
        int t = s - 1;
        while (t >= b && D.sorted[t] > v) { D.sorted[t + 1] = D.sorted[t]; --t; }
        D.sorted[t + 1] = v;
    }
    if (write_cpos)
        for (int s = b; s < e; ++s) {
            int idx = D.sorted[s];
            float4 p = pos[idx];
            D.cpos[s] = make_float4(p.x, p.y, p.z, __int_as_float(idx));
        }
}

void gm_launch_sort_keys(const GmParams &P, const GmDev &D, const float4 *pos, int use_sfc_rank, int gate,
                         int parity, cudaStream_t st)
{
    int nb = (P.n + SORT_BLOCK - 1) / SORT_BLOCK;
    int per = GM_SCAN_BLOCK * GM_SCAN_ITEMS;
    int nsb = (P.n_cells + 1 + per - 1) / per;
    int ncb = (P.n_cells + 1 + SORT_BLOCK - 1) / SORT_BLOCK;
    if (ncb > 1184) ncb = 1184;
    k_sort_clear<<<ncb, SORT_BLOCK, 0, st>>>(P, D, use_sfc_rank, gate, parity);
    k_sort_keys<<<nb, SORT_BLOCK, 0, st>>>(P, D, pos, use_sfc_rank, gate, parity);
    k_scan_local<<<nsb, GM_SCAN_BLOCK, 0, st>>>(P, D, gate, parity);
    k_scan_sums<<<1, GM_SCAN_BLOCK, 0, st>>>(P, D, nsb, gate, parity);
    k_scan_add<<<nsb, GM_SCAN_BLOCK, 0, st>>>(P, D, gate, parity);
    k_sort_scatter<<<nb, SORT_BLOCK, 0, st>>>(P, D, gate, parity);
}

void gm_launch_cell_finish(const GmParams &P, const GmDev &D, const float4 *pos, int write_cpos, int gate,
                           int parity, cudaStream_t st)
{
    int nb = (P.n_cells + SORT_BLOCK - 1) / SORT_BLOCK;
    k_cell_finish<<<nb, SORT_BLOCK, 0, st>>>(P, D, pos, write_cpos, gate, parity);
}

// ---- a2: apply the permutation sorted[new] = old to every per-bead array --------------------------
__global__ void __launch_bounds__(SORT_BLOCK)
k_permute4(int n, const int *__restrict__ perm, const float4 *__restrict__ src, float4 *__restrict__ dst)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[perm[i]];
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_permute_tag(int n, const int *__restrict__ perm, const int *__restrict__ src, int *__restrict__ dst)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[perm[i]];
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_set_rtag(int n, const int *__restrict__ tag_new, int *__restrict__ tag, int *__restrict__ rtag)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { int t = tag_new[i]; tag[i] = t; rtag[t] = i; }
}

void gm_launch_reorder(const GmParams &P, GmDev &D, int cur, cudaStream_t st)
{
    int n = P.n, nb = (n + SORT_BLOCK - 1) / SORT_BLOCK;
    size_t b4 = (size_t)n * sizeof(float4);
    k_permute4<<<nb, SORT_BLOCK, 0, st>>>(n, D.sorted, D.pos[cur], D.tmp4);
    cudaMemcpyAsync(D.pos[cur], D.tmp4, b4, cudaMemcpyDeviceToDevice, st);
    k_permute4<<<nb, SORT_BLOCK, 0, st>>>(n, D.sorted, D.vel, D.tmp4);
    cudaMemcpyAsync(D.vel, D.tmp4, b4, cudaMemcpyDeviceToDevice, st);
    if (D.vt[0]) {
        k_permute4<<<nb, SORT_BLOCK, 0, st>>>(n, D.sorted, D.vt[cur], D.tmp4);
        cudaMemcpyAsync(D.vt[cur], D.tmp4, b4, cudaMemcpyDeviceToDevice, st);
    }
    k_permute_tag<<<nb, SORT_BLOCK, 0, st>>>(n, D.sorted, D.tag, D.tmpi);
    k_set_rtag<<<nb, SORT_BLOCK, 0, st>>>(n, D.tmpi, D.tag, D.rtag);
}

// BL/BN in index space from the tag-space master table (the tags in column i of BL
// are the beads bonded to i; stored under both ends).
__global__ void __launch_bounds__(SORT_BLOCK) k_bonds_to_index(GmParams P, GmDev D)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    int t = D.tag[i];
    int nb = D.bn_tag[t];
    D.bn[i] = nb;
    for (int k = 0; k < nb; ++k) {
        int e = D.bl_tag[(size_t)k * P.n + t];
        D.bl[(size_t)k * P.ns + i] = D.rtag[e & GM_BOND_MASK] | (e & ~GM_BOND_MASK);
    }
}

void gm_launch_bonds_to_index(const GmParams &P, const GmDev &D, cudaStream_t st)
{
    if (P.max_bonds <= 0) return;
    k_bonds_to_index<<<(P.n + SORT_BLOCK - 1) / SORT_BLOCK, SORT_BLOCK, 0, st>>>(P, D);
}
