// gm_sort.cu -- a1 cell binning by counting sort, fused with a2, the space-filling-curve reorder of the
// particle arrays (PAPER.md:L57 and Alg. 1 Kernel 1 L376-388 for what a cell list holds;
// L33/L199 for the memory sort).
//
// The paper claims a slot per particle with atomicInc into a fixed-slot CL table and re-sorts memory
// now and then with SFCPACK.  Here ONE counting sort does both, at every rebuild: the sort key of a
// bead is the rank of its cell along the curve (cells run along x inside a row; the (y, z) rows follow
// a 2-D Hilbert curve), and all per-bead state is moved into that order.  Afterwards
//   - the sorted position array `ref` IS the cell list (CSR: cell c = slots [cstart[c], cstart[c+1])),
//     the three x-adjacent cells of a row are one contiguous run, and slot index == bead index, so the
//     neighbor search (gm_nlist.cu) needs no indirection and writes whole tiles of the NL table;
//   - the 32 beads of a warp of the force kernel sit in a few adjacent cells: their gathers hit the
//     same cache lines and their list lengths are alike.
// Within a cell, beads are ordered by their previous slot, so the result (and with it every fp32 sum
// downstream) is the same on every run whatever order the histogram atomics were served in.
//
// Chain: k_gate (decide, publish ctl->go) -> k_keys (key + histogram) -> k_scan_local / k_scan_add
// (exclusive scan -> cstart) -> k_scatter (slot lists per cell) -> k_permute (canonical slot, move state)
// -> k_bl_remap, k_nl_build (gm_nlist.cu).
#include "gm_internal.cuh"

#define SORT_BLOCK 256
static_assert(GM_SCAN_ITEMS == 4, "the scan kernels move one int4 per thread");

// Decide whether the rebuild runs at this time level and publish the decision (every later kernel of
// the chain only reads ctl->go).  With a conditional graph node the body is skipped altogether.
__device__ __forceinline__ int gate_decide(GmCtl *c, int gate, int parity)
{
    const int go = gm_rebuild_off(c, gate, parity) ? 0 : 1;
    c->go = go;
    if (go) {
        c->rebuilt_at = c->step[parity];
        c->n_rebuilds += 1;
        c->max_nn = 0;
        c->sum_nn = 0;
        c->n_glob_tiles = 0;
    }
    return go;
}

__global__ void k_gate(GmDev D, int gate, int parity) { gate_decide(D.ctl, gate, parity); }

__global__ void k_gate_cond(GmDev D, int gate, int parity, cudaGraphConditionalHandle h)
{
    cudaGraphSetConditional(h, (unsigned)gate_decide(D.ctl, gate, parity));
}

void gm_launch_gate(const GmDev &D, int gate, int parity, unsigned long long cond_handle, int use_handle,
                    cudaStream_t st)
{
    if (use_handle) k_gate_cond<<<1, 1, 0, st>>>(D, gate, parity, (cudaGraphConditionalHandle)cond_handle);
    else k_gate<<<1, 1, 0, st>>>(D, gate, parity);
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_keys(const __grid_constant__ GmParams P, GmDev D, int parity)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    float4 p = D.pos[parity][i];
    int key = 0;
    if (isfinite(p.x) && isfinite(p.y) && isfinite(p.z)) {
        // the step kernel leaves positions unwrapped between rebuilds (at most skin/2 outside the box)
        p.x = gm_wrap(p.x, P.half[0], P.box[0]); p.y = gm_wrap(p.y, P.half[1], P.box[1]);
        p.z = gm_wrap(p.z, P.half[2], P.box[2]);
        const int cx = gm_cell_coord(p.x, P.half[0], P.inv_w[0], P.nc[0]);
        const int cy = gm_cell_coord(p.y, P.half[1], P.inv_w[1], P.nc[1]);
        const int cz = gm_cell_coord(p.z, P.half[2], P.inv_w[2], P.nc[2]);
        key = (int)D.row_rank[cz * P.nc[1] + cy] * P.nc[0] + cx;
    } else {
        atomicOr(&D.ctl->err, GM_DEV_ERR_NONFINITE);
    }
    D.key[i] = key;
    D.rank[i] = atomicAdd(&D.ccount[key], 1);     // arrival order; made canonical in k_permute
}

// ---- exclusive scan of ccount[0 .. n_cells] into cstart (n_cells + 1 entries, the last count is 0) ----
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

// A single-pass scan (tickets + look-back over the tile totals) measured SLOWER inside the step graphs than these
// two launches (C3: 72.1 vs 71.5 us per timestep, same box): kept as two kernels.
// Block-local exclusive scan; leaves ccount zeroed for the next rebuild.
__global__ void __launch_bounds__(GM_SCAN_BLOCK)
k_scan_local(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    __shared__ int total;
    const int n = P.n_cells + 1;
    const int base = (blockIdx.x * GM_SCAN_BLOCK + threadIdx.x) * GM_SCAN_ITEMS;
    int v[GM_SCAN_ITEMS], s = 0;
    if (base + GM_SCAN_ITEMS <= n) {
        const int4 q = *reinterpret_cast<const int4 *>(D.ccount + base);
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        *reinterpret_cast<int4 *>(D.ccount + base) = make_int4(0, 0, 0, 0);
    } else {
#pragma unroll
        for (int q = 0; q < GM_SCAN_ITEMS; ++q) {
            v[q] = (base + q < n) ? D.ccount[base + q] : 0;
            if (base + q < n) D.ccount[base + q] = 0;
        }
    }
#pragma unroll
    for (int q = 0; q < GM_SCAN_ITEMS; ++q) s += v[q];
    int off = block_exclusive_scan(s, &total);
    if (base + GM_SCAN_ITEMS <= n) {          // one 16-byte store per thread (cstart is 256-byte aligned)
        *reinterpret_cast<int4 *>(D.cstart + base) = make_int4(off, off + v[0], off + v[0] + v[1], off + v[0] + v[1] + v[2]);
    } else {
#pragma unroll
        for (int q = 0; q < GM_SCAN_ITEMS; ++q) {
            if (base + q < n) D.cstart[base + q] = off;
            off += v[q];
        }
    }
    if (threadIdx.x == 0) D.scan_sums[blockIdx.x] = total;
}

// Each block adds the sum of the totals of the blocks before it (a few hundred at most).
__global__ void __launch_bounds__(GM_SCAN_BLOCK)
k_scan_add(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    __shared__ int warp_part[32];
    __shared__ int add_sh;
    int part = 0;
    for (int b = threadIdx.x; b < (int)blockIdx.x; b += GM_SCAN_BLOCK) part += D.scan_sums[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_down_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x < 32) {
        int v = warp_part[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) add_sh = v;
    }
    __syncthreads();
    const int add = add_sh;
    const int n = P.n_cells + 1;
    const int base = (blockIdx.x * GM_SCAN_BLOCK + threadIdx.x) * GM_SCAN_ITEMS;
    if (base + GM_SCAN_ITEMS <= n) {
        int4 c = *reinterpret_cast<const int4 *>(D.cstart + base);
        c.x += add; c.y += add; c.z += add; c.w += add;
        *reinterpret_cast<int4 *>(D.cstart + base) = c;
    } else {
#pragma unroll
        for (int q = 0; q < GM_SCAN_ITEMS; ++q)
            if (base + q < n) D.cstart[base + q] += add;
    }
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_scatter(const __grid_constant__ GmParams P, GmDev D)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    D.sorted[D.cstart[D.key[i]] + D.rank[i]] = i;
}

// a2: thread i = old slot.  Its new slot is the start of its cell plus the number of beads of that cell
// that had a smaller old slot (canonical order); then every per-bead array follows.
__global__ void __launch_bounds__(SORT_BLOCK)
k_permute(const __grid_constant__ GmParams P, GmDev D, int parity)
{
    if (!D.ctl->go) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const int sel = (int)(D.ctl->n_rebuilds & 1ull);       // buffers this rebuild writes
    float4 p = D.pos[parity][i];
    p.x = gm_wrap(p.x, P.half[0], P.box[0]); p.y = gm_wrap(p.y, P.half[1], P.box[1]);
    p.z = gm_wrap(p.z, P.half[2], P.box[2]);
    const float4 u = D.vel[i];
    const int t = D.tag[sel ^ 1][i];
    const int c = D.key[i];
    const int b = D.cstart[c], e = D.cstart[c + 1];
    int r = 0;
    for (int s = b; s < e; ++s) r += (D.sorted[s] < i) ? 1 : 0;
    const int d = b + r;
    D.ref[d] = p;
    D.svel[d] = u;
    if (D.svt) D.svt[d] = D.vt[parity][i];
    D.tag[sel][d] = t;
    D.rtag[t] = d;
    const size_t ns = (size_t)P.ns;
    for (int k = 0; k < P.max_bonds; ++k) D.blt[sel][k * ns + d] = D.blt[sel ^ 1][k * ns + i];
}

void gm_launch_sort(const GmParams &P, const GmDev &D, int parity, cudaStream_t st)
{
    const int nb = (P.n + SORT_BLOCK - 1) / SORT_BLOCK;
    const int per = GM_SCAN_BLOCK * GM_SCAN_ITEMS;
    const int nsb = (P.n_cells + 1 + per - 1) / per;
    k_keys<<<nb, SORT_BLOCK, 0, st>>>(P, D, parity);
    k_scan_local<<<nsb, GM_SCAN_BLOCK, 0, st>>>(P, D);
    k_scan_add<<<nsb, GM_SCAN_BLOCK, 0, st>>>(P, D);
    k_scatter<<<nb, SORT_BLOCK, 0, st>>>(P, D);
    k_permute<<<nb, SORT_BLOCK, 0, st>>>(P, D, parity);
}

// BL in tag space, storage order, from the tag-order master table written by gm_set_bonds
// (column i of BL holds the beads bonded to i; each bond is stored under both ends).
__global__ void __launch_bounds__(SORT_BLOCK) k_bonds_from_master(const __grid_constant__ GmParams P, GmDev D)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const int sel = (int)(D.ctl->n_rebuilds & 1ull);
    const int t = D.tag[sel][i];
    const size_t ns = (size_t)P.ns;
    for (int k = 0; k < P.max_bonds; ++k) {
        const int e = D.bl_tag[k * ns + t];
        D.blt[sel][k * ns + i] = e;
        D.bl[k * ns + i] = e < 0 ? -1 : (D.rtag[e & GM_BOND_MASK] | (e & ~GM_BOND_MASK));
    }
}

void gm_launch_bonds_from_master(const GmParams &P, const GmDev &D, cudaStream_t st)
{
    if (P.max_bonds <= 0) return;
    k_bonds_from_master<<<(P.n + SORT_BLOCK - 1) / SORT_BLOCK, SORT_BLOCK, 0, st>>>(P, D);
}
