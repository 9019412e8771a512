// gm_static.cu -- gm_kinetic_static: kinetic energy and momentum of a set of beads (the a9 sums of k_energy) through an
// entry point that needs no gm_system, no workspace and allocates nothing: the per-block partial sums, which the a9
// reduction otherwise keeps in the caller's workspace (GmDev::esum), live in a file-scope __device__ array of fixed size.
// For callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The array is held by every GPU that loads the library, until exit (GM_STATIC_BYTES = 262,400 bytes).  ALL calls share
// it: two calls that overlap on one GPU (different streams, or two host threads) race on the partial sums and on the
// ticket; calls on one stream are ordered and safe.  The array keeps the last call's contents: the only part that must
// start at zero, the ticket counter, is cleared on the stream at the start of every call.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <mutex>

#include "../../include/gm.h"

#define ST_BLOCK 256
#define ST_PER_THREAD 4                       // beads per thread: a CTA takes 1,024 consecutive beads
#define ST_MAX_BLOCKS (GM_STATIC_MAX_BEADS / (ST_BLOCK * ST_PER_THREAD))
#define ST_TICKET_OFFSET (ST_MAX_BLOCKS * 4 * sizeof(double))
#define GM_STATIC_BYTES (ST_TICKET_OFFSET + 256)
#define ST_MAX_DEVICES 64
static_assert(GM_STATIC_MAX_BEADS % (ST_BLOCK * ST_PER_THREAD) == 0, "whole CTAs");

// [ST_MAX_BLOCKS][4] doubles (ke, px, py, pz of each CTA), then the ticket counter.  In HOST code this name is a stand-in,
// not a device address: the address kernels are given comes from cudaGetSymbolAddress (static_scratch below).
static __device__ __align__(256) unsigned char gm_static_scratch[GM_STATIC_BYTES];

// One launch: every CTA writes its four partial sums (fixed order inside the CTA, no atomics on the sums), takes a
// ticket, and the CTA that draws the last ticket adds the partials in an order that depends on nothing but the grid size.
__global__ void __launch_bounds__(ST_BLOCK)
k_kinetic_static(const float *__restrict__ vel3, const float *__restrict__ mass, long long n, double *part,
                 unsigned int *ticket, double *__restrict__ out4)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double acc[4] = { 0.0, 0.0, 0.0, 0.0 };
    const long long base = (long long)blockIdx.x * (ST_BLOCK * ST_PER_THREAD);
#pragma unroll
    for (int k = 0; k < ST_PER_THREAD; ++k) {
        const long long i = base + (long long)k * ST_BLOCK + tid;
        if (i < n) {
            // as k_energy: fp32 inputs, every term and every sum in fp64
            const double vx = (double)vel3[3 * i + 0], vy = (double)vel3[3 * i + 1], vz = (double)vel3[3 * i + 2];
            const double m = mass ? (double)mass[i] : 1.0;
            acc[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
            acc[1] += m * vx; acc[2] += m * vy; acc[3] += m * vz;
        }
    }
    __shared__ double sh[ST_BLOCK / 32][4];
    __shared__ bool last;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        double v = acc[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) sh[wid][q] = v;
    }
    __syncthreads();
    if (tid < 4) {
        double v = 0.0;
        for (int w = 0; w < ST_BLOCK / 32; ++w) v += sh[w][tid];
        part[(size_t)blockIdx.x * 4 + tid] = v;
        __threadfence();                                   // the partials are visible before the ticket is taken
    }
    __syncthreads();
    if (tid == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (wid < 4) {                                         // warp q sums quantity q: lane l takes CTAs l, l + 32, ... in order
        double v = 0.0;
        for (unsigned int b = lane; b < gridDim.x; b += 32) v += __ldcg(part + (size_t)b * 4 + wid);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) out4[wid] = v;
    }
    if (tid == 0) *ticket = 0u;
}

// The device address of the scratch array on `device` (made current here): resolved once per device and kept.
static cudaError_t static_scratch(int device, unsigned char **ptr)
{
    static std::mutex mu;
    static unsigned char *known[ST_MAX_DEVICES];
    std::lock_guard<std::mutex> lock(mu);
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return e;
    if (!known[device]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, gm_static_scratch);
        if (e != cudaSuccess) return e;
        known[device] = static_cast<unsigned char *>(p);
    }
    *ptr = known[device];
    return cudaSuccess;
}

#define ST_FAIL(code, ...)                                      \
    do {                                                        \
        if (err && err_len) snprintf(err, err_len, __VA_ARGS__); \
        return (code);                                          \
    } while (0)

extern "C" gm_status gm_kinetic_static(const float *vel3, const float *mass, int64_t n, int device, void *stream,
                                       double *out4, char *err, size_t err_len)
{
    if (err && err_len) err[0] = 0;
    if ((!vel3 && n > 0) || !out4 || n < 0)
        ST_FAIL(GM_ERR_INVALID_ARG, "gm_kinetic_static: NULL vel3 / out4, or n < 0 (n = %lld)", (long long)n);
    if (n > (int64_t)GM_STATIC_MAX_BEADS)
        ST_FAIL(GM_ERR_INVALID_ARG, "gm_kinetic_static: n = %lld exceeds the static scratch array (at most %lld beads per call)",
                (long long)n, (long long)GM_STATIC_MAX_BEADS);
    if (device < 0 || device >= ST_MAX_DEVICES)
        ST_FAIL(GM_ERR_INVALID_ARG, "gm_kinetic_static: device %d outside [0, %d)", device, ST_MAX_DEVICES);
    unsigned char *scratch = nullptr;
    cudaError_t e = static_scratch(device, &scratch);
    cudaStream_t st = (cudaStream_t)stream;
    if (e == cudaSuccess) e = cudaMemsetAsync(scratch + ST_TICKET_OFFSET, 0, 256, st);      // the ticket starts at zero
    if (e == cudaSuccess) {
        const long long per = ST_BLOCK * ST_PER_THREAD;
        const unsigned int nb = (unsigned int)((n + per - 1) / per);
        k_kinetic_static<<<nb ? nb : 1u, ST_BLOCK, 0, st>>>(vel3, mass, (long long)n, reinterpret_cast<double *>(scratch),
                                                             reinterpret_cast<unsigned int *>(scratch + ST_TICKET_OFFSET), out4);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) ST_FAIL(GM_ERR_CUDA, "gm_kinetic_static: CUDA: %s", cudaGetErrorString(e));
    return GM_OK;
}
