// gm_io.cu -- boundary marshalling kernels: tag-order (N,3) float arrays <-> the float4 storage
// arrays, the device control block, and the conditional-graph gate.  No arithmetic of the method
// except the half-kick that completes a half-step velocity for output (a8; see gm_force.cu).
#include "gm_internal.cuh"

#define IO_BLOCK 256

__device__ __forceinline__ float wrap_any(float x, float half, float L)
{
    if (x >= half || x < -half) x -= L * floorf((x + half) / L);
    return gm_wrap(x, half, L);
}

__global__ void __launch_bounds__(IO_BLOCK)
k_pack(GmParams P, GmDev D, int cur, const float *__restrict__ pos3, const float *__restrict__ vel3,
       const int *__restrict__ type, const float *__restrict__ mass)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    float x = wrap_any(pos3[3 * i + 0], P.half[0], P.box[0]);
    float y = wrap_any(pos3[3 * i + 1], P.half[1], P.box[1]);
    float z = wrap_any(pos3[3 * i + 2], P.half[2], P.box[2]);
    D.pos[cur][i] = make_float4(x, y, z, __int_as_float(type[i]));
    float vx = vel3[3 * i + 0], vy = vel3[3 * i + 1], vz = vel3[3 * i + 2];
    D.vel[i] = make_float4(vx, vy, vz, mass ? mass[i] : 1.0f);
    if (D.vt[0]) D.vt[cur][i] = make_float4(vx, vy, vz, __int_as_float(i));
    D.tag[i] = i;
    D.rtag[i] = i;
}

__global__ void __launch_bounds__(IO_BLOCK)
k_unpack(GmParams P, GmDev D, int cur, float *__restrict__ pos3, float *__restrict__ vel3,
         float *__restrict__ force3, int lagged)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    int t = D.tag[i];
    if (pos3) {
        float4 p = D.pos[cur][i];
        pos3[3 * t + 0] = p.x; pos3[3 * t + 1] = p.y; pos3[3 * t + 2] = p.z;
    }
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    if (force3 || (vel3 && lagged)) f = D.frc[i];
    if (vel3) {
        float4 u = D.vel[i];
        if (lagged) {   // v^m = u^{m-1} + dt/2 a^m
            float h = 0.5f * P.dt / u.w;
            u.x += h * f.x; u.y += h * f.y; u.z += h * f.z;
        }
        vel3[3 * t + 0] = u.x; vel3[3 * t + 1] = u.y; vel3[3 * t + 2] = u.z;
    }
    if (force3) { force3[3 * t + 0] = f.x; force3[3 * t + 1] = f.y; force3[3 * t + 2] = f.z; }
}

void gm_launch_pack(const GmParams &P, const GmDev &D, int cur, const float *pos3, const float *vel3,
                    const int *type, const float *mass, cudaStream_t st)
{
    k_pack<<<(P.n + IO_BLOCK - 1) / IO_BLOCK, IO_BLOCK, 0, st>>>(P, D, cur, pos3, vel3, type, mass);
}

void gm_launch_unpack(const GmParams &P, const GmDev &D, int cur, float *pos3, float *vel3, float *force3,
                      int lagged, cudaStream_t st)
{
    k_unpack<<<(P.n + IO_BLOCK - 1) / IO_BLOCK, IO_BLOCK, 0, st>>>(P, D, cur, pos3, vel3, force3, lagged);
}

__global__ void k_set_ctl(GmDev D, unsigned long long step, int reset_all)
{
    GmCtl *c = D.ctl;
    c->step[0] = step;
    c->step[1] = step;
    c->need = ~0ull;
    if (reset_all) {
        c->n_rebuilds = 0; c->sum_nn = 0; c->max_nn = 0; c->err = 0; c->built = 0; c->pad = 0;
    }
}

void gm_launch_set_ctl(const GmDev &D, unsigned long long step, int reset_all, cudaStream_t st)
{
    k_set_ctl<<<1, 1, 0, st>>>(D, step, reset_all);
}

// Gate of the conditional graph node that holds the rebuild kernels: body runs iff a rebuild is due
// at this time level (a4).
__global__ void k_gate(GmDev D, int parity, cudaGraphConditionalHandle h)
{
    cudaGraphSetConditional(h, D.ctl->need == D.ctl->step[parity] ? 1u : 0u);
}

void gm_launch_gate(const GmDev &D, int parity, unsigned long long cond_handle, cudaStream_t st)
{
    k_gate<<<1, 1, 0, st>>>(D, parity, (cudaGraphConditionalHandle)cond_handle);
}
