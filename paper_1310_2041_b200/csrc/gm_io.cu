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
k_pack(const __grid_constant__ GmParams P, GmDev D, int cur, const float *__restrict__ pos3,
       const float *__restrict__ vel3, const int *__restrict__ type, const float *__restrict__ mass)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    float x = wrap_any(pos3[3 * i + 0], P.half[0], P.box[0]);
    float y = wrap_any(pos3[3 * i + 1], P.half[1], P.box[1]);
    float z = wrap_any(pos3[3 * i + 2], P.half[2], P.box[2]);
    // a type outside [0, n_types) would index the pair table out of bounds, a mass <= 0 has no acceleration:
    // latched, reported as GM_ERR_INVALID_ARG by the next synchronising call; the bead is stored as type 0, mass 1
    int ty = type[i];
    float m = mass ? mass[i] : 1.0f;
    if (ty < 0 || ty >= P.n_types || !(m > 0.0f) || !isfinite(m)) {
        atomicOr(&D.ctl->err, GM_DEV_ERR_BAD_INPUT);
        ty = (ty < 0 || ty >= P.n_types) ? 0 : ty;
        m = (m > 0.0f && isfinite(m)) ? m : 1.0f;
    }
    D.pos[cur][i] = make_float4(x, y, z, __int_as_float(ty));
    float vx = vel3[3 * i + 0], vy = vel3[3 * i + 1], vz = vel3[3 * i + 2];
    D.vel[i] = make_float4(vx, vy, vz, m);
    if (D.vt[0]) D.vt[cur][i] = make_float4(vx, vy, vz, __int_as_float(i));
    D.tag[0][i] = i;            // k_set_ctl(reset_all) selects buffer 0
    D.rtag[i] = i;
}

__global__ void __launch_bounds__(IO_BLOCK)
k_unpack(const __grid_constant__ GmParams P, GmDev D, int cur, float *__restrict__ pos3,
         float *__restrict__ vel3, float *__restrict__ force3, int lagged)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const Src S = current_src(D, cur, D.ctl->step[cur]);
    int t = S.tag[i];
    if (pos3) {
        float4 p = S.pos[i];     // may sit up to skin/2 outside the box between rebuilds: wrapped on the way out
        pos3[3 * t + 0] = gm_wrap(p.x, P.half[0], P.box[0]);
        pos3[3 * t + 1] = gm_wrap(p.y, P.half[1], P.box[1]);
        pos3[3 * t + 2] = gm_wrap(p.z, P.half[2], P.box[2]);
    }
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    if (force3 || (vel3 && lagged)) f = D.frc[i];
    if (vel3) {
        float4 u = S.vel[i];
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

// The far-away pad bead in slot n of every position array (NL quads are padded with index n), and
// "no bond" (-1) in every bond table.
__global__ void k_init_pad(const __grid_constant__ GmParams P, GmDev D)
{
    const float4 far = make_float4(1e18f, 1e18f, 1e18f, 0.f);
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = P.n + threadIdx.x; i < P.ns; i += blockDim.x) {
        D.pos[0][i] = far; D.pos[1][i] = far; D.ref[i] = far;
        D.vel[i] = zero; D.svel[i] = zero;
        if (D.vt[0]) { D.vt[0][i] = zero; D.vt[1][i] = zero; D.svt[i] = zero; }
        D.nn[i] = 0;
    }
}

void gm_launch_init_pad(const GmParams &P, const GmDev &D, cudaStream_t st)
{
    k_init_pad<<<1, 256, 0, st>>>(P, D);
}

__global__ void k_set_ctl(GmDev D, unsigned long long step, int reset_all, int parity)
{
    GmCtl *c = D.ctl;
    const bool fresh = !reset_all && c->rebuilt_at == c->step[parity];
    c->step[0] = step;
    c->step[1] = step;
    c->need = GM_NEVER;
    c->rebuilt_at = fresh ? step : GM_NEVER;
    c->go = 0;
    for (int q = 0; q < 3; ++q) { c->ke2[q] = 0.0; c->xi[q] = 0.0; }
    c->thermo_start = step;
    if (reset_all) {
        c->n_rebuilds = 0; c->sum_nn = 0; c->max_nn = 0; c->err = 0; c->n_glob_tiles = 0;
    }
}

// gm_set_integrator: the thermostat state starts afresh at the current time level
__global__ void k_thermo_reset(GmDev D, int parity)
{
    GmCtl *c = D.ctl;
    for (int q = 0; q < 3; ++q) { c->ke2[q] = 0.0; c->xi[q] = 0.0; }
    c->thermo_start = c->step[parity];
}

void gm_launch_thermo_reset(const GmDev &D, int parity, cudaStream_t st) { k_thermo_reset<<<1, 1, 0, st>>>(D, parity); }

void gm_launch_set_ctl(const GmDev &D, unsigned long long step, int reset_all, int parity, cudaStream_t st)
{
    k_set_ctl<<<1, 1, 0, st>>>(D, step, reset_all, parity);
}
