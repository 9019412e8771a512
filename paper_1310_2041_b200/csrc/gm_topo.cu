// gm_topo.cu -- angle and dihedral forces from per-particle tables.
//
// "For angles and torsions, we store them with the same form as bonds, except that the position (side or
// middle) of the target particle in an angle or a dihedral needs to be indicated.  Although the force of a bond will be
// computed twice (three times for an angle and four times for a torsion) ... it casts the computation well into parallel
// mode for separated threads".  One thread owns one bead and sums the forces of all angles and dihedrals it is a member
// of: no atomics.  Potentials: Eq. (8) U = k (theta - theta0)^2, Eq. (9) U = k (cos theta - cos theta0)^2, Eq. (10)
// U = k [1 + cos(n phi - delta)] (L103-114); theta is the angle at the middle bead (pi = straight), phi = 0 for cis
// (readings c-26, c-27).
//
// The tables stay in TAG order (they are never permuted by the SFC sort): thread t finds its bead and its partners
// through rtag[].  The result goes to ftopo[slot] (force, and the bead's share of the energy: a third of an angle, a
// quarter of a dihedral) and is added by the fused force + integrate kernels, which run right after.
#include "gm_internal.cuh"

__device__ __forceinline__ float3 mi3(const float4 a, const float4 b, const GmParams &P)
{
    return make_float3(gm_min_image(a.x, b.x, P.half[0]), gm_min_image(a.y, b.y, P.half[1]), gm_min_image(a.z, b.z, P.half[2]));
}

__device__ __forceinline__ float dot3(const float3 a, const float3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

__device__ __forceinline__ float3 cross3(const float3 a, const float3 b)
{
    return make_float3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}

__global__ void __launch_bounds__(128)
k_topo(const __grid_constant__ GmParams P, GmDev D, int parity)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= P.n) return;
    const Src S = current_src(D, parity, D.ctl->step[parity]);
    const int *__restrict__ rtag = D.rtag;
    const size_t ns = (size_t)P.ns;
    const int slot = rtag[t];
    const float4 own = S.pos[slot];
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f;
    for (int k = 0; k < P.max_angles; ++k) {
        const int4 e = D.at[k * ns + t];
        if (e.x < 0) break;                               // rows are filled from the top
        const float4 pa = S.pos[rtag[e.x]], pb = S.pos[rtag[e.y]];
        // members in order (i, j, k), j the middle bead; e.z = own position
        const float4 ri = e.z == 0 ? own : pa;
        const float4 rj = e.z == 1 ? own : (e.z == 0 ? pa : pb);
        const float4 rk = e.z == 2 ? own : pb;
        const float3 a = mi3(ri, rj, P), b = mi3(rk, rj, P);
        const float ia = rsqrtf(dot3(a, a)), ib = rsqrtf(dot3(b, b));
        const float c = fminf(1.0f, fmaxf(-1.0f, dot3(a, b) * ia * ib));
        const float kk = P.angle_k[e.w];
        float dudc;
        if (P.angle_style == GM_ANGLE_HARMONIC) {         // Eq. (8)
            // sin(theta) from the cross product and theta from atan2: 1 - c^2 and acos(c) lose their digits in fp32
            // near a straight angle, where the force 2 k (theta - theta0) / |a| is perfectly regular
            const float3 x = cross3(a, b);
            const float sn = fmaxf(sqrtf(dot3(x, x)) * ia * ib, 1e-12f);
            const float th = atan2f(sn, c);
            const float d = th - P.angle_t0[e.w];
            pe += kk * d * d * (1.0f / 3.0f);
            dudc = -2.0f * kk * d / sn;
        } else if (P.angle_style == GM_ANGLE_TABLE) {     // Eq. (12) with x = theta
            const float3 x = cross3(a, b);
            const float sn = fmaxf(sqrtf(dot3(x, x)) * ia * ib, 1e-12f);
            const float th = atan2f(sn, c);
            const int np = P.angle_table_points;
            const float h = 3.14159265358979323846f / (float)np;
            const int point = min((int)(th / h), np - 1);
            const float4 cf = __ldg(P.atable + e.w * np + point);
            const float d = th - (float)point * h;
            pe += (cf.x + d * (cf.y + d * (cf.z + d * cf.w))) * (1.0f / 3.0f);
            dudc = -(cf.y + d * (2.0f * cf.z + 3.0f * cf.w * d)) / sn;
        } else {                                          // Eq. (9)
            const float d = c - P.angle_c0[e.w];
            pe += kk * d * d * (1.0f / 3.0f);
            dudc = 2.0f * kk * d;
        }
        // d cos / d r_i = (b^ - c a^) / |a|,  d cos / d r_k = (a^ - c b^) / |b|,  middle bead: minus their sum
        const float3 gi = make_float3((b.x * ib - c * a.x * ia) * ia, (b.y * ib - c * a.y * ia) * ia, (b.z * ib - c * a.z * ia) * ia);
        const float3 gk = make_float3((a.x * ia - c * b.x * ib) * ib, (a.y * ia - c * b.y * ib) * ib, (a.z * ia - c * b.z * ib) * ib);
        float3 g;
        if (e.z == 0) g = gi;
        else if (e.z == 2) g = gk;
        else g = make_float3(-gi.x - gk.x, -gi.y - gk.y, -gi.z - gk.z);
        fx -= dudc * g.x; fy -= dudc * g.y; fz -= dudc * g.z;
    }
    for (int k = 0; k < P.max_dihedrals; ++k) {
        const int4 e = D.dt[k * ns + t];
        if (e.x < 0) break;
        const int pos = e.w & 3, ty = e.w >> 2;
        const float4 q0 = S.pos[rtag[e.x]], q1 = S.pos[rtag[e.y]], q2 = S.pos[rtag[e.z]];
        // members in order (i, j, k, l): the three partners fill the positions the owner does not hold
        const float4 ri = pos == 0 ? own : q0;
        const float4 rj = pos == 1 ? own : (pos == 0 ? q0 : q1);
        const float4 rk = pos == 2 ? own : (pos == 3 ? q2 : q1);
        const float4 rl = pos == 3 ? own : q2;
        const float3 b1 = mi3(rj, ri, P), b2 = mi3(rk, rj, P), b3 = mi3(rl, rk, P);
        const float3 n1 = cross3(b1, b2), n2 = cross3(b2, b3);
        const float n1s = dot3(n1, n1), n2s = dot3(n2, n2), b2s = dot3(b2, b2);
        if (n1s < 1e-20f || n2s < 1e-20f) continue;       // three beads in line: phi undefined, no force
        const float l2 = sqrtf(b2s);
        const float phi = atan2f(l2 * dot3(b1, n2), dot3(n1, n2));
        float dudphi;
        if (P.dihedral_table_points > 0) {                // Eq. (12) with x = phi, grid point k at -pi + k h
            const int np = P.dihedral_table_points;
            const float h = 6.28318530717958647692f / (float)np;
            const float x = phi + 3.14159265358979323846f;
            const int point = min(max((int)(x / h), 0), np - 1);
            const float4 cf = __ldg(P.dtable + ty * np + point);
            const float d = x - (float)point * h;
            pe += (cf.x + d * (cf.y + d * (cf.z + d * cf.w))) * 0.25f;
            dudphi = cf.y + d * (2.0f * cf.z + 3.0f * cf.w * d);
        } else {
            const float arg = (float)P.dih_n[ty] * phi - P.dih_delta[ty];
            float sn, cs;
            sincosf(arg, &sn, &cs);
            pe += P.dih_k[ty] * (1.0f + cs) * 0.25f;
            dudphi = -P.dih_k[ty] * (float)P.dih_n[ty] * sn;
        }
        const float wi = -l2 / n1s, wl = l2 / n2s;        // d phi / d r_i = wi n1,  d phi / d r_l = wl n2
        const float s12 = dot3(b1, b2) / b2s, s32 = dot3(b3, b2) / b2s;
        float ci, cl;                                     // d phi / d r_own = ci wi n1 + cl wl n2
        if (pos == 0) { ci = 1.0f; cl = 0.0f; }
        else if (pos == 3) { ci = 0.0f; cl = 1.0f; }
        else if (pos == 1) { ci = -(1.0f + s12); cl = s32; }
        else { ci = s12; cl = -(1.0f + s32); }
        const float u = ci * wi, v = cl * wl;
        fx -= dudphi * (u * n1.x + v * n2.x); fy -= dudphi * (u * n1.y + v * n2.y); fz -= dudphi * (u * n1.z + v * n2.z);
    }
    D.ftopo[slot] = make_float4(fx, fy, fz, pe);
}

void gm_launch_topo(const GmParams &P, const GmDev &D, int parity, cudaStream_t st)
{
    if (P.max_angles <= 0 && P.max_dihedrals <= 0) return;
    k_topo<<<(P.n + 127) / 128, 128, 0, st>>>(P, D, parity);
}
