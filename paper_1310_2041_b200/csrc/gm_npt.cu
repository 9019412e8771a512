// gm_npt.cu -- f3: Andersen barostat, NPH and NPT (reading c-31; scheme in gm_npt.cuh).
// Plain kernels, one thread per bead over the 32-bit rows of the neighbor list (an NPT system runs without tile windows):
// this path is about the ensemble, the tuned fixed-box kernels of gm_force_impl.cuh are not touched by it.
#include "gm_npt.cuh"
#include "gm_force_impl.cuh"

#define NPT_BLOCK 128
#ifndef NPT_FBLOCK
#define NPT_FBLOCK 32            // threads per CTA of the force kernel (no block-level step in it): one-warp CTAs, 32 per SM,
#define NPT_FMINB 32             // as the short-list step kernel (measured on C3: 103.1 us per timestep; 64 x 16 and 128 x 8 the same)
#endif

// sum of v[0..NQ) over the warp -> one of the GM_NPT_SLOTS copies of the sums (lane q adds quantity q: one double atomic
// per warp and quantity, spread over 64 x NQ addresses; no block barrier, a warp leaves when it is done)
template <int NQ>
__device__ __forceinline__ void npt_warp_add(double (&v)[NQ], double (*dst)[8])
{
    const int lane = threadIdx.x & 31;
    const int warp = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    double mine = 0.0;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        double x = v[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if (lane == q) mine = x;
    }
    if (lane < NQ) atomicAdd(&dst[warp & (GM_NPT_SLOTS - 1)][lane], mine);
}

// the 8 sums of slot array `src`: every thread of the block gets all of them, summed in an order that depends on nothing
// but the slot layout (all blocks derive bit-identical piston scalars)
__device__ __forceinline__ void npt_sums(const double (*src)[8], double (&out)[8])
{
    __shared__ double sh[8];
    if (threadIdx.x < 8) {
        double x = 0.0;
        for (int c = 0; c < GM_NPT_SLOTS; ++c) x += src[c][threadIdx.x];
        sh[threadIdx.x] = x;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 8; ++q) out[q] = sh[q];
}

// Eq. (1) over row i of the neighbor list at the real distances lambda * s; e0: the row's first quad (already loaded).
// MI: minimum-image differences (a warp with a bead near a face), else plain ones.  The four gathers of a quad are
// issued together; slots past NN hold the far-away pad bead, which the branch-free term turns into zero.
template <bool NT1, bool MI>
__device__ __forceinline__ void npt_pairs(const GmParams &P, const GmDev &D, const Src &S, int i, const float4 pi, int nn,
                                          int4 e0, float lam, float lam2, float &fx, float &fy, float &fz, float &w,
                                          float &pe_pair)
{
    const int ti = __float_as_int(pi.w);
    const int4 *__restrict__ t = nl_row(P, D, i);
    const GmPair p0 = P.pair[0];
    int4 en = e0;
    for (int q = 0; 4 * q < nn; ++q) {
        const int4 e = en;
        if (4 * (q + 1) < nn) en = t[(q + 1) * 32];
        float4 pj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) pj[u] = __ldg(S.pos + quad_get(e, u));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float dx, dy, dz;
            if (MI) {
                dx = gm_min_image(pi.x, pj[u].x, P.half[0]);
                dy = gm_min_image(pi.y, pj[u].y, P.half[1]);
                dz = gm_min_image(pi.z, pj[u].z, P.half[2]);
            } else {
                dx = pi.x - pj[u].x; dy = pi.y - pj[u].y; dz = pi.z - pj[u].z;
            }
            const float r2 = lam2 * (dx * dx + dy * dy + dz * dz);
            GmPair k = p0;
            if (!NT1) k = P.pair[ti * P.n_types + __float_as_int(pj[u].w)];
            // Eq. (1): F_i = r^-2 r^-6 (48 eps s^12 r^-6 - 24 eps s^6) r_ij, r_ij = lambda s_ij
            const bool in = r2 < k.c0;
            const float r2i = gm_rcp(r2);
            const float r6i = r2i * r2i * r2i;
            const float fs = in ? r2i * r6i * (k.c1 * r6i - k.c2) : 0.0f;
            const float fl = fs * lam;
            fx += fl * dx; fy += fl * dy; fz += fl * dz;
            w += in ? fs * r2 : 0.0f;
            pe_pair += in ? r6i * (k.c1 * (1.0f / 12.0f) * r6i - k.c2 * (1.0f / 6.0f)) - k.c3 : 0.0f;
        }
    }
}

// Forces at the real distances lambda * s (Eq. 1 pairs from the neighbor list, bonds from BL), the virial and the sums
// the piston needs.  D.frc[i] = (F, the bead's half share of the potential energy).
template <bool NT1, int BOND, bool PAIRS>
__global__ void __launch_bounds__(NPT_FBLOCK, NPT_FMINB)
k_npt_force(const __grid_constant__ GmParams P, GmDev D, int parity, int probe)
{
    GmNpt *N = gm_npt_state(D);
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    const float lam = (float)N->lam[parity];
    const float lam2 = lam * lam;
    const int i = blockIdx.x * NPT_FBLOCK + threadIdx.x;
    double acc[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    if (i < P.n) {
        // every stream of the bead is requested before anything is used
        const float4 pi = S.pos[i];
        const int4 e0 = PAIRS ? nl_row(P, D, i)[0] : make_int4(0, 0, 0, 0);
        const int nn = PAIRS ? D.nn[i] : 0;
        const float4 c = S.vel[i];
        float fx = 0.f, fy = 0.f, fz = 0.f, w = 0.f, pe_pair = 0.f, pe_bond = 0.f;
        if (PAIRS) {
            // a bead further than r_list + skin (scaled) from every face has no listed partner across the boundary:
            // plain differences; decided per warp so that a warp runs one of the two loops
            const float m = P.edge_margin;
            const bool interior = fabsf(pi.x) < P.half[0] - m && fabsf(pi.y) < P.half[1] - m && fabsf(pi.z) < P.half[2] - m;
            if (__all_sync(__activemask(), interior)) npt_pairs<NT1, false>(P, D, S, i, pi, nn, e0, lam, lam2, fx, fy, fz, w, pe_pair);
            else npt_pairs<NT1, true>(P, D, S, i, pi, nn, e0, lam, lam2, fx, fy, fz, w, pe_pair);
        }
        if (BOND != GM_BOND_NONE) {
            for (int b = 0; b < P.max_bonds; ++b) {
                const int e = __ldg(D.bl + i + (size_t)b * P.ns);
                if (e < 0) continue;
                const int bt = (unsigned)e >> GM_BOND_SHIFT;
                const float4 pj = __ldg(S.pos + (e & GM_BOND_MASK));
                const float dx = gm_min_image(pi.x, pj.x, P.half[0]);
                const float dy = gm_min_image(pi.y, pj.y, P.half[1]);
                const float dz = gm_min_image(pi.z, pj.z, P.half[2]);
                const float r2 = lam2 * (dx * dx + dy * dy + dz * dz);
                const float kb = P.bond_k[bt], r0 = P.bond_r0[bt];
                float fs;
                if (BOND == GM_BOND_FENE) {
                    const float q = 1.0f - r2 * P.bond_c[bt];
                    if (!(q > 0.0f)) { atomicOr(&D.ctl->err, GM_DEV_ERR_OVERSTRETCH); continue; }
                    fs = -kb / q;
                    pe_bond += -0.5f * kb * r0 * r0 * logf(q);
                } else if (BOND == GM_BOND_TABLE) {
                    const int point = (int)(r2 * kb);
                    if (!(point < P.bond_table_points)) { atomicOr(&D.ctl->err, GM_DEV_ERR_OVERSTRETCH); continue; }
                    const float4 cf = __ldg(P.btable + bt * P.bond_table_points + point);
                    const float d = r2 - (float)point * r0;
                    fs = -2.0f * (cf.y + d * (2.0f * cf.z + 3.0f * cf.w * d));
                    pe_bond += cf.x + d * (cf.y + d * (cf.z + d * cf.w));
                } else {
                    const float r = sqrtf(r2);
                    fs = (r0 == 0.0f) ? -2.0f * kb : ((r > 0.0f) ? -2.0f * kb * (1.0f - r0 / r) : 0.0f);
                    pe_bond += kb * (r - r0) * (r - r0);
                }
                const float fl = fs * lam;
                fx += fl * dx; fy += fl * dy; fz += fl * dz;
                w += fs * r2;
            }
        }
        // a7: angle and dihedral forces were evaluated on the scaled coordinates (gm_topo.cu); an angle does not change
        // under a uniform scaling, so U is the same, F = -dU/dr = (1 / lambda) (-dU/ds), and the virial gets nothing
        if (P.max_angles + P.max_dihedrals > 0) {
            const float4 ft = D.ftopo[i];
            const float il = 1.0f / lam;
            fx += il * ft.x; fy += il * ft.y; fz += il * ft.z;
            pe_bond += 2.0f * ft.w;
        }
        D.frc[i] = make_float4(fx, fy, fz, 0.5f * (pe_pair + pe_bond));
        const float im = 1.0f / c.w;
        acc[0] = 0.5 * (double)w;
        acc[1] = (double)c.w * ((double)c.x * c.x + (double)c.y * c.y + (double)c.z * c.z);
        acc[2] = (double)c.x * fx + (double)c.y * fy + (double)c.z * fz;
        acc[3] = (double)im * ((double)fx * fx + (double)fy * fy + (double)fz * fz);
        acc[4] = 0.5 * (double)pe_pair;
        acc[5] = 0.5 * (double)pe_bond;
    }
    npt_warp_add<6>(acc, N->sum[probe ? 2 : parity]);
}

// Piston, kick, drift, collisions, displacement test (scheme in gm_npt.cuh).  Every thread derives the same scalars from
// the control block; thread 0 of block 0 stores the new volume and piston momentum in the slots of the next time level.
__global__ void __launch_bounds__(NPT_BLOCK)
k_npt_update(const __grid_constant__ GmParams P, GmDev D, int parity, float kick)
{
    GmNpt *N = gm_npt_state(D);
    const unsigned long long step = D.ctl->step[parity];
    const Src S = current_src(D, parity, step);
    const double dt = (double)P.dt, kk = (double)kick;
    const double V = N->V[parity], lam = N->lam[parity];
    double sm[8];
    npt_sums(N->sum[parity], sm);
    double Pi = N->Pi[parity] + kk * (sm[0] / (3.0 * V) - N->p_ext);
    const double s_new = sm[1] + 2.0 * kk * lam * sm[2] + kk * kk * lam * lam * sm[3];
    Pi += 0.5 * dt * s_new / (3.0 * V * lam * lam);
    const double Vn = V + dt * Pi / N->mass;
    const double lamn = cbrt(Vn / N->vol0);
    Pi += 0.5 * dt * s_new / (3.0 * Vn * lamn * lamn);
    // the list holds every pair with s < r_list; a pair outside it stays beyond r_cut_max while both beads moved less than
    // (r_list - r_cut_max / lambda') / 2 in scaled coordinates since the build
    const float r_list = sqrtf(P.r_list2);
    const float rc_max = r_list - 2.0f * sqrtf(P.half_skin2);
    const float thr = 0.5f * (r_list - rc_max / (float)lamn);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        D.ctl->step[parity ^ 1] = step + 1;
        N->V[parity ^ 1] = Vn; N->Pi[parity ^ 1] = Pi; N->lam[parity ^ 1] = lamn;
        if (!(Vn > 0.0) || !(thr > 0.0f)) atomicOr(&D.ctl->err, GM_DEV_ERR_BOX);
        if (P.sfc_period > 0 && D.ctl->rebuilt_at != GM_NEVER &&
            step + 1 - D.ctl->rebuilt_at >= (unsigned long long)P.sfc_period)
            raise_rebuild(D, step);
    }
    if (blockIdx.x == 0)                    // the slots of the next time level (nobody reads or adds to them in this launch)
        for (int q = threadIdx.x; q < GM_NPT_SLOTS * 8; q += NPT_BLOCK) (&N->sum[parity ^ 1][0][0])[q] = 0.0;
    const int i = blockIdx.x * NPT_BLOCK + threadIdx.x;
    if (i >= P.n) return;
    const float4 pi = S.pos[i];
    const float4 c = S.vel[i];
    const float4 f = D.frc[i];
    const float4 rf = D.ref[i];
    const float kl = (float)(kk * lam) / c.w;
    float cx = c.x + kl * f.x, cy = c.y + kl * f.y, cz = c.z + kl * f.z;
    const float drift = (float)(0.5 * dt * (1.0 / (lam * lam) + 1.0 / (lamn * lamn)));
    const float x = pi.x + drift * cx, y = pi.y + drift * cy, z = pi.z + drift * cz;
    if (P.integrator == GM_NPT_ANDERSEN) {
        float ux = cx, uy = cy, uz = cz;
        andersen_collide(P, S, i, step, c.w, ux, uy, uz);
        if (ux != cx || uy != cy || uz != cz) {         // hit: a fresh Maxwell velocity v, stored as c = lambda' v
            cx = (float)lamn * ux; cy = (float)lamn * uy; cz = (float)lamn * uz;
        }
    }
    D.vel[i] = make_float4(cx, cy, cz, c.w);
    D.pos[parity ^ 1][i] = make_float4(x, y, z, pi.w);
    const float dx = x - rf.x, dy = y - rf.y, dz = z - rf.z;
    if (!(dx * dx + dy * dy + dz * dz <= thr * thr)) raise_rebuild(D, step);
}

// tag-order output in real units: r = lambda s (wrapped), v = (c + dt/2 lambda F / m) / lambda, F
__global__ void __launch_bounds__(256)
k_npt_unpack(const __grid_constant__ GmParams P, GmDev D, int parity, float *__restrict__ pos3, float *__restrict__ vel3,
             float *__restrict__ force3, int lagged)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n) return;
    const Src S = current_src(D, parity, D.ctl->step[parity]);
    const float lam = (float)gm_npt_state(D)->lam[parity];
    const int t = S.tag[i];
    if (pos3) {
        const float4 p = S.pos[i];
        pos3[3 * t + 0] = lam * gm_wrap(p.x, P.half[0], P.box[0]);
        pos3[3 * t + 1] = lam * gm_wrap(p.y, P.half[1], P.box[1]);
        pos3[3 * t + 2] = lam * gm_wrap(p.z, P.half[2], P.box[2]);
    }
    const float4 f = D.frc[i];
    if (vel3) {
        float4 c = S.vel[i];
        if (lagged) {
            const float h = 0.5f * P.dt * lam / c.w;
            c.x += h * f.x; c.y += h * f.y; c.z += h * f.z;
        }
        vel3[3 * t + 0] = c.x / lam; vel3[3 * t + 1] = c.y / lam; vel3[3 * t + 2] = c.z / lam;
    }
    if (force3) { force3[3 * t + 0] = f.x; force3[3 * t + 1] = f.y; force3[3 * t + 2] = f.z; }
}

__global__ void k_npt_init(GmDev D, int parity, double vol0, double V, double Pi, double p_ext, double mass)
{
    GmNpt *N = gm_npt_state(D);
    for (int b = 0; b < 2; ++b) { N->V[b] = V; N->Pi[b] = Pi; N->lam[b] = cbrt(V / vol0); }
    for (int b = 0; b < 3; ++b)
        for (int c = 0; c < GM_NPT_SLOTS; ++c)
            for (int q = 0; q < 8; ++q) N->sum[b][c][q] = 0.0;
    N->p_ext = p_ext; N->mass = mass; N->vol0 = vol0;
    (void)parity;
}

__global__ void __launch_bounds__(256) k_scale3(float *__restrict__ x, size_t count, float factor)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) x[i] *= factor;
}

void gm_launch_npt_init(const GmDev &D, int parity, double vol0, double V, double Pi, double p_ext, double mass, cudaStream_t st)
{
    k_npt_init<<<1, 1, 0, st>>>(D, parity, vol0, V, Pi, p_ext, mass);
}

template <bool NT1, int BOND>
static void npt_force_p(const GmParams &P, const GmDev &D, int parity, int probe, cudaStream_t st)
{
    const int nb = (P.n + NPT_FBLOCK - 1) / NPT_FBLOCK;
    if (P.pair_style == GM_PAIR_LJ) k_npt_force<NT1, BOND, true><<<nb, NPT_FBLOCK, 0, st>>>(P, D, parity, probe);
    else k_npt_force<NT1, BOND, false><<<nb, NPT_FBLOCK, 0, st>>>(P, D, parity, probe);
}

template <bool NT1>
static void npt_force_b(const GmParams &P, const GmDev &D, int parity, int probe, cudaStream_t st)
{
    const int bond = (P.max_bonds > 0) ? P.bond_style : GM_BOND_NONE;
    if (bond == GM_BOND_FENE) npt_force_p<NT1, GM_BOND_FENE>(P, D, parity, probe, st);
    else if (bond == GM_BOND_HARMONIC) npt_force_p<NT1, GM_BOND_HARMONIC>(P, D, parity, probe, st);
    else if (bond == GM_BOND_TABLE) npt_force_p<NT1, GM_BOND_TABLE>(P, D, parity, probe, st);
    else npt_force_p<NT1, GM_BOND_NONE>(P, D, parity, probe, st);
}

// probe != 0: a force evaluation outside the time stepping; its sums go to the scratch slot, cleared here first
void gm_launch_npt_force(const GmParams &P, const GmDev &D, int parity, int probe, cudaStream_t st)
{
    if (probe) cudaMemsetAsync(gm_npt_state(D)->sum[2], 0, GM_NPT_SLOTS * 8 * sizeof(double), st);
    gm_launch_topo(P, D, parity, st);        // angle + dihedral forces of this time level -> D.ftopo (no-op without them)
    if (P.n_types == 1) npt_force_b<true>(P, D, parity, probe, st);
    else npt_force_b<false>(P, D, parity, probe, st);
}

void gm_launch_npt_update(const GmParams &P, const GmDev &D, int parity, float kick, cudaStream_t st)
{
    k_npt_update<<<(P.n + NPT_BLOCK - 1) / NPT_BLOCK, NPT_BLOCK, 0, st>>>(P, D, parity, kick);
}

void gm_launch_npt_unpack(const GmParams &P, const GmDev &D, int parity, float *pos3, float *vel3, float *force3, int lagged,
                          cudaStream_t st)
{
    k_npt_unpack<<<(P.n + 255) / 256, 256, 0, st>>>(P, D, parity, pos3, vel3, force3, lagged);
}

void gm_launch_scale3(float *x, size_t count, float factor, cudaStream_t st)
{
    if (count) k_scale3<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(x, count, factor);
}
