// gm_npt.cuh -- state and launch wrappers of the Andersen barostat (f3: NPH / NPT; PAPER.md:L133 names the barostat,
// DESIGN.md reading c-31 gives the equations).  Nothing here is used by, or derived from, the CPU oracle.
//
// Andersen (1980): scaled coordinates rho_i = r_i / V^(1/3) with momenta pi_i, the volume V with momentum Pi,
//     H = sum pi_i^2 / (2 m_i V^(2/3)) + U(V^(1/3) rho) + Pi^2 / (2 M) + P_ext V.
// Device representation: the position arrays hold s_i = r_i / lambda, lambda = (V / V_0)^(1/3), i.e. positions in the box
// of gm_create -- cells, sort, neighbor build and the periodic images work on them unchanged; the velocity arrays hold
// c_i = lambda * v_i (v: physical velocity), which only a force changes: c' = lambda F / m.  One timestep is the symmetric
// product  pot(dt/2) kin(dt/2) pis(dt) kin(dt/2) pot(dt/2)  in leapfrog form (the two pot halves of neighboring steps merge):
//     k_npt_force:   F_i, virial W = sum r_ij . F_ij, and the sums S_cc = sum m c^2, S_cF = sum c . F, S_FF = sum F^2 / m
//     k_npt_update:  Pi += kick (W / 3V - P_ext);  c += kick lambda F / m;  S' = S_cc + 2 kick lambda S_cF + kick^2 lambda^2 S_FF
//                    Pi += dt/2 S' / (3 V lambda^2);  V' = V + dt Pi / M;  Pi += dt/2 S' / (3 V' lambda'^2)
//                    s += dt/2 (1 / lambda^2 + 1 / lambda'^2) c;   (NPT) Andersen collisions: c = lambda' sqrt(kT / m) g
// The sum of the new m c^2 follows from the three sums of the force kernel, so the piston needs no reduction between kick
// and drift: two kernels per timestep.
#pragma once
#include "gm_internal.cuh"

#define GM_DEV_ERR_BOX 32          // the box shrank below what the neighbor list of gm_create covers

// Lives in the tail of the energy scratch (GmDev::esum + (GM_ESUM_BLOCKS + 1) * 8); slots [parity] follow the position
// buffers; sum[2] is the scratch of force evaluations outside the time stepping (gm_compute_forces, gm_energies, ...)
#define GM_NPT_SLOTS 64            // the sums are spread over this many copies (warp w adds to copy w % 64): no hot atomic address
struct GmNpt {
    double V[2], Pi[2], lam[2];
    double p_ext, mass, vol0;
    double pad[7];
    double sum[3][GM_NPT_SLOTS][8];    // W, S_cc, S_cF, S_FF, pair PE, bond PE
};
#define GM_NPT_DOUBLES 2048
static_assert(sizeof(GmNpt) <= GM_NPT_DOUBLES * sizeof(double), "GmNpt outgrew its slot");

__host__ __device__ __forceinline__ GmNpt *gm_npt_state(const GmDev &D)
{
    return reinterpret_cast<GmNpt *>(D.esum + (size_t)(GM_ESUM_BLOCKS + 1) * 8);
}

void gm_launch_npt_init(const GmDev &D, int parity, double vol0, double V, double Pi, double p_ext, double mass, cudaStream_t st);
void gm_launch_npt_force(const GmParams &P, const GmDev &D, int parity, int probe, cudaStream_t st);
void gm_launch_npt_update(const GmParams &P, const GmDev &D, int parity, float kick, cudaStream_t st);
void gm_launch_npt_unpack(const GmParams &P, const GmDev &D, int parity, float *pos3, float *vel3, float *force3, int lagged,
                          cudaStream_t st);
void gm_launch_scale3(float *x, size_t count, float factor, cudaStream_t st);
