// gm_force.cu -- dispatch of the force / step / energy kernels (gm_force_impl.cuh) by pair style, and the
// instantiations for GM_PAIR_NONE and GM_PAIR_LJ.
#include "gm_force_impl.cuh"

GM_DEFINE_PAIR_LAUNCH(gm_launch_force_lj, GM_PAIR_LJ)

void gm_launch_force_dpd(const GmParams &, const GmDev &, int, int, float, float, int, cudaStream_t);
void gm_launch_force_harmonic(const GmParams &, const GmDev &, int, int, float, float, int, cudaStream_t);
void gm_launch_force_gauss(const GmParams &, const GmDev &, int, int, float, float, int, cudaStream_t);
void gm_launch_force_table(const GmParams &, const GmDev &, int, int, float, float, int, cudaStream_t);

void gm_launch_force(const GmParams &P, const GmDev &D, int mode, int parity, float kick, float kick_vt,
                     int lagged, cudaStream_t st)
{
    gm_launch_topo(P, D, parity, st);        // a7: angle + dihedral forces of this time level -> D.ftopo (no-op without them)
    switch (P.pair_style) {
    case GM_PAIR_LJ: gm_launch_force_lj(P, D, mode, parity, kick, kick_vt, lagged, st); break;
    case GM_PAIR_DPD: gm_launch_force_dpd(P, D, mode, parity, kick, kick_vt, lagged, st); break;
    case GM_PAIR_HARMONIC: gm_launch_force_harmonic(P, D, mode, parity, kick, kick_vt, lagged, st); break;
    case GM_PAIR_GAUSS: gm_launch_force_gauss(P, D, mode, parity, kick, kick_vt, lagged, st); break;
    case GM_PAIR_TABLE: gm_launch_force_table(P, D, mode, parity, kick, kick_vt, lagged, st); break;
    default: launch_force_b<GM_PAIR_NONE, true>(P, D, mode, parity, kick, kick_vt, lagged, st);
    }
}
