// gm_force_dpd.cu -- the force / step / energy kernels of gm_force_impl.cuh for GM_PAIR_DPD (a6).
#include "gm_force_impl.cuh"

GM_DEFINE_PAIR_LAUNCH(gm_launch_force_dpd, GM_PAIR_DPD)
