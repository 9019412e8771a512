// gm_force_gauss.cu -- the kernels of gm_force_impl.cuh for Gaussian repulsion, Eq. (3).
#include "gm_force_impl.cuh"

GM_DEFINE_PAIR_LAUNCH(gm_launch_force_gauss, GM_PAIR_GAUSS)
