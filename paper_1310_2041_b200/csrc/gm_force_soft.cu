// gm_force_soft.cu -- the kernels of gm_force_impl.cuh for harmonic repulsion, Eq. (2).
#include "gm_force_impl.cuh"

GM_DEFINE_PAIR_LAUNCH(gm_launch_force_harmonic, GM_PAIR_HARMONIC)
