// gm_force_table.cu -- the kernels of gm_force_impl.cuh for the tabulated potential, Eqs. (11)-(12) / Algorithm 2
// (PAPER.md:L118-129, L458).
#include "gm_force_impl.cuh"

GM_DEFINE_PAIR_LAUNCH(gm_launch_force_table, GM_PAIR_TABLE)
