// cfs_kernels_static2d_a.cu -- the 2-D kernels compiled for one chain: BASELINE cfg 1
#define CFS_STATIC2D_PART a
#define CFS_STATIC2D_SIG chain_sig(T_SWIRL, T_SCALE)
#include "cfs_kernels_static2d.inc"
