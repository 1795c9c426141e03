// cfs_kernels_static2d_b.cu -- the 2-D kernels compiled for one chain: BASELINE cfg 2
#define CFS_STATIC2D_PART b
#define CFS_STATIC2D_SIG chain_sig(T_AFFINE, T_SINUSOIDAL)
#include "cfs_kernels_static2d.inc"
