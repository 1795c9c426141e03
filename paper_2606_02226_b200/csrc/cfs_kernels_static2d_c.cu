// cfs_kernels_static2d_c.cu -- the 2-D kernels compiled for one chain: PAPER Eq. 2
#define CFS_STATIC2D_PART c
#define CFS_STATIC2D_SIG chain_sig(T_STRETCH_COS, T_AFFINE)
#include "cfs_kernels_static2d.inc"
