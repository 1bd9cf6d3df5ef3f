// The fused force kernel in its DENSE launch configuration (see the head of tc_kernels.cu): 4 CTAs x 3 warps per SM,
// 168 registers per thread, 320 cell records / 512 bodies staged per warp.  Same source, other constants.
#define TC_CFG_NS dense
#define TC_FORCES_ONLY 1
#define TC_WARPS 3
#define TC_CELLCAP 320
#define TC_BODYCAP 512
#include "tc_kernels.cu"
