// The fused force kernel in its DENSE launch configuration (see the head of tc_kernels.cu): 4 CTAs x 3 warps per SM,
// 168 registers per thread, 320 cell records / 512 bodies staged per warp, tails in the lane mapping.  Same source,
// other constants (the TC_DENSE_* macros exist for tuning sweeps).
#ifndef TC_DENSE_WARPS
#define TC_DENSE_WARPS 3
#endif
#ifndef TC_DENSE_MINB
#define TC_DENSE_MINB 4
#endif
#ifndef TC_DENSE_CELLCAP
#define TC_DENSE_CELLCAP 320
#endif
#ifndef TC_DENSE_BODYCAP
#define TC_DENSE_BODYCAP 512
#endif
#ifndef TC_DENSE_UNROLL2_MAXK
#define TC_DENSE_UNROLL2_MAXK 2
#endif
#define TC_CFG_NS dense
#define TC_FORCES_ONLY 1
#define TC_WARPS TC_DENSE_WARPS
#define TC_MINB TC_DENSE_MINB
#define TC_CELLCAP TC_DENSE_CELLCAP
#define TC_BODYCAP TC_DENSE_BODYCAP
#define TC_UNROLL2_MAXK TC_DENSE_UNROLL2_MAXK
#include "tc_kernels.cu"
