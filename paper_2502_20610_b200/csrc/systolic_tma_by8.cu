// systolic_tma_by8.cu -- the TMA-staged systolic kernel built for a 32 x 8 x 8 box (tile 31x7x7), two CTAs per SM.
// Same source as systolic_tma.cu (see there); only the box height, the register split and the exported names differ.
#define FDTD_BY 8
#define FDTD_TMA_NAME(x) x##_by8
#include "systolic_tma.cu"
