// systolic_tma_h16.cu -- the TMA-staged systolic kernel for binary16 field storage with f32 arithmetic (row f1,
// "utilizing 16-bit floating-point representations for the field values").  Same source as
// systolic_tma.cu (see there); only the storage type of the six field arrays, their TMA box geometry and the exported
// names differ.
#define FDTD_FLD16 1
#define FDTD_TMA_NAME(x) x##_h16
#include "systolic_tma.cu"
