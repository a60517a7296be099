// systolic_tma_lut.cu -- the TMA-staged systolic kernel for compressed coefficients (row f2): one material
// index (a byte) per cell and component in global memory and a (ca, cb) table, instead of six float arrays.  Same source
// as systolic_tma.cu (see there); only the coefficient shell (byte boxes, expansion through the table when a cell enters
// the chip) and the exported names differ.  Launched with coef = 1 only.
#define FDTD_COEF_LUT 1
#define FDTD_TMA_NAME(x) x##_lut
#include "systolic_tma.cu"
