// fdtd_internal.h -- launch entry points of libfdtd_b200 (CUDA path only).
#pragma once
#include <cuda_runtime.h>

#include "../../include/fdtd.h"
#include "fdtd_types.h"

// implemented in naive_kernels.cu
cudaError_t launch_e_half_naive(const GridParams& g, cudaStream_t st);
cudaError_t launch_h_half_naive(const GridParams& g, cudaStream_t st);
cudaError_t launch_source_w(const GridParams& g, float w, cudaStream_t st);   // w = wave[t], looked up by the host

cudaError_t launch_monitor_naive(const GridParams& g, const MonitorParams& m, int isH, long long t, cudaStream_t st);   // row f4

// implemented in systolic_kernel.cu
int systolic_num_configs();
const SysConfig* systolic_config(int idx);
// returns cudaSuccess and launches `ctas` persistent CTAs of configuration cfg_idx
cudaError_t launch_systolic(int cfg_idx, const SysParams& p, int ctas, cudaStream_t st);
// set the max-dynamic-shared-memory attribute; *blocks_per_sm = resident CTAs per SM by the occupancy query
cudaError_t systolic_prepare(int cfg_idx, int* blocks_per_sm);

// implemented in systolic_reg.cu: the register-resident systolic kernel, tile 31x15x7 in a 32x16x8 box
size_t systolic_reg_smem(int coef);
int systolic_reg_threads();
cudaError_t systolic_reg_prepare(int coef, int* blocks_per_sm);
cudaError_t launch_systolic_reg(int coef, const SysParams& p, int ctas, cudaStream_t st);

// implemented in systolic_tma.cu: the TMA-staged systolic kernel (PEC grids, nx % 4 == 0), tile 31x15x7
size_t systolic_tma_smem(int coef);
int systolic_tma_threads();
void systolic_tma_boxes(int fld[3][3], int coef[3][3]);   // TMA box extents (x,y,z) of the z-plane, y-row and x-column shell pieces
cudaError_t systolic_tma_prepare(int coef, int* blocks_per_sm);
cudaError_t launch_systolic_tma(int coef, const SysParams& p, const TmaMaps& maps, int ctas, cudaStream_t st);
// implemented in systolic_tma_by8.cu: the same kernel for tile 31x7x7 (box 32x8x8), two CTAs per SM
size_t systolic_tma_smem_by8(int coef);
int systolic_tma_threads_by8();
void systolic_tma_boxes_by8(int fld[3][3], int coef[3][3]);
cudaError_t systolic_tma_prepare_by8(int coef, int* blocks_per_sm);
cudaError_t launch_systolic_tma_by8(int coef, const SysParams& p, const TmaMaps& maps, int ctas, cudaStream_t st);

// implemented in systolic_tma_h16.cu: the same kernel for binary16 field storage (GridParams::fld16), tile 31x15x7
size_t systolic_tma_smem_h16(int coef);
int systolic_tma_threads_h16();
void systolic_tma_boxes_h16(int fld[3][3], int coef[3][3]);
cudaError_t systolic_tma_prepare_h16(int coef, int* blocks_per_sm);
cudaError_t launch_systolic_tma_h16(int coef, const SysParams& p, const TmaMaps& maps, int ctas, cudaStream_t st);

// implemented in systolic_tma_lut.cu: the same kernel for material-index coefficients (GridParams::cidx), tile 31x15x7, coef = 1
size_t systolic_tma_smem_lut(int coef);
int systolic_tma_threads_lut();
void systolic_tma_boxes_lut(int fld[3][3], int coef[3][3]);
cudaError_t systolic_tma_prepare_lut(int coef, int* blocks_per_sm);
cudaError_t launch_systolic_tma_lut(int coef, const SysParams& p, const TmaMaps& maps, int ctas, cudaStream_t st);

// implemented in pad_kernels.cu: copies between the caller's arrays and the padded working copy (periodic images)
cudaError_t launch_pad_copy_in(const PadGeom& g, const PadArrays& a, cudaStream_t st);     // all padded cells <- images
cudaError_t launch_pad_ghost_fill(const PadGeom& g, const PadArrays& a, cudaStream_t st);  // ghost cells <- interior
cudaError_t launch_pad_copy_out(const PadGeom& g, const PadArrays& a, cudaStream_t st);    // interior -> caller

// implemented in absorber_kernels.cu: graded-conductivity update coefficients written to device arrays (row f3)
cudaError_t launch_absorber(const int n[3], float dt, const float* const eps[3], const int L[6], const float smax[6], int order,
                            float* const ca[3], float* const cb[3], cudaStream_t st);
