// pad_kernels.cu -- the padded working copy of the grid on which the systolic kernel runs when an axis is periodic
// or nx is not a multiple of 4.
//
// The time-skewed tile schedule moves boundary values upwind -> downwind only; a periodic axis closes the
// chain of tiles into a ring whose members must advance in lock step through global memory.  Instead the ring is cut:
// the axis is extended by G ghost cells on either side, filled with the periodic images of the interior before each
// launch of T <= G steps, and runs as an open axis.  A wrong value at the open ends spreads inwards by one cell per step
// (E reads H one cell back, H reads E one cell ahead), so after T steps exactly the interior [G, G+n) is still exact --
// the halo of PAPER.md:79, Fig. 4, paid once per launch at the seam instead of once per subdomain and step.
// These kernels are plain copies (index wrap, no arithmetic of the method).
#include <cuda_fp16.h>

#include "fdtd_internal.h"

namespace {

constexpr int kThreads = 128;

__device__ __forceinline__ int wrap(int e, int G, int n)
{
    int s = (e - G) % n;
    return s < 0 ? s + n : s;
}

// one block per (row j,k of the padded grid, array); threads stride over x
template <typename T>
__global__ void __launch_bounds__(kThreads) pad_copy_in_kernel(PadGeom g, PadArrays a)
{
    const long long row = blockIdx.x;
    const int q = blockIdx.y;
    const int j = (int)(row % g.m[1]), k = (int)(row / g.m[1]);
    const int sj = g.G[1] ? wrap(j, g.G[1], g.n[1]) : j;
    const int sk = g.G[2] ? wrap(k, g.G[2], g.n[2]) : k;
    const T* __restrict__ src = reinterpret_cast<const T*>(a.usr[q]) + (long long)g.n[0] * (sj + (long long)g.n[1] * sk);
    T* __restrict__ dst = reinterpret_cast<T*>(a.ext) + (long long)q * a.stride + g.ldx * (j + (long long)g.m[1] * k);
    for (int i = threadIdx.x; i < g.ldx; i += kThreads) {
        T v = T(0.0f);                                    // the pitch padding beyond m[0] reads as "outside the grid"
        if (i < g.m[0]) v = src[g.G[0] ? wrap(i, g.G[0], g.n[0]) : i];
        dst[i] = v;
    }
}

// ghost cells <- their periodic image inside the interior of the same padded array (interior cells are skipped)
template <typename T>
__global__ void __launch_bounds__(kThreads) pad_ghost_fill_kernel(PadGeom g, PadArrays a)
{
    const long long row = blockIdx.x;
    const int q = blockIdx.y;
    const int j = (int)(row % g.m[1]), k = (int)(row / g.m[1]);
    const int sj = g.G[1] ? g.G[1] + wrap(j, g.G[1], g.n[1]) : j;
    const int sk = g.G[2] ? g.G[2] + wrap(k, g.G[2], g.n[2]) : k;
    const bool row_interior = (sj == j) & (sk == k);
    T* base = reinterpret_cast<T*>(a.ext) + (long long)q * a.stride;
    const T* src = base + g.ldx * (sj + (long long)g.m[1] * sk);
    T* dst = base + g.ldx * (j + (long long)g.m[1] * k);
    for (int i = threadIdx.x; i < g.m[0]; i += kThreads) {
        const int si = g.G[0] ? g.G[0] + wrap(i, g.G[0], g.n[0]) : i;
        if (!(row_interior && si == i)) dst[i] = src[si];
    }
}

template <typename T>
__global__ void __launch_bounds__(kThreads) pad_copy_out_kernel(PadGeom g, PadArrays a)
{
    const long long row = blockIdx.x;
    const int q = blockIdx.y;
    const int j = (int)(row % g.n[1]), k = (int)(row / g.n[1]);
    const T* __restrict__ src = reinterpret_cast<const T*>(a.ext) + (long long)q * a.stride + g.ldx * ((j + g.G[1]) + (long long)g.m[1] * (k + g.G[2])) + g.G[0];
    T* __restrict__ dst = reinterpret_cast<T*>(a.usr[q]) + (long long)g.n[0] * (j + (long long)g.n[1] * k);
    for (int i = threadIdx.x; i < g.n[0]; i += kThreads) dst[i] = src[i];
}

}  // namespace

cudaError_t launch_pad_copy_in(const PadGeom& g, const PadArrays& a, cudaStream_t st)
{
    if (a.elem16 == 2) pad_copy_in_kernel<unsigned char><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else if (a.elem16) pad_copy_in_kernel<__half><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else pad_copy_in_kernel<float><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    return cudaGetLastError();
}

cudaError_t launch_pad_ghost_fill(const PadGeom& g, const PadArrays& a, cudaStream_t st)
{
    if (a.elem16 == 2) pad_ghost_fill_kernel<unsigned char><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else if (a.elem16) pad_ghost_fill_kernel<__half><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else pad_ghost_fill_kernel<float><<<dim3((unsigned)((long long)g.m[1] * g.m[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    return cudaGetLastError();
}

cudaError_t launch_pad_copy_out(const PadGeom& g, const PadArrays& a, cudaStream_t st)
{
    if (a.elem16 == 2) pad_copy_out_kernel<unsigned char><<<dim3((unsigned)((long long)g.n[1] * g.n[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else if (a.elem16) pad_copy_out_kernel<__half><<<dim3((unsigned)((long long)g.n[1] * g.n[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    else pad_copy_out_kernel<float><<<dim3((unsigned)((long long)g.n[1] * g.n[2]), (unsigned)a.narr), kThreads, 0, st>>>(g, a);
    return cudaGetLastError();
}
