// absorber_kernels.cu -- adiabatic-absorber coefficient generator.
//
// PAPER.md:103 (section 4): the engine "does not use PMLs, but instead relies on the imaginary part of the permittivity
// to allow for the formation of adiabatic absorbers [5]": a conductivity that rises polynomially from zero over a layer
// in front of a wall (Oskooi et al. 2008).  DESIGN.md reading #14 fixes the formula; this kernel writes the six
// per-cell update-coefficient arrays of fdtd_set_coeffs straight into device memory (config 5's are 43 GB: they are
// generated where they are used).  One thread per cell, one statement per rounded operation: with -fmad=false the
// arrays are bit-identical to the fp32 CPU oracle's.
//
//   component E_a of cell g sits at s_q = g_q + 1/2 (q == a) or g_q (q != a) along axis q;  domain [0, n_q]
//   low layer of L cells:  u = (L - s)/L where s < L;   high layer:  u = (s - (n - L))/L where s > n - L
//   sigma_q = smax * u^p;  sigma = (sigma_x + sigma_y) + sigma_z
//   ca = (2 eps - sigma dt)/(2 eps + sigma dt),  cb = (2 dt)/(2 eps + sigma dt)
#include <stdint.h>

#include "fdtd_internal.h"

namespace {

struct AbsorberParams {
    int n[3];
    int L[6];          // x_lo x_hi y_lo y_hi z_lo z_hi, cells
    float smax[6];
    int order;
    float dt;
    const float* eps[3];   // NULL: 1
    float* ca[3];
    float* cb[3];
};

__device__ __forceinline__ float layer_sigma(const AbsorberParams& p, int q, int g, bool own)
{
    const float s = (float)g + (own ? 0.5f : 0.0f);
    float sig = 0.0f;
#pragma unroll
    for (int side = 0; side < 2; ++side) {
        const int L = p.L[2 * q + side];
        if (L <= 0) continue;
        const float fl = (float)L;
        float num;
        if (side == 0) {
            if (!(s < fl)) continue;
            num = fl - s;
        } else {
            const float edge = (float)(p.n[q] - L);
            if (!(s > edge)) continue;
            num = s - edge;
        }
        const float u = num / fl;
        float w = 1.0f;
        for (int i = 0; i < p.order; ++i) w = w * u;
        const float term = p.smax[2 * q + side] * w;
        sig = sig + term;
    }
    return sig;
}

__global__ void __launch_bounds__(256) absorber_kernel(const __grid_constant__ AbsorberParams p)
{
    const long long cells = (long long)p.n[0] * p.n[1] * p.n[2];
    const float dt2 = 2.0f * p.dt;
    for (long long idx = blockIdx.x * 256ll + threadIdx.x; idx < cells; idx += 256ll * gridDim.x) {
        const int i = (int)(idx % p.n[0]);
        const int j = (int)((idx / p.n[0]) % p.n[1]);
        const int k = (int)(idx / ((long long)p.n[0] * p.n[1]));
        const int g[3] = {i, j, k};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float sx = layer_sigma(p, 0, g[0], a == 0);
            const float sy = layer_sigma(p, 1, g[1], a == 1);
            const float sz = layer_sigma(p, 2, g[2], a == 2);
            const float sxy = sx + sy;
            const float sig = sxy + sz;
            const float e = p.eps[a] ? __ldg(p.eps[a] + idx) : 1.0f;
            const float e2 = 2.0f * e;
            const float sd = sig * p.dt;
            const float den = e2 + sd;
            const float num = e2 - sd;
            p.ca[a][idx] = num / den;
            p.cb[a][idx] = dt2 / den;
        }
    }
}

// The same arithmetic, four consecutive cells of a row per thread: 128-bit loads and stores, one index decomposition per
// group instead of one per cell (the one-cell kernel above spends more issue slots on 64-bit divisions than on the
// formula and reaches 0.31 of the 36 B/cell HBM roof).  Needs nx % 4 == 0 and 16-byte aligned arrays; every value is
// produced by the same sequence of rounded operations, so the output is bit-identical.
template <typename index_t>
__global__ void __launch_bounds__(256) absorber_kernel_x4(const __grid_constant__ AbsorberParams p)
{
    const int G = p.n[0] >> 2;                                     // groups per row
    const index_t groups = (index_t)G * p.n[1] * p.n[2];
    const float dt2 = 2.0f * p.dt;
    for (index_t q = blockIdx.x * (index_t)256 + threadIdx.x; q < groups; q += (index_t)256 * gridDim.x) {
        const index_t row = q / G;
        const int i0 = (int)(q - row * G) << 2;
        const int k = (int)(row / p.n[1]);
        const int j = (int)(row - (index_t)k * p.n[1]);
        const long long idx = (long long)q << 2;
        float sx[2][4] = {{0.0f, 0.0f, 0.0f, 0.0f}, {0.0f, 0.0f, 0.0f, 0.0f}};       // [own][cell]
        // a low layer of L cells reaches cells g < L, a high one cells g >= n - L (either Yee offset): most groups lie in
        // neither and keep the 0 that layer_sigma would return
        if (i0 < p.L[0] || i0 + 3 >= p.n[0] - p.L[1]) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                sx[0][c] = layer_sigma(p, 0, i0 + c, false);
                sx[1][c] = layer_sigma(p, 0, i0 + c, true);
            }
        }
        const float sy[2] = {layer_sigma(p, 1, j, false), layer_sigma(p, 1, j, true)};
        const float sz[2] = {layer_sigma(p, 2, k, false), layer_sigma(p, 2, k, true)};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float e[4] = {1.0f, 1.0f, 1.0f, 1.0f};
            if (p.eps[a]) {
                const float4 v = __ldcs(reinterpret_cast<const float4*>(p.eps[a] + idx));
                e[0] = v.x; e[1] = v.y; e[2] = v.z; e[3] = v.w;
            }
            float ca[4], cb[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float sxy = sx[a == 0][c] + sy[a == 1];
                const float sig = sxy + sz[a == 2];
                const float e2 = 2.0f * e[c];
                const float sd = sig * p.dt;
                const float den = e2 + sd;
                const float num = e2 - sd;
                ca[c] = num / den;
                cb[c] = dt2 / den;
            }
            __stcs(reinterpret_cast<float4*>(p.ca[a] + idx), make_float4(ca[0], ca[1], ca[2], ca[3]));
            __stcs(reinterpret_cast<float4*>(p.cb[a] + idx), make_float4(cb[0], cb[1], cb[2], cb[3]));
        }
    }
}

bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

}  // namespace

cudaError_t launch_absorber(const int n[3], float dt, const float* const eps[3], const int L[6], const float smax[6], int order,
                            float* const ca[3], float* const cb[3], cudaStream_t st)
{
    AbsorberParams p;
    for (int a = 0; a < 3; ++a) {
        p.n[a] = n[a];
        p.eps[a] = eps ? eps[a] : nullptr;
        p.ca[a] = ca[a];
        p.cb[a] = cb[a];
    }
    for (int f = 0; f < 6; ++f) {
        p.L[f] = L[f];
        p.smax[f] = smax[f];
    }
    p.order = order;
    p.dt = dt;
    const long long cells = (long long)n[0] * n[1] * n[2];
    bool x4 = n[0] % 4 == 0;
    for (int a = 0; a < 3; ++a) x4 = x4 && aligned16(p.eps[a]) && aligned16(p.ca[a]) && aligned16(p.cb[a]);
    const long long work = x4 ? cells / 4 : cells;
    long long blocks = (work + 255) / 256;
    if (blocks > 148ll * 32) blocks = 148ll * 32;      // grid-stride: a multiple of the SM count
    if (!x4) absorber_kernel<<<(unsigned)blocks, 256, 0, st>>>(p);
    else if (work + 148ll * 32 * 256 < (1ll << 31)) absorber_kernel_x4<unsigned int><<<(unsigned)blocks, 256, 0, st>>>(p);
    else absorber_kernel_x4<unsigned long long><<<(unsigned)blocks, 256, 0, st>>>(p);
    return cudaGetLastError();
}
