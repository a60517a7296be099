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
    long long blocks = (cells + 255) / 256;
    if (blocks > 148ll * 32) blocks = 148ll * 32;      // grid-stride: a multiple of the SM count
    absorber_kernel<<<(unsigned)blocks, 256, 0, st>>>(p);
    return cudaGetLastError();
}
