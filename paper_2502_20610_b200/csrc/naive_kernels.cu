// naive_kernels.cu -- the internal baseline: one HBM-bound kernel per half-step.
//
// This is the B200 version of the paper's "very straightforward" implementation (section 2):
// every cell is loaded, updated once and stored, with a kernel boundary (= grid-wide barrier, PAPER.md:61
// item 1) between the E and the H half-step.  Per cell-update it moves 72 B of HBM with uniform coefficients
// (12 loads + 6 stores of 4 B: the paper's "6 memory operations" per component) and 96 B with
// the six coefficient arrays.
//
// Mapping: the (x,y) plane is flattened (the layout is x-fastest with no padding, so a plane is one
// contiguous run); a thread owns VEC consecutive x cells (float4 when nx % 4 == 0) of one (x,y) column and
// marches ZC planes in z, carrying the z-neighbour plane in registers so that it is read from memory once.
// y- and x-neighbours come through L1/L2 (the same CTA, or its neighbour, has just loaded those lines).
//
// Arithmetic: the expression tree of eq. (1) with coefficients, one rounding per operation when compiled
// with -fmad=false (then bit-identical to the fp32 oracle); the default build lets ptxas contract mul+add.
#include <cuda_fp16.h>

#include "fdtd_internal.h"
#include "yee_update.h"

namespace {

constexpr int kThreads = 256;
constexpr int kZChunk = 16;

template <int VEC>
__device__ __forceinline__ void ldv(const float* __restrict__ p, float (&v)[VEC])
{
    if constexpr (VEC == 4) {
        const float4 t = *reinterpret_cast<const float4*>(p);
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    } else {
#pragma unroll
        for (int q = 0; q < VEC; ++q) v[q] = p[q];
    }
}

template <int VEC>
__device__ __forceinline__ void stv(float* __restrict__ p, const float (&v)[VEC])
{
    if constexpr (VEC == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    } else {
#pragma unroll
        for (int q = 0; q < VEC; ++q) p[q] = v[q];
    }
}

// binary16 field storage (row f1): exact conversion to f32 on load, round-to-nearest-even on store
template <int VEC>
__device__ __forceinline__ void ldv(const __half* __restrict__ p, float (&v)[VEC])
{
    if constexpr (VEC == 4) {
        const uint2 t = *reinterpret_cast<const uint2*>(p);
        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&t.x));
        const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&t.y));
        v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
    } else {
#pragma unroll
        for (int q = 0; q < VEC; ++q) v[q] = __half2float(p[q]);
    }
}

template <int VEC>
__device__ __forceinline__ void stv(__half* __restrict__ p, const float (&v)[VEC])
{
    if constexpr (VEC == 4) {
        const __half2 a = __floats2half2_rn(v[0], v[1]), b = __floats2half2_rn(v[2], v[3]);
        uint2 t;
        t.x = *reinterpret_cast<const unsigned*>(&a);
        t.y = *reinterpret_cast<const unsigned*>(&b);
        *reinterpret_cast<uint2*>(p) = t;
    } else {
#pragma unroll
        for (int q = 0; q < VEC; ++q) p[q] = __float2half_rn(v[q]);
    }
}
__device__ __forceinline__ float ld1(const float* p) { return *p; }
__device__ __forceinline__ float ld1(const __half* p) { return __half2float(*p); }
__device__ __forceinline__ void st1(float* p, float v) { *p = v; }
__device__ __forceinline__ void st1(__half* p, float v) { *p = __float2half_rn(v); }

template <int VEC>
__device__ __forceinline__ void zerov(float (&v)[VEC])
{
#pragma unroll
    for (int q = 0; q < VEC; ++q) v[q] = 0.0f;
}

// per-component arithmetic: yee_update.h (the one expression tree of reading #3, shared with the systolic kernels);
// the coefficient-array choice is a run-time flag here
__device__ __forceinline__ float e_update(float e, float hc, float hc_m, float hb, float hb_m, float rdb, float rdc,
                                          bool has_ca, float ca, float cb)
{
    return has_ca ? yee_e_update<true>(e, hc, hc_m, hb, hb_m, rdb, rdc, ca, cb) : yee_e_update<false>(e, hc, hc_m, hb, hb_m, rdb, rdc, ca, cb);
}
__device__ __forceinline__ float h_update(float h, float ec_p, float ec, float eb_p, float eb, float rdb, float rdc, float db)
{
    return yee_h_update(h, ec_p, ec, eb_p, eb, rdb, rdc, db);
}

template <int VEC, typename FT>
__global__ void __launch_bounds__(kThreads) e_half_naive(const __grid_constant__ GridParams g)
{
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long plane = (long long)nx * ny;
    const long long q = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (q * VEC >= plane) return;
    const long long cell0 = q * VEC;
    const int j = (int)(cell0 / nx);
    const int i0 = (int)(cell0 - (long long)j * nx);
    const int k0 = blockIdx.y * kZChunk;
    const int k1 = min(k0 + kZChunk, nz);
    const bool perx = g.per[0], pery = g.per[1], perz = g.per[2];
    const bool wall_y = !pery && j == 0;
    const long long ym_off = (j > 0) ? -(long long)nx : (long long)nx * (ny - 1);
    const long long xm_off = (i0 > 0) ? -1 : (long long)(nx - 1);
    const float rdx = g.rd[0], rdy = g.rd[1], rdz = g.rd[2];
    const bool has_lut = g.cidx[0] != nullptr;       // material-index tables instead of coefficient arrays (row f2)
    const bool has_ca = g.ca[0] != nullptr || has_lut, has_cb = g.cb[0] != nullptr || has_lut;
    const FT* __restrict__ Hx = reinterpret_cast<const FT*>(g.H[0]);
    const FT* __restrict__ Hy = reinterpret_cast<const FT*>(g.H[1]);
    const FT* __restrict__ Hz = reinterpret_cast<const FT*>(g.H[2]);
    FT* __restrict__ Ex = reinterpret_cast<FT*>(g.E[0]);
    FT* __restrict__ Ey = reinterpret_cast<FT*>(g.E[1]);
    FT* __restrict__ Ez = reinterpret_cast<FT*>(g.E[2]);

    float hx_m[VEC], hy_m[VEC];   // H_x, H_y one plane back in z
    if (k0 > 0 || perz) {
        const long long pm = cell0 + plane * (k0 > 0 ? k0 - 1 : nz - 1);
        ldv<VEC>(Hx + pm, hx_m);
        ldv<VEC>(Hy + pm, hy_m);
    } else {
        zerov<VEC>(hx_m);
        zerov<VEC>(hy_m);
    }
    for (int k = k0; k < k1; ++k) {
        const long long p = cell0 + plane * k;
        const bool wall_z = !perz && k == 0;
        float hx[VEC], hy[VEC], hz[VEC], hz_ym[VEC], hx_ym[VEC], ex[VEC], ey[VEC], ez[VEC];
        ldv<VEC>(Hx + p, hx);
        ldv<VEC>(Hy + p, hy);
        ldv<VEC>(Hz + p, hz);
        ldv<VEC>(Hz + p + ym_off, hz_ym);
        ldv<VEC>(Hx + p + ym_off, hx_ym);
        const float hz_xm = ld1(Hz + p + xm_off);
        const float hy_xm = ld1(Hy + p + xm_off);
        ldv<VEC>(Ex + p, ex);
        ldv<VEC>(Ey + p, ey);
        ldv<VEC>(Ez + p, ez);
        float ca0[VEC], ca1[VEC], ca2[VEC], cb0[VEC], cb1[VEC], cb2[VEC];
        if (has_lut) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const int m0 = g.cidx[0][p + v], m1 = g.cidx[1][p + v], m2 = g.cidx[2][p + v];
                const float2 q0 = __ldg(reinterpret_cast<const float2*>(g.lut) + m0);
                const float2 q1 = __ldg(reinterpret_cast<const float2*>(g.lut) + g.nmat + m1);
                const float2 q2 = __ldg(reinterpret_cast<const float2*>(g.lut) + 2 * g.nmat + m2);
                ca0[v] = q0.x; cb0[v] = q0.y; ca1[v] = q1.x; cb1[v] = q1.y; ca2[v] = q2.x; cb2[v] = q2.y;
            }
        } else {
            if (has_ca) { ldv<VEC>(g.ca[0] + p, ca0); ldv<VEC>(g.ca[1] + p, ca1); ldv<VEC>(g.ca[2] + p, ca2); }
            if (has_cb) { ldv<VEC>(g.cb[0] + p, cb0); ldv<VEC>(g.cb[1] + p, cb1); ldv<VEC>(g.cb[2] + p, cb2); }
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const bool wall_x = !perx && (i0 + v) == 0;
            const float hz_x = (v == 0) ? hz_xm : hz[v > 0 ? v - 1 : 0];
            const float hy_x = (v == 0) ? hy_xm : hy[v > 0 ? v - 1 : 0];
            if (!(wall_y || wall_z))   // E_x: (Hz - Hz[j-1])/dy - (Hy - Hy[k-1])/dz
                ex[v] = e_update(ex[v], hz[v], hz_ym[v], hy[v], hy_m[v], rdy, rdz, has_ca, has_ca ? ca0[v] : 1.0f,
                                 has_cb ? cb0[v] : g.cb_scalar);
            if (!(wall_z || wall_x))   // E_y: (Hx - Hx[k-1])/dz - (Hz - Hz[i-1])/dx
                ey[v] = e_update(ey[v], hx[v], hx_m[v], hz[v], hz_x, rdz, rdx, has_ca, has_ca ? ca1[v] : 1.0f,
                                 has_cb ? cb1[v] : g.cb_scalar);
            if (!(wall_x || wall_y))   // E_z: (Hy - Hy[i-1])/dx - (Hx - Hx[j-1])/dy
                ez[v] = e_update(ez[v], hy[v], hy_x, hx[v], hx_ym[v], rdx, rdy, has_ca, has_ca ? ca2[v] : 1.0f,
                                 has_cb ? cb2[v] : g.cb_scalar);
        }
        stv<VEC>(Ex + p, ex);
        stv<VEC>(Ey + p, ey);
        stv<VEC>(Ez + p, ez);
#pragma unroll
        for (int v = 0; v < VEC; ++v) { hx_m[v] = hx[v]; hy_m[v] = hy[v]; }
    }
}

template <int VEC, typename FT>
__global__ void __launch_bounds__(kThreads) h_half_naive(const __grid_constant__ GridParams g)
{
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long plane = (long long)nx * ny;
    const long long q = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (q * VEC >= plane) return;
    const long long cell0 = q * VEC;
    const int j = (int)(cell0 / nx);
    const int i0 = (int)(cell0 - (long long)j * nx);
    const int k0 = blockIdx.y * kZChunk;
    const int k1 = min(k0 + kZChunk, nz);
    const bool perx = g.per[0], pery = g.per[1], perz = g.per[2];
    const bool last_y = (j == ny - 1);
    const bool ghost_y = last_y && !pery;          // E beyond the high y wall is 0 (reading #5)
    const long long yp_off = last_y ? -(long long)nx * (ny - 1) : (long long)nx;
    const bool last_x = (i0 + VEC >= nx);
    const bool ghost_x = last_x && !perx;
    const long long xp_off = last_x ? (long long)VEC - nx : (long long)VEC;
    const float rdx = g.rd[0], rdy = g.rd[1], rdz = g.rd[2];
    const FT* __restrict__ Ex = reinterpret_cast<const FT*>(g.E[0]);
    const FT* __restrict__ Ey = reinterpret_cast<const FT*>(g.E[1]);
    const FT* __restrict__ Ez = reinterpret_cast<const FT*>(g.E[2]);
    FT* __restrict__ Hx = reinterpret_cast<FT*>(g.H[0]);
    FT* __restrict__ Hy = reinterpret_cast<FT*>(g.H[1]);
    FT* __restrict__ Hz = reinterpret_cast<FT*>(g.H[2]);

    float ex[VEC], ey[VEC];
    ldv<VEC>(Ex + cell0 + plane * k0, ex);
    ldv<VEC>(Ey + cell0 + plane * k0, ey);
    for (int k = k0; k < k1; ++k) {
        const long long p = cell0 + plane * k;
        float ex_p[VEC], ey_p[VEC], ez[VEC], ez_yp[VEC], ex_yp[VEC], hx[VEC], hy[VEC], hz[VEC];
        if (k < nz - 1) {
            ldv<VEC>(Ex + p + plane, ex_p);
            ldv<VEC>(Ey + p + plane, ey_p);
        } else if (perz) {
            ldv<VEC>(Ex + cell0, ex_p);
            ldv<VEC>(Ey + cell0, ey_p);
        } else {
            zerov<VEC>(ex_p);
            zerov<VEC>(ey_p);
        }
        ldv<VEC>(Ez + p, ez);
        if (ghost_y) {
            zerov<VEC>(ez_yp);
            zerov<VEC>(ex_yp);
        } else {
            ldv<VEC>(Ez + p + yp_off, ez_yp);
            ldv<VEC>(Ex + p + yp_off, ex_yp);
        }
        const float ey_xp = ghost_x ? 0.0f : ld1(Ey + p + xp_off);
        const float ez_xp = ghost_x ? 0.0f : ld1(Ez + p + xp_off);
        ldv<VEC>(Hx + p, hx);
        ldv<VEC>(Hy + p, hy);
        ldv<VEC>(Hz + p, hz);
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const float ey_x = (v == VEC - 1) ? ey_xp : ey[v < VEC - 1 ? v + 1 : v];
            const float ez_x = (v == VEC - 1) ? ez_xp : ez[v < VEC - 1 ? v + 1 : v];
            hx[v] = h_update(hx[v], ez_yp[v], ez[v], ey_p[v], ey[v], rdy, rdz, g.db[0]);   // (Ez[j+1]-Ez)/dy - (Ey[k+1]-Ey)/dz
            hy[v] = h_update(hy[v], ex_p[v], ex[v], ez_x, ez[v], rdz, rdx, g.db[1]);       // (Ex[k+1]-Ex)/dz - (Ez[i+1]-Ez)/dx
            hz[v] = h_update(hz[v], ey_x, ey[v], ex_yp[v], ex[v], rdx, rdy, g.db[2]);      // (Ey[i+1]-Ey)/dx - (Ex[j+1]-Ex)/dy
        }
        stv<VEC>(Hx + p, hx);
        stv<VEC>(Hy + p, hy);
        stv<VEC>(Hz + p, hz);
#pragma unroll
        for (int v = 0; v < VEC; ++v) { ex[v] = ex_p[v]; ey[v] = ey_p[v]; }
    }
}

// E_comp[box] += amp[q] * wave[t]   (reading #6)
template <typename FT>
__global__ void source_kernel(const __grid_constant__ GridParams g, float w)
{
    const int ni = g.src_box[3], nj = g.src_box[4], nk = g.src_box[5];
    const long long total = (long long)ni * nj * nk;
    FT* __restrict__ Ec = reinterpret_cast<FT*>(g.E[g.src_comp]);
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int ii = (int)(q % ni);
        const int jj = (int)((q / ni) % nj);
        const int kk = (int)(q / ((long long)ni * nj));
        const long long p = (long long)(g.src_box[0] + ii) + (long long)g.n[0] * ((long long)(g.src_box[1] + jj) + (long long)g.n[1] * (g.src_box[2] + kk));
        const float inj = g.src_amp[q] * w;
        st1(Ec + p, ld1(Ec + p) + inj);
    }
}

dim3 naive_grid(const GridParams& g, int vec)
{
    const long long plane_vecs = ((long long)g.n[0] * g.n[1] + vec - 1) / vec;
    return dim3((unsigned)((plane_vecs + kThreads - 1) / kThreads), (unsigned)((g.n[2] + kZChunk - 1) / kZChunk), 1);
}

}  // namespace

cudaError_t launch_e_half_naive(const GridParams& g, cudaStream_t st)
{
    if (g.fld16) {
        if (g.n[0] % 4 == 0) e_half_naive<4, __half><<<naive_grid(g, 4), kThreads, 0, st>>>(g);
        else e_half_naive<1, __half><<<naive_grid(g, 1), kThreads, 0, st>>>(g);
    } else if (g.n[0] % 4 == 0)
        e_half_naive<4, float><<<naive_grid(g, 4), kThreads, 0, st>>>(g);
    else
        e_half_naive<1, float><<<naive_grid(g, 1), kThreads, 0, st>>>(g);
    return cudaGetLastError();
}

cudaError_t launch_h_half_naive(const GridParams& g, cudaStream_t st)
{
    if (g.fld16) {
        if (g.n[0] % 4 == 0) h_half_naive<4, __half><<<naive_grid(g, 4), kThreads, 0, st>>>(g);
        else h_half_naive<1, __half><<<naive_grid(g, 1), kThreads, 0, st>>>(g);
    } else if (g.n[0] % 4 == 0)
        h_half_naive<4, float><<<naive_grid(g, 4), kThreads, 0, st>>>(g);
    else
        h_half_naive<1, float><<<naive_grid(g, 1), kThreads, 0, st>>>(g);
    return cudaGetLastError();
}

// host passes wave[t] by value (the host keeps a copy of the table), so the kernel needs no index
cudaError_t launch_source_w(const GridParams& g, float w, cudaStream_t st)
{
    const long long total = (long long)g.src_box[3] * g.src_box[4] * g.src_box[5];
    const int blocks = (int)((total + 255) / 256 > 1184 ? 1184 : (total + 255) / 256);
    if (g.fld16) source_kernel<__half><<<blocks, 256, 0, st>>>(g, w);
    else source_kernel<float><<<blocks, 256, 0, st>>>(g, w);
    return cudaGetLastError();
}

// ---- running-DFT monitor (row f4): one thread per plane cell and component, all frequencies ----------------------------
namespace {
__global__ void __launch_bounds__(128) monitor_kernel(const __grid_constant__ GridParams g, const __grid_constant__ MonitorParams m, int isH, long long t)
{
    const long long q = blockIdx.x * 128ll + threadIdx.x;
    if (q >= 3 * m.pcells) return;
    const int c = (int)(q / m.pcells);
    const long long cell = q % m.pcells;
    // plane cell -> grid coordinates (the naive kernels run on the caller's grid: G = 0)
    int i, j, k;
    if (m.axis == 0)      { i = m.index; j = (int)(cell % m.n[1]); k = (int)(cell / m.n[1]); }
    else if (m.axis == 1) { j = m.index; i = (int)(cell % m.n[0]); k = (int)(cell / m.n[0]); }
    else                  { k = m.index; i = (int)(cell % m.n[0]); j = (int)(cell / m.n[0]); }
    const long long off = i + (long long)g.n[0] * (j + (long long)g.n[1] * k);
    const float* fa = isH ? g.H[c] : g.E[c];
    const float v = g.fld16 ? __half2float(reinterpret_cast<const __half*>(fa)[off]) : fa[off];
    const float* w = (isH ? m.wH : m.wE) + t * m.F * 2;
    float* acc = m.acc + ((long long)(isH ? 3 + c : c) * m.F * 2) * m.pcells + cell;
    for (int f = 0; f < m.F; ++f) {
        const float pr = v * w[2 * f];
        const float pi = v * w[2 * f + 1];
        acc[(2 * f) * m.pcells] = acc[(2 * f) * m.pcells] + pr;
        acc[(2 * f + 1) * m.pcells] = acc[(2 * f + 1) * m.pcells] + pi;
    }
}
}  // namespace

cudaError_t launch_monitor_naive(const GridParams& g, const MonitorParams& m, int isH, long long t, cudaStream_t st)
{
    const long long items = 3 * m.pcells;
    monitor_kernel<<<(unsigned)((items + 127) / 128), 128, 0, st>>>(g, m, isH, t);
    return cudaGetLastError();
}
