// systolic_reg.cu -- the systolic FDTD kernel for sm_100a, register-resident cp.async version: a slow CROSS-CHECK
// implementation (explicit FDTD_KERNEL_SYSTOLIC_REG only; the product kernel is systolic_tma.cu).
//
// Same schedule as systolic_kernel.cu (tile regions R_k = [a-k, a+w-k) sliding along the x-y-z-t diagonal,
// PAPER.md:94; minus-shell loads, plus-shell publishes, per-tile acquire/release flags on all seven upwind
// neighbours, readings #10/#11), but the subdomain does not live in shared memory:
//
//   * box 32 x 16 x 8 cells (tile 31 x 15 x 7).  Compute thread (lane, warp) owns the (x,y) slot
//     (gx mod 32, gy mod 16) = (lane, warp) and keeps the 8-cell z column of all six field components in
//     REGISTERS.  x/y are addressed modulo the box (the slide moves no data, a10); z is indexed by the local
//     coordinate, so the slide in z is a register renaming inside the fully unrolled z march (each phase writes
//     cell l into register l+1).
//   * z neighbours come from the march (registers), x neighbours by warp shuffle (lane +-1, rotating), y
//     neighbours through a small shared-memory exchange buffer holding only the two components the other phase
//     needs (Hz,Hx for the E phase; Ez,Ex for the H phase).
//   * the six coefficient arrays of the resident cells stay in shared memory (96 KB), addressed modulo the box.
//   * global memory is touched by compute threads only to publish leaving cells (fire-and-forget stores).
//     Minus-shell loads are done by three LOADER warps with cp.async into shared-memory staging (fields) and
//     straight into the coefficient slots of the leaving cells; they poll the upwind flags and run up to one
//     phase ahead of the compute warps, so flag latency and L2/HBM latency overlap the other phase's arithmetic.
//     A SIGNAL warp turns "all publishes of this phase are issued" into fence + st.release of the tile's flag.
//
//   compute (16 warps)      H-loaders (2 warps)           E-loader (1 warp)            signal (1 warp)
//   ------------------      -------------------           -----------------            ---------------
//   wait Hfull(k)           wait Edone(k-1)               wait Hdone(k-1)
//   grab H shell            poll flagH[u] >= base+k       poll flagE[u] >= base+k+1
//   E phase k               cp.async H shell + coefs      cp.async E shell
//   publish E, Edone(k) ->  -> Hfull(k)                   -> Efull(k)                  wait Edone(k): fence, flagE=base+k+1
//   wait Efull(k), grab E
//   H phase k
//   publish H, Hdone(k) ->                                                             wait Hdone(k): fence, flagH=base+k+1
//
// Per-cell arithmetic is yee_update.h, unchanged: with -fmad=false the result is bit-identical to the oracle.
#include "fdtd_internal.h"
#include "yee_update.h"

namespace {

constexpr int BX = 32, BY = 16, BZ = 8;
constexpr int PLANE = BX * BY;            // 512 (x,y) slots = compute threads
constexpr int NCOMPUTE = PLANE;
constexpr int NAUX = 128;                 // warps 16,17: H loaders; 18: E loader; 19: signal
constexpr int NT = NCOMPUTE + NAUX;
constexpr int W_HLOAD = 16, W_ELOAD = 18;   // warp 19: signal
constexpr int N_HLOAD_THREADS = 64, N_ELOAD_THREADS = 32;

enum { BAR_COMPUTE = 1, BAR_EDONE = 2, BAR_HDONE = 3 };
constexpr int N_EDONE = NCOMPUTE + N_HLOAD_THREADS + 32;   // compute arrive; H loaders + signal wait
constexpr int N_HDONE = NCOMPUTE + N_ELOAD_THREADS + 32;   // compute arrive; E loader + signal wait

// shared-memory layout, in floats
constexpr int SZ_EXCH = BZ * PLANE;                  // one exchange array, [m][y slot][x slot]
constexpr int SZ_STG_Z = 3 * PLANE;                  // [arr][y slot][x slot]      plane l_z = 0
constexpr int SZ_STG_Y = 3 * BZ * BX;                // [arr][l_z][x slot]         row   l_y = 0
constexpr int SZ_STG_X = BY * 3 * BZ;                // [y slot][arr][l_z]         column l_x = 0 (16-byte rows)
constexpr int SZ_STG = SZ_STG_Z + SZ_STG_Y + SZ_STG_X;
template <bool COEF>
struct Lay {
    static constexpr int exch = COEF ? 6 * BZ * PLANE : 0;
    static constexpr int stgh = exch + 4 * SZ_EXCH;
    static constexpr int stge = stgh + SZ_STG;
    static constexpr int total = stge + SZ_STG;
};

struct TileGeom {
    int a[3], w[3];
    int nbr[7];
};

struct Ctl {
    int tile;
    int abort;
};

// ---- small PTX helpers ----------------------------------------------------------------------------------
__device__ __forceinline__ int ld_acquire(const int* p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_volatile(const int* p)
{
    int v;
    asm volatile("ld.volatile.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void bar_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int count)
{
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// the executing thread's earlier cp.async copies arrive on the mbarrier when they have landed
__device__ __forceinline__ void cp_async_arrive(unsigned long long* bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// 4-byte asynchronous copy global -> shared; ok == false writes 0.0f (cells outside a PEC domain, a3/a11)
__device__ __forceinline__ void cp_async4(float* dst, const float* src, bool ok)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(ok ? 4 : 0) : "memory");
}

// unwrapped global coordinate -> stored coordinate; false if outside the domain on a PEC axis
__device__ __forceinline__ bool resolve(const SysParams& P, int axis, int gu, int& g)
{
    const int n = P.g.n[axis];
    if (P.ax[axis].per) {
        while (gu < 0) gu += n;
        while (gu >= n) gu -= n;
        g = gu;
        return true;
    }
    g = gu;
    return gu >= 0 && gu < n;
}

__device__ __forceinline__ void tile_init(const SysParams& P, int tile, TileGeom& t)
{
    const int nbx = P.ax[0].nb, nby = P.ax[1].nb;
    int b[3];
    b[0] = tile % nbx;
    b[1] = (tile / nbx) % nby;
    b[2] = tile / (nbx * nby);
    for (int q = 0; q < 3; ++q) {
        t.a[q] = P.ax[q].start(b[q]);
        t.w[q] = P.ax[q].width(b[q]);
    }
    for (int d = 1; d < 8; ++d) {
        int idx[3];
        bool ok = true;
        for (int q = 0; q < 3; ++q) {
            int bq = b[q] - ((d >> q) & 1);
            if (bq < 0) {
                if (P.ax[q].per) bq += P.ax[q].nb; else ok = false;
            }
            idx[q] = bq;
        }
        t.nbr[d - 1] = ok ? idx[0] + nbx * (idx[1] + nby * idx[2]) : -1;
    }
}

// lanes 0..6 of the calling warp each watch one upwind neighbour (a9); on a watchdog hit the whole launch is
// flagged and every later wait returns at once (the host reports FDTD_ETIMEOUT; fields are then invalid).
__device__ __forceinline__ void wait_upwind(const SysParams& P, const TileGeom& t, const int* flags, int target, Ctl* ctl)
{
    const int lane = threadIdx.x & 31;
    if (lane < 7 && *(volatile int*)&ctl->abort == 0 && !FDTD_DBG(P, 1)) {
        const int u = t.nbr[lane];
        if (u >= 0) {
            const long long t_start = clock64();
            unsigned spins = 0;
            while (ld_acquire(flags + u) < target) {
                if ((++spins & 63u) == 0u) {
                    if (ld_volatile(P.abort_flag) != 0) { *(volatile int*)&ctl->abort = 1; break; }
                    if (clock64() - t_start > P.spin_budget) {
                        atomicExch(P.abort_flag, 1);
                        *(volatile int*)&ctl->abort = 1;
                        break;
                    }
                }
                __nanosleep(20);
            }
        }
    }
    __syncwarp();
}

#ifdef FDTD_DEBUG
__device__ __forceinline__ void debug_delay(const SysParams& P, int tile, int k, int phase)
{
    if (P.delay_seed == 0u) return;
    unsigned h = P.delay_seed ^ (unsigned)(tile * 2654435761u) ^ (unsigned)(k * 40503u + phase * 97u);
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13; h *= 3266489917u; h ^= h >> 16;
    if ((h & 3u) == 0u) __nanosleep((h >> 8) & 0x3fffu);   // up to ~16 us, one phase in four
}
#endif

// ---- loader warps: minus shell of the box of step k, NARR field arrays (+ six coefficient arrays) ---------
// part / nparts split the work between the loader warps of one kind.
template <bool COEF, bool WITH_COEF>
__device__ __forceinline__ void load_shell(const SysParams& P, const TileGeom& t, int k, float* const* fld, float* stg,
                                           float* coef, int part, int nparts)
{
    const int lane = threadIdx.x & 31;
    const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
    const long long nx = P.g.n[0], ny = P.g.n[1];
    float* stgZ = stg;
    float* stgY = stg + SZ_STG_Z;
    float* stgX = stg + SZ_STG_Z + SZ_STG_Y;

    auto cell = [&](int lx, int ly, int lz, float* d0, int dstride) {
        int gx, gy, gz;
        const bool in = resolve(P, 0, o0 + lx, gx) & resolve(P, 1, o1 + ly, gy) & resolve(P, 2, o2 + lz, gz);
        const long long off = in ? gx + nx * (gy + ny * (long long)gz) : 0;
        if (FDTD_DBG(P, 2)) return;
#pragma unroll
        for (int c = 0; c < 3; ++c) cp_async4(d0 + c * dstride, fld[c] + off, in);
        if (COEF && WITH_COEF) {
            float* cs = coef + (((o2 + lz) & (BZ - 1)) * BY + ((o1 + ly) & (BY - 1))) * BX + ((o0 + lx) & (BX - 1));
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                cp_async4(cs + c * (BZ * PLANE), P.g.ca[c] + off, in);
                cp_async4(cs + (3 + c) * (BZ * PLANE), P.g.cb[c] + off, in);
            }
        }
    };

    int task = 0;
    // plane l_z = 0: rows l_y = 0..w1, lane = l_x
    for (int ly = 0; ly <= t.w[1]; ++ly, ++task) {
        if (task % nparts != part) continue;
        if (lane <= t.w[0]) cell(lane, ly, 0, stgZ + ((o1 + ly) & (BY - 1)) * BX + ((o0 + lane) & (BX - 1)), PLANE);
    }
    // row l_y = 0: l_z = 1..w2, lane = l_x
    for (int lz = 1; lz <= t.w[2]; ++lz, ++task) {
        if (task % nparts != part) continue;
        if (lane <= t.w[0]) cell(lane, 0, lz, stgY + lz * BX + ((o0 + lane) & (BX - 1)), BZ * BX);
    }
    // column l_x = 0: (l_y = 1..w1) x (l_z = 0..BZ-1), 32 cells per pass
    for (int base = 0; base < t.w[1] * BZ; base += 32, ++task) {
        if (task % nparts != part) continue;
        const int idx = base + lane;
        const int lz = idx & (BZ - 1), ly = 1 + (idx >> 3);
        if (ly <= t.w[1] && lz <= t.w[2]) cell(0, ly, lz, stgX + ((o1 + ly) & (BY - 1)) * (3 * BZ) + lz, BZ);
    }
}

// ---- compute warps ----------------------------------------------------------------------------------------
template <bool COEF>
__device__ __forceinline__ void compute_tile(const SysParams& P, const TileGeom& t, int tile, float* sm, unsigned long long* mbH,
                                             unsigned long long* mbE, unsigned& phH, unsigned& phE)
{
    const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5;
    const int slot = wy * BX + lane;
    const int slot_ym = ((wy - 1) & (BY - 1)) * BX + lane, slot_yp = ((wy + 1) & (BY - 1)) * BX + lane;
    const int lane_m = (lane - 1) & 31, lane_p = (lane + 1) & 31;
    const int w0 = t.w[0], w1 = t.w[1], w2 = t.w[2];
    const long long nx = P.g.n[0], plane = nx * P.g.n[1];

    float* coef = sm;
    float* exHz = sm + Lay<COEF>::exch;
    float* exHx = exHz + SZ_EXCH;
    float* exEz = exHx + SZ_EXCH;
    float* exEx = exEz + SZ_EXCH;
    const float* sgH = sm + Lay<COEF>::stgh;
    const float* sgE = sm + Lay<COEF>::stge;

    const float rdx = P.g.rd[0], rdy = P.g.rd[1], rdz = P.g.rd[2];
    const float dbx = P.g.db[0], dby = P.g.db[1], dbz = P.g.db[2];
    const float cbs = P.g.cb_scalar;

    float ex[BZ + 1], ey[BZ + 1], ez[BZ + 1], hx[BZ], hy[BZ], hz[BZ];
#pragma unroll
    for (int l = 0; l <= BZ; ++l) ex[l] = ey[l] = ez[l] = 0.0f;
#pragma unroll
    for (int l = 0; l < BZ; ++l) hx[l] = hy[l] = hz[l] = 0.0f;

    for (int k = 0; k < P.T; ++k) {
        const bool last = (k == P.T - 1);
        const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
        const int lx = (lane - o0) & (BX - 1), ly = (wy - o1) & (BY - 1);
        int gx, gy;
        const bool col_in = resolve(P, 0, o0 + lx, gx) & resolve(P, 1, o1 + ly, gy) & (lx <= w0) & (ly <= w1);
        const long long col_off = col_in ? gx + nx * gy : 0;
        const bool wall_x = !P.ax[0].per && gx == 0, wall_y = !P.ax[1].per && gy == 0;
        // z: stored index and validity of local plane l (uniform over the CTA)
        int gz[BZ];
        bool zin[BZ];
#pragma unroll
        for (int l = 0; l < BZ; ++l) zin[l] = resolve(P, 2, o2 + l, gz[l]) & (l <= w2);

        // ---------------- H (+ coefficient) minus shell ----------------------------------------------------
        if (k == 0) {
            // a6: the whole box; H and coefficients on [0,w]^3, E on R_0 = [1,w]^3
#pragma unroll
            for (int l = 0; l < BZ; ++l) {
                const bool ok = col_in && zin[l];
                const long long off = ok ? col_off + plane * gz[l] : 0;
                hx[l] = ok ? __ldcg(P.g.H[0] + off) : 0.0f;
                hy[l] = ok ? __ldcg(P.g.H[1] + off) : 0.0f;
                hz[l] = ok ? __ldcg(P.g.H[2] + off) : 0.0f;
                const bool oke = ok && lx >= 1 && ly >= 1 && l >= 1;
                ex[l] = oke ? __ldcg(P.g.E[0] + off) : 0.0f;
                ey[l] = oke ? __ldcg(P.g.E[1] + off) : 0.0f;
                ez[l] = oke ? __ldcg(P.g.E[2] + off) : 0.0f;
                if (COEF) {
                    float* cs = coef + ((o2 + l) & (BZ - 1)) * PLANE + slot;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        cs[c * (BZ * PLANE)] = ok ? __ldg(P.g.ca[c] + off) : 0.0f;
                        cs[(3 + c) * (BZ * PLANE)] = ok ? __ldg(P.g.cb[c] + off) : 0.0f;
                    }
                }
            }
#pragma unroll
            for (int l = 1; l < BZ; ++l) {
                exHz[l * PLANE + slot] = hz[l];
                exHx[l * PLANE + slot] = hx[l];
            }
        } else {
            mbar_wait(mbH, phH & 1u);
            ++phH;
            hx[0] = sgH[0 * PLANE + slot];
            hy[0] = sgH[1 * PLANE + slot];
            hz[0] = sgH[2 * PLANE + slot];
            if (ly == 0) {            // warp-uniform: the entering row
                const float* sy = sgH + SZ_STG_Z + lane;
#pragma unroll
                for (int l = 1; l < BZ; ++l) {
                    hx[l] = sy[(0 * BZ + l) * BX];
                    hy[l] = sy[(1 * BZ + l) * BX];
                    hz[l] = sy[(2 * BZ + l) * BX];
                    exHz[l * PLANE + slot] = hz[l];
                    exHx[l * PLANE + slot] = hx[l];
                }
            } else if (lx == 0) {     // one lane per warp: the entering column
                const float4* s4 = reinterpret_cast<const float4*>(sgH + SZ_STG_Z + SZ_STG_Y + wy * (3 * BZ));
                const float4 a0 = s4[0], a1 = s4[1], b0 = s4[2], b1 = s4[3], c0 = s4[4], c1 = s4[5];
                hx[1] = a0.y; hx[2] = a0.z; hx[3] = a0.w; hx[4] = a1.x; hx[5] = a1.y; hx[6] = a1.z; hx[7] = a1.w;
                hy[1] = b0.y; hy[2] = b0.z; hy[3] = b0.w; hy[4] = b1.x; hy[5] = b1.y; hy[6] = b1.z; hy[7] = b1.w;
                hz[1] = c0.y; hz[2] = c0.z; hz[3] = c0.w; hz[4] = c1.x; hz[5] = c1.y; hz[6] = c1.z; hz[7] = c1.w;
            }
        }
        bar_sync(BAR_COMPUTE, NCOMPUTE);   // exchange rows of H (shell + last H phase) are visible

        // ---------------- E phase on R_k = [1,w]^3 (a1) ---------------------------------------------------------
        if (ly >= 1 && ly <= w1) {        // warp-uniform
            const bool colE = col_in && lx >= 1;
            const bool pEx = colE && !wall_y, pEy = colE && !wall_x, pEz = colE && !wall_x && !wall_y;
#pragma unroll
            for (int l = BZ - 1; l >= 1; --l) {
                const float hz_xm = __shfl_sync(0xffffffffu, hz[l], lane_m);
                const float hy_xm = __shfl_sync(0xffffffffu, hy[l], lane_m);
                const float hz_ym = exHz[l * PLANE + slot_ym];
                const float hx_ym = exHx[l * PLANE + slot_ym];
                float cax = 1.0f, cay = 1.0f, caz = 1.0f, cbx = cbs, cby = cbs, cbz = cbs;
                if (COEF) {
                    const float* cs = coef + ((o2 + l) & (BZ - 1)) * PLANE + slot;
                    cax = cs[0 * (BZ * PLANE)]; cay = cs[1 * (BZ * PLANE)]; caz = cs[2 * (BZ * PLANE)];
                    cbx = cs[3 * (BZ * PLANE)]; cby = cs[4 * (BZ * PLANE)]; cbz = cs[5 * (BZ * PLANE)];
                }
                const bool wall_z = !P.ax[2].per && gz[l] == 0;
                const bool zu = zin[l], zw = zin[l] && !wall_z;
                // E_x: (Hz - Hz[j-1])/dy - (Hy - Hy[k-1])/dz      eq. (1)
                const float nex = yee_e_update<COEF>(ex[l], hz[l], hz_ym, hy[l], hy[l - 1], rdy, rdz, cax, cbx);
                // E_y: (Hx - Hx[k-1])/dz - (Hz - Hz[i-1])/dx
                const float ney = yee_e_update<COEF>(ey[l], hx[l], hx[l - 1], hz[l], hz_xm, rdz, rdx, cay, cby);
                // E_z: (Hy - Hy[i-1])/dx - (Hx - Hx[j-1])/dy
                const float nez = yee_e_update<COEF>(ez[l], hy[l], hy_xm, hx[l], hx_ym, rdx, rdy, caz, cbz);
                ex[l + 1] = (pEx && zw) ? nex : ex[l];
                ey[l + 1] = (pEy && zw) ? ney : ey[l];
                ez[l + 1] = (pEz && zu) ? nez : ez[l];
            }
            // soft source after the E update of step t0 + k (a4)
            const long long ts = P.t0 + k;
            if (P.g.src_comp >= 0 && ts >= 0 && ts < P.g.src_nwave) {
                const int sx = gx - P.g.src_box[0], sy = gy - P.g.src_box[1];
                if (colE && sx >= 0 && sx < P.g.src_box[3] && sy >= 0 && sy < P.g.src_box[4]) {
                    const float wsrc = __ldg(P.g.src_wave + ts);
#pragma unroll
                    for (int l = 1; l < BZ; ++l) {
                        const int sz = gz[l] - P.g.src_box[2];
                        if (zin[l] && sz >= 0 && sz < P.g.src_box[5]) {
                            const float amp = __ldg(P.g.src_amp + (sx + P.g.src_box[3] * (sy + (long long)P.g.src_box[4] * sz)));
                            const float inj = amp * wsrc;
                            if (P.g.src_comp == 0) ex[l + 1] = ex[l + 1] + inj;
                            else if (P.g.src_comp == 1) ey[l + 1] = ey[l + 1] + inj;
                            else ez[l + 1] = ez[l + 1] + inj;
                        }
                    }
                }
            }
#pragma unroll
            for (int l = 1; l < BZ - 1; ++l) {   // E(l) lives in register l+1 from here on; H phase reads m = 1..BZ-1
                exEz[(l + 1) * PLANE + slot] = ez[l + 1];
                exEx[(l + 1) * PLANE + slot] = ex[l + 1];
            }
            // publish E of R_k \ R_{k+1} (everything at the last step)                                  (a8, a6)
            if (colE && !FDTD_DBG(P, 4)) {
                const bool whole = last || lx == w0 || ly == w1;
                if (whole) {
#pragma unroll
                    for (int l = 1; l < BZ; ++l) {
                        if (zin[l]) {
                            const long long off = col_off + plane * gz[l];
                            __stcg(P.g.E[0] + off, ex[l + 1]);
                            __stcg(P.g.E[1] + off, ey[l + 1]);
                            __stcg(P.g.E[2] + off, ez[l + 1]);
                        }
                    }
                } else {
#pragma unroll
                    for (int l = 1; l < BZ; ++l) {
                        if (l == w2 && zin[l]) {
                            const long long off = col_off + plane * gz[l];
                            __stcg(P.g.E[0] + off, ex[l + 1]);
                            __stcg(P.g.E[1] + off, ey[l + 1]);
                            __stcg(P.g.E[2] + off, ez[l + 1]);
                        }
                    }
                }
            }
        }
        bar_arrive(BAR_EDONE, N_EDONE);
        FDTD_DEBUG_ONLY(if (P.delay_seed != 0u) debug_delay(P, tile, k, 1);)

        // ---------------- E minus shell -------------------------------------------------------------------------
        mbar_wait(mbE, phE & 1u);
        ++phE;
        ex[1] = sgE[0 * PLANE + slot];
        ey[1] = sgE[1 * PLANE + slot];
        ez[1] = sgE[2 * PLANE + slot];
        exEz[1 * PLANE + slot] = ez[1];
        exEx[1 * PLANE + slot] = ex[1];
        if (ly == 0) {
            const float* sy = sgE + SZ_STG_Z + lane;
#pragma unroll
            for (int l = 1; l < BZ; ++l) {
                ex[l + 1] = sy[(0 * BZ + l) * BX];
                ey[l + 1] = sy[(1 * BZ + l) * BX];
                ez[l + 1] = sy[(2 * BZ + l) * BX];
            }
        } else if (lx == 0) {
            const float4* s4 = reinterpret_cast<const float4*>(sgE + SZ_STG_Z + SZ_STG_Y + wy * (3 * BZ));
            const float4 a0 = s4[0], a1 = s4[1], b0 = s4[2], b1 = s4[3], c0 = s4[4], c1 = s4[5];
            ex[2] = a0.y; ex[3] = a0.z; ex[4] = a0.w; ex[5] = a1.x; ex[6] = a1.y; ex[7] = a1.z; ex[8] = a1.w;
            ey[2] = b0.y; ey[3] = b0.z; ey[4] = b0.w; ey[5] = b1.x; ey[6] = b1.y; ey[7] = b1.z; ey[8] = b1.w;
            ez[2] = c0.y; ez[3] = c0.z; ez[4] = c0.w; ez[5] = c1.x; ez[6] = c1.y; ez[7] = c1.z; ez[8] = c1.w;
#pragma unroll
            for (int m = 2; m < BZ; ++m) {
                exEz[m * PLANE + slot] = ez[m];
                exEx[m * PLANE + slot] = ex[m];
            }
        }
        bar_sync(BAR_COMPUTE, NCOMPUTE);   // exchange rows of E are visible

        // ---------------- H phase on R_{k+1} = [0,w-1]^3 (a2) ------------------------------------------------
        if (ly <= w1 - 1) {               // warp-uniform
            const bool colH = col_in && lx <= w0 - 1;
#pragma unroll
            for (int l = BZ - 2; l >= 0; --l) {
                const float ey_xp = __shfl_sync(0xffffffffu, ey[l + 1], lane_p);
                const float ez_xp = __shfl_sync(0xffffffffu, ez[l + 1], lane_p);
                const float ez_yp = exEz[(l + 1) * PLANE + slot_yp];
                const float ex_yp = exEx[(l + 1) * PLANE + slot_yp];
                const bool up = colH && zin[l] && (l <= w2 - 1);
                const float nhx = yee_h_update(hx[l], ez_yp, ez[l + 1], ey[l + 2], ey[l + 1], rdy, rdz, dbx);   // (Ez[j+1]-Ez)/dy - (Ey[k+1]-Ey)/dz
                const float nhy = yee_h_update(hy[l], ex[l + 2], ex[l + 1], ez_xp, ez[l + 1], rdz, rdx, dby);   // (Ex[k+1]-Ex)/dz - (Ez[i+1]-Ez)/dx
                const float nhz = yee_h_update(hz[l], ey_xp, ey[l + 1], ex_yp, ex[l + 1], rdx, rdy, dbz);       // (Ey[i+1]-Ey)/dx - (Ex[j+1]-Ex)/dy
                hx[l + 1] = up ? nhx : hx[l];
                hy[l + 1] = up ? nhy : hy[l];
                hz[l + 1] = up ? nhz : hz[l];
            }
#pragma unroll
            for (int m = 1; m < BZ; ++m) {
                exHz[m * PLANE + slot] = hz[m];
                exHx[m * PLANE + slot] = hx[m];
            }
            // publish H of R_{k+1} \ R_{k+2}: frame-k planes l = w-1 (everything at the last step)       (a8, a6)
            if (colH && !FDTD_DBG(P, 4)) {
                const bool whole = last || lx == w0 - 1 || ly == w1 - 1;
                if (whole) {
#pragma unroll
                    for (int l = 0; l < BZ - 1; ++l) {
                        if (zin[l] && l <= w2 - 1) {
                            const long long off = col_off + plane * gz[l];
                            __stcg(P.g.H[0] + off, hx[l + 1]);
                            __stcg(P.g.H[1] + off, hy[l + 1]);
                            __stcg(P.g.H[2] + off, hz[l + 1]);
                        }
                    }
                } else {
#pragma unroll
                    for (int l = 0; l < BZ - 1; ++l) {
                        if (l == w2 - 1 && zin[l]) {
                            const long long off = col_off + plane * gz[l];
                            __stcg(P.g.H[0] + off, hx[l + 1]);
                            __stcg(P.g.H[1] + off, hy[l + 1]);
                            __stcg(P.g.H[2] + off, hz[l + 1]);
                        }
                    }
                }
            }
        }
        bar_arrive(BAR_HDONE, N_HDONE);
        FDTD_DEBUG_ONLY(if (P.delay_seed != 0u) debug_delay(P, tile, k, 2);)
    }
}

template <bool COEF>
__global__ void __launch_bounds__(NT, 1) systolic_reg_kernel(const __grid_constant__ SysParams P)
{
    extern __shared__ __align__(16) float sm[];
    __shared__ __align__(8) unsigned long long mbar[2];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        ctl.abort = 0;
        mbar_init(&mbar[0], N_HLOAD_THREADS);
        mbar_init(&mbar[1], N_ELOAD_THREADS);
    }
    unsigned phH = 0, phE = 0;   // completed phases of the two mbarriers, tracked identically by every user

    for (;;) {
        __syncthreads();
        if (tid == 0) {
            ctl.tile = (int)atomicAdd(P.counter, 1u);
            if (ld_volatile(P.abort_flag) != 0) ctl.abort = 1;
        }
        __syncthreads();
        const int tile = ctl.tile;
        if (tile >= P.ntiles || ctl.abort) break;
        TileGeom t;
        tile_init(P, tile, t);
        const int T = P.T;

        if (warp < W_HLOAD) {
            compute_tile<COEF>(P, t, tile, sm, &mbar[0], &mbar[1], phH, phE);
        } else if (warp < W_ELOAD) {
            // H loaders: shell of step k needs the coefficient slots and the staging of step k-1 released
            // (E phase k-1 done) and the upwind tiles' H of step k-1 published
            for (int k = 1; k < T; ++k) {
                bar_sync(BAR_EDONE, N_EDONE);
                wait_upwind(P, t, P.flagH, P.flag_base + k, &ctl);
                load_shell<COEF, true>(P, t, k, P.g.H, sm + Lay<COEF>::stgh, sm, warp - W_HLOAD, 2);
                cp_async_arrive(&mbar[0]);
            }
            bar_sync(BAR_EDONE, N_EDONE);
        } else if (warp == W_ELOAD) {
            for (int k = 0; k < T; ++k) {
                if (k > 0) bar_sync(BAR_HDONE, N_HDONE);
                wait_upwind(P, t, P.flagE, P.flag_base + k + 1, &ctl);
                load_shell<COEF, false>(P, t, k, P.g.E, sm + Lay<COEF>::stge, sm, 0, 1);
                cp_async_arrive(&mbar[1]);
            }
            bar_sync(BAR_HDONE, N_HDONE);
        } else {
            // signal warp: every publish of the phase has been issued (bar.arrive follows the stores);
            // make them visible, then raise the flag                                                   (a9)
            for (int k = 0; k < T; ++k) {
                bar_sync(BAR_EDONE, N_EDONE);
                if (lane == 0) {
                    if (!FDTD_DBG(P, 8)) __threadfence();
                    st_release(P.flagE + tile, P.flag_base + k + 1);
                }
                bar_sync(BAR_HDONE, N_HDONE);
                if (lane == 0) {
                    if (!FDTD_DBG(P, 8)) __threadfence();
                    st_release(P.flagH + tile, P.flag_base + k + 1);
                }
            }
        }
    }
}

}  // namespace

size_t systolic_reg_smem(int coef) { return (size_t)(coef ? Lay<true>::total : Lay<false>::total) * sizeof(float); }
int systolic_reg_threads() { return NT; }

cudaError_t systolic_reg_prepare(int coef, int* blocks_per_sm)
{
    const void* fn = coef ? (const void*)&systolic_reg_kernel<true> : (const void*)&systolic_reg_kernel<false>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)systolic_reg_smem(coef));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, fn, NT, systolic_reg_smem(coef));
}

cudaError_t launch_systolic_reg(int coef, const SysParams& p, int ctas, cudaStream_t st)
{
    const void* fn = coef ? (const void*)&systolic_reg_kernel<true> : (const void*)&systolic_reg_kernel<false>;
    void* args[] = {(void*)&p};
    return cudaLaunchKernel(fn, dim3((unsigned)ctas), dim3((unsigned)NT), args, systolic_reg_smem(coef), st);
}
