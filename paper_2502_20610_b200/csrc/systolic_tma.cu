// systolic_tma.cu -- the systolic FDTD kernel for sm_100a, TMA-staged version (the product kernel).
//
// Schedule: DESIGN.md section 6.2 (tile regions R_k = [a-k, a+w-k) sliding along the x-y-z-t diagonal, PAPER.md:94;
// one E phase and one H phase per step; minus-shell loads and plus-shell publishes through global
// memory; per-tile acquire/release flags on the seven upwind neighbours).  How a B200 SM
// executes it:
//
//   * box 32 x 16 x 8 cells (tile 31 x 15 x 7), 640 threads: 16 compute warps (warps 0-15) and 4 auxiliary warps
//     (16-19).  Compute thread (lane, warp w) owns the x slot gx mod 32 and the ONE y slot w (gy mod 16) and keeps the
//     8-cell z column of all six field components in REGISTERS (FDTD_NROW = 1: 104 registers per compute thread, 64 per
//     auxiliary thread via setmaxnreg); the slide in x/y is modular addressing, the slide in z a register renaming
//     inside the unrolled z march.  Neighbours: z = registers, x = warp shuffle, y = a shared-memory exchange row
//     written by the neighbouring warp.  (FDTD_NROW = 2, two rows per thread and 8 compute warps, is a rejected
//     experiment that still compiles; FDTD_BY = 8 is the 31x7x7 build with two CTAs per SM.)
//   * the (ca, cb) pair of every resident cell and component sits in a thread-private shared-memory slot and is read
//     with one 64-bit load.
//   * the compute warps execute NO per-cell predicate: walls and the outside of the domain are data.  Cells
//     outside the grid are zero-filled by TMA (fields and coefficients), so E stays 0 there (the PEC ghost,
//     reading #5); frozen wall components get (ca, cb) = (1, 0) when their coefficients enter the chip; shell
//     slots compute garbage that the next shell absorb overwrites.  Stores are predicated, arithmetic is not.
//   * the minus shell of every step is fetched by TMA (cp.async.bulk.tensor, three boxes per array or -- when the
//     component arrays sit at a uniform stride -- per group of arrays: a z plane 36x16x1, a y row 36x1x8, an x column
//     4x16x7, each starting on a 16-byte boundary in x) into shared-memory staging, completing on mbarriers;
//     auxiliary warps poll the upwind flags, issue the copies one step ahead of the compute warps and repack the x
//     column so that its single owner lane absorbs it with 16-byte loads.  The coefficient shell is copied by an
//     auxiliary warp too, but scattered into the owner threads' private slots by the compute warps (one row or column
//     piece per warp) after E phase k, a whole step before E phase k+1 reads it.
//   * every hand-off inside the CTA is an mbarrier with one elected arrive per warp; the only CTA-wide barriers are the
//     two 512-thread named barriers of a step (exchange rows of H visible before the E phase, of E before the H phase).
//   * ONE gpu-scope fence per step: the signal warp copies the leaving x columns of E and of H out of shared memory
//     (acknowledging each at once, so the compute warps never wait for the fence), stores them, fences, and raises
//     flagE and flagH together.
//   * tiles are claimed in wavefront order (bx+by+bz) and skip the steps at which their region lies outside the grid;
//     consecutive launches of one tile grid overlap (griddepcontrol + the pred_final wait in next_tile).
//
//   compute (warps 0-15)         warp 16: field H shell      warp 17: coefficient shell   warp 18: field E shell     warp 19: flags
//   --------------------         ------------------------    -------------------------    -----------------------    ---------------
//   wait HREADY(k), absorb H     poll flagH[u] >= base+k     wait CFREE(k-1)              poll flagE[u] >= base+k+1
//     -> HFREE                   fence.proxy.async           TMA coefficient shell k      fence.proxy.async
//   barrier (512)                wait HFREE(k-1)               -> CFULL(k) on landing     wait EFREE(k-1)
//   E phase k, source, monitor   TMA H shell k                                            TMA E shell k, landed
//   wait ACKE(k-1), publish E    wait landed, pack x column                               pack x column
//     -> EDONE                   -> HREADY(k)                                             wait HDONE(k-1)            wait EDONE(k): x column
//   wait EREADY(k), absorb E                                                              write E exchange column      -> registers -> ACKE
//     -> EFREE                                                                            -> EREADY(k)               wait HDONE(k): x column
//   barrier (512)                                                                                                      -> registers -> ACKH
//   wait CFULL(k), scatter the                                                                                       store both columns, fence,
//     coefficient shell -> CFREE                                                                                       flagE = flagH = base+k+1
//   H phase k, monitor
//   wait ACKH(k-1), publish H -> HDONE
//
// Per-cell arithmetic is yee_update.h, unchanged: with -fmad=false the result is bit-identical to the oracle.
// Scope: every axis is a wall axis of the (possibly padded) grid and nx % 4 == 0 (TMA strides are
// multiples of 16 bytes); P.g.per[] only says which low walls freeze tangential E.
#include <cuda.h>
#include <cuda_fp16.h>
#include <string.h>

#include <type_traits>

#include "fdtd_internal.h"
#include "yee_update.h"

namespace {

// FDTD_BY = 16 (default): one CTA of 16 compute warps per SM, tile 31x15x7.  FDTD_BY = 8 (systolic_tma_by8.cu): tile 31x7x7,
// 8 compute warps, half the shared memory and registers: TWO CTAs per SM, whose latency-bound sections (shell absorb,
// publish, hand-offs) overlap each other's arithmetic.
#ifndef FDTD_BY
#define FDTD_BY 16
#endif
#ifndef FDTD_TMA_NAME
#define FDTD_TMA_NAME(x) x
#endif
constexpr int BX = 32, BY = FDTD_BY, BZ = 8;
constexpr int CTAS_PER_SM = BY == 16 ? 1 : 2;
constexpr int W0 = BX - 1, W1 = BY - 1, W2 = BZ - 1;   // tile widths (PEC axes: always full)
#ifndef FDTD_NROW
#define FDTD_NROW 1
#endif
constexpr int NROW = FDTD_NROW;                         // y slots (rows) per compute thread: 1 or 2
constexpr int NWARPS_C = BY / NROW;                     // compute warps: warp w owns the y slots NROW*w .. NROW*w + NROW-1
constexpr int NCOMPUTE = 32 * NWARPS_C;                 // compute threads
constexpr int SX = BX + 1;                              // row stride of the slot-indexed shared arrays: a column of
constexpr int PLANE = SX * BY;                          // slots (the entering x column) then spans 16 banks, not one
constexpr int NT = NCOMPUTE + 128;
// NROW = 1: the launch gives each of the 640 threads 96 registers: compute warps grow to 104, auxiliary warps shrink to 64
// (512*104 + 128*64 = 61440 = 640*96).  NROW = 2: 384 threads of 168 registers: 256*208 + 128*64 = 61440 <= 64512.
// BY = 8: 384 threads of 80 registers at launch (two CTAs per SM): 256*96 + 128*48 = 30720 = 384*80.
constexpr int REGS_COMPUTE = BY == 8 ? 96 : NROW == 1 ? 104 : 208, REGS_AUX = BY == 8 ? 48 : 64;
constexpr int W_HPROD = NWARPS_C, W_HAUX = NWARPS_C + 1, W_EPROD = NWARPS_C + 2;   // warp NWARPS_C + 3: signal

// staging of one array's minus shell (floats); every TMA destination is 128-byte aligned
// TMA needs the innermost start coordinate on a 16-byte boundary, the shell slides by one cell per step: every
// box starts at q0 = o0 & ~3 and is RX = 36 cells wide; r0 = o0 & 3 is where the shell begins inside a staged row
// Box extents are chosen so that every piece is a multiple of 128 bytes: a group of arrays at uniform stride can
// then be fetched by ONE 4-D box per piece and lands exactly where per-array 3-D boxes would put it.
// Field storage (row f1): FDTD_FLD16 builds keep the six field arrays in IEEE binary16 (systolic_tma_h16.cu);
// arithmetic and the on-chip copies stay f32, every newly computed value is rounded to binary16 before it is used again
// (reading #16), so the result does not depend on the schedule.  A binary16 box needs 8 elements per 16 bytes:
// field boxes start at o0 & ~7, are 40 cells wide, and the x column box is 8 cells wide.
#ifdef FDTD_FLD16
using fld_t = __half;
constexpr int RXF = BX + 8, CWF = 8;
__device__ __forceinline__ float fld_round(float v) { return __half2float(__float2half_rn(v)); }
__device__ __forceinline__ float fld_get(const fld_t* p) { return __half2float(*p); }
__device__ __forceinline__ float fld_ldcg(const float* base, long long off) { return __half2float(__ldcg(reinterpret_cast<const __half*>(base) + off)); }
__device__ __forceinline__ void fld_stcg(float* base, long long off, float v) { __stcg(reinterpret_cast<__half*>(base) + off, __float2half_rn(v)); }
#else
using fld_t = float;
constexpr int RXF = BX + 4, CWF = 4;
__device__ __forceinline__ float fld_round(float v) { return v; }
__device__ __forceinline__ float fld_get(const fld_t* p) { return *p; }
__device__ __forceinline__ float fld_ldcg(const float* base, long long off) { return __ldcg(base + off); }
__device__ __forceinline__ void fld_stcg(float* base, long long off, float v) { __stcg(base + off, v); }
#endif
constexpr int XMASK_F = CWF - 1;
// staged group of the three field arrays, in elements of fld_t: [3][FZF] [3][FYF] [3][FXF]
constexpr int FZF = RXF * BY, FYF = RXF * BZ, FXF = CWF * BY * W2;
constexpr int F_ARR_F = (FZF + FYF + FXF) * (int)sizeof(fld_t) / 4;      // floats of staging per field array and step
static_assert((FZF * sizeof(fld_t)) % 128 == 0 && (FYF * sizeof(fld_t)) % 128 == 0 && (FXF * sizeof(fld_t)) % 128 == 0, "TMA destinations are 128-byte aligned");
__device__ __forceinline__ int zidxF(int a, int ly, int x) { return a * FZF + ly * RXF + x; }
__device__ __forceinline__ int yidxF(int a, int l, int x) { return 3 * FZF + a * FYF + (l - 1) * RXF + x; }
__device__ __forceinline__ int xidxF(int a, int ly, int l) { return 3 * (FZF + FYF) + a * FXF + ((l - 1) * BY + ly) * CWF; }
// Compressed coefficients (row f2, "doubles the number of memory operations"): FDTD_COEF_LUT builds
// (systolic_tma_lut.cu) read one material index (a byte) per cell and component instead of two floats and expand it through
// a table of (ca, cb) pairs held in shared memory when the cell ENTERS the chip; the resident copy stays a float2 pair, so
// the E phase is the one of the coefficient-array build.  A byte box needs 16 elements per 16 bytes: index boxes start at
// o0 & ~15, are 48 cells wide, and the x column box is 16 cells wide.
#ifndef FDTD_COEF_LUT
#define FDTD_COEF_LUT 0
#endif
constexpr bool LUT = FDTD_COEF_LUT != 0;
constexpr int RXB = BX + 16, CWB = 16, MAXMAT = 256;
constexpr int ZB = RXB * BY, YB = RXB * BZ, XB = CWB * BY * W2;              // bytes of one index array's shell pieces
static_assert(ZB % 128 == 0 && YB % 128 == 0 && XB % 128 == 0, "TMA destinations are 128-byte aligned");
constexpr int B_ARR = (ZB + YB + XB) / 4;                                    // floats of staging per index array and step
__device__ __forceinline__ int zidxB(int a, int ly, int x) { return a * ZB + ly * RXB + x; }
__device__ __forceinline__ int yidxB(int a, int l, int x) { return 3 * ZB + a * YB + (l - 1) * RXB + x; }
__device__ __forceinline__ int xidxB(int a, int ly, int l) { return 3 * (ZB + YB) + a * XB + ((l - 1) * BY + ly) * CWB; }
// coefficient arrays are always f32
constexpr int RX = BX + 4;
constexpr int FZ = RX * BY;                  // box (36,16,1)   [y][x]      576 floats: plane l_z = 0
constexpr int FY = RX * BZ;                  // box (36,1,8)    [z][x]      288 floats: row l_y = 0, l_z = 1..8 (8 unused)
constexpr int FX = 4 * BY * W2;              // box (4,16,7)    [z][y][4]   448 floats: column l_x = 0 (x index r0), l_y = 0..15, l_z = 1..7
constexpr int F_ARR = FZ + FY + FX;          // 1312 floats per array and step
// a staged group of NA arrays: [NA][FZ] [NA][FY] [NA][FX]
template <int NA> __device__ __forceinline__ int zidx(int a, int ly, int x) { return a * FZ + ly * RX + x; }
template <int NA> __device__ __forceinline__ int yidx(int a, int l, int x) { return NA * FZ + a * FY + (l - 1) * RX + x; }
template <int NA> __device__ __forceinline__ int xidx(int a, int ly, int l) { return NA * (FZ + FY) + a * FX + ((l - 1) * BY + ly) * 4; }
constexpr int XPK = BY * 3 * 8;              // packed x column [y slot][component][8]
constexpr int EXP = 7 * PLANE;               // one exchange array: 7 planes of (x,y) slots

template <bool COEF>
struct Lay {
    static constexpr int NC = COEF ? 6 : 3;            // resident coefficient floats per cell: COEF: three (ca, cb) pairs,
                                                       // [(c*BZ + z slot)*PLANE + slot] as float2; else three cb masks as float
    static constexpr int stgh = 0;
    static constexpr int stge = stgh + 3 * F_ARR_F;
    static constexpr int stgc = stge + 3 * F_ARR_F;
    static constexpr int lut = stgc + (COEF ? (LUT ? 3 * B_ARR : 6 * F_ARR) : 0);     // (ca, cb) table [3][MAXMAT] of the index build
    static constexpr int xpkh = lut + (COEF && LUT ? 3 * MAXMAT * 2 : 0);
    static constexpr int xpke = xpkh + XPK;
    static constexpr int xoute = xpke + XPK;           // leaving x column of E, [y slot][component][8], stored by the signal warp
    static constexpr int xouth = xoute + XPK;
    static constexpr int exch = xouth + XPK;           // y exchange: float2 (H_z, H_x)[W2][PLANE] then float2 (E_z, E_x)[W2][PLANE]
    static constexpr int coef = exch + 4 * EXP;
    static constexpr int total = coef + NC * BZ * PLANE;
};

enum { MB_HFULL = 0, MB_CFULL, MB_EFULL, MB_HREADY, MB_EREADY, MB_HFREE, MB_EFREE, MB_EDONE, MB_HDONE, MB_ACKE, MB_ACKH, MB_CFREE, MB_COUNT };

struct TileGeom {
    int a[3];
    int nbr[7];
};

struct TileJob {
    int tile, k0, k1;
    bool fast;
    TileGeom t;
};

struct Ctl {
    int tile;
    int abort;
};

// ---- PTX helpers --------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
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
// a9: publish "tile has finished phase v - flag_base"; cumulative over every store the calling thread has observed
__device__ __forceinline__ void raise_flag(const SysParams& P, int* flags, int tile, int v)
{
    FDTD_DEBUG_ONLY(if (tile == P.withhold_tile) return;)   // fault injection: the downwind tiles' watchdog must fire
    st_release(flags + tile, v);
}
// The same for the one raise that no tile of the launch itself waits for (the trailing jump to flag_base + T of a tile
// that left the grid early): with launch overlap the tile of the same index of the NEXT launch may already have raised
// this flag past that value, and a plain store arriving late would lower it (its downwind tiles would then spin until the
// watchdog).  max keeps every flag monotone whatever the timing.
__device__ __forceinline__ void raise_flag_max(const SysParams& P, int* flags, int tile, int v)
{
    FDTD_DEBUG_ONLY(if (tile == P.withhold_tile) return;)
    asm volatile("red.release.gpu.global.max.s32 [%0], %1;" ::"l"(flags + tile), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void st_relaxed(int* p, int v)
{
    asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_volatile(const int* p)
{
    int v;
    asm volatile("ld.volatile.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
#ifdef FDTD_DEBUG
// Time-level shadow arrays (race detection; compute-sanitizer is closed on this pool): one int per
// cell and field = number of updates of this launch that the value in global memory has received.  Every value a tile
// takes from global memory is checked against the level the schedule promises, every publish records its level.
__device__ __forceinline__ void lev_check(const SysParams& P, const int* lev, long long off, int expect, int kind)
{
    if (!lev) return;
    const int v = ld_volatile(lev + off);
    if (v != expect && atomicAdd(P.lev_err, 1ull) == 0ull) {
        P.lev_err[1] = (unsigned long long)kind;
        P.lev_err[2] = (unsigned long long)off;
        P.lev_err[3] = (unsigned long long)(long long)v;
        P.lev_err[4] = (unsigned long long)(long long)expect;
    }
}
__device__ __forceinline__ void lev_set(int* lev, long long off, int v)
{
    if (lev) __stcg(lev + off, v);
}
#endif
__device__ __forceinline__ void bar_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)   // suspend-time hint: the warp sleeps in hardware instead of spinning
        : "memory");
}
// one elected arrive per warp, after every lane's earlier shared/global accesses
__device__ __forceinline__ void warp_arrive(unsigned long long* bar)
{
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
// TMA: box of the 3-D tensor `map` at element coordinates (c0,c1,c2) -> shared memory; out-of-bounds elements
// are written as zeros; completes `bytes of the box` on the mbarrier
__device__ __forceinline__ void tma_load_3d(float* dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
                 "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}

// ---- geometry ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tile_init(const SysParams& P, int tile, TileGeom& t)
{
    const int nbx = P.ax[0].nb, nby = P.ax[1].nb;
    int b[3];
    b[0] = tile % nbx;
    b[1] = (tile / nbx) % nby;
    b[2] = tile / (nbx * nby);
    t.a[0] = b[0] * W0;
    t.a[1] = b[1] * W1;
    t.a[2] = b[2] * W2;
    for (int d = 1; d < 8; ++d) {
        int idx[3];
        bool ok = true;
        for (int q = 0; q < 3; ++q) {
            idx[q] = b[q] - ((d >> q) & 1);
            if (idx[q] < 0) ok = false;
        }
        t.nbr[d - 1] = ok ? idx[0] + nbx * (idx[1] + nby * idx[2]) : -1;
    }
}

// frozen tangential E on the low PEC walls (reading #5): component c of the cell at (gx,gy,gz).  An axis with
// P.g.per[a] != 0 has no wall (a periodic axis running on its padded copy): nothing freezes there.
__device__ __forceinline__ bool frozen(const SysParams& P, int c, int gx, int gy, int gz)
{
    const bool fx = (gx == 0) & (P.g.per[0] == 0), fy = (gy == 0) & (P.g.per[1] == 0), fz = (gz == 0) & (P.g.per[2] == 0);
    return c == 0 ? fy | fz : c == 1 ? fz | fx : fx | fy;
}

// lanes 0..6 of the calling warp each watch one upwind neighbour (a9); watchdog as in systolic_reg.cu
__device__ __forceinline__ void wait_upwind(const SysParams& P, const TileGeom& t, const int* flags, int target, Ctl* ctl)
{
    const int lane = threadIdx.x & 31;
    if (lane < 7 && *(volatile int*)&ctl->abort == 0 && !FDTD_DBG(P, 1)) {
        const int u = t.nbr[lane];
        if (u >= 0 && ld_acquire(flags + u) < target) {
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
                __nanosleep(32);
            }
        }
    }
    __syncwarp();
}

#ifdef FDTD_DEBUG
__device__ __forceinline__ void debug_delay(const SysParams& P, int tile, int k, int phase)
{
    unsigned h = P.delay_seed ^ (unsigned)(tile * 2654435761u) ^ (unsigned)(k * 40503u + phase * 97u);
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13; h *= 3266489917u; h ^= h >> 16;
    if ((h & 3u) == 0u) __nanosleep((h >> 8) & 0x3fffu);   // up to ~16 us, one phase in four
}
#endif

__device__ __forceinline__ void tma_load_4d(float* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(smem_u32(dst)),
                 "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
                 : "memory");
}

// One lane issues the minus shell of step k for a group of NA arrays into stg = [NA][FZ] [NA][FY] [NA][FX].
// grouped == 1: the arrays sit at a uniform stride and maps[0..2] are 4-D (x, y, z, array) maps, one box per piece;
// grouped == 2 (NA = 6): two such triples (maps[0..2], maps[9..11]); grouped == 0: per-array 3-D maps maps[a*3 + piece].
// FLD: the group is the three field arrays (elements of fld_t, field box geometry); else f32 coefficient arrays.
template <int NA, bool FLD>
__device__ __forceinline__ void issue_shell(const CUtensorMap* maps, int grouped, float* stg, int o0, int o1, int o2, unsigned long long* bar)
{
    // piece sizes in floats of staging
    constexpr int FZ = FLD ? FZF * (int)sizeof(fld_t) / 4 : ::FZ, FY = FLD ? FYF * (int)sizeof(fld_t) / 4 : ::FY, FX = FLD ? FXF * (int)sizeof(fld_t) / 4 : ::FX;
    const int q0 = FLD ? (o0 & ~XMASK_F) : (o0 & ~3);
    mbar_expect_tx(bar, (unsigned)NA * (unsigned)(FZ + FY + FX) * 4u);
    float* dz = stg;
    float* dy = stg + NA * FZ;
    float* dx = stg + NA * (FZ + FY);
    if (grouped == 1) {
        tma_load_4d(dz, maps + 0, q0, o1, o2, 0, bar);
        tma_load_4d(dy, maps + 1, q0, o1, o2 + 1, 0, bar);
        tma_load_4d(dx, maps + 2, q0, o1, o2 + 1, 0, bar);
    } else if (grouped == 2) {
        for (int h = 0; h < 2; ++h) {
            tma_load_4d(dz + h * 3 * FZ, maps + h * 9 + 0, q0, o1, o2, 0, bar);
            tma_load_4d(dy + h * 3 * FY, maps + h * 9 + 1, q0, o1, o2 + 1, 0, bar);
            tma_load_4d(dx + h * 3 * FX, maps + h * 9 + 2, q0, o1, o2 + 1, 0, bar);
        }
    } else {
        for (int a = 0; a < NA; ++a) {
            tma_load_3d(dz + a * FZ, maps + a * 3 + 0, q0, o1, o2, bar);          // z plane  l_z = 0
            tma_load_3d(dy + a * FY, maps + a * 3 + 1, q0, o1, o2 + 1, bar);      // y row    l_y = 0, l_z = 1..
            tma_load_3d(dx + a * FX, maps + a * 3 + 2, q0, o1, o2 + 1, bar);      // x column l_x = 0, l_y = 0.., l_z = 1..7
        }
    }
}

// the same for the three material-index arrays (bytes): maps[0..2] one 4-D map per piece when grouped, else maps[a*3 + piece]
__device__ __forceinline__ void issue_index_shell(const CUtensorMap* maps, int grouped, float* stg, int o0, int o1, int o2, unsigned long long* bar)
{
    const int q0 = o0 & ~(CWB - 1);
    mbar_expect_tx(bar, 3u * (unsigned)(ZB + YB + XB));
    float* dz = stg;
    float* dy = stg + 3 * ZB / 4;
    float* dx = stg + 3 * (ZB + YB) / 4;
    if (grouped == 1) {
        tma_load_4d(dz, maps + 0, q0, o1, o2, 0, bar);
        tma_load_4d(dy, maps + 1, q0, o1, o2 + 1, 0, bar);
        tma_load_4d(dx, maps + 2, q0, o1, o2 + 1, 0, bar);
    } else {
        for (int a = 0; a < 3; ++a) {
            tma_load_3d(dz + a * ZB / 4, maps + a * 3 + 0, q0, o1, o2, bar);
            tma_load_3d(dy + a * YB / 4, maps + a * 3 + 1, q0, o1, o2 + 1, bar);
            tma_load_3d(dx + a * XB / 4, maps + a * 3 + 2, q0, o1, o2 + 1, bar);
        }
    }
}

// cb mask of component c for the cell at (gx,gy,gz) when there are no coefficient arrays: dt inside the grid, 0 on
// frozen wall components and outside the grid
__device__ __forceinline__ float cb_mask(const SysParams& P, int c, int gx, int gy, int gz)
{
    const bool in = ((unsigned)gx < (unsigned)P.g.n[0]) & ((unsigned)gy < (unsigned)P.g.n[1]) & ((unsigned)gz < (unsigned)P.g.n[2]);
    return (in && !frozen(P, c, gx, gy, gz)) ? P.g.cb_scalar : 0.0f;
}
// (ca, cb) pair of component c as it enters the chip: the staged values, except frozen wall components -> (1, 0)
__device__ __forceinline__ float2 coef_pair(const SysParams& P, int c, float a, float b, int gx, int gy, int gz)
{
    return frozen(P, c, gx, gy, gz) ? make_float2(1.0f, 0.0f) : make_float2(a, b);
}
// the same when the caller knows (CTA-uniform) whether the box touches a low wall at all
__device__ __forceinline__ float2 coef_pair(const SysParams& P, bool wall, int c, float a, float b, int gx, int gy, int gz)
{
    return wall ? coef_pair(P, c, a, b, gx, gy, gz) : make_float2(a, b);
}

// ---- coefficients of the cells that enter with the shell of a step -> their owner threads' private slots -------------
// All compute threads take part, one shell cell each (after the barrier that follows E phase k, so nobody still reads the
// slots of the cells that left): every thread its own cell of the entering plane l_z = 0, warps 0..6 the entering row
// l_y = 0 (one plane each, lane = x), warps 7..10 the 105 cells of the entering column l_x = 0.  The slots are first read
// by E phase k+1, behind the next CTA barrier.
template <bool COEF>
__device__ __forceinline__ void absorb_coef_shell(const SysParams& P, float* sm, int o0, int o1, int o2, int lx, const int (&ly)[NROW], int ys0)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const float* stg = sm + Lay<COEF>::stgc;
    const unsigned char* stgb = reinterpret_cast<const unsigned char*>(sm + Lay<COEF>::stgc);
    const float2* lut = reinterpret_cast<const float2*>(sm + Lay<COEF>::lut);
    float* const cmask = sm + Lay<COEF>::coef;
    float2* const cpair = reinterpret_cast<float2*>(sm + Lay<COEF>::coef);
    const int r0 = o0 & 3, r0b = o0 & (CWB - 1);
    const bool wall = (o0 <= 0) | (o1 <= 0) | (o2 <= 0);   // CTA-uniform: only then can a shell cell be frozen
    auto put = [&](int slot, int gx, int gy, int gz, const float (&v)[6]) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (COEF) cpair[slot + c * (BZ * PLANE)] = coef_pair(P, wall, c, v[c], v[3 + c], gx, gy, gz);
            else cmask[slot + c * (BZ * PLANE)] = cb_mask(P, c, gx, gy, gz);
        }
    };
    // index build: the staged bytes of a cell -> its three (ca, cb) pairs.  A cell outside the grid was delivered as index 0
    // (TMA zero fill), which is a real material: it gets (0, 0) like the zero-filled arrays of the other build.
    auto expand = [&](int b0, int b1, int b2, int gx, int gy, int gz, float (&v)[6]) {
        const bool in = ((unsigned)gx < (unsigned)P.g.n[0]) & ((unsigned)gy < (unsigned)P.g.n[1]) & ((unsigned)gz < (unsigned)P.g.n[2]);
        const float2 p0 = lut[stgb[b0]], p1 = lut[MAXMAT + stgb[b1]], p2 = lut[2 * MAXMAT + stgb[b2]];
        v[0] = in ? p0.x : 0.0f; v[3] = in ? p0.y : 0.0f;
        v[1] = in ? p1.x : 0.0f; v[4] = in ? p1.y : 0.0f;
        v[2] = in ? p2.x : 0.0f; v[5] = in ? p2.y : 0.0f;
    };
    // the entering plane: this thread's own cells
#pragma unroll
    for (int r = 0; r < NROW; ++r) {
        float v[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) v[c] = (COEF && !LUT) ? stg[zidx<6>(c, ly[r], r0 + lx)] : 0.0f;
        if (COEF && LUT) expand(zidxB(0, ly[r], r0b + lx), zidxB(1, ly[r], r0b + lx), zidxB(2, ly[r], r0b + lx), o0 + lx, o1 + ly[r], o2, v);
        put((o2 & (BZ - 1)) * PLANE + (ys0 + r) * SX + lane, o0 + lx, o1 + ly[r], o2, v);
    }
    constexpr int ROW_WARPS = W2, COL_WARPS = (W1 * W2 + 31) / 32;
#pragma unroll
    for (int it = w; it < ROW_WARPS + COL_WARPS; it += NWARPS_C) {   // one work item per warp (two for one warp when BY = 8)
    if (it < ROW_WARPS) {                      // the entering row, plane l = it + 1: lane = x offset inside the box
        const int l = it + 1, gx = o0 + lane;
        float v[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) v[c] = (COEF && !LUT) ? stg[yidx<6>(c, l, r0 + lane)] : 0.0f;
        if (COEF && LUT) expand(yidxB(0, l, r0b + lane), yidxB(1, l, r0b + lane), yidxB(2, l, r0b + lane), gx, o1, o2 + l, v);
        put(((o2 + l) & (BZ - 1)) * PLANE + (o1 & (BY - 1)) * SX + (gx & (BX - 1)), gx, o1, o2 + l, v);
    } else {                                   // the entering column: idx = (l-1)*W1 + (ly-1)
        const int idx = (it - ROW_WARPS) * 32 + lane;
        if (idx < W1 * W2) {
            const int cy = 1 + idx % W1, l = 1 + idx / W1;
            float v[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) v[c] = (COEF && !LUT) ? stg[xidx<6>(c, cy, l) + r0] : 0.0f;
            if (COEF && LUT) expand(xidxB(0, cy, l) + r0b, xidxB(1, cy, l) + r0b, xidxB(2, cy, l) + r0b, o0, o1 + cy, o2 + l, v);
            put(((o2 + l) & (BZ - 1)) * PLANE + ((o1 + cy) & (BY - 1)) * SX + (o0 & (BX - 1)), o0, o1 + cy, o2 + l, v);
        }
    }
    }
}

// x column of the three field arrays in `stg` -> xpk[(y slot*3 + c)*8 + l], l = 1..7 (16-byte rows for the owner lane)
__device__ __forceinline__ void pack_xcol(const fld_t* stg, float* xpk, int o0, int o1)
{
    const int lane = threadIdx.x & 31;
    const int r0 = o0 & XMASK_F;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        float v[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = r * 32 + lane;
            v[r] = idx < W1 * W2 ? fld_get(stg + xidxF(c, 1 + idx % W1, 1 + idx / W1) + r0) : 0.0f;
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = r * 32 + lane;
            if (idx < W1 * W2) xpk[(((o1 + 1 + idx % W1) & (BY - 1)) * 3 + c) * 8 + 1 + idx / W1] = v[r];
        }
    }
}

// signal warp: the leaving x column of three field arrays, rows ly = ly_lo..ly_hi, six planes starting at local plane
// l_lo, is copied from xo[(y slot*3 + c)*8 + l] into registers (load_xcol; the shared rows are free again as soon as
// it returns) and later stored to global memory at x = gx (store_xcol)                                        (a8)
constexpr int XROUNDS = (BY * (W2 - 1) + 31) / 32;
struct XCol {
    float v[XROUNDS][3];
};
__device__ __forceinline__ void load_xcol(XCol& x, const float* xo, int l_lo)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int r = 0; r < XROUNDS; ++r) {
        const int item = min(r * 32 + lane, BY * (W2 - 1) - 1);            // y slot * 6 + plane
        const float* v = xo + (item / (W2 - 1)) * 24 + l_lo + item % (W2 - 1);
        x.v[r][0] = v[0];
        x.v[r][1] = v[8];
        x.v[r][2] = v[16];
    }
}
__device__ __forceinline__ void store_xcol(const SysParams& P, float* const* fld, const XCol& x, int gx, int o1, int o2, int ly_lo, int ly_hi, int l_lo,
                                           int* lev, int level)
{
    const int lane = threadIdx.x & 31;
    if ((unsigned)gx >= (unsigned)P.g.n[0]) return;
    const long long nx = P.ldx, plane = nx * P.g.n[1];
#pragma unroll
    for (int r = 0; r < XROUNDS; ++r) {
        const int item = r * 32 + lane;
        const int ys = item / (W2 - 1), l = l_lo + item % (W2 - 1);
        const int ly = (ys - o1) & (BY - 1);
        const int gy = o1 + ly, gz = o2 + l;
        if (item < BY * (W2 - 1) && ly >= ly_lo && ly <= ly_hi && (unsigned)gy < (unsigned)P.g.n[1] && (unsigned)gz < (unsigned)P.g.n[2]) {
            const long long off = gx + nx * gy + plane * gz;
            fld_stcg(fld[0], off, x.v[r][0]);
            fld_stcg(fld[1], off, x.v[r][1]);
            fld_stcg(fld[2], off, x.v[r][2]);
            FDTD_DEBUG_ONLY(lev_set(lev, off, level);)
        }
    }
}

// ---- compute warps ---------------------------------------------------------------------------------------------
// FDTD_PROFILE build only: lane 0 of compute warp 0 accumulates clock64 ticks per section of the step into
// P.prof[0..7] (0 wait HREADY + absorb H, 1 barrier, 2 E phase + source + exchange stores, 3 wait ACKE + publish E,
// 4 wait EREADY, 5 absorb E + barrier, 6 H phase + wait ACKH + publish H, 7 wait CREADY + absorb coefficient plane);
// aux warps add theirs to P.prof[8..].
#ifdef FDTD_PROFILE
#define PROF_DECL long long pt_ = clock64(), pacc_[8] = {0, 0, 0, 0, 0, 0, 0, 0}
#define PROF_MARK(i) do { const long long n_ = clock64(); pacc_[i] += n_ - pt_; pt_ = n_; } while (0)
#define PROF_FLUSH(base) do { if ((threadIdx.x & 31) == 0 && P.prof) for (int i_ = 0; i_ < 8; ++i_) atomicAdd((unsigned long long*)P.prof + (base) + i_, (unsigned long long)pacc_[i_]); } while (0)
// event trace of one CTA (the tiles CTA 0 claims in the second half of the claim order): P.prof[32 ...]
#define TRACE_C(ev, k) do { if (w == 0 || w == NWARPS_C - 1) TRACE(w == 0 ? 0 : 5, ev, k); } while (0)
#define TRACE(role, ev, k) do { if (trace_on_ && (threadIdx.x & 31) == 0) { const unsigned i_ = atomicAdd(&trace_cur_, 1u); \
    if (i_ < (unsigned)FDTD_TRACE_CAP) P.prof[32 + i_] = (clock64() << 20) | ((long long)(role) << 16) | ((long long)(ev) << 12) | (long long)((k) & 4095); } } while (0)
__shared__ int trace_on_;
__shared__ unsigned trace_cur_;
#else
#define PROF_DECL
#define PROF_MARK(i)
#define PROF_FLUSH(base)
#define TRACE(role, ev, k)
#define TRACE_C(ev, k)
#endif

// Running-DFT monitor (row f4, reading #15): the cells of the plane that this thread has just updated in step
// t0 + k are accumulated into the caller's device array.  Every (cell, step) pair is updated by exactly one thread of one
// tile; successive steps of a cell are ordered by program order inside a tile and by the flag hand-off between tiles (the
// read-modify-write below is issued before the warp arrives on the DONE barrier that the signal warp's fence covers, and
// goes through L2).  Rare path: the caller tests the CTA-uniform conditions first.
// Kept small on purpose.  The path is rare (only tile steps whose region the plane cuts), but how it is written decides the
// speed of EVERY step of the instantiation: unrolled over the seven planes it doubled the step loop (11.7k instead of 5.4k
// instructions), and as a non-inlined call it made ptxas spill loop-carried values inside the step loop; both ran config 2
// 22-28 % slower even on steps that never take it.  Here: a run-time loop over the planes, the plane's three values picked
// from the register columns by a select chain, and per frequency six accumulator loads in flight, then six stores.
// ax, ay, az: the thread's register columns; plane gz0 + l holds a?[OFF + l].
template <int OFF, int NA>
__device__ __forceinline__ void monitor_add(const MonitorParams& m, const float* w, int base, int gx, int gy, int gz0,
                                            const float (&ax)[NA], const float (&ay)[NA], const float (&az)[NA])
{
    static_assert(OFF + W2 <= NA, "register column too short");
    const long long ps = m.pcells, fs = 2 * ps, cs = fs * m.F;       // strides: re -> im, frequency, component
#pragma unroll 1
    for (int l = 0; l < W2; ++l) {
        const long long cell = m.cell(gx, gy, gz0 + l);
        if (cell < 0) continue;
        float vx = ax[OFF], vy = ay[OFF], vz = az[OFF];
#pragma unroll
        for (int q = 1; q < W2; ++q)
            if (l == q) { vx = ax[OFF + q]; vy = ay[OFF + q]; vz = az[OFF + q]; }
        float* p0 = m.acc + (long long)base * cs + cell;
#pragma unroll 1
        for (int f = 0; f < m.F; ++f, p0 += fs) {
            const float wr = __ldg(w + 2 * f), wi = __ldg(w + 2 * f + 1);
            const float xr = __ldcg(p0), xi = __ldcg(p0 + ps);
            const float yr = __ldcg(p0 + cs), yi = __ldcg(p0 + cs + ps);
            const float zr = __ldcg(p0 + 2 * cs), zi = __ldcg(p0 + 2 * cs + ps);
            const float qxr = vx * wr, qxi = vx * wi, qyr = vy * wr, qyi = vy * wi, qzr = vz * wr, qzi = vz * wi;
            __stcg(p0, xr + qxr);
            __stcg(p0 + ps, xi + qxi);
            __stcg(p0 + cs, yr + qyr);
            __stcg(p0 + cs + ps, yi + qyi);
            __stcg(p0 + 2 * cs, zr + qzr);
            __stcg(p0 + 2 * cs + ps, zi + qzi);
        }
    }
}
// CTA-uniform: does the monitor plane cut the region [lo, lo + W) of this step, and is step ts inside the weight table
__device__ __forceinline__ bool monitor_hits(const MonitorParams& m, long long ts, int lo0, int lo1, int lo2)
{
    if (!m.on || ts < 0 || ts >= m.nt) return false;
    const int lo = m.axis == 0 ? lo0 : m.axis == 1 ? lo1 : lo2;
    const int wd = m.axis == 0 ? W0 : m.axis == 1 ? W1 : W2;
    return m.index >= lo && m.index < lo + wd;
}

struct Phases {   // completed phases of each mbarrier as seen by this thread's role (all users count alike)
    unsigned hready, eready, acke, ackh, cfull;
};

template <bool COEF, bool MON>
__device__ __forceinline__ void compute_tile(const SysParams& P, const TileGeom& t, int tile, int k0, int k1, bool fast, float* sm, unsigned long long* mb, Phases& ph)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    constexpr int RL = NROW - 1;                                // the thread's last row
    const int ys0 = NROW * w;                                   // this thread's y slots (rows): ys0 .. ys0 + RL
    const int slot0 = ys0 * SX + lane, slot1 = slot0 + RL * SX; // slots of the first and of the last row
    const int slot_ym = ((ys0 - 1) & (BY - 1)) * SX + lane;     // the row below row 0 = last row of warp w-1
    const int slot_yp = ((ys0 + NROW) & (BY - 1)) * SX + lane;  // the row above the last row = row 0 of warp w+1
    const int lane_m = (lane - 1) & 31, lane_p = (lane + 1) & 31;
    const int nx = P.g.n[0], ny = P.g.n[1], nz = P.g.n[2];
    const long long ldx = P.ldx, plane = ldx * ny;

    const fld_t* stgH = reinterpret_cast<const fld_t*>(sm + Lay<COEF>::stgh);
    const fld_t* stgE = reinterpret_cast<const fld_t*>(sm + Lay<COEF>::stge);
    const float* xpkH = sm + Lay<COEF>::xpkh;
    const float* xpkE = sm + Lay<COEF>::xpke;
    // y exchange: only the links between a thread's row 1 and the next warp's row 0 go through shared memory
    // (z, x) component pairs: one 64-bit access per link
    float2* exH = reinterpret_cast<float2*>(sm + Lay<COEF>::exch);   // (H_z, H_x) of the last row for the E phase of the next warp's row 0
    float2* exE = exH + EXP;                                         // (E_z, E_x) of row 0 for the H phase of the previous warp's last row
    // this thread's private coefficient slots, row 0 (row 1: + SX): index (c*BZ + z slot)*PLANE; float2 (ca, cb) pairs
    // with coefficient arrays, float cb masks without
    float* const cmask = sm + Lay<COEF>::coef + slot0;
    float2* const cpair = reinterpret_cast<float2*>(sm + Lay<COEF>::coef) + slot0;

    const float rdx = P.g.rd[0], rdy = P.g.rd[1], rdz = P.g.rd[2];
    const float dbx = P.g.db[0], dby = P.g.db[1], dbz = P.g.db[2];
    float* const Ex = P.g.E[0]; float* const Ey = P.g.E[1]; float* const Ez = P.g.E[2];
    float* const Hx = P.g.H[0]; float* const Hy = P.g.H[1]; float* const Hz = P.g.H[2];

    // frame k: local l <-> global z = o2 + l.  E(l) lives in e?[r][l] before the E phase and in e?[r][l+1] after it;
    // H(l) lives in h?[r][l] before the H phase and in h?[r][l+1] (= frame k+1 index) after it.  r = row 0 / 1.
    float ex[NROW][BZ + 1], ey[NROW][BZ + 1], ez[NROW][BZ + 1], hx[NROW][BZ], hy[NROW][BZ], hz[NROW][BZ];
#pragma unroll
    for (int r = 0; r < NROW; ++r) {
#pragma unroll
        for (int l = 0; l <= BZ; ++l) ex[r][l] = ey[r][l] = ez[r][l] = 0.0f;
#pragma unroll
        for (int l = 0; l < BZ; ++l) hx[r][l] = hy[r][l] = hz[r][l] = 0.0f;
    }

    const int T = P.T;
    PROF_DECL;
    for (int k = k0; k < k1; ++k) {
        const bool last = (k == T - 1);
        const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
        const int lx = (lane - o0) & (BX - 1);
        const int gx = o0 + lx;
        const int xs = (o0 & XMASK_F) + lx;    // position inside a staged field row
        int ly[NROW], gy[NROW];
        bool col_in[NROW];
        long long col_off[NROW];
#pragma unroll
        for (int r = 0; r < NROW; ++r) {
            ly[r] = (ys0 + r - o1) & (BY - 1);
            gy[r] = o1 + ly[r];
            col_in[r] = ((unsigned)gx < (unsigned)nx) & ((unsigned)gy[r] < (unsigned)ny);
            col_off[r] = col_in[r] ? gx + ldx * gy[r] : 0;
        }
        // the entering shell row l_y = 0 is row 0 of one warp or row 1 of one warp (warp-uniform tests)

        // ---------------- H (+ coefficient) minus shell ----------------------------------------------------
        if (k == 0) {
            // a6: the whole box straight from global memory; H and coefficients on [0,w]^3, E on R_0 = [1,w]^3
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
#pragma unroll
                for (int l = 0; l < BZ; ++l) {
                    const int gz = o2 + l;
                    const bool ok = col_in[r] && (unsigned)gz < (unsigned)nz;
                    const long long off = ok ? col_off[r] + plane * gz : 0;
                    hx[r][l] = ok ? fld_ldcg(Hx, off) : 0.0f;
                    hy[r][l] = ok ? fld_ldcg(Hy, off) : 0.0f;
                    hz[r][l] = ok ? fld_ldcg(Hz, off) : 0.0f;
                    const bool oke = ok && lx >= 1 && ly[r] >= 1 && l >= 1;
                    ex[r][l] = oke ? fld_ldcg(Ex, off) : 0.0f;
                    ey[r][l] = oke ? fld_ldcg(Ey, off) : 0.0f;
                    ez[r][l] = oke ? fld_ldcg(Ez, off) : 0.0f;
                    FDTD_DEBUG_ONLY(if (ok) lev_check(P, P.levH, off, 0, 1); if (oke) lev_check(P, P.levE, off, 0, 2);)
                    const int cidx = r * SX + (gz & (BZ - 1)) * PLANE;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        if (COEF && LUT) {
                            const float2* lut = reinterpret_cast<const float2*>(sm + Lay<COEF>::lut);
                            const float2 pr = ok ? lut[c * MAXMAT + __ldg(P.g.cidx[c] + off)] : make_float2(0.0f, 0.0f);
                            cpair[cidx + c * (BZ * PLANE)] = coef_pair(P, c, pr.x, pr.y, gx, gy[r], gz);
                        } else if (COEF) {
                            const float a = ok ? __ldg(P.g.ca[c] + off) : 0.0f;
                            const float b = ok ? __ldg(P.g.cb[c] + off) : 0.0f;
                            cpair[cidx + c * (BZ * PLANE)] = coef_pair(P, c, a, b, gx, gy[r], gz);
                        } else {
                            cmask[cidx + c * (BZ * PLANE)] = cb_mask(P, c, gx, gy[r], gz);
                        }
                    }
                }
            }
#pragma unroll
            for (int l = 1; l < BZ; ++l) {
                exH[(l - 1) * PLANE + slot1] = make_float2(hz[RL][l], hx[RL][l]);
            }
        } else {
            TRACE_C(0, k);
            mbar_wait(mb + MB_HREADY, ph.hready & 1u);
            ++ph.hready;
            TRACE_C(1, k);
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                hx[r][0] = fld_get(stgH + zidxF(0, ly[r], xs));
                hy[r][0] = fld_get(stgH + zidxF(1, ly[r], xs));
                hz[r][0] = fld_get(stgH + zidxF(2, ly[r], xs));
            }
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                if (ly[r] == 0) {         // warp-uniform: the entering row
#pragma unroll
                    for (int l = 1; l < BZ; ++l) {
                        hx[r][l] = fld_get(stgH + yidxF(0, l, xs));
                        hy[r][l] = fld_get(stgH + yidxF(1, l, xs));
                        hz[r][l] = fld_get(stgH + yidxF(2, l, xs));
                        if (r == RL) {    // its y+1 neighbour is the next warp's row 0, which reads it from the exchange
                            exH[(l - 1) * PLANE + slot1] = make_float2(hz[r][l], hx[r][l]);
                        }
                    }
                }
            }
            if (lx == 0) {                // one lane per warp: the entering column, packed by the H-side warp
#pragma unroll
                for (int r = 0; r < NROW; ++r) {
                    if (ly[r] != 0) {
                        const float4* s4 = reinterpret_cast<const float4*>(xpkH + (ys0 + r) * 24);
                        const float4 a0 = s4[0], a1 = s4[1], b0 = s4[2], b1 = s4[3], c0 = s4[4], c1 = s4[5];
                        hx[r][1] = a0.y; hx[r][2] = a0.z; hx[r][3] = a0.w; hx[r][4] = a1.x; hx[r][5] = a1.y; hx[r][6] = a1.z; hx[r][7] = a1.w;
                        hy[r][1] = b0.y; hy[r][2] = b0.z; hy[r][3] = b0.w; hy[r][4] = b1.x; hy[r][5] = b1.y; hy[r][6] = b1.z; hy[r][7] = b1.w;
                        hz[r][1] = c0.y; hz[r][2] = c0.z; hz[r][3] = c0.w; hz[r][4] = c1.x; hz[r][5] = c1.y; hz[r][6] = c1.z; hz[r][7] = c1.w;
                    }
                }
            }
            warp_arrive(mb + MB_HFREE);
#ifdef FDTD_DEBUG
            // every H value just taken from the shell must have received exactly k updates in this launch
#pragma unroll
            for (int r = 0; r < NROW; ++r)
                for (int l = 0; l < BZ; ++l)
                    if ((l == 0 || ly[r] == 0 || lx == 0) && col_in[r] && (unsigned)(o2 + l) < (unsigned)nz)
                        lev_check(P, P.levH, col_off[r] + plane * (o2 + l), k, 3);
#endif
        }
        PROF_MARK(0);
        bar_sync(1, NCOMPUTE);   // exchange rows of H (shell + last H phase) and the scattered coefficients are visible

        PROF_MARK(1);
        TRACE_C(2, k);
        // ---------------- E phase on R_k = [1,w]^3 (a1): every slot computes, shell slots produce garbage ----
        // fast (no coefficient arrays, box never touches a wall or the outside): cb is the scalar dt, no mask loads
        auto e_phase = [&](auto fastc) {
        constexpr bool FAST = decltype(fastc)::value;
#pragma unroll
        for (int l = BZ - 1; l >= 1; --l) {
            const int cidx = ((o2 + l) & (BZ - 1)) * PLANE;
            const float2 h_ym = exH[(l - 1) * PLANE + slot_ym];
            const float hz_ym = h_ym.x, hx_ym = h_ym.y;
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                const float hz_xm = __shfl_sync(0xffffffffu, hz[r][l], lane_m);
                const float hy_xm = __shfl_sync(0xffffffffu, hy[r][l], lane_m);
                // y-1 neighbour: row 0 reads the previous warp's last row from the exchange, row 1 reads row 0's registers
                const float hz_y = r == 0 ? hz_ym : hz[r > 0 ? r - 1 : 0][l];
                const float hx_y = r == 0 ? hx_ym : hx[r > 0 ? r - 1 : 0][l];
                float cax = 1.0f, cay = 1.0f, caz = 1.0f, cbx, cby, cbz;
                if (COEF) {
                    const float2 px = cpair[cidx + r * SX], py = cpair[cidx + r * SX + BZ * PLANE], pz = cpair[cidx + r * SX + 2 * BZ * PLANE];
                    cax = px.x; cbx = px.y; cay = py.x; cby = py.y; caz = pz.x; cbz = pz.y;
                } else if (FAST) {
                    cbx = cby = cbz = P.g.cb_scalar;
                } else {
                    cbx = cmask[cidx + r * SX]; cby = cmask[cidx + r * SX + BZ * PLANE]; cbz = cmask[cidx + r * SX + 2 * BZ * PLANE];
                }
                // E_x: (Hz - Hz[j-1])/dy - (Hy - Hy[k-1])/dz      eq. (1)
                ex[r][l + 1] = fld_round(yee_e_update<COEF>(ex[r][l], hz[r][l], hz_y, hy[r][l], hy[r][l - 1], rdy, rdz, cax, cbx));
                // E_y: (Hx - Hx[k-1])/dz - (Hz - Hz[i-1])/dx
                ey[r][l + 1] = fld_round(yee_e_update<COEF>(ey[r][l], hx[r][l], hx[r][l - 1], hz[r][l], hz_xm, rdz, rdx, cay, cby));
                // E_z: (Hy - Hy[i-1])/dx - (Hx - Hx[j-1])/dy
                ez[r][l + 1] = fld_round(yee_e_update<COEF>(ez[r][l], hy[r][l], hy_xm, hx[r][l], hx_y, rdx, rdy, caz, cbz));
            }
        }
        };
        if (!COEF && fast) e_phase(std::true_type{});
        else e_phase(std::false_type{});
        // soft source after the E update of step t0 + k (a4): rare, CTA-uniform tests first.  P.src_org lists the images
        // of the source box (one on a wall grid; a box on a periodic axis also drives its copies in the ghost zones).
        {
            const long long ts = P.t0 + k;
            if (P.nsrc > 0 && ts >= 0 && ts < P.g.src_nwave) {
                for (int si = 0; si < P.nsrc; ++si) {
                    const int b0 = P.src_org[si][0], b1 = P.src_org[si][1], b2 = P.src_org[si][2];
                    if (b0 <= o0 + W0 && b0 + P.g.src_box[3] > o0 + 1 && b1 <= o1 + W1 && b1 + P.g.src_box[4] > o1 + 1 &&
                        b2 <= o2 + W2 && b2 + P.g.src_box[5] > o2 + 1) {
                        const float wsrc = __ldg(P.g.src_wave + ts);
                        const int sx = gx - b0;
#pragma unroll
                        for (int r = 0; r < NROW; ++r) {
                            const int sy = gy[r] - b1;
                            if ((lx >= 1) & (ly[r] >= 1) && sx >= 0 && sx < P.g.src_box[3] && sy >= 0 && sy < P.g.src_box[4]) {
#pragma unroll
                                for (int l = 1; l < BZ; ++l) {
                                    const int sz = o2 + l - b2;
                                    if (sz >= 0 && sz < P.g.src_box[5]) {
                                        const float amp = __ldg(P.g.src_amp + (sx + P.g.src_box[3] * (sy + (long long)P.g.src_box[4] * sz)));
                                        const float inj = amp * wsrc;
                                        if (P.g.src_comp == 0) ex[r][l + 1] = fld_round(ex[r][l + 1] + inj);
                                        else if (P.g.src_comp == 1) ey[r][l + 1] = fld_round(ey[r][l + 1] + inj);
                                        else ez[r][l + 1] = fld_round(ez[r][l + 1] + inj);
                                    }
                                }
                            }
                        }
                    }
                }
            }
        }
        // running DFT of E on the monitor plane: R_k = [o+1, o+W] on every axis
        if (MON && monitor_hits(P.mon, P.t0 + k, o0 + 1, o1 + 1, o2 + 1)) {
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                if ((lx >= 1) & (ly[r] >= 1) && col_in[r]) {
                    // planes o2 + 1 + l, l = 0..6, hold e?[r][l + 2]
                    monitor_add<2>(P.mon, P.mon.wE + (P.t0 + k) * P.mon.F * 2, 0, gx, gy[r], o2 + 1, ex[r], ey[r], ez[r]);
                }
            }
        }
        // E of row 0, planes 1..6, for the previous warp's row 1 in the H phase; the shell column lx = 0 is written by the
        // E-side warp
        if (lx != 0) {
#pragma unroll
            for (int l = 1; l < BZ - 1; ++l) {
                exE[l * PLANE + slot0] = make_float2(ez[0][l + 1], ex[0][l + 1]);
            }
        }
        PROF_MARK(2);
        TRACE_C(3, k);
        if (k > k0) {   // the signal warp has copied the x-out rows of step k-1 (and the DONE barriers cannot lap it)
            mbar_wait(mb + MB_ACKE, ph.acke & 1u);
            ++ph.acke;
        }
        // publish E of R_k \ R_{k+1} (everything at the last step)                                      (a8, a6)
#pragma unroll
        for (int r = 0; r < NROW; ++r) {
            if ((lx >= 1) & (ly[r] >= 1) && col_in[r] && !FDTD_DBG(P, 4)) {
                if ((unsigned)(o2 + W2) < (unsigned)nz) {            // the leaving plane l = 7: every column
                    const long long off = col_off[r] + plane * (o2 + W2);
                    fld_stcg(Ex, off, ex[r][W2 + 1]);
                    fld_stcg(Ey, off, ey[r][W2 + 1]);
                    fld_stcg(Ez, off, ez[r][W2 + 1]);
                    FDTD_DEBUG_ONLY(lev_set(P.levE, off, k + 1);)
                }
                if (last | (ly[r] == W1)) {                          // warp-uniform: the leaving row (or the whole tile), planes 1..6
                    long long off = col_off[r] + plane * (o2 + 1);
#pragma unroll
                    for (int l = 1; l < W2; ++l) {
                        if ((unsigned)(o2 + l) < (unsigned)nz) {
                            fld_stcg(Ex, off, ex[r][l + 1]);
                            fld_stcg(Ey, off, ey[r][l + 1]);
                            fld_stcg(Ez, off, ez[r][l + 1]);
                            FDTD_DEBUG_ONLY(lev_set(P.levE, off, k + 1);)
                        }
                        off += plane;
                    }
                } else if (lx == W0) {                               // one lane per warp: the leaving column goes out through
                    float* xo = sm + Lay<COEF>::xoute + (ys0 + r) * 24;   // shared memory; the signal warp stores it
#pragma unroll
                    for (int l = 1; l < W2; ++l) {
                        xo[l] = ex[r][l + 1];
                        xo[8 + l] = ey[r][l + 1];
                        xo[16 + l] = ez[r][l + 1];
                    }
                }
            }
        }
        warp_arrive(mb + MB_EDONE);
        TRACE_C(4, k);
        FDTD_DEBUG_ONLY(if (P.delay_seed != 0u) debug_delay(P, tile, k, 1);)

        // ---------------- E minus shell -------------------------------------------------------------------------
        PROF_MARK(3);
        mbar_wait(mb + MB_EREADY, ph.eready & 1u);
        ++ph.eready;
        PROF_MARK(4);
        TRACE_C(5, k);
#pragma unroll
        for (int r = 0; r < NROW; ++r) {
            ex[r][1] = fld_get(stgE + zidxF(0, ly[r], xs));
            ey[r][1] = fld_get(stgE + zidxF(1, ly[r], xs));
            ez[r][1] = fld_get(stgE + zidxF(2, ly[r], xs));
        }
        exE[slot0] = make_float2(ez[0][1], ex[0][1]);
#pragma unroll
        for (int r = 0; r < NROW; ++r) {
            if (ly[r] == 0) {             // warp-uniform: the entering row
#pragma unroll
                for (int l = 1; l < BZ; ++l) {
                    ex[r][l + 1] = fld_get(stgE + yidxF(0, l, xs));
                    ey[r][l + 1] = fld_get(stgE + yidxF(1, l, xs));
                    ez[r][l + 1] = fld_get(stgE + yidxF(2, l, xs));
                }
            }
        }
        if (lx == 0) {
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                if (ly[r] != 0) {
                    const float4* s4 = reinterpret_cast<const float4*>(xpkE + (ys0 + r) * 24);
                    const float4 a0 = s4[0], a1 = s4[1], b0 = s4[2], b1 = s4[3], c0 = s4[4], c1 = s4[5];
                    ex[r][2] = a0.y; ex[r][3] = a0.z; ex[r][4] = a0.w; ex[r][5] = a1.x; ex[r][6] = a1.y; ex[r][7] = a1.z; ex[r][8] = a1.w;
                    ey[r][2] = b0.y; ey[r][3] = b0.z; ey[r][4] = b0.w; ey[r][5] = b1.x; ey[r][6] = b1.y; ey[r][7] = b1.z; ey[r][8] = b1.w;
                    ez[r][2] = c0.y; ez[r][3] = c0.z; ez[r][4] = c0.w; ez[r][5] = c1.x; ez[r][6] = c1.y; ez[r][7] = c1.z; ez[r][8] = c1.w;
                }
            }
        }
        warp_arrive(mb + MB_EFREE);
#ifdef FDTD_DEBUG
        // every E value just taken from the shell must have received exactly k+1 updates in this launch
#pragma unroll
        for (int r = 0; r < NROW; ++r)
            for (int l = 0; l < BZ; ++l)
                if ((l == 0 || ly[r] == 0 || lx == 0) && col_in[r] && (unsigned)(o2 + l) < (unsigned)nz)
                    lev_check(P, P.levE, col_off[r] + plane * (o2 + l), k + 1, 4);
#endif
        bar_sync(1, NCOMPUTE);   // exchange rows of E are visible; every warp has finished E phase k
        PROF_MARK(5);
        TRACE_C(6, k);
        // ---------------- coefficients of the cells that entered with this step's shell ------------------------------
        // first used by E phase k+1 (shell cells are not in R_k); copied a whole step ahead (issued after CFREE(k-1))
        if (k >= 1 && !fast) {
            if (COEF) {
                mbar_wait(mb + MB_CFULL, ph.cfull & 1u);
                ++ph.cfull;
            }
            absorb_coef_shell<COEF>(P, sm, o0, o1, o2, lx, ly, ys0);
            warp_arrive(mb + MB_CFREE);
        }
        PROF_MARK(7);
        TRACE_C(7, k);

        // ---------------- H phase on R_{k+1} = [0,w-1]^3 (a2): every slot computes ----------------------------
#pragma unroll
        for (int l = BZ - 2; l >= 0; --l) {
            const float2 e_yp = exE[l * PLANE + slot_yp];
            const float ez_yp = e_yp.x, ex_yp = e_yp.y;
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                const float ey_xp = __shfl_sync(0xffffffffu, ey[r][l + 1], lane_p);
                const float ez_xp = __shfl_sync(0xffffffffu, ez[r][l + 1], lane_p);
                // y+1 neighbour: the last row reads the next warp's row 0 from the exchange, row 0 of two reads row 1's registers
                const float ez_y = r == RL ? ez_yp : ez[r < RL ? r + 1 : RL][l + 1];
                const float ex_y = r == RL ? ex_yp : ex[r < RL ? r + 1 : RL][l + 1];
                hx[r][l + 1] = fld_round(yee_h_update(hx[r][l], ez_y, ez[r][l + 1], ey[r][l + 2], ey[r][l + 1], rdy, rdz, dbx));   // (Ez[j+1]-Ez)/dy - (Ey[k+1]-Ey)/dz
                hy[r][l + 1] = fld_round(yee_h_update(hy[r][l], ex[r][l + 2], ex[r][l + 1], ez_xp, ez[r][l + 1], rdz, rdx, dby));   // (Ex[k+1]-Ex)/dz - (Ez[i+1]-Ez)/dx
                hz[r][l + 1] = fld_round(yee_h_update(hz[r][l], ey_xp, ey[r][l + 1], ex_y, ex[r][l + 1], rdx, rdy, dbz));           // (Ey[i+1]-Ey)/dx - (Ex[j+1]-Ex)/dy
            }
            exH[l * PLANE + slot1] = make_float2(hz[RL][l + 1], hx[RL][l + 1]);
        }
        // running DFT of H on the monitor plane: R_{k+1} = [o, o+W-1] on every axis
        if (MON && monitor_hits(P.mon, P.t0 + k, o0, o1, o2)) {
#pragma unroll
            for (int r = 0; r < NROW; ++r) {
                if ((lx <= W0 - 1) & (ly[r] <= W1 - 1) && col_in[r]) {
                    // planes o2 + l, l = 0..6, hold h?[r][l + 1]
                    monitor_add<1>(P.mon, P.mon.wH + (P.t0 + k) * P.mon.F * 2, 3, gx, gy[r], o2, hx[r], hy[r], hz[r]);
                }
            }
        }
        TRACE_C(8, k);
        if (k > k0) {   // the signal warp has copied the H x-out rows of step k-1 (HDONE cannot lap its waiters)
            mbar_wait(mb + MB_ACKH, ph.ackh & 1u);
            ++ph.ackh;
        }
        // publish H of R_{k+1} \ R_{k+2} (everything at the last step)                                  (a8, a6)
#pragma unroll
        for (int r = 0; r < NROW; ++r) {
            if ((lx <= W0 - 1) & (ly[r] <= W1 - 1) && col_in[r] && !FDTD_DBG(P, 4)) {
                if ((unsigned)(o2 + W2 - 1) < (unsigned)nz) {        // the leaving plane l = 6: every column
                    const long long off = col_off[r] + plane * (o2 + W2 - 1);
                    fld_stcg(Hx, off, hx[r][W2]);
                    fld_stcg(Hy, off, hy[r][W2]);
                    fld_stcg(Hz, off, hz[r][W2]);
                    FDTD_DEBUG_ONLY(lev_set(P.levH, off, k + 1);)
                }
                if (last | (ly[r] == W1 - 1)) {                      // warp-uniform: leaving row (or whole tile), planes 0..5
                    long long off = col_off[r] + plane * o2;
#pragma unroll
                    for (int l = 0; l < W2 - 1; ++l) {
                        if ((unsigned)(o2 + l) < (unsigned)nz) {
                            fld_stcg(Hx, off, hx[r][l + 1]);
                            fld_stcg(Hy, off, hy[r][l + 1]);
                            fld_stcg(Hz, off, hz[r][l + 1]);
                            FDTD_DEBUG_ONLY(lev_set(P.levH, off, k + 1);)
                        }
                        off += plane;
                    }
                } else if (lx == W0 - 1) {                           // the leaving column: out through shared memory
                    float* xo = sm + Lay<COEF>::xouth + (ys0 + r) * 24;
#pragma unroll
                    for (int l = 0; l < W2 - 1; ++l) {
                        xo[l] = hx[r][l + 1];
                        xo[8 + l] = hy[r][l + 1];
                        xo[16 + l] = hz[r][l + 1];
                    }
                }
            }
        }
        warp_arrive(mb + MB_HDONE);
        TRACE_C(9, k);
        FDTD_DEBUG_ONLY(if (P.delay_seed != 0u) debug_delay(P, tile, k, 2);)
        PROF_MARK(6);
    }
    if (threadIdx.x < 32) PROF_FLUSH(0);
    // the signal warp's last ack of this tile is covered by the CTA barrier at the tile boundary
    if (k1 > k0) { ++ph.acke; ++ph.ackh; }
}

// MON: a running-DFT monitor is set (a separate instantiation keeps its rare path out of the product loop)
template <bool COEF, bool MON>
__global__ void __launch_bounds__(NT, CTAS_PER_SM) systolic_tma_kernel(const __grid_constant__ SysParams P, const __grid_constant__ TmaMaps M)
{
    extern __shared__ __align__(128) float sm[];
    __shared__ __align__(8) unsigned long long mb[MB_COUNT];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // the next launch of the stream may be scheduled as soon as SMs drain (its tiles wait on flags, see pred_final)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (blockIdx.x == 0 && tid == 0 && P.counter_zero) *P.counter_zero = 0u;
    if (tid == 0) {
#ifdef FDTD_PROFILE
        trace_on_ = 0;
        trace_cur_ = 0u;
#endif
        ctl.abort = 0;
        mbar_init(mb + MB_HFULL, 1);
        mbar_init(mb + MB_CFULL, 1);
        mbar_init(mb + MB_EFULL, 1);
        mbar_init(mb + MB_HREADY, 1);
        mbar_init(mb + MB_CFREE, NWARPS_C);
        mbar_init(mb + MB_EREADY, 1);
        mbar_init(mb + MB_HFREE, NWARPS_C);
        mbar_init(mb + MB_EFREE, NWARPS_C);
        mbar_init(mb + MB_EDONE, NWARPS_C);
        mbar_init(mb + MB_HDONE, NWARPS_C);
        mbar_init(mb + MB_ACKE, 1);
        mbar_init(mb + MB_ACKH, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // Shell slots and cells outside the grid compute on whatever the shared arrays hold and rely on 0 * garbage = 0:
    // the garbage must be finite.  Shared memory keeps the bits of earlier kernels (possibly NaN patterns), so it is
    // cleared once per CTA; from then on every value in it derives from finite data.
    for (int i = tid; i < Lay<COEF>::total; i += NT) sm[i] = 0.0f;
    if (COEF && LUT) {      // the (ca, cb) table of the index build: [3][nmat] pairs from global memory, rest stays 0
        __syncthreads();
        const float2* src = reinterpret_cast<const float2*>(P.g.lut);
        float2* dst = reinterpret_cast<float2*>(sm + Lay<COEF>::lut);
        for (int i = tid; i < 3 * P.g.nmat; i += NT) dst[(i / P.g.nmat) * MAXMAT + i % P.g.nmat] = src[i];
    }
    const CUtensorMap* maps = reinterpret_cast<const CUtensorMap*>(M.bytes);   // [E0 E1 E2 H0 H1 H2 ca0..2 cb0..2][3 faces]
    // Acquire the flags of step k+1 (and run the ~0.7 us proxy fence) while the copy of step k is in flight, instead of
    // at the top of iteration k+1.  Measured: +5 % at 768^3 without coefficient arrays, -2 % on config 2 with them (the
    // field copies then queue earlier against the coefficient copies), hence per instantiation.
    constexpr bool EARLY = !COEF;
    Phases ph = {0u, 0u, 0u, 0u, 0u};

    // One tile claim: CTA-wide barriers around the claim and around the late-start clearing.  Both role loops below call
    // it the same number of times, so the barriers match although they are executed from two places.
    auto next_tile = [&](TileJob& J) -> bool {
        bar_sync(0, NT);
        if (tid == 0) {
            ctl.tile = (int)atomicAdd(P.counter, 1u);
            if (ld_volatile(P.abort_flag) != 0) ctl.abort = 1;
#ifdef FDTD_PROFILE
            trace_on_ = (blockIdx.x == 0 && P.prof != nullptr && (int)ctl.tile >= P.ntiles / 2) ? 1 : 0;
#endif
        }
        bar_sync(0, NT);
        if (ctl.tile >= P.ntiles || ctl.abort) return false;
        // claim order = wavefront order (P.order sorts the tiles by bx+by+bz): the tiles in flight at any time lie on
        // one or two anti-diagonal planes and do not depend on each other, their upwind tiles were claimed a whole
        // tile lifetime earlier -- the hand-off latency then never stalls a step
        const int tile = P.order ? P.order[ctl.tile] : ctl.tile;
        TileGeom& t = J.t;
        tile_init(P, tile, t);
        const int T = P.T;
        // a11: steps at which the tile's region lies wholly outside the grid do nothing and publish nothing.  The region
        // [a-k, a+w-k) meets [0,n) on every axis for k in [kin, kout); the tile runs [k0, k1) = [kin-1, kout) -- one step
        // early, because the cells of R_kin enter as the minus shell of step kin-1 -- and its flags jump over the rest.
        int k0 = 0, k1 = T;
        for (int q = 0; q < 3; ++q) {
            const int wq = q == 0 ? W0 : q == 1 ? W1 : W2;
            k0 = max(k0, t.a[q] - P.g.n[q]);          // kin - 1 = a - n
            k1 = min(k1, t.a[q] + wq);
        }
        if (k1 < k0) k1 = k0;
        if (FDTD_DBG(P, 64)) { k0 = 0; k1 = T; }
        // no coefficient arrays and the box stays strictly inside the grid (never index 0, never outside) for the whole
        // launch: every cb mask would be dt -- the tile runs without masks, without their scatter and without CREADY/CFREE
        bool fast = !COEF && !FDTD_DBG(P, 256);
        for (int q = 0; q < 3; ++q) {
            const int wq = q == 0 ? W0 : q == 1 ? W1 : W2;
            fast = fast && (t.a[q] - k1 >= 1) && (t.a[q] - k0 + wq <= P.g.n[q]);
        }
        if (P.pred_final != 0 && tid < 27 && !ctl.abort) {
            // Launch-to-launch overlap.  Read-after-write: the cells of the box [a-1, a+w) were finalised, at step T-1 of the
            // previous launch, by the tiles whose start lies in (a-1+T-w, a+w-1+T] on every axis: two per axis, indices jlo
            // and jlo+1.  Write-after-read: those final values are also the last minus shells of the downwind neighbours of
            // these tiles (index +1 per axis), which must have read them before anything of this launch overwrites them.
            // Every tile of this launch therefore waits for the last flag of the 3 x 3 x 3 tiles jlo .. jlo+2 of the previous
            // launch (cells that reach a tile later, through shells, were covered by the tile that loaded them in its box).
            int u = 0, div = 9;
            const bool ok = true;
            for (int q = 2; q >= 0; --q) {
                const int wq = q == 0 ? W0 : q == 1 ? W1 : W2;
                const int lo = t.a[q] - 1 + T - wq;
                const int jlo = (lo >= 0 ? lo / wq : -((-lo + wq - 1) / wq)) + 1;      // floor(lo / w) + 1
                // clamped to the tile grid: beyond it there is nothing to wait for on this axis, but the other axes still
                // count, and a tile must never raise a flag that its own predecessor (same index, <= every tile waited for)
                // has not finished with -- the flag values of the two launches share one array
                const int j = min(max(jlo + (tid / div) % 3, 0), P.ax[q].nb - 1);
                div /= 3;
                u = u * P.ax[q].nb + j;
            }
            if (ok && ld_acquire(P.flagH + u) < P.pred_final) {
                const long long t_start = clock64();
                unsigned spins = 0;
                while (ld_acquire(P.flagH + u) < P.pred_final) {
                    if ((++spins & 63u) == 0u) {
                        if (ld_volatile(P.abort_flag) != 0) { *(volatile int*)&ctl.abort = 1; break; }
                        if (clock64() - t_start > P.spin_budget) {
                            atomicExch(P.abort_flag, 1);
                            *(volatile int*)&ctl.abort = 1;
                            break;
                        }
                    }
                    __nanosleep(64);
                }
            }
        }
        if (k0 > 0 && warp < NWARPS_C) {
            // started late: nothing is loaded from the grid; the box holds zero fields (registers) and zero coefficients
            float* cs = sm + Lay<COEF>::coef;
            for (int i = tid; i < Lay<COEF>::NC * BZ * PLANE; i += NCOMPUTE) cs[i] = 0.0f;
        }
        bar_sync(0, NT);
        J.tile = tile; J.k0 = k0; J.k1 = k1; J.fast = fast;
        return true;
    };

    // Register split (setmaxnreg): the launch gives each of the 384 threads 168 registers; the compute code keeps 102 field
    // values per thread and wants room to hoist loads, the auxiliary warps need few.  Each role has its own tile loop so
    // that the register budget of a region is the one set at its head.
    if (warp < NWARPS_C) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_COMPUTE));
        TileJob J;
        while (next_tile(J)) compute_tile<COEF, MON>(P, J.t, J.tile, J.k0, J.k1, J.fast, sm, mb, ph);
        return;
    }
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_AUX));
    // one instantiation of the auxiliary tile loop per role (the role is a compile-time constant inside): each keeps only
    // its own phase counters and geometry alive
    auto aux_loop = [&](auto rolec) {
    constexpr int warp = decltype(rolec)::value;      // shadows the run-time warp index
    // completed phases of every mbarrier this role waits on (each role counts only what it uses)
    unsigned n_hfull = 0, n_cfull = 0, n_efull = 0, n_hfree = 0, n_cfree = 0, n_efree = 0, n_edone = 0, n_hdone = 0;
    TileJob J;
    while (next_tile(J)) {
        const TileGeom& t = J.t;
        const int tile = J.tile, k0 = J.k0, k1 = J.k1, T = P.T;
        const bool fast = J.fast;
        if (warp == W_HPROD || warp == W_HAUX) {
            // H side: shell of step k needs the staging of step k-1 absorbed (HFREE), the upwind tiles' H of
            // step k-1 published (flagH), and -- before the coefficient slots are overwritten -- E phase k-1 done
            PROF_DECL;
            const int hk0 = max(k0, 1);       // step 0 loads its whole box itself
            for (int j = k0; j <= k1; ++j) {
                if (j >= hk0 && j < k1) {
                    const int k = j;
                    const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
                    PROF_MARK(7);
                    if (warp == W_HPROD) {
                        TRACE(1, 0, k);
                        // field shell: acquire the upwind flags and order the async proxy after them while the staging is
                        // still in use, copy, repack the entering column -> HREADY(k)
                        if (k == hk0 || !EARLY) {      // later steps: acquired while the previous copy was in flight
                            wait_upwind(P, t, P.flagH, P.flag_base + k, &ctl);
                            if (lane == 0 && !FDTD_DBG(P, 32)) fence_proxy_async();
                        }
                        PROF_MARK(0);
                        TRACE(1, 1, k);
                        if (k > hk0) { mbar_wait(mb + MB_HFREE, n_hfree & 1u); ++n_hfree; }
                        PROF_MARK(1);
                        TRACE(1, 2, k);
                        if (lane == 0 && !FDTD_DBG(P, 2)) issue_shell<3, true>(maps + 3 * 3, P.tma_group[1], sm + Lay<COEF>::stgh, o0, o1, o2, mb + MB_HFULL);
                        __syncwarp();
                        if (k + 1 < k1 && EARLY) {
                            wait_upwind(P, t, P.flagH, P.flag_base + k + 1, &ctl);
                            if (lane == 0 && !FDTD_DBG(P, 32)) fence_proxy_async();
                        }
                        PROF_MARK(2);
                        TRACE(1, 3, k);
                        if (!FDTD_DBG(P, 2)) { mbar_wait(mb + MB_HFULL, n_hfull & 1u); ++n_hfull; }
                        PROF_MARK(3);
                        TRACE(1, 4, k);
                        pack_xcol(reinterpret_cast<const fld_t*>(sm + Lay<COEF>::stgh), sm + Lay<COEF>::xpkh, o0, o1);
                        warp_arrive(mb + MB_HREADY);
                        TRACE(1, 5, k);
                        PROF_MARK(4);
                    } else {
                        // coefficient shell (constants of the run: no flag, no proxy fence): copied as soon as the compute
                        // warps have taken the previous one out of the staging (CFREE), a whole step before it is needed
                        if (COEF && !fast) {         // (a uniform tile has no coefficient copy)
                        TRACE(2, 0, k);
                        if (k > hk0) { mbar_wait(mb + MB_CFREE, n_cfree & 1u); ++n_cfree; }
                        PROF_MARK(0);
                        TRACE(2, 1, k);
                        if (lane == 0 && !FDTD_DBG(P, 2)) {
                            if (LUT) issue_index_shell(maps + 6 * 3, P.tma_group[2], sm + Lay<COEF>::stgc, o0, o1, o2, mb + MB_CFULL);
                            else issue_shell<6, false>(maps + 6 * 3, P.tma_group[2], sm + Lay<COEF>::stgc, o0, o1, o2, mb + MB_CFULL);
                        }
                        __syncwarp();
                        PROF_MARK(1);
                        }
                    }
                }
            }
            if (warp == W_HPROD) PROF_FLUSH(8);
            if (warp == W_HAUX) PROF_FLUSH(16);
            // phases of the last step that this warp does not wait for: covered by the CTA barrier at the tile boundary
            if (k1 > hk0) { if (warp == W_HPROD) ++n_hfree; else if (COEF && !fast) ++n_cfree; }
        } else if (warp == W_EPROD) {
            // the flags of step k are acquired (and the async proxy ordered after them) while the copy of step k-1 is in
            // flight: the ~0.7 us proxy fence is off the EFREE -> EREADY chain
            if (k0 < k1) {
                wait_upwind(P, t, P.flagE, P.flag_base + k0 + 1, &ctl);
                if (lane == 0 && !FDTD_DBG(P, 32)) fence_proxy_async();
            }
            for (int k = k0; k < k1; ++k) {
                const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
                if (k > k0 && !EARLY) {
                    wait_upwind(P, t, P.flagE, P.flag_base + k + 1, &ctl);
                    if (lane == 0 && !FDTD_DBG(P, 32)) fence_proxy_async();
                }
                TRACE(3, 0, k);
                if (k > k0) {
                    mbar_wait(mb + MB_EFREE, n_efree & 1u); ++n_efree;     // staging of step k-1 absorbed
                }
                TRACE(3, 1, k);
                if (lane == 0 && !FDTD_DBG(P, 2)) issue_shell<3, true>(maps, P.tma_group[0], sm + Lay<COEF>::stge, o0, o1, o2, mb + MB_EFULL);
                __syncwarp();
                if (k + 1 < k1 && EARLY) {
                    wait_upwind(P, t, P.flagE, P.flag_base + k + 2, &ctl);
                    if (lane == 0 && !FDTD_DBG(P, 32)) fence_proxy_async();
                }
                TRACE(3, 2, k);
                if (!FDTD_DBG(P, 2)) { mbar_wait(mb + MB_EFULL, n_efull & 1u); ++n_efull; }
                TRACE(3, 4, k);
                const fld_t* stg = reinterpret_cast<const fld_t*>(sm + Lay<COEF>::stge);
                pack_xcol(stg, sm + Lay<COEF>::xpke, o0, o1);
                TRACE(3, 5, k);
                if (k > k0) { mbar_wait(mb + MB_HDONE, n_hdone & 1u); ++n_hdone; }   // H phase k-1 has read the E exchange rows
                TRACE(3, 6, k);
                // the shell column's Ez, Ex of planes 1..6 for its y-1 readers in the H phase
                float2* exE = reinterpret_cast<float2*>(sm + Lay<COEF>::exch) + EXP;
                for (int r = 0; r < 3; ++r) {
                    const int idx = r * 32 + lane;            // (l-1)*15 + (ly-1), l = 1..6
                    if (idx < W1 * (W2 - 1)) {
                        const int ly = 1 + idx % W1, l = 1 + idx / W1;
                        const int s = ((o1 + ly) & (BY - 1)) * SX + (o0 & (BX - 1));
                        exE[l * PLANE + s] = make_float2(fld_get(stg + xidxF(2, ly, l) + (o0 & XMASK_F)), fld_get(stg + xidxF(0, ly, l) + (o0 & XMASK_F)));
                    }
                }
                warp_arrive(mb + MB_EREADY);
                TRACE(3, 7, k);
            }
            if (k1 > k0) { ++n_efree; ++n_hdone; }   // phases of the last step: covered by the CTA barrier at the tile boundary
        } else {
            // signal warp.  Every publish of a phase has been issued before its warp arrived on the DONE barrier.  The
            // leaving x columns are copied out of shared memory as soon as their phase is done and acknowledged at once, so
            // the compute warps never wait for the fence; both columns are stored, ONE gpu-scope fence orders every publish
            // of the step (cumulative over what this warp observed through the mbarriers), then both flags go up.     (a9)
            // Steps outside [k0, k1) publish nothing: their flags are raised at once.
            if (k0 > 0 && lane == 0) {
                raise_flag(P, P.flagE, tile, P.flag_base + k0);
                raise_flag(P, P.flagH, tile, P.flag_base + k0);
            }
            for (int k = k0; k < k1; ++k) {
                const int o0 = t.a[0] - k - 1, o1 = t.a[1] - k - 1, o2 = t.a[2] - k - 1;
                XCol ce, ch;
                TRACE(4, 0, k);
                mbar_wait(mb + MB_EDONE, n_edone & 1u); ++n_edone;
                TRACE(4, 1, k);
                load_xcol(ce, sm + Lay<COEF>::xoute, 1);
                __syncwarp();
                if (lane == 0) mbar_arrive(mb + MB_ACKE);
                TRACE(4, 2, k);
                mbar_wait(mb + MB_HDONE, n_hdone & 1u); ++n_hdone;
                TRACE(4, 3, k);
                load_xcol(ch, sm + Lay<COEF>::xouth, 0);
                __syncwarp();
                if (lane == 0) mbar_arrive(mb + MB_ACKH);
                if (k != T - 1 && !FDTD_DBG(P, 4)) {
                    store_xcol(P, P.g.E, ce, o0 + W0, o1, o2, 1, W1 - 1, 1, P.levE, k + 1);
                    store_xcol(P, P.g.H, ch, o0 + W0 - 1, o1, o2, 0, W1 - 2, 0, P.levH, k + 1);
                }
                __syncwarp();
                TRACE(4, 5, k);
                if (lane == 0) {
                    fence_acq_rel_gpu();
                    FDTD_DEBUG_ONLY(if (tile != P.withhold_tile))
                    {
                        st_relaxed(P.flagE + tile, P.flag_base + k + 1);
                        st_relaxed(P.flagH + tile, P.flag_base + k + 1);
                    }
                }
                __syncwarp();
                TRACE(4, 6, k);
            }
            if (k1 < T && lane == 0) {
                raise_flag_max(P, P.flagE, tile, P.flag_base + T);
                raise_flag_max(P, P.flagH, tile, P.flag_base + T);
            }
        }
    }
    };
    if (warp == W_HPROD) aux_loop(std::integral_constant<int, W_HPROD>{});
    else if (warp == W_HAUX) aux_loop(std::integral_constant<int, W_HAUX>{});
    else if (warp == W_EPROD) aux_loop(std::integral_constant<int, W_EPROD>{});
    else aux_loop(std::integral_constant<int, W_EPROD + 1>{});
}

}  // namespace

size_t FDTD_TMA_NAME(systolic_tma_smem)(int coef) { return (size_t)(coef ? Lay<true>::total : Lay<false>::total) * sizeof(float); }
int FDTD_TMA_NAME(systolic_tma_threads)() { return NT; }
void FDTD_TMA_NAME(systolic_tma_boxes)(int fld[3][3], int coef[3][3])
{
    const int bf[3][3] = {{RXF, BY, 1}, {RXF, 1, BZ}, {CWF, BY, W2}};
    const int bc[3][3] = {{LUT ? RXB : RX, BY, 1}, {LUT ? RXB : RX, 1, BZ}, {LUT ? CWB : 4, BY, W2}};
    for (int f = 0; f < 3; ++f)
        for (int q = 0; q < 3; ++q) {
            fld[f][q] = bf[f][q];
            coef[f][q] = bc[f][q];
        }
}

cudaError_t FDTD_TMA_NAME(systolic_tma_prepare)(int coef, int* blocks_per_sm)
{
    const void* fn = coef ? (const void*)&systolic_tma_kernel<true, false> : (const void*)&systolic_tma_kernel<false, false>;
    const void* fm = coef ? (const void*)&systolic_tma_kernel<true, true> : (const void*)&systolic_tma_kernel<false, true>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FDTD_TMA_NAME(systolic_tma_smem)(coef));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fm, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FDTD_TMA_NAME(systolic_tma_smem)(coef));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, fn, NT, FDTD_TMA_NAME(systolic_tma_smem)(coef));
}

cudaError_t FDTD_TMA_NAME(launch_systolic_tma)(int coef, const SysParams& p, const TmaMaps& maps, int ctas, cudaStream_t st)
{
    static_assert(sizeof(CUtensorMap) == 128, "TmaMaps layout");
    const void* fn = p.mon.on ? (coef ? (const void*)&systolic_tma_kernel<true, true> : (const void*)&systolic_tma_kernel<false, true>)
                              : (coef ? (const void*)&systolic_tma_kernel<true, false> : (const void*)&systolic_tma_kernel<false, false>);
    void* args[] = {(void*)&p, (void*)&maps};
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)ctas);
    cfg.blockDim = dim3((unsigned)NT);
    cfg.dynamicSmemBytes = FDTD_TMA_NAME(systolic_tma_smem)(coef);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.pred_final != 0 ? 1 : 0;       // overlap with the previous launch only when its flags are this launch's gate
    return cudaLaunchKernelExC(&cfg, fn, args);
}
