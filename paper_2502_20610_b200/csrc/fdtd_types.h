// fdtd_types.h -- plain structs of libfdtd_b200 shared by host and device code (CUDA path only; nothing under
// oracle/ includes this).  No CUDA headers: tests/emu builds the tile stage functions with plain g++.
#pragma once
#include <stddef.h>
#include <stdint.h>

#ifndef FDTD_HD
#ifdef __CUDACC__
#define FDTD_HD __host__ __device__ __forceinline__
#else
#define FDTD_HD inline
#endif
#endif

// Everything a kernel needs about the grid (passed by value as a __grid_constant__ kernel parameter).
struct GridParams {
    float* E[3];
    float* H[3];
    const float* ca[3];  // all NULL or all set
    const float* cb[3];  // all NULL or all set
    // compressed coefficients (row f2): one material index per cell and component and a table of (ca, cb)
    // pairs per component; replaces ca / cb (which are then NULL):  ca_a[p] = lut[(a*nmat + cidx[a][p])*2], cb_a[p] = ...*2 + 1
    const unsigned char* cidx[3];   // all NULL or all set
    const float* lut;               // device, [3][nmat][2]
    int nmat;
    int fld16;           // 1: E and H point to IEEE binary16 arrays (row f1); arithmetic stays f32
    int n[3];
    int per[3];          // 1 = periodic axis
    float rd[3];         // (float)(1.0 / (double)d_a)                    (reading #2)
    float cb_scalar;     // dt, used where cb == NULL
    float db[3];
    // soft source (reading #6)
    int src_comp;        // -1: none
    int src_box[6];      // i0 j0 k0 ni nj nk
    const float* src_amp;   // device copy, ni*nj*nk
    const float* src_wave;  // device copy, nwave
    int src_nwave;
};

// One axis of the systolic tile schedule (SURVEY.md section 7 hard part 3 / DESIGN.md reading #11).
//   PEC axis:      tiles b = 0 .. nb-1, nb = ceil((n+T)/N), start(b) = b*N, width N; regions are clipped to
//                  [0,n): tiles enter empty at the high wall and drain at the low wall.
//   periodic axis: a ring of nb = ceil(n/N) tiles of widths base+1 (first rem tiles) or base, all <= N.
// At step s of a launch tile b owns [start(b) - s, start(b) + width(b) - s)  (the x-y-z-t diagonal).
struct AxisPlan {
    int n, per, N, nb, base, rem;
    FDTD_HD int start(int b) const { return per ? b * base + (b < rem ? b : rem) : b * N; }
    FDTD_HD int width(int b) const { return per ? base + (b < rem ? 1 : 0) : N; }
};

inline AxisPlan make_axis_plan(int n, int per, int N, int T)
{
    AxisPlan a;
    a.n = n; a.per = per; a.N = N;
    if (per) {
        a.nb = (n + N - 1) / N;
        a.base = n / a.nb;
        a.rem = n % a.nb;
    } else {
        a.nb = (n + T + N - 1) / N;
        a.base = N;
        a.rem = 0;
    }
    return a;
}

// Developer builds only (-DFDTD_DEBUG: the "dbg" and "prof" variants of build.py): timing probes that skip work
// (results invalid), fault injection (pseudo-random sleeps, a withheld flag) and the time-level shadow arrays.
// The product libraries compile every one of them out: FDTD_DBG() is the constant false there.
#ifdef FDTD_DEBUG
#define FDTD_DBG(P, bit) (((P).dbg & (bit)) != 0)
#define FDTD_DEBUG_ONLY(...) __VA_ARGS__
#else
#define FDTD_DBG(P, bit) false
#define FDTD_DEBUG_ONLY(...)
#endif

constexpr int MAX_SRC_IMAGES = 125;
constexpr int FDTD_TRACE_CAP = 1 << 16;   // FDTD_PROFILE build: events of the traced CTA, behind the 32 tick accumulators of SysParams::prof

// The padded working copy of the grid (pad_kernels.cu): a periodic axis a carries G[a] ghost cells on
// either side (m[a] = n[a] + 2 G[a]); wall axes have G[a] = 0; rows are ldx >= m[0] elements long (a multiple of 4).
struct PadGeom {
    int n[3];
    int m[3];
    int G[3];
    long long ldx;
};
struct PadArrays {
    float* usr[6];        // the caller's arrays (n[0]*n[1]*n[2] each)
    float* ext;           // narr padded arrays of ldx*m[1]*m[2] elements at a uniform stride
    long long stride;     // in elements
    int narr;
    int elem16;           // 1: binary16 elements, 2: one-byte elements (material indices); usr / ext then hide them behind float pointers
};

// Running-DFT monitor on one plane of the grid (PAPER.md:106 names outputs as what real runs carry;
// DESIGN.md reading #15).  During step t (0 <= t < nt), for every cell of the plane and every frequency f:
//     after the E half-step and the source:  acc[a][f][re|im][cell]     += E_a * wE[t][f][re|im]     a = 0..2
//     after the H half-step:                 acc[3 + a][f][re|im][cell] += H_a * wH[t][f][re|im]
// (product rounded, then the add).  Plane cells are numbered x fastest over the two remaining axes of the CALLER's grid.
struct MonitorParams {
    int on;               // 0: no monitor
    int axis, index;      // plane axis; plane index in WORKING coordinates (caller index + G[axis])
    int F, nt;
    int n[3];             // extents of the caller's grid
    int G[3];             // working coordinate = caller coordinate + G (the padded copy of DESIGN.md 6.4), else 0
    const float* wE;      // device, [nt][F][2]
    const float* wH;
    float* acc;           // device, [6][F][2][pcells], borrowed from the caller
    long long pcells;
    // cell number inside the plane of the working-grid cell (gx,gy,gz), or -1 when the cell is not on the plane or is a
    // ghost image outside the caller's grid
    FDTD_HD long long cell(int gx, int gy, int gz) const
    {
        const int g[3] = {gx, gy, gz};
        if (g[axis] != index) return -1;
        const int u0 = gx - G[0], u1 = gy - G[1], u2 = gz - G[2];
        if ((unsigned)u0 >= (unsigned)n[0] || (unsigned)u1 >= (unsigned)n[1] || (unsigned)u2 >= (unsigned)n[2]) return -1;
        return axis == 0 ? u1 + (long long)n[1] * u2 : axis == 1 ? u0 + (long long)n[0] * u2 : u0 + (long long)n[0] * u1;
    }
};

struct SysParams {
    GridParams g;
    AxisPlan ax[3];
    int T;                 // steps in this launch
    long long t0;          // ctx time at launch start (indexes wave[])
    int flag_base;         // epoch: flags of this launch count up from flag_base
    int ntiles;
    int* flagE;            // [ntiles]  = flag_base + (number of E phases published)
    int* flagH;            // [ntiles]
    unsigned int* counter; // tile claim counter of this launch (zero at launch)
    unsigned int* counter_zero;  // systolic_tma.cu: the claim counter of a launch 32 launches ahead, zeroed by this one (NULL: none)
    // Launch-to-launch overlap (row f2, "global synchronization operations are still required"): the launch may
    // start while the previous launch of the same tile grid is still draining (programmatic dependent launch); a tile then
    // waits until the tiles of the previous launch that finalised the cells of its box have raised their last flag.
    int pred_final;        // 0: the previous launch has completed (stream order); else the value those flags reach
    int* abort_flag;       // != 0: a watchdog fired; every CTA leaves
    long long spin_budget; // clock64 ticks a single wait may take
    const int* order;      // systolic_tma.cu: claim index -> tile, sorted by wavefront bx+by+bz (NULL: identity)
    int tma_group[3];      // systolic_tma.cu, per group (E, H, coefficients): 0 per-array 3-D maps, 1 one 4-D map per piece, 2 two triples
    // systolic_tma.cu on a padded copy of the grid: row pitch of the arrays in elements (>= g.n[0], a
    // multiple of 4), and the images of the source box (a box on a periodic axis also drives its ghost copies)
    int ldx;
    int nsrc;              // 0: no source; else number of images of g.src_box
    int src_org[MAX_SRC_IMAGES][3];
    MonitorParams mon;     // running-DFT monitor (mon.on == 0: none)
    long long* prof;       // FDTD_PROFILE build: 32 tick accumulators (NULL otherwise)
    // FDTD_DEBUG builds only (always 0 / NULL in the product libraries, and never read there):
    int dbg;               // FDTD_DEBUG_SKIP timing probes (results invalid): 1 no upwind waits, 2 no shell loads, 4 no publishes,
                           // 16 no coefficient scatter, 32 no proxy fence, 64 no skipping of empty tile steps
    unsigned int delay_seed; // != 0 inserts pseudo-random sleeps to perturb the inter-CTA order (FDTD_DEBUG_DELAY)
    int withhold_tile;     // >= 0: this tile never raises its flags, so the hand-off watchdog must fire (FDTD_DEBUG_WITHHOLD)
    int* levE;             // time-level shadow arrays, one int per cell (FDTD_DEBUG_LEVELS): number of E / H updates the
    int* levH;             //   value stored in global memory has received; every shell load asserts the level it expects
    unsigned long long* lev_err;   // [0] = number of violations, [1..4] = first violation (kind, cell index, found, expected)
};

// 36 CUtensorMap (128 bytes each) passed to systolic_tma.cu as a __grid_constant__ kernel parameter:
// [12 arrays: E0..2 H0..2 ca0..2 cb0..2][3 shell pieces: z plane, y row, x column]
struct alignas(64) TmaMaps {
    unsigned char bytes[36 * 128];
};

struct SysConfig {        // one compiled instantiation
    int Bx, By, Bz;       // cached box (powers of two); updated tile = (Bx-1, By-1, Bz-1)
    int coef;             // 1: carries the six coefficient arrays on chip
    int threads;
    size_t smem;
};

