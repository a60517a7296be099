// fdtd_api.cu -- the C ABI of include/fdtd.h: context, argument checking, schedule planning and launches.
// Every step of the hot path runs in the kernels of naive_kernels.cu / systolic_kernel.cu; this file only
// marshals.  There is no CPU fallback: without a device fdtd_create fails with FDTD_ECUDA.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <string>
#include <vector>

#include <cuda.h>

#include "fdtd_internal.h"

struct fdtd_ctx {
    GridParams g;
    float d[3];
    float dt;
    cudaStream_t stream;
    bool fields_set;
    float* d_amp;
    float* d_wave;
    std::vector<float> h_wave;
    long long t;
    MonitorParams mon;   // running-DFT monitor in CALLER coordinates (G = 0); mon.on == 0: none
    float* d_lut;        // device copy of the (ca, cb) table of fdtd_set_coeff_lut: [3][nmat][2]
    float* d_mon_w;      // device copy of the weight tables: wE[nt][F][2] then wH[nt][F][2]
    // schedule
    int which;
    bool which_explicit;   // fdtd_set_kernel was called: no automatic choice
    int reqN[3];      // requested tile (0 = default)
    int reqT;         // requested temporal depth (0 = default)
    int cfg_idx;      // resolved shared-memory systolic configuration, -1 = unresolved / not used
    bool use_reg;     // resolved: the register-resident kernel (tile 31x15x7) runs
    bool use_tma;     // resolved: its TMA-staged version runs
    bool tma_by8;     // resolved: the 31x7x7 build of it (two CTAs per SM)
    bool tma_h16;     // resolved: the binary16-field-storage build of it (g.fld16)
    bool tma_lut;     // resolved: the material-index build of it (g.cidx)
    // resolved: the TMA kernel runs on a padded working copy of the grid (periodic axis or nx % 4 != 0)
    bool use_pad;
    PadGeom pg;
    float* pad_fld;   // 6 padded arrays E0..2 H0..2 at stride pad_stride (library-owned)
    float* pad_coef;  // 6 padded arrays ca0..2 cb0..2, or NULL
    long long pad_stride;
    bool pad_coef_valid;
    TmaMaps tmaps;    // 36 CUtensorMap: [E0..2 H0..2 ca0..2 cb0..2][z plane, y row, x column]
    int tma_group[3]; // per group (E, H, coefficients): 0 per-array maps, 1 one 4-D map per piece, 2 two triples
    bool tmaps_valid;
    bool resolved;
    int N[3];         // resolved tile
    size_t smem;      // resolved dynamic shared memory per CTA
    int T;            // resolved temporal depth
    int ctas;
    // systolic state
    int* d_flags;     // flagE[cap] then flagH[cap]
    size_t flags_cap;
    // ring of kCounterRing tile-claim counters for the TMA kernel: its launch L uses slot L % ring and zeroes slot
    // (L + ring/2) % ring; one more slot behind the ring serves every launch of the other systolic kernels (memset before
    // each of them), which therefore never touch the ring
    unsigned int* d_counter;
    unsigned long long launch_seq;   // TMA launches so far
    // launch-to-launch overlap (row f2): shape and final flag value of the previous TMA launch, 0 = none / not reusable
    int prev_nb[3], prev_T, prev_final;
    bool no_overlap;           // FDTD_NO_OVERLAP in the environment at fdtd_create: every launch waits for the previous one
    bool timing;               // fdtd_set_timing: record events around every fdtd_step call (they serialise consecutive launches)
    int* d_abort;
    long long* d_prof;   // FDTD_PROFILE build only
    int* d_order;        // wavefront claim order of the TMA kernel for the launch being enqueued
    struct OrderEntry { int nb[3]; int* d; };
    std::vector<OrderEntry> orders;   // one per tile-grid shape seen (fdtd_step(n) ends with a shorter launch: n = qT + r)
    int flag_base;
    long long spin_budget;
    // tuning variables, read from the environment ONCE in fdtd_create (FDTD_T, FDTD_TILE, FDTD_SPIN_BUDGET_MS)
    int env_T;
    int env_tile[3];
    // FDTD_DEBUG builds only (dbg / prof variants); always zero in the product libraries
    unsigned int delay_seed;
    int dbg_skip, dbg_withhold;
    bool dbg_no_tma, dbg_no_group, dbg_lex_order, dbg_levels;
    int* d_lev;                      // time-level shadow arrays levE, levH of the working grid (FDTD_DEBUG_LEVELS)
    size_t lev_cells;
    unsigned long long* d_lev_err;   // [0] violations, [1..4] the first one
    // device
    int device, num_sms, clock_khz;
    cudaEvent_t ev0, ev1;
    bool ev_valid;
    long long counters[4];
    std::string err;
};

namespace {

constexpr int kCounterRing = 64;

// Every entry point that touches the device runs on the device the context was created on, whatever device is
// current in the calling thread, and leaves the caller's current device unchanged.
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(const fdtd_ctx* c) : prev(-1), switched(false)
    {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

int fail(fdtd_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    return code;
}

int cuda_fail(fdtd_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, FDTD_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool has_lut(const fdtd_ctx* c) { return c->g.cidx[0] != nullptr; }
bool has_coef(const fdtd_ctx* c) { return c->g.ca[0] != nullptr || has_lut(c); }

// both-or-neither rule for the systolic kernel (the naive kernel takes any combination)
bool coef_mixed(const fdtd_ctx* c) { return (c->g.ca[0] != nullptr) != (c->g.cb[0] != nullptr); }

int default_T(const fdtd_ctx* c)
{
    // Temporal depth: a launch costs each tile one whole-box load and one whole-tile store (a6) and widens every PEC
    // axis by T cells of ramp tiles (a11).  Since tiles skip the steps at which their region is outside the grid, a deep
    // launch is cheap even on small grids; measured on B200 (TCUPS at T = 16 / 64 / 128): 64^3 0.021 / - / 0.044,
    // 128^3 0.077 / - / 0.100, 256^3 (config 2) - / 0.102 / 0.106, 1024^3 - / 0.165 / 0.165.  (fdtd_step(n) with n < T
    // runs one launch of n steps.)
    return c->env_T > 0 ? c->env_T : 128;
}

// Temporal depth on a padded periodic axis: the ghost zones are 2T cells of redundant work per n cells of the axis, so T
// follows the shortest periodic extent (n/8: 25 % redundant cells), within [8, 128].
int default_T_padded(const fdtd_ctx* c)
{
    if (c->env_T > 0) return c->env_T;
    int nmin = 1 << 30;
    for (int a = 0; a < 3; ++a)
        if (c->g.per[a] && c->g.n[a] < nmin) nmin = c->g.n[a];
    if (nmin == (1 << 30)) return default_T(c);      // no periodic axis: only the row pitch is padded
    int T = nmin / 8;
    T = T < 8 ? 8 : T > 128 ? 128 : T;
    return T;
}

void free_pad(fdtd_ctx* c)
{
    if (c->pad_fld) cudaFree(c->pad_fld);
    if (c->pad_coef) cudaFree(c->pad_coef);
    c->pad_fld = c->pad_coef = nullptr;
    c->pad_coef_valid = false;
}

int resolve_systolic(fdtd_ctx* c)
{
    if (coef_mixed(c)) return fail(c, FDTD_EINVAL, "systolic kernel needs ca and cb both bound or both NULL");
    const int want_coef = has_coef(c) ? 1 : 0;
    const bool smem_only = c->which == FDTD_KERNEL_SYSTOLIC_SMEM;
    int N[3] = {c->reqN[0], c->reqN[1], c->reqN[2]};
    if (N[0] == 0) {
        if (!smem_only || want_coef) { N[0] = 31; N[1] = 15; N[2] = 7; }
        else                         { N[0] = 31; N[1] = 15; N[2] = 15; }
        if (c->env_tile[0] > 0) { N[0] = c->env_tile[0]; N[1] = c->env_tile[1]; N[2] = c->env_tile[2]; }
    }
    c->use_reg = !smem_only && N[0] == 31 && N[1] == 15 && N[2] == 7;
    c->tma_by8 = c->which == FDTD_KERNEL_SYSTOLIC && N[0] == 31 && N[1] == 7 && N[2] == 7;
    c->tma_h16 = c->g.fld16 != 0;
    c->tma_lut = has_lut(c);
    if (c->tma_lut && (c->tma_h16 || !(c->which == FDTD_KERNEL_SYSTOLIC && N[0] == 31 && N[1] == 15 && N[2] == 7)))
        return fail(c, FDTD_EINVAL, "material-index coefficients run FDTD_KERNEL_NAIVE or FDTD_KERNEL_SYSTOLIC with tile 31x15x7 and f32 fields");
    if (c->tma_h16 && !(c->which == FDTD_KERNEL_SYSTOLIC && N[0] == 31 && N[1] == 15 && N[2] == 7))
        return fail(c, FDTD_EINVAL, "binary16 field storage runs FDTD_KERNEL_NAIVE or FDTD_KERNEL_SYSTOLIC with tile 31x15x7");
    c->use_tma = (c->use_reg && c->which == FDTD_KERNEL_SYSTOLIC && !c->dbg_no_tma) || c->tma_by8;
    c->use_pad = c->use_tma && (c->g.per[0] || c->g.per[1] || c->g.per[2] || c->g.n[0] % (c->tma_lut ? 16 : c->tma_h16 ? 8 : 4) != 0);
    int found = -1;
    int per_sm = 0;
    if (c->use_tma) {
        cudaError_t e = c->tma_lut   ? systolic_tma_prepare_lut(want_coef, &per_sm)
                        : c->tma_h16 ? systolic_tma_prepare_h16(want_coef, &per_sm)
                        : c->tma_by8 ? systolic_tma_prepare_by8(want_coef, &per_sm)
                                     : systolic_tma_prepare(want_coef, &per_sm);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaFuncSetAttribute(max dynamic shared memory) / occupancy query");
        c->smem = c->tma_lut ? systolic_tma_smem_lut(want_coef) : c->tma_h16 ? systolic_tma_smem_h16(want_coef) : c->tma_by8 ? systolic_tma_smem_by8(want_coef) : systolic_tma_smem(want_coef);
    } else if (c->use_reg) {
        cudaError_t e = systolic_reg_prepare(want_coef, &per_sm);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaFuncSetAttribute(max dynamic shared memory) / occupancy query");
        c->smem = systolic_reg_smem(want_coef);
    } else {
        for (int i = 0; i < systolic_num_configs(); ++i) {
            const SysConfig* s = systolic_config(i);
            if (s->Bx - 1 == N[0] && s->By - 1 == N[1] && s->Bz - 1 == N[2] && s->coef == want_coef) { found = i; break; }
        }
        if (found < 0) {
            char buf[160];
            snprintf(buf, sizeof buf, "no systolic kernel built for tile %dx%dx%d %s coefficient arrays", N[0], N[1], N[2],
                     want_coef ? "with" : "without");
            return fail(c, FDTD_EINVAL, buf);
        }
        cudaError_t e = systolic_prepare(found, &per_sm);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaFuncSetAttribute(max dynamic shared memory) / occupancy query");
        c->smem = systolic_config(found)->smem;
    }
    // persistent grid: every CTA resident at once.  Residency comes from the occupancy query of the chosen function
    // (registers, threads and shared memory), because a ring of tiles deadlocks if a CTA of it is not resident.
    if (per_sm < 1) return fail(c, FDTD_ECUDA, "the systolic kernel does not fit on an SM of this device");
    if (per_sm > 4) per_sm = 4;
    c->ctas = c->num_sms * per_sm;
    c->T = c->reqT > 0 ? c->reqT : c->use_pad ? default_T_padded(c) : default_T(c);
    if (!c->use_tma) {
        // a ring of tiles along a periodic axis advances in lock step: all of it (and everything the claim order
        // interleaves with it) must be resident at once (SURVEY.md section 7 hard part 2)
        int span = 1, ring = 1;
        for (int a = 0; a < 3; ++a) {
            const AxisPlan ap = make_axis_plan(c->g.n[a], c->g.per[a], N[a], c->T);
            span *= ap.nb;
            if (c->g.per[a]) ring = span;
        }
        if (ring > c->ctas) {
            char buf[160];
            snprintf(buf, sizeof buf, "periodic ring of %d tiles exceeds the %d resident CTAs; use a larger tile or the naive kernel", ring, c->ctas);
            return fail(c, FDTD_EINVAL, buf);
        }
    }
    free_pad(c);
    if (c->use_pad) {
        // the padded working copy: G = T ghost cells on either side of every periodic axis, rows of a multiple of 4 cells
        long long cells = 1;
        for (int a = 0; a < 3; ++a) {
            c->pg.n[a] = c->g.n[a];
            c->pg.G[a] = c->g.per[a] ? c->T : 0;
            c->pg.m[a] = c->g.n[a] + 2 * c->pg.G[a];
        }
        c->pg.ldx = c->tma_lut ? (c->pg.m[0] + 15) / 16 * 16 : c->tma_h16 ? (c->pg.m[0] + 7) / 8 * 8 : (c->pg.m[0] + 3) / 4 * 4;   // rows are multiples of 16 bytes
        cells = c->pg.ldx * c->pg.m[1] * c->pg.m[2];
        if (c->pg.m[0] > (1 << 16) || c->pg.m[1] > (1 << 16) || c->pg.m[2] > (1 << 16) || cells >= (1ll << 40))
            return fail(c, FDTD_EINVAL, "padded working grid too large; use a smaller temporal depth");
        c->pad_stride = (cells + 63) / 64 * 64;
        cudaError_t e = cudaMalloc(&c->pad_fld, (size_t)c->pad_stride * 6 * sizeof(float));
        if (e == cudaSuccess && want_coef) e = cudaMalloc(&c->pad_coef, c->tma_lut ? (size_t)c->pad_stride * 3 : (size_t)c->pad_stride * 6 * sizeof(float));
        if (e != cudaSuccess) {
            free_pad(c);
            return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(padded working copy): ") + cudaGetErrorString(e));
        }
    }
    c->tmaps_valid = false;
    c->prev_final = 0;
    c->cfg_idx = found;
    for (int a = 0; a < 3; ++a) c->N[a] = N[a];
    c->resolved = true;
    return FDTD_OK;
}

// The grid the systolic kernel works on: the caller's arrays, or the padded working copy (then every axis is an open /
// wall axis of extent m, and the source box moves with the interior).  *ldx = row pitch in elements.
GridParams work_grid(const fdtd_ctx* c, long long* ldx)
{
    GridParams g = c->g;
    *ldx = c->g.n[0];
    if (!c->use_pad) return g;
    for (int a = 0; a < 3; ++a) {
        // the padded field arrays hold elements of the storage type (binary16 arrays sit behind float pointers)
        const size_t es = c->g.fld16 ? 2 : 4;
        g.E[a] = reinterpret_cast<float*>(reinterpret_cast<char*>(c->pad_fld) + es * (size_t)c->pad_stride * a);
        g.H[a] = reinterpret_cast<float*>(reinterpret_cast<char*>(c->pad_fld) + es * (size_t)c->pad_stride * (3 + a));
        const bool lutm = has_lut(c);
        g.ca[a] = (c->pad_coef && !lutm) ? c->pad_coef + c->pad_stride * a : nullptr;
        g.cb[a] = (c->pad_coef && !lutm) ? c->pad_coef + c->pad_stride * (3 + a) : nullptr;
        g.cidx[a] = (c->pad_coef && lutm) ? reinterpret_cast<const unsigned char*>(c->pad_coef) + c->pad_stride * a : nullptr;
        g.n[a] = c->pg.m[a];
        g.src_box[a] = c->g.src_box[a] + c->pg.G[a];
    }
    *ldx = c->pg.ldx;
    return g;
}

int ensure_flags(fdtd_ctx* c, size_t ntiles)
{
    if (ntiles <= c->flags_cap) return FDTD_OK;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    if (c->d_flags) cudaFree(c->d_flags);
    c->d_flags = nullptr;
    c->flags_cap = 0;
    e = cudaMalloc(&c->d_flags, 2 * ntiles * sizeof(int));
    if (e != cudaSuccess) return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(flags): ") + cudaGetErrorString(e));
    e = cudaMemsetAsync(c->d_flags, 0, 2 * ntiles * sizeof(int), c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemsetAsync(flags)");
    c->flags_cap = ntiles;
    c->flag_base = 0;
    c->prev_final = 0;
    return FDTD_OK;
}

// Tensor maps of the TMA-staged kernel: each field / coefficient array is a rank-3 fp32 tensor (nx, ny, nz) with
// byte strides (4 nx, 4 nx ny); one map per array and shell piece (the box extents are part of the map).
// Elements outside the tensor are delivered as zeros: the PEC ghost of reading #5 and the empty part of clipped tiles.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int ensure_tmaps(fdtd_ctx* c)
{
    if (c->tmaps_valid) return FDTD_OK;
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) return fail(c, FDTD_ECUDA, "cuTensorMapEncodeTiled is not available in this driver");
        encode = (EncodeTiledFn)fn;
    }
    int box_fld[3][3], box_coef[3][3];
    if (c->tma_h16) systolic_tma_boxes_h16(box_fld, box_coef);
    else if (c->tma_lut) systolic_tma_boxes_lut(box_fld, box_coef);
    else if (c->tma_by8) systolic_tma_boxes_by8(box_fld, box_coef);
    else systolic_tma_boxes(box_fld, box_coef);
    long long ldx = 0;
    const GridParams wg = work_grid(c, &ldx);
    const void* arr[12];
    for (int a = 0; a < 3; ++a) {
        arr[a] = wg.E[a];
        arr[3 + a] = wg.H[a];
        arr[6 + a] = wg.cidx[a] ? (const void*)wg.cidx[a] : (const void*)wg.ca[a];
        arr[9 + a] = wg.cb[a];
    }
    static_assert(sizeof(CUtensorMap) * 36 == sizeof(TmaMaps), "TmaMaps layout");
    CUtensorMap* host = reinterpret_cast<CUtensorMap*>(c->tmaps.bytes);
    memset(c->tmaps.bytes, 0, sizeof c->tmaps.bytes);
    const cuuint64_t ncells = (cuuint64_t)ldx * wg.n[1] * wg.n[2];
    // arrays first..first+count-1 at one positive stride (multiple of 16 bytes, no overlap)? -> the stride, else 0
    auto uniform_stride = [&](int first, int count) -> cuuint64_t {
        if (!arr[first] || c->dbg_no_group) return 0;
        const cuuint64_t nbytes = ncells * ((first < 6 && c->g.fld16) ? 2u : (first >= 6 && has_lut(c)) ? 1u : 4u);
        const char* b0 = (const char*)arr[first];
        const char* b1 = (const char*)arr[first + 1];
        if (b1 <= b0) return 0;
        const cuuint64_t d = (cuuint64_t)(b1 - b0);
        if (d < nbytes || (d & 15u) || d >= (1ull << 40)) return 0;
        for (int a = 2; a < count; ++a)
            if ((const char*)arr[first + a] != b0 + d * a) return 0;
        return d;
    };
    auto encode_maps = [&](CUtensorMap* dst, const void* base, int narr, cuuint64_t astride, bool fld) -> int {
        // extents are the logical grid (elements beyond it are delivered as zeros), strides follow the row pitch
        const bool h16 = fld && c->g.fld16;
        const bool u8 = !fld && has_lut(c);
        const cuuint64_t es = h16 ? 2u : u8 ? 1u : 4u;
        const int (*box)[3] = fld ? box_fld : box_coef;
        const cuuint64_t dims[4] = {(cuuint64_t)wg.n[0], (cuuint64_t)wg.n[1], (cuuint64_t)wg.n[2], (cuuint64_t)narr};
        const cuuint64_t strides[3] = {(cuuint64_t)ldx * es, (cuuint64_t)ldx * wg.n[1] * es, astride};
        const cuuint32_t estr[4] = {1, 1, 1, 1};
        for (int f = 0; f < 3; ++f) {
            const cuuint32_t b[4] = {(cuuint32_t)box[f][0], (cuuint32_t)box[f][1], (cuuint32_t)box[f][2], (cuuint32_t)narr};
            const CUresult r = encode(dst + f, h16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : u8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, narr > 1 ? 4 : 3, const_cast<void*>(base), dims, strides, b, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) {
                char buf[96];
                snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d), %d array(s), piece %d", (int)r, narr, f);
                return fail(c, FDTD_ECUDA, buf);
            }
        }
        return FDTD_OK;
    };
    // groups: E = arrays 0..2 (slot 0), H = 3..5 (slot 9), coefficients = 6..11 (slot 18)
    const int first[3] = {0, 3, 6}, count[3] = {3, 3, has_lut(c) ? 3 : 6};
    for (int g = 0; g < 3; ++g) {
        c->tma_group[g] = 0;
        if (!arr[first[g]]) continue;
        CUtensorMap* dst = host + first[g] * 3;
        int rc = FDTD_OK;
        cuuint64_t d = uniform_stride(first[g], count[g]);
        cuuint64_t da = 0, db = 0;
        if (d) {
            c->tma_group[g] = 1;
            rc = encode_maps(dst, arr[first[g]], count[g], d, g < 2);
        } else if (g == 2 && !has_lut(c) && (da = uniform_stride(6, 3)) && (db = uniform_stride(9, 3))) {
            c->tma_group[g] = 2;
            rc = encode_maps(dst, arr[6], 3, da, false);
            if (rc == FDTD_OK) rc = encode_maps(dst + 9, arr[9], 3, db, false);
        } else {
            for (int a = 0; a < count[g] && rc == FDTD_OK; ++a) rc = encode_maps(dst + a * 3, arr[first[g] + a], 1, 0, g < 2);
        }
        if (rc != FDTD_OK) return rc;
    }
    c->tmaps_valid = true;
    return FDTD_OK;
}

// Claim order of the TMA kernel: tiles sorted by wavefront index bx+by+bz (ties: z, y, x).  Every upwind neighbour
// of a tile has a smaller index, so it is claimed earlier (forward progress as with the lexicographic order), and the
// tiles in flight at one time are mutually independent once a wavefront holds more tiles than there are CTAs.
int ensure_order(fdtd_ctx* c, const int nb[3])
{
    for (const auto& o : c->orders)
        if (o.nb[0] == nb[0] && o.nb[1] == nb[1] && o.nb[2] == nb[2]) {
            c->d_order = o.d;
            return FDTD_OK;
        }
    const size_t nt = (size_t)nb[0] * nb[1] * nb[2];
    std::vector<int> h;
    h.reserve(nt);
    for (int d = 0; d <= nb[0] + nb[1] + nb[2] - 3; ++d)
        for (int z = 0; z < nb[2]; ++z) {
            if (d - z < 0) break;
            for (int y = 0; y < nb[1]; ++y) {
                const int x = d - z - y;
                if (x < 0) break;
                if (x < nb[0]) h.push_back(x + nb[0] * (y + nb[1] * z));
            }
        }
    if (c->orders.size() >= 8) {       // launches still in flight may read the oldest table: drain before freeing it
        cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
        cudaFree(c->orders.front().d);
        c->orders.erase(c->orders.begin());
    }
    fdtd_ctx::OrderEntry o;
    for (int a = 0; a < 3; ++a) o.nb[a] = nb[a];
    o.d = nullptr;
    cudaError_t e = cudaMalloc(&o.d, nt * sizeof(int));
    if (e != cudaSuccess) return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(order): ") + cudaGetErrorString(e));
    e = cudaMemcpyAsync(o.d, h.data(), nt * sizeof(int), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);     // h is a local; once per tile-grid shape
    if (e != cudaSuccess) { cudaFree(o.d); return cuda_fail(c, e, "cudaMemcpy(order)"); }
    c->orders.push_back(o);
    c->d_order = o.d;
    return FDTD_OK;
}

// Library default (no fdtd_set_kernel call): the systolic schedule on every grid (its TMA-staged kernel; grids with a
// periodic axis or nx % 4 != 0 run it on the padded working copy).  Only a half-bound coefficient set (ca without cb or
// the reverse), which the systolic kernel does not take, falls back to the naive kernel.
int effective_kernel(const fdtd_ctx* c)
{
    if (!c->which_explicit && c->which == FDTD_KERNEL_SYSTOLIC && coef_mixed(c)) return FDTD_KERNEL_NAIVE;
    return c->which;
}

int step_naive(fdtd_ctx* c, int n)
{
    for (int s = 0; s < n; ++s) {
        cudaError_t e = launch_e_half_naive(c->g, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "E half-step launch");
        c->counters[0]++;
        if (c->g.src_comp >= 0 && c->t >= 0 && c->t < c->g.src_nwave) {
            e = launch_source_w(c->g, c->h_wave[(size_t)c->t], c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "source launch");
            c->counters[0]++;
        }
        const bool mon = c->mon.on && c->t >= 0 && c->t < c->mon.nt;
        if (mon) {
            e = launch_monitor_naive(c->g, c->mon, 0, c->t, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "monitor launch");
            c->counters[0]++;
        }
        e = launch_h_half_naive(c->g, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "H half-step launch");
        c->counters[0]++;
        if (mon) {
            e = launch_monitor_naive(c->g, c->mon, 1, c->t, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "monitor launch");
            c->counters[0]++;
        }
        c->t++;
        c->counters[1]++;
    }
    return FDTD_OK;
}

int step_systolic(fdtd_ctx* c, int n)
{
    if (!c->resolved) {
        const int rc = resolve_systolic(c);
        if (rc != FDTD_OK) return rc;
    }
    if (c->use_tma) {
        const int rc = ensure_tmaps(c);
        if (rc != FDTD_OK) return rc;
    }
    if (c->mon.on && !c->use_tma)
        return fail(c, FDTD_EINVAL, "a monitor needs FDTD_KERNEL_SYSTOLIC with tile 31x15x7 or 31x7x7, or FDTD_KERNEL_NAIVE");
    const int N[3] = {c->N[0], c->N[1], c->N[2]};
    long long ldx = 0;
    const GridParams wg = work_grid(c, &ldx);
    // source images on the working grid: the box itself and, on the padded copy, its periodic copies that meet a ghost zone
    int nsrc = 0, src_org[MAX_SRC_IMAGES][3];
    if (c->use_tma && c->g.src_comp >= 0) {
        int lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
        for (int a = 0; a < 3; ++a) {
            if (!c->use_pad || c->pg.G[a] == 0) continue;
            // images j * n[a] of the box [b, b + w) that intersect [0, m[a])
            const int b0 = wg.src_box[a], w = wg.src_box[3 + a], na = c->g.n[a], ma = wg.n[a];
            while (b0 + (lo[a] - 1) * na + w > 0) --lo[a];
            while (b0 + (hi[a] + 1) * na < ma) ++hi[a];
        }
        for (int jz = lo[2]; jz <= hi[2]; ++jz)
            for (int jy = lo[1]; jy <= hi[1]; ++jy)
                for (int jx = lo[0]; jx <= hi[0]; ++jx) {
                    if (nsrc == MAX_SRC_IMAGES) return fail(c, FDTD_EINVAL, "temporal depth too large for this periodic grid: more than 125 source images");
                    src_org[nsrc][0] = wg.src_box[0] + jx * c->g.n[0];
                    src_org[nsrc][1] = wg.src_box[1] + jy * c->g.n[1];
                    src_org[nsrc][2] = wg.src_box[2] + jz * c->g.n[2];
                    ++nsrc;
                }
    }
    PadArrays pf, pc;
    if (c->use_pad && n > 0) {
        memset(&pf, 0, sizeof pf);
        memset(&pc, 0, sizeof pc);
        for (int a = 0; a < 3; ++a) {
            pf.usr[a] = c->g.E[a];
            pf.usr[3 + a] = c->g.H[a];
            pc.usr[a] = has_lut(c) ? reinterpret_cast<float*>(const_cast<unsigned char*>(c->g.cidx[a])) : const_cast<float*>(c->g.ca[a]);
            pc.usr[3 + a] = const_cast<float*>(c->g.cb[a]);
        }
        pf.ext = c->pad_fld; pf.stride = c->pad_stride; pf.narr = 6; pf.elem16 = c->g.fld16;
        pc.ext = c->pad_coef; pc.stride = c->pad_stride; pc.narr = has_lut(c) ? 3 : 6; pc.elem16 = has_lut(c) ? 2 : 0;
        if (c->pad_coef && !c->pad_coef_valid) {           // constants of the run: copied (with their images) once
            cudaError_t e = launch_pad_copy_in(c->pg, pc, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "padded copy of the coefficient arrays");
            c->pad_coef_valid = true;
            c->counters[0]++;
        }
        // the caller's arrays are the state between calls (they may have been rewritten): copy in, interior and ghosts
        cudaError_t e = launch_pad_copy_in(c->pg, pf, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "padded copy of the field arrays");
        c->counters[0]++;
    }
    bool first = true;
    int left = n;
    while (left > 0) {
        const int T = left < c->T ? left : c->T;
        if (c->use_pad && !first) {      // ghost zones <- periodic images of the interior the last launch left behind
            cudaError_t e = launch_pad_ghost_fill(c->pg, pf, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "ghost fill");
            c->counters[0]++;
        }
        first = false;
        SysParams P;
        memset(&P, 0, sizeof P);
        P.g = c->use_tma ? wg : c->g;
        P.ldx = (int)ldx;
        P.nsrc = nsrc;
        memcpy(P.src_org, src_org, sizeof src_org);
        long long ntiles = 1;
        for (int a = 0; a < 3; ++a) {
            P.ax[a] = make_axis_plan(P.g.n[a], c->use_tma ? 0 : c->g.per[a], N[a], T);
            ntiles *= P.ax[a].nb;
        }
        if (ntiles >= (1ll << 30)) return fail(c, FDTD_EINVAL, "too many tiles for one launch");
        const int rc = ensure_flags(c, (size_t)ntiles);
        if (rc != FDTD_OK) return rc;
        if (c->flag_base > (1 << 30)) {   // monotone epochs: rewind long before int overflow
            cudaError_t e = cudaMemsetAsync(c->d_flags, 0, 2 * c->flags_cap * sizeof(int), c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemsetAsync(flags)");
            c->flag_base = 0;
            c->prev_final = 0;
        }
        P.order = nullptr;
        if (c->use_tma && !c->dbg_lex_order) {
            const int nb[3] = {P.ax[0].nb, P.ax[1].nb, P.ax[2].nb};
            const int rc2 = ensure_order(c, nb);
            if (rc2 != FDTD_OK) return rc2;
            P.order = c->d_order;
        }
        P.T = T;
        P.t0 = c->t;
        P.flag_base = c->flag_base;
        P.ntiles = (int)ntiles;
        P.flagE = c->d_flags;
        P.flagH = c->d_flags + c->flags_cap;
        P.counter = c->use_tma ? c->d_counter + (c->launch_seq % kCounterRing) : c->d_counter + kCounterRing;
        P.counter_zero = c->use_tma ? c->d_counter + ((c->launch_seq + kCounterRing / 2) % kCounterRing) : nullptr;
        // overlap with the previous launch: same tile grid, same flag arrays still holding its final values, nothing but that
        // kernel before this one in the stream (a ghost refill or a copy in between serialises anyway: the wait is then free)
        P.pred_final = 0;
        if (c->use_tma && !c->use_pad && c->prev_final != 0 && c->prev_T == T && c->prev_nb[0] == P.ax[0].nb && c->prev_nb[1] == P.ax[1].nb &&
            c->prev_nb[2] == P.ax[2].nb && T >= 2 && !c->dbg_levels && !c->no_overlap)
            P.pred_final = c->prev_final;
        P.abort_flag = c->d_abort;
        P.spin_budget = c->spin_budget;
        P.delay_seed = c->delay_seed;
        P.prof = c->d_prof;
        P.mon = c->mon;
        if (c->mon.on && c->use_pad) {
            for (int a = 0; a < 3; ++a) P.mon.G[a] = c->pg.G[a];
            P.mon.index = c->mon.index + c->pg.G[c->mon.axis];
        }
        for (int g = 0; g < 3; ++g) P.tma_group[g] = c->tma_group[g];
        P.dbg = c->dbg_skip;
        P.withhold_tile = c->dbg_withhold;
        if (c->dbg_levels && c->use_tma) {
            // developer build: per-cell time levels of this launch start at 0 everywhere (all cells are at time t0)
            const size_t cells = (size_t)ldx * P.g.n[1] * P.g.n[2];
            if (cells > c->lev_cells) {
                cudaStreamSynchronize(c->stream);
                if (c->d_lev) cudaFree(c->d_lev);
                c->d_lev = nullptr;
                c->lev_cells = 0;
                if (cudaMalloc(&c->d_lev, 2 * cells * sizeof(int)) != cudaSuccess) return fail(c, FDTD_ENOMEM, "cudaMalloc(level shadow arrays)");
                c->lev_cells = cells;
            }
            if (!c->d_lev_err) {
                if (cudaMalloc(&c->d_lev_err, 8 * sizeof(unsigned long long)) != cudaSuccess) return fail(c, FDTD_ENOMEM, "cudaMalloc(level errors)");
                cudaMemsetAsync(c->d_lev_err, 0, 8 * sizeof(unsigned long long), c->stream);
            }
            cudaMemsetAsync(c->d_lev, 0, 2 * cells * sizeof(int), c->stream);
            P.levE = c->d_lev;
            P.levH = c->d_lev + cells;
            P.lev_err = c->d_lev_err;
        }
        cudaError_t e = cudaSuccess;
        if (!c->use_tma) {      // the other kernels do not maintain the ring: their own slot, cleared before every launch
            e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int), c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemsetAsync(counter)");
        }
        const int ctas = ntiles < c->ctas ? (int)ntiles : c->ctas;
        e = c->tma_lut   ? launch_systolic_tma_lut(1, P, c->tmaps, ctas, c->stream)
            : c->tma_h16 ? launch_systolic_tma_h16(has_coef(c) ? 1 : 0, P, c->tmaps, ctas, c->stream)
            : c->tma_by8 ? launch_systolic_tma_by8(has_coef(c) ? 1 : 0, P, c->tmaps, ctas, c->stream)
            : c->use_tma ? launch_systolic_tma(has_coef(c) ? 1 : 0, P, c->tmaps, ctas, c->stream)
            : c->use_reg ? launch_systolic_reg(has_coef(c) ? 1 : 0, P, ctas, c->stream)
                         : launch_systolic(c->cfg_idx, P, ctas, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "systolic launch");
        c->prev_final = 0;
        if (c->use_tma) {
            c->prev_final = c->flag_base + T;
            c->prev_T = T;
            for (int a = 0; a < 3; ++a) c->prev_nb[a] = P.ax[a].nb;
        }
        if (c->use_tma) c->launch_seq++;      // the ring position moves with TMA launches only (slot L is zeroed by TMA launch L - ring/2)
        c->flag_base += T + 2;
        c->t += T;
        left -= T;
        c->counters[0]++;
        c->counters[1] += T;
        c->counters[2]++;
        c->counters[3] += ntiles;
    }
    if (c->use_pad && n > 0) {
        cudaError_t e = launch_pad_copy_out(c->pg, pf, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "copy out of the padded working copy");
        c->counters[0]++;
    }
    return FDTD_OK;
}

int check_async(fdtd_ctx* c)
{
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    int flag = 0;
    e = cudaMemcpy(&flag, c->d_abort, sizeof(int), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(abort flag)");
    if (flag != 0) {
        cudaMemset(c->d_abort, 0, sizeof(int));
        c->prev_final = 0;      // the flags of the aborted launch are not final: the next launch must not wait on them
        return fail(c, FDTD_ETIMEOUT, "systolic hand-off watchdog fired: a tile waited longer than the spin budget; fields are invalid");
    }
    return FDTD_OK;
}

}  // namespace

extern "C" {

int fdtd_create(fdtd_ctx** out, int nx, int ny, int nz, float dx, float dy, float dz, float dt, const int boundary[3],
                void* cuda_stream)
{
    if (!out || !boundary) return FDTD_EINVAL;
    const int n[3] = {nx, ny, nz};
    const float d[3] = {dx, dy, dz};
    for (int a = 0; a < 3; ++a) {
        if (n[a] < 1 || n[a] > (1 << 15)) return FDTD_EINVAL;
        if (!(d[a] > 0.0f) || !isfinite(d[a])) return FDTD_EINVAL;
        if (boundary[a] != FDTD_PEC && boundary[a] != FDTD_PERIODIC) return FDTD_EINVAL;
    }
    if (!(dt > 0.0f) || !isfinite(dt)) return FDTD_EINVAL;
    if ((long long)nx * ny * nz >= (1ll << 40)) return FDTD_EINVAL;

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return FDTD_ECUDA;
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return FDTD_ECUDA;
    if (prop.major != 10) return FDTD_ECUDA;   // built for sm_100a only

    fdtd_ctx* c = new fdtd_ctx();
    memset(&c->g, 0, sizeof c->g);
    for (int a = 0; a < 3; ++a) {
        c->g.n[a] = n[a];
        c->g.per[a] = boundary[a] == FDTD_PERIODIC;
        c->g.rd[a] = (float)(1.0 / (double)d[a]);
        c->g.db[a] = dt;
        c->d[a] = d[a];
        c->reqN[a] = 0;
    }
    c->g.cb_scalar = dt;
    c->g.src_comp = -1;
    c->dt = dt;
    c->stream = (cudaStream_t)cuda_stream;
    c->fields_set = false;
    c->d_amp = c->d_wave = nullptr;
    c->t = 0;
    c->which = FDTD_KERNEL_SYSTOLIC;
    c->which_explicit = false;
    c->reqT = 0;
    c->cfg_idx = -1;
    c->use_reg = false;
    c->use_tma = false;
    c->tma_by8 = false;
    c->tma_h16 = false;
    c->tma_lut = false;
    c->d_lut = nullptr;
    c->use_pad = false;
    c->pad_fld = c->pad_coef = nullptr;
    c->pad_stride = 0;
    c->pad_coef_valid = false;
    memset(&c->pg, 0, sizeof c->pg);
    c->tmaps_valid = false;
    c->resolved = false;
    c->smem = 0;
    c->T = 0;
    c->ctas = 0;
    c->d_flags = nullptr;
    c->flags_cap = 0;
    c->d_counter = nullptr;
    c->launch_seq = 0;
    c->prev_final = 0;
    c->prev_T = 0;
    c->timing = false;
    c->no_overlap = false;
    c->d_abort = nullptr;
    c->d_prof = nullptr;
    c->d_mon_w = nullptr;
    memset(&c->mon, 0, sizeof c->mon);
    c->d_order = nullptr;
    c->flag_base = 0;
    c->delay_seed = 0;
    c->dbg_skip = 0;
    c->dbg_withhold = -1;
    c->dbg_no_tma = c->dbg_no_group = c->dbg_lex_order = c->dbg_levels = false;
    c->d_lev = nullptr;
    c->lev_cells = 0;
    c->d_lev_err = nullptr;
    c->env_T = 0;
    c->env_tile[0] = c->env_tile[1] = c->env_tile[2] = 0;
    if (const char* env = getenv("FDTD_T")) c->env_T = atoi(env);
    c->no_overlap = getenv("FDTD_NO_OVERLAP") != nullptr;
    if (const char* env = getenv("FDTD_TILE")) {
        int x, y, z;
        if (sscanf(env, "%dx%dx%d", &x, &y, &z) == 3 && x > 0 && y > 0 && z > 0) { c->env_tile[0] = x; c->env_tile[1] = y; c->env_tile[2] = z; }
    }
#ifdef FDTD_DEBUG
    if (const char* env = getenv("FDTD_DEBUG_DELAY")) c->delay_seed = (unsigned int)strtoul(env, nullptr, 10);
    if (const char* env = getenv("FDTD_DEBUG_SKIP")) c->dbg_skip = atoi(env);
    if (const char* env = getenv("FDTD_DEBUG_WITHHOLD")) c->dbg_withhold = atoi(env);
    c->dbg_no_tma = getenv("FDTD_DEBUG_NO_TMA") != nullptr;
    c->dbg_no_group = getenv("FDTD_DEBUG_NO_GROUP") != nullptr;
    c->dbg_lex_order = getenv("FDTD_DEBUG_LEX_ORDER") != nullptr;
    c->dbg_levels = getenv("FDTD_DEBUG_LEVELS") != nullptr;
#endif
    c->device = dev;
    c->num_sms = prop.multiProcessorCount;
    c->clock_khz = prop.clockRate;
    double budget_ms = 10000.0;
    if (const char* env = getenv("FDTD_SPIN_BUDGET_MS")) budget_ms = atof(env);
    c->spin_budget = (long long)(budget_ms * (double)(prop.clockRate > 0 ? prop.clockRate : 1965000));
    c->ev_valid = false;
    memset(c->counters, 0, sizeof c->counters);
    e = cudaMalloc(&c->d_counter, (kCounterRing + 1) * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(c->d_counter, 0, (kCounterRing + 1) * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_abort, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(c->d_abort, 0, sizeof(int));
#ifdef FDTD_PROFILE
    if (e == cudaSuccess) e = cudaMalloc(&c->d_prof, (32 + FDTD_TRACE_CAP) * sizeof(long long));
    if (e == cudaSuccess) e = cudaMemset(c->d_prof, 0, (32 + FDTD_TRACE_CAP) * sizeof(long long));
#endif
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    if (e != cudaSuccess) {
        fdtd_destroy(c);
        return FDTD_ECUDA;
    }
    *out = c;
    return FDTD_OK;
}

int fdtd_set_fields(fdtd_ctx* c, float* const E[3], float* const H[3])
{
    if (!c) return FDTD_EINVAL;
    if (!E || !H) return fail(c, FDTD_EINVAL, "fdtd_set_fields: NULL array");
    for (int a = 0; a < 3; ++a) {
        if (!E[a] || !H[a]) return fail(c, FDTD_EINVAL, "fdtd_set_fields: NULL field pointer");
        if (!aligned16(E[a]) || !aligned16(H[a])) return fail(c, FDTD_EINVAL, "fdtd_set_fields: pointers must be 16-byte aligned");
    }
    for (int a = 0; a < 3; ++a) {
        c->g.E[a] = E[a];
        c->g.H[a] = H[a];
    }
    if (c->g.fld16) c->resolved = false;     // the storage type selects the kernel build
    c->g.fld16 = 0;
    c->fields_set = true;
    c->tmaps_valid = false;
    return FDTD_OK;
}

int fdtd_set_fields_f16(fdtd_ctx* c, void* const E[3], void* const H[3])
{
    if (!c) return FDTD_EINVAL;
    if (!E || !H) return fail(c, FDTD_EINVAL, "fdtd_set_fields_f16: NULL array");
    for (int a = 0; a < 3; ++a) {
        if (!E[a] || !H[a]) return fail(c, FDTD_EINVAL, "fdtd_set_fields_f16: NULL field pointer");
        if (!aligned16(E[a]) || !aligned16(H[a])) return fail(c, FDTD_EINVAL, "fdtd_set_fields_f16: pointers must be 16-byte aligned");
    }
    for (int a = 0; a < 3; ++a) {
        c->g.E[a] = static_cast<float*>(E[a]);     // binary16 arrays behind float pointers; g.fld16 tells the kernels
        c->g.H[a] = static_cast<float*>(H[a]);
    }
    if (!c->g.fld16) c->resolved = false;
    c->g.fld16 = 1;
    c->fields_set = true;
    c->tmaps_valid = false;
    return FDTD_OK;
}

int fdtd_load_fields(fdtd_ctx* c, const float* const E[3], const float* const H[3])
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    if (!c->fields_set) return fail(c, FDTD_ESTATE, "fdtd_load_fields before fdtd_set_fields");
    const size_t bytes = (size_t)c->g.n[0] * c->g.n[1] * c->g.n[2] * (c->g.fld16 ? 2 : sizeof(float));
    for (int a = 0; a < 3; ++a) {
        if (E && E[a] && E[a] != c->g.E[a]) {
            cudaError_t e = cudaMemcpyAsync(c->g.E[a], E[a], bytes, cudaMemcpyDefault, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(E in)");
        }
        if (H && H[a] && H[a] != c->g.H[a]) {
            cudaError_t e = cudaMemcpyAsync(c->g.H[a], H[a], bytes, cudaMemcpyDefault, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(H in)");
        }
    }
    return FDTD_OK;
}

int fdtd_set_coeffs(fdtd_ctx* c, const float* const ca[3], const float* const cb[3], const float db[3])
{
    if (!c) return FDTD_EINVAL;
    for (int a = 0; a < 3; ++a) {
        if (ca && (!ca[a] || !aligned16(ca[a]))) return fail(c, FDTD_EINVAL, "fdtd_set_coeffs: ca needs three aligned device pointers");
        if (cb && (!cb[a] || !aligned16(cb[a]))) return fail(c, FDTD_EINVAL, "fdtd_set_coeffs: cb needs three aligned device pointers");
        if (db && !isfinite(db[a])) return fail(c, FDTD_EINVAL, "fdtd_set_coeffs: db not finite");
    }
    for (int a = 0; a < 3; ++a) {
        c->g.ca[a] = ca ? ca[a] : nullptr;
        c->g.cb[a] = cb ? cb[a] : nullptr;
        c->g.db[a] = db ? db[a] : c->dt;
        c->g.cidx[a] = nullptr;          // coefficient arrays replace a material-index binding
    }
    c->g.lut = nullptr;
    c->g.nmat = 0;
    c->cfg_idx = -1;   // the coefficient-carrying kernels are separate instantiations
    c->resolved = false;
    c->tmaps_valid = false;
    c->pad_coef_valid = false;
    return FDTD_OK;
}

int fdtd_set_coeff_lut(fdtd_ctx* c, const unsigned char* const idx[3], int nmat, const float* ca_lut, const float* cb_lut, const float db[3])
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    if (!idx || !ca_lut || !cb_lut || nmat < 1 || nmat > 256) return fail(c, FDTD_EINVAL, "fdtd_set_coeff_lut: NULL argument or nmat outside 1..256");
    for (int a = 0; a < 3; ++a) {
        if (!idx[a] || !aligned16(idx[a])) return fail(c, FDTD_EINVAL, "fdtd_set_coeff_lut: idx needs three 16-byte aligned device pointers");
        if (db && !isfinite(db[a])) return fail(c, FDTD_EINVAL, "fdtd_set_coeff_lut: db not finite");
    }
    cudaError_t e = cudaStreamSynchronize(c->stream);   // the old table may still be in use
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    if (c->d_lut) cudaFree(c->d_lut);
    c->d_lut = nullptr;
    // 256 pairs of zero padding behind the table: an index >= nmat (a caller error) reads (0, 0), never past the allocation
    std::vector<float> h((size_t)3 * nmat * 2 + 512, 0.0f);
    for (int a = 0; a < 3; ++a)
        for (int m = 0; m < nmat; ++m) {
            h[((size_t)a * nmat + m) * 2] = ca_lut[a * nmat + m];
            h[((size_t)a * nmat + m) * 2 + 1] = cb_lut[a * nmat + m];
        }
    e = cudaMalloc(&c->d_lut, h.size() * sizeof(float));
    if (e != cudaSuccess) return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(coefficient table): ") + cudaGetErrorString(e));
    e = cudaMemcpy(c->d_lut, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(coefficient table)");
    for (int a = 0; a < 3; ++a) {
        c->g.cidx[a] = idx[a];
        c->g.ca[a] = c->g.cb[a] = nullptr;
        c->g.db[a] = db ? db[a] : c->dt;
    }
    c->g.lut = c->d_lut;
    c->g.nmat = nmat;
    c->cfg_idx = -1;
    c->resolved = false;
    c->tmaps_valid = false;
    c->pad_coef_valid = false;
    return FDTD_OK;
}

int fdtd_set_source(fdtd_ctx* c, int comp, int i0, int j0, int k0, int ni, int nj, int nk, const float* amp,
                    const float* wave, int nwave)
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    cudaError_t e = cudaStreamSynchronize(c->stream);   // the old tables may still be in use
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    if (c->d_amp) cudaFree(c->d_amp);
    if (c->d_wave) cudaFree(c->d_wave);
    c->d_amp = c->d_wave = nullptr;
    c->g.src_comp = -1;
    c->g.src_amp = c->g.src_wave = nullptr;
    c->g.src_nwave = 0;
    c->h_wave.clear();
    if (!amp) return FDTD_OK;
    const int o[3] = {i0, j0, k0}, m[3] = {ni, nj, nk};
    if (comp < 0 || comp > 2 || !wave || nwave < 1) return fail(c, FDTD_EINVAL, "fdtd_set_source: bad component, wave or nwave");
    for (int a = 0; a < 3; ++a)
        if (o[a] < 0 || m[a] < 1 || o[a] + m[a] > c->g.n[a]) return fail(c, FDTD_EINVAL, "fdtd_set_source: box outside the grid");
    const size_t na = (size_t)ni * nj * nk;
    e = cudaMalloc(&c->d_amp, na * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_wave, (size_t)nwave * sizeof(float));
    if (e != cudaSuccess) return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(source): ") + cudaGetErrorString(e));
    e = cudaMemcpy(c->d_amp, amp, na * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_wave, wave, (size_t)nwave * sizeof(float), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(source)");
    c->h_wave.assign(wave, wave + nwave);
    c->g.src_comp = comp;
    for (int a = 0; a < 3; ++a) {
        c->g.src_box[a] = o[a];
        c->g.src_box[3 + a] = m[a];
    }
    c->g.src_amp = c->d_amp;
    c->g.src_wave = c->d_wave;
    c->g.src_nwave = nwave;
    return FDTD_OK;
}

int fdtd_set_monitor(fdtd_ctx* c, int axis, int index, int nfreq, int nt, const float* wE, const float* wH, float* acc)
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    cudaError_t e = cudaStreamSynchronize(c->stream);   // the old tables may still be in use
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    if (c->d_mon_w) cudaFree(c->d_mon_w);
    c->d_mon_w = nullptr;
    memset(&c->mon, 0, sizeof c->mon);
    if (!acc) return FDTD_OK;
    if (axis < 0 || axis > 2 || index < 0 || index >= c->g.n[axis] || nfreq < 1 || nfreq > 64 || nt < 1 || !wE || !wH)
        return fail(c, FDTD_EINVAL, "fdtd_set_monitor: bad axis, index, nfreq (1..64), nt or weight table");
    if (!aligned16(acc)) return fail(c, FDTD_EINVAL, "fdtd_set_monitor: misaligned accumulator");
    const size_t nw = (size_t)nt * nfreq * 2;
    e = cudaMalloc(&c->d_mon_w, 2 * nw * sizeof(float));
    if (e != cudaSuccess) return fail(c, FDTD_ENOMEM, std::string("cudaMalloc(monitor weights): ") + cudaGetErrorString(e));
    e = cudaMemcpy(c->d_mon_w, wE, nw * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_mon_w + nw, wH, nw * sizeof(float), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(monitor weights)");
    c->mon.on = 1;
    c->mon.axis = axis;
    c->mon.index = index;
    c->mon.F = nfreq;
    c->mon.nt = nt;
    for (int a = 0; a < 3; ++a) c->mon.n[a] = c->g.n[a];
    c->mon.wE = c->d_mon_w;
    c->mon.wH = c->d_mon_w + nw;
    c->mon.acc = acc;
    c->mon.pcells = (long long)c->g.n[0] * c->g.n[1] * c->g.n[2] / c->g.n[axis];
    return FDTD_OK;
}

int fdtd_step(fdtd_ctx* c, int n)
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    if (n < 0) return fail(c, FDTD_EINVAL, "fdtd_step: n < 0");
    if (!c->fields_set) return fail(c, FDTD_ESTATE, "fdtd_step before fdtd_set_fields");
    cudaError_t e = cudaSuccess;
    if (c->timing) {
        e = cudaEventRecord(c->ev0, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventRecord");
    }
    const int rc = (effective_kernel(c) == FDTD_KERNEL_NAIVE) ? step_naive(c, n) : step_systolic(c, n);
    if (c->timing) {
        e = cudaEventRecord(c->ev1, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventRecord");
        c->ev_valid = true;
    }
    return rc;
}

int fdtd_sync(fdtd_ctx* c)
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    return check_async(c);
}

int fdtd_get_fields(fdtd_ctx* c, float* const E[3], float* const H[3])
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    const int rc = check_async(c);
    if (rc != FDTD_OK) return rc;
    if (!E && !H) return FDTD_OK;
    if (!c->fields_set) return fail(c, FDTD_ESTATE, "fdtd_get_fields before fdtd_set_fields");
    const size_t bytes = (size_t)c->g.n[0] * c->g.n[1] * c->g.n[2] * (c->g.fld16 ? 2 : sizeof(float));
    for (int a = 0; a < 3; ++a) {
        if (E && E[a] && E[a] != c->g.E[a]) {
            cudaError_t e = cudaMemcpyAsync(E[a], c->g.E[a], bytes, cudaMemcpyDefault, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(E out)");
        }
        if (H && H[a] && H[a] != c->g.H[a]) {
            cudaError_t e = cudaMemcpyAsync(H[a], c->g.H[a], bytes, cudaMemcpyDefault, c->stream);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpyAsync(H out)");
        }
    }
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    return FDTD_OK;
}

int fdtd_set_time(fdtd_ctx* c, long long t)
{
    if (!c) return FDTD_EINVAL;
    c->t = t;
    return FDTD_OK;
}

long long fdtd_get_time(const fdtd_ctx* c) { return c ? c->t : -1; }

int fdtd_set_kernel(fdtd_ctx* c, int which, int Nx, int Ny, int Nz, int T)
{
    if (!c) return FDTD_EINVAL;
    DeviceGuard guard(c);
    if (which != FDTD_KERNEL_NAIVE && which != FDTD_KERNEL_SYSTOLIC && which != FDTD_KERNEL_SYSTOLIC_SMEM && which != FDTD_KERNEL_SYSTOLIC_REG) return fail(c, FDTD_EINVAL, "fdtd_set_kernel: unknown kernel");
    if (Nx < 0 || Ny < 0 || Nz < 0 || T < 0) return fail(c, FDTD_EINVAL, "fdtd_set_kernel: negative argument");
    if ((Nx == 0) != (Ny == 0) || (Nx == 0) != (Nz == 0)) return fail(c, FDTD_EINVAL, "fdtd_set_kernel: give all of Nx,Ny,Nz or none");
    const int oldN[3] = {c->reqN[0], c->reqN[1], c->reqN[2]};
    const int oldT = c->reqT, oldw = c->which;
    const bool old_explicit = c->which_explicit;
    c->which = which;
    c->which_explicit = true;
    c->reqN[0] = Nx; c->reqN[1] = Ny; c->reqN[2] = Nz;
    c->reqT = T;
    c->cfg_idx = -1;
    c->resolved = false;
    if (which != FDTD_KERNEL_NAIVE) {
        const int rc = resolve_systolic(c);
        if (rc != FDTD_OK) {
            c->which = oldw; c->reqT = oldT;
            c->which_explicit = old_explicit;
            c->reqN[0] = oldN[0]; c->reqN[1] = oldN[1]; c->reqN[2] = oldN[2];
            c->cfg_idx = -1;
            c->resolved = false;
            return rc;
        }
    }
    return FDTD_OK;
}

int fdtd_get_kernel(const fdtd_ctx* cc, int out[8])
{
    fdtd_ctx* c = const_cast<fdtd_ctx*>(cc);
    if (!c || !out) return FDTD_EINVAL;
    DeviceGuard guard(c);
    memset(out, 0, 8 * sizeof(int));
    out[0] = effective_kernel(c);
    if (out[0] != FDTD_KERNEL_NAIVE) {
        if (!c->resolved) {
            const int rc = resolve_systolic(c);
            if (rc != FDTD_OK) return rc;
        }
        out[1] = c->N[0]; out[2] = c->N[1]; out[3] = c->N[2];
        out[4] = c->T;
        long long nt = 1;
        const int N[3] = {out[1], out[2], out[3]};
        for (int a = 0; a < 3; ++a)
            nt *= c->use_tma ? make_axis_plan(c->use_pad ? c->pg.m[a] : c->g.n[a], 0, N[a], c->T).nb
                             : make_axis_plan(c->g.n[a], c->g.per[a], N[a], c->T).nb;
        out[5] = (int)nt;
        out[6] = nt < c->ctas ? (int)nt : c->ctas;
        out[7] = (int)c->smem;
    }
    return FDTD_OK;
}

int fdtd_get_counters(const fdtd_ctx* c, long long out[4])
{
    if (!c || !out) return FDTD_EINVAL;
    for (int q = 0; q < 4; ++q) out[q] = c->counters[q];
    return FDTD_OK;
}

int fdtd_set_timing(fdtd_ctx* c, int on)
{
    if (!c) return FDTD_EINVAL;
    c->timing = on != 0;
    if (!c->timing) c->ev_valid = false;
    return FDTD_OK;
}

int fdtd_last_step_ms(fdtd_ctx* c, float* ms)
{
    if (!c || !ms) return FDTD_EINVAL;
    DeviceGuard guard(c);
    if (!c->ev_valid) return fail(c, FDTD_ESTATE, "fdtd_last_step_ms: no timed fdtd_step call yet (fdtd_set_timing(ctx, 1) first)");
    cudaError_t e = cudaEventSynchronize(c->ev1);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventSynchronize");
    e = cudaEventElapsedTime(ms, c->ev0, c->ev1);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventElapsedTime");
    return FDTD_OK;
}

int fdtd_plan_tiles(const int n[3], const int boundary[3], const int N[3], int T, int ntiles[3])
{
    if (!n || !boundary || !N || !ntiles || T < 1) return FDTD_EINVAL;
    for (int a = 0; a < 3; ++a) {
        if (n[a] < 1 || N[a] < 1) return FDTD_EINVAL;
        if (boundary[a] != FDTD_PEC && boundary[a] != FDTD_PERIODIC) return FDTD_EINVAL;
    }
    for (int a = 0; a < 3; ++a) ntiles[a] = make_axis_plan(n[a], boundary[a] == FDTD_PERIODIC, N[a], T).nb;
    return FDTD_OK;
}

int fdtd_plan_owner(int n, int boundary, int N, int T, int g, int s, int* tile, int* offset)
{
    if (n < 1 || N < 1 || T < 1 || g < 0 || g >= n || s < 0 || s >= T || !tile || !offset) return FDTD_EINVAL;
    if (boundary != FDTD_PEC && boundary != FDTD_PERIODIC) return FDTD_EINVAL;
    const AxisPlan ap = make_axis_plan(n, boundary == FDTD_PERIODIC, N, T);
    int u = g + s;                      // position in the frame that moves with the tiles
    if (ap.per) u %= n;
    for (int b = 0; b < ap.nb; ++b) {
        const int a0 = ap.start(b), w = ap.width(b);
        if (u >= a0 && u < a0 + w) {
            *tile = b;
            *offset = u - a0;
            return FDTD_OK;
        }
    }
    return FDTD_EINVAL;
}

int fdtd_debug_level_errors(fdtd_ctx* c, long long out[5])
{
    if (!c || !out) return FDTD_EINVAL;
    for (int q = 0; q < 5; ++q) out[q] = 0;
    if (!c->dbg_levels) return fail(c, FDTD_ESTATE, "time-level shadow arrays are off (developer build with FDTD_DEBUG_LEVELS=1 only)");
    DeviceGuard guard(c);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
    if (!c->d_lev_err) return FDTD_OK;
    unsigned long long h[5];
    e = cudaMemcpy(h, c->d_lev_err, sizeof h, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(level errors)");
    for (int q = 0; q < 5; ++q) out[q] = (long long)h[q];
    return FDTD_OK;
}

const char* fdtd_last_error(const fdtd_ctx* c) { return c ? c->err.c_str() : "null context"; }

const char* fdtd_build_info(void)
{
#ifdef FDTD_NOFMA
    return "libfdtd_b200 sm_100a fmad=false (bit-exact build)";
#else
    return "libfdtd_b200 sm_100a fmad=true";
#endif
}

void fdtd_destroy(fdtd_ctx* c)
{
    if (!c) return;
    DeviceGuard guard(c);
    cudaStreamSynchronize(c->stream);
    if (c->d_amp) cudaFree(c->d_amp);
    if (c->d_wave) cudaFree(c->d_wave);
    if (c->d_mon_w) cudaFree(c->d_mon_w);
    if (c->d_lut) cudaFree(c->d_lut);
    if (c->d_flags) cudaFree(c->d_flags);
    if (c->d_counter) cudaFree(c->d_counter);
    if (c->d_abort) cudaFree(c->d_abort);
    free_pad(c);
    if (c->d_lev) cudaFree(c->d_lev);
    if (c->d_lev_err) cudaFree(c->d_lev_err);
    for (auto& o : c->orders) cudaFree(o.d);
    if (c->d_prof) {
        long long h[32];
        if (cudaMemcpy(h, c->d_prof, sizeof h, cudaMemcpyDeviceToHost) == cudaSuccess) {
            fprintf(stderr, "fdtd profile (clock64 ticks summed over CTAs):");
            for (int i = 0; i < 32; ++i) fprintf(stderr, "%s%lld", i % 8 == 0 ? "\n  " : " ", h[i]);
            fprintf(stderr, "\n");
        }
#ifdef FDTD_PROFILE
        // event trace of one CTA (systolic_tma.cu TRACE): clock << 20 | role << 16 | event << 12 | step
        if (const char* path = getenv("FDTD_TRACE_FILE")) {
            std::vector<long long> tr(FDTD_TRACE_CAP);
            if (cudaMemcpy(tr.data(), c->d_prof + 32, tr.size() * sizeof(long long), cudaMemcpyDeviceToHost) == cudaSuccess) {
                if (FILE* f = fopen(path, "w")) {
                    for (long long v : tr) {
                        if (v == 0) break;
                        fprintf(f, "%lld %d %d %d\n", v >> 20, (int)((v >> 16) & 15), (int)((v >> 12) & 15), (int)(v & 4095));
                    }
                    fclose(f);
                }
            }
        }
#endif
        cudaFree(c->d_prof);
    }
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    delete c;
}

int fdtd_absorber_coeffs(int nx, int ny, int nz, float dt, const float* const eps[3], const int thickness[6],
                         const float sigma_max[6], int order, float* const ca[3], float* const cb[3], void* cuda_stream)
{
    if (nx < 1 || ny < 1 || nz < 1 || nx > (1 << 15) || ny > (1 << 15) || nz > (1 << 15)) return FDTD_EINVAL;
    if (!(dt > 0.0f) || !std::isfinite(dt) || !thickness || !sigma_max || !ca || !cb || order < 0 || order > 8) return FDTD_EINVAL;
    const int n[3] = {nx, ny, nz};
    for (int f = 0; f < 6; ++f)
        if (thickness[f] < 0 || thickness[f] > n[f / 2] || !(sigma_max[f] >= 0.0f) || !std::isfinite(sigma_max[f])) return FDTD_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (!ca[a] || !cb[a]) return FDTD_EINVAL;
    const cudaError_t e = launch_absorber(n, dt, eps, thickness, sigma_max, order, ca, cb, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? FDTD_OK : FDTD_ECUDA;
}

}  // extern "C"
