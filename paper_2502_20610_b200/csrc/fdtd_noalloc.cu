// fdtd_noalloc.cu -- fdtd_step_noalloc (include/fdtd.h): the systolic TMA kernel for callers that must not allocate.
//
// The context path (fdtd_create / fdtd_step) cudaMallocs what the systolic schedule needs besides the caller's fields:
// two hand-off flags per tile, a ring of tile-claim counters, the wavefront claim order and the watchdog word.  Some
// hosts cannot let a library do that: a framework that has handed all of HBM to its own pool (config 5 is 81 GiB of
// fields on a 180 GB part, the rest usually belongs to the host application's allocator), or a time-stepping loop that
// shares the device with other streams and cannot take the device-wide stall a cudaMalloc / cudaFree may cause.  For
// them the same kernel runs here on ONE file-scope __device__ array of fixed size.  Nothing in this file calls
// cudaMalloc, cudaFree, cudaMallocAsync or a library routine that allocates device memory; host memory comes from
// static arrays as well.
//
// The array belongs to the module image: every GPU that loads libfdtd_b200 holds kScratchBytes of it until the process
// exits, whether or not this entry point is ever called.  All calls on one device share it and it keeps what the last
// call left there, so each call clears the part that must start at zero (flags, counters, watchdog word) in stream order
// before its first launch.  Two runs in flight on one device would raise and poll the same flags; a lock held until the
// GPU work of a call has finished keeps callers of one process apart (the call synchronises its stream anyway, to read
// the watchdog word).
//
// In HOST code the name g_scratch is only a handle for the runtime, not a device address: a kernel handed &g_scratch[0]
// would fault (or quietly use host memory where the GPU can reach it).  The device address comes from
// cudaGetSymbolAddress, asked once per device with that device current; see device_state().
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include <cuda.h>

#include "fdtd_internal.h"

namespace {

constexpr int kMaxTiles = FDTD_NOALLOC_MAX_TILES;     // tiles of one launch
constexpr int kRing = 64;                             // tile-claim counters: launch L uses slot L % kRing and zeroes slot (L + kRing/2) % kRing
constexpr int kMaxDevices = 64;
// layout in ints: flagE[kMaxTiles] | flagH[kMaxTiles] | order[kMaxTiles] | counters[kRing] | watchdog word, padded
constexpr size_t kOffFlagE = 0, kOffFlagH = kMaxTiles, kOffOrder = 2 * (size_t)kMaxTiles, kOffCounter = 3 * (size_t)kMaxTiles, kOffAbort = kOffCounter + kRing;
constexpr size_t kScratchInts = kOffAbort + 64;
constexpr size_t kScratchBytes = kScratchInts * sizeof(int);     // 1.5 MiB + 512 B

static __device__ __align__(256) int g_scratch[kScratchInts];

struct DeviceState {
    bool ready;
    int* scratch;        // DEVICE address of g_scratch on this device
    int num_sms;
    int clock_khz;
    int per_sm[2];       // resident CTAs per SM of the kernel without / with coefficient arrays (0 = not prepared yet)
};

std::mutex g_lock;                       // one run at a time per process: every call shares g_scratch
DeviceState g_dev[kMaxDevices];
int g_host_order[kMaxTiles];             // host staging of the claim order (static: no heap either)

int fail(char* errbuf, int len, int code, const char* fmt, ...)
{
    if (errbuf && len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, (size_t)len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Set-up of the current device, done by the first call that runs on it: the device address of the scratch array, the
// SM count and clock (watchdog budget).  Must not run while a stream of this device is being captured.
int device_state(int dev, DeviceState** out, char* errbuf, int len)
{
    if (dev < 0 || dev >= kMaxDevices) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: device ordinal %d is beyond the %d this entry point tracks", dev, kMaxDevices);
    DeviceState& s = g_dev[dev];
    if (!s.ready) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: built for sm_100a, the current device has compute capability %d.x", major);
        int* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_scratch);      // device current: the address is this device's copy of the array
        if (e != cudaSuccess || !p) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
        s.scratch = p;
        e = cudaDeviceGetAttribute(&s.num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&s.clock_khz, cudaDevAttrClockRate, dev);
        if (e != cudaSuccess) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        s.per_sm[0] = s.per_sm[1] = 0;
        s.ready = true;
    }
    *out = &s;
    return FDTD_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Tensor maps of the f32 kernel on the caller's arrays (rank 3, or rank 4 when the arrays of a group sit at one stride);
// they live in the kernel's parameter space, not in device memory.
int encode_maps(TmaMaps* maps, int group[3], const int n[3], const void* const arr[12], bool coef, char* errbuf, int len)
{
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: cuTensorMapEncodeTiled is not available in this driver");
        encode = (EncodeTiledFn)fn;
    }
    int box_fld[3][3], box_coef[3][3];
    systolic_tma_boxes(box_fld, box_coef);
    static_assert(sizeof(CUtensorMap) * 36 == sizeof(TmaMaps), "TmaMaps layout");
    CUtensorMap* host = reinterpret_cast<CUtensorMap*>(maps->bytes);
    memset(maps->bytes, 0, sizeof maps->bytes);
    const cuuint64_t nbytes = (cuuint64_t)n[0] * n[1] * n[2] * 4u;
    auto stride_of = [&](int first, int count) -> cuuint64_t {      // one positive stride over the group, else 0
        const char* b0 = (const char*)arr[first];
        const char* b1 = (const char*)arr[first + 1];
        if (b1 <= b0) return 0;
        const cuuint64_t d = (cuuint64_t)(b1 - b0);
        if (d < nbytes || (d & 15u) || d >= (1ull << 40)) return 0;
        for (int a = 2; a < count; ++a)
            if ((const char*)arr[first + a] != b0 + d * a) return 0;
        return d;
    };
    auto encode3 = [&](CUtensorMap* dst, const void* base, int narr, cuuint64_t astride, const int (*box)[3]) -> int {
        const cuuint64_t dims[4] = {(cuuint64_t)n[0], (cuuint64_t)n[1], (cuuint64_t)n[2], (cuuint64_t)narr};
        const cuuint64_t strides[3] = {(cuuint64_t)n[0] * 4u, (cuuint64_t)n[0] * n[1] * 4u, astride};
        const cuuint32_t estr[4] = {1, 1, 1, 1};
        for (int f = 0; f < 3; ++f) {          // shell pieces: z plane, y row, x column
            const cuuint32_t b[4] = {(cuuint32_t)box[f][0], (cuuint32_t)box[f][1], (cuuint32_t)box[f][2], (cuuint32_t)narr};
            const CUresult r = encode(dst + f, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, narr > 1 ? 4 : 3, const_cast<void*>(base), dims, strides, b, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);     // outside the grid: zeros (the PEC ghost)
            if (r != CUDA_SUCCESS) return fail(errbuf, len, FDTD_ECUDA, "fdtd_step_noalloc: cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
        }
        return FDTD_OK;
    };
    const int first[3] = {0, 3, 6}, count[3] = {3, 3, 6};
    for (int g = 0; g < 3; ++g) {
        group[g] = 0;
        if (g == 2 && !coef) continue;
        const int (*box)[3] = g < 2 ? box_fld : box_coef;
        CUtensorMap* dst = host + first[g] * 3;
        int rc = FDTD_OK;
        cuuint64_t d = stride_of(first[g], count[g]), da = 0, db = 0;
        if (d) {
            group[g] = 1;
            rc = encode3(dst, arr[first[g]], count[g], d, box);
        } else if (g == 2 && (da = stride_of(6, 3)) && (db = stride_of(9, 3))) {
            group[g] = 2;
            rc = encode3(dst, arr[6], 3, da, box);
            if (rc == FDTD_OK) rc = encode3(dst + 9, arr[9], 3, db, box);
        } else {
            for (int a = 0; a < count[g] && rc == FDTD_OK; ++a) rc = encode3(dst + a * 3, arr[first[g] + a], 1, 0, box);
        }
        if (rc != FDTD_OK) return rc;
    }
    return FDTD_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" int fdtd_step_noalloc(int nx, int ny, int nz, float dx, float dy, float dz, float dt, float* const E[3], float* const H[3],
                                 const float* const ca[3], const float* const cb[3], const float db[3], int nsteps, int T,
                                 void* cuda_stream, char* errbuf, int errbuf_len)
{
    char* const eb = errbuf;
    const int el = errbuf_len;
    if (eb && el > 0) eb[0] = 0;
    // ---- arguments and limits: nothing is dereferenced and no CUDA call is made before these pass
    const int n[3] = {nx, ny, nz};
    const float d[3] = {dx, dy, dz};
    const int N[3] = {31, 15, 7};
    for (int a = 0; a < 3; ++a) {
        if (n[a] < 1 || n[a] > (1 << 15)) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: grid extent %d outside 1..32768", n[a]);
        if (!(d[a] > 0.0f) || !isfinite(d[a])) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: cell sizes must be positive and finite");
    }
    if (!(dt > 0.0f) || !isfinite(dt)) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: dt must be positive and finite");
    if (nsteps < 0 || T < 0) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: nsteps and T must not be negative");
    if (nx % 4 != 0)
        return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: nx = %d is not a multiple of 4; such grids run on a padded working copy, which needs an allocation (use fdtd_create / fdtd_step)", nx);
    if (!E || !H || (ca == nullptr) != (cb == nullptr)) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: E and H are required; ca and cb come together or not at all");
    for (int a = 0; a < 3; ++a) {
        if (!E[a] || !H[a] || !aligned16(E[a]) || !aligned16(H[a])) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: field pointers must be non-NULL and 16-byte aligned");
        if (ca && (!ca[a] || !cb[a] || !aligned16(ca[a]) || !aligned16(cb[a]))) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: coefficient pointers must be non-NULL and 16-byte aligned");
        if (db && !isfinite(db[a])) return fail(eb, el, FDTD_EINVAL, "fdtd_step_noalloc: db not finite");
    }
    const int depth = T > 0 ? T : 128;
    const int T0 = nsteps < depth ? nsteps : depth;       // the deepest launch of this call has the most tiles
    if (T0 > 0) {
        long long ntiles = 1;
        for (int a = 0; a < 3; ++a) ntiles *= make_axis_plan(n[a], 0, N[a], T0).nb;
        if (ntiles > kMaxTiles)
            return fail(eb, el, FDTD_EINVAL,
                        "fdtd_step_noalloc: %lld tiles per launch (grid %dx%dx%d, temporal depth %d, tile 31x15x7) exceed FDTD_NOALLOC_MAX_TILES = %d, the size of the "
                        "static scratch array; pass a smaller T or use fdtd_create / fdtd_step",
                        ntiles, nx, ny, nz, T0, kMaxTiles);
    }
    if (nsteps == 0) return FDTD_OK;

    std::lock_guard<std::mutex> guard(g_lock);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: no CUDA device (%s); there is no CPU fallback", cudaGetErrorString(e));
    DeviceState* ds = nullptr;
    int rc = device_state(dev, &ds, eb, el);
    if (rc != FDTD_OK) return rc;
    const int coef = ca ? 1 : 0;
    if (ds->per_sm[coef] == 0) {
        int per_sm = 0;
        e = systolic_tma_prepare(coef, &per_sm);          // shared-memory attribute of the kernel + occupancy query (no allocation)
        if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: kernel set-up: %s", cudaGetErrorString(e));
        if (per_sm < 1) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: the systolic kernel does not fit on an SM of this device");
        ds->per_sm[coef] = per_sm > 4 ? 4 : per_sm;
    }
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    int* const base = ds->scratch;

    GridParams g;
    memset(&g, 0, sizeof g);
    const void* arr[12] = {};
    for (int a = 0; a < 3; ++a) {
        g.E[a] = E[a];
        g.H[a] = H[a];
        g.ca[a] = ca ? ca[a] : nullptr;
        g.cb[a] = cb ? cb[a] : nullptr;
        g.n[a] = n[a];
        g.rd[a] = (float)(1.0 / (double)d[a]);
        g.db[a] = db ? db[a] : dt;
        arr[a] = E[a];
        arr[3 + a] = H[a];
        arr[6 + a] = g.ca[a];
        arr[9 + a] = g.cb[a];
    }
    g.cb_scalar = dt;
    g.src_comp = -1;
    static TmaMaps maps;          // 4.5 KiB, copied into the kernel's parameter space at every launch; guarded by g_lock
    int group[3];
    rc = encode_maps(&maps, group, n, arr, coef != 0, eb, el);
    if (rc != FDTD_OK) return rc;

    // what must start at zero: every flag, every claim counter, the watchdog word (stream order, before the first launch)
    e = cudaMemsetAsync(base + kOffFlagE, 0, 2 * (size_t)kMaxTiles * sizeof(int), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(base + kOffCounter, 0, (kRing + 64) * sizeof(int), st);
    if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: cudaMemsetAsync(scratch): %s", cudaGetErrorString(e));

    int flag_base = 0, order_nb[3] = {0, 0, 0};
    unsigned long long seq = 0;
    int left = nsteps;
    while (left > 0) {
        const int Tl = left < depth ? left : depth;
        SysParams P;
        memset(&P, 0, sizeof P);
        P.g = g;
        P.ldx = nx;
        long long ntiles = 1;
        for (int a = 0; a < 3; ++a) {
            P.ax[a] = make_axis_plan(n[a], 0, N[a], Tl);
            ntiles *= P.ax[a].nb;
        }
        if (flag_base > (1 << 30)) {          // flags count up across launches: rewind long before int overflow
            e = cudaMemsetAsync(base + kOffFlagE, 0, 2 * (size_t)kMaxTiles * sizeof(int), st);
            if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: cudaMemsetAsync(flags): %s", cudaGetErrorString(e));
            flag_base = 0;
        }
        if (order_nb[0] != P.ax[0].nb || order_nb[1] != P.ax[1].nb || order_nb[2] != P.ax[2].nb) {
            // claim order: tiles sorted by wavefront bx+by+bz (ties z, y, x), so every upwind tile is claimed first.  The copy
            // is ordered on the stream behind the launches that still read the previous table; a pageable source is staged
            // before cudaMemcpyAsync returns, so g_host_order may be rewritten afterwards.
            for (int a = 0; a < 3; ++a) order_nb[a] = P.ax[a].nb;
            const int* nb = order_nb;
            size_t q = 0;
            for (int w = 0; w <= nb[0] + nb[1] + nb[2] - 3; ++w)
                for (int z = 0; z < nb[2] && z <= w; ++z)
                    for (int y = 0; y < nb[1] && y <= w - z; ++y) {
                        const int x = w - z - y;
                        if (x < nb[0]) g_host_order[q++] = x + nb[0] * (y + nb[1] * z);
                    }
            e = cudaMemcpyAsync(base + kOffOrder, g_host_order, q * sizeof(int), cudaMemcpyHostToDevice, st);
            if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: cudaMemcpyAsync(claim order): %s", cudaGetErrorString(e));
        }
        P.order = base + kOffOrder;
        P.T = Tl;
        P.t0 = 0;
        P.flag_base = flag_base;
        P.ntiles = (int)ntiles;
        P.flagE = base + kOffFlagE;
        P.flagH = base + kOffFlagH;
        P.counter = reinterpret_cast<unsigned int*>(base + kOffCounter) + (seq % kRing);
        P.counter_zero = reinterpret_cast<unsigned int*>(base + kOffCounter) + ((seq + kRing / 2) % kRing);
        P.pred_final = 0;                     // launches of a call follow each other in stream order, no overlap
        P.abort_flag = base + kOffAbort;
        P.spin_budget = 10000ll * (ds->clock_khz > 0 ? ds->clock_khz : 1965000);      // 10 s of SM clock ticks
        for (int q = 0; q < 3; ++q) P.tma_group[q] = group[q];
        P.withhold_tile = -1;
        const int resident = ds->num_sms * ds->per_sm[coef];
        const int ctas = ntiles < resident ? (int)ntiles : resident;
        e = launch_systolic_tma(coef, P, maps, ctas, st);
        if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: kernel launch: %s", cudaGetErrorString(e));
        ++seq;
        flag_base += Tl + 2;
        left -= Tl;
    }
    // the watchdog word tells whether a hand-off ever timed out; reading it means waiting for the work
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: cudaStreamSynchronize: %s", cudaGetErrorString(e));
    int fired = 0;
    e = cudaMemcpy(&fired, base + kOffAbort, sizeof(int), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(eb, el, FDTD_ECUDA, "fdtd_step_noalloc: cudaMemcpy(watchdog word): %s", cudaGetErrorString(e));
    if (fired != 0) return fail(eb, el, FDTD_ETIMEOUT, "fdtd_step_noalloc: hand-off watchdog fired: a tile waited longer than 10 s; fields are invalid");
    return FDTD_OK;
}
