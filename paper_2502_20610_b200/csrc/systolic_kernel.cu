// systolic_kernel.cu -- the systolic FDTD kernel for sm_100a: persistent CTAs, one resident tile each,
// hand-off through global memory with per-tile acquire/release flags instead of grid-wide barriers.
//
// "each subdomain can be considered to be a single node which communicates ... only boundary values to
// neighboring nodes ... in a directional manner which minimizes the need for global synchronization"
// (section 3); "an upwind subdomain can leave behind a trail of boundary values for a downwind
// subdomain to pick up whenever it is ready to consume them".
//
// Protocol (a9; reading #11).  Tiles are claimed from an atomic counter in lexicographic order
// (x fastest), so every upwind tile (b - delta, delta in {0,1}^3 \ 0) of a claimed tile has been claimed by a
// resident CTA before it: the lowest unfinished tile can always advance and no spin can deadlock.  Per tile
// two monotone counters: flagE = base + (E phases published), flagH = base + (H phases published).
//   E phase of step k needs the H shell published by step k-1 of ALL SEVEN upwind tiles: wait flagH[u] >= base+k
//   H phase of step k needs their E shell of step k:                                     wait flagE[u] >= base+k+1
// Producer: shell stores (st.global.cg) -> __syncthreads -> thread 0: __threadfence + st.release.gpu.
// Consumer: threads 0..6 poll ld.acquire.gpu -> __syncthreads -> shell loads (ld.global.cg, never L1).
// The same waits order the in-place overwrites (a cell is rewritten by its next owner only after every
// reader of the previous value has passed the corresponding phase), so there is no double buffering.
//
// Watchdog: a wait that exceeds its clock64 budget sets *abort_flag; every CTA polls it and leaves, and the
// host reports FDTD_ETIMEOUT instead of hanging the device.
#include "fdtd_internal.h"
#include "systolic_tile.cuh"

namespace {

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

struct Ctl {
    int tile;
    int abort;
};

// threads 0..6 each watch one upwind neighbour; returns false (block-uniform) if the launch is aborting
template <class Tile>
__device__ __forceinline__ bool wait_upwind(const SysParams& P, const Tile& t, const int* flags, int target, Ctl* ctl)
{
    const int tid = threadIdx.x;
    if (tid < 7) {
        const int u = t.nbr[tid];
        if (u >= 0) {
            const long long t_start = clock64();
            unsigned spins = 0;
            while (ld_acquire(flags + u) < target) {
                if ((++spins & 63u) == 0u) {
                    if (ld_volatile(P.abort_flag) != 0) { ctl->abort = 1; break; }
                    if (clock64() - t_start > P.spin_budget) {
                        atomicExch(P.abort_flag, 1);
                        ctl->abort = 1;
                        break;
                    }
                }
                __nanosleep(20);
            }
        }
    }
    __syncthreads();
    return ctl->abort == 0;
}

// all shell stores of this CTA are done (they precede the barrier); make them visible, then raise the flag
__device__ __forceinline__ void publish_flag(int* flag, int value)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        st_release(flag, value);
    }
}

#ifdef FDTD_DEBUG
__device__ __forceinline__ void debug_delay(const SysParams& P, int tile, int k, int phase)
{
    if (P.delay_seed == 0u) return;
    if (threadIdx.x == 0) {
        unsigned h = P.delay_seed ^ (unsigned)(tile * 2654435761u) ^ (unsigned)(k * 40503u + phase * 97u);
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13; h *= 3266489917u; h ^= h >> 16;
        if ((h & 3u) == 0u) __nanosleep((h >> 8) & 0x3fffu);   // up to ~16 us, one phase in four
    }
    __syncthreads();
}
#endif

template <int BX, int BY, int BZ, bool COEF, int ZSPLIT>
__global__ void __launch_bounds__(BX * BY * ZSPLIT, 1) systolic_kernel(const __grid_constant__ SysParams P)
{
    using Tile = SysTile<BX, BY, BZ, COEF, ZSPLIT>;
    extern __shared__ __align__(16) float sm[];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x;
    if (tid == 0) ctl.abort = 0;

    for (;;) {
        __syncthreads();   // the previous tile's last publish has read shared memory; ctl.tile may be rewritten
        if (tid == 0) {
            ctl.tile = (int)atomicAdd(P.counter, 1u);
            if (ld_volatile(P.abort_flag) != 0) ctl.abort = 1;
        }
        __syncthreads();
        const int tile = ctl.tile;
        if (tile >= P.ntiles || ctl.abort) break;

        Tile t;
        t.init(P, tile);
        for (int k = 0; k < P.T; ++k) {
            t.begin_step(k, P.T);
            if (k == 0) {
                t.load_initial(P, sm, tid);
            } else {
                if (!wait_upwind(P, t, P.flagH, P.flag_base + k, &ctl)) return;
                t.load_h_shell(P, sm, tid);
            }
            __syncthreads();
            FDTD_DEBUG_ONLY(debug_delay(P, tile, k, 0);)
            t.e_phase(P, sm, tid);
            __syncthreads();
            t.publish_e(P, sm, tid);
            publish_flag(P.flagE + tile, P.flag_base + k + 1);
            FDTD_DEBUG_ONLY(debug_delay(P, tile, k, 1);)
            if (!wait_upwind(P, t, P.flagE, P.flag_base + k + 1, &ctl)) return;
            t.load_e_shell(P, sm, tid);
            __syncthreads();
            t.h_phase(P, sm, tid);
            __syncthreads();
            t.publish_h(P, sm, tid);
            publish_flag(P.flagH + tile, P.flag_base + k + 1);
        }
    }
}

struct Entry {
    SysConfig cfg;
    const void* fn;
};

template <int BX, int BY, int BZ, bool COEF, int ZSPLIT>
Entry make_entry()
{
    using Tile = SysTile<BX, BY, BZ, COEF, ZSPLIT>;
    Entry e;
    e.cfg.Bx = BX; e.cfg.By = BY; e.cfg.Bz = BZ;
    e.cfg.coef = COEF ? 1 : 0;
    e.cfg.threads = Tile::NT;
    e.cfg.smem = Tile::kSmemBytes;
    e.fn = (const void*)&systolic_kernel<BX, BY, BZ, COEF, ZSPLIT>;
    return e;
}

const Entry* table(int* count)
{
    static const Entry entries[] = {
        make_entry<32, 16, 16, false, 1>(),   // the paper's 31x15x15 tile in a 32x16x16 box, fp32: 192 KB
        make_entry<32, 16, 8, true, 1>(),     // with the six coefficient arrays on chip: 31x15x7, 192 KB
        make_entry<16, 16, 16, true, 2>(),    // 15x15x15 with coefficients, 192 KB
        make_entry<32, 16, 8, false, 1>(),
        make_entry<16, 16, 16, false, 2>(),
        make_entry<16, 8, 8, false, 2>(),     // small tiles: many-tile schedules on small grids (tests)
        make_entry<16, 8, 8, true, 2>(),
        make_entry<8, 8, 8, false, 2>(),
        make_entry<8, 8, 8, true, 2>(),
    };
    *count = (int)(sizeof(entries) / sizeof(entries[0]));
    return entries;
}

}  // namespace

int systolic_num_configs()
{
    int n;
    table(&n);
    return n;
}

const SysConfig* systolic_config(int idx)
{
    int n;
    const Entry* e = table(&n);
    return (idx >= 0 && idx < n) ? &e[idx].cfg : nullptr;
}

cudaError_t systolic_prepare(int idx, int* blocks_per_sm)
{
    int n;
    const Entry* e = table(&n);
    if (idx < 0 || idx >= n) return cudaErrorInvalidValue;
    cudaError_t err = cudaFuncSetAttribute(e[idx].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e[idx].cfg.smem);
    if (err != cudaSuccess) return err;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, e[idx].fn, e[idx].cfg.threads, e[idx].cfg.smem);
}

cudaError_t launch_systolic(int idx, const SysParams& p, int ctas, cudaStream_t st)
{
    int n;
    const Entry* e = table(&n);
    if (idx < 0 || idx >= n) return cudaErrorInvalidValue;
    void* args[] = {(void*)&p};
    return cudaLaunchKernel(e[idx].fn, dim3((unsigned)ctas), dim3((unsigned)e[idx].cfg.threads), args, e[idx].cfg.smem, st);
}
