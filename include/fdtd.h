/*
 * include/fdtd.h -- C ABI of libfdtd_b200: the 3-D FDTD Yee update of arXiv 2502.20610 on one B200.
 *
 * The library advances Maxwell's curl equations on a Yee grid with the leapfrog update of the paper's
 * eq. (1) (section 2: "E_x += dt/dy (H_z[i,j,k]-H_z[i,j-1,k]) - dt/dz (H_y[i,j,k]-H_y[i,j,k-1])"),
 * the five sibling updates "in the vein of" it, and per-cell structural fields
 * ("permittivity and conductivity", section 4) expressed as update coefficients:
 *
 *     E_a <- ca_a * E_a + cb_a * [ (H_c - H_c[-e_b]) / d_b - (H_b - H_b[-e_c]) / d_c ]      (a,b,c) cyclic
 *     H_a <- H_a  - db_a * [ (E_c[+e_b] - E_c) / d_b - (E_b[+e_c] - E_b) / d_c ]
 *
 * One step = E half-step over the whole grid, soft source, H half-step over the whole grid (Fig. 7 caption,
 * "all the E-field nodes ... after which all the H-field nodes").  Two schedules compute it:
 *   FDTD_KERNEL_NAIVE     one HBM-bound kernel per half-step (the paper's "very straightforward" baseline,
 *                         PAPER.md:54-57, section 2);
 *   FDTD_KERNEL_SYSTOLIC  the paper's systolic scheme (sections 3-4): persistent CTAs keep a
 *                         subdomain on chip, slide it along the x-y-z-t diagonal, exchange only faces through
 *                         global memory and hand off with per-tile flags.  It performs "the exact same update
 *                         equations", so results are identical per cell to the naive schedule.
 *                         Tile 31x15x7 (the default) runs the TMA-staged register kernel (fields in registers,
 *                         coefficients in shared memory, shells fetched by TMA boxes) on every grid: a grid with
 *                         a periodic axis, or with nx % 4 != 0, runs it on a library-owned padded working copy
 *                         (ghost zones of T cells on either side of a periodic axis, refilled before each launch
 *                         of T steps; copy-in / copy-out of the bound arrays around every fdtd_step call).
 *                         Other built tile shapes run FDTD_KERNEL_SYSTOLIC_SMEM.
 *   FDTD_KERNEL_SYSTOLIC_REG   the same schedule and register residency with loader warps staging the shells by
 *                         cp.async (any wall type, any nx; tile 31x15x7 only).
 *   FDTD_KERNEL_SYSTOLIC_SMEM  the same schedule with the whole subdomain in shared memory (the first,
 *                         simpler implementation; kept as a cross-check and for other tile shapes).
 *
 * Layout contract.  Every field / coefficient component is ONE contiguous fp32 array of nx*ny*nz elements,
 * x fastest:  idx = i + nx*(j + ny*k).  Yee positions: E_x(i+1/2,j,k) E_y(i,j+1/2,k) E_z(i,j,k+1/2)
 * H_x(i,j+1/2,k+1/2) H_y(i+1/2,j,k+1/2) H_z(i+1/2,j+1/2,k)  (fixed by eq. (1)'s index pattern).
 * Device pointers must be 16-byte aligned.
 *
 * Time contract.  At entry E holds E^n and H holds H^{n+1/2}; fdtd_step(ctx, n) leaves E^{n0+n}, H^{n0+n+1/2}.
 *
 * Walls (the paper is silent; reading #5).  FDTD_PEC on an axis: tangential E stored at index 0 of
 * that axis is never updated (keeps what the caller put there), tangential E one past the last index is a
 * ghost equal to 0.  FDTD_PERIODIC: indices wrap, every cell is updated.
 *
 * Errors.  Every function except fdtd_destroy / fdtd_last_error returns an FDTD_* status; no exception crosses
 * the ABI.  The Courant limit is NOT enforced.  There is no CPU fallback: without a CUDA device fdtd_create
 * returns FDTD_ECUDA.
 *
 * Thread safety: one ctx per host thread at a time.
 *
 * Environment (read ONCE, in fdtd_create; tuning only, none of them changes a result): FDTD_T = default temporal depth,
 * FDTD_TILE = "NXxNYxNZ" default tile, FDTD_SPIN_BUDGET_MS = hand-off watchdog budget (default 10 s), FDTD_NO_OVERLAP =
 * consecutive systolic launches wait for each other instead of overlapping.  Debug switches exist only in the developer
 * builds (libfdtd_b200_dbg.so / _prof.so).
 */
#ifndef FDTD_B200_H
#define FDTD_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdtd_ctx fdtd_ctx; /* opaque; owned by the library */

enum { FDTD_PEC = 0, FDTD_PERIODIC = 1 };
enum { FDTD_OK = 0, FDTD_EINVAL = 1, FDTD_ENOMEM = 2, FDTD_ECUDA = 3, FDTD_ESTATE = 4, FDTD_ETIMEOUT = 5 };
enum { FDTD_KERNEL_NAIVE = 0, FDTD_KERNEL_SYSTOLIC = 1, FDTD_KERNEL_SYSTOLIC_SMEM = 2, FDTD_KERNEL_SYSTOLIC_REG = 3 };

/* Create a context for an nx*ny*nz grid with cell sizes dx,dy,dz (> 0, finite), time step dt (> 0, finite)
 * and per-axis wall type boundary[3] (host array of FDTD_PEC | FDTD_PERIODIC).
 * cuda_stream: a cudaStream_t (as void*) on which all work is enqueued; NULL = the legacy default stream.
 * Default schedule (no fdtd_set_kernel call): FDTD_KERNEL_SYSTOLIC with library-chosen tile shape and temporal depth
 * on every grid (FDTD_KERNEL_NAIVE only while ca is bound without cb or the reverse); fdtd_get_kernel tells.
 * All later calls run on the device that was current here, whatever device is current in the calling thread.
 * *out is written only on FDTD_OK.  FDTD_EINVAL: bad dims (each 1..2^15, product < 2^40), spacings, dt, boundary.
 * FDTD_ECUDA: no usable sm_100 device / CUDA failure.   (problem statement: PAPER.md:35-37) */
int fdtd_create(fdtd_ctx** out, int nx, int ny, int nz, float dx, float dy, float dz, float dt,
                const int boundary[3], void* cuda_stream);

/* Bind the six field arrays: E[3] = {Ex,Ey,Ez}, H[3] = {Hx,Hy,Hz}; host arrays of DEVICE pointers.
 * The buffers are BORROWED (config 5 is 81 GiB: no copy is affordable) and updated in place by fdtd_step;
 * they must stay valid until rebinding or fdtd_destroy, and must not alias each other.
 * Performance note: when E[0..2] (and H[0..2]) sit at one positive stride (e.g. views of one [3][nz][ny][nx] block)
 * the TMA kernel fetches all three components of a shell piece with a single 4-D box; any placement is correct.
 * FDTD_EINVAL: NULL or misaligned pointer.   (the six arrays of eq. (1) and its siblings) */
int fdtd_set_fields(fdtd_ctx* ctx, float* const E[3], float* const H[3]);

/* The same with the six field arrays stored as IEEE binary16 (row f1; section 4: the paper's engine "halves
 * the number of bytes needed to be loaded per field value, by utilizing 16-bit floating-point representations for the
 * field values"; reading #16).  E[3], H[3]: host arrays of DEVICE pointers to nx*ny*nz binary16 values each,
 * same layout, 16-byte aligned, borrowed and updated in place.  Arithmetic is unchanged (f32, the same expression tree;
 * coefficients, 1/d and source tables stay f32); every newly computed field value -- each half-step, and the source add --
 * is rounded to binary16, nearest-even, before it is stored or used again, so the result does not depend on the schedule
 * and equals the f16-storage build of the oracle bit for bit.  Runs FDTD_KERNEL_NAIVE and FDTD_KERNEL_SYSTOLIC (tile
 * 31x15x7; a periodic axis or nx % 8 != 0 uses the padded working copy); other schedules return FDTD_EINVAL from
 * fdtd_step.  fdtd_load_fields / fdtd_get_fields then copy binary16 arrays (pass the pointers cast to float*). */
int fdtd_set_fields_f16(fdtd_ctx* ctx, void* const E[3], void* const H[3]);

/* Copy initial data from six caller arrays (HOST or device pointers, same layout) into the bound field
 * buffers, asynchronously on the ctx stream.  NULL entries are skipped.  This is the host-buffer entry of
 * the end-to-end path (bench.py `e2e`).  FDTD_ESTATE before fdtd_set_fields. */
int fdtd_load_fields(fdtd_ctx* ctx, const float* const E[3], const float* const H[3]);

/* Bind update coefficients ("structural fields"; reading #2).
 * ca[3], cb[3]: host arrays of DEVICE pointers to per-cell, per-component fp32 arrays (borrowed, read-only),
 *   ca == NULL -> ca_a = 1 everywhere (the multiply is skipped, which is exact);
 *   cb == NULL -> cb_a = dt everywhere (eq. (1)'s vacuum form with 1/d applied inside the curl).
 *   If ca / cb is non-NULL all three entries must be non-NULL.  (Same note as for the fields: six arrays at one
 *   stride, ca first, are fetched with one box per shell piece.)
 * db[3]: HOST array of three scalars (non-magnetic media); NULL -> {dt, dt, dt}.
 * Generator side (not the library's business): ca=(2eps-sigma dt)/(2eps+sigma dt), cb=2dt/(2eps+sigma dt).
 * Contents are constants of the run: treat the arrays as frozen from this call until the next fdtd_set_coeffs /
 * fdtd_set_coeff_lut.  On grids that run on the padded working copy (a periodic axis, or nx % 4 != 0; % 8 with binary16
 * fields, % 16 with material indices) the library copies them once, at the first fdtd_step after this call, and does not
 * look at the caller's arrays again; elsewhere the kernels read the caller's arrays at every launch.  A caller that
 * edits them in place must call fdtd_set_coeffs again (same pointers) to have the edit seen on every grid. */
int fdtd_set_coeffs(fdtd_ctx* ctx, const float* const ca[3], const float* const cb[3], const float db[3]);

/* Compressed coefficients for grids of few materials (row f2; the structural fields "double the number of
 * memory operations needed per iteration"): instead of six float arrays, one material index per cell and component and a
 * table,   ca_a[cell] = ca_lut[a*nmat + idx[a][cell]],   cb_a[cell] = cb_lut[a*nmat + idx[a][cell]].
 * idx[3]: host array of DEVICE pointers to nx*ny*nz bytes each (x fastest, 16-byte aligned, borrowed, read-only, values
 * < nmat); ca_lut, cb_lut: HOST arrays [3][nmat], copied; nmat 1..256; db as in fdtd_set_coeffs.  Replaces any arrays
 * bound with fdtd_set_coeffs (and vice versa).  The update is the one of fdtd_set_coeffs with the expanded arrays, bit for
 * bit; the systolic kernel moves 3 bytes per entering cell instead of 24 and expands them through the table on chip.
 * Runs FDTD_KERNEL_NAIVE and FDTD_KERNEL_SYSTOLIC (tile 31x15x7, f32 fields; a periodic axis or nx % 16 != 0 uses the
 * padded working copy); other schedules return FDTD_EINVAL from fdtd_step. */
int fdtd_set_coeff_lut(fdtd_ctx* ctx, const unsigned char* const idx[3], int nmat, const float* ca_lut, const float* cb_lut,
                       const float db[3]);

/* Additive soft source on one E component over a box (excluded from the paper's own benchmark, PAPER.md:106;
 * DESIGN.md reading #6): after the E half-step of step t,  E_comp[box] += amp[q] * wave[t]  while 0 <= t < nwave
 * (product rounded to fp32, then the add).  comp 0..2 = Ex,Ey,Ez; box origin (i0,j0,k0), extent (ni,nj,nk);
 * amp: HOST array ni*nj*nk, x fastest; wave: HOST array nwave.  Both are copied (caller may free them).
 * amp == NULL removes the source.  FDTD_EINVAL: box outside the grid, comp out of range, nwave < 1. */
int fdtd_set_source(fdtd_ctx* ctx, int comp, int i0, int j0, int k0, int ni, int nj, int nk,
                    const float* amp, const float* wave, int nwave);

/* Running-DFT output monitor on one plane (outputs are excluded from the paper's benchmark but named as what real runs
 * carry; reading #15).  While the step counter t is in [0, nt), every step adds, for each cell of
 * the plane `axis` = `index`, each frequency f < nfreq and each component a:
 *     after the E half-step and the source:  acc[a][f][0|1][cell]     += E_a * wE[t][f][0|1]
 *     after the H half-step:                 acc[3 + a][f][0|1][cell] += H_a * wH[t][f][0|1]
 * (product rounded to fp32, then the add; [0|1] = real | imaginary part of the complex weight).  The weights are the
 * caller's: e.g. wE[t][f] = exp(-i w_f (t+1) dt), wH[t][f] = exp(-i w_f (t+3/2) dt), or a window times these.
 * wE, wH: HOST arrays [nt][nfreq][2], copied.  acc: DEVICE array [6][nfreq][2][cells], BORROWED, not cleared by the
 * library; cells of the plane are numbered x fastest over the two remaining axes (axis 0: j + ny*k; 1: i + nx*k; 2: i + nx*j).
 * One monitor per context; acc == NULL removes it.  Runs inside FDTD_KERNEL_NAIVE and FDTD_KERNEL_SYSTOLIC (tiles
 * 31x15x7 and 31x7x7); other schedules make fdtd_step return FDTD_EINVAL while a monitor is set.
 * FDTD_EINVAL: axis/index outside the grid, nfreq not in 1..64, nt < 1, NULL table, misaligned acc. */
int fdtd_set_monitor(fdtd_ctx* ctx, int axis, int index, int nfreq, int nt, const float* wE, const float* wH, float* acc);

/* Advance n >= 0 steps; enqueues on the ctx stream and returns without synchronising; ctx time += n.
 * FDTD_ESTATE before fdtd_set_fields.  A device-side failure (hand-off watchdog) is reported by the next
 * fdtd_get_fields / fdtd_sync as FDTD_ETIMEOUT.   (eq. (1); sections 3-4 for the schedule) */
int fdtd_step(fdtd_ctx* ctx, int n);

/* Synchronise the ctx stream, then copy the fields out to E[3], H[3] (HOST or device pointers; a NULL array or
 * NULL entry, or an entry equal to the bound pointer, is skipped -- fdtd_get_fields(ctx, NULL, NULL) = sync only).
 * Returns FDTD_ETIMEOUT / FDTD_ECUDA if the enqueued work failed. */
int fdtd_get_fields(fdtd_ctx* ctx, float* const E[3], float* const H[3]);
int fdtd_sync(fdtd_ctx* ctx);

/* Step counter used to index wave[] (resume after a checkpoint: state = six arrays + t). */
int fdtd_set_time(fdtd_ctx* ctx, long long t);
long long fdtd_get_time(const fdtd_ctx* ctx);

/* Choose the schedule.  which = FDTD_KERNEL_NAIVE | FDTD_KERNEL_SYSTOLIC | FDTD_KERNEL_SYSTOLIC_SMEM |
 * FDTD_KERNEL_SYSTOLIC_REG (all four are accepted; the last two are slow cross-check implementations).
 * For the systolic kernel (Nx,Ny,Nz) is the updated tile ("subdomain": 31x15x15 updated inside a
 * 32x16x16 cached block) and T the temporal depth (steps a tile stays resident per launch); 0 = library default.
 * FDTD_EINVAL if the shape is not one the kernel was built for or the grid cannot run it (see fdtd_last_error);
 * the context then keeps the schedule it had before the call. */
int fdtd_set_kernel(fdtd_ctx* ctx, int which, int Nx, int Ny, int Nz, int T);

/* What fdtd_step will run: out[0]=which, out[1..3]=tile Nx,Ny,Nz, out[4]=T, out[5]=tiles per launch,
 * out[6]=CTAs per launch, out[7]=dynamic shared memory bytes per CTA. */
int fdtd_get_kernel(const fdtd_ctx* ctx, int out[8]);

/* Counters since creation: out[0] = kernels launched by fdtd_step, out[1] = steps advanced,
 * out[2] = systolic chunks launched, out[3] = tiles processed. */
int fdtd_get_counters(const fdtd_ctx* ctx, long long out[4]);

/* GPU time of the most recent fdtd_step call in milliseconds (CUDA events recorded on the ctx stream around the enqueued
 * kernels).  Synchronises on the closing event.  Timing is OFF by default: the events sit between the last launch of one
 * call and the first launch of the next and would serialise them, whereas consecutive systolic launches of the same
 * tile grid overlap (the next launch fills the SMs the previous one drains, gated by per-tile flags; PAPER.md:112,
 * DESIGN.md 6.6).  fdtd_set_timing(ctx, 1) switches the events on for later calls; FDTD_ESTATE until a timed call exists. */
int fdtd_set_timing(fdtd_ctx* ctx, int on);
int fdtd_last_step_ms(fdtd_ctx* ctx, float* ms);

/* Pure host function (no device needed): the tile schedule the systolic kernel would use for this grid.
 * ntiles[3] = tiles per axis for a launch of T steps with tile (Nx,Ny,Nz): ceil((n+T)/N) on a PEC axis
 * (tiles enter empty at the high wall and drain at the low wall), ceil(n/N) on a periodic axis (a ring).
 * Returns FDTD_EINVAL for non-positive arguments. */
int fdtd_plan_tiles(const int n[3], const int boundary[3], const int N[3], int T, int ntiles[3]);

/* Pure host function: which tile updates cell coordinate g (0 <= g < n) of one axis at step s of a launch
 * (0 <= s < T) and the cell's offset inside that tile's current region.  start[] are the nb tile starts the
 * library uses for that axis (uniform b*N on a PEC axis; as even as possible on a ring).
 * Writes *tile, *offset.  (reading #11: cell g at step s belongs to the tile whose region [a_b - s, a_{b+1} - s) holds it) */
int fdtd_plan_owner(int n, int boundary, int N, int T, int g, int s, int* tile, int* offset);

/* Developer builds only (libfdtd_b200_dbg.so with FDTD_DEBUG_LEVELS=1 in the environment at fdtd_create): the systolic
 * kernel keeps per-cell time-level shadow arrays and checks every value a tile takes from global memory against the
 * level the schedule promises (the race detector of the hand-off protocol, "delayed synchronization").
 * Synchronises; out[0] = number of violations so far, out[1..4] = the first one (kind: 1/2 H/E at the box load, 3 H
 * shell, 4 E shell; cell offset; level found; level expected).  FDTD_ESTATE when the arrays are off (always in the
 * product library: out is zeroed). */
int fdtd_debug_level_errors(fdtd_ctx* ctx, long long out[5]);

/* Adiabatic-absorber coefficient generator (section 4: "does not use PMLs, but instead relies on the
 * imaginary part of the permittivity to allow for the formation of adiabatic absorbers [5]"; reading #14).
 * Context-free; runs one kernel on `cuda_stream` of the current device and returns without synchronising.
 * Writes the six per-cell update-coefficient arrays that fdtd_set_coeffs takes, for a conductivity that rises as
 * sigma_max * u^order (u = 0 at the inner edge of a layer, 1 at the wall) over `thickness` cells in front of each face:
 *     thickness[6], sigma_max[6]: HOST arrays ordered x-low, x-high, y-low, y-high, z-low, z-high (0 = no layer);
 *     order: integer 0..8 (0 = uniform conductivity inside the layer);  layers of different axes add;
 *     eps[3]: host array of DEVICE pointers to per-cell relative permittivities of E_x, E_y, E_z (NULL, or NULL
 *             entries: 1); ca[3], cb[3]: host arrays of DEVICE pointers, written (nx*ny*nz floats each, x fastest).
 *     E_a of cell (i,j,k) is evaluated at its own Yee position (half a cell further along axis a);
 *     ca = (2 eps - sigma dt)/(2 eps + sigma dt),  cb = 2 dt/(2 eps + sigma dt), every operation rounded to fp32.
 * A round-trip power reflection R0 in a medium of index n_r needs sigma_max = -(order+1) n_r ln(R0) / (2 L d).
 * FDTD_EINVAL: bad dims, negative thickness or sigma_max, thickness > n, order out of range, NULL output. */
int fdtd_absorber_coeffs(int nx, int ny, int nz, float dt, const float* const eps[3], const int thickness[6],
                         const float sigma_max[6], int order, float* const ca[3], float* const cb[3], void* cuda_stream);

/* The systolic kernel for callers that must not allocate device memory.
 *
 * Who this is for: fdtd_create / fdtd_step cudaMalloc the bookkeeping of the systolic schedule (two hand-off flags per
 * tile, tile-claim counters, the claim order, a watchdog word).  A host application that has given all of HBM to its own
 * memory pool has nothing left for that (and config 5 alone is 81 GiB of fields); a stepping loop that shares the GPU
 * with other streams cannot afford the device-wide stall a cudaMalloc or cudaFree may bring.  This one call serves them:
 * it advances the fields by nsteps steps with the same kernel as FDTD_KERNEL_SYSTOLIC (tile 31x15x7, f32), and calls no
 * cudaMalloc, cudaFree or other allocating routine.  The bookkeeping lives in a fixed __device__ array inside the
 * library, about 1.5 MiB, which every GPU that loads the library holds until the process exits.
 *
 * Scope: PEC walls on all three axes, nx a multiple of 4 (other grids need the padded working copy, i.e. an allocation),
 * no source, no monitor, f32 fields.  Inputs and outputs stay the caller's: E[3], H[3] (updated in place), and either
 * ca[3] and cb[3] or neither (NULL, NULL = ca 1, cb dt), all host arrays of 16-byte aligned DEVICE pointers to
 * nx*ny*nz floats, x fastest; db: HOST array of three scalars or NULL (= dt).  T = temporal depth, 0 = 128.
 * Limit: a launch of min(T, nsteps) steps may have at most FDTD_NOALLOC_MAX_TILES tiles,
 *     ceil((nx+T)/31) * ceil((ny+T)/15) * ceil((nz+T)/7)      (fdtd_plan_tiles computes it on the host);
 * e.g. 512^3 at T = 128 is 83 076 tiles and fits, 768^3 at T = 128 does not (pass T = 32).  A larger job returns
 * FDTD_EINVAL and says so in errbuf; it is checked before anything touches the GPU.
 *
 * Behaviour to know about.
 *   - The call works on the CURRENT device and on cuda_stream (NULL = legacy default stream), and returns only after
 *     the GPU work has finished: it has to read the watchdog word.  FDTD_ETIMEOUT = a hand-off waited more than 10 s,
 *     fields invalid.
 *   - The first call on each device does a one-time set-up (it asks the runtime for the array's device address and sets
 *     the kernel's shared-memory attribute).  Make that first call before any stream capture begins.
 *   - All calls share the one array, and it still holds whatever the previous call wrote.  Each call therefore clears
 *     the flags, counters and watchdog word on cuda_stream before its first launch.  Two runs in flight on one GPU
 *     would raise and poll the same flags and corrupt each other, so the library holds a lock for the whole call:
 *     a second host thread calling in waits until the first run is done.
 *   - The step counter is not kept anywhere: state = the six arrays.
 * errbuf (may be NULL): receives a NUL-terminated message of at most errbuf_len bytes on failure, "" on success.
 * Results are bit-identical to fdtd_step on the same inputs (same kernel, same per-cell arithmetic). */
enum { FDTD_NOALLOC_MAX_TILES = 131072 };
int fdtd_step_noalloc(int nx, int ny, int nz, float dx, float dy, float dz, float dt, float* const E[3], float* const H[3],
                      const float* const ca[3], const float* const cb[3], const float db[3], int nsteps, int T,
                      void* cuda_stream, char* errbuf, int errbuf_len);

const char* fdtd_last_error(const fdtd_ctx* ctx); /* text of the last failure on this ctx; never NULL */
const char* fdtd_build_info(void);                /* e.g. "sm_100a fmad=true" */
void fdtd_destroy(fdtd_ctx* ctx);                 /* NULL-safe; never frees borrowed buffers */

#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_H */
