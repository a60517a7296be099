/*
 * oracle/yee_oracle.c -- CPU oracle for the 3-D FDTD Yee update of arXiv 2502.20610.
 *
 * *** TEST INFRASTRUCTURE.  NOT THE PRODUCT. ***
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, link, import or execute anything under oracle/.  It shares no code,
 * header, table or helper with paper_2502_20610_b200/ (the CUDA path), and neither
 * imports the other.
 *
 * What it computes.  The paper's systolic scheme performs "the exact same update
 * equations" as plain FDTD (section 1) and in its final form updates "all the
 * E-field nodes ... simultaneously, after which all the H-field nodes" (Fig. 7 caption,
 * PAPER.md:161).  The result therefore has a plain definition -- n repetitions of
 *     { E half-step over the whole grid ; source ; H half-step over the whole grid } --
 * and this file is that definition written out as literal triple loops, one C statement
 * per rounded floating-point operation, no blocking, fusion or reordering.
 *
 *   E half-step: eq. (1), PAPER.md:37 (section 2), printed for E_x only:
 *       E_x += (dt/dy)(H_z[i,j,k]-H_z[i,j-1,k]) - (dt/dz)(H_y[i,j,k]-H_y[i,j,k-1])
 *   The other five updates are "in the vein of" eq. (1): cyclic permutation of
 *   (x,y,z) for E_y, E_z; Faraday's law with forward differences for H (Yee, ref. [8],
 *   PAPER.md:133) -- the staggering is fixed by eq. (1)'s backward differences on H.
 *   Structural fields ("permittivity and conductivity", section 4) enter as
 *   per-cell, per-component coefficients ca, cb:  E_a <- ca_a E_a + cb_a curl_a(H),
 *   H_a <- H_a - db_a curl_a(E).
 *
 * Readings where the paper is silent (all listed in DESIGN.md):
 *   #1 other five components: cyclic permutation + Faraday sign.
 *   #2 coefficient form above; 1/d_a applied inside the curl, rd_a = (REAL)(1.0/(double)d_a).
 *   #3 expression tree, each operation rounded to nearest-even separately:
 *        d1 = Hc[p]-Hc[p-e_b]; d2 = Hb[p]-Hb[p-e_c]; curl = d1*rd_b - d2*rd_c;
 *        Ea = ca*Ea + cb*curl      (ca absent: the multiply by 1 is skipped, which is exact)
 *        Ha = Ha - db*curl(E)      with e1 = Ec[p+e_b], e2 = Eb[p+e_c] forward neighbours.
 *   #4 one step = E half-step, source, H half-step; inputs are (E^0, H^{1/2}).
 *   #5 walls: PEC box -- tangential E stored at index 0 of a PEC axis is never updated,
 *      tangential E one past the last index is a ghost equal to 0; periodic = index wrap.
 *   #6 source: additive on one E component over a box, E += amp[q]*wave[t] (product rounded,
 *      then the add), after the E half-step of step t, only while 0 <= t < nwave.
 *   #7 fp32 storage and arithmetic (BASELINE.json); the fp64 build exists for the physics pins.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): PEC-cavity eigenfrequency closed form,
 * oblique plane-wave dispersion in a periodic box, div H and div D conservation, exact
 * leapfrog energy conservation, lossy three-term recurrence, magic-time-step exact shift,
 * cyclic-permutation symmetry, hand-expanded 4^3 grids in exact rational arithmetic.
 * Parity unpinned: none of the arithmetic; the *wave physics* of heterogeneous-eps
 * interfaces has no closed form in the paper and is covered only by the div D / energy
 * invariants and the 4^3 brute force (stated in DESIGN.md).
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC (oracle/build_oracle.py).
 * No flush-to-zero: Gaussian source tails go subnormal and must stay so.
 */
#include <stddef.h>

enum { YEE_PEC = 0, YEE_PERIODIC = 1 };

#define YEE_GRID_STRUCT(REAL, NAME)                                                              \
    typedef struct {                                                                             \
        int n[3];            /* nx, ny, nz */                                                    \
        int bnd[3];          /* YEE_PEC | YEE_PERIODIC per axis */                               \
        REAL rd[3];          /* 1/dx, 1/dy, 1/dz, rounded once from double */                    \
        REAL *E[3];          /* Ex, Ey, Ez: n cells each, x fastest, updated in place */         \
        REAL *H[3];          /* Hx, Hy, Hz */                                                    \
        const REAL *ca[3];   /* per-cell E decay factor per component, or NULL (= 1) */          \
        const REAL *cb[3];   /* per-cell E curl factor per component, or NULL (= cb_scalar) */   \
        REAL cb_scalar;      /* used where cb[a] == NULL; caller passes (REAL)dt */              \
        REAL db[3];          /* H curl factor per component */                                   \
        int src_comp;        /* 0..2 = Ex, Ey, Ez */                                             \
        int src_box[6];      /* i0, j0, k0, ni, nj, nk */                                        \
        const REAL *src_amp; /* ni*nj*nk, x fastest, or NULL (no source) */                      \
        const REAL *src_wave;/* nwave samples */                                                 \
        int src_nwave;                                                                           \
        int nthreads;        /* OpenMP threads over k; does not change per-cell arithmetic */    \
    } NAME

YEE_GRID_STRUCT(float, yee_grid_f32);
YEE_GRID_STRUCT(double, yee_grid_f64);

#define REAL float
#define FN(x) x##_f32
#define STORE(x) (x)
#include "yee_oracle_impl.h"
#undef REAL
#undef FN
#undef STORE

/* f16 field storage with f32 arithmetic (section 4: "halves the number of bytes needed
 * to be loaded per field value, by utilizing 16-bit floating-point representations for the field values").
 * reading #16: the six field arrays hold IEEE binary16 values; every update reads them (exact conversion to f32),
 * evaluates the same f32 expression tree, and rounds the new value to binary16 (nearest-even) when it is stored -- at every
 * half-step, so that the result does not depend on how long a value stays on chip.  The source add rounds likewise.
 * Coefficients, 1/d and the source tables stay f32.  The arrays of this build are float arrays whose values are
 * binary16-representable (the caller rounds the inputs). */
typedef yee_grid_f32 yee_grid_h16;
#define REAL float
#define FN(x) x##_h16
#define STORE(x) ((float)(_Float16)(x))
#include "yee_oracle_impl.h"
#undef REAL
#undef FN
#undef STORE

#define REAL double
#define FN(x) x##_f64
#define STORE(x) (x)
#include "yee_oracle_impl.h"
#undef REAL
#undef FN
