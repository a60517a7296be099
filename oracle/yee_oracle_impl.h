/*
 * oracle/yee_oracle_impl.h -- body of the CPU oracle, included once per precision.
 *
 * TEST INFRASTRUCTURE ONLY.  See yee_oracle.c for the header comment, the
 * citations and the list of readings.  This file is included with
 *   REAL   = float | double
 *   FN(x)  = x##_f32 | x##_f64
 * and holds literal triple loops, one statement per rounded operation.
 *   STORE(x) = x for the f32 / f64 builds; the f16-storage build (row f1) rounds every value it
 *   stores to IEEE binary16, nearest-even, and keeps it in a float array.
 *
 * Index convention: idx = i + nx*(j + ny*k), x fastest.
 */

/* ---- E half-step:  E <- ca*E + cb*curl(H), backward differences on H (eq. (1)) ---- */
static void FN(e_half)(const FN(yee_grid) *g)
{
    const int nx = g->n[0], ny = g->n[1], nz = g->n[2];
    const int px = g->bnd[0] == YEE_PERIODIC, py = g->bnd[1] == YEE_PERIODIC, pz = g->bnd[2] == YEE_PERIODIC;
    const REAL rdx = g->rd[0], rdy = g->rd[1], rdz = g->rd[2];
    REAL *Ex = g->E[0], *Ey = g->E[1], *Ez = g->E[2];
    const REAL *Hx = g->H[0], *Hy = g->H[1], *Hz = g->H[2];
    int k;
#pragma omp parallel for schedule(static) num_threads(g->nthreads)
    for (k = 0; k < nz; ++k) {
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) {
                const size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                /* neighbour one cell back along each axis; wraps on a periodic axis.
                 * On a PEC axis index 0 has no back neighbour: the components that
                 * would need it are the frozen tangential ones (reading #5). */
                const size_t pxm = (i > 0) ? p - 1 : p + (size_t)(nx - 1);
                const size_t pym = (j > 0) ? p - (size_t)nx : p + (size_t)nx * (size_t)(ny - 1);
                const size_t pzm = (k > 0) ? p - (size_t)nx * ny : p + (size_t)nx * ny * (size_t)(nz - 1);
                const int wall_x = (!px && i == 0), wall_y = (!py && j == 0), wall_z = (!pz && k == 0);

                /* E_x: eq. (1) verbatim:  (Hz - Hz[j-1])/dy - (Hy - Hy[k-1])/dz */
                if (!(wall_y || wall_z)) {
                    const REAL d1 = Hz[p] - Hz[pym];
                    const REAL d2 = Hy[p] - Hy[pzm];
                    const REAL t1 = d1 * rdy;
                    const REAL t2 = d2 * rdz;
                    const REAL curl = t1 - t2;
                    const REAL keep = g->ca[0] ? (REAL)(g->ca[0][p] * Ex[p]) : Ex[p];
                    const REAL cb = g->cb[0] ? g->cb[0][p] : g->cb_scalar;
                    const REAL gain = cb * curl;
                    Ex[p] = STORE(keep + gain);
                }
                /* E_y:  (Hx - Hx[k-1])/dz - (Hz - Hz[i-1])/dx */
                if (!(wall_z || wall_x)) {
                    const REAL d1 = Hx[p] - Hx[pzm];
                    const REAL d2 = Hz[p] - Hz[pxm];
                    const REAL t1 = d1 * rdz;
                    const REAL t2 = d2 * rdx;
                    const REAL curl = t1 - t2;
                    const REAL keep = g->ca[1] ? (REAL)(g->ca[1][p] * Ey[p]) : Ey[p];
                    const REAL cb = g->cb[1] ? g->cb[1][p] : g->cb_scalar;
                    const REAL gain = cb * curl;
                    Ey[p] = STORE(keep + gain);
                }
                /* E_z:  (Hy - Hy[i-1])/dx - (Hx - Hx[j-1])/dy */
                if (!(wall_x || wall_y)) {
                    const REAL d1 = Hy[p] - Hy[pxm];
                    const REAL d2 = Hx[p] - Hx[pym];
                    const REAL t1 = d1 * rdx;
                    const REAL t2 = d2 * rdy;
                    const REAL curl = t1 - t2;
                    const REAL keep = g->ca[2] ? (REAL)(g->ca[2][p] * Ez[p]) : Ez[p];
                    const REAL cb = g->cb[2] ? g->cb[2][p] : g->cb_scalar;
                    const REAL gain = cb * curl;
                    Ez[p] = STORE(keep + gain);
                }
            }
        }
    }
}

/* ---- soft source: E_comp[box] += amp[q]*wave[t]   (reading #6; excluded from the paper's benchmark) ---- */
static void FN(add_source)(const FN(yee_grid) *g, long long t)
{
    if (!g->src_amp || !g->src_wave || t < 0 || t >= (long long)g->src_nwave) return;
    const int nx = g->n[0], ny = g->n[1];
    REAL *Ec = g->E[g->src_comp];
    const REAL w = g->src_wave[t];
    for (int kk = 0; kk < g->src_box[5]; ++kk)
        for (int jj = 0; jj < g->src_box[4]; ++jj)
            for (int ii = 0; ii < g->src_box[3]; ++ii) {
                const size_t q = (size_t)ii + (size_t)g->src_box[3] * ((size_t)jj + (size_t)g->src_box[4] * (size_t)kk);
                const size_t p = (size_t)(g->src_box[0] + ii)
                               + (size_t)nx * ((size_t)(g->src_box[1] + jj) + (size_t)ny * (size_t)(g->src_box[2] + kk));
                const REAL inj = g->src_amp[q] * w;
                Ec[p] = STORE(Ec[p] + inj);
            }
}

/* ---- H half-step:  H <- H - db*curl(E), forward differences on E (reading #1; Yee [8]) ---- */
static void FN(h_half)(const FN(yee_grid) *g)
{
    const int nx = g->n[0], ny = g->n[1], nz = g->n[2];
    const int px = g->bnd[0] == YEE_PERIODIC, py = g->bnd[1] == YEE_PERIODIC, pz = g->bnd[2] == YEE_PERIODIC;
    const REAL rdx = g->rd[0], rdy = g->rd[1], rdz = g->rd[2];
    const REAL *Ex = g->E[0], *Ey = g->E[1], *Ez = g->E[2];
    REAL *Hx = g->H[0], *Hy = g->H[1], *Hz = g->H[2];
    int k;
#pragma omp parallel for schedule(static) num_threads(g->nthreads)
    for (k = 0; k < nz; ++k) {
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) {
                const size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                /* neighbour one cell forward; periodic: wrap; PEC: ghost tangential E beyond the high wall is 0 */
                const int last_x = (i == nx - 1), last_y = (j == ny - 1), last_z = (k == nz - 1);
                const size_t pxp = last_x ? p - (size_t)(nx - 1) : p + 1;
                const size_t pyp = last_y ? p - (size_t)nx * (size_t)(ny - 1) : p + (size_t)nx;
                const size_t pzp = last_z ? p - (size_t)nx * ny * (size_t)(nz - 1) : p + (size_t)nx * ny;
                const REAL zero = (REAL)0;
                const REAL Ey_xp = (last_x && !px) ? zero : Ey[pxp];
                const REAL Ez_xp = (last_x && !px) ? zero : Ez[pxp];
                const REAL Ex_yp = (last_y && !py) ? zero : Ex[pyp];
                const REAL Ez_yp = (last_y && !py) ? zero : Ez[pyp];
                const REAL Ex_zp = (last_z && !pz) ? zero : Ex[pzp];
                const REAL Ey_zp = (last_z && !pz) ? zero : Ey[pzp];

                /* H_x -= db_x * [ (Ez[j+1]-Ez)/dy - (Ey[k+1]-Ey)/dz ] */
                {
                    const REAL d1 = Ez_yp - Ez[p];
                    const REAL d2 = Ey_zp - Ey[p];
                    const REAL t1 = d1 * rdy;
                    const REAL t2 = d2 * rdz;
                    const REAL curl = t1 - t2;
                    const REAL loss = g->db[0] * curl;
                    Hx[p] = STORE(Hx[p] - loss);
                }
                /* H_y -= db_y * [ (Ex[k+1]-Ex)/dz - (Ez[i+1]-Ez)/dx ] */
                {
                    const REAL d1 = Ex_zp - Ex[p];
                    const REAL d2 = Ez_xp - Ez[p];
                    const REAL t1 = d1 * rdz;
                    const REAL t2 = d2 * rdx;
                    const REAL curl = t1 - t2;
                    const REAL loss = g->db[1] * curl;
                    Hy[p] = STORE(Hy[p] - loss);
                }
                /* H_z -= db_z * [ (Ey[i+1]-Ey)/dx - (Ex[j+1]-Ex)/dy ] */
                {
                    const REAL d1 = Ey_xp - Ey[p];
                    const REAL d2 = Ex_yp - Ex[p];
                    const REAL t1 = d1 * rdx;
                    const REAL t2 = d2 * rdy;
                    const REAL curl = t1 - t2;
                    const REAL loss = g->db[2] * curl;
                    Hz[p] = STORE(Hz[p] - loss);
                }
            }
        }
    }
}

/* n full steps: { E half-step; source with wave[t]; H half-step; t++ }  (Fig. 7 caption; reading #4) */
int FN(yee_oracle_run)(const FN(yee_grid) *g, long long t0, int nsteps)
{
    if (!g || nsteps < 0) return 1;
    for (int a = 0; a < 3; ++a) {
        if (g->n[a] < 1 || !g->E[a] || !g->H[a]) return 1;
        if (g->bnd[a] != YEE_PEC && g->bnd[a] != YEE_PERIODIC) return 1;
    }
    if (g->src_amp) {
        if (g->src_comp < 0 || g->src_comp > 2) return 1;
        for (int a = 0; a < 3; ++a)
            if (g->src_box[a] < 0 || g->src_box[3 + a] < 1 || g->src_box[a] + g->src_box[3 + a] > g->n[a]) return 1;
    }
    for (int s = 0; s < nsteps; ++s) {
        FN(e_half)(g);
        FN(add_source)(g, t0 + s);
        FN(h_half)(g);
    }
    return 0;
}

/* single half-steps, exported so the pins can look between them (energy pin P5 needs H at consecutive half-levels) */
int FN(yee_oracle_e_half)(const FN(yee_grid) *g) { FN(e_half)(g); return 0; }
int FN(yee_oracle_h_half)(const FN(yee_grid) *g) { FN(h_half)(g); return 0; }
