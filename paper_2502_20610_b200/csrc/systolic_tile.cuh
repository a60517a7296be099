// systolic_tile.cuh -- the stages one tile ("subdomain") goes through in the systolic schedule.
//
// A tile of (w_x, w_y, w_z) <= (BX-1, BY-1, BZ-1) cells lives in shared memory inside a BX x BY x BZ box
// ("a 32x16x16 block of Yee cells is stored in cache, to allow for loading of boundary values").
// At step k of a launch its region is R_k = [a - k, a + w - k) per axis: it slides one cell toward -x,-y,-z per
// time step ("traverse ... along the x-y-z-t diagonal") and the box [a-k-1, a+w-k) holds R_k and
// R_{k+1}.  Shared-memory slots are addressed by the global cell coordinate modulo the box size, so the slide
// moves no data (a10).
//
//   step k:  [wait H of upwind tiles]  load H (+coefficients) on the minus shell of the box   (a7)
//            E phase on R_k: all E nodes at once (Fig. 7), soft source          (a1, a4)
//            publish E of the cells leaving the tile, R_k \ R_{k+1}; release flagE            (a8, a9)
//            [wait E of upwind tiles]  load E on the minus shell                              (a7)
//            H phase on R_{k+1}                                                               (a2)
//            publish H of R_{k+1} \ R_{k+2}; release flagH                                    (a8, a9)
//   step 0 loads the whole box instead of a shell; step T-1 publishes the whole region (a6).
//
// "Local" coordinates l = g - o, o = a - k - 1 (the box origin), l in [0, w]:  R_k = [1,w]^3, R_{k+1} = [0,w-1]^3.
// Cells outside the domain on a PEC axis are zero-filled on load and never updated or stored; that realises
// both "ghost tangential E beyond the high wall = 0" and the clipped entry/drain tiles of the launch ramp (a11).
//
// Every stage is a function of the thread index so that the same code runs as CUDA threads separated by
// __syncthreads() (systolic_kernel.cu) and, for the CPU-side schedule tests, as plain loops (tests/emu).
#pragma once
#include "fdtd_types.h"
#include "yee_update.h"

#if defined(__CUDA_ARCH__)
#define SYS_LDCG(p) __ldcg(p)            // L2-only: shell data is written by other SMs, L1 is not coherent
#define SYS_STCG(p, v) __stcg((p), (v))
#define SYS_LDRO(p) __ldg(p)
#else
#define SYS_LDCG(p) (*(p))
#define SYS_STCG(p, v) (*(p) = (v))
#define SYS_LDRO(p) (*(p))
#endif

enum { SYS_MINUS_SHELL = 0, SYS_PLUS_SHELL = 1, SYS_FULL = 2 };

template <int BX, int BY, int BZ, bool COEF, int ZSPLIT>
struct SysTile {
    static constexpr int BV = BX * BY * BZ;
    static constexpr int NT = BX * BY * ZSPLIT;
    static constexpr int NF = COEF ? 12 : 6;   // arrays on chip: Ex Ey Ez Hx Hy Hz [cax cay caz cbx cby cbz]
    static constexpr size_t kSmemBytes = (size_t)BV * NF * sizeof(float);

    int b[3], a[3], w[3];   // tile coordinates, start, width
    int nbr[7];             // the seven upwind neighbours (3 faces, 3 edges, 1 corner) or -1   (reading #11)
    int o[3];               // box origin at the current step (unwrapped global coordinate of local 0)
    int k;
    bool last;

    FDTD_HD void init(const SysParams& P, int tile)
    {
        const int nbx = P.ax[0].nb, nby = P.ax[1].nb;
        b[0] = tile % nbx;
        b[1] = (tile / nbx) % nby;
        b[2] = tile / (nbx * nby);
        for (int q = 0; q < 3; ++q) {
            a[q] = P.ax[q].start(b[q]);
            w[q] = P.ax[q].width(b[q]);
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
            nbr[d - 1] = ok ? idx[0] + nbx * (idx[1] + nby * idx[2]) : -1;
        }
    }

    FDTD_HD void begin_step(int kk, int T)
    {
        k = kk;
        last = (kk == T - 1);
        for (int q = 0; q < 3; ++q) o[q] = a[q] - kk - 1;
    }

    // unwrapped global coordinate -> stored coordinate; false if outside the domain on a PEC axis
    static FDTD_HD bool resolve(const SysParams& P, int axis, int gu, int& g)
    {
        const int n = P.g.n[axis];
        if (P.ax[axis].per) {
            gu %= n;
            g = gu < 0 ? gu + n : gu;
            return true;
        }
        g = gu;
        return gu >= 0 && gu < n;
    }

    static FDTD_HD int slot(int gxu, int gyu, int gzu)
    {
        return ((gzu & (BZ - 1)) * BY + (gyu & (BY - 1))) * BX + (gxu & (BX - 1));
    }

    // ---- enumeration of a box / of the shell of a box, x fastest --------------------------------------------
    // SYS_FULL: [lo,hi]^3.  SYS_MINUS_SHELL: cells with some l_a == lo_a.  SYS_PLUS_SHELL: some l_a == hi_a.
    static FDTD_HD int region_count(const int lo[3], const int hi[3], int mode)
    {
        const int ex = hi[0] - lo[0] + 1, ey = hi[1] - lo[1] + 1, ez = hi[2] - lo[2] + 1;
        if (ex <= 0 || ey <= 0 || ez <= 0) return 0;
        if (mode == SYS_FULL) return ex * ey * ez;
        return ex * ey + ex * (ez - 1) + (ey - 1) * (ez - 1);
    }

    static FDTD_HD void region_cell(int idx, const int lo[3], const int hi[3], int mode, int l[3])
    {
        const int ex = hi[0] - lo[0] + 1, ey = hi[1] - lo[1] + 1, ez = hi[2] - lo[2] + 1;
        if (mode == SYS_FULL) {
            l[0] = lo[0] + idx % ex;
            l[1] = lo[1] + (idx / ex) % ey;
            l[2] = lo[2] + idx / (ex * ey);
            return;
        }
        const int sh = (mode == SYS_MINUS_SHELL) ? 1 : 0;   // the non-face range starts one above lo on a minus shell
        const int nZ = ex * ey, nY = ex * (ez - 1);
        if (idx < nZ) {                                     // slab l_z = face
            l[0] = lo[0] + idx % ex;
            l[1] = lo[1] + idx / ex;
            l[2] = sh ? lo[2] : hi[2];
        } else if (idx < nZ + nY) {                         // slab l_y = face, l_z off the face
            const int r = idx - nZ;
            l[0] = lo[0] + r % ex;
            l[1] = sh ? lo[1] : hi[1];
            l[2] = lo[2] + sh + r / ex;
        } else {                                            // slab l_x = face, l_y and l_z off their faces
            const int r = idx - nZ - nY;
            l[0] = sh ? lo[0] : hi[0];
            l[1] = lo[1] + sh + r % (ey - 1);
            l[2] = lo[2] + sh + r / (ey - 1);
        }
    }

    static FDTD_HD const float* array_ptr(const SysParams& P, int c)
    {
        return c < 3 ? P.g.E[c] : c < 6 ? P.g.H[c - 3] : c < 9 ? P.g.ca[c - 6] : P.g.cb[c - 9];
    }

    // Move arrays c in [c0,c1) between global memory and the box for every cell of a region (a6, a7, a8).
    template <bool LOAD>
    FDTD_HD void transfer(const SysParams& P, float* sm, int tid, int c0, int c1, const int lo[3], const int hi[3], int mode) const
    {
        const int ncell = region_count(lo, hi, mode);
        const int total = ncell * (c1 - c0);
        const long long nx = P.g.n[0], ny = P.g.n[1];
        for (int q = tid; q < total; q += NT) {
            const int c = c0 + q / ncell;
            int l[3], g[3];
            region_cell(q % ncell, lo, hi, mode, l);
            const int gxu = o[0] + l[0], gyu = o[1] + l[1], gzu = o[2] + l[2];
            const bool in = resolve(P, 0, gxu, g[0]) & resolve(P, 1, gyu, g[1]) & resolve(P, 2, gzu, g[2]);
            const long long gi = g[0] + nx * (g[1] + ny * (long long)g[2]);
            const int s = c * BV + slot(gxu, gyu, gzu);
            if (LOAD) {
                float v = 0.0f;
                if (in) v = (c < 6) ? SYS_LDCG(array_ptr(P, c) + gi) : SYS_LDRO(array_ptr(P, c) + gi);
                sm[s] = v;
            } else if (in) {
                SYS_STCG(const_cast<float*>(array_ptr(P, c)) + gi, sm[s]);
            }
        }
    }

    // step 0: the whole box of H (+ coefficients), E on R_0                                           (a6)
    FDTD_HD void load_initial(const SysParams& P, float* sm, int tid) const
    {
        const int lo0[3] = {0, 0, 0}, lo1[3] = {1, 1, 1}, hi[3] = {w[0], w[1], w[2]};
        transfer<true>(P, sm, tid, 3, NF, lo0, hi, SYS_FULL);
        transfer<true>(P, sm, tid, 0, 3, lo1, hi, SYS_FULL);
    }
    // steps k > 0: H (+ coefficients) on the full minus shell of the box                                (a7)
    FDTD_HD void load_h_shell(const SysParams& P, float* sm, int tid) const
    {
        const int lo[3] = {0, 0, 0}, hi[3] = {w[0], w[1], w[2]};
        transfer<true>(P, sm, tid, 3, NF, lo, hi, SYS_MINUS_SHELL);
    }
    // E on the full minus shell (faces + edges + corner: reading #10)                                   (a7)
    FDTD_HD void load_e_shell(const SysParams& P, float* sm, int tid) const
    {
        const int lo[3] = {0, 0, 0}, hi[3] = {w[0], w[1], w[2]};
        transfer<true>(P, sm, tid, 0, 3, lo, hi, SYS_MINUS_SHELL);
    }
    // E of R_k \ R_{k+1} (the plus shell of [1,w]^3); everything at the last step                        (a8, a6)
    FDTD_HD void publish_e(const SysParams& P, float* sm, int tid) const
    {
        const int lo[3] = {1, 1, 1}, hi[3] = {w[0], w[1], w[2]};
        transfer<false>(P, sm, tid, 0, 3, lo, hi, last ? SYS_FULL : SYS_PLUS_SHELL);
    }
    // H of R_{k+1} \ R_{k+2} (the plus shell of [0,w-1]^3); everything at the last step
    FDTD_HD void publish_h(const SysParams& P, float* sm, int tid) const
    {
        const int lo[3] = {0, 0, 0}, hi[3] = {w[0] - 1, w[1] - 1, w[2] - 1};
        transfer<false>(P, sm, tid, 3, 6, lo, hi, last ? SYS_FULL : SYS_PLUS_SHELL);
    }

    // E phase on R_k = [1,w]^3: thread = one (x,y) column of the box, marching its share of z with the
    // z-neighbour H carried in registers.  Soft source after the update (a1, a4).
    FDTD_HD void e_phase(const SysParams& P, float* sm, int tid) const
    {
        const int xs = tid % BX, ys = (tid / BX) % BY, zp = tid / (BX * BY);
        const int lx = (xs - o[0]) & (BX - 1), ly = (ys - o[1]) & (BY - 1);
        if (lx < 1 || lx > w[0] || ly < 1 || ly > w[1]) return;
        int gx, gy;
        if (!(resolve(P, 0, o[0] + lx, gx) & resolve(P, 1, o[1] + ly, gy))) return;
        const int per = (w[2] + ZSPLIT - 1) / ZSPLIT;
        const int z0 = 1 + zp * per;
        const int z1 = (z0 + per - 1 < w[2]) ? z0 + per - 1 : w[2];
        const bool wall_x = !P.ax[0].per && gx == 0, wall_y = !P.ax[1].per && gy == 0;
        const float rdx = P.g.rd[0], rdy = P.g.rd[1], rdz = P.g.rd[2];
        const int col = ys * BX + xs;
        const int col_xm = ys * BX + ((xs - 1) & (BX - 1));
        const int col_ym = ((ys - 1) & (BY - 1)) * BX + xs;
        const long long t = P.t0 + k;
        const bool has_src = P.g.src_comp >= 0 && t >= 0 && t < P.g.src_nwave;
        const float wsrc = has_src ? SYS_LDRO(P.g.src_wave + t) : 0.0f;
        const int sx = gx - P.g.src_box[0], sy = gy - P.g.src_box[1];
        const bool src_col = has_src && sx >= 0 && sx < P.g.src_box[3] && sy >= 0 && sy < P.g.src_box[4];
        const float* Hx = sm + 3 * BV;
        const float* Hy = sm + 4 * BV;
        const float* Hz = sm + 5 * BV;

        const int pl0 = ((o[2] + z0 - 1) & (BZ - 1)) * (BX * BY);
        float hx_m = Hx[pl0 + col], hy_m = Hy[pl0 + col];
        for (int lz = z0; lz <= z1; ++lz) {
            const int pl = ((o[2] + lz) & (BZ - 1)) * (BX * BY);
            const float hx = Hx[pl + col], hy = Hy[pl + col], hz = Hz[pl + col];
            int gz;
            if (resolve(P, 2, o[2] + lz, gz)) {
                const bool wall_z = !P.ax[2].per && gz == 0;
                float ex = sm[0 * BV + pl + col], ey = sm[1 * BV + pl + col], ez = sm[2 * BV + pl + col];
                float cax = 1.0f, cay = 1.0f, caz = 1.0f, cbx = P.g.cb_scalar, cby = cbx, cbz = cbx;
                if (COEF) {
                    cax = sm[6 * BV + pl + col]; cay = sm[7 * BV + pl + col]; caz = sm[8 * BV + pl + col];
                    cbx = sm[9 * BV + pl + col]; cby = sm[10 * BV + pl + col]; cbz = sm[11 * BV + pl + col];
                }
                if (!(wall_y || wall_z))   // E_x: (Hz - Hz[j-1])/dy - (Hy - Hy[k-1])/dz      eq. (1)
                    ex = yee_e_update<COEF>(ex, hz, Hz[pl + col_ym], hy, hy_m, rdy, rdz, cax, cbx);
                if (!(wall_z || wall_x))   // E_y: (Hx - Hx[k-1])/dz - (Hz - Hz[i-1])/dx
                    ey = yee_e_update<COEF>(ey, hx, hx_m, hz, Hz[pl + col_xm], rdz, rdx, cay, cby);
                if (!(wall_x || wall_y))   // E_z: (Hy - Hy[i-1])/dx - (Hx - Hx[j-1])/dy
                    ez = yee_e_update<COEF>(ez, hy, Hy[pl + col_xm], hx, Hx[pl + col_ym], rdx, rdy, caz, cbz);
                if (src_col) {
                    const int sz = gz - P.g.src_box[2];
                    if (sz >= 0 && sz < P.g.src_box[5]) {
                        const float amp = SYS_LDRO(P.g.src_amp + (sx + P.g.src_box[3] * (sy + (long long)P.g.src_box[4] * sz)));
                        const float inj = amp * wsrc;
                        if (P.g.src_comp == 0) ex = ex + inj;
                        else if (P.g.src_comp == 1) ey = ey + inj;
                        else ez = ez + inj;
                    }
                }
                sm[0 * BV + pl + col] = ex;
                sm[1 * BV + pl + col] = ey;
                sm[2 * BV + pl + col] = ez;
            }
            hx_m = hx;
            hy_m = hy;
        }
    }

    // H phase on R_{k+1} = [0,w-1]^3; the z-neighbour E (one plane up) is carried to the next iteration (a2).
    FDTD_HD void h_phase(const SysParams& P, float* sm, int tid) const
    {
        const int xs = tid % BX, ys = (tid / BX) % BY, zp = tid / (BX * BY);
        const int lx = (xs - o[0]) & (BX - 1), ly = (ys - o[1]) & (BY - 1);
        if (lx > w[0] - 1 || ly > w[1] - 1) return;
        int gx, gy;
        if (!(resolve(P, 0, o[0] + lx, gx) & resolve(P, 1, o[1] + ly, gy))) return;
        const int per = (w[2] + ZSPLIT - 1) / ZSPLIT;
        const int z0 = zp * per;
        const int z1 = (z0 + per - 1 < w[2] - 1) ? z0 + per - 1 : w[2] - 1;
        const float rdx = P.g.rd[0], rdy = P.g.rd[1], rdz = P.g.rd[2];
        const float dbx = P.g.db[0], dby = P.g.db[1], dbz = P.g.db[2];
        const int col = ys * BX + xs;
        const int col_xp = ys * BX + ((xs + 1) & (BX - 1));
        const int col_yp = ((ys + 1) & (BY - 1)) * BX + xs;
        const float* Ex = sm + 0 * BV;
        const float* Ey = sm + 1 * BV;
        const float* Ez = sm + 2 * BV;

        if (z0 > z1) return;
        const int pl0 = ((o[2] + z0) & (BZ - 1)) * (BX * BY);
        float ex = Ex[pl0 + col], ey = Ey[pl0 + col];
        for (int lz = z0; lz <= z1; ++lz) {
            const int pl = ((o[2] + lz) & (BZ - 1)) * (BX * BY);
            const int plp = ((o[2] + lz + 1) & (BZ - 1)) * (BX * BY);
            const float ex_p = Ex[plp + col], ey_p = Ey[plp + col];
            int gz;
            if (resolve(P, 2, o[2] + lz, gz)) {
                const float ez = Ez[pl + col];
                float hx = sm[3 * BV + pl + col], hy = sm[4 * BV + pl + col], hz = sm[5 * BV + pl + col];
                hx = yee_h_update(hx, Ez[pl + col_yp], ez, ey_p, ey, rdy, rdz, dbx);   // (Ez[j+1]-Ez)/dy - (Ey[k+1]-Ey)/dz
                hy = yee_h_update(hy, ex_p, ex, Ez[pl + col_xp], ez, rdz, rdx, dby);   // (Ex[k+1]-Ex)/dz - (Ez[i+1]-Ez)/dx
                hz = yee_h_update(hz, Ey[pl + col_xp], ey, Ex[pl + col_yp], ex, rdx, rdy, dbz);   // (Ey[i+1]-Ey)/dx - (Ex[j+1]-Ex)/dy
                sm[3 * BV + pl + col] = hx;
                sm[4 * BV + pl + col] = hy;
                sm[5 * BV + pl + col] = hz;
            }
            ex = ex_p;
            ey = ey_p;
        }
    }
};
