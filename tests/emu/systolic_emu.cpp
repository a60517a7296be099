// tests/emu/systolic_emu.cpp -- CPU-side schedule harness for the systolic kernel's tile stages.  TEST CODE ONLY.
//
// It compiles paper_2502_20610_b200/csrc/systolic_tile.cuh (the very stage functions the CUDA kernel calls)
// with plain g++ and drives them as per-tile state machines under an adversarial scheduler, so that the tile
// geometry, shell enumeration, wall clipping, ring wrap, flag protocol and in-place hazards can be checked
// against the oracle without a GPU (-m "not gpu").  It is not a fallback: nothing in the package loads it.
//
// Each tile advances through sub-stages; a sub-stage that starts with a wait is runnable only when all seven
// upwind flags have reached the target, exactly as systolic_kernel.cu spins on them:
//   4k+0: [k>0: wait flagH >= k] load box / H shell       4k+1: E phase, publish E, flagE = k+1
//   4k+2: wait flagE >= k+1, load E shell                 4k+3: H phase, publish H, flagH = k+1
// Tiles are claimed in lexicographic order by `ctas` virtual CTAs (the persistent grid); the scheduler picks a
// runnable (cta, sub-stage) by policy: 0 serial upwind-first, 1 uniformly random, 2 prefer the most advanced,
// 3 prefer the least advanced, 4 prefer the highest tile index.  Shared memory is poisoned with NaN at claim.
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "../../paper_2502_20610_b200/csrc/systolic_tile.cuh"

namespace {

struct Rng {
    uint64_t s;
    uint32_t next() { s = s * 6364136223846793005ull + 1442695040888963407ull; return (uint32_t)(s >> 33); }
};

template <int BX, int BY, int BZ, bool COEF, int ZSPLIT>
int run_launch(SysParams P, int ctas, int policy, uint64_t seed, long long* stage_count)
{
    using Tile = SysTile<BX, BY, BZ, COEF, ZSPLIT>;
    struct Cta { int tile; int sp; Tile t; std::vector<float> sm; };
    std::vector<int> flagE(P.ntiles, 0), flagH(P.ntiles, 0);
    std::vector<Cta> cta(ctas);
    int next_tile = 0, done = 0;
    Rng rng{seed * 2 + 1};
    auto claim = [&](Cta& c) {
        if (next_tile >= P.ntiles) { c.tile = -1; return; }
        c.tile = next_tile++;
        c.sp = 0;
        c.t.init(P, c.tile);
        c.sm.assign((size_t)Tile::BV * Tile::NF, nanf(""));
    };
    for (auto& c : cta) claim(c);
    auto ready = [&](const Cta& c) {
        const int k = c.sp / 4, sub = c.sp % 4;
        if (sub == 0 && k > 0) {
            for (int q = 0; q < 7; ++q) if (c.t.nbr[q] >= 0 && flagH[c.t.nbr[q]] < k) return false;
        } else if (sub == 2) {
            for (int q = 0; q < 7; ++q) if (c.t.nbr[q] >= 0 && flagE[c.t.nbr[q]] < k + 1) return false;
        }
        return true;
    };
    auto run = [&](Cta& c) {
        const int k = c.sp / 4, sub = c.sp % 4;
        float* sm = c.sm.data();
        c.t.begin_step(k, P.T);
        if (sub == 0) {
            for (int tid = 0; tid < Tile::NT; ++tid) { if (k == 0) c.t.load_initial(P, sm, tid); else c.t.load_h_shell(P, sm, tid); }
        } else if (sub == 1) {
            for (int tid = 0; tid < Tile::NT; ++tid) c.t.e_phase(P, sm, tid);
            for (int tid = 0; tid < Tile::NT; ++tid) c.t.publish_e(P, sm, tid);
            flagE[c.tile] = k + 1;
        } else if (sub == 2) {
            for (int tid = 0; tid < Tile::NT; ++tid) c.t.load_e_shell(P, sm, tid);
        } else {
            for (int tid = 0; tid < Tile::NT; ++tid) c.t.h_phase(P, sm, tid);
            for (int tid = 0; tid < Tile::NT; ++tid) c.t.publish_h(P, sm, tid);
            flagH[c.tile] = k + 1;
        }
        ++*stage_count;
        if (++c.sp == 4 * P.T) { ++done; claim(c); }
    };
    while (done < P.ntiles) {
        std::vector<int> cand;
        for (int i = 0; i < ctas; ++i) if (cta[i].tile >= 0 && ready(cta[i])) cand.push_back(i);
        if (cand.empty()) return 2;   // deadlock: the protocol or the claim order is wrong
        int pick = cand[0];
        if (policy == 0) {            // serial: always the lowest tile index (upwind first)
            for (int i : cand) if (cta[i].tile < cta[pick].tile) pick = i;
        } else if (policy == 1) {
            pick = cand[rng.next() % cand.size()];
        } else {
            // biased policies, with a random pick one time in four so that everybody eventually moves
            if (rng.next() % 4 == 0) pick = cand[rng.next() % cand.size()];
            else for (int i : cand) {
                const Cta &x = cta[i], &y = cta[pick];
                if (policy == 2 && x.sp > y.sp) pick = i;
                if (policy == 3 && x.sp < y.sp) pick = i;
                if (policy == 4 && x.tile > y.tile) pick = i;
            }
        }
        run(cta[pick]);
    }
    return 0;
}

}  // namespace

extern "C" {

// Runs nsteps steps in launches of at most T steps on host arrays.  g: GridParams with HOST pointers.
// box = {Bx,By,Bz}; returns 0 ok, 1 unsupported box, 2 deadlock.
int systolic_emu_run(const GridParams* g, const int box[3], int T, int nsteps, long long t0, int ctas, int policy,
                     unsigned long long seed, long long* stage_count)
{
    const bool coef = g->ca[0] != nullptr;
    int left = nsteps;
    long long t = t0;
    long long dummy = 0;
    if (!stage_count) stage_count = &dummy;
    while (left > 0) {
        const int Tl = left < T ? left : T;
        SysParams P;
        memset(&P, 0, sizeof P);
        P.g = *g;
        P.T = Tl;
        P.t0 = t;
        long long nt = 1;
        const int N[3] = {box[0] - 1, box[1] - 1, box[2] - 1};
        for (int a = 0; a < 3; ++a) {
            P.ax[a] = make_axis_plan(g->n[a], g->per[a], N[a], Tl);
            nt *= P.ax[a].nb;
        }
        P.ntiles = (int)nt;
        int rc = 1;
#define EMU_CASE(BX, BY, BZ, ZS)                                                                              \
        if (box[0] == BX && box[1] == BY && box[2] == BZ)                                                         \
            rc = coef ? run_launch<BX, BY, BZ, true, ZS>(P, ctas, policy, seed + (unsigned long long)t, stage_count)  \
                      : run_launch<BX, BY, BZ, false, ZS>(P, ctas, policy, seed + (unsigned long long)t, stage_count);
        EMU_CASE(8, 8, 8, 2)
        EMU_CASE(16, 8, 8, 2)
        EMU_CASE(4, 4, 4, 1)
        EMU_CASE(8, 4, 4, 2)
        EMU_CASE(32, 16, 8, 1)
        EMU_CASE(16, 16, 16, 2)
        EMU_CASE(32, 16, 16, 1)
#undef EMU_CASE
        if (rc != 0) return rc;
        t += Tl;
        left -= Tl;
    }
    return 0;
}

}  // extern "C"

// layout check for the ctypes mirror in harness.py
extern "C" int systolic_emu_sizeof_grid() { return (int)sizeof(GridParams); }
