// yee_update.h -- the per-component arithmetic of the Yee update, shared by the naive and the systolic kernels
// (CUDA path only).  One statement per rounded operation; with -fmad=false this is the expression tree of
// DESIGN.md reading #3 and the result is bit-identical to the fp32 oracle, in any schedule.
#pragma once
#include "fdtd_types.h"

// E_a <- ca_a E_a + cb_a [ (H_c - H_c[-e_b]) rd_b - (H_b - H_b[-e_c]) rd_c ]      (eq. (1))
template <bool HAS_CA>
FDTD_HD float yee_e_update(float e, float hc, float hc_m, float hb, float hb_m, float rdb, float rdc, float ca, float cb)
{
    const float d1 = hc - hc_m;
    const float d2 = hb - hb_m;
    const float t1 = d1 * rdb;
    const float t2 = d2 * rdc;
    const float curl = t1 - t2;
    const float keep = HAS_CA ? ca * e : e;
    const float gain = cb * curl;
    return keep + gain;
}

// H_a <- H_a - db_a [ (E_c[+e_b] - E_c) rd_b - (E_b[+e_c] - E_b) rd_c ]         (Faraday; Yee [8])
FDTD_HD float yee_h_update(float h, float ec_p, float ec, float eb_p, float eb, float rdb, float rdc, float db)
{
    const float d1 = ec_p - ec;
    const float d2 = eb_p - eb;
    const float t1 = d1 * rdb;
    const float t2 = d2 * rdc;
    const float curl = t1 - t2;
    const float loss = db * curl;
    return h - loss;
}
