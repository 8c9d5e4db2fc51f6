// The position rule O2-O4 (DESIGN.md section 3; PAPER.md:66 "closest w-plane", :78 the per-region lists), shared by the
// binning kernels (ws_bin.cu) and the fp64-mesh gridder (ws_f64.cu).
#pragma once
#include "ws_internal.h"

// Position rule.  Each line is one correctly rounded binary64 operation,
// in the order the header states; the oracle performs the same operations on the host.
struct Placed {
    int i0, j0, k;
    double fu, fv;
};

__device__ __forceinline__ bool place(const WsChanConsts& cc, const WsGeom& g, float u, float v, float w, double su,
                                      double sw, Placed& o) {
    const double pu = __fma_rn((double)u, su, cc.half);
    const double pv = __fma_rn((double)v, su, cc.half);
    const double pw = __fma_rn((double)w, sw, cc.ow);
    const double ci = floor(__dadd_rn(pu, 0.5));   // nearest cell centre, ties up (R4)
    const double cj = floor(__dadd_rn(pv, 0.5));
    double ck = floor(pw);                          // N_w equal bins over [w_min, w_max] (R6)
    ck = ck < 0.0 ? 0.0 : ck;
    const double ktop = (double)(g.n_wplanes - 1);
    ck = ck > ktop ? ktop : ck;
    const double lo = (double)g.halo, hi = (double)(g.n_pix - 1 - g.halo);
    if (!(ci >= lo && ci <= hi && cj >= lo && cj <= hi && pw == pw)) return false;   // drop rule O3 (R5); a NaN in u, v or w drops (R33)
    if (ck < (double)g.plane_lo || ck >= (double)g.plane_hi) return false;           // another rank's planes (ws_plan_set_plane_range)
    o.k = (int)ck;
    o.i0 = (int)ci;
    o.j0 = (int)cj;
    o.fu = __dsub_rn(pu, ci);                       // exact, in [-1/2, 1/2)
    o.fv = __dsub_rn(pv, cj);
    return true;
}

__device__ __forceinline__ uint32_t bin_of(const WsGeom& g, int k, int ty, int tx) {
    return ((uint32_t)k * (uint32_t)g.nt + (uint32_t)ty) * (uint32_t)g.nt + (uint32_t)tx;
}

