// Tap evaluation shared by the gridder (ws_grid.cu, Eq. 3 at PAPER.md:80) and the degridder (ws_degrid.cu, :459):
// the 1-D convolution function at the S integer offsets around a visibility, in registers.
#pragma once
#include "ws_internal.h"

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// The 2 S taps of one record: gu[i] = g(i - h - fx) / norm1, gv likewise (norm1^2 is folded into weight * vis).
template <int S, bool KB>
__device__ __forceinline__ void eval_taps(const WsGeom& g, float fx, float fy, float* gu, float* gv) {
    constexpr int H = (S - 1) / 2;
    if constexpr (!KB) {
        const float tap_c = g.tap_c;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const float dx = (float)(i - H) - fx, dy = (float)(i - H) - fy;
            gu[i] = ex2_approx(tap_c * dx * dx);
            gv[i] = ex2_approx(tap_c * dy * dy);
        }
    } else {
        // I0(beta sqrt(y)) / I0(beta) = sum_k c_k y^k, y = 1 - (2x/S)^2 in [0, 1], c_k > 0: Horner without cancellation
        float yu[S], yv[S];
        const float ky = g.kb_y;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const float dx = (float)(i - H) - fx, dy = (float)(i - H) - fy;
            yu[i] = fmaxf(fmaf(-ky * dx, dx, 1.0f), 0.0f);
            yv[i] = fmaxf(fmaf(-ky * dy, dy, 1.0f), 0.0f);
        }
        int k = g.kb_terms - 1;
        const float top = g.kb_c[k];
#pragma unroll
        for (int i = 0; i < S; ++i) gu[i] = gv[i] = top;
        for (--k; k >= 0; --k) {
            const float c = g.kb_c[k];
#pragma unroll
            for (int i = 0; i < S; ++i) {
                gu[i] = fmaf(gu[i], yu[i], c);
                gv[i] = fmaf(gv[i], yv[i], c);
            }
        }
    }
}

