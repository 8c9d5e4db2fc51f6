// Phase screen of the w-correction, Eq. 2:  exp(2 pi i w_k (sqrt(1 - l^2 - m^2) - 1)),
// w_k = w_min + (k + 1/2) dw.  Shared by the stand-alone pass (ws_wcorrect.cu) and the fused FFT epilogue
// (ws_fft.cu).  The phases of one pixel over the planes are a geometric sequence exp(2 pi i (phi0 + k delta));
// phi0 and delta are formed and range-reduced in fp64 (|w (n-1)| reaches ~10^2 turns, where an fp32 product
// is 1e-5 rad off), n - 1 as -r^2 / (1 + sqrt(1 - r^2)), never by subtraction; only the fraction of a turn
// goes to sincospif.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct WcParams {
    int32_t n_pix, n_wplanes;
    double cell, w0, dw;      // w0 = w_min + dw/2
};

__device__ __forceinline__ float2 ws_cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// acc * r + p  (one Horner step of the plane sum)
__device__ __forceinline__ float2 ws_horner(float2 acc, float2 r, float px, float py) {
    return make_float2(fmaf(acc.x, r.x, fmaf(-acc.y, r.y, px)), fmaf(acc.x, r.y, fmaf(acc.y, r.x, py)));
}
__device__ __forceinline__ float2 ws_expi_turns(double turns) {
    const float f = (float)(turns - rint(turns));   // fraction in [-1/2, 1/2], reduced in fp64
    float s, c;
    sincospif(2.0f * f, &s, &c);
    return make_float2(c, s);
}
// n - 1 of logical pixel (q, p); *inside = false where l^2 + m^2 >= 1 (reading R14: such pixels receive 0)
__device__ __forceinline__ double ws_n_minus_1(const WcParams& prm, int q, int p, bool* inside) {
    const int half = prm.n_pix >> 1;
    const double l = (double)(p - half) * prm.cell, m = (double)(q - half) * prm.cell;
    const double r2 = l * l + m * m;
    *inside = r2 < 1.0;
    return *inside ? -r2 / (1.0 + sqrt(1.0 - r2)) : 0.0;
}
