// a4: w-correction and reduction over the planes, Eq. 2 (PAPER.md:68; step 4 at :86, :152):
//   D(l, m) = sum_k exp(2 pi i w_k (sqrt(1 - l^2 - m^2) - 1)) P_k(l, m),   w_k = w_min + (k + 1/2) dw.
// The paper runs one CUDA thread per (i, j, k) cell with atomicAdd into the image.  Here
// the whole sum is ONE streaming pass: a thread owns two adjacent pixels, reads them from every plane once
// (16-byte loads, 8 in flight), keeps the sum in registers and writes the image once -- no atomics.
// The phases of one pixel are a geometric sequence, exp(2 pi i (phi0 + k delta)), so the planes are summed by
// Horner's rule in blocks of WS_WC_GROUP planes: inside a block with r = exp(2 pi i delta), between blocks
// with R = exp(2 pi i GROUP delta) evaluated exactly, which bounds the fp32 drift to GROUP roundings.
// phi0, delta and GROUP*delta are formed and range-reduced in fp64 (|w (n-1)| reaches ~10^2 turns, where an
// fp32 product is 1e-5 rad off), n - 1 as -r^2 / (1 + sqrt(1 - r^2)); only the fraction goes to sincospif.
#include "ws_internal.h"
#include "ws_phase.cuh"

namespace {

constexpr int G = WS_WC_GROUP;

struct PixelPhase {
    float2 e0, r, R;
    bool inside;
};
__device__ __forceinline__ PixelPhase pixel_phase(const WcParams& prm, int q, int p) {
    PixelPhase o;
    const double t = ws_n_minus_1(prm, q, p, &o.inside);   // n - 1, never by subtraction
    const double delta = prm.dw * t;
    o.e0 = ws_expi_turns(prm.w0 * t);
    o.r = ws_expi_turns(delta);
    o.R = ws_expi_turns((double)G * delta);
    return o;
}

__global__ void __launch_bounds__(256)
k_wcorrect(const __grid_constant__ WcParams prm, const float4* __restrict__ planes, float4* __restrict__ image,
           int accumulate, float2* __restrict__ dirty) {
    const uint32_t N = (uint32_t)prm.n_pix, halfN = N >> 1, pairs = N >> 1;
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= (uint64_t)N * pairs) return;
    const uint32_t q = (uint32_t)(tid / pairs), p = (uint32_t)(tid - (uint64_t)q * pairs) * 2u;
    // wrapped (FFT-native) position of logical pixel (q, p) inside a plane
    const uint32_t sq = q >= halfN ? q - halfN : q + halfN;
    const uint32_t sp = p >= halfN ? p - halfN : p + halfN;
    const size_t plane_stride = (size_t)N * pairs;                 // in float4 units
    const float4* src = planes + (size_t)sq * pairs + (sp >> 1);

    const PixelPhase A = pixel_phase(prm, (int)q, (int)p), B = pixel_phase(prm, (int)q, (int)p + 1);
    float2 dA = make_float2(0.f, 0.f), dB = make_float2(0.f, 0.f);
    const int nw = prm.n_wplanes;
    const int n_groups = (nw + G - 1) / G;
    for (int gI = n_groups - 1; gI >= 0; --gI) {
        const int lo = gI * G;
        float4 v[G];
#pragma unroll
        for (int j = 0; j < G; ++j)
            v[j] = lo + j < nw ? __ldcs(src + (size_t)(lo + j) * plane_stride) : make_float4(0.f, 0.f, 0.f, 0.f);
        float2 hA = make_float2(0.f, 0.f), hB = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = G - 1; j >= 0; --j) {
            hA = ws_horner(hA, A.r, v[j].x, v[j].y);
            hB = ws_horner(hB, B.r, v[j].z, v[j].w);
        }
        dA = ws_horner(dA, A.R, hA.x, hA.y);
        dB = ws_horner(dB, B.R, hB.x, hB.y);
    }
    dA = ws_cmul(dA, A.e0);
    dB = ws_cmul(dB, B.e0);
    if (!A.inside) dA = make_float2(0.f, 0.f);   // R14
    if (!B.inside) dB = make_float2(0.f, 0.f);
    float4* dst = image + tid;                    // centred image, row q, pixels p, p+1
    float4 out = make_float4(dA.x, dA.y, dB.x, dB.y);
    if (accumulate) {
        const float4 old = *dst;
        out.x += old.x; out.y += old.y; out.z += old.z; out.w += old.w;
    }
    *dst = out;
    if (dirty) dirty[tid] = make_float2(out.x, out.z);
}

// a5: dirty = Re(image)
__global__ void __launch_bounds__(256)
k_dirty(const float4* __restrict__ image, float2* __restrict__ dirty, uint64_t n_pairs) {
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= n_pairs) return;
    const float4 v = __ldcs(image + tid);
    dirty[tid] = make_float2(v.x, v.z);
}

// a5 with normalisation (wstack.h WS_NORM_*; Eq. 2 solved for I): Re(image) times 1 / sum of weights,
// n = sqrt(1 - l^2 - m^2) (fp64, 0 outside the unit circle) and 1 / (ghat(xi_p) ghat(xi_q)) from the plan's table.
__global__ void __launch_bounds__(256)
k_dirty_norm(const float4* __restrict__ image, float2* __restrict__ dirty, uint32_t N, double cell, uint32_t flags,
             const double* __restrict__ sum_wt, const float* __restrict__ inv_taper) {
    const uint32_t pairs = N >> 1;
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= (uint64_t)N * pairs) return;
    const uint32_t q = (uint32_t)(tid / pairs), p = (uint32_t)(tid - (uint64_t)q * pairs) * 2u;
    const float4 v = __ldcs(image + tid);
    double fa = 1.0, fb = 1.0;
    if (flags & WS_NORM_SUMWT) fa = fb = 1.0 / *sum_wt;
    if (flags & WS_NORM_N) {
        const int half = (int)(N >> 1);
        const double m = (double)((int)q - half) * cell, la = (double)((int)p - half) * cell, lb = (double)((int)p + 1 - half) * cell;
        const double ra = la * la + m * m, rb = lb * lb + m * m;
        fa *= ra < 1.0 ? sqrt(1.0 - ra) : 0.0;
        fb *= rb < 1.0 ? sqrt(1.0 - rb) : 0.0;
    }
    if (flags & WS_NORM_TAPER) {
        const double tq = (double)inv_taper[q];
        fa *= tq * (double)inv_taper[p];
        fb *= tq * (double)inv_taper[p + 1];
    }
    dirty[tid] = make_float2((float)((double)v.x * fa), (float)((double)v.z * fb));
}

}  // namespace

int ws_launch_wcorrect(ws_plan* plan, const float2* planes, float2* image, int accumulate, float* dirty,
                       cudaStream_t st) {
    const ws_params& P = plan->prm;
    WcParams prm;
    prm.n_pix = P.n_pix;
    prm.n_wplanes = P.n_wplanes;
    prm.cell = P.cell_rad;
    prm.dw = (P.w_max - P.w_min) / (double)P.n_wplanes;
    prm.w0 = P.w_min + 0.5 * prm.dw;
    const uint64_t n_pairs = (uint64_t)P.n_pix * (uint64_t)(P.n_pix / 2);
    k_wcorrect<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>(prm, (const float4*)planes, (float4*)image, accumulate,
                                                                  (float2*)dirty);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_dirty(ws_plan* plan, const float2* image, float* dirty, uint32_t norm_flags, cudaStream_t st) {
    const uint64_t n_pairs = (uint64_t)plan->prm.n_pix * (uint64_t)(plan->prm.n_pix / 2);
    if (norm_flags) {
        k_dirty_norm<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>((const float4*)image, (float2*)dirty,
                                                                        (uint32_t)plan->prm.n_pix, plan->prm.cell_rad, norm_flags,
                                                                        plan->d_sumwt, plan->d_taper);
        if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
        return 1;
    }
    k_dirty<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>((const float4*)image, (float2*)dirty, n_pairs);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_zero(ws_plan* plan, void* ptr, size_t bytes, cudaStream_t st) {
    (void)plan;
    if (cudaMemsetAsync(ptr, 0, bytes, st) != cudaSuccess) return WS_ERR_CUDA;
    return 0;
}
