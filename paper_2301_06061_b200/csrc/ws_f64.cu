// WS_FLAG_MESH_F64: the path with the paper's own arithmetic -- mesh, image and every sum in fp64 (PAPER.md:392,
// Table 3 :306-314: "mesh ... double precision, real and imaginary part") -- for like-for-like context against its
// Table 4 (:428-443), not for speed.  The gridder also takes the paper's own GPU kernel shape: one thread per measurement,
// atomicAdd on the mesh in global memory (:207, :219); nothing is binned, no workspace is needed.  The per-plane FFT is
// cuFFT Z2Z (ws_api.cu); the w-correction evaluates exp(2 pi i w_k (n - 1)) in fp64 for every pixel and plane.
// Positions follow the same rule O2-O4 as the fp32 path (ws_place.cuh); the taps are evaluated in fp64 at the exact offset.
#include "ws_internal.h"
#include "ws_place.cuh"

namespace {

struct F64Kernel {
    int32_t type, support;
    double param;            // sigma (Gaussian) or beta (Kaiser-Bessel)
    double norm1;            // Gaussian: 1 / (sigma sqrt(2 pi)); Kaiser-Bessel: beta / (S sinh beta)
};

__device__ __forceinline__ double i0_series(double x) {      // I0(x) = sum_k (x^2/4)^k / (k!)^2
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}
__device__ __forceinline__ double tap64(const F64Kernel& kk, double x) {
    if (kk.type == WS_KERNEL_KAISER_BESSEL) {
        const double t = 2.0 * x / (double)kk.support, y = 1.0 - t * t;
        return y < 0.0 ? 0.0 : kk.norm1 * i0_series(kk.param * sqrt(y));
    }
    return kk.norm1 * exp(-x * x / (2.0 * kk.param * kk.param));
}

// thread = visibility (presum = 0) or row whose n_chan visibilities share one position (presum = 1: sum_c wt V first)
__global__ void __launch_bounds__(256)
k_grid_f64(const __grid_constant__ WsChanConsts cc, const __grid_constant__ WsGeom g, const __grid_constant__ F64Kernel kk,
           const float* __restrict__ uvw, const float2* __restrict__ vis, const float* __restrict__ wt, uint64_t n_items,
           uint32_t n_chan, int presum, double* __restrict__ grid, double* __restrict__ sum_wt) {
    const uint64_t m = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    double wsum = 0.0;
    if (m < n_items) {
        const uint64_t row = presum ? m : m / n_chan;
        const uint32_t c = presum ? 0u : (uint32_t)(m - row * n_chan);
        Placed pl;
        if (place(cc, g, __ldg(uvw + 3 * row), __ldg(uvw + 3 * row + 1), __ldg(uvw + 3 * row + 2), cc.su[c], cc.sw[c], pl)) {
            double vr = 0.0, vi = 0.0;
            if (presum) {
                for (uint32_t ch = 0; ch < n_chan; ++ch) {
                    const float2 v = vis[row * n_chan + ch];
                    const double w = (double)wt[row * n_chan + ch];
                    vr += w * (double)v.x;
                    vi += w * (double)v.y;
                    wsum += w;
                }
            } else {
                const float2 v = vis[m];
                const double w = (double)wt[m];
                vr = w * (double)v.x;
                vi = w * (double)v.y;
                wsum = w;
            }
            const int S = g.support, h = g.halo, N = g.n_pix, half = N >> 1;
            double gu[2 * WS_HALO_MAX + 1], gv[2 * WS_HALO_MAX + 1];
            for (int a = 0; a < S; ++a) {
                gu[a] = tap64(kk, (double)(a - h) - pl.fu);
                gv[a] = tap64(kk, (double)(a - h) - pl.fv);
            }
            double* plane = grid + (size_t)pl.k * N * N * 2;
            for (int b = 0; b < S; ++b) {
                const int sy = (pl.j0 + b - h + half) & (N - 1);                 // FFT-native storage (wstack.h)
                for (int a = 0; a < S; ++a) {
                    const int sx = (pl.i0 + a - h + half) & (N - 1);
                    const double t = gu[a] * gv[b];
                    double* cell = plane + ((size_t)sy * N + sx) * 2;
                    atomicAdd(cell, vr * t);
                    atomicAdd(cell + 1, vi * t);
                }
            }
        }
    }
    if (sum_wt) {
#pragma unroll
        for (int d = 16; d; d >>= 1) wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        if ((threadIdx.x & 31) == 0 && wsum != 0.0) atomicAdd(sum_wt, wsum);
    }
}

// a4 in fp64: thread = pixel; image (+)= sum_k exp(2 pi i w_k t) P_k, the phase reduced to a fraction of a turn first
__global__ void __launch_bounds__(256)
k_wcorrect_f64(int N, int nw, double cell, double w0, double dw, const double2* __restrict__ planes,
               double2* __restrict__ image, int accumulate, double* __restrict__ dirty) {
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= (uint64_t)N * N) return;
    const int q = (int)(tid / N), p = (int)(tid - (uint64_t)q * N), half = N >> 1;
    const double l = (double)(p - half) * cell, mm = (double)(q - half) * cell, r2 = l * l + mm * mm;
    double2 acc = make_double2(0.0, 0.0);
    if (r2 < 1.0) {
        const double t = -r2 / (1.0 + sqrt(1.0 - r2));
        const size_t off = (size_t)((q + half) & (N - 1)) * N + ((p + half) & (N - 1));
        for (int k = 0; k < nw; ++k) {
            const double turns = (w0 + (double)k * dw) * t;
            double s, c;
            sincospi(2.0 * (turns - rint(turns)), &s, &c);
            const double2 v = planes[(size_t)k * N * N + off];
            acc.x += c * v.x - s * v.y;
            acc.y += c * v.y + s * v.x;
        }
    }
    if (accumulate) {
        const double2 old = image[tid];
        acc.x += old.x;
        acc.y += old.y;
    }
    image[tid] = acc;
    if (dirty) dirty[tid] = acc.x;
}

__device__ __forceinline__ double taper64(const F64Kernel& kk, double xi) {
    const double PI = 3.14159265358979323846264338327950288;
    if (kk.type == WS_KERNEL_KAISER_BESSEL) {
        const double a = PI * (double)kk.support * xi, d = kk.param * kk.param - a * a;
        double f = 1.0;
        if (d > 1e-12) f = sinh(sqrt(d)) / sqrt(d);
        else if (d < -1e-12) f = sin(sqrt(-d)) / sqrt(-d);
        return f * kk.param / sinh(kk.param);
    }
    return exp(-2.0 * PI * PI * kk.param * kk.param * xi * xi);
}

__global__ void __launch_bounds__(256)
k_dirty_f64(int N, double cell, const __grid_constant__ F64Kernel kk, uint32_t flags, const double* __restrict__ sum_wt,
            const double2* __restrict__ image, double* __restrict__ dirty) {
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= (uint64_t)N * N) return;
    const int q = (int)(tid / N), p = (int)(tid - (uint64_t)q * N), half = N >> 1;
    double f = 1.0;
    if (flags & WS_NORM_SUMWT) f /= *sum_wt;
    if (flags & WS_NORM_N) {
        const double l = (double)(p - half) * cell, mm = (double)(q - half) * cell, r2 = l * l + mm * mm;
        f *= r2 < 1.0 ? sqrt(1.0 - r2) : 0.0;
    }
    if (flags & WS_NORM_TAPER) f /= taper64(kk, (double)(p - half) / (double)N) * taper64(kk, (double)(q - half) / (double)N);
    dirty[tid] = image[tid].x * f;
}

F64Kernel make_kernel(const ws_plan* plan) {
    const double PI = 3.14159265358979323846264338327950288;
    F64Kernel kk;
    kk.type = plan->prm.kernel_type;
    kk.support = plan->prm.support;
    kk.param = plan->prm.kernel_param;
    kk.norm1 = kk.type == WS_KERNEL_KAISER_BESSEL ? kk.param / ((double)kk.support * sinh(kk.param))
                                                  : 1.0 / (kk.param * sqrt(2.0 * PI));
    return kk;
}

}  // namespace

int ws_launch_grid_f64(ws_plan* plan, const WsChanConsts& cc, const float* uvw, const float2* vis, const float* wt,
                       int64_t n_rows, int32_t n_chan, int presum, double* grid, cudaStream_t st) {
    const uint64_t n_items = presum ? (uint64_t)n_rows : (uint64_t)n_rows * (uint64_t)n_chan;
    if (n_items == 0) return 0;
    double* sw = (plan->prm.flags & WS_FLAG_TRACK_SUMWT) ? plan->d_sumwt : nullptr;
    k_grid_f64<<<(unsigned)((n_items + 255) / 256), 256, 0, st>>>(cc, plan->geom, make_kernel(plan), uvw, vis, wt, n_items,
                                                                  (uint32_t)n_chan, presum, grid, sw);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}

int ws_launch_wcorrect_f64(ws_plan* plan, const void* planes, void* image, int accumulate, void* dirty, cudaStream_t st) {
    const ws_params& P = plan->prm;
    const double dw = (P.w_max - P.w_min) / (double)P.n_wplanes, w0 = P.w_min + 0.5 * dw;
    const uint64_t n = (uint64_t)P.n_pix * (uint64_t)P.n_pix;
    k_wcorrect_f64<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(P.n_pix, P.n_wplanes, P.cell_rad, w0, dw, (const double2*)planes,
                                                                (double2*)image, accumulate, (double*)dirty);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}

int ws_launch_dirty_f64(ws_plan* plan, const void* image, void* dirty, uint32_t norm_flags, cudaStream_t st) {
    const uint64_t n = (uint64_t)plan->prm.n_pix * (uint64_t)plan->prm.n_pix;
    k_dirty_f64<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(plan->prm.n_pix, plan->prm.cell_rad, make_kernel(plan), norm_flags,
                                                             plan->d_sumwt, (const double2*)image, (double*)dirty);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}
