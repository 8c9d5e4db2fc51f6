// Diagnostic, not on the hot path: the fp32 FMA rate a register-only loop reaches on this GPU.  bench.py prints it
// beside the DERIVED fp32 peak (SMs x lanes x 2 x clock) it holds the arithmetic-bound row pass of the FFT against.
#include "ws_internal.h"

namespace {

__global__ void __launch_bounds__(256)
k_probe_ffma(float* __restrict__ out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);      // 16 independent chains per thread
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;                               // keeps the loop alive, never true in practice
}

}  // namespace

extern "C" int ws_measure_fp32_tflops(ws_plan* plan, double* tflops, void* stream) {
    if (!plan || !tflops) return WS_ERR_INVALID_ARG;
    int prev = -1;
    const bool switched = cudaGetDevice(&prev) == cudaSuccess && prev != plan->prm.device && cudaSetDevice(plan->prm.device) == cudaSuccess;
    struct Restore { int d; bool on; ~Restore() { if (on) cudaSetDevice(d); } } restore{prev, switched};
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return WS_ERR_CUDA;
    const int iters = 4096, ctas = plan->sm_count * 16;
    float* sink = (float*)plan->d_sumwt + 2;                       // 8 spare bytes of a plan-owned block
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        k_probe_ffma<<<ctas, 256, 0, st>>>(sink, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * 16.0 * (double)iters * 256.0 * (double)ctas;
        if (ms > 0.f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    plan->launches += 4;
    *tflops = best;
    return cudaGetLastError() == cudaSuccess && best > 0.0 ? WS_OK : WS_ERR_CUDA;
}
