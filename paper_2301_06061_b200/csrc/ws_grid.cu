// a2: convolutional gridding, Eq. 3:  V~(u_i, v_j, w_k) = sum_m V_m G(u_i - u_m, v_j - v_m),
// Gaussian G of S x S cells, weights per measurement (:74).
//
// The paper's GPU kernel gives one thread per measurement and resolves collisions with atomicAdd on the fp64
// mesh in global memory, and names the accumulation as "the main potential bottleneck"
// (:191).  Here the bins of ws_bin.cu make the mesh output-stationary instead:
//   * one WARP owns one 32 x 32 tile of one w-plane, accumulates it in its private shared-memory tile with
//     plain LDS / FFMA / STS (the lanes of a warp cover distinct taps of one visibility, so there are no
//     collisions and no atomics), and writes it ONCE with coalesced stores -- in WS_GRID_OVERWRITE mode the
//     tile (zeros included) is simply stored, so the mesh needs no memset and no read-modify-write;
//   * taps are evaluated in registers: lane (a, b) computes g(a - fu) and g(b - fv) itself (ex2.approx);
//   * bins with more than WS_CHUNK records are cut into chunks; chunk 0 is handled as above, the others are
//     work items of k_grid_items, which adds its tile with vector red.global.add.f32x2.
#include "ws_internal.h"

namespace {

constexpr int T = WS_TILE;
constexpr int GRID_WARPS = 8;                 // warps per CTA
constexpr int GRID_THREADS = GRID_WARPS * 32;

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int S>
struct TileCfg {
    static constexpr int H = (S - 1) / 2;
    static constexpr int P = T + S;                 // row pitch in complex cells: P = S mod 16 -> conflict-free taps
    static constexpr int R = 32 / S;                // footprint rows a warp covers per round
    static constexpr int NR = (S + R - 1) / R;      // rounds per visibility
    static constexpr int TILE_CELLS = T * P;
    static constexpr size_t WARP_BYTES = (size_t)TILE_CELLS * sizeof(float2) + 32 * sizeof(float4);
};

// storage origin (FFT-native order, wstack.h) of tile `bin`: returns the pointer to its first cell
__device__ __forceinline__ float2* tile_origin(const WsGeom& g, float2* grid, uint32_t bin) {
    const uint32_t nt = (uint32_t)g.nt;
    const uint32_t tx = bin % nt, r = bin / nt;
    const uint32_t ty = r % nt, k = r / nt;
    const uint32_t N = (uint32_t)g.n_pix, half = N >> 1;
    uint32_t sx = tx * T + half, sy = ty * T + half;
    sx = sx >= N ? sx - N : sx;
    sy = sy >= N ? sy - N : sy;
    return grid + ((size_t)k * N + sy) * N + sx;
}

// Accumulates records [lo, hi) into the warp's shared tile.
template <int S>
__device__ __forceinline__ void accumulate(const WsGeom& g, const float4* __restrict__ records, uint32_t lo, uint32_t hi,
                                           float2* tile, float4* stage, int lane) {
    using C = TileCfg<S>;
    const int a = lane % S, br = lane / S;
    const bool active = br < C::R;
    const float da = (float)(a - C::H);
    const float tap_c = g.tap_c;
    float4 nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    if (lo + lane < hi) nxt = __ldcs(records + lo + lane);
    for (uint32_t base = lo; base < hi; base += 32) {
        const int n = (int)min(32u, hi - base);
        stage[lane] = nxt;
        if (base + 32 + lane < hi) nxt = __ldcs(records + base + 32 + lane);   // prefetch the next batch
        __syncwarp();
        for (int r = 0; r < n; ++r) {
            const float4 q = stage[r];                       // broadcast
            const uint32_t X = __float_as_uint(q.x), Y = __float_as_uint(q.y);
            const int cx = (int)X >> 24, cy = (int)Y >> 24;  // centre cell relative to the tile origin
            const float fx = (float)(X & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            const float fy = (float)(Y & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            const int x = cx - C::H + a;
            const float dx = da - fx;
            const float gu = ex2_approx(tap_c * dx * dx);
            const bool okx = active && (unsigned)x < (unsigned)T;
            float2 cell[C::NR];
            float t[C::NR];
            bool ok[C::NR];
            int idx[C::NR];
#pragma unroll
            for (int rr = 0; rr < C::NR; ++rr) {
                const int b = br + rr * C::R;
                const int y = cy - C::H + b;
                const float dy = (float)(b - C::H) - fy;
                t[rr] = gu * ex2_approx(tap_c * dy * dy);
                ok[rr] = okx && b < S && (unsigned)y < (unsigned)T;
                idx[rr] = y * C::P + x;
                if (ok[rr]) cell[rr] = tile[idx[rr]];
            }
#pragma unroll
            for (int rr = 0; rr < C::NR; ++rr) {
                if (ok[rr]) {
                    cell[rr].x = fmaf(q.z, t[rr], cell[rr].x);
                    cell[rr].y = fmaf(q.w, t[rr], cell[rr].y);
                    tile[idx[rr]] = cell[rr];
                }
            }
            __syncwarp();
        }
    }
}

template <int S>
__device__ __forceinline__ void zero_tile(float2* tile, int lane) {
    using C = TileCfg<S>;
    for (int i = lane; i < C::TILE_CELLS; i += 32) tile[i] = make_float2(0.f, 0.f);
    __syncwarp();
}

// One warp per tile-plane, tiles strided over all warps of the (persistent) grid.
template <int S>
__global__ void __launch_bounds__(GRID_THREADS, 2)
k_grid_tiles(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ rec_start,
             const float4* __restrict__ records, float2* __restrict__ grid, int mode,
             const WsStatus* __restrict__ status) {
    using C = TileCfg<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float4* stage = (float4*)(smem_raw + (size_t)wid * C::WARP_BYTES);
    float2* tile = (float2*)(stage + 32);
    if (status->overflow) return;
    const uint32_t n_warps = gridDim.x * GRID_WARPS;
    const size_t N = (size_t)g.n_pix;
    for (uint32_t bin = blockIdx.x * GRID_WARPS + wid; bin < g.n_bins; bin += n_warps) {
        const uint32_t s = rec_start[bin], e = rec_start[bin + 1];
        float2* out = tile_origin(g, grid, bin);
        if (s == e) {
            if (mode == WS_GRID_OVERWRITE) {
                // 32 rows x 256 B of zeros: 16 lanes x 16 B per row, two rows per store instruction
                float4* o4 = (float4*)(out + (size_t)(lane >> 4) * N) + (lane & 15);
                const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int y = 0; y < T; y += 2) __stcs(o4 + (size_t)y * (N / 2), z);
            }
            continue;
        }
        zero_tile<S>(tile, lane);
        accumulate<S>(g, records, s, min(e, s + (uint32_t)WS_CHUNK), tile, stage, lane);
        if (mode == WS_GRID_OVERWRITE) {
#pragma unroll 4
            for (int y = 0; y < T; ++y) __stcs(out + (size_t)y * N + lane, tile[y * C::P + lane]);
        } else {
#pragma unroll 4
            for (int y = 0; y < T; ++y) {
                float2 v = tile[y * C::P + lane];
                float2* p = out + (size_t)y * N + lane;
                const float2 old = *p;
                v.x += old.x;
                v.y += old.y;
                *p = v;
            }
        }
        __syncwarp();
    }
}

// Heavy bins: chunks 1.. of a bin, added onto the tile chunk 0 already stored (stream order).
template <int S>
__global__ void __launch_bounds__(GRID_THREADS, 2)
k_grid_items(const __grid_constant__ WsGeom g, const uint4* __restrict__ items, const float4* __restrict__ records,
             float2* __restrict__ grid, const WsStatus* __restrict__ status) {
    using C = TileCfg<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float4* stage = (float4*)(smem_raw + (size_t)wid * C::WARP_BYTES);
    float2* tile = (float2*)(stage + 32);
    if (status->overflow) return;
    const uint32_t n_items = status->n_items;
    const uint32_t n_warps = gridDim.x * GRID_WARPS;
    const size_t N = (size_t)g.n_pix;
    for (uint32_t it = blockIdx.x * GRID_WARPS + wid; it < n_items; it += n_warps) {
        const uint4 w = items[it];
        float2* out = tile_origin(g, grid, w.x);
        zero_tile<S>(tile, lane);
        accumulate<S>(g, records, w.y, w.z, tile, stage, lane);
#pragma unroll 4
        for (int y = 0; y < T; ++y) {
            const float2 v = tile[y * C::P + lane];
            if (v.x != 0.f || v.y != 0.f) atomicAdd(out + (size_t)y * N + lane, v);   // RED.E.ADD.F32x2
        }
        __syncwarp();
    }
}

template <int S>
int launch_s(ws_plan* plan, const WsLayout& L, char* ws, float2* grid, int mode, cudaStream_t st) {
    using C = TileCfg<S>;
    const size_t smem = C::WARP_BYTES * GRID_WARPS;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_grid_tiles<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaFuncSetAttribute(k_grid_items<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return WS_ERR_CUDA;
        attr_set = true;
    }
    const uint32_t* rec_start = (const uint32_t*)(ws + L.off_counts_all);
    const float4* records = (const float4*)(ws + L.off_records);
    const WsStatus* status = plan->d_status;
    const uint4* items = (const uint4*)(ws + L.off_items);
    const int ctas = plan->sm_count * 2;
    k_grid_tiles<S><<<ctas, GRID_THREADS, smem, st>>>(plan->geom, rec_start, records, grid, mode, status);
    k_grid_items<S><<<ctas, GRID_THREADS, smem, st>>>(plan->geom, items, records, grid, status);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 2;
}

}  // namespace

int ws_launch_grid(ws_plan* plan, const WsLayout& L, char* ws, float2* grid, int mode, cudaStream_t st) {
    switch (plan->geom.support) {
        case 1: return launch_s<1>(plan, L, ws, grid, mode, st);
        case 3: return launch_s<3>(plan, L, ws, grid, mode, st);
        case 5: return launch_s<5>(plan, L, ws, grid, mode, st);
        case 7: return launch_s<7>(plan, L, ws, grid, mode, st);
        case 9: return launch_s<9>(plan, L, ws, grid, mode, st);
        case 11: return launch_s<11>(plan, L, ws, grid, mode, st);
        case 13: return launch_s<13>(plan, L, ws, grid, mode, st);
        case 15: return launch_s<15>(plan, L, ws, grid, mode, st);
    }
    return WS_ERR_UNSUPPORTED;
}
