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
//   * taps are evaluated in registers, 32 visibilities at a time (lane r evaluates the 2 S taps of record r
//     -- Gaussian: ex2.approx; Kaiser-Bessel: the power series of I0 by Horner's rule, all 2 S
//     taps side by side -- and parks them in shared memory), then lane (a, b) of the warp applies tap (a, b) of
//     one record after the other;
//   * a bin with more than WS_CHUNK records ("heavy": the dense core of the uv plane) is cut
//     into chunks that become work items of their own; k_prepare_heavy queues them and clears their tiles,
//     and the chunks are added with vector red.global.add.f32x2.  Tiles and items are interleaved in ONE
//     persistent kernel so that the store stream of the (mostly empty) tiles overlaps the arithmetic of the
//     dense ones.
#include "ws_internal.h"
#include "ws_taps.cuh"

namespace {

constexpr int T = WS_TILE;

template <int S>
struct TileCfg {
    static constexpr int H = (S - 1) / 2;
    static constexpr int P = T + S;                 // row pitch in complex cells: P = S mod 16 -> conflict-free taps
    static constexpr int R = 32 / S;                // footprint rows a warp covers per round
    static constexpr int NR = (S + R - 1) / R;      // rounds per visibility
    static constexpr int TILE_CELLS = T * P;
    // per warp: tile | meta[32] float4 | gu[32][S] | gv[32][S]
    static constexpr size_t WARP_BYTES =
        ((size_t)TILE_CELLS * sizeof(float2) + 32 * sizeof(float4) + 2 * 32 * S * sizeof(float) + 15) / 16 * 16;
    static constexpr int WARPS = (113 * 1024) / WARP_BYTES >= 8 ? 8 : (int)((113 * 1024) / WARP_BYTES);
    static constexpr int THREADS = WARPS * 32;
};

// storage origin (FFT-native order, wstack.h) of tile `bin`: returns the pointer to its first cell.  tr: the planes
// are stored transposed ([k][u][v], the private layout a WS_GRID_SPARSE mesh may take): cell (y, x) of the tile is
// then at origin + x N + y.
__device__ __forceinline__ float2* tile_origin(const WsGeom& g, float2* grid, uint32_t bin, bool tr) {
    const uint32_t nt = (uint32_t)g.nt;
    const uint32_t tx = bin % nt, r = bin / nt;
    const uint32_t ty = r % nt, k = r / nt;
    const uint32_t N = (uint32_t)g.n_pix, half = N >> 1;
    uint32_t sx = tx * T + half, sy = ty * T + half;
    sx = sx >= N ? sx - N : sx;
    sy = sy >= N ? sy - N : sy;
    return tr ? grid + ((size_t)k * N + sx) * N + sy : grid + ((size_t)k * N + sy) * N + sx;
}

// 32 rows x 256 B of zeros: 16 lanes x 16 B per row, two rows per store instruction
__device__ __forceinline__ void store_zero_tile(float2* out, size_t N, int lane) {
    float4* o4 = (float4*)(out + (size_t)(lane >> 4) * N) + (lane & 15);
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int y = 0; y < T; y += 2) __stcs(o4 + (size_t)y * (N / 2), z);
}

template <int S>
struct WarpSmem {
    float2* tile;
    float4* meta;
    float* gu;
    float* gv;
    __device__ __forceinline__ WarpSmem(unsigned char* base) {
        using C = TileCfg<S>;
        tile = (float2*)base;
        meta = (float4*)(tile + C::TILE_CELLS);
        gu = (float*)(meta + 32);
        gv = gu + 32 * S;
    }
};

// Accumulates records [lo, hi) into the warp's shared tile.
template <int S, bool KB>
__device__ __forceinline__ void accumulate(const WsGeom& g, const float4* __restrict__ records, uint32_t lo, uint32_t hi,
                                           const WarpSmem<S>& sm, int lane) {
    using C = TileCfg<S>;
    const int a = lane % S, br = lane / S;
    const bool active = br < C::R;
    const int lane_idx = br * C::P + a;            // tap (a, br) relative to the footprint's first cell
    float4 nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    if (lo + lane < hi) nxt = __ldcs(records + lo + lane);
    for (uint32_t base = lo; base < hi; base += 32) {
        const int n = (int)min(32u, hi - base);
        {   // vector phase: lane r prepares record r of the batch
            const uint32_t X = __float_as_uint(nxt.x), Y = __float_as_uint(nxt.y);
            const int cxp = ((int)X >> 24) - C::H, cyp = ((int)Y >> 24) - C::H;   // footprint's first cell, tile frame
            const float fx = (float)(X & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            const float fy = (float)(Y & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            if constexpr (!KB) {
                const float tap_c = g.tap_c;
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    const float dx = (float)(i - C::H) - fx, dy = (float)(i - C::H) - fy;
                    sm.gu[lane * S + i] = ex2_approx(tap_c * dx * dx);
                    sm.gv[lane * S + i] = ex2_approx(tap_c * dy * dy);
                }
            } else {
                float gu[S], gv[S];
                eval_taps<S, true>(g, fx, fy, gu, gv);
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    sm.gu[lane * S + i] = gu[i];
                    sm.gv[lane * S + i] = gv[i];
                }
            }
            sm.meta[lane] = make_float4(nxt.z, nxt.w, __int_as_float((cxp & 0xFFFF) | (cyp << 16)),
                                        __int_as_float(cyp * C::P + cxp));
        }
        if (base + 32 + lane < hi) nxt = __ldcs(records + base + 32 + lane);   // prefetch the next batch
        __syncwarp();
        for (int r = 0; r < n; ++r) {
            const float4 m = sm.meta[r];                       // broadcast
            const float u = sm.gu[r * S + a];
            const int xy = __float_as_int(m.z);
            const int cxp = (int)(short)(xy & 0xFFFF), cyp = xy >> 16;
            const bool okx = active && (unsigned)(cxp + a) < (unsigned)T;
            const int idx0 = __float_as_int(m.w) + lane_idx;
            float2 cell[C::NR];
            float t[C::NR];
            bool ok[C::NR];
#pragma unroll
            for (int rr = 0; rr < C::NR; ++rr) {
                const int b = br + rr * C::R;
                ok[rr] = okx && b < S && (unsigned)(cyp + b) < (unsigned)T;
                t[rr] = u * sm.gv[r * S + (b < S ? b : 0)];
                if (ok[rr]) cell[rr] = sm.tile[idx0 + rr * C::R * C::P];
            }
#pragma unroll
            for (int rr = 0; rr < C::NR; ++rr) {
                if (ok[rr]) {
                    cell[rr].x = fmaf(m.x, t[rr], cell[rr].x);
                    cell[rr].y = fmaf(m.y, t[rr], cell[rr].y);
                    sm.tile[idx0 + rr * C::R * C::P] = cell[rr];
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

// Queues the chunks of the heavy bins as work items and (OVERWRITE mode) clears their tiles.
__global__ void __launch_bounds__(256)
k_prepare_heavy(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ rec_start, uint4* __restrict__ items,
                uint32_t item_capacity, WsStatus* __restrict__ status, float2* __restrict__ grid, int mode,
                const uint32_t* __restrict__ orient, const WsMaskView mv) {
    if (status->overflow) return;
    const bool tr = orient && *orient;
    const uint32_t b = blockIdx.x * 256u + threadIdx.x;
    const int lane = threadIdx.x & 31;
    uint32_t s = 0, cnt = 0;
    if (b < g.n_bins) {
        s = rec_start[b];
        cnt = rec_start[b + 1] - s;
    }
    const bool heavy = cnt > WS_CHUNK;
    const uint32_t chunks = heavy ? (cnt + WS_CHUNK - 1) / WS_CHUNK : 0u;
    const unsigned hm = __ballot_sync(0xffffffffu, heavy);
    if (!hm) return;
    uint32_t inc = chunks;                       // inclusive warp scan of the chunk counts
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
    uint32_t base = 0;
    if (lane == 0) base = atomicAdd(&status->n_items, total);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base + total > item_capacity) {
        if (lane == 0) status->overflow = status->sticky_overflow = 1u;
        return;
    }
    if (heavy) {
        uint32_t o = base + inc - chunks;
        for (uint32_t lo = s; lo < s + cnt; lo += WS_CHUNK) items[o++] = make_uint4(b, lo, min(lo + WS_CHUNK, s + cnt), 0u);
    }
    if (mode != WS_GRID_ACCUMULATE) {
        for (unsigned m = hm; m; m &= m - 1) {
            const uint32_t hb = (b - lane) + (__ffs(m) - 1);
            if (mode == WS_GRID_SPARSE_ADD) {                   // a tile earlier chunks filled is added to, not cleared
                const uint32_t nt = (uint32_t)g.nt, tx = hb % nt, r = hb / nt;
                if (ws_tile_occupied(mv, g.nt, r / nt, r % nt, tx)) continue;
            }
            store_zero_tile(tile_origin(g, grid, hb, tr), (size_t)g.n_pix, lane);
        }
    }
}

// Persistent kernel: warp w takes tiles w, w + W, ... and items w, w + W, ..., interleaved.
template <int S, bool KB>
__global__ void __launch_bounds__(TileCfg<S>::THREADS, 2)
k_grid(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ rec_start, const uint4* __restrict__ items,
       const float4* __restrict__ records, float2* __restrict__ grid, int mode, const WsStatus* __restrict__ status,
       const uint32_t* __restrict__ orient, const WsMaskView mv) {
    using C = TileCfg<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const WarpSmem<S> sm(smem_raw + (size_t)wid * C::WARP_BYTES);
    if (status->overflow) return;
    const bool tr = orient && *orient;          // transposed planes: lane = row of the tile, one tile column per store
    const uint32_t n_items = status->n_items;
    const uint32_t n_warps = gridDim.x * C::WARPS;
    const uint32_t gw = blockIdx.x * C::WARPS + wid;
    const size_t N = (size_t)g.n_pix;
    const uint32_t my_tiles = gw < g.n_bins ? (g.n_bins - gw + n_warps - 1) / n_warps : 0u;
    const uint32_t my_items = gw < n_items ? (n_items - gw + n_warps - 1) / n_warps : 0u;
    const uint32_t gap = my_items ? max(1u, my_tiles / my_items) : 0xFFFFFFFFu;
    uint32_t it = gw, since = 0;

    auto do_item = [&]() {
        const uint4 w = items[it];
        it += n_warps;
        float2* out = tile_origin(g, grid, w.x, tr);
        zero_tile<S>(sm.tile, lane);
        accumulate<S, KB>(g, records, w.y, w.z, sm, lane);
#pragma unroll 4
        for (int y = 0; y < T; ++y) {
            const float2 v = tr ? sm.tile[lane * C::P + y] : sm.tile[y * C::P + lane];
            if (v.x != 0.f || v.y != 0.f) atomicAdd(out + (size_t)y * N + lane, v);   // RED.E.ADD.F32x2
        }
        __syncwarp();
    };

    for (uint32_t bin = gw; bin < g.n_bins; bin += n_warps) {
        if (it < n_items && since >= gap) {
            do_item();
            since = 0;
        }
        ++since;
        const uint32_t s = rec_start[bin], e = rec_start[bin + 1];
        if (e - s > WS_CHUNK) continue;                     // heavy: its chunks are items
        float2* out = tile_origin(g, grid, bin, tr);
        if (s == e) {
            if (mode == WS_GRID_OVERWRITE) store_zero_tile(out, N, lane);
            continue;
        }
        zero_tile<S>(sm.tile, lane);
        accumulate<S, KB>(g, records, s, e, sm, lane);
        bool add = mode == WS_GRID_ACCUMULATE;
        if (mode == WS_GRID_SPARSE_ADD) {                       // warp-uniform: did an earlier chunk fill this tile?
            const uint32_t nt = (uint32_t)g.nt, tx = bin % nt, r = bin / nt;
            add = ws_tile_occupied(mv, g.nt, r / nt, r % nt, tx);
        }
        if (!add) {
#pragma unroll 4
            for (int y = 0; y < T; ++y) __stcs(out + (size_t)y * N + lane, tr ? sm.tile[lane * C::P + y] : sm.tile[y * C::P + lane]);
        } else {        // no other warp writes this tile in this launch except through red: fire-and-forget vector adds
#pragma unroll 4
            for (int y = 0; y < T; ++y) {
                const float2 v = tr ? sm.tile[lane * C::P + y] : sm.tile[y * C::P + lane];
                if (v.x != 0.f || v.y != 0.f) atomicAdd(out + (size_t)y * N + lane, v);   // RED.E.ADD.F32x2
            }
        }
        __syncwarp();
    }
    while (it < n_items) do_item();
}

template <int S, bool KB>
int launch_s(ws_plan* plan, const WsLayout& L, char* ws, float2* grid, int mode, cudaStream_t st) {
    const uint32_t* orient = (mode == WS_GRID_SPARSE || mode == WS_GRID_SPARSE_ADD) ? ws_fft_orientation_flag(plan) : nullptr;
    const WsMaskView mv = ws_fft_mask_view(plan);
    if (mode == WS_GRID_SPARSE_ADD && !mv.masks) return WS_ERR_UNSUPPORTED;
    using C = TileCfg<S>;
    const size_t smem = C::WARP_BYTES * C::WARPS;
    // per device, and cheap: set on every launch rather than cached in a process-wide flag
    if (cudaFuncSetAttribute(k_grid<S, KB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return WS_ERR_CUDA;
    const uint32_t* rec_start = (const uint32_t*)(ws + L.off_rec_start);
    const float4* records = (const float4*)(ws + L.off_records);
    WsStatus* status = plan->d_status;
    uint4* items = (uint4*)(ws + L.off_items);
    const WsGeom& g = plan->geom;
    if (cudaMemsetAsync(&status->n_items, 0, sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;
    k_prepare_heavy<<<(g.n_bins + 255) / 256, 256, 0, st>>>(g, rec_start, items, L.item_capacity, status, grid, mode, orient, mv);
    k_grid<S, KB><<<plan->sm_count * 2, C::THREADS, smem, st>>>(g, rec_start, items, records, grid, mode, status, orient, mv);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 2;
}

}  // namespace

// Work items for the lists of `starts` ([n_bins + 1] offsets) longer than WS_CHUNK: used by the degridder on the home lists.
int ws_launch_items(ws_plan* plan, const uint32_t* starts, uint4* items, uint32_t item_capacity, cudaStream_t st) {
    const WsGeom& g = plan->geom;
    if (cudaMemsetAsync(&plan->d_status->n_items, 0, sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;
    k_prepare_heavy<<<(g.n_bins + 255) / 256, 256, 0, st>>>(g, starts, items, item_capacity, plan->d_status, nullptr,
                                                          WS_GRID_ACCUMULATE, nullptr, WsMaskView{nullptr, 0u, 1});
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_grid(ws_plan* plan, const WsLayout& L, char* ws, float2* grid, int mode, cudaStream_t st) {
    const bool kb = plan->geom.kb_terms > 0;
    switch (plan->geom.support) {
        case 1: return kb ? launch_s<1, true>(plan, L, ws, grid, mode, st) : launch_s<1, false>(plan, L, ws, grid, mode, st);
        case 3: return kb ? launch_s<3, true>(plan, L, ws, grid, mode, st) : launch_s<3, false>(plan, L, ws, grid, mode, st);
        case 5: return kb ? launch_s<5, true>(plan, L, ws, grid, mode, st) : launch_s<5, false>(plan, L, ws, grid, mode, st);
        case 7: return kb ? launch_s<7, true>(plan, L, ws, grid, mode, st) : launch_s<7, false>(plan, L, ws, grid, mode, st);
        case 9: return kb ? launch_s<9, true>(plan, L, ws, grid, mode, st) : launch_s<9, false>(plan, L, ws, grid, mode, st);
        case 11: return kb ? launch_s<11, true>(plan, L, ws, grid, mode, st) : launch_s<11, false>(plan, L, ws, grid, mode, st);
        case 13: return kb ? launch_s<13, true>(plan, L, ws, grid, mode, st) : launch_s<13, false>(plan, L, ws, grid, mode, st);
        case 15: return kb ? launch_s<15, true>(plan, L, ws, grid, mode, st) : launch_s<15, false>(plan, L, ws, grid, mode, st);
    }
    return WS_ERR_UNSUPPORTED;
}
