// a2: convolutional gridding, Eq. 3:  V~(u_i, v_j, w_k) = sum_m V_m G(u_i - u_m, v_j - v_m),
// Gaussian G of S x S cells, weights per measurement (:74).
//
// The paper's GPU kernel gives one thread per measurement and resolves collisions with atomicAdd on the fp64
// mesh in global memory, and names the accumulation as "the main potential bottleneck"
// (:191).  Here the bins of ws_bin.cu make the mesh output-stationary instead:
//   * one WARP owns one 32 x 32 tile of one w-plane and accumulates the records of the visibilities whose centre
//     cell lies in it in a private shared-memory buffer -- the tile plus a ring of (S-1)/2 cells, so that no
//     footprint leaves the buffer -- with plain LDS / FFMA / STS (the lanes of a warp cover distinct taps of one
//     visibility: no collisions, no atomics, no bounds tests);
//   * taps are evaluated in registers, 32 visibilities at a time (lane r evaluates the 2 S taps of record r
//     -- Gaussian: ex2.approx; Kaiser-Bessel: the power series of I0 by Horner's rule, all 2 S
//     taps side by side -- and parks them in shared memory), then lane (a, b) of the warp applies tap (a, b) of
//     one record after the other;
//   * the buffer is then ADDED to the mesh once, tile and ring alike (red.global.add.v2.f32, skipping zeros): the
//     ring is what this tile's visibilities put onto the neighbours' cells, and it is the only place where two
//     writers can meet ("atomics only at tile borders").  The tiles that receive anything -- from their own
//     records or from a neighbour's ring: the halo histogram of ws_bin.cu knows -- are cleared first by
//     k_prepare_heavy (WS_GRID_SPARSE_ADD: unless an earlier chunk filled them; WS_GRID_ACCUMULATE: never);
//     WS_GRID_OVERWRITE also stores the zeros of the tiles that receive nothing, from inside the persistent kernel,
//     so that their store stream overlaps the arithmetic of the dense tiles.  (Round 1 copied a record into every
//     tile its footprint reaches and let one owner store each tile: 1.41 records per visibility on Large, 1.56
//     with S = 9.)
//   * a bin with more than WS_CHUNK records ("heavy": the dense core of the uv plane) is cut
//     into chunks that become work items of their own (k_prepare_heavy); ONE persistent kernel takes the chunks and
//     then the other non-empty bins (a list k_prepare_heavy writes) from one work counter.
#include "ws_internal.h"
#include "ws_taps.cuh"

namespace {

constexpr int T = WS_TILE;

constexpr int pow2_ceil(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// The warp's shared buffer covers the 32 x 32 cells of its tile PLUS a ring of H cells: the footprint of a record whose
// centre lies inside the tile never leaves the buffer, so the inner loop needs no bounds test.  What lands in the ring
// belongs to the neighbour tiles and reaches them when the whole buffer is added to the mesh (flush_ring).
template <int S>
struct TileCfg {
    static constexpr int H = (S - 1) / 2;
    static constexpr int P = T + S;                 // row pitch in complex cells: P = S mod 16 -> conflict-free taps
    static constexpr int ROWS = T + S - 1;          // rows (and used columns) of the buffer: tile + ring
    static constexpr int R = 32 / S < S ? 32 / S : S;   // footprint rows a warp covers per round
    static constexpr int NR = (S + R - 1) / R;      // rounds per visibility
    static constexpr int NRP = pow2_ceil(NR);       // taps of one lane along v, padded: one vector load
    static constexpr int SP = S;                    // pitch of the u taps of a record (odd: lane r's scalar stores are conflict-free)
    static constexpr int GP = NRP * (R | 1);        // pitch of its v taps, [R][NRP] + padding: an odd number of NRP-vectors, so
                                                    // that the lanes' vector stores of one br fall into distinct banks
    static constexpr int TILE_CELLS = (ROWS - 1) * P + ROWS;   // (the last row needs no padding)
    static constexpr int GU_FLOATS = (32 * SP + 3) / 4 * 4;    // (keeps gv 16-byte aligned)
    static constexpr int GV_FLOATS = (31 * GP + R * NRP + 1) / 2 * 2;   // (the last record needs no padding; keeps the tile 8-byte aligned)
    // per warp: meta[32] float4 | gu[32][SP] | gv[32][GP] | tile.  Sized to the byte: S = 7 comes to 14528 bytes, and sixteen of
    // those are exactly the 227 KB a CTA may have
    static constexpr size_t WARP_BYTES =
        (32 * sizeof(float4) + (size_t)(GU_FLOATS + GV_FLOATS) * sizeof(float) + (size_t)TILE_CELLS * sizeof(float2) + 15) / 16 * 16;
    // one CTA per SM with as many (independent) warps as the 227 KB of shared memory hold, at most 16
    static constexpr int WARPS = (227 * 1024) / WARP_BYTES >= 16 ? 16 : (int)((227 * 1024) / WARP_BYTES);
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
        meta = (float4*)base;
        gu = (float*)(meta + 32);
        gv = gu + C::GU_FLOATS;
        tile = (float2*)(gv + C::GV_FLOATS);
    }
};

template <int N>
struct TapVec { float v[N]; };
template <int N>
__device__ __forceinline__ void store_taps(float* p, const TapVec<N>& t) {
    if constexpr (N == 1) p[0] = t.v[0];
    else if constexpr (N == 2) *(float2*)p = make_float2(t.v[0], t.v[1]);
    else {
#pragma unroll
        for (int i = 0; i < N; i += 4) *(float4*)(p + i) = make_float4(t.v[i], t.v[i + 1], t.v[i + 2], t.v[i + 3]);
    }
}
template <int N>
__device__ __forceinline__ TapVec<N> load_taps(const float* p) {
    TapVec<N> t;
    if constexpr (N == 1) t.v[0] = p[0];
    else if constexpr (N == 2) { const float2 q = *(const float2*)p; t.v[0] = q.x; t.v[1] = q.y; }
    else {
#pragma unroll
        for (int i = 0; i < N; i += 4) {
            const float4 q = *(const float4*)(p + i);
            t.v[i] = q.x; t.v[i + 1] = q.y; t.v[i + 2] = q.z; t.v[i + 3] = q.w;
        }
    }
    return t;
}

// vector phase of a batch: the 2 S taps of lane r's record, parked where the lanes (a, br) find them.  The Kaiser-Bessel
// series is kept out of line: inlined, its register demand makes the compiler turn the predicated read-modify-writes of the
// record loop into divergent branches (measured: 15.3 ms against 10.9 on Large).
template <int S>
__device__ __forceinline__ void park_store(const float* gu, const float* gv, const WarpSmem<S>& sm, int lane) {
    using C = TileCfg<S>;
#pragma unroll
    for (int i = 0; i < S; ++i) sm.gu[lane * C::SP + i] = gu[i];
#pragma unroll
    for (int b0 = 0; b0 < C::R; ++b0) {                 // the taps lane (., b0) applies in its rounds, as one vector
        TapVec<C::NRP> tv;
#pragma unroll
        for (int rr = 0; rr < C::NRP; ++rr) tv.v[rr] = b0 + rr * C::R < S ? gv[b0 + rr * C::R < S ? b0 + rr * C::R : 0] : 0.f;
        store_taps<C::NRP>(sm.gv + lane * C::GP + b0 * C::NRP, tv);
    }
}
template <int S>
__device__ __noinline__ void park_taps_kb(const WsGeom& g, float fx, float fy, float* gu_s, float* gv_s, int lane) {
    float gu[S], gv[S];
    eval_taps<S, true>(g, fx, fy, gu, gv);
    WarpSmem<S> sm(nullptr);
    sm.gu = gu_s;
    sm.gv = gv_s;
    park_store<S>(gu, gv, sm, lane);
}
template <int S, bool KB>
__device__ __forceinline__ void park_taps(const WsGeom& g, float fx, float fy, const WarpSmem<S>& sm, int lane) {
    if constexpr (KB) {
        park_taps_kb<S>(g, fx, fy, sm.gu, sm.gv, lane);
    } else {
        using C = TileCfg<S>;
        float gu[S], gv[S];
        const float tap_c = g.tap_c;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const float dx = (float)(i - C::H) - fx, dy = (float)(i - C::H) - fy;
            gu[i] = ex2_approx(tap_c * dx * dx);
            gv[i] = ex2_approx(tap_c * dy * dy);
        }
        park_store<S>(gu, gv, sm, lane);
    }
}

// One record of the batch onto the buffer: lane (a, br) applies its taps.  The record's centre cell lies inside the tile,
// so its footprint stays inside the buffer (tile + ring): no bounds tests.
template <int S>
__device__ __forceinline__ void apply_record(const WarpSmem<S>& sm, int r, const bool* okb, unsigned char* tile_b,
                                             const float* gu_l, const float* gv_l) {
    using C = TileCfg<S>;
    const float4 m = sm.meta[r];                       // broadcast
    const float u = gu_l[r * C::SP];
    const TapVec<C::NRP> gvv = load_taps<C::NRP>(gv_l + r * C::GP);
    float2* const cell0 = (float2*)(tile_b + __float_as_int(m.z));
#pragma unroll
    for (int rr = 0; rr < C::NR; ++rr) {
        if (okb[rr]) {                                  // (distinct cells per round: the loads of all rounds can go first)
            float2 c = cell0[rr * C::R * C::P];
            const float t = u * gvv.v[rr];
            c.x = fmaf(m.x, t, c.x);
            c.y = fmaf(m.y, t, c.y);
            cell0[rr * C::R * C::P] = c;
        }
    }
    __syncwarp();
}

// Accumulates records [lo, hi) (all of one tile) into the warp's shared buffer.
template <int S, bool KB>
__device__ __forceinline__ void accumulate_records(const WsGeom& g, const float4* __restrict__ records, uint32_t lo, uint32_t hi,
                                                   const WarpSmem<S>& sm, int lane) {
    using C = TileCfg<S>;
    const int a = lane % S, br = lane / S;
    const bool active = br < C::R;
    bool okb[C::NR];                               // lane constants: this lane has a tap in round rr
#pragma unroll
    for (int rr = 0; rr < C::NR; ++rr) okb[rr] = active && br + rr * C::R < S;
    unsigned char* const tile_b = (unsigned char*)sm.tile + (size_t)((active ? br : 0) * C::P + a) * sizeof(float2);
    const float* const gu_l = sm.gu + a;
    const float* const gv_l = sm.gv + (active ? br : 0) * C::NRP;
    float4 nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    if (lo + lane < hi) nxt = __ldcs(records + lo + lane);
    for (uint32_t base = lo; base < hi; base += 32) {
        const int n = (int)min(32u, hi - base);
        {   // vector phase: lane r prepares record r of the batch
            const uint32_t X = __float_as_uint(nxt.x), Y = __float_as_uint(nxt.y);
            const int cx = (int)(X >> 24), cy = (int)(Y >> 24);   // centre cell in the tile's frame = first footprint cell in the buffer's
            const float fx = (float)(X & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            const float fy = (float)(Y & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
            park_taps<S, KB>(g, fx, fy, sm, lane);
            sm.meta[lane] = make_float4(nxt.z, nxt.w, __int_as_float((cy * C::P + cx) * (int)sizeof(float2)), 0.f);
        }
        if (base + 32 + lane < hi) nxt = __ldcs(records + base + 32 + lane);   // prefetch the next batch
        __syncwarp();
        for (int r = 0; r < n; ++r) apply_record<S>(sm, r, okb, tile_b, gu_l, gv_l);
    }
}

template <int S>
__device__ __forceinline__ void zero_tile(float2* tile, int lane) {
    using C = TileCfg<S>;
    for (int i = lane; i < C::TILE_CELLS; i += 32) tile[i] = make_float2(0.f, 0.f);
    __syncwarp();
}

// Queues the chunks of the heavy bins (more than WS_CHUNK records) as work items and, for the gridder (clear_occupied),
// clears every tile that will be ADDED to: every tile that receives anything at all -- its own records or a neighbour's
// ring (occ_start: home + halo counts).  starts: offsets of the record lists ([n_bins + 1]).  In WS_GRID_SPARSE_ADD mode
// a tile that earlier chunks filled is left alone; WS_GRID_ACCUMULATE clears nothing.
__global__ void __launch_bounds__(256)
k_prepare_heavy(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ starts, const uint32_t* __restrict__ occ_start,
                int clear_occupied, uint32_t* __restrict__ light, uint4* __restrict__ items, uint32_t item_capacity,
                WsStatus* __restrict__ status,
                float2* __restrict__ grid, int mode, const uint32_t* __restrict__ orient, const WsMaskView mv) {
    if (status->overflow) return;
    const bool tr = orient && *orient;
    const uint32_t b = blockIdx.x * 256u + threadIdx.x;
    const int lane = threadIdx.x & 31;
    uint32_t s = 0, cnt = 0, occ = 0;
    if (b < g.n_bins) {
        s = starts[b];
        cnt = starts[b + 1] - s;
        occ = clear_occupied ? occ_start[b + 1] - occ_start[b] : 0u;
    }
    const bool heavy = cnt > WS_CHUNK;
    const uint32_t chunks = heavy ? (cnt + WS_CHUNK - 1) / WS_CHUNK : 0u;
    const unsigned hm = __ballot_sync(0xffffffffu, heavy);
    bool clear = mode != WS_GRID_ACCUMULATE && occ > 0;
    if (clear && mode == WS_GRID_SPARSE_ADD) {              // a tile earlier chunks filled is added to, not cleared
        const uint32_t nt = (uint32_t)g.nt, tx = b % nt, r = b / nt;
        clear = !ws_tile_occupied(mv, g.nt, r / nt, r % nt, tx);
    }
    for (unsigned m = __ballot_sync(0xffffffffu, clear); m; m &= m - 1) {
        const uint32_t hb = (b - lane) + (__ffs(m) - 1);
        store_zero_tile(tile_origin(g, grid, hb, tr), (size_t)g.n_pix, lane);
    }
    if (light) {                                 // the bins the gridder takes whole, as a list: it need not walk the empty ones
        const unsigned lm = __ballot_sync(0xffffffffu, cnt > 0 && !heavy);
        if (lm) {
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(&status->n_light, (uint32_t)__popc(lm));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (cnt > 0 && !heavy) light[base + __popc(lm & ((1u << lane) - 1u))] = b;
        }
    }
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
}

// Ring scheme: adds the whole shared buffer -- the 32 x 32 tile AND its ring, which holds what this tile's records put onto
// the neighbours' cells -- to the mesh with red.global.add.v2.f32 (PAPER.md:191 names the accumulation as the bottleneck;
// here the atomics are confined to this one flush per tile, and only the ring's share of it ever meets another writer).
// Every target tile was cleared (or filled by an earlier chunk) before this kernel started.  Cells off the mesh cannot
// hold anything (drop rule) and are skipped, like zeros.
template <int S>
__device__ __forceinline__ void flush_ring(const WsGeom& g, const WarpSmem<S>& sm, float2* __restrict__ grid, uint32_t bin, bool tr,
                                           int lane) {
    using C = TileCfg<S>;
    const uint32_t nt = (uint32_t)g.nt, tx = bin % nt, r = bin / nt, ty = r % nt, k = r / nt;
    const int N = g.n_pix, half = N >> 1;
    const int gx0 = (int)tx * T - C::H, gy0 = (int)ty * T - C::H;     // logical cell of buffer cell (0, 0)
    float2* const plane = grid + (size_t)k * N * N;
    // lanes run along the storage line: x (rows of the plane are v) or, transposed, y
    const int l0 = tr ? gx0 : gy0, c0 = tr ? gy0 : gx0;               // logical coordinate of buffer line 0 / of lane 0's cell
    for (int line = 0; line < C::ROWS; ++line) {
        const int gl = l0 + line;
        if ((unsigned)gl >= (unsigned)N) continue;
        float2* const row = plane + (size_t)((gl + half) & (N - 1)) * N;
#pragma unroll
        for (int seg = 0; seg < C::ROWS; seg += 32) {
            const int i = seg + lane;
            if (i < C::ROWS) {
                const float2 v = tr ? sm.tile[i * C::P + line] : sm.tile[line * C::P + i];
                const int gc = c0 + i;
                if ((v.x != 0.f || v.y != 0.f) && (unsigned)gc < (unsigned)N) atomicAdd(row + ((gc + half) & (N - 1)), v);
            }
        }
    }
    __syncwarp();
}

// Persistent kernel, one CTA per SM of independent warps.  The warps take their work from one counter (WS_GRID_OVERWRITE: by
// a fixed stride over ALL bins, warp w takes tiles w, w + W, ... and items w, w + W, ..., interleaved -- it stores zeros too).
// bin_start: offsets of the record lists (one record per visibility, in its home bin); occ_start: home + halo counts,
// scanned -- a tile whose entry does not grow receives nothing, and WS_GRID_OVERWRITE stores its zeros here (every other
// tile was cleared by k_prepare_heavy, or holds what earlier calls put there, and is only ever added to).
template <int S, bool KB>
__global__ void __launch_bounds__(TileCfg<S>::THREADS, 1)
k_grid(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ occ_start,
       const uint32_t* __restrict__ light, const uint4* __restrict__ items, const float4* __restrict__ records,
       float2* __restrict__ grid, int mode, WsStatus* __restrict__ status, const uint32_t* __restrict__ orient) {
    using C = TileCfg<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const WarpSmem<S> sm(smem_raw + (size_t)wid * C::WARP_BYTES);
    if (status->overflow) return;
    const bool tr = orient && *orient;          // transposed planes: lanes run along v instead of u
    const uint32_t n_items = status->n_items;
    const uint32_t n_warps = gridDim.x * C::WARPS;
    const uint32_t gw = blockIdx.x * C::WARPS + wid;
    const uint32_t my_tiles = gw < g.n_bins ? (g.n_bins - gw + n_warps - 1) / n_warps : 0u;
    const uint32_t my_items = gw < n_items ? (n_items - gw + n_warps - 1) / n_warps : 0u;
    const uint32_t gap = my_items ? max(1u, my_tiles / my_items) : 0xFFFFFFFFu;
    uint32_t it = gw, since = 0;

    auto do_item = [&]() {
        const uint4 w = items[it];
        it += n_warps;
        zero_tile<S>(sm.tile, lane);
        accumulate_records<S, KB>(g, records, w.y, w.z, sm, lane);
        flush_ring<S>(g, sm, grid, w.x, tr, lane);
    };

    if (mode != WS_GRID_OVERWRITE) {
        // only the listed bins matter (k_prepare_heavy: non-empty, not heavy); 96 % of the tiles of Large hold nothing, and
        // walking them costs every warp a dependent load each -- again in every call of a chunked run
        // The warps take their work from one counter: the chunks of the heavy bins first (1024 records each), then the
        // listed bins (1 .. 1024 records), so that the short ones fill the end of the kernel evenly.
        const uint32_t total = n_items + status->n_light;
        for (;;) {
            uint32_t q = 0;
            if (lane == 0) q = atomicAdd(&status->queue, 1u);
            q = __shfl_sync(0xffffffffu, q, 0);
            if (q >= total) break;
            uint32_t bin, lo, hi;
            if (q < n_items) {
                const uint4 w = items[q];
                bin = w.x, lo = w.y, hi = w.z;
            } else {
                bin = light[q - n_items];
                lo = bin_start[bin], hi = bin_start[bin + 1];
            }
            zero_tile<S>(sm.tile, lane);
            accumulate_records<S, KB>(g, records, lo, hi, sm, lane);
            flush_ring<S>(g, sm, grid, bin, tr, lane);
        }
        return;
    }
    for (uint32_t bin = gw; bin < g.n_bins; bin += n_warps) {
        if (it < n_items && since >= gap) {
            do_item();
            since = 0;
        }
        ++since;
        const uint32_t s = bin_start[bin], e = bin_start[bin + 1];
        if (e - s > WS_CHUNK) continue;                     // heavy: its chunks are items
        if (s == e) {
            if (mode == WS_GRID_OVERWRITE && occ_start[bin + 1] == occ_start[bin])
                store_zero_tile(tile_origin(g, grid, bin, tr), (size_t)g.n_pix, lane);
            continue;
        }
        zero_tile<S>(sm.tile, lane);
        accumulate_records<S, KB>(g, records, s, e, sm, lane);
        flush_ring<S>(g, sm, grid, bin, tr, lane);
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
    const uint32_t* occ_start = (const uint32_t*)(ws + L.off_rec_start);
    const uint32_t* bin_start = (const uint32_t*)(ws + L.off_counts_home);
    const float4* records = (const float4*)(ws + L.off_records);
    WsStatus* status = plan->d_status;
    uint4* items = (uint4*)(ws + L.off_items);
    const WsGeom& g = plan->geom;
    uint32_t* light = (uint32_t*)(ws + L.off_cursor_home);        // (the scatter's cursors are spent)
    if (cudaMemsetAsync(&status->n_items, 0, 3 * sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;    // n_items, n_light, queue
    k_prepare_heavy<<<(g.n_bins + 255) / 256, 256, 0, st>>>(g, bin_start, occ_start, 1, light, items, L.item_capacity, status, grid,
                                                          mode, orient, mv);
    k_grid<S, KB><<<plan->sm_count, C::THREADS, smem, st>>>(g, bin_start, occ_start, light, items, records, grid, mode, status, orient);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 2;
}

}  // namespace

// Work items for the lists of `starts` ([n_bins + 1] offsets) longer than WS_CHUNK, and the list of the other non-empty bins:
// used by the degridder on the home lists.
int ws_launch_items(ws_plan* plan, const uint32_t* starts, uint32_t* light, uint4* items, uint32_t item_capacity, cudaStream_t st) {
    const WsGeom& g = plan->geom;
    if (cudaMemsetAsync(&plan->d_status->n_items, 0, 3 * sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;    // n_items, n_light, queue
    k_prepare_heavy<<<(g.n_bins + 255) / 256, 256, 0, st>>>(g, starts, starts, 0, light, items, item_capacity, plan->d_status, nullptr,
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
