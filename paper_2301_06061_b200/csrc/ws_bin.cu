// a1: binning of the visibilities by (w-plane, uv-tile)  --  PAPER.md:78 (sub-step 1, the per-region lists of
// visibilities), :144-150 (bucketing then gather into contiguous arrays).  The paper builds linked lists on the
// CPU; here it is a one-digit counting sort on the device (the whole key is the digit; the order INSIDE a bin is
// unspecified, R19): histogram over all bins, exclusive prefix scan (warp shuffles), and a scatter that
// writes, per bin, contiguous 16-byte records the gridder streams: one record per visibility, in the bin of the tile
// that holds its centre cell.  (Round 1 copied a record into every tile its footprint reaches; the gridder now carries a
// ring around each tile instead, ws_grid.cu.)
#include <stddef.h>

#include <algorithm>

#include "ws_internal.h"
#include "ws_place.cuh"

namespace {

constexpr int T = WS_TILE;
constexpr int T_LOG2 = 5;

// Warp-aggregated counting (the dense core of the uv plane, sends a large share of all
// visibilities to a few bins; one atomic per visibility serialises on those addresses).  The lanes of a warp
// that share the home bin are found with ONE match.any; the lanes among them that also share a neighbour tile
// (same side) follow from ballots.  Each group elects its lowest lane, which adds the group's size.
struct Groups {
    unsigned home, nx, ny, nc;     // peer masks: home bin, x-neighbour, y-neighbour, corner neighbour (0 if none)
};
__device__ __forceinline__ Groups warp_groups(uint32_t home, int dx, int dy) {
    Groups q;
    q.home = __match_any_sync(0xffffffffu, home);
    const unsigned xm = __ballot_sync(0xffffffffu, dx < 0), xp = __ballot_sync(0xffffffffu, dx > 0);
    const unsigned ym = __ballot_sync(0xffffffffu, dy < 0), yp = __ballot_sync(0xffffffffu, dy > 0);
    const unsigned sx = dx < 0 ? xm : (dx > 0 ? xp : 0u), sy = dy < 0 ? ym : (dy > 0 ? yp : 0u);
    q.nx = q.home & sx;
    q.ny = q.home & sy;
    q.nc = q.home & sx & sy;
    return q;
}
__device__ __forceinline__ bool leads(unsigned group, int lane) { return group && lane == __ffs(group) - 1; }
__device__ __forceinline__ uint32_t rank_in(unsigned group, int lane) { return (uint32_t)__popc(group & ((1u << lane) - 1u)); }

// The per-channel constants are staged in shared memory: indexing the kernel parameter with a per-lane channel
// would be a divergent constant-bank load, replayed once per distinct channel in the warp.
__device__ __forceinline__ void stage_consts(const WsChanConsts& cc, uint32_t n_chan, double* s_su, double* s_sw) {
    for (uint32_t i = threadIdx.x; i < n_chan; i += blockDim.x) {
        s_su[i] = cc.su[i];
        s_sw[i] = cc.sw[i];
    }
    __syncthreads();
}

// thread index -> flat visibility index (WsRemap, ws_internal.h).  Warp w = (snapshot block tb, adjacent group f_hi);
// lane = f_lo * ts + tt: the ts consecutive snapshots of one (baseline, channel) sit in consecutive lanes, so that
// the slots they take in a bin are consecutive too.
__device__ __forceinline__ uint32_t remap(const WsRemap& r, uint32_t mp) {
    if (r.cw == 0u || mp >= r.n_main) return mp;
    const uint32_t L = mp & 31u, wq = mp >> 5, ts_log2 = 5u - r.cw_log2;
    const uint32_t tt = L & ((1u << ts_log2) - 1u), f_lo = L >> ts_log2;
    const uint32_t f_hi = wq / r.n_t, tb = wq - f_hi * r.n_t;               // n_t: whole blocks of ts snapshots
    return ((tb << ts_log2) + tt) * r.per_snap + (f_hi << r.cw_log2) + f_lo;
}

__device__ __forceinline__ void row_chan(uint32_t m, uint32_t n_chan, int chan_shift, uint32_t& row, uint32_t& c) {
    if (chan_shift >= 0) {
        row = m >> chan_shift;
        c = m & (n_chan - 1u);
    } else {
        row = m / n_chan;
        c = m - row * n_chan;
    }
}

// ---- pass A: keys + histograms -------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_keys_hist(const __grid_constant__ WsChanConsts cc, const __grid_constant__ WsGeom g,
            const float* __restrict__ uvw, uint32_t n_vis, uint32_t n_chan, int chan_shift,
            uint32_t* __restrict__ keys, uint32_t* __restrict__ counts_home, uint32_t* __restrict__ counts_halo,
            int home_only, const __grid_constant__ WsRemap rm) {
    __shared__ double s_su[WS_MAX_CHAN], s_sw[WS_MAX_CHAN];
    stage_consts(cc, n_chan, s_su, s_sw);
    const uint32_t m = remap(rm, blockIdx.x * 256u + threadIdx.x);
    const int lane = threadIdx.x & 31;
    Placed pl;
    bool kept = false;
    if (m < n_vis) {
        uint32_t row, c;
        row_chan(m, n_chan, chan_shift, row, c);
        const float* p = uvw + 3ull * row;
        kept = place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), s_su[c], s_sw[c], pl);
    }
    uint32_t home = 0xFFFFFFFFu;
    int tx = 0, ty = 0, dx = 0, dy = 0, k = 0;
    if (kept) {
        tx = pl.i0 >> T_LOG2; ty = pl.j0 >> T_LOG2; k = pl.k;
        const int lx = pl.i0 & (T - 1), ly = pl.j0 & (T - 1);
        home = bin_of(g, k, ty, tx);
        // tiles the footprint overlaps: own, and the neighbour on each side it sticks out of
        dx = lx < g.halo ? -1 : (lx >= T - g.halo ? 1 : 0);
        dy = ly < g.halo ? -1 : (ly >= T - g.halo ? 1 : 0);
        if (home_only) dx = dy = 0;               // bins for the degridder: a gather reaches nothing outside its staged region
                                                  // (the gridder needs the halo counts: which tiles receive anything)
    }
    if (m < n_vis) keys[m] = home;
    // two histograms: visibilities per home bin (-> bin_start) and halo copies received per bin; the record
    // list of a bin is its home records followed by its halo records (rec_start = their sum, k_finish_offsets)
    const Groups q = warp_groups(home, dx, dy);
    if (kept && leads(q.home, lane)) atomicAdd(counts_home + home, (uint32_t)__popc(q.home));
    if (leads(q.nx, lane)) atomicAdd(counts_halo + bin_of(g, k, ty, tx + dx), (uint32_t)__popc(q.nx));
    if (leads(q.ny, lane)) atomicAdd(counts_halo + bin_of(g, k, ty + dy, tx), (uint32_t)__popc(q.ny));
    if (leads(q.nc, lane)) atomicAdd(counts_halo + bin_of(g, k, ty + dy, tx + dx), (uint32_t)__popc(q.nc));
}

// ---- exclusive prefix scan over n entries of two arrays (blockIdx.y selects), in place ------------------
constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_BLOCK = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += t;
    }
    return v;
}

// inclusive scan of one value per thread over the block; returns the inclusive value, *total = block sum
__device__ __forceinline__ uint32_t block_incl_scan(uint32_t v, uint32_t* total) {
    __shared__ uint32_t wsum[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = warp_incl_scan(v);
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < (int)(blockDim.x >> 5) ? wsum[lane] : 0u;
        s = warp_incl_scan(s);
        wsum[lane] = s;
    }
    __syncthreads();
    const uint32_t base = wid ? wsum[wid - 1] : 0u;
    *total = wsum[(blockDim.x >> 5) - 1];
    __syncthreads();
    return inc + base;
}

__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_reduce(const uint32_t* __restrict__ a0, const uint32_t* __restrict__ a1, uint32_t n,
              uint32_t* __restrict__ block_sums, uint32_t n_blocks) {
    const uint32_t* a = blockIdx.y ? a1 : a0;
    const uint32_t base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_ITEMS;
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < n) s += a[base + i];
    uint32_t total;
    block_incl_scan(s, &total);
    if (threadIdx.x == 0) block_sums[blockIdx.y * n_blocks + blockIdx.x] = total;
}

__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_block_sums(uint32_t* __restrict__ block_sums, uint32_t n_blocks) {
    uint32_t* b = block_sums + blockIdx.y * n_blocks;
    uint32_t carry = 0;
    for (uint32_t lo = 0; lo < n_blocks; lo += SCAN_THREADS) {
        const uint32_t i = lo + threadIdx.x;
        const uint32_t v = i < n_blocks ? b[i] : 0u;
        uint32_t total;
        const uint32_t inc = block_incl_scan(v, &total);
        if (i < n_blocks) b[i] = carry + inc - v;   // exclusive
        carry += total;
    }
}

// Writes the exclusive scans in place (bin_start, halo_start).
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_apply(uint32_t* __restrict__ a0, uint32_t* __restrict__ a1, uint32_t n, const uint32_t* __restrict__ block_sums,
             uint32_t n_blocks) {
    uint32_t* a = blockIdx.y ? a1 : a0;
    const uint32_t base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        v[i] = base + i < n ? a[base + i] : 0u;
        s += v[i];
    }
    uint32_t total;
    const uint32_t inc = block_incl_scan(s, &total);
    uint32_t run = block_sums[blockIdx.y * n_blocks + blockIdx.x] + inc - s;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        if (base + i < n) a[base + i] = run;
        run += v[i];
    }
}

// rec_start = bin_start + halo_start (home + halo counts, scanned: rec_start[b + 1] > rec_start[b] <=> tile b receives
// something from its own visibilities or from a neighbour's footprints); slot cursors start at bin_start[b]; totals
// and the capacity check.
__global__ void __launch_bounds__(256)
k_finish_offsets(const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ halo_start,
                 uint32_t* __restrict__ rec_start, uint32_t* __restrict__ cursor_home,
                 uint32_t n_bins, WsStatus* __restrict__ status, uint64_t rec_capacity) {
    const uint32_t b = blockIdx.x * 256u + threadIdx.x;
    if (b > n_bins) return;
    const uint32_t bs = bin_start[b], hs = halo_start[b];
    rec_start[b] = bs + hs;
    if (b < n_bins) {
        cursor_home[b] = bs;
    } else {
        status->n_kept = bs;
        status->n_records = bs;                         // one record per kept visibility, in its home bin
        if ((uint64_t)bs > rec_capacity) status->overflow = status->sticky_overflow = 1u;
    }
}

// ---- pass B: scatter into per-bin record lists ----------------------------------------------------------
// One record (16 B) per kept visibility, in the list of its HOME bin (the tile that holds its centre cell): X, Y = centre
// cell minus tile origin (0 .. T-1) in the top byte, 24-bit fraction of fu + 1/2 below it; then weight * norm * vis
// (re, im).  The record slot is the perm slot: the lists are indexed by bin_start.  What a footprint puts onto neighbour
// tiles is the gridder's business (it accumulates every tile with a ring, ws_grid.cu); the halo HISTOGRAM of pass A only
// tells which tiles receive anything.
__global__ void __launch_bounds__(256)
k_scatter(const __grid_constant__ WsChanConsts cc, const __grid_constant__ WsGeom g,
          const float* __restrict__ uvw, const float2* __restrict__ vis, const float* __restrict__ wt,
          uint32_t n_vis, uint32_t n_chan, int chan_shift, uint32_t* __restrict__ cursor_home, uint32_t* __restrict__ perm,
          float4* __restrict__ records, const WsStatus* __restrict__ status, const __grid_constant__ WsRemap rm) {
    if (status->overflow) return;
    __shared__ double s_su[WS_MAX_CHAN], s_sw[WS_MAX_CHAN];
    stage_consts(cc, n_chan, s_su, s_sw);
    const uint32_t m = remap(rm, blockIdx.x * 256u + threadIdx.x);
    const int lane = threadIdx.x & 31;
    Placed pl;
    bool kept = false;
    float2 v = make_float2(0.f, 0.f);
    float w = 0.f;
    if (m < n_vis) {
        uint32_t row, c;
        row_chan(m, n_chan, chan_shift, row, c);
        const float* p = uvw + 3ull * row;
        // the value and the weight are asked for together with the position, not after the drop test: the kernel is bound by
        // its chain of round trips (position -> value -> slot), and dropped visibilities are rare
        if (vis) {                                  // NULL: bins for the degridder, the records carry positions only
            v = __ldcs(vis + m);
            w = wt ? __ldcs(wt + m) : 1.0f;         // NULL: pre-summed rows, the weights are already inside
        }
        kept = place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), s_su[c], s_sw[c], pl);
    }
    uint32_t home = 0xFFFFFFFFu;
    int lx = 0, ly = 0;
    if (kept) {
        lx = pl.i0 & (T - 1); ly = pl.j0 & (T - 1);
        home = bin_of(g, pl.k, pl.j0 >> T_LOG2, pl.i0 >> T_LOG2);
    }
    // slots: one atomic per group of lanes that share the bin, the result broadcast by shuffle
    const unsigned peers = __match_any_sync(0xffffffffu, home);
    uint32_t bh = 0;
    if (kept && leads(peers, lane)) bh = atomicAdd(cursor_home + home, (uint32_t)__popc(peers));
    uint32_t qx = 0, qy = 0;
    float vr = 0.f, vi = 0.f;
    if (kept) {
        const float wn = w * g.norm2;
        qx = __double2uint_rn(__dadd_rn(pl.fu, 0.5) * 16777216.0);
        qy = __double2uint_rn(__dadd_rn(pl.fv, 0.5) * 16777216.0);
        qx = qx > 0xFFFFFFu ? 0xFFFFFFu : qx;
        qy = qy > 0xFFFFFFu ? 0xFFFFFFu : qy;
        vr = v.x * wn; vi = v.y * wn;
    }
    bh = __shfl_sync(0xffffffffu, bh, __ffs(peers) - 1) + rank_in(peers, lane);
    if (!kept) return;
    perm[bh] = m;
    records[bh] = make_float4(__uint_as_float(((uint32_t)lx << 24) | qx), __uint_as_float(((uint32_t)ly << 24) | qy), vr, vi);
}

// ---- parity export: sorted_keys[] expanded from bin_start (run lengths) ---------------------------------
__global__ void __launch_bounds__(256)
k_sorted_keys(const uint32_t* __restrict__ bin_start, uint32_t n_bins, uint32_t* __restrict__ sorted_keys) {
    const uint32_t w = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_bins) return;
    const uint32_t s = bin_start[w], e = bin_start[w + 1];
    for (uint32_t i = s + lane; i < e; i += 32) sorted_keys[i] = w;
}

// ---- WS_FLAG_TRACK_SUMWT: sum of the weights of the kept visibilities (keys[] != 0xFFFFFFFF), fp64 --------------
__global__ void __launch_bounds__(256)
k_sum_weights(const uint32_t* __restrict__ keys, const float* __restrict__ wt, uint32_t n_vis, uint32_t chan_per_key,
              double* __restrict__ sum) {
    __shared__ double s_part[8];
    double acc = 0.0;
    for (uint32_t m = blockIdx.x * 256u + threadIdx.x; m < n_vis; m += gridDim.x * 256u)
        if (__ldg(keys + (chan_per_key == 1u ? m : m / chan_per_key)) != 0xFFFFFFFFu) acc += (double)__ldcs(wt + m);
#pragma unroll
    for (int d = 16; d; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) t += s_part[i];
        atomicAdd(sum, t);
    }
}

// ---- WS_FLAG_PRESUM_CHANNELS: out[row] = sum_c wt[row][c] * vis[row][c] (narrow-band mode) ----------
__global__ void __launch_bounds__(256)
k_presum_rows(const float2* __restrict__ vis, const float* __restrict__ wt, uint32_t n_rows, uint32_t n_chan,
              float2* __restrict__ out) {
    const uint32_t n_warps = gridDim.x * 8u, lane = threadIdx.x & 31u;
    for (uint32_t row = blockIdx.x * 8u + (threadIdx.x >> 5); row < n_rows; row += n_warps) {
        const size_t base = (size_t)row * n_chan;
        float ar = 0.f, ai = 0.f;
        for (uint32_t c = lane; c < n_chan; c += 32u) {
            const float2 v = __ldcs(vis + base + c);
            const float w = __ldcs(wt + base + c);
            ar = fmaf(w, v.x, ar);
            ai = fmaf(w, v.y, ai);
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            ar += __shfl_xor_sync(0xffffffffu, ar, d);
            ai += __shfl_xor_sync(0xffffffffu, ai, d);
        }
        if (lane == 0) out[row] = make_float2(ar, ai);
    }
}

}  // namespace

int ws_launch_presum(ws_plan* plan, const float2* vis, const float* wt, int64_t n_rows, int32_t n_chan, float2* out,
                     cudaStream_t st) {
    if (n_rows <= 0) return 0;
    const unsigned blocks = (unsigned)std::min<int64_t>((n_rows + 7) / 8, (int64_t)plan->sm_count * 32);
    k_presum_rows<<<blocks, 256, 0, st>>>(vis, wt, (uint32_t)n_rows, (uint32_t)n_chan, out);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_sum_weights(ws_plan* plan, const WsLayout& L, char* ws, const float* wt, int64_t n_vis, int32_t chan_per_key,
                          cudaStream_t st) {
    if (n_vis <= 0) return 0;
    const unsigned blocks = (unsigned)std::min<int64_t>((n_vis + 255) / 256, (int64_t)plan->sm_count * 8);
    k_sum_weights<<<blocks, 256, 0, st>>>((const uint32_t*)(ws + L.off_keys), wt, (uint32_t)n_vis, (uint32_t)chan_per_key,
                                          plan->d_sumwt);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_bin(ws_plan* plan, const WsLayout& L, char* ws, const WsChanConsts& cc, const float* uvw,
                  const float2* vis, const float* wt, int64_t n_rows, int32_t n_chan, cudaStream_t st) {
    const WsGeom& g = plan->geom;
    const int home_only = vis == nullptr;          // positions only: the degridder's gather (no halo histogram)
    WsRemap rm = {0u, 0u, 0u, 0u, 0u};
    if (plan->snapshot_rows > 0 && n_rows >= 2 * plan->snapshot_rows) {
        const uint64_t F = (uint64_t)plan->snapshot_rows * (uint64_t)n_chan;
        uint32_t lg = 2;                              // cw = 4 adjacent visibilities x 8 snapshots per warp
        while (lg > 0 && (F & ((1u << lg) - 1u))) --lg;
        rm.cw_log2 = lg;
        rm.cw = 1u << lg;
        rm.n_t = (uint32_t)((n_rows / plan->snapshot_rows) >> (5u - lg));    // blocks of ts = 32 / cw snapshots
        rm.per_snap = (uint32_t)F;
        rm.n_main = (uint32_t)(((uint64_t)rm.n_t << (5u - lg)) * F);
        if (rm.n_t == 0) rm.cw = 0u;
    }
    const uint32_t n_vis = (uint32_t)(n_rows * n_chan);
    uint32_t* counts_home = (uint32_t*)(ws + L.off_counts_home);   // -> bin_start
    uint32_t* counts_halo = (uint32_t*)(ws + L.off_counts_halo);   // -> halo_start
    uint32_t* rec_start = (uint32_t*)(ws + L.off_rec_start);
    uint32_t* cursor_home = (uint32_t*)(ws + L.off_cursor_home);
    uint32_t* block_sums = (uint32_t*)(ws + L.off_block_sums);
    WsStatus* status = plan->d_status;
    uint32_t* keys = (uint32_t*)(ws + L.off_keys);
    uint32_t* perm = (uint32_t*)(ws + L.off_perm);
    float4* records = (float4*)(ws + L.off_records);
    int launches = 0;
    int chan_shift = -1;   // log2(n_chan) when it is a power of two: row = m >> shift instead of a division
    for (int b = 0; b < 8; ++b)
        if (n_chan == (1 << b)) chan_shift = b;

    // the two histograms are contiguous at the head of the workspace: one clear, plus the plan's status block
    if (cudaMemsetAsync(ws, 0, L.off_rec_start, st) != cudaSuccess) return WS_ERR_CUDA;
    if (cudaMemsetAsync(status, 0, offsetof(WsStatus, sticky_overflow), st) != cudaSuccess) return WS_ERR_CUDA;

    const uint32_t n_scan = g.n_bins + 1;
    const uint32_t n_blocks = (n_scan + SCAN_BLOCK - 1) / SCAN_BLOCK;
    if (n_vis) {
        k_keys_hist<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, n_vis, (uint32_t)n_chan, chan_shift, keys,
                                                         counts_home, counts_halo, home_only, rm);
        ++launches;
    }
    k_scan_reduce<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_halo, n_scan, block_sums, n_blocks);
    k_scan_block_sums<<<dim3(1, 2), SCAN_THREADS, 0, st>>>(block_sums, n_blocks);
    k_scan_apply<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_halo, n_scan, block_sums, n_blocks);
    k_finish_offsets<<<(n_scan + 255) / 256, 256, 0, st>>>(counts_home, counts_halo, rec_start, cursor_home,
                                                          g.n_bins, status, L.rec_capacity);
    launches += 4;
    if (n_vis) {
        k_scatter<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, vis, wt, n_vis, (uint32_t)n_chan, chan_shift,
                                                       cursor_home, perm, records, status, rm);
        ++launches;
    }
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return launches;
}

int ws_launch_sorted_keys(ws_plan* plan, const WsLayout& L, char* ws, cudaStream_t st) {
    const WsGeom& g = plan->geom;
    const uint64_t threads = (uint64_t)g.n_bins * 32;
    k_sorted_keys<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>((const uint32_t*)(ws + L.off_counts_home), g.n_bins,
                                                                     (uint32_t*)(ws + L.off_sorted_keys));
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}
