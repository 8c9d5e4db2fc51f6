// a1: binning of the visibilities by (w-plane, uv-tile)  --  PAPER.md:78 (sub-step 1, the per-region lists of
// visibilities), :144-150 (bucketing then gather into contiguous arrays).  The paper builds linked lists on the
// CPU; here it is a radix-2^b counting sort on the device: histogram over all bins (one digit = the whole
// key), exclusive prefix scan (warp shuffles), and a scatter that writes, per bin, contiguous 16-byte records
// the gridder streams.  A visibility whose S x S footprint crosses a tile border is written into every tile
// it touches (up to 4), so that each tile-plane of the mesh is produced by exactly one warp (ws_grid.cu).
#include "ws_internal.h"

namespace {

constexpr int T = WS_TILE;
constexpr int T_LOG2 = 5;

// ---- O2-O4: position rule.  Each line is one correctly rounded binary64 operation,
// in the order the header states; the oracle performs the same operations on the host.
struct Placed {
    int i0, j0, k;
    double fu, fv;
};

__device__ __forceinline__ bool place(const WsChanConsts& cc, const WsGeom& g, float u, float v, float w, int c,
                                      Placed& o) {
    const double su = cc.su[c], sw = cc.sw[c];
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
    if (!(ci >= lo && ci <= hi && cj >= lo && cj <= hi)) return false;   // drop rule O3 (R5); NaN drops
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
            uint32_t* __restrict__ keys, uint32_t* __restrict__ counts_home, uint32_t* __restrict__ counts_all) {
    const uint32_t m = blockIdx.x * 256u + threadIdx.x;
    const int lane = threadIdx.x & 31;
    Placed pl;
    bool kept = false;
    if (m < n_vis) {
        uint32_t row, c;
        row_chan(m, n_chan, chan_shift, row, c);
        const float* p = uvw + 3ull * row;
        kept = place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), (int)c, pl);
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
    }
    if (m < n_vis) keys[m] = home;
    const Groups q = warp_groups(home, dx, dy);
    if (kept && leads(q.home, lane)) {
        const uint32_t n = (uint32_t)__popc(q.home);
        atomicAdd(counts_home + home, n);
        atomicAdd(counts_all + home, n);
    }
    if (leads(q.nx, lane)) atomicAdd(counts_all + bin_of(g, k, ty, tx + dx), (uint32_t)__popc(q.nx));
    if (leads(q.ny, lane)) atomicAdd(counts_all + bin_of(g, k, ty + dy, tx), (uint32_t)__popc(q.ny));
    if (leads(q.nc, lane)) atomicAdd(counts_all + bin_of(g, k, ty + dy, tx + dx), (uint32_t)__popc(q.nc));
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

// Writes the exclusive scan in place, seeds the scatter cursors, and records the totals.
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_apply(uint32_t* __restrict__ a0, uint32_t* __restrict__ a1, uint32_t* __restrict__ cur0,
             uint32_t* __restrict__ cur1, uint32_t n, const uint32_t* __restrict__ block_sums, uint32_t n_blocks,
             WsStatus* __restrict__ status, uint64_t rec_capacity) {
    uint32_t* a = blockIdx.y ? a1 : a0;
    uint32_t* cur = blockIdx.y ? cur1 : cur0;
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
        const uint32_t idx = base + i;
        if (idx < n) {
            a[idx] = run;
            if (idx < n - 1) cur[idx] = run;
            else {   // entry n-1 = n_bins: the grand total
                if (blockIdx.y == 0) status->n_kept = run;
                else {
                    status->n_records = run;
                    if ((uint64_t)run > rec_capacity) status->overflow = 1u;
                }
            }
        }
        run += v[i];
    }
}

// ---- pass B: scatter into per-bin record lists ----------------------------------------------------------
// Record (16 B): X, Y = position relative to the RECEIVING tile: signed 8-bit integer part = centre cell minus
// tile origin (i0 - tile_x0, in [-h, T-1+h]) in the top byte, 24-bit fraction of fu + 1/2 below it; then
// weight * norm * vis (re, im).
__global__ void __launch_bounds__(256)
k_scatter(const __grid_constant__ WsChanConsts cc, const __grid_constant__ WsGeom g,
          const float* __restrict__ uvw, const float2* __restrict__ vis, const float* __restrict__ wt,
          uint32_t n_vis, uint32_t n_chan, int chan_shift, uint32_t* __restrict__ cursor_home,
          uint32_t* __restrict__ cursor_all, uint32_t* __restrict__ perm, float4* __restrict__ records,
          const WsStatus* __restrict__ status) {
    if (status->overflow) return;
    const uint32_t m = blockIdx.x * 256u + threadIdx.x;
    const int lane = threadIdx.x & 31;
    Placed pl;
    bool kept = false;
    if (m < n_vis) {
        uint32_t row, c;
        row_chan(m, n_chan, chan_shift, row, c);
        const float* p = uvw + 3ull * row;
        kept = place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), (int)c, pl);
    }
    uint32_t home = 0xFFFFFFFFu;
    int tx = 0, ty = 0, lx = 0, ly = 0, dx = 0, dy = 0, k = 0;
    float2 v = make_float2(0.f, 0.f);
    float w = 0.f;
    if (kept) {
        v = __ldcs(vis + m);
        w = __ldcs(wt + m);
        tx = pl.i0 >> T_LOG2; ty = pl.j0 >> T_LOG2; k = pl.k;
        lx = pl.i0 & (T - 1); ly = pl.j0 & (T - 1);
        home = bin_of(g, k, ty, tx);
        dx = lx < g.halo ? -1 : (lx >= T - g.halo ? 1 : 0);
        dy = ly < g.halo ? -1 : (ly >= T - g.halo ? 1 : 0);
    }
    // slots: every group leader issues its atomics back to back, the results are broadcast afterwards
    const Groups q = warp_groups(home, dx, dy);
    uint32_t bh = 0, ba = 0, bx = 0, by = 0, bc = 0;
    if (kept && leads(q.home, lane)) {
        const uint32_t n = (uint32_t)__popc(q.home);
        bh = atomicAdd(cursor_home + home, n);
        ba = atomicAdd(cursor_all + home, n);
    }
    if (leads(q.nx, lane)) bx = atomicAdd(cursor_all + bin_of(g, k, ty, tx + dx), (uint32_t)__popc(q.nx));
    if (leads(q.ny, lane)) by = atomicAdd(cursor_all + bin_of(g, k, ty + dy, tx), (uint32_t)__popc(q.ny));
    if (leads(q.nc, lane)) bc = atomicAdd(cursor_all + bin_of(g, k, ty + dy, tx + dx), (uint32_t)__popc(q.nc));

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
    const int lh = __ffs(q.home) - 1;
    bh = __shfl_sync(0xffffffffu, bh, lh) + rank_in(q.home, lane);
    ba = __shfl_sync(0xffffffffu, ba, lh) + rank_in(q.home, lane);
    bx = __shfl_sync(0xffffffffu, bx, q.nx ? __ffs(q.nx) - 1 : lane) + rank_in(q.nx, lane);
    by = __shfl_sync(0xffffffffu, by, q.ny ? __ffs(q.ny) - 1 : lane) + rank_in(q.ny, lane);
    bc = __shfl_sync(0xffffffffu, bc, q.nc ? __ffs(q.nc) - 1 : lane) + rank_in(q.nc, lane);
    if (!kept) return;
    // centre cell relative to the receiving tile's origin: lx - ddx*T (negative wraps into the signed byte)
    auto emit = [&](uint32_t slot, int ddx, int ddy) {
        const uint32_t X = ((uint32_t)(lx - ddx * T) << 24) | qx;
        const uint32_t Y = ((uint32_t)(ly - ddy * T) << 24) | qy;
        records[slot] = make_float4(__uint_as_float(X), __uint_as_float(Y), vr, vi);
    };
    perm[bh] = m;
    emit(ba, 0, 0);
    if (q.nx) emit(bx, dx, 0);
    if (q.ny) emit(by, 0, dy);
    if (q.nc) emit(bc, dx, dy);
}

// ---- parity export: sorted_keys[] expanded from bin_start (run lengths) ---------------------------------
__global__ void __launch_bounds__(256)
k_sorted_keys(const uint32_t* __restrict__ bin_start, uint32_t n_bins, uint32_t* __restrict__ sorted_keys) {
    const uint32_t w = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_bins) return;
    const uint32_t s = bin_start[w], e = bin_start[w + 1];
    for (uint32_t i = s + lane; i < e; i += 32) sorted_keys[i] = w;
}

}  // namespace

int ws_launch_bin(ws_plan* plan, const WsLayout& L, char* ws, const WsChanConsts& cc, const float* uvw,
                  const float2* vis, const float* wt, int64_t n_rows, int32_t n_chan, cudaStream_t st) {
    const WsGeom& g = plan->geom;
    const uint32_t n_vis = (uint32_t)(n_rows * n_chan);
    uint32_t* counts_home = (uint32_t*)(ws + L.off_counts_home);
    uint32_t* counts_all = (uint32_t*)(ws + L.off_counts_all);
    uint32_t* cursor_home = (uint32_t*)(ws + L.off_cursor_home);
    uint32_t* cursor_all = (uint32_t*)(ws + L.off_cursor_all);
    uint32_t* block_sums = (uint32_t*)(ws + L.off_block_sums);
    WsStatus* status = plan->d_status;
    uint32_t* keys = (uint32_t*)(ws + L.off_keys);
    uint32_t* perm = (uint32_t*)(ws + L.off_perm);
    float4* records = (float4*)(ws + L.off_records);
    int launches = 0;
    int chan_shift = -1;   // log2(n_chan) when it is a power of two: row = m >> shift instead of a division
    for (int b = 0; b < 8; ++b)
        if (n_chan == (1 << b)) chan_shift = b;

    // the counters are contiguous at the head of the workspace: one clear, plus the plan's status block
    if (cudaMemsetAsync(ws, 0, L.off_keys, st) != cudaSuccess) return WS_ERR_CUDA;
    if (cudaMemsetAsync(status, 0, sizeof(WsStatus), st) != cudaSuccess) return WS_ERR_CUDA;

    const uint32_t n_scan = g.n_bins + 1;
    const uint32_t n_blocks = (n_scan + SCAN_BLOCK - 1) / SCAN_BLOCK;
    if (n_vis) {
        k_keys_hist<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, n_vis, (uint32_t)n_chan, chan_shift, keys, counts_home,
                                                         counts_all);
        ++launches;
    }
    k_scan_reduce<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_all, n_scan, block_sums, n_blocks);
    k_scan_block_sums<<<dim3(1, 2), SCAN_THREADS, 0, st>>>(block_sums, n_blocks);
    k_scan_apply<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_all, cursor_home, cursor_all, n_scan,
                                                             block_sums, n_blocks, status, L.rec_capacity);
    launches += 3;
    if (n_vis) {
        k_scatter<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, vis, wt, n_vis, (uint32_t)n_chan, chan_shift, cursor_home,
                                                       cursor_all, perm, records, status);
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
