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

// ---- pass A: keys + histograms -------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_keys_hist(const __grid_constant__ WsChanConsts cc, const __grid_constant__ WsGeom g,
            const float* __restrict__ uvw, uint32_t n_vis, uint32_t n_chan,
            uint32_t* __restrict__ keys, uint32_t* __restrict__ counts_home, uint32_t* __restrict__ counts_all) {
    const uint32_t m = blockIdx.x * 256u + threadIdx.x;
    if (m >= n_vis) return;
    const uint32_t row = m / n_chan, c = m - row * n_chan;
    const float* p = uvw + 3ull * row;
    Placed pl;
    if (!place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), (int)c, pl)) {
        keys[m] = 0xFFFFFFFFu;
        return;
    }
    const int tx = pl.i0 >> T_LOG2, ty = pl.j0 >> T_LOG2;
    const int lx = pl.i0 & (T - 1), ly = pl.j0 & (T - 1);
    const uint32_t home = bin_of(g, pl.k, ty, tx);
    keys[m] = home;
    atomicAdd(counts_home + home, 1u);
    // tiles the footprint overlaps: own, and the neighbour on each side it sticks out of
    const int dx = lx < g.halo ? -1 : (lx >= T - g.halo ? 1 : 0);
    const int dy = ly < g.halo ? -1 : (ly >= T - g.halo ? 1 : 0);
    atomicAdd(counts_all + home, 1u);
    if (dx) atomicAdd(counts_all + bin_of(g, pl.k, ty, tx + dx), 1u);
    if (dy) atomicAdd(counts_all + bin_of(g, pl.k, ty + dy, tx), 1u);
    if (dx && dy) atomicAdd(counts_all + bin_of(g, pl.k, ty + dy, tx + dx), 1u);
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
          uint32_t n_vis, uint32_t n_chan, uint32_t* __restrict__ cursor_home, uint32_t* __restrict__ cursor_all,
          uint32_t* __restrict__ perm, float4* __restrict__ records, const WsStatus* __restrict__ status) {
    if (status->overflow) return;
    const uint32_t m = blockIdx.x * 256u + threadIdx.x;
    if (m >= n_vis) return;
    const uint32_t row = m / n_chan, c = m - row * n_chan;
    const float* p = uvw + 3ull * row;
    Placed pl;
    if (!place(cc, g, __ldg(p), __ldg(p + 1), __ldg(p + 2), (int)c, pl)) return;
    const int tx = pl.i0 >> T_LOG2, ty = pl.j0 >> T_LOG2;
    const int lx = pl.i0 & (T - 1), ly = pl.j0 & (T - 1);
    const uint32_t home = bin_of(g, pl.k, ty, tx);
    perm[atomicAdd(cursor_home + home, 1u)] = m;

    const float2 v = __ldg(vis + m);
    const float wn = __ldg(wt + m) * g.norm2;
    uint32_t qx = __double2uint_rn(__dadd_rn(pl.fu, 0.5) * 16777216.0);
    uint32_t qy = __double2uint_rn(__dadd_rn(pl.fv, 0.5) * 16777216.0);
    qx = qx > 0xFFFFFFu ? 0xFFFFFFu : qx;
    qy = qy > 0xFFFFFFu ? 0xFFFFFFu : qy;
    const float vr = v.x * wn, vi = v.y * wn;
    const int dx = lx < g.halo ? -1 : (lx >= T - g.halo ? 1 : 0);
    const int dy = ly < g.halo ? -1 : (ly >= T - g.halo ? 1 : 0);
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const int ddx = (t & 1) ? dx : 0, ddy = (t & 2) ? dy : 0;
        if (((t & 1) && !dx) || ((t & 2) && !dy)) continue;
        const uint32_t b = bin_of(g, pl.k, ty + ddy, tx + ddx);
        const uint32_t slot = atomicAdd(cursor_all + b, 1u);
        // centre cell relative to the receiving tile's origin: lx - ddx*T (negative wraps into the signed byte)
        const uint32_t X = ((uint32_t)(lx - ddx * T) << 24) | qx;
        const uint32_t Y = ((uint32_t)(ly - ddy * T) << 24) | qy;
        records[slot] = make_float4(__uint_as_float(X), __uint_as_float(Y), vr, vi);
    }
}

// ---- heavy bins: every chunk after the first becomes a work item of the reduce-add kernel ---------------
__global__ void __launch_bounds__(256)
k_build_items(const uint32_t* __restrict__ rec_start, uint32_t n_bins, uint4* __restrict__ items,
              uint32_t item_capacity, WsStatus* __restrict__ status) {
    const uint32_t b = blockIdx.x * 256u + threadIdx.x;
    if (b >= n_bins || status->overflow) return;
    const uint32_t s = rec_start[b], e = rec_start[b + 1];
    const uint32_t cnt = e - s;
    if (cnt <= WS_CHUNK) return;
    const uint32_t extra = (cnt - 1) / WS_CHUNK;
    const uint32_t base = atomicAdd(&status->n_items, extra);
    if (base + extra > item_capacity) {
        status->overflow = 1u;
        return;
    }
    for (uint32_t i = 0; i < extra; ++i) {
        const uint32_t lo = s + (i + 1) * WS_CHUNK;
        const uint32_t hi = lo + WS_CHUNK < e ? lo + WS_CHUNK : e;
        items[base + i] = make_uint4(b, lo, hi, 0u);
    }
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
    uint4* items = (uint4*)(ws + L.off_items);
    float4* records = (float4*)(ws + L.off_records);
    int launches = 0;

    // the counters are contiguous at the head of the workspace: one clear, plus the plan's status block
    if (cudaMemsetAsync(ws, 0, L.off_keys, st) != cudaSuccess) return WS_ERR_CUDA;
    if (cudaMemsetAsync(status, 0, sizeof(WsStatus), st) != cudaSuccess) return WS_ERR_CUDA;

    const uint32_t n_scan = g.n_bins + 1;
    const uint32_t n_blocks = (n_scan + SCAN_BLOCK - 1) / SCAN_BLOCK;
    if (n_vis) {
        k_keys_hist<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, n_vis, (uint32_t)n_chan, keys, counts_home,
                                                         counts_all);
        ++launches;
    }
    k_scan_reduce<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_all, n_scan, block_sums, n_blocks);
    k_scan_block_sums<<<dim3(1, 2), SCAN_THREADS, 0, st>>>(block_sums, n_blocks);
    k_scan_apply<<<dim3(n_blocks, 2), SCAN_THREADS, 0, st>>>(counts_home, counts_all, cursor_home, cursor_all, n_scan,
                                                             block_sums, n_blocks, status, L.rec_capacity);
    launches += 3;
    if (n_vis) {
        k_scatter<<<(n_vis + 255) / 256, 256, 0, st>>>(cc, g, uvw, vis, wt, n_vis, (uint32_t)n_chan, cursor_home,
                                                       cursor_all, perm, records, status);
        ++launches;
    }
    k_build_items<<<(g.n_bins + 255) / 256, 256, 0, st>>>(counts_all, g.n_bins, items, L.item_capacity, status);
    ++launches;
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
