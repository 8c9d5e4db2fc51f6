// Degridding: model image -> predicted visibilities ("the degridding procedure (transforming from the
// image to the visibility space)"; Eq. 1 at :59 discretised the way Eq. 2 / Eq. 3 discretise the imaging direction).
// With unit weights it is the exact adjoint of a1..a4:
//   D1  Q_k(l, m) = M(l, m) exp(-2 pi i w_k (sqrt(1 - l^2 - m^2) - 1))          k_wscreen_fwd
//   D2  H_k = forward un-normalised 2-D DFT of Q_k, per plane                     cuFFT (ws_api.cu)
//   D3  V_m = sum_{a,b} g(a - fu) g(b - fv) H_k[j0 + b][i0 + a]                    k_degrid
// D3 reuses the bins of ws_bin.cu: the paper expects "the same parallelization strategy" to work, with "a specific
// implementation ... required by the distribution of the visibilities on the cell back to the single measurements"
// (:459).  Here a warp owns a tile-plane, stages the tile plus its halo ((T + S - 1)^2 cells) in shared memory once,
// and each lane then gathers the S x S footprint of one visibility with its taps in registers -- a pure gather, no
// atomics; the home lists of the bins give each visibility exactly one owner.
#include "ws_internal.h"
#include "ws_phase.cuh"
#include "ws_taps.cuh"

namespace {

constexpr int T = WS_TILE;
constexpr int G = WS_WC_GROUP;

// ---- D1: the N_w screened copies of the model image, FFT-native storage order -------------------------------
// A thread owns two adjacent pixels; the phases over the planes are a geometric sequence, advanced by one complex
// multiply per plane inside a block of G planes and restarted from an exactly reduced (fp64) phase per block.
__global__ void __launch_bounds__(256)
k_wscreen_fwd(const __grid_constant__ WcParams prm, const float2* __restrict__ image, float4* __restrict__ planes,
              int conj_out, const uint32_t* __restrict__ orient) {
    const uint32_t N = (uint32_t)prm.n_pix, halfN = N >> 1, pairs = N >> 1;
    const uint64_t tid = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    if (tid >= (uint64_t)N * pairs) return;
    // a: line of the stored plane, b, b + 1: the two adjacent cells of it.  [k][v][u]: a = q (m), b = p (l);
    // transposed ([k][u][v], orient set): a = p, b = q -- the screen is symmetric in l and m, only the model is read across
    const bool tr = orient && *orient;
    const uint32_t a = (uint32_t)(tid / pairs), b = (uint32_t)(tid - (uint64_t)a * pairs) * 2u;
    const uint32_t sa = a >= halfN ? a - halfN : a + halfN;
    const uint32_t sb = b >= halfN ? b - halfN : b + halfN;
    const size_t plane_stride = (size_t)N * pairs;                 // in float4 units
    float4* dst = planes + (size_t)sa * pairs + (sb >> 1);
    float4 m;
    if (!tr) {
        m = __ldcs((const float4*)image + tid);
    } else {
        const float2 m0 = __ldg(image + (size_t)b * N + a), m1 = __ldg(image + (size_t)(b + 1) * N + a);
        m = make_float4(m0.x, m0.y, m1.x, m1.y);
    }
    bool inA, inB;
    const double tA = ws_n_minus_1(prm, (int)a, (int)b, &inA), tB = ws_n_minus_1(prm, (int)a, (int)b + 1, &inB);
    if (!inA) m.x = m.y = 0.f;                                      // R14
    if (!inB) m.z = m.w = 0.f;
    const float2 rA = ws_expi_turns(-prm.dw * tA), rB = ws_expi_turns(-prm.dw * tB);
    const int nw = prm.n_wplanes;
    for (int lo = 0; lo < nw; lo += G) {
        const double wk = prm.w0 + (double)lo * prm.dw;
        float2 eA = ws_expi_turns(-wk * tA), eB = ws_expi_turns(-wk * tB);
#pragma unroll
        for (int j = 0; j < G; ++j) {
            if (lo + j < nw) {
                const float2 a = ws_cmul(make_float2(m.x, m.y), eA), b = ws_cmul(make_float2(m.z, m.w), eB);
                __stcs(dst + (size_t)(lo + j) * plane_stride,
                       conj_out ? make_float4(a.x, -a.y, b.x, -b.y) : make_float4(a.x, a.y, b.x, b.y));
                eA = ws_cmul(eA, rA);
                eB = ws_cmul(eB, rB);
            }
        }
    }
}

// ---- D3: the gather ------------------------------------------------------------------------------------------
template <int S>
struct DgCfg {
    static constexpr int H = (S - 1) / 2;
    static constexpr int W = T + 2 * H;             // side of the staged region: the tile and its halo
    static constexpr int P = W | 1;                 // odd row pitch (in cells)
    static constexpr size_t WARP_BYTES = ((size_t)W * P * sizeof(float2) + 15) / 16 * 16;
    static constexpr int WARPS = (113 * 1024) / WARP_BYTES >= 8 ? 8 : (int)((113 * 1024) / WARP_BYTES);
    static constexpr int THREADS = WARPS * 32;
};

// Stages logical cells [x0 - H, x0 + T + H) x [y0 - H, y0 + T + H) of plane k (cells off the mesh: 0; no kept
// visibility reads them, drop rule O3).
template <int S>
__device__ __forceinline__ void load_region(const WsGeom& g, const float2* __restrict__ planes, uint32_t bin, float2* region,
                                            int lane, int xf_lr0, bool tr) {
    using C = DgCfg<S>;
    const uint32_t nt = (uint32_t)g.nt;
    const uint32_t tx = bin % nt, r = bin / nt;
    const uint32_t ty = r % nt, k = r / nt;
    const int N = g.n_pix, half = N >> 1;
    const int x0 = (int)tx * T - C::H, y0 = (int)ty * T - C::H;
    const float2* plane = planes + (size_t)k * (size_t)N * (size_t)N;
#pragma unroll 8
    for (int idx = lane; idx < C::W * C::W; idx += 32) {     // independent loads: eight in flight per lane
        const int i0 = idx / C::W, i1 = idx - i0 * C::W;     // consecutive lanes walk the stored line: x, or y if transposed
        const int ry = tr ? i1 : i0, rx = tr ? i0 : i1;
        const int ly = y0 + ry, lx = x0 + rx;
        float2 v = make_float2(0.f, 0.f);
        if ((unsigned)ly < (unsigned)N && (unsigned)lx < (unsigned)N) {
            const int sy = ly >= half ? ly - half : ly + half, sx = lx >= half ? lx - half : lx + half;
            int line = tr ? sx : sy;                         // the axis the column passes transformed
            const int col = tr ? sy : sx;
            if (xf_lr0 >= 0) line = ((line & ((1 << xf_lr0) - 1)) << 8) | (line >> xf_lr0);   // where ws_fft_columns left that frequency
            v = __ldg(plane + (size_t)line * N + col);
            if (xf_lr0 >= 0) v.y = -v.y;                     // ... of the conjugate transform
        }
        region[ry * C::P + rx] = v;
    }
    __syncwarp();
}

// Home records [lo, hi) (perm slots) of one bin, whose records start `hs` after their perm slots.
template <int S, bool KB>
__device__ __forceinline__ void gather(const WsGeom& g, const float4* __restrict__ records, const uint32_t* __restrict__ perm,
                                       uint32_t lo, uint32_t hi, uint32_t hs, const float2* region, float2* __restrict__ vis_out,
                                       float scale, int accumulate, int lane) {
    using C = DgCfg<S>;
    float4 nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    uint32_t m_nxt = 0;
    if (lo + lane < hi) {
        nxt = __ldcs(records + lo + lane + hs);
        m_nxt = __ldcs(perm + lo + lane);
    }
    for (uint32_t slot = lo + lane; slot < hi; slot += 32) {
        const float4 rec = nxt;
        const uint32_t m = m_nxt;
        if (slot + 32 < hi) {                                       // next batch in flight while this one gathers
            nxt = __ldcs(records + slot + 32 + hs);
            m_nxt = __ldcs(perm + slot + 32);
        }
        const uint32_t X = __float_as_uint(rec.x), Y = __float_as_uint(rec.y);
        const int cx = (int)X >> 24, cy = (int)Y >> 24;            // centre cell in the tile frame = first footprint cell in the region
        const float fx = (float)(X & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
        const float fy = (float)(Y & 0xFFFFFFu) * (1.0f / 16777216.0f) - 0.5f;
        float gu[S], gv[S];
        eval_taps<S, KB>(g, fx, fy, gu, gv);
        const float2* base = region + cy * C::P + cx;
        float ar = 0.f, ai = 0.f;
#pragma unroll
        for (int b = 0; b < S; ++b) {
            float rr = 0.f, ri = 0.f;
#pragma unroll
            for (int a = 0; a < S; ++a) {
                const float2 c = base[b * C::P + a];
                rr = fmaf(gu[a], c.x, rr);
                ri = fmaf(gu[a], c.y, ri);
            }
            ar = fmaf(gv[b], rr, ar);
            ai = fmaf(gv[b], ri, ai);
        }
        const float f = scale * g.norm2;
        float2 out = make_float2(ar * f, ai * f);
        if (accumulate) {
            const float2 old = vis_out[m];
            out.x += old.x;
            out.y += old.y;
        }
        vis_out[m] = out;
    }
    __syncwarp();
}

// Persistent kernel: the warps take the chunks of the heavy bins (items) and then the listed (non-empty, not heavy) bins from one counter.
template <int S, bool KB>
__global__ void __launch_bounds__(DgCfg<S>::THREADS, 2)
k_degrid(const __grid_constant__ WsGeom g, const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ halo_start,
         const uint32_t* __restrict__ light, const uint4* __restrict__ items, const float4* __restrict__ records, const uint32_t* __restrict__ perm,
         const float2* __restrict__ planes, float2* __restrict__ vis_out, float scale, int accumulate,
         WsStatus* __restrict__ status, int xf_lr0, const uint32_t* __restrict__ orient) {
    using C = DgCfg<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float2* region = (float2*)(smem_raw + (size_t)wid * C::WARP_BYTES);
    if (status->overflow) return;
    const bool tr = orient && *orient;           // planes stored [k][u][v] (ws_predict_visibilities may choose so)
    const uint32_t n_items = status->n_items;
    const uint32_t total = n_items + status->n_light;    // the non-empty bins that are not heavy, listed by k_prepare_heavy
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
        load_region<S>(g, planes, bin, region, lane, xf_lr0, tr);
        gather<S, KB>(g, records, perm, lo, hi, halo_start[bin], region, vis_out, scale, accumulate, lane);
    }
}

template <int S, bool KB>
int launch_s(ws_plan* plan, const WsLayout& L, char* ws, const float2* planes, float2* vis_out, float scale, int accumulate,
             int xf_lr0, cudaStream_t st) {
    using C = DgCfg<S>;
    const uint32_t* orient = xf_lr0 >= 0 ? ws_fft_orientation_flag(plan) : nullptr;
    const size_t smem = C::WARP_BYTES * C::WARPS;
    // per device, and cheap: set on every launch rather than cached in a process-wide flag
    if (cudaFuncSetAttribute(k_degrid<S, KB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return WS_ERR_CUDA;
    const uint32_t* bin_start = (const uint32_t*)(ws + L.off_counts_home);
    const uint32_t* halo_start = (const uint32_t*)(ws + L.off_counts_halo);
    uint4* items = (uint4*)(ws + L.off_items);
    uint32_t* light = (uint32_t*)(ws + L.off_cursor_home);        // (the scatter's cursors are spent)
    int rc = ws_launch_items(plan, bin_start, light, items, L.item_capacity, st);
    if (rc < 0) return rc;
    k_degrid<S, KB><<<plan->sm_count * 2, C::THREADS, smem, st>>>(plan->geom, bin_start, halo_start, light, items,
                                                                  (const float4*)(ws + L.off_records),
                                                                  (const uint32_t*)(ws + L.off_perm), planes, vis_out, scale,
                                                                  accumulate, plan->d_status, xf_lr0, orient);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return rc + 1;
}

}  // namespace

int ws_launch_wscreen_fwd(ws_plan* plan, const float2* image, float2* planes, int conj_out, cudaStream_t st) {
    const ws_params& P = plan->prm;
    WcParams prm;
    prm.n_pix = P.n_pix;
    prm.n_wplanes = P.n_wplanes;
    prm.cell = P.cell_rad;
    prm.dw = (P.w_max - P.w_min) / (double)P.n_wplanes;
    prm.w0 = P.w_min + 0.5 * prm.dw;
    const uint64_t n_pairs = (uint64_t)P.n_pix * (uint64_t)(P.n_pix / 2);
    k_wscreen_fwd<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>(prm, image, (float4*)planes, conj_out,
                                                                     conj_out ? ws_fft_orientation_flag(plan) : nullptr);
    if (cudaGetLastError() != cudaSuccess) return WS_ERR_CUDA;
    return 1;
}

int ws_launch_degrid(ws_plan* plan, const WsLayout& L, char* ws, const float2* planes, float2* vis_out, float scale,
                     int accumulate, int xf_lr0, cudaStream_t st) {
    const bool kb = plan->geom.kb_terms > 0;
#define WS_DG_CASE(S_)                                                                                        \
    case S_:                                                                                                  \
        return kb ? launch_s<S_, true>(plan, L, ws, planes, vis_out, scale, accumulate, xf_lr0, st)           \
                  : launch_s<S_, false>(plan, L, ws, planes, vis_out, scale, accumulate, xf_lr0, st);
    switch (plan->geom.support) {
        WS_DG_CASE(1) WS_DG_CASE(3) WS_DG_CASE(5) WS_DG_CASE(7) WS_DG_CASE(9) WS_DG_CASE(11) WS_DG_CASE(13) WS_DG_CASE(15)
    }
#undef WS_DG_CASE
    return WS_ERR_UNSUPPORTED;
}
