// Host side of libwstack: the C ABI of include/wstack.h.  Argument validation, the workspace carve-up, the
// fp64 per-channel constants of the position rule (O1), the cuFFT plan for a3
// and the sequencing of the kernels in ws_bin.cu / ws_grid.cu / ws_wcorrect.cu.  No device arithmetic here.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "ws_internal.h"

namespace {

constexpr double C_LIGHT = 299792458.0;
constexpr double PI = 3.14159265358979323846264338327950288;
constexpr int64_t MAX_VIS = (int64_t)1 << 30;

// Makes the plan's device current for the duration of a call and restores the caller's afterwards: a process that holds
// plans on several devices (or whose current device simply differs) must not launch against another device's pointers.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const ws_plan* plan) {
        if (!plan) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != plan->prm.device) switched = cudaSetDevice(plan->prm.device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

int fail(ws_plan* plan, int code, const char* msg) {
    if (plan) plan->last_error = msg;
    return code;
}

int cuda_fail(ws_plan* plan, cudaError_t e, const char* where) {
    if (plan) plan->last_error = std::string(where) + ": " + cudaGetErrorString(e);
    return WS_ERR_CUDA;
}

// Workspace layout for n_vis visibilities and a record capacity.  The two histograms at the head are cleared per call.
WsLayout make_layout(const ws_plan* plan, int64_t n_vis, uint64_t rec_capacity, int64_t presum_rows = 0) {
    WsLayout L;
    const size_t nb = plan->geom.n_bins;
    const size_t A = 256;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = ws_align_up(off + bytes, A); return o; };
    L.off_counts_home = take((nb + 1) * 4);
    L.off_counts_halo = take((nb + 1) * 4);
    L.off_rec_start = take((nb + 1) * 4);
    L.off_cursor_home = take(nb * 4);
    L.off_block_sums = take(2 * ((nb + 1) / 4096 + 2) * 4);
    L.off_keys = take((size_t)n_vis * 4);
    L.off_perm = take((size_t)n_vis * 4);
    L.off_sorted_keys = take((size_t)n_vis * 4);
    L.rec_capacity = rec_capacity;
    L.item_capacity = (uint32_t)(2 * rec_capacity / WS_CHUNK + 2);   // sum of ceil(cnt/CHUNK) over bins with cnt > CHUNK
    L.off_presum = take((size_t)presum_rows * sizeof(float2));
    L.off_items = take((size_t)L.item_capacity * sizeof(uint4));
    L.off_records = take((size_t)rec_capacity * sizeof(float4));
    L.total = off;
    return L;
}

// Largest record capacity whose layout fits into `bytes` (0 if even the fixed part does not fit).
bool fit_layout(const ws_plan* plan, int64_t n_vis, size_t bytes, WsLayout* out, int64_t presum_rows = 0) {
    WsLayout L0 = make_layout(plan, n_vis, 0, presum_rows);
    if (L0.total > bytes) return false;
    const uint64_t want = (uint64_t)n_vis;                          // one record per visibility
    const size_t spare = bytes - L0.total;
    // per record: 16 B + 32/WS_CHUNK B of items; keep a page of slack for the alignment of the two regions
    uint64_t cap = spare > 1024 ? (uint64_t)((spare - 1024) / (16.0 + 32.0 / WS_CHUNK)) : 0;
    if (cap > want) cap = want;
    WsLayout L = make_layout(plan, n_vis, cap, presum_rows);
    while (L.total > bytes && cap > 0) {
        cap = cap > 64 ? cap - 64 : 0;
        L = make_layout(plan, n_vis, cap, presum_rows);
    }
    if (L.total > bytes) return false;
    *out = L;
    return true;
}

int make_fft_plan(ws_plan* plan) {
    const long long n[2] = {plan->prm.n_pix, plan->prm.n_pix};
    const size_t plane_bytes = (size_t)plan->prm.n_pix * plan->prm.n_pix * ((plan->prm.flags & WS_FLAG_MESH_F64) ? 16 : 8);
    // all planes in one batched transform unless its work area is out of proportion; else plane by plane
    for (int attempt = 0; attempt < 2; ++attempt) {
        const int batch = attempt == 0 ? plan->prm.n_wplanes : 1;
        cufftHandle h;
        if (cufftCreate(&h) != CUFFT_SUCCESS) return WS_ERR_CUFFT;
        size_t work = 0;
        if (cufftSetAutoAllocation(h, 0) != CUFFT_SUCCESS ||
            cufftMakePlanMany64(h, 2, const_cast<long long*>(n), nullptr, 1, 0, nullptr, 1, 0,
                                (plan->prm.flags & WS_FLAG_MESH_F64) ? CUFFT_Z2Z : CUFFT_C2C, batch, &work) != CUFFT_SUCCESS) {
            cufftDestroy(h);
            if (attempt == 0) continue;
            return WS_ERR_CUFFT;
        }
        if (attempt == 0 && batch > 1 && work > 2 * plane_bytes + (64u << 20)) {
            cufftDestroy(h);
            continue;
        }
        plan->fft = h;
        plan->fft_ok = true;
        plan->fft_work_bytes = work;
        plan->fft_batch = batch;
        return WS_OK;
    }
    return WS_ERR_CUFFT;
}

// Continuous Fourier transform of the 1-D convolution function at xi cycles per cell (WS_NORM_TAPER, wstack.h).
double kernel_taper(const ws_params& p, double xi) {
    if (p.kernel_type == WS_KERNEL_KAISER_BESSEL) {
        const double beta = p.kernel_param, a = PI * (double)p.support * xi, d = beta * beta - a * a;
        double f = 1.0;
        if (d > 1e-12) f = std::sinh(std::sqrt(d)) / std::sqrt(d);
        else if (d < -1e-12) f = std::sin(std::sqrt(-d)) / std::sqrt(-d);
        return f * beta / std::sinh(beta);
    }
    return std::exp(-2.0 * PI * PI * p.kernel_param * p.kernel_param * xi * xi);
}

// Tap constants of the gridder.  Gaussian: g(x) = norm1 2^(tap_c x^2).  Kaiser-Bessel: I0(beta sqrt(y)) as its power
// series in y = 1 - (2x/S)^2, scaled by 1/I0(beta) so that the fp32 Horner sum stays in (0, 1]; every coefficient is
// positive, so the sum has no cancellation.  Terms are kept until the tail is below 1e-9 of the peak.
int make_taps(const ws_params& p, WsGeom& g) {
    std::memset(g.kb_c, 0, sizeof(g.kb_c));
    g.kb_terms = 0;
    g.kb_y = 0.f;
    if (p.kernel_type == WS_KERNEL_GAUSSIAN) {
        const double sigma = p.kernel_param;
        g.tap_c = (float)(-1.4426950408889634 / (2.0 * sigma * sigma));
        g.norm2 = (float)(1.0 / (2.0 * PI * sigma * sigma));
        return WS_OK;
    }
    const double beta = p.kernel_param, q = 0.25 * beta * beta, S = (double)p.support;
    if (beta > 24.0) return WS_ERR_UNSUPPORTED;
    double c[WS_KB_MAX_TERMS + 64], sum = 0.0;
    const int n_all = WS_KB_MAX_TERMS + 64;
    c[0] = 1.0;
    for (int k = 1; k < n_all; ++k) c[k] = c[k - 1] * q / ((double)k * (double)k);
    for (int k = 0; k < n_all; ++k) sum += c[k];          // = I0(beta) to fp64 accuracy (k up to 112 >> beta)
    double tail = 0.0;
    int terms = n_all;
    while (terms > 1 && tail + c[terms - 1] < 1e-9 * sum) tail += c[--terms];
    if (terms > WS_KB_MAX_TERMS) return WS_ERR_UNSUPPORTED;
    for (int k = 0; k < terms; ++k) g.kb_c[k] = (float)(c[k] / sum);
    g.kb_terms = terms;
    g.kb_y = (float)(4.0 / (S * S));
    g.tap_c = 0.f;
    const double norm1 = beta / (S * std::sinh(beta)) * sum;   // g(x) = norm1 * (series / I0(beta))
    g.norm2 = (float)(norm1 * norm1);
    return WS_OK;
}

}  // namespace

// Bytes of workspace a1 + a2 need for n_vis visibilities (the layout alone, with fit_layout's alignment margin; no FFT
// work area): what ws_grid_visibilities_static (ws_static.cu) holds against the size of its static array.
size_t ws_bin_layout_bytes(const ws_plan* plan, int64_t n_vis, int64_t presum_rows) {
    return make_layout(plan, n_vis, (uint64_t)n_vis + 64, presum_rows).total + 4096;
}

extern "C" {

int ws_version(void) { return WS_VERSION; }

const char* ws_strerror(int code) {
    switch (code) {
        case WS_OK: return "ok";
        case WS_ERR_INVALID_ARG: return "invalid argument";
        case WS_ERR_UNSUPPORTED: return "unsupported configuration";
        case WS_ERR_WORKSPACE: return "workspace too small";
        case WS_ERR_CUDA: return "CUDA error";
        case WS_ERR_CUFFT: return "cuFFT error";
    }
    return "unknown error";
}

const char* ws_last_error(const ws_plan* plan) { return plan ? plan->last_error.c_str() : ""; }

int ws_plan_create(const ws_params* p, ws_plan** out) {
    if (!out) return WS_ERR_INVALID_ARG;
    *out = nullptr;
    if (!p) return WS_ERR_INVALID_ARG;
    if (p->n_pix <= 0 || p->n_wplanes <= 0 || p->support <= 0 || (p->support & 1) == 0) return WS_ERR_INVALID_ARG;
    if (!(p->kernel_param > 0.0) || !(p->cell_rad > 0.0) || !(p->w_max > p->w_min)) return WS_ERR_INVALID_ARG;
    if (!std::isfinite(p->w_min) || !std::isfinite(p->w_max) || !std::isfinite(p->cell_rad)) return WS_ERR_INVALID_ARG;
    if ((p->flags & ~(uint32_t)(WS_FLAG_LIBRARY_FFT | WS_FLAG_NO_TRANSPOSE | WS_FLAG_TRACK_SUMWT | WS_FLAG_PRESUM_CHANNELS |
                                WS_FLAG_MESH_F64)) != 0 ||
        p->device < 0)
        return WS_ERR_INVALID_ARG;
    if (!std::isfinite(p->kernel_param)) return WS_ERR_INVALID_ARG;
    if (p->support > 2 * WS_HALO_MAX + 1) return WS_ERR_UNSUPPORTED;
    if (p->kernel_type != WS_KERNEL_GAUSSIAN && p->kernel_type != WS_KERNEL_KAISER_BESSEL) return WS_ERR_UNSUPPORTED;
    if (p->tile != 0 && p->tile != WS_TILE) return WS_ERR_UNSUPPORTED;
    if (p->n_pix % (2 * WS_TILE) != 0 || p->n_pix > 32768) return WS_ERR_INVALID_ARG;
    const uint64_t nt = (uint64_t)p->n_pix / WS_TILE;
    if (nt * nt * (uint64_t)p->n_wplanes >= 0xFFFFFFFFull / 2) return WS_ERR_UNSUPPORTED;

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || p->device >= n_dev) return WS_ERR_CUDA;
    if (cudaSetDevice(p->device) != cudaSuccess) return WS_ERR_CUDA;
    ws_plan* plan = new (std::nothrow) ws_plan();
    if (!plan) return WS_ERR_CUDA;
    plan->prm = *p;
    plan->prm.tile = WS_TILE;
    WsGeom& g = plan->geom;
    g.n_pix = p->n_pix;
    g.n_wplanes = p->n_wplanes;
    g.support = p->support;
    g.halo = (p->support - 1) / 2;
    g.plane_lo = 0;
    g.plane_hi = p->n_wplanes;
    g.nt = (int32_t)nt;
    g.n_bins = (uint32_t)(nt * nt * (uint64_t)p->n_wplanes);
    const int taps_rc = make_taps(*p, g);
    if (taps_rc != WS_OK) {
        delete plan;
        return taps_rc;
    }
    plan->fft_ok = false;
    plan->d_sumwt = nullptr;
    plan->d_taper = nullptr;
    plan->last_weights = nullptr;
    plan->snapshot_rows = 0;
    plan->last_has_values = false;
    plan->last_chan_per_key = 1;
    plan->launches = 0;
    plan->last_valid = false;
    plan->sorted_keys_valid = false;
    plan->sticky_status = WS_OK;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) {
        delete plan;
        return WS_ERR_CUDA;
    }
    plan->sm_count = prop.multiProcessorCount;
    plan->d_status = nullptr;
    plan->last_ws = nullptr;
    {   // 1 / ghat per image column (= per row: the kernel is separable and the image square), fp64 on the host
        std::vector<float> inv_taper((size_t)p->n_pix);
        for (int i = 0; i < p->n_pix; ++i)
            inv_taper[(size_t)i] = (float)(1.0 / kernel_taper(*p, (double)(i - p->n_pix / 2) / (double)p->n_pix));
        if (cudaMalloc((void**)&plan->d_status, sizeof(WsStatus)) != cudaSuccess ||
            cudaMemset(plan->d_status, 0, sizeof(WsStatus)) != cudaSuccess ||
            cudaMalloc((void**)&plan->d_sumwt, 16) != cudaSuccess || cudaMemset(plan->d_sumwt, 0, 16) != cudaSuccess ||
            cudaMalloc((void**)&plan->d_taper, inv_taper.size() * 4) != cudaSuccess ||
            cudaMemcpy(plan->d_taper, inv_taper.data(), inv_taper.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
            if (plan->d_status) cudaFree(plan->d_status);
            if (plan->d_sumwt) cudaFree(plan->d_sumwt);
            if (plan->d_taper) cudaFree(plan->d_taper);
            delete plan;
            return WS_ERR_CUDA;
        }
    }
    // a3: the FFT of ws_fft.cu where it exists (N = 2^8 .. 2^13), else (or on request) the library's
    plan->fft_own = !(p->flags & (WS_FLAG_LIBRARY_FFT | WS_FLAG_MESH_F64)) && ws_fft_own_supported(p->n_pix, p->n_wplanes);
    plan->e2e_ready = false;
    plan->e2e_chunk_bytes = 0;
    plan->d_twiddles = nullptr;
    plan->d_masks = nullptr;
    plan->mask_words = 0;
    plan->occ_grid = nullptr;
    plan->occ_sparse = false;
    int rc = make_fft_plan(plan);                       // ws_fft_planes is always the library's
    if (rc == WS_OK && plan->fft_own) rc = ws_fft_own_init(plan);
    plan->fft_rows1d_ok = false;
    plan->fft_rows1d_work = 0;
    if (rc == WS_OK && plan->fft_own) {                 // degridding fast path: every row of the stack along u in one batch
        long long n1[1] = {p->n_pix};
        size_t work = 0;
        cufftHandle h;
        if (cufftCreate(&h) == CUFFT_SUCCESS) {
            if (cufftSetAutoAllocation(h, 0) == CUFFT_SUCCESS &&
                cufftMakePlanMany64(h, 1, n1, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C,
                                    (long long)p->n_pix * (long long)p->n_wplanes, &work) == CUFFT_SUCCESS) {
                plan->fft_rows1d = h;                   // (its work area, a few bytes per row, comes from the workspace's end)
                plan->fft_rows1d_work = work;
                plan->fft_rows1d_ok = true;
            } else {
                cufftDestroy(h);
            }
        }
    }
    if (rc != WS_OK) {
        if (plan->fft_rows1d_ok) cufftDestroy(plan->fft_rows1d);
        if (plan->fft_ok) cufftDestroy(plan->fft);
        if (plan->d_twiddles) cudaFree(plan->d_twiddles);
        if (plan->d_masks) cudaFree(plan->d_masks);
        cudaFree(plan->d_status);
        cudaFree(plan->d_sumwt);
        cudaFree(plan->d_taper);
        delete plan;
        return rc;
    }
    *out = plan;
    return WS_OK;
}

int ws_plan_destroy(ws_plan* plan) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (plan->e2e_ready) {
        cudaStreamDestroy(plan->copy_stream);
        cudaEventDestroy(plan->ev_start);
        cudaEventDestroy(plan->ev_orient);
        cudaFreeHost(plan->h_orient);
        for (int i = 0; i < WS_E2E_MAX_CHUNKS; ++i) cudaEventDestroy(plan->ev_chunk[i]);
    }
    if (plan->fft_ok) cufftDestroy(plan->fft);
    if (plan->fft_rows1d_ok) cufftDestroy(plan->fft_rows1d);
    if (plan->d_status) cudaFree(plan->d_status);
    if (plan->d_sumwt) cudaFree(plan->d_sumwt);
    if (plan->d_taper) cudaFree(plan->d_taper);
    if (plan->d_twiddles) cudaFree(plan->d_twiddles);
    if (plan->d_masks) cudaFree(plan->d_masks);
    delete plan;
    return WS_OK;
}

int ws_plan_set_snapshot_rows(ws_plan* plan, int64_t rows_per_snapshot) {
    if (!plan) return WS_ERR_INVALID_ARG;
    if (rows_per_snapshot < 0 || rows_per_snapshot > MAX_VIS)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_plan_set_snapshot_rows: bad count");
    plan->snapshot_rows = rows_per_snapshot;
    return WS_OK;
}

int ws_plan_set_plane_range(ws_plan* plan, int32_t plane_lo, int32_t plane_hi) {
    if (!plan) return WS_ERR_INVALID_ARG;
    if (plane_lo < 0 || plane_hi > plan->prm.n_wplanes || plane_lo >= plane_hi)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_plan_set_plane_range: need 0 <= plane_lo < plane_hi <= n_wplanes");
    plan->geom.plane_lo = plane_lo;
    plan->geom.plane_hi = plane_hi;
    return WS_OK;
}

int ws_plan_set_e2e_chunk_bytes(ws_plan* plan, size_t bytes) {
    if (!plan) return WS_ERR_INVALID_ARG;
    plan->e2e_chunk_bytes = bytes;
    return WS_OK;
}

static inline size_t f64_factor(const ws_plan* plan) { return (plan->prm.flags & WS_FLAG_MESH_F64) ? 2 : 1; }
static inline bool is_f64(const ws_plan* plan) { return (plan->prm.flags & WS_FLAG_MESH_F64) != 0; }
size_t ws_grid_bytes(const ws_plan* plan) {
    return plan ? f64_factor(plan) * 8 * plan->prm.n_pix * plan->prm.n_pix * plan->prm.n_wplanes : 0;
}
size_t ws_image_bytes(const ws_plan* plan) { return plan ? f64_factor(plan) * 8 * plan->prm.n_pix * plan->prm.n_pix : 0; }
size_t ws_dirty_bytes(const ws_plan* plan) { return plan ? f64_factor(plan) * 4 * plan->prm.n_pix * plan->prm.n_pix : 0; }
size_t ws_fft_workspace_bytes(const ws_plan* plan) { return plan ? plan->fft_work_bytes : 0; }
int ws_plan_tile(const ws_plan* plan) { return plan ? WS_TILE : 0; }
int ws_plan_fft_is_own(const ws_plan* plan) { return plan && plan->fft_own ? 1 : 0; }
int64_t ws_plan_n_bins(const ws_plan* plan) { return plan ? (int64_t)plan->geom.n_bins : 0; }

size_t ws_workspace_bytes_for(const ws_plan* plan, int64_t max_vis, double dup_factor) {
    if (!plan || max_vis < 0 || max_vis > MAX_VIS) return 0;
    (void)dup_factor;      // one record per visibility since round 2 (the gridder carries a ring instead of copies)
    const uint64_t cap = (uint64_t)max_vis + 64;
    const bool presum = (plan->prm.flags & WS_FLAG_PRESUM_CHANNELS) != 0;          // sized for n_chan = 1, the worst case
    const size_t a = make_layout(plan, max_vis, cap, presum ? max_vis : 0).total + 4096 +   // slack for fit_layout's alignment margin
                     ws_align_up(plan->fft_rows1d_work, 256) + 256;                         // ws_predict_visibilities' row transforms
    return a > plan->fft_work_bytes ? a : plan->fft_work_bytes;
}

size_t ws_workspace_bytes(const ws_plan* plan, int64_t max_vis) { return ws_workspace_bytes_for(plan, max_vis, 1.0); }

int ws_grid_zero(ws_plan* plan, void* grid, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !grid) return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_zero: null argument");
    int rc = ws_launch_zero(plan, grid, ws_grid_bytes(plan), (cudaStream_t)stream);
    if (rc >= 0) rc = ws_launch_fft_masks_clear(plan, (cudaStream_t)stream);
    if (rc >= 0 && cudaMemsetAsync(plan->d_sumwt, 0, sizeof(double), (cudaStream_t)stream) != cudaSuccess) rc = WS_ERR_CUDA;
    if (rc < 0) return fail(plan, rc, "ws_grid_zero: memset failed");
    plan->occ_grid = grid;                               // an empty mesh: the occupancy masks describe it
    plan->occ_sparse = false;
    return WS_OK;
}

// O1: per-channel constants, fp64, in exactly this operation order (the bit-exact bin contract)
static int make_chan_consts(ws_plan* plan, const double* freq_hz, int32_t n_chan, WsChanConsts& cc) {
    const ws_params& P = plan->prm;
    std::memset(&cc, 0, sizeof(cc));
    const double dw = (P.w_max - P.w_min) / (double)P.n_wplanes;
    for (int c = 0; c < n_chan; ++c) {
        if (freq_hz) {
            if (!(freq_hz[c] > 0.0) || !std::isfinite(freq_hz[c]))
                return fail(plan, WS_ERR_INVALID_ARG, "ws_bin_visibilities: bad frequency");
            cc.su[c] = (freq_hz[c] / C_LIGHT) * ((double)P.n_pix * P.cell_rad);
            cc.sw[c] = (freq_hz[c] / C_LIGHT) / dw;
        } else {
            cc.su[c] = (double)P.n_pix * P.cell_rad;
            cc.sw[c] = 1.0 / dw;
        }
    }
    cc.ow = -P.w_min / dw;
    cc.half = (double)(P.n_pix / 2);
    return WS_OK;
}

// a1 for the gridder (with_values) and for the degridder (positions only: vis and weights are not read)
static int bin_impl(ws_plan* plan, const float* uvw, const void* vis, const float* weights, const double* freq_hz,
                    int64_t n_rows, int32_t n_chan, void* workspace, size_t workspace_bytes, void* stream, bool with_values) {
    if (!plan) return WS_ERR_INVALID_ARG;
    if (is_f64(plan)) return fail(plan, WS_ERR_UNSUPPORTED, "WS_FLAG_MESH_F64: nothing is binned (ws_grid_visibilities grids directly); no degridding");
    if (n_rows < 0 || n_chan <= 0) return fail(plan, WS_ERR_INVALID_ARG, "ws_bin_visibilities: bad n_rows / n_chan");
    if (n_chan > WS_MAX_CHAN) return fail(plan, WS_ERR_UNSUPPORTED, "ws_bin_visibilities: n_chan > 128");
    if (n_rows > MAX_VIS || n_rows * n_chan > MAX_VIS)
        return fail(plan, WS_ERR_UNSUPPORTED, "ws_bin_visibilities: more than 2^30 visibilities in one call");
    if (!with_values) vis = nullptr, weights = nullptr;
    if (!workspace || (n_rows > 0 && (!uvw || (with_values && (!vis || !weights)))))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_bin_visibilities: null pointer");
    if (((uintptr_t)uvw | (uintptr_t)vis | (uintptr_t)weights | (uintptr_t)workspace) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_bin_visibilities: pointers must be 16-byte aligned");
    // WS_FLAG_PRESUM_CHANNELS: the rows are what is binned, each carrying sum_c weight * vis
    const bool presum = with_values && (plan->prm.flags & WS_FLAG_PRESUM_CHANNELS) != 0;
    if (presum && freq_hz)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_bin_visibilities: WS_FLAG_PRESUM_CHANNELS needs freq_hz == NULL (shared uvw)");
    const int64_t n_vis = presum ? n_rows : n_rows * n_chan;
    const int32_t n_chan_in = n_chan;
    WsLayout L;
    if (!fit_layout(plan, n_vis, workspace_bytes, &L, presum ? n_rows : 0) ||
        (n_vis > 0 && L.rec_capacity < (uint64_t)n_vis))
        return fail(plan, WS_ERR_WORKSPACE, "ws_bin_visibilities: workspace too small (see ws_workspace_bytes_for)");
    const void* vis_in = vis;
    const float* wt_in = weights;
    if (presum) {
        float2* sums = (float2*)((char*)workspace + L.off_presum);
        const int prc = ws_launch_presum(plan, (const float2*)vis, weights, n_rows, n_chan, sums, (cudaStream_t)stream);
        if (prc < 0) return fail(plan, prc, "ws_bin_visibilities: launch failed");
        plan->launches += prc;
        vis_in = sums;
        wt_in = nullptr;
        n_chan = 1;
    }

    WsChanConsts cc;
    const int crc = make_chan_consts(plan, freq_hz, n_chan, cc);
    if (crc != WS_OK) return crc;

    plan->last_valid = false;
    plan->sorted_keys_valid = false;
    const int rc = ws_launch_bin(plan, L, (char*)workspace, cc, uvw, (const float2*)vis_in, wt_in, n_rows, n_chan,
                                 (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_bin_visibilities: launch failed");
    plan->launches += rc;
    plan->last_ws = workspace;
    plan->last_layout = L;
    plan->last_n_vis = n_vis;
    plan->last_weights = weights;
    plan->last_chan_per_key = presum ? n_chan_in : 1;
    plan->last_has_values = with_values;
    plan->last_valid = true;
    return WS_OK;
}

int ws_bin_visibilities(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                        const double* freq_hz, int64_t n_rows, int32_t n_chan, void* workspace,
                        size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    return bin_impl(plan, uvw, vis, weights, freq_hz, n_rows, n_chan, workspace, workspace_bytes, stream, true);
}

int ws_grid_binned(ws_plan* plan, void* grid, int32_t mode, void* workspace, size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!grid || !workspace) return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: null pointer");
    if (mode != WS_GRID_ACCUMULATE && mode != WS_GRID_OVERWRITE && mode != WS_GRID_SPARSE && mode != WS_GRID_SPARSE_ADD)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: bad mode");
    const bool sparse_mode = mode == WS_GRID_SPARSE || mode == WS_GRID_SPARSE_ADD;
    if (sparse_mode && !plan->fft_own)
        return fail(plan, WS_ERR_UNSUPPORTED, "ws_grid_binned: WS_GRID_SPARSE needs the own FFT (N = 2^8..2^14, no WS_FLAG_LIBRARY_FFT)");
    if ((uintptr_t)grid & 15) return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: grid must be 16-byte aligned");
    if (!plan->last_valid || !plan->last_has_values || plan->last_ws != workspace || plan->last_layout.total > workspace_bytes)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: workspace does not hold the bins of ws_bin_visibilities");
    if (mode == WS_GRID_ACCUMULATE && plan->occ_sparse && plan->occ_grid == grid)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: cannot accumulate onto a WS_GRID_SPARSE mesh (its empty tiles were never written): use WS_GRID_SPARSE_ADD");
    if (mode == WS_GRID_SPARSE_ADD && !(plan->occ_sparse && plan->occ_grid == grid))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_binned: WS_GRID_SPARSE_ADD needs a mesh this plan wrote with WS_GRID_SPARSE");
    cudaStream_t st = (cudaStream_t)stream;
    // Tile occupancy of the mesh, for the sparse FFT passes: restarted by OVERWRITE / SPARSE, OR-ed by ACCUMULATE /
    // SPARSE_ADD.  It comes BEFORE the gridding kernel -- a SPARSE mesh is stored in the orientation the masks favour --
    // except for SPARSE_ADD, whose kernel must see the occupancy of the EARLIER chunks to know which tiles to add to.
    int rc;
    auto update_masks = [&]() -> int {
        if (!plan->d_masks) return WS_OK;
        if (mode == WS_GRID_OVERWRITE || mode == WS_GRID_SPARSE) {
            if (ws_launch_fft_masks_clear(plan, st) < 0) return fail(plan, WS_ERR_CUDA, "ws_grid_binned: mask clear failed");
            plan->occ_grid = grid;
            plan->occ_sparse = mode == WS_GRID_SPARSE;
        }
        if (plan->occ_grid == grid) {
            const int r = ws_launch_fft_masks(plan, (const uint32_t*)((char*)workspace + plan->last_layout.off_rec_start),
                                              mode == WS_GRID_SPARSE ? 1 : (mode == WS_GRID_OVERWRITE ? 0 : -1), st);
            if (r < 0) return fail(plan, r, "ws_grid_binned: launch failed");
            plan->launches += r;
        } else {
            plan->occ_grid = nullptr;                    // accumulation onto a mesh this plan has no record of
        }
        return WS_OK;
    };
    if (mode != WS_GRID_SPARSE_ADD && (rc = update_masks()) != WS_OK) return rc;
    if (plan->prm.flags & WS_FLAG_TRACK_SUMWT) {
        if ((mode == WS_GRID_OVERWRITE || mode == WS_GRID_SPARSE) &&
            cudaMemsetAsync(plan->d_sumwt, 0, sizeof(double), st) != cudaSuccess)
            return fail(plan, WS_ERR_CUDA, "ws_grid_binned: memset failed");
        rc = ws_launch_sum_weights(plan, plan->last_layout, (char*)workspace, plan->last_weights,
                                   plan->last_n_vis * plan->last_chan_per_key, plan->last_chan_per_key, st);
        if (rc < 0) return fail(plan, rc, "ws_grid_binned: launch failed");
        plan->launches += rc;
    }
    rc = ws_launch_grid(plan, plan->last_layout, (char*)workspace, (float2*)grid, mode, st);
    if (rc < 0) return fail(plan, rc, "ws_grid_binned: launch failed");
    plan->launches += rc;
    if (mode == WS_GRID_SPARSE_ADD && (rc = update_masks()) != WS_OK) return rc;
    return WS_OK;
}

int ws_grid_visibilities(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                         const double* freq_hz, int64_t n_rows, int32_t n_chan, void* grid, int32_t mode,
                         void* workspace, size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!grid) return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: null pointer");
    if (mode != WS_GRID_ACCUMULATE && mode != WS_GRID_OVERWRITE && mode != WS_GRID_SPARSE && mode != WS_GRID_SPARSE_ADD)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: bad mode");
    if (is_f64(plan)) {    // fp64 mesh: one thread per measurement, atomicAdd on the mesh (ws_f64.cu); nothing is binned
        if (mode != WS_GRID_ACCUMULATE && mode != WS_GRID_OVERWRITE)
            return fail(plan, WS_ERR_UNSUPPORTED, "ws_grid_visibilities: WS_FLAG_MESH_F64 grids with WS_GRID_ACCUMULATE or WS_GRID_OVERWRITE");
        if (n_rows < 0 || n_chan <= 0 || n_chan > WS_MAX_CHAN || n_rows > MAX_VIS || n_rows * n_chan > MAX_VIS)
            return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: bad n_rows / n_chan");
        if (n_rows > 0 && (!uvw || !vis || !weights)) return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: null pointer");
        if (((uintptr_t)uvw | (uintptr_t)vis | (uintptr_t)weights | (uintptr_t)grid) & 15)
            return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: pointers must be 16-byte aligned");
        const bool presum = (plan->prm.flags & WS_FLAG_PRESUM_CHANNELS) != 0;
        if (presum && freq_hz)
            return fail(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities: WS_FLAG_PRESUM_CHANNELS needs freq_hz == NULL (shared uvw)");
        WsChanConsts cc;
        int rc = make_chan_consts(plan, freq_hz, n_chan, cc);
        if (rc != WS_OK) return rc;
        cudaStream_t st = (cudaStream_t)stream;
        if (mode == WS_GRID_OVERWRITE) {
            if (cudaMemsetAsync(grid, 0, ws_grid_bytes(plan), st) != cudaSuccess ||
                cudaMemsetAsync(plan->d_sumwt, 0, sizeof(double), st) != cudaSuccess)
                return fail(plan, WS_ERR_CUDA, "ws_grid_visibilities: memset failed");
        }
        plan->last_valid = false;
        rc = ws_launch_grid_f64(plan, cc, uvw, (const float2*)vis, weights, n_rows, n_chan, presum ? 1 : 0, (double*)grid, st);
        if (rc < 0) return fail(plan, rc, "ws_grid_visibilities: launch failed");
        plan->launches += rc;
        return WS_OK;
    }
    const int rc = ws_bin_visibilities(plan, uvw, vis, weights, freq_hz, n_rows, n_chan, workspace, workspace_bytes, stream);
    if (rc != WS_OK) return rc;
    return ws_grid_binned(plan, grid, mode, workspace, workspace_bytes, stream);
}

static int fft_planes_dir(ws_plan* plan, void* grid, void* workspace, size_t workspace_bytes, void* stream, int direction) {
    if (!plan || !grid) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_planes: null argument");
    if ((uintptr_t)grid & 15) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_planes: grid must be 16-byte aligned");
    if (plan->fft_work_bytes > 0 && (!workspace || workspace_bytes < plan->fft_work_bytes))
        return fail(plan, WS_ERR_WORKSPACE, "ws_fft_planes: workspace smaller than ws_fft_workspace_bytes");
    if (cufftSetStream(plan->fft, (cudaStream_t)stream) != CUFFT_SUCCESS)
        return fail(plan, WS_ERR_CUFFT, "ws_fft_planes: cufftSetStream");
    if (plan->fft_work_bytes > 0 && cufftSetWorkArea(plan->fft, workspace) != CUFFT_SUCCESS)
        return fail(plan, WS_ERR_CUFFT, "ws_fft_planes: cufftSetWorkArea");
    // the records of the last grid call share the workspace with the FFT work area
    plan->last_valid = plan->last_valid && plan->fft_work_bytes == 0;
    const size_t plane = (size_t)plan->prm.n_pix * plan->prm.n_pix;
    for (int k = 0; k < plan->prm.n_wplanes; k += plan->fft_batch) {
        if (is_f64(plan)) {
            cufftDoubleComplex* p = (cufftDoubleComplex*)grid + (size_t)k * plane;
            if (cufftExecZ2Z(plan->fft, p, p, direction) != CUFFT_SUCCESS)
                return fail(plan, WS_ERR_CUFFT, "ws_fft_planes: cufftExecZ2Z");
            continue;
        }
        cufftComplex* p = (cufftComplex*)grid + (size_t)k * plane;
        if (cufftExecC2C(plan->fft, p, p, direction) != CUFFT_SUCCESS)
            return fail(plan, WS_ERR_CUFFT, "ws_fft_planes: cufftExecC2C");
    }
    return WS_OK;
}

int ws_fft_planes(ws_plan* plan, void* grid, void* workspace, size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    return fft_planes_dir(plan, grid, workspace, workspace_bytes, stream, CUFFT_INVERSE);
}

int ws_predict_planes(ws_plan* plan, const void* model_image, void* planes, void* workspace, size_t workspace_bytes,
                      void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !model_image || !planes) return fail(plan, WS_ERR_INVALID_ARG, "ws_predict_planes: null argument");
    if (is_f64(plan)) return fail(plan, WS_ERR_UNSUPPORTED, "ws_predict_planes: no degridding with WS_FLAG_MESH_F64");
    if (((uintptr_t)model_image | (uintptr_t)planes) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_predict_planes: pointers must be 16-byte aligned");
    if (plan->fft_work_bytes > 0 && (!workspace || workspace_bytes < plan->fft_work_bytes))
        return fail(plan, WS_ERR_WORKSPACE, "ws_predict_planes: workspace smaller than ws_fft_workspace_bytes");
    if (plan->occ_grid == planes) plan->occ_grid = nullptr;      // no longer a mesh the gridder filled
    const int rc = ws_launch_wscreen_fwd(plan, (const float2*)model_image, (float2*)planes, 0, (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_predict_planes: launch failed");
    plan->launches += rc;
    return fft_planes_dir(plan, planes, workspace, workspace_bytes, stream, CUFFT_FORWARD);
}

int ws_degrid_visibilities(ws_plan* plan, const float* uvw, const double* freq_hz, int64_t n_rows, int32_t n_chan,
                           const void* planes, void* vis_out, float scale, int32_t accumulate, void* workspace,
                           size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!planes || (n_rows > 0 && !vis_out)) return fail(plan, WS_ERR_INVALID_ARG, "ws_degrid_visibilities: null pointer");
    if (accumulate != 0 && accumulate != 1) return fail(plan, WS_ERR_INVALID_ARG, "ws_degrid_visibilities: bad flag");
    if (((uintptr_t)planes | (uintptr_t)vis_out) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_degrid_visibilities: pointers must be 16-byte aligned");
    int rc = bin_impl(plan, uvw, nullptr, nullptr, freq_hz, n_rows, n_chan, workspace, workspace_bytes, stream, false);
    if (rc != WS_OK) return rc;
    if (n_rows == 0) return WS_OK;
    if (!accumulate &&
        cudaMemsetAsync(vis_out, 0, (size_t)n_rows * n_chan * 8, (cudaStream_t)stream) != cudaSuccess)   // dropped ones predict 0
        return fail(plan, WS_ERR_CUDA, "ws_degrid_visibilities: memset failed");
    rc = ws_launch_degrid(plan, plan->last_layout, (char*)workspace, (const float2*)planes, (float2*)vis_out, scale,
                          accumulate, -1, (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_degrid_visibilities: launch failed");
    plan->launches += rc;
    return WS_OK;
}

int ws_predict_visibilities(ws_plan* plan, const void* model_image, const float* uvw, const double* freq_hz, int64_t n_rows,
                            int32_t n_chan, void* planes, void* vis_out, float scale, int32_t accumulate, void* workspace,
                            size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!plan->fft_own || !plan->fft_rows1d_ok) {      // the two library calls in sequence
        const int rc = ws_predict_planes(plan, model_image, planes, workspace, workspace_bytes, stream);
        if (rc != WS_OK) return rc;
        return ws_degrid_visibilities(plan, uvw, freq_hz, n_rows, n_chan, planes, vis_out, scale, accumulate, workspace,
                                      workspace_bytes, stream);
    }
    if (!model_image || !planes || (n_rows > 0 && !vis_out))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_predict_visibilities: null pointer");
    if (accumulate != 0 && accumulate != 1) return fail(plan, WS_ERR_INVALID_ARG, "ws_predict_visibilities: bad flag");
    if (((uintptr_t)model_image | (uintptr_t)planes | (uintptr_t)vis_out) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_predict_visibilities: pointers must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    // positions first: the bins say which column bands of the planes the gather will read
    int rc = bin_impl(plan, uvw, nullptr, nullptr, freq_hz, n_rows, n_chan, workspace, workspace_bytes, stream, false);
    if (rc != WS_OK) return rc;
    if (n_rows == 0) return WS_OK;
    const WsLayout& L = plan->last_layout;
    // the work area of the row transforms sits at the end of the workspace, behind the bins
    const size_t w1 = ws_align_up(plan->fft_rows1d_work, 256);
    if (L.total + w1 + 256 > workspace_bytes)
        return fail(plan, WS_ERR_WORKSPACE, "ws_predict_visibilities: workspace too small (see ws_workspace_bytes)");
    void* work1 = (char*)workspace + ((workspace_bytes - w1) & ~(size_t)255);
    rc = ws_launch_fft_masks_degrid(plan, (const uint32_t*)((char*)workspace + L.off_counts_home), st);
    if (rc < 0) return fail(plan, rc, "ws_predict_visibilities: launch failed");
    plan->launches += rc;
    plan->occ_grid = nullptr;                            // the masks no longer describe a gridded mesh
    plan->occ_sparse = false;
    // conj(M screen) -> inverse transforms (cuFFT along u, own column passes on the wanted bands) = conj(forward transform)
    rc = ws_launch_wscreen_fwd(plan, (const float2*)model_image, (float2*)planes, 1, st);
    if (rc < 0) return fail(plan, rc, "ws_predict_visibilities: launch failed");
    plan->launches += rc;
    if (cufftSetStream(plan->fft_rows1d, st) != CUFFT_SUCCESS ||
        (plan->fft_rows1d_work > 0 && cufftSetWorkArea(plan->fft_rows1d, work1) != CUFFT_SUCCESS) ||
        cufftExecC2C(plan->fft_rows1d, (cufftComplex*)planes, (cufftComplex*)planes, CUFFT_INVERSE) != CUFFT_SUCCESS)
        return fail(plan, WS_ERR_CUFFT, "ws_predict_visibilities: cufftExecC2C");
    rc = ws_launch_fft_cols(plan, (float2*)planes, true, st);
    if (rc < 0) return fail(plan, rc, "ws_predict_visibilities: launch failed");
    plan->launches += rc;
    if (!accumulate && cudaMemsetAsync(vis_out, 0, (size_t)n_rows * n_chan * 8, st) != cudaSuccess)
        return fail(plan, WS_ERR_CUDA, "ws_predict_visibilities: memset failed");
    int lr0 = 0;
    while ((256 << lr0) < plan->prm.n_pix) ++lr0;
    rc = ws_launch_degrid(plan, L, (char*)workspace, (const float2*)planes, (float2*)vis_out, scale, accumulate, lr0, st);
    if (rc < 0) return fail(plan, rc, "ws_predict_visibilities: launch failed");
    plan->launches += rc;
    return WS_OK;
}

int ws_wcorrect_accumulate(ws_plan* plan, const void* planes, void* image, int32_t accumulate, float* dirty,
                           void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !planes || !image) return fail(plan, WS_ERR_INVALID_ARG, "ws_wcorrect_accumulate: null argument");
    if (accumulate != 0 && accumulate != 1) return fail(plan, WS_ERR_INVALID_ARG, "ws_wcorrect_accumulate: bad flag");
    if (((uintptr_t)planes | (uintptr_t)image | (uintptr_t)dirty) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_wcorrect_accumulate: pointers must be 16-byte aligned");
    const int rc = is_f64(plan) ? ws_launch_wcorrect_f64(plan, planes, image, accumulate, dirty, (cudaStream_t)stream)
                                : ws_launch_wcorrect(plan, (const float2*)planes, (float2*)image, accumulate, dirty, (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_wcorrect_accumulate: launch failed");
    plan->launches += rc;
    return WS_OK;
}

// 0 = dense, 1 = sparse, negative = error
static int fft_sparse_flag(ws_plan* plan, const void* grid, uint32_t fft_flags, const char* who) {
    if (fft_flags & ~(uint32_t)WS_FFT_USE_OCCUPANCY) return fail(plan, WS_ERR_INVALID_ARG, who);
    if (!(fft_flags & WS_FFT_USE_OCCUPANCY)) return 0;
    if (!plan->d_masks || plan->occ_grid != grid) return fail(plan, WS_ERR_INVALID_ARG, who);
    return 1;
}

int ws_fft_columns(ws_plan* plan, void* grid, uint32_t fft_flags, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !grid) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_columns: null argument");
    if ((uintptr_t)grid & 15) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_columns: grid must be 16-byte aligned");
    if (!plan->fft_own) return fail(plan, WS_ERR_UNSUPPORTED, "ws_fft_columns: this plan uses the library FFT");
    const int sparse = fft_sparse_flag(plan, grid, fft_flags, "ws_fft_columns: bad fft_flags, or no occupancy recorded for this mesh");
    if (sparse < 0) return sparse;
    const int rc = ws_launch_fft_cols(plan, (float2*)grid, sparse != 0, (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_fft_columns: launch failed");
    plan->launches += rc;
    return WS_OK;
}

int ws_fft_rows_wcorrect(ws_plan* plan, const void* grid, void* image, int32_t accumulate, float* dirty,
                         uint32_t fft_flags, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !grid || !image) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_rows_wcorrect: null argument");
    if (accumulate != 0 && accumulate != 1) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_rows_wcorrect: bad flag");
    if (((uintptr_t)grid | (uintptr_t)image | (uintptr_t)dirty) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_rows_wcorrect: pointers must be 16-byte aligned");
    if (!plan->fft_own) return fail(plan, WS_ERR_UNSUPPORTED, "ws_fft_rows_wcorrect: this plan uses the library FFT");
    const int sparse = fft_sparse_flag(plan, grid, fft_flags, "ws_fft_rows_wcorrect: bad fft_flags, or no occupancy recorded for this mesh");
    if (sparse < 0) return sparse;
    const int rc = ws_launch_fft_rows(plan, (const float2*)grid, (float2*)image, dirty, accumulate, sparse != 0, 0, 1,
                                      (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_fft_rows_wcorrect: launch failed");
    plan->launches += rc;
    return WS_OK;
}

int ws_fft_wcorrect(ws_plan* plan, void* grid, void* image, int32_t accumulate, float* dirty, uint32_t fft_flags,
                    void* workspace, size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !grid || !image) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_wcorrect: null argument");
    if (!plan->fft_own) {     // library FFT (needs a fully written mesh), then the stand-alone a4 pass
        if (fft_flags & ~(uint32_t)WS_FFT_USE_OCCUPANCY) return fail(plan, WS_ERR_INVALID_ARG, "ws_fft_wcorrect: bad fft_flags");
        const int rc = ws_fft_planes(plan, grid, workspace, workspace_bytes, stream);
        if (rc != WS_OK) return rc;
        return ws_wcorrect_accumulate(plan, grid, image, accumulate, dirty, stream);
    }
    const int rc = ws_fft_columns(plan, grid, fft_flags, stream);
    if (rc != WS_OK) return rc;
    return ws_fft_rows_wcorrect(plan, grid, image, accumulate, dirty, fft_flags, stream);
}

int ws_dirty_image(ws_plan* plan, const void* image, float* dirty, uint32_t norm_flags, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !image || !dirty) return fail(plan, WS_ERR_INVALID_ARG, "ws_dirty_image: null argument");
    if (norm_flags & ~(uint32_t)(WS_NORM_SUMWT | WS_NORM_N | WS_NORM_TAPER))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_dirty_image: unknown norm_flags");
    if ((norm_flags & WS_NORM_SUMWT) && !(plan->prm.flags & WS_FLAG_TRACK_SUMWT))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_dirty_image: WS_NORM_SUMWT needs a plan created with WS_FLAG_TRACK_SUMWT");
    if (((uintptr_t)image | (uintptr_t)dirty) & 15)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_dirty_image: pointers must be 16-byte aligned");
    const int rc = is_f64(plan) ? ws_launch_dirty_f64(plan, image, dirty, norm_flags, (cudaStream_t)stream)
                                : ws_launch_dirty(plan, (const float2*)image, dirty, norm_flags, (cudaStream_t)stream);
    if (rc < 0) return fail(plan, rc, "ws_dirty_image: launch failed");
    plan->launches += rc;
    return WS_OK;
}

int ws_get_sum_weights(ws_plan* plan, double* sum_weights, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan || !sum_weights) return fail(plan, WS_ERR_INVALID_ARG, "ws_get_sum_weights: null argument");
    if (!(plan->prm.flags & WS_FLAG_TRACK_SUMWT))
        return fail(plan, WS_ERR_INVALID_ARG, "ws_get_sum_weights: plan was not created with WS_FLAG_TRACK_SUMWT");
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_sum_weights: synchronize");
    e = cudaMemcpy(sum_weights, plan->d_sumwt, sizeof(double), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_sum_weights: copy");
    return WS_OK;
}

size_t ws_dev_inputs_bytes(int64_t n_rows, int32_t n_chan) {
    if (n_rows < 0 || n_chan <= 0) return 0;
    const size_t n_vis = (size_t)n_rows * (size_t)n_chan;
    return ws_align_up((size_t)n_rows * 12, 16) + ws_align_up(n_vis * 8, 16) + ws_align_up(n_vis * 4, 16);
}

int ws_image_from_host(ws_plan* plan, const float* uvw_h, const void* vis_h, const float* weights_h,
                       const double* freq_hz, int64_t n_rows, int32_t n_chan, void* dev_inputs,
                       size_t dev_inputs_bytes, void* grid, void* image, float* dirty_d, float* dirty_h,
                       void* workspace, size_t workspace_bytes, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!uvw_h || !vis_h || !weights_h || !dev_inputs || !grid || !image || !dirty_d || !dirty_h || !workspace)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_image_from_host: null argument");
    if (n_rows <= 0 || n_chan <= 0 || n_rows * n_chan > MAX_VIS)
        return fail(plan, WS_ERR_INVALID_ARG, "ws_image_from_host: bad sizes");
    if (is_f64(plan)) return fail(plan, WS_ERR_UNSUPPORTED, "ws_image_from_host: not with WS_FLAG_MESH_F64");
    const size_t n_vis = (size_t)n_rows * n_chan;
    // every sub-buffer starts on a 16-byte boundary (bin_impl's alignment rule): uvw | vis | weights
    const size_t b_uvw = ws_align_up((size_t)n_rows * 12, 16), b_vis = ws_align_up(n_vis * 8, 16), b_wt = n_vis * 4;
    if (dev_inputs_bytes < b_uvw + b_vis + b_wt) return fail(plan, WS_ERR_WORKSPACE, "ws_image_from_host: dev_inputs too small");
    if ((uintptr_t)dev_inputs & 15) return fail(plan, WS_ERR_INVALID_ARG, "ws_image_from_host: dev_inputs must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if (!plan->e2e_ready) {
        if ((e = cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking)) != cudaSuccess)
            return cuda_fail(plan, e, "ws_image_from_host: stream");
        bool ok = cudaEventCreateWithFlags(&plan->ev_start, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&plan->ev_orient, cudaEventDisableTiming) == cudaSuccess &&
                  cudaHostAlloc((void**)&plan->h_orient, 64, cudaHostAllocDefault) == cudaSuccess;
        for (int i = 0; i < WS_E2E_MAX_CHUNKS; ++i)
            ok = ok && cudaEventCreateWithFlags(&plan->ev_chunk[i], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) return fail(plan, WS_ERR_CUDA, "ws_image_from_host: events");
        plan->e2e_ready = true;
    }
    // Row chunks: the copy of chunk c + 1 (copy stream) runs beside the binning + gridding of chunk c (caller's stream),
    // which therefore hide under the PCIe time; what remains exposed is the last chunk's gridding, the FFT and the
    // copy out.  Chunk starts are multiples of 4 rows (16-byte alignment of every array) and of eight snapshots (the
    // snapshot-ordered walk of the binning, if the hint is set).
    const size_t total_in = (size_t)n_rows * 12 + n_vis * 12;
    const size_t chunk_bytes = plan->e2e_chunk_bytes ? plan->e2e_chunk_bytes : ((size_t)160 << 20);
    int64_t n_chunks = (int64_t)((total_in + chunk_bytes - 1) / chunk_bytes);
    n_chunks = n_chunks < 1 ? 1 : (n_chunks > WS_E2E_MAX_CHUNKS ? WS_E2E_MAX_CHUNKS : n_chunks);
    int64_t quantum = 4;
    if (plan->snapshot_rows > 0) quantum = plan->snapshot_rows * 8 % 4 == 0 ? plan->snapshot_rows * 8 : plan->snapshot_rows * 32;
    int64_t chunk_rows = (n_rows + n_chunks - 1) / n_chunks;
    chunk_rows = (chunk_rows + quantum - 1) / quantum * quantum;
    n_chunks = (n_rows + chunk_rows - 1) / chunk_rows;
    char* d = (char*)dev_inputs;
    float* uvw_d = (float*)d;
    char* vis_d = d + b_uvw;
    float* wt_d = (float*)(d + b_uvw + b_vis);
    if ((e = cudaEventRecord(plan->ev_start, st)) != cudaSuccess ||               // dev_inputs may still be read by earlier work
        (e = cudaStreamWaitEvent(plan->copy_stream, plan->ev_start, 0)) != cudaSuccess)
        return cuda_fail(plan, e, "ws_image_from_host: event");
    for (int64_t c = 0; c < n_chunks; ++c) {
        const int64_t r0 = c * chunk_rows, nr = (r0 + chunk_rows <= n_rows ? chunk_rows : n_rows - r0);
        const size_t v0 = (size_t)r0 * n_chan, nv = (size_t)nr * n_chan;
        if ((e = cudaMemcpyAsync(uvw_d + 3 * r0, uvw_h + 3 * r0, (size_t)nr * 12, cudaMemcpyHostToDevice, plan->copy_stream)) != cudaSuccess ||
            (e = cudaMemcpyAsync(vis_d + v0 * 8, (const char*)vis_h + v0 * 8, nv * 8, cudaMemcpyHostToDevice, plan->copy_stream)) != cudaSuccess ||
            (e = cudaMemcpyAsync(wt_d + v0, weights_h + v0, nv * 4, cudaMemcpyHostToDevice, plan->copy_stream)) != cudaSuccess ||
            (e = cudaEventRecord(plan->ev_chunk[c], plan->copy_stream)) != cudaSuccess)
            return cuda_fail(plan, e, "ws_image_from_host: H2D copy");
    }
    // the mesh is never cleared nor completely written where the own FFT can skip what the gridder left empty
    for (int64_t c = 0; c < n_chunks; ++c) {
        const int64_t r0 = c * chunk_rows, nr = (r0 + chunk_rows <= n_rows ? chunk_rows : n_rows - r0);
        const size_t v0 = (size_t)r0 * n_chan;
        if ((e = cudaStreamWaitEvent(st, plan->ev_chunk[c], 0)) != cudaSuccess) return cuda_fail(plan, e, "ws_image_from_host: event");
        const int mode = plan->fft_own ? (c == 0 ? WS_GRID_SPARSE : WS_GRID_SPARSE_ADD) : (c == 0 ? WS_GRID_OVERWRITE : WS_GRID_ACCUMULATE);
        const int rc = ws_grid_visibilities(plan, uvw_d + 3 * r0, vis_d + v0 * 8, wt_d + v0, freq_hz, nr, n_chan, grid, mode,
                                            workspace, workspace_bytes, stream);
        if (rc != WS_OK) return rc;
        if (c == 0 && plan->fft_own &&        // the orientation the sparse mesh took, for the copy out (read back asynchronously)
            ((e = cudaMemcpyAsync(plan->h_orient, ws_fft_orientation_flag(plan), 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
             (e = cudaEventRecord(plan->ev_orient, st)) != cudaSuccess))
            return cuda_fail(plan, e, "ws_image_from_host: orientation read");
    }
    int rc;
    const size_t N = (size_t)plan->prm.n_pix;
    const int n_parts = 8;        // (measured on Large: 4 parts 43.8 ms, 8: 43.5, 16: 45.0)
    if (plan->fft_own && N >= 8192) {     // (N >= 8192: one row position per item, items ordered by the line they produce)
        // The row pass in eight launches, each producing an eighth of the image lines: the lines of part p travel to
        // the host (copy stream) while part p + 1 is computed.  Item = v-frequency F, line (F + N/2) mod N; a
        // transposed mesh yields columns instead, copied as a strided block.
        if ((rc = ws_fft_columns(plan, grid, WS_FFT_USE_OCCUPANCY, stream)) != WS_OK) return rc;
        if (cudaEventSynchronize(plan->ev_orient) != cudaSuccess)      // (decided by the first chunk: long since known)
            return fail(plan, WS_ERR_CUDA, "ws_image_from_host: orientation read");
        const int32_t tr = *plan->h_orient;
        for (int p = 0; p < n_parts; ++p) {
            rc = ws_launch_fft_rows(plan, (const float2*)grid, (float2*)image, dirty_d, 0, true, p, n_parts, st);
            if (rc < 0) return fail(plan, rc, "ws_image_from_host: launch failed");
            plan->launches += rc;
            if ((e = cudaEventRecord(plan->ev_chunk[p], st)) != cudaSuccess ||
                (e = cudaStreamWaitEvent(plan->copy_stream, plan->ev_chunk[p], 0)) != cudaSuccess)
                return cuda_fail(plan, e, "ws_image_from_host: event");
            const size_t l0 = ((size_t)p * (N / n_parts) + N / 2) % N, nl = N / n_parts;     // lines (or columns) of this part
            if (!tr)
                e = cudaMemcpyAsync(dirty_h + l0 * N, dirty_d + l0 * N, nl * N * 4, cudaMemcpyDeviceToHost, plan->copy_stream);
            else
                e = cudaMemcpy2DAsync(dirty_h + l0, N * 4, dirty_d + l0, N * 4, nl * 4, N, cudaMemcpyDeviceToHost, plan->copy_stream);
            if (e != cudaSuccess) return cuda_fail(plan, e, "ws_image_from_host: D2H copy");
        }
        if ((e = cudaEventRecord(plan->ev_start, plan->copy_stream)) != cudaSuccess ||
            (e = cudaStreamWaitEvent(st, plan->ev_start, 0)) != cudaSuccess)
            return cuda_fail(plan, e, "ws_image_from_host: event");
        return ws_async_status(plan, stream);
    }
    if ((rc = ws_fft_wcorrect(plan, grid, image, 0, dirty_d, plan->fft_own ? WS_FFT_USE_OCCUPANCY : 0u, workspace,
                              workspace_bytes, stream)) != WS_OK)
        return rc;
    if ((e = cudaMemcpyAsync(dirty_h, dirty_d, ws_dirty_bytes(plan), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(plan, e, "ws_image_from_host: D2H copy");
    // synchronises and reads the deferred status: a record overflow means the gridder was skipped and dirty_h is garbage
    return ws_async_status(plan, stream);
}

int ws_async_status(ws_plan* plan, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_async_status: synchronize");
    WsStatus s;
    e = cudaMemcpy(&s, plan->d_status, sizeof(s), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_async_status: status read");
    if (s.overflow || s.sticky_overflow) {
        cudaMemset(&plan->d_status->sticky_overflow, 0, sizeof(uint32_t));
        return fail(plan, WS_ERR_WORKSPACE, "record capacity of the workspace exceeded: gridding was skipped");
    }
    return WS_OK;
}

int ws_get_bins(ws_plan* plan, const uint32_t** keys, const uint32_t** sorted_keys, const uint32_t** perm,
                const uint32_t** bin_start, int64_t* n_vis, int64_t* n_bins, int64_t* n_dropped,
                int64_t* n_records, void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!plan->last_valid) return fail(plan, WS_ERR_INVALID_ARG, "ws_get_bins: no bins (no grid call, or workspace reused by the FFT)");
    cudaStream_t st = (cudaStream_t)stream;
    char* ws = (char*)plan->last_ws;
    const WsLayout& L = plan->last_layout;
    if (sorted_keys && !plan->sorted_keys_valid) {
        const int rc = ws_launch_sorted_keys(plan, L, ws, st);
        if (rc < 0) return fail(plan, rc, "ws_get_bins: launch failed");
        plan->launches += rc;
        plan->sorted_keys_valid = true;
    }
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_bins: synchronize");
    WsStatus s;
    e = cudaMemcpy(&s, plan->d_status, sizeof(s), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_bins: status read");
    if (keys) *keys = (const uint32_t*)(ws + L.off_keys);
    if (sorted_keys) *sorted_keys = (const uint32_t*)(ws + L.off_sorted_keys);
    if (perm) *perm = (const uint32_t*)(ws + L.off_perm);
    if (bin_start) *bin_start = (const uint32_t*)(ws + L.off_counts_home);
    if (n_vis) *n_vis = plan->last_n_vis;
    if (n_bins) *n_bins = (int64_t)plan->geom.n_bins;
    if (n_dropped) *n_dropped = plan->last_n_vis - (int64_t)s.n_kept;
    if (n_records) *n_records = (int64_t)s.n_records;
    if (s.overflow) return fail(plan, WS_ERR_WORKSPACE, "record capacity of the workspace exceeded: gridding was skipped");
    return WS_OK;
}

int ws_get_occupancy(ws_plan* plan, double* tiles, double* classes, double* bands, double* planes, int32_t* transposed,
                     void* stream) {
    const DeviceGuard device_guard(plan);
    if (!plan) return WS_ERR_INVALID_ARG;
    if (!plan->d_masks || !plan->occ_grid) return fail(plan, WS_ERR_INVALID_ARG, "ws_get_occupancy: no occupancy recorded");
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_occupancy: synchronize");
    std::vector<uint32_t> all(plan->mask_words);
    e = cudaMemcpy(all.data(), plan->d_masks, all.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(plan, e, "ws_get_occupancy: copy");
    const bool tr = all[2] != 0;
    const uint32_t* m = all.data() + 8 + (tr ? plan->mask_set_words : 0);      // the set of the orientation in use
    const size_t nw = (size_t)plan->prm.n_wplanes, nt = (size_t)plan->geom.nt, n_class = nw * nt * 8;
    const size_t cw = (size_t)plan->mask_class_words, bw = (size_t)plan->mask_band_words;
    size_t t = 0, c = 0, b = 0, p = 0;
    for (size_t i = 0; i < n_class; ++i) {
        size_t bits = 0;
        for (size_t j = 0; j < cw; ++j) bits += (size_t)__builtin_popcount(m[i * cw + j]);
        t += bits;
        c += bits != 0;
    }
    for (size_t k = 0; k < nw; ++k) {
        size_t nb = 0;
        for (size_t i = 0; i < bw; ++i) nb += (size_t)__builtin_popcount(m[n_class * cw + k * bw + i]);
        b += nb;
        p += nb != 0;
    }
    if (tiles) *tiles = (double)t / (double)(nw * nt * nt);
    if (classes) *classes = (double)c / (double)n_class;
    if (bands) *bands = (double)b / (double)(nw * nt);
    if (planes) *planes = (double)p / (double)nw;
    if (transposed) *transposed = tr ? 1 : 0;
    return WS_OK;
}

int64_t ws_launch_count(const ws_plan* plan) { return plan ? plan->launches : 0; }

}  // extern "C"
