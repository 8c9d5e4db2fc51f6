// ws_grid_visibilities_static (wstack.h): a1 + a2 with the workspace in a file-scope device array instead of a buffer
// the caller allocates, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that
// forbid it).  The kernels are the ones ws_grid_visibilities launches (k_keys_hist, the scan, k_scatter,
// k_prepare_heavy, k_grid: ws_bin.cu / ws_grid.cu); what differs is where their scratch -- histograms, cursors, keys,
// the permutation, the sorted records, the work items -- lives.
//
// `ws_static_scratch` below is a HOST-side stand-in for the device array when it is named in host code: it is not a
// device address.  The address the kernels get comes from cudaGetSymbolAddress, asked once per device with that device
// current (a library loaded on several GPUs has one copy of the array on each).
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>
#include <string>

#include "ws_internal.h"

static_assert(WS_STATIC_SCRATCH_BYTES % 256 == 0, "the scratch array is carved up in 256-byte units");
static __device__ __align__(256) unsigned char ws_static_scratch[WS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_lock;
void* g_scratch[MAX_DEVICES];          // device address of ws_static_scratch on device d (NULL: not asked yet)

// The device address of the array on the CURRENT device, which must be `device`.
cudaError_t scratch_address(int device, void** out) {
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, ws_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch[device] = p;
    }
    *out = g_scratch[device];
    return cudaSuccess;
}

struct OnDevice {                       // makes `device` current, restores the caller's on the way out
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit OnDevice(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) {
            err = cudaSetDevice(device);
            switched = err == cudaSuccess;
        }
    }
    ~OnDevice() {
        if (switched) cudaSetDevice(prev);
    }
};

int refuse(ws_plan* plan, int code, const std::string& msg) {
    plan->last_error = msg;
    return code;
}

}  // namespace

extern "C" {

size_t ws_static_scratch_bytes(void) { return WS_STATIC_SCRATCH_BYTES; }

int ws_grid_visibilities_static(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                                const double* freq_hz, int64_t n_rows, int32_t n_chan, void* grid, int32_t mode,
                                void* stream) {
    if (!plan) return WS_ERR_INVALID_ARG;
    if (plan->prm.flags & WS_FLAG_MESH_F64)
        return refuse(plan, WS_ERR_UNSUPPORTED,
                      "ws_grid_visibilities_static: a WS_FLAG_MESH_F64 plan grids without scratch memory: call ws_grid_visibilities");
    if (n_rows < 0 || n_chan <= 0 || n_chan > WS_MAX_CHAN)
        return refuse(plan, WS_ERR_INVALID_ARG, "ws_grid_visibilities_static: bad n_rows / n_chan");
    const int device = plan->prm.device;
    if (device < 0 || device >= MAX_DEVICES)
        return refuse(plan, WS_ERR_UNSUPPORTED, "ws_grid_visibilities_static: device ordinal beyond 63");
    // the size test comes first: it needs no device, and its message has to name the limit
    const bool presum = (plan->prm.flags & WS_FLAG_PRESUM_CHANNELS) != 0;
    const double n_vis_d = presum ? (double)n_rows : (double)n_rows * (double)n_chan;
    const size_t need = n_vis_d > (double)(1 << 30) ? (size_t)-1
                                                    : ws_bin_layout_bytes(plan, presum ? n_rows : n_rows * n_chan, presum ? n_rows : 0);
    if (need > (size_t)WS_STATIC_SCRATCH_BYTES) {
        char msg[320];
        if (need == (size_t)-1)
            std::snprintf(msg, sizeof msg, "ws_grid_visibilities_static: more than 2^30 visibilities in one call");
        else
            std::snprintf(msg, sizeof msg,
                          "ws_grid_visibilities_static: %.0f visibilities in %lld bins need %zu bytes of scratch, the static "
                          "array holds WS_STATIC_SCRATCH_BYTES = %zu: split the call, or use ws_grid_visibilities with a "
                          "workspace of your own",
                          n_vis_d, (long long)plan->geom.n_bins, need, (size_t)WS_STATIC_SCRATCH_BYTES);
        return refuse(plan, WS_ERR_WORKSPACE, msg);
    }
    const OnDevice on(device);
    if (on.err != cudaSuccess)
        return refuse(plan, WS_ERR_CUDA, std::string("ws_grid_visibilities_static: cudaSetDevice: ") + cudaGetErrorString(on.err));
    void* scratch = nullptr;
    const cudaError_t e = scratch_address(device, &scratch);
    if (e != cudaSuccess)
        return refuse(plan, WS_ERR_CUDA, std::string("ws_grid_visibilities_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    // From here on the call is ws_grid_visibilities on that address: the binning clears the histograms at the head of the
    // workspace on `stream` before it counts, every other region is written before it is read, so nothing the previous
    // call left in the array is seen.
    return ws_grid_visibilities(plan, uvw, vis, weights, freq_hz, n_rows, n_chan, grid, mode, scratch,
                                (size_t)WS_STATIC_SCRATCH_BYTES, stream);
}

}  // extern "C"
