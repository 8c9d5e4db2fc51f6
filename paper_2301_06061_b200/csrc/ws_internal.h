// Internal declarations shared by the translation units of libwstack (CUDA product path only).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <stddef.h>
#include <string>

#include "../../include/wstack.h"

#define WS_TILE 32            // T: uv-tile side of the bin key, one warp owns one tile-plane
#define WS_MAX_CHAN 128       // per-channel constants travel as a kernel parameter
#define WS_CHUNK 1024         // records a warp accumulates in shared memory before it flushes
#define WS_HALO_MAX 7         // (S-1)/2 for S <= 15
#define WS_KB_MAX_TERMS 48    // terms of the I0 power series kept for the Kaiser-Bessel taps (beta <= 24)
#define WS_E2E_MAX_CHUNKS 32   // row chunks ws_image_from_host pipelines (copy of chunk c + 1 beside the gridding of chunk c)
#define WS_WC_GROUP 8          // planes per Horner block in the w-correction (exact restart between blocks)

// Per-channel position constants (O1): fp64, computed on the host exactly as the header states.
struct WsChanConsts {
    double su[WS_MAX_CHAN];   // cells per stored-uvw unit
    double sw[WS_MAX_CHAN];   // planes per stored-uvw unit
    double ow;                // plane offset = -w_min / dw
    double half;              // N/2
};

// Geometry the binning and gridding kernels need.
struct WsGeom {
    int32_t n_pix, n_wplanes, support, halo;   // N, N_w, S, h
    int32_t plane_lo, plane_hi;                 // only visibilities whose plane k lies in [plane_lo, plane_hi) are kept (default: all)
    int32_t nt;                                 // N / T
    uint32_t n_bins;                            // N_w nt^2
    float tap_c;                                // -log2(e) / (2 sigma^2): g(x) = norm1 * 2^(tap_c x^2)
    float norm2;                                // product of the two 1-D normalisations (folded into weight * vis once)
    // Kaiser-Bessel: g(x) / norm1 = sum_k kb_c[k] y^k, y = 1 - kb_y x^2, kb_c[k] = (beta^2/4)^k / (k!)^2 / I0(beta)
    int32_t kb_terms;                           // 0: Gaussian
    float kb_y;                                 // 4 / S^2
    float kb_c[WS_KB_MAX_TERMS];
};

// Order in which the binning kernels walk the visibilities (ws_plan_set_snapshot_rows).  The input is time-major: a
// snapshot holds F = rows_per_snapshot * n_chan visibilities that lie next to each other in memory, and one (baseline,
// channel) moves by about a cell from one snapshot to the next.  A warp takes `cw` memory-adjacent
// visibilities of 32 / cw CONSECUTIVE SNAPSHOTS, so that most of its lanes fall into the same few bins: their slots
// are adjacent, the record / perm stores coalesce and one atomic serves many lanes.  cw = 0: input order.
struct WsRemap {
    uint32_t cw_log2, cw;      // cw: power of two dividing F (4 where possible); ts = 32 / cw snapshots per warp
    uint32_t n_t;              // whole blocks of ts snapshots in this call
    uint32_t per_snap;         // F
    uint32_t n_main;           // n_t * ts * F: visibilities beyond (ragged last block / snapshot) keep the input order
};

// Workspace carve-up for one ws_grid_visibilities call (all offsets 256-byte aligned).
struct WsLayout {
    size_t off_counts_home, off_counts_halo;    // [n_bins + 1] u32 each: histograms -> exclusive scans (bin_start / halo_start)
    size_t off_rec_start;                       // [n_bins + 1] u32: bin_start + halo_start: a tile receives something iff its entry grows
    size_t off_cursor_home;                     // [n_bins] u32: running slot cursors of the scatter; afterwards the gridder's list of light bins
    size_t off_block_sums;                      // scan scratch
    size_t off_keys, off_perm, off_sorted_keys; // [n_vis] u32 each
    size_t off_presum;                          // [presum_rows] float2: per-row sums of weight * vis (WS_FLAG_PRESUM_CHANNELS)
    size_t off_items;                           // heavy-chunk work items (uint4)
    size_t off_records;                         // float4 records, one per kept visibility, lists indexed by bin_start
    size_t total;                               // bytes used for capacity `rec_capacity`
    uint64_t rec_capacity;                      // records that fit
    uint32_t item_capacity;
};

struct WsStatus {                               // device-side, 64 bytes
    uint32_t n_kept;                            // kept visibilities (home histogram total)
    uint32_t n_records;                         // records incl. halo copies
    uint32_t n_items;                           // heavy chunks queued
    uint32_t n_light;                           // non-empty bins that are not heavy, listed for the gridder
    uint32_t queue;                             // k_grid's work counter: heavy chunks first, then the listed bins (zeroed with the two above)
    uint32_t overflow;                          // 1: record or item capacity exceeded, gridding skipped (cleared by every binning call)
    uint32_t sticky_overflow;                   // ... of ANY call since the last ws_async_status (which clears it)
    uint32_t pad[9];
};

struct ws_plan {
    ws_params prm;
    WsGeom geom;
    int sm_count;
    cufftHandle fft;
    bool fft_ok;
    cufftHandle fft_rows1d;                     // batched 1-D transforms along u of the whole stack (degridding fast path)
    bool fft_rows1d_ok;
    size_t fft_rows1d_work;                     // its work area (taken from the end of the caller's workspace)
    size_t fft_work_bytes;
    int fft_batch;                              // planes per cufftExec call
    int64_t launches;
    std::string last_error;
    // state of the last grid call (for ws_get_bins)
    void* last_ws;
    WsLayout last_layout;
    int64_t last_n_vis;
    bool last_valid;
    bool sorted_keys_valid;
    int sticky_status;
    WsStatus* d_status;                         // plan-owned 64-byte device block: totals and the overflow flag
    // own FFT (ws_fft.cu): available for N = 2^8 .. 2^13 unless WS_FLAG_LIBRARY_FFT is set
    bool fft_own;
    void* d_twiddles;                           // plan-owned inter-stage twiddle tables (fp64-computed, < 140 KB)
    size_t tw_off_a, tw_off_b, tw_off_c;        // entry offsets of the pass 1a / 1b tables and of the row kernel's register constants
    int mask_class_words, mask_band_words;      // words per class mask (2 for N = 16384) and band words per plane (16 for N = 16384)
    void* d_masks;                              // plan-owned tile-occupancy masks of the mesh (class masks, band masks)
    size_t mask_words, mask_set_words;          // whole buffer; one set (class masks, band masks, band list) of the two orientations
    double* d_sumwt;                            // plan-owned: sum of the weights of the kept visibilities (WS_FLAG_TRACK_SUMWT)
    float* d_taper;                             // plan-owned [N]: 1 / ghat((p - N/2)/N), fp64-computed on the host
    int64_t snapshot_rows;                      // ws_plan_set_snapshot_rows hint (0: none)
    const float* last_weights;                  // weights of the last ws_bin_visibilities call
    int32_t last_chan_per_key;                  // visibilities per binned entry: 1, or n_chan after a pre-summed call
    bool last_has_values;                       // false: the bins were made by ws_degrid_visibilities (records carry no visibilities)
    cudaStream_t copy_stream;                   // ws_image_from_host: the H2D copies of the next chunk run beside the gridding
    cudaEvent_t ev_start, ev_chunk[WS_E2E_MAX_CHUNKS];    // of this one (created on first use)
    cudaEvent_t ev_orient;
    int32_t* h_orient;                          // pinned host word: the orientation flag of the sparse mesh, read back asynchronously
    bool e2e_ready;
    size_t e2e_chunk_bytes;                     // input bytes per chunk (0: 160 MiB)
    const void* occ_grid;                       // mesh the masks describe (NULL: none)
    bool occ_sparse;                            // ... and it was written by WS_GRID_SPARSE (private layout, empty tiles unwritten)
};

static inline size_t ws_align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Tile-occupancy masks of the mesh (built by ws_fft.cu, also read by the gridder in WS_GRID_SPARSE_ADD mode).
// Buffer: ctrl[8] = {bands of set 0, bands of set 1, transposed, ...} | set 0 | set 1; a set = class masks, band masks.
// class mask ((k nt + band) 8 + c) x cw words: bit m <=> the tile at (other coordinate = c + 8 m, band) of plane k holds
// visibilities, in STORAGE (FFT-native) tile coordinates; set 0: band = tx, other = ty; set 1 (transposed mesh): swapped.
#define WS_MASK_CTRL 8
struct WsMaskView {
    const uint32_t* masks;     // NULL: no occupancy available
    uint32_t set_words;
    int32_t class_words;
};
#ifdef __CUDACC__
// was the logical tile (k, ty, tx) marked occupied?  (the set of the orientation the mesh is stored in)
__device__ __forceinline__ bool ws_tile_occupied(const WsMaskView& mv, int nt, uint32_t k, uint32_t ty, uint32_t tx) {
    const uint32_t tr = mv.masks[2];
    const uint32_t* cm = mv.masks + WS_MASK_CTRL + (tr ? mv.set_words : 0u);
    const uint32_t sx = (tx + (uint32_t)nt / 2) & ((uint32_t)nt - 1), sy = (ty + (uint32_t)nt / 2) & ((uint32_t)nt - 1);
    const uint32_t band = tr ? sy : sx, other = tr ? sx : sy;
    const uint32_t m = other >> 3;
    return (cm[(((size_t)k * nt + band) * 8 + (other & 7)) * mv.class_words + (m >> 5)] >> (m & 31)) & 1u;
}
#endif

// ---- launchers (each returns the number of kernels it launched, or a negative WS_ERR_*) ----------------
size_t ws_bin_layout_bytes(const ws_plan* plan, int64_t n_vis, int64_t presum_rows);      // ws_api.cu
int ws_launch_bin(ws_plan* plan, const WsLayout& L, char* ws, const WsChanConsts& cc, const float* uvw,
                  const float2* vis, const float* wt, int64_t n_rows, int32_t n_chan, cudaStream_t st);
int ws_launch_grid(ws_plan* plan, const WsLayout& L, char* ws, float2* grid, int mode, cudaStream_t st);
WsMaskView ws_fft_mask_view(const ws_plan* plan);
int ws_launch_items(ws_plan* plan, const uint32_t* starts, uint32_t* light, uint4* items, uint32_t item_capacity, cudaStream_t st);
int ws_launch_wscreen_fwd(ws_plan* plan, const float2* image, float2* planes, int conj_out, cudaStream_t st);
// xf_lr0 < 0: planes in natural (FFT-native) order; >= 0: log2(N / 256), the planes hold the CONJUGATE of the transform
// with the rows where ws_fft_columns leaves them (frequency f at row ((f mod R0) << 8) | (f / R0))
int ws_launch_degrid(ws_plan* plan, const WsLayout& L, char* ws, const float2* planes, float2* vis_out, float scale,
                     int accumulate, int xf_lr0, cudaStream_t st);
int ws_launch_fft_masks_degrid(ws_plan* plan, const uint32_t* bin_start, cudaStream_t st);
int ws_launch_sorted_keys(ws_plan* plan, const WsLayout& L, char* ws, cudaStream_t st);
int ws_launch_wcorrect(ws_plan* plan, const float2* planes, float2* image, int accumulate, float* dirty,
                       cudaStream_t st);
int ws_launch_dirty(ws_plan* plan, const float2* image, float* dirty, uint32_t norm_flags, cudaStream_t st);
int ws_launch_sum_weights(ws_plan* plan, const WsLayout& L, char* ws, const float* wt, int64_t n_vis, int32_t chan_per_key,
                          cudaStream_t st);
int ws_launch_presum(ws_plan* plan, const float2* vis, const float* wt, int64_t n_rows, int32_t n_chan, float2* out,
                     cudaStream_t st);
int ws_launch_zero(ws_plan* plan, void* ptr, size_t bytes, cudaStream_t st);
// WS_FLAG_MESH_F64 (ws_f64.cu): fp64 mesh, image and dirty image
int ws_launch_grid_f64(ws_plan* plan, const WsChanConsts& cc, const float* uvw, const float2* vis, const float* wt,
                       int64_t n_rows, int32_t n_chan, int presum, double* grid, cudaStream_t st);
int ws_launch_wcorrect_f64(ws_plan* plan, const void* planes, void* image, int accumulate, void* dirty, cudaStream_t st);
int ws_launch_dirty_f64(ws_plan* plan, const void* image, void* dirty, uint32_t norm_flags, cudaStream_t st);
bool ws_fft_own_supported(int n_pix, int n_wplanes);
int ws_fft_own_init(ws_plan* plan);             // twiddle table + kernel attributes; WS_OK or an error
int ws_launch_fft_cols(ws_plan* plan, float2* grid, bool sparse, cudaStream_t st);
int ws_launch_fft_rows(ws_plan* plan, const float2* grid, float2* image, float* dirty, int accumulate, bool sparse,
                       int part, int n_parts, cudaStream_t st);
int ws_launch_fft_masks_clear(ws_plan* plan, cudaStream_t st);
int ws_launch_fft_masks(ws_plan* plan, const uint32_t* rec_start, int decide, cudaStream_t st);
const uint32_t* ws_fft_orientation_flag(const ws_plan* plan);   // device word: 1 = the sparse mesh is stored transposed
