/*
 * wstack.h -- C ABI of the B200-native w-stacking hot path (arxiv 2301.06061).
 *
 * The chain follows the paper's statement of the problem (PAPER.md:66-68 Eq. 2, :76-88 steps 1-5):
 *
 *   ws_grid_visibilities   a1 + a2: bin the visibilities by (w-plane, uv-tile) and convolve them onto
 *                          the stack of w-planes (Eq. 3 at :80)
 *   ws_fft_planes          a3: one 2-D inverse FFT per w-plane -- cuFFT
 *   ws_fft_wcorrect        a3 + a4 in one call: the library's own FFT with Eq. 2 fused into its last pass
 *   ws_wcorrect_accumulate a4: phase screen exp(2 pi i w_k (sqrt(1-l^2-m^2)-1)) times plane k, summed
 *                          over planes (PAPER.md:68 Eq. 2, :86)
 *   ws_dirty_image         a5: real part of the accumulated image, optionally normalised
 *   ws_predict_planes,
 *   ws_degrid_visibilities the opposite direction, image -> visibilities, the adjoint of the chain above
 *
 * Kernels: Gaussian or Kaiser-Bessel (:82, :459), both evaluated in registers.  Narrow-band data (one uvw
 * per row shared by all channels, :207) can be pre-summed per row (WS_FLAG_PRESUM_CHANNELS).
 *
 * Conventions (DESIGN.md sections 2-3 give the readings R1-R16 of the paper behind them):
 *   - All data pointers are DEVICE pointers unless the argument is marked "host".  The caller owns every
 *     buffer and the stream; the library owns only the opaque plan.  Pointers must be 16-byte aligned.
 *   - Every call enqueues work on `stream` and returns; buffers must stay alive until the stream drains.
 *     Only ws_plan_create/destroy, ws_get_bins, ws_get_occupancy, ws_get_sum_weights, ws_async_status and
 *     ws_image_from_host synchronise.
 *   - Every call returns WS_OK (0) or a negative WS_ERR_* code; nothing throws, exits or prints.
 *     Arguments are validated before any launch.
 *   - Mesh ("grid") layout: complex64 [n_wplanes][n_pix][n_pix], u fastest, FFT-NATIVE storage order:
 *     logical cell (j, i)  <->  (v, u) = ((j - N/2) du, (i - N/2) du), du = 1/(N cell_rad), is stored at
 *     row (j + N/2) mod N, column (i + N/2) mod N, so that the FFT needs no shift pass.  After
 *     ws_fft_planes logical pixel (q, p) of plane k sits at the same wrapped position.
 *   - Image layout: complex64 [n_pix][n_pix], CENTRED: pixel (q, p) <-> (m, l) = ((q-N/2), (p-N/2)) cell_rad.
 *   - One plan per host thread.  Every call that touches the device makes the plan's device current for its duration and
 *     restores the caller's afterwards (ws_plan_create leaves the plan's device current).
 *   - With WS_FLAG_MESH_F64 the mesh, image and dirty image are complex128 / complex128 / float64 wherever this header says
 *     complex64 / complex64 / float32 (the `float* dirty` arguments then point to doubles).
 */
#ifndef WSTACK_H
#define WSTACK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WS_VERSION 200

/* error codes */
#define WS_OK 0
#define WS_ERR_INVALID_ARG (-1)
#define WS_ERR_UNSUPPORTED (-2)
#define WS_ERR_WORKSPACE (-3)   /* workspace too small */
#define WS_ERR_CUDA (-4)
#define WS_ERR_CUFFT (-5)

/* ws_grid_visibilities mode */
#define WS_GRID_ACCUMULATE 0 /* add onto the existing mesh (call ws_grid_zero first, or start with an OVERWRITE call); tiles
                                without visibilities untouched */
#define WS_GRID_OVERWRITE 1  /* the mesh is taken as zero on entry and EVERY cell is written: no ws_grid_zero needed */
#define WS_GRID_SPARSE 2     /* as OVERWRITE, but only the 32 x 32 tiles that receive visibilities are written; every
                                other cell keeps whatever it held, and the layout is PRIVATE: the library stores the
                                planes transposed ([k][u][v]) when that leaves fewer 32-line bands to transform.  Only
                                ws_fft_* with WS_FFT_USE_OCCUPANCY can consume such a mesh (own FFT: N = 2^8..2^13
                                and no WS_FLAG_LIBRARY_FFT), and nothing can be accumulated onto it */

#define WS_GRID_SPARSE_ADD 3 /* a further chunk of visibilities onto a WS_GRID_SPARSE mesh (same plan, same `grid`, nothing else
                                having written it since): tiles the earlier calls filled are added to, tiles that are new are
                                stored, the recorded occupancy grows.  The orientation the first call chose is kept.  This is
                                how chunks are streamed through the gridder without ever clearing the mesh (Extreme) */

/* fft_flags of ws_fft_wcorrect / ws_fft_columns / ws_fft_rows_wcorrect */
#define WS_FFT_USE_OCCUPANCY 1u /* skip the tiles / column bands the gridding calls on this plan left empty.  The plan
                                   records which tiles of a mesh its ws_grid_* calls filled (restarted by ws_grid_zero
                                   and by an OVERWRITE / SPARSE call, extended by ACCUMULATE calls); valid only if
                                   nothing else wrote the mesh in between (else WS_ERR_INVALID_ARG, or wrong results
                                   if the library cannot know) */

/* ws_params.flags */
#define WS_FLAG_LIBRARY_FFT 1u /* a3 through cuFFT even where the library's own two-pass FFT exists (N = 2^8..2^14) */
#define WS_FLAG_NO_TRANSPOSE 2u /* WS_GRID_SPARSE keeps the [k][v][u] orientation (default: it may store the mesh transposed) */

#define WS_FLAG_TRACK_SUMWT 4u  /* every gridding call also sums the weights of the visibilities it kept (one extra
                                   reduction kernel); needed by WS_NORM_SUMWT.  The sum restarts with ws_grid_zero and
                                   with an OVERWRITE / SPARSE call and grows with ACCUMULATE calls */

#define WS_FLAG_PRESUM_CHANNELS 8u /* the paper's narrow-band mode at scale (one thread grids "all frequencies and
                                     polarisations" of a measurement): with freq_hz == NULL the n_chan visibilities of a row
                                     share one position, so sum_c weight * vis is formed per row first (one streaming pass)
                                     and ROWS are binned and gridded: n_chan times fewer records.  The bins ws_get_bins
                                     exports are then per row (n_vis = n_rows).  Ignored by ws_degrid_visibilities; a
                                     gridding call with freq_hz != NULL on such a plan is WS_ERR_INVALID_ARG */

#define WS_FLAG_MESH_F64 16u /* the paper's own arithmetic (Table 3: fp64 mesh, real and imaginary part): grid, image
                               and dirty image are complex128 / complex128 / float64 (sizes from ws_grid_bytes etc.), taps and phases
                               are evaluated in fp64.  For like-for-like context against the paper's Table 4, not for speed: the
                               gridder is the paper's own kernel shape, one thread per measurement with atomicAdd on the mesh
                               (:207, :219; nothing is binned, no workspace needed, ws_get_bins has nothing to export), the FFT is
                               cuFFT Z2Z.  Calls: ws_grid_zero, ws_grid_visibilities (ACCUMULATE / OVERWRITE), ws_fft_planes,
                               ws_wcorrect_accumulate, ws_fft_wcorrect (= the two), ws_dirty_image, ws_get_sum_weights; every
                               other entry returns WS_ERR_UNSUPPORTED.  With WS_FLAG_PRESUM_CHANNELS a thread takes a whole row */

/* kernel_type: the separable 1-D convolution function g(x), x in cells, unit integral (R2, R28) */
#define WS_KERNEL_GAUSSIAN 0      /* g(x) = exp(-x^2 / (2 sigma^2)) / (sigma sqrt(2 pi)), kernel_param = sigma */
#define WS_KERNEL_KAISER_BESSEL 1 /* g(x) = I0(beta sqrt(1 - (2x/S)^2)) beta / (S sinh beta) on |x| <= S/2, kernel_param =
                                     beta in (0, 24]; the production kernel PAPER.md:82 and :459 name (Jackson et al. 1991).
                                     I0 is evaluated in registers from its power series, not from a table */

/* norm_flags of ws_dirty_image: dirty = Re(image) times the product of the selected factors (R29) */
#define WS_NORM_SUMWT 1u /* 1 / (sum of the weights of the gridded visibilities); plan needs WS_FLAG_TRACK_SUMWT          */
#define WS_NORM_N 2u     /* n = sqrt(1 - l^2 - m^2): the 1/n on the left side of Eq. 2; 0 where l^2+m^2 >= 1 */
#define WS_NORM_TAPER 4u /* 1 / (ghat(xi_p) ghat(xi_q)), xi = (p - N/2)/N, ghat the continuous Fourier transform of g:
                            Gaussian exp(-2 pi^2 sigma^2 xi^2); Kaiser-Bessel (beta / sinh beta) sinh(r)/r,
                            r = sqrt(beta^2 - (pi S xi)^2) (sin(r')/r' with r' = sqrt(-(..)) beyond) */

typedef struct ws_plan ws_plan; /* opaque */

typedef struct ws_params {
    int32_t n_pix;        /* N: mesh and image side; multiple of 2*tile                                   */
    int32_t n_wplanes;    /* N_w >= 1                                                                      */
    int32_t support;      /* S: odd, 1..15; full S x S footprint ("kernel size of 7 cells")    */
    int32_t kernel_type;  /* WS_KERNEL_GAUSSIAN or WS_KERNEL_KAISER_BESSEL                                 */
    double kernel_param;  /* Gaussian: sigma in cells (> 0), 1.0 is the default reading R1; KB: beta        */
    double cell_rad;      /* image pixel size in radians (> 0)                                             */
    double w_min, w_max;  /* w range covered by the planes, wavelengths; w_max > w_min.  Plane k covers    */
                          /* [w_min + k dw, w_min + (k+1) dw), dw = (w_max-w_min)/N_w, value = midpoint     */
    int32_t tile;         /* uv-tile side T of the bin key; 0 = auto (32); only 32 is supported            */
    int32_t device;       /* CUDA device ordinal                                                           */
    uint32_t flags;       /* 0 or WS_FLAG_*                                                                */
} ws_params;

/* ---- plan ------------------------------------------------------------------------------------------- */
/* Validates `p`, selects the device, creates the cuFFT plan (work area NOT allocated: it comes from the
 * caller's workspace).  *out is NULL on failure. */
int ws_plan_create(const ws_params* p, ws_plan** out);
int ws_plan_destroy(ws_plan* plan);

/* Performance hint, never needed for correctness: the rows of every later gridding / degridding call are recorded
 * snapshot after snapshot with `rows_per_snapshot` rows (all baselines) per snapshot, in the same baseline order each
 * time (measurement sets are stored this way).  The binning kernels then walk the visibilities so that a
 * warp holds a few memory-adjacent visibilities of consecutive snapshots, which fall into the same bins: binning is
 * about twice as fast.  0 switches the hint off.  The results are the same sets either way (the order inside a bin
 * is unspecified in both cases); a wrong hint only costs speed. */
int ws_plan_set_snapshot_rows(ws_plan* plan, int64_t rows_per_snapshot);

/* Plane-sharded imaging over several GPUs (one plan per rank; the paper distributes slabs of the mesh over
 * MPI ranks and reduces the WHOLE mesh, Eq. 8 at :180): after this call the plan keeps only the
 * visibilities whose w-plane k (computed with the GLOBAL w_min, w_max, n_wplanes of the plan: the keys stay bit-exact)
 * lies in [plane_lo, plane_hi); all others are dropped like visibilities off the mesh.  Every rank runs the unchanged
 * chain on all the data and its own plane range -- planes outside it stay empty and cost nothing on the sparse path --
 * and the N x N images of the ranks are summed (one reduce of 8 N^2 bytes instead of the mesh).  Default: all planes. */
int ws_plan_set_plane_range(ws_plan* plan, int32_t plane_lo, int32_t plane_hi);

/* ---- sizes: all device memory is allocated by the caller ---------------------------------------------- */
size_t ws_grid_bytes(const ws_plan* plan);   /* 8 N^2 N_w */
size_t ws_image_bytes(const ws_plan* plan);  /* 8 N^2     */
size_t ws_dirty_bytes(const ws_plan* plan);  /* 4 N^2     */
/* Workspace that is enough for ws_grid_visibilities with up to max_vis_per_call visibilities (keys, perm, one 16-byte
 * record per visibility, the per-tile offset arrays) and for ws_fft_planes.  A workspace that cannot hold a call's
 * visibilities is refused by that call (WS_ERR_WORKSPACE). */
size_t ws_workspace_bytes(const ws_plan* plan, int64_t max_vis_per_call);   /* WS_FLAG_PRESUM_CHANNELS: count ROWS */
/* The same (dup_factor is ignored: round 1 stored a copy of a record in every tile its footprint reaches and sized the
 * workspace by that factor; since round 2 there is one record per visibility). */
size_t ws_workspace_bytes_for(const ws_plan* plan, int64_t max_vis_per_call, double dup_factor);
size_t ws_fft_workspace_bytes(const ws_plan* plan);
int ws_plan_tile(const ws_plan* plan);       /* T */
int64_t ws_plan_n_bins(const ws_plan* plan); /* N_w (N/T)^2 */

/* ---- a0: clear the mesh (needed before WS_GRID_ACCUMULATE calls only) ---------------------------------- */
int ws_grid_zero(ws_plan* plan, void* grid, void* stream);

/* ---- a1 + a2: binning and gridding, Eq. 3 ----------------------------------------------- */
/* uvw     [n_rows][3] float32: (u, v, w) per (baseline, time) row.
 * vis     [n_rows][n_chan] complex64 (re, im).      weights [n_rows][n_chan] float32.
 * freq_hz HOST pointer, [n_chan] doubles, or NULL.  Not NULL: uvw are metres, channel c is scaled by
 *         freq_hz[c]/c, c = 299792458 m/s.  NULL: uvw are wavelengths shared by the n_chan visibilities
 *         of the row (the paper's narrow-band mode).
 * Position rule (bit-exact contract, O2-O4): pu = fma(u, su_c, N/2), i0 = floor(pu + 1/2),
 * plane k = clamp(floor(fma(w, sw_c, ow))), dropped unless the S x S footprint lies on the mesh;
 * key = (k nt + j0/T) nt + i0/T, nt = N/T.  Contribution: weight * vis * g(a - fu) g(b - fv) at logical
 * cell (k, j0 + b, i0 + a), |a|,|b| <= (S-1)/2, fp32.  n_rows * n_chan <= 2^30, n_chan <= 128.
 * A visibility with a NaN coordinate is dropped (R33).  mode: one of WS_GRID_*.
 * Every tile of the mesh is accumulated by one warp in shared memory together with a ring of (S-1)/2 cells and added to
 * the mesh once (red.global.add: the ring is the only place where two writers meet); the tiles that receive anything
 * are cleared first, except in WS_GRID_ACCUMULATE mode and for tiles earlier WS_GRID_SPARSE(_ADD) chunks filled. */
int ws_grid_visibilities(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                         const double* freq_hz, int64_t n_rows, int32_t n_chan, void* grid, int32_t mode,
                         void* workspace, size_t workspace_bytes, void* stream);

/* The two halves of ws_grid_visibilities as separate calls (same arguments, same workspace): a1 leaves the bins
 * and the per-tile record lists in `workspace`; a2 consumes them.  ws_grid_visibilities == a1 then a2. */
int ws_bin_visibilities(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                        const double* freq_hz, int64_t n_rows, int32_t n_chan, void* workspace,
                        size_t workspace_bytes, void* stream);
int ws_grid_binned(ws_plan* plan, void* grid, int32_t mode, void* workspace, size_t workspace_bytes, void* stream);

/* ---- a3: per-plane un-normalised inverse 2-D FFT, in place -------------------------- */
/* P_k[q][p] = sum_ji G_k[j][i] exp(+2 pi i ((i-N/2)(p-N/2) + (j-N/2)(q-N/2)) / N) in logical indices. */
int ws_fft_planes(ws_plan* plan, void* grid, void* workspace, size_t workspace_bytes, void* stream);

/* 1 if ws_fft_wcorrect runs the library's own FFT kernels, 0 if it calls cuFFT + the stand-alone a4 pass. */
int ws_plan_fft_is_own(const ws_plan* plan);

/* ---- a4: w-correction and reduction over planes, Eq. 2 ------------------------------ */
/* image[q][p] (+)= sum_k exp(2 pi i w_k t) P_k[q][p], t = sqrt(1-l^2-m^2) - 1, w_k = w_min + (k+1/2) dw;
 * pixels with l^2 + m^2 >= 1 receive 0.  accumulate: 0 overwrite, 1 add to image.
 * dirty may be NULL; otherwise Re(image) after this call is also written there (float32 [N][N]). */
int ws_wcorrect_accumulate(ws_plan* plan, const void* planes, void* image, int32_t accumulate, float* dirty,
                           void* stream);

/* ---- a3 + a4 fused: ws_fft_planes followed by ws_wcorrect_accumulate, same image --------- */
/* With the own FFT (N = 2^8..2^13) a plane makes two trips through memory instead of four: columns (two in-place
 * steps), then rows, whose last pass multiplies each transformed row by the phase screen and sums it over the
 * planes in registers -- the transformed planes are never written.  `grid` is DESTROYED (it holds the
 * column-transformed planes afterwards, rows in digit-reversed order).  With cuFFT (WS_FLAG_LIBRARY_FFT or other
 * N) it is exactly the two calls in sequence and needs `workspace` >= ws_fft_workspace_bytes.  dirty may be NULL.
 * fft_flags: 0 (any mesh contents) or WS_FFT_USE_OCCUPANCY. */
int ws_fft_wcorrect(ws_plan* plan, void* grid, void* image, int32_t accumulate, float* dirty, uint32_t fft_flags,
                    void* workspace, size_t workspace_bytes, void* stream);
/* The two halves of ws_fft_wcorrect as separate calls (own FFT only, else WS_ERR_UNSUPPORTED).
 * ws_fft_columns transforms every plane along v in place: afterwards row position r of a plane holds
 * v-frequency (r / 256) + (N / 256) (r mod 256).  ws_fft_rows_wcorrect transforms such rows along u and applies
 * Eq. 2 without writing them back (grid is read only). */
int ws_fft_columns(ws_plan* plan, void* grid, uint32_t fft_flags, void* stream);
int ws_fft_rows_wcorrect(ws_plan* plan, const void* grid, void* image, int32_t accumulate, float* dirty,
                         uint32_t fft_flags, void* stream);

/* ---- a5: dirty[q][p] = Re image[q][p] x normalisation (PAPER.md:86-88; Eq. 2 solved for I, :68) ---------- */
/* norm_flags = 0: the plain real part.  Otherwise an OR of WS_NORM_*: with all three set and a Kaiser-Bessel
 * kernel the result is the weighted-mean brightness, comparable to the direct sum
 * n / sum(wt) * Re sum_k wt_k V_k exp(2 pi i (u l + v m + w (n - 1))) in the inner half of the field.
 * WS_NORM_SUMWT without WS_FLAG_TRACK_SUMWT, or unknown bits: WS_ERR_INVALID_ARG. */
int ws_dirty_image(ws_plan* plan, const void* image, float* dirty, uint32_t norm_flags, void* stream);

/* Sum of the weights of the visibilities gridded so far (plan with WS_FLAG_TRACK_SUMWT; synchronises `stream`). */
int ws_get_sum_weights(ws_plan* plan, double* sum_weights, void* stream);

/* ---- degridding: model image -> predicted visibilities (Eq. 1 at :59) -------------------- */
/* The adjoint of ws_grid_visibilities (unit weights) -> ws_fft_planes -> ws_wcorrect_accumulate, in two calls:
 *   ws_predict_planes       planes[k] = forward un-normalised 2-D DFT of model_image x exp(-2 pi i w_k (n - 1)),
 *                           k = 0..N_w-1, FFT-native storage order like the mesh (cuFFT; needs `workspace` >=
 *                           ws_fft_workspace_bytes).  model_image: complex64 [N][N], centred, the APPARENT sky
 *                           (Eq. 1's I / n), already divided by the kernel taper ghat(xi_p) ghat(xi_q) if calibrated
 *                           visibilities are wanted; pixels with l^2 + m^2 >= 1 are ignored.
 *   ws_degrid_visibilities  vis_out[row][chan] (complex64) = [accumulate ? vis_out : 0] + scale x
 *                           sum_{a,b} g(a - fu) g(b - fv) planes[k][j0 + b][i0 + a], positions by the rule of
 *                           ws_grid_visibilities; a dropped visibility predicts 0.  scale = -1 with accumulate = 1 turns
 *                           measured visibilities into residuals.  Bins the positions into `workspace` first (same
 *                           size rules as ws_grid_visibilities; ws_get_bins works afterwards, ws_grid_binned does not). */
int ws_predict_planes(ws_plan* plan, const void* model_image, void* planes, void* workspace, size_t workspace_bytes,
                      void* stream);
int ws_degrid_visibilities(ws_plan* plan, const float* uvw, const double* freq_hz, int64_t n_rows, int32_t n_chan,
                           const void* planes, void* vis_out, float scale, int32_t accumulate, void* workspace,
                           size_t workspace_bytes, void* stream);
/* The two calls above as ONE, same result in vis_out (`planes` is scratch of ws_grid_bytes, its contents afterwards are
 * private).  Where the library's own FFT exists (N = 2^8..2^13) the positions are binned FIRST, so that only the
 * column bands of the planes that hold visibilities are transformed along v (the own column passes; along u: cuFFT),
 * and the gather reads the column-transformed planes where those passes leave them.  Elsewhere it is the two calls. */
int ws_predict_visibilities(ws_plan* plan, const void* model_image, const float* uvw, const double* freq_hz, int64_t n_rows,
                            int32_t n_chan, void* planes, void* vis_out, float scale, int32_t accumulate, void* workspace,
                            size_t workspace_bytes, void* stream);

/* ---- the whole path from HOST buffers (end-to-end entry) ----------------------------------------------- */
/* uvw_h, vis_h, weights_h, dirty_h are HOST pointers (pinned memory gives asynchronous copies); dev_inputs
 * is a 16-byte aligned device scratch of at least ws_dev_inputs_bytes(n_rows, n_chan) bytes (uvw | vis | weights,
 * each padded to 16 bytes); grid, image, dirty_d, workspace are device buffers as above.  Copies the inputs in,
 * runs a1..a5 (own FFT: WS_GRID_SPARSE + WS_FFT_USE_OCCUPANCY, so `grid` is private scratch whose empty tiles are
 * never written; library FFT: WS_GRID_OVERWRITE), copies the dirty image out, synchronises the stream and returns
 * the deferred status (WS_ERR_WORKSPACE if the record capacity of `workspace` was exceeded: dirty_h is then
 * meaningless). */
size_t ws_dev_inputs_bytes(int64_t n_rows, int32_t n_chan);
/* The rows are fed through the gridder in chunks of about `bytes` input bytes (0: the default, 160 MiB; at most 32
 * chunks): the copy of chunk c + 1 runs on a second stream beside the binning and gridding of chunk c (first chunk
 * WS_GRID_SPARSE, later ones WS_GRID_SPARSE_ADD), so that only the last chunk's gridding, the FFT and the copy out
 * are exposed behind the PCIe time (the paper's GPU timings include the copies). */
int ws_plan_set_e2e_chunk_bytes(ws_plan* plan, size_t bytes);
int ws_image_from_host(ws_plan* plan, const float* uvw_h, const void* vis_h, const float* weights_h,
                       const double* freq_hz, int64_t n_rows, int32_t n_chan, void* dev_inputs,
                       size_t dev_inputs_bytes, void* grid, void* image, float* dirty_d, float* dirty_h,
                       void* workspace, size_t workspace_bytes, void* stream);

/* ---- parity export of the bins of the LAST ws_grid_visibilities call ----------------------------------- */
/* Device pointers into that call's workspace, valid until the next call on the plan: keys[n_vis] in input
 * order (0xFFFFFFFF = dropped), sorted_keys[n_kept] ascending, perm[n_kept] flat visibility indices
 * (row * n_chan + c) grouped by ascending key -- the order INSIDE a bin is unspecified (atomic slot
 * assignment) -- and bin_start[n_bins + 1].  Synchronises `stream`.  Any output pointer may be NULL. */
int ws_get_bins(ws_plan* plan, const uint32_t** keys, const uint32_t** sorted_keys, const uint32_t** perm,
                const uint32_t** bin_start, int64_t* n_vis, int64_t* n_bins, int64_t* n_dropped,
                int64_t* n_records, void* stream);

/* Fractions of the mesh the recorded occupancy marks non-empty (synchronises `stream`): 32 x 32 tiles; row classes
 * pass 1a of the FFT writes; 32-column bands per plane (what pass 1b writes and pass 2 reads); planes with any;
 * *transposed = 1 if the WS_GRID_SPARSE mesh is stored [k][u][v] (then "column" means a line along u). */
int ws_get_occupancy(ws_plan* plan, double* tiles, double* classes, double* bands, double* planes, int32_t* transposed,
                     void* stream);

/* Synchronises `stream` and returns the deferred status of the work enqueued so far (record capacity
 * exceeded -> WS_ERR_WORKSPACE, CUDA fault -> WS_ERR_CUDA). */
int ws_async_status(ws_plan* plan, void* stream);

/* a1 + a2 WITHOUT a caller-allocated workspace, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * serving loops, harnesses that forbid it): ws_grid_visibilities (Eq. 3 at :80) with its scratch -- the
 * histograms, keys, permutation, sorted records and work items of the binning -- in a static device array of
 * WS_STATIC_SCRATCH_BYTES that every GPU holding the library keeps until the process exits.  Same arguments, layouts,
 * modes and results as ws_grid_visibilities (all device pointers, 16-byte aligned; freq_hz host or NULL); the call
 * allocates and frees nothing on the device and calls no library routine that does.
 *   Limit: the layout for n_rows * n_chan visibilities (n_rows under WS_FLAG_PRESUM_CHANNELS) and the plan's bins must
 * fit the array: about 16 (n_bins + 1) + 28.1 n_vis bytes, e.g. the 1.13 million visibilities of a 2048^2 x 16-plane mesh.
 * Beyond it the call returns WS_ERR_WORKSPACE before anything is launched and ws_last_error names the bytes needed and
 * the limit; a WS_FLAG_MESH_F64 plan (which uses no scratch) is WS_ERR_UNSUPPORTED.
 *   The array is SHARED by every plan and stream of the process on that device and keeps the last call's contents: the
 * call clears what must start at zero (on `stream`), but two calls whose work overlaps on the GPU race -- keep them on
 * one stream or order them with events -- and ws_get_bins after it reads the array, so it must come before the next
 * static call.  The plan itself is created beforehand (ws_plan_create allocates). */
#define WS_STATIC_SCRATCH_BYTES (32u << 20)
int ws_grid_visibilities_static(ws_plan* plan, const float* uvw, const void* vis, const float* weights,
                                const double* freq_hz, int64_t n_rows, int32_t n_chan, void* grid, int32_t mode,
                                void* stream);
size_t ws_static_scratch_bytes(void); /* = WS_STATIC_SCRATCH_BYTES of the library that is loaded */

/* Diagnostic (not part of the path): the fp32 FMA rate, in TFLOP/s, that a register-only FFMA loop reaches on the plan's
 * device (best of four short launches; synchronises `stream`).  bench.py prints it beside the derived fp32 peak. */
int ws_measure_fp32_tflops(ws_plan* plan, double* tflops, void* stream);

/* Number of kernels this library has launched through `plan` since it was created. */
int64_t ws_launch_count(const ws_plan* plan);

const char* ws_strerror(int code);
const char* ws_last_error(const ws_plan* plan);
int ws_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WSTACK_H */
