// a3 + a4: the per-plane un-normalised inverse 2-D FFT written for this path, with the
// phase correction and the reduction over the w-planes (Eq. 2) fused into its last pass.
//
// The paper leaves the FFT to FFTW on the CPU (55-80 % of its GPU runs) and names a GPU FFT as
// future work (:459).  A library 2-D FFT of an 8192^2 plane reads and writes the mesh three times (rows, and the
// columns in two steps), and a4 reads it a fourth time.  Here, for N = R0 * 256 (N = 2^8 .. 2^14):
//   pass 1a              columns, first radix-R0 step across the N/R0-spaced rows, in registers: a warp = 32
//                        adjacent columns, so every access is a whole 256-byte row segment; twiddles are
//                        warp-uniform; no shared memory;
//   pass 1b              columns, the remaining 256-point transforms of a [256 rows x 16 columns] block per item
//                        (lane = column: conflict-free, coalesced), radix 16 x 16, in place.  Row position
//                        256 m0 + f of the mesh then holds v-frequency m0 + R0 f;
//                        both in ONE launch, k_fft_cols: items of the two passes from one queue, pass 1b of a band a
//                        few bands behind its pass 1a, so that what pass 1a writes is read back from L2
//                        (N = 256: pass 1b alone, k_fft_colB);
//   pass 2  k_fft_rows   rows.  A CTA owns 8192 contiguous points (whole rows) of EVERY plane: bulk copies (TMA,
//                        cp.async.bulk + mbarrier) land the next plane's rows in shared memory while the current one
//                        is transformed (radix 32/16/8 in registers, in-place exchanges through padded shared memory).
//                        The transformed row never returns to memory: it is multiplied by the phase screen and
//                        summed over the planes in registers (Horner's rule on the geometric phase sequence of a
//                        pixel), and the image row is written once.
// All three skip what the gridder left empty (tile occupancy masks, ws_grid.cu): the uv coverage of one w-plane
// touches a few per cent of its tiles, so pass 1a reads almost nothing, and whole column bands of a plane stay
// zero and are neither written by pass 1 nor read by pass 2.
// Decimation in frequency; the digit-reversed order costs nothing because pass 2 accumulates in registers and
// un-permutes once per image row.  Inter-stage twiddles come from fp64-computed tables.
// Tensor cores are not used: an FFT at fp32 accuracy is not a dense contraction (north_star).
#include <math.h>

#include <vector>

#include "ws_internal.h"
#include "ws_phase.cuh"

namespace {

constexpr int CT = 256;            // threads per CTA of the column kernels
constexpr int FT = 512;            // threads per CTA of the row kernel: two groups of 8 warps
constexpr int GT = 256;            // threads per group
constexpr int PT = 128;            // the producer's warpgroup (one warp of it works): register re-allocation is per warpgroup
constexpr int EPT = 16;            // points per thread
constexpr int PTS = FT * EPT;      // points per CTA (8192)
constexpr int MAX_PLANES = 4096;   // w-planes the row kernel's per-plane occupancy bits provide for
constexpr int WC_SPAN = 64;        // planes per Horner chain of the fused w-correction (exact restart between chains)

// ---- stage plan of the row transform: N = prod R_s ---------------------------------------------------------------
__host__ __device__ constexpr int n_stages(int logn) { return logn == 8 ? 2 : 3; }
__host__ __device__ constexpr int log2r(int logn, int s) {
    if (s >= n_stages(logn)) return 0;
    switch (logn) {
        case 8: return 4;                                   // 16 16
        case 9: return s < 2 ? 4 : 1;                       // 16 16 2
        case 10: return s < 2 ? 4 : 2;                      // 16 16 4
        case 11: return s < 2 ? 4 : 3;                      // 16 16 8
        case 12: return 4;                                  // 16 16 16
        case 13: return s == 0 ? 5 : 4;                     // 32 16 16 (the radix-32 butterflies are split over two threads)
        case 14: return s == 0 ? 6 : 4;                     // 64 16 16 (radix 64 split over two threads of each of two CTAs)
    }
    return 0;
}
// log2 of the sub-transform length entering stage s
__host__ __device__ constexpr int log2l(int logn, int s) {
    int l = logn;
    for (int i = 0; i < s; ++i) l -= log2r(logn, i);
    return l;
}
// offset (entries) of stage s in the twiddle table; stage s holds (R-1) * Q entries [(m'-1) Q + j] = W_L^(j m')
__host__ __device__ constexpr int tw_offset(int logn, int s) {
    int o = 0;
    for (int i = 0; i < s; ++i) o += ((1 << log2r(logn, i)) - 1) << (log2l(logn, i) - log2r(logn, i));
    return o;
}
__host__ __device__ constexpr int tw_entries(int logn) { return tw_offset(logn, n_stages(logn) - 1); }   // last stage: Q = 1, none
// what of it the row kernel keeps in shared memory: everything, except for N = 16384, where the 128 KB landing buffer
// leaves no room for the first-stage table (63 x 256 entries): there the first-stage twiddle of output digit d = 4 (4 a + b) + q
// is the product of two factors from two small tables, W_N^(ug (4 b + q)) (the two q of the CTA: 2 x 4 x 256 entries) and
// W_N^(16 a ug) (3 x 256), beside the stage-1 table.  (Measured at N = 8192: factored twiddles + a second landing buffer in the
// freed shared memory, 12.06 ms against 11.72 with the full table -- the second, dependent complex multiply per output costs
// more issue slots and latency than the table's loads; not used there.)
__host__ __device__ constexpr bool tw_factored(int logn) { return logn >= 14; }
// (+ 3 x 256 entries W_N^(4 M a ug), a = 1..3: the second factor of the register twiddles, fetched per use)
// and 2 x 4 x 256 entries W_N^(ug (M b + q)) for the two q of the CTA's groups: the first factor)
__host__ __device__ constexpr int tw_smem_entries(int logn) { return tw_factored(logn) ? tw_entries(logn) - tw_offset(logn, 1) + 768 + 2048 : tw_entries(logn); }
__host__ __device__ constexpr int tw_smem_off1(int logn) { return tw_factored(logn) ? 0 : tw_offset(logn, 1); }

__host__ __device__ constexpr int brev(int i, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
    return r;
}
__device__ __forceinline__ int pad(int p) { return p + (p >> 4); }
constexpr int PAD_PTS = PTS + (PTS >> 4);

// position n inside a transformed sequence -> frequency index (mixed-radix digit reversal)
template <int LOGN>
__device__ __forceinline__ int freq_of(int n) {
    int f = 0, in = LOGN, out = 0;
#pragma unroll
    for (int s = 0; s < n_stages(LOGN); ++s) {
        const int lr = log2r(LOGN, s);
        in -= lr;
        f |= ((n >> in) & ((1 << lr) - 1)) << out;
        out += lr;
    }
    return f;
}


// ---- complex helpers -------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 sadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 ssub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// complex add / subtract as ONE packed instruction (add.f32x2 -> FADD2 on sm_100a): same lane throughput as two
// FADDs, half the issue slots -- the butterflies are mostly additions and the row kernel is issue-bound
__device__ __forceinline__ float2 eadd(float2 a, float2 b) {
    unsigned long long ra, rb, rc;
    float2 c;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rc) : "l"(ra), "l"(rb));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(c.x), "=f"(c.y) : "l"(rc));
    return c;
}
__device__ __forceinline__ float2 esub(float2 a, float2 b) {
    unsigned long long ra, rb, rc;
    float2 c;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(rc) : "l"(ra), "l"(rb));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(c.x), "=f"(c.y) : "l"(rc));
    return c;
}
// a * (c + i s)
__device__ __forceinline__ float2 emul(float2 a, float c, float s) {
    return make_float2(fmaf(a.x, c, -(a.y * s)), fmaf(a.x, s, a.y * c));
}
__device__ __forceinline__ float2 emul_i(float2 a) { return make_float2(-a.y, a.x); }
// a * (1 + i) and a * (-1 + i), unscaled
__device__ __forceinline__ float2 emul_1pi(float2 a) { return make_float2(a.x - a.y, a.x + a.y); }
__device__ __forceinline__ float2 emul_m1pi(float2 a) { return make_float2(-a.x - a.y, a.x - a.y); }
__device__ __forceinline__ float2 escale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }

// a * exp(+2 pi i k / 32), k = 0..15 a compile-time constant after unrolling
template <typename E>
__device__ __forceinline__ E mul_w32(E a, int k) {
    switch (k) {
        case 0: return a;
        case 1: return emul(a, 0.98078528040323043f, 0.19509032201612825f);
        case 2: return emul(a, 0.92387953251128674f, 0.38268343236508978f);
        case 3: return emul(a, 0.83146961230254524f, 0.55557023301960218f);
        case 4: return escale(emul_1pi(a), 0.70710678118654752f);
        case 5: return emul(a, 0.55557023301960218f, 0.83146961230254524f);
        case 6: return emul(a, 0.38268343236508978f, 0.92387953251128674f);
        case 7: return emul(a, 0.19509032201612825f, 0.98078528040323043f);
        case 8: return emul_i(a);
        case 9: return emul(a, -0.19509032201612825f, 0.98078528040323043f);
        case 10: return emul(a, -0.38268343236508978f, 0.92387953251128674f);
        case 11: return emul(a, -0.55557023301960218f, 0.83146961230254524f);
        case 12: return escale(emul_m1pi(a), 0.70710678118654752f);
        case 13: return emul(a, -0.83146961230254524f, 0.55557023301960218f);
        case 14: return emul(a, -0.92387953251128674f, 0.38268343236508978f);
        default: return emul(a, -0.98078528040323043f, 0.19509032201612825f);
    }
}

// a * exp(+2 pi i k / 64), k = 0..63 a compile-time constant after unrolling (radix-64 first stage, N = 16384)
__device__ __forceinline__ float2 mul_w64(float2 a, int k) {
    switch (k & 63) {
        case 0: return a;
        case 1: return emul(a, 0.99518472667219693f, 0.098017140329560604f);
        case 2: return emul(a, 0.98078528040323043f, 0.19509032201612825f);
        case 3: return emul(a, 0.95694033573220882f, 0.29028467725446233f);
        case 4: return emul(a, 0.92387953251128674f, 0.38268343236508978f);
        case 5: return emul(a, 0.88192126434835505f, 0.47139673682599764f);
        case 6: return emul(a, 0.83146961230254524f, 0.55557023301960218f);
        case 7: return emul(a, 0.77301045336273699f, 0.63439328416364549f);
        case 8: return escale(emul_1pi(a), 0.70710678118654752f);
        case 9: return emul(a, 0.63439328416364549f, 0.77301045336273699f);
        case 10: return emul(a, 0.55557023301960229f, 0.83146961230254524f);
        case 11: return emul(a, 0.47139673682599781f, 0.88192126434835494f);
        case 12: return emul(a, 0.38268343236508984f, 0.92387953251128674f);
        case 13: return emul(a, 0.29028467725446233f, 0.95694033573220894f);
        case 14: return emul(a, 0.19509032201612833f, 0.98078528040323043f);
        case 15: return emul(a, 0.09801714032956077f, 0.99518472667219682f);
        case 16: return emul_i(a);
        case 17: return emul(a, -0.098017140329560645f, 0.99518472667219693f);
        case 18: return emul(a, -0.19509032201612819f, 0.98078528040323043f);
        case 19: return emul(a, -0.29028467725446216f, 0.95694033573220894f);
        case 20: return emul(a, -0.38268343236508973f, 0.92387953251128674f);
        case 21: return emul(a, -0.4713967368259977f, 0.88192126434835505f);
        case 22: return emul(a, -0.55557023301960196f, 0.83146961230254546f);
        case 23: return emul(a, -0.63439328416364538f, 0.7730104533627371f);
        case 24: return escale(emul_m1pi(a), 0.70710678118654752f);
        case 25: return emul(a, -0.77301045336273699f, 0.63439328416364549f);
        case 26: return emul(a, -0.83146961230254535f, 0.55557023301960218f);
        case 27: return emul(a, -0.88192126434835494f, 0.47139673682599786f);
        case 28: return emul(a, -0.92387953251128674f, 0.38268343236508989f);
        case 29: return emul(a, -0.95694033573220882f, 0.29028467725446239f);
        case 30: return emul(a, -0.98078528040323043f, 0.19509032201612861f);
        case 31: return emul(a, -0.99518472667219682f, 0.098017140329560826f);
        case 32: return make_float2(-a.x, -a.y);
        case 33: return emul(a, -0.99518472667219693f, -0.09801714032956059f);
        case 34: return emul(a, -0.98078528040323043f, -0.19509032201612836f);
        case 35: return emul(a, -0.95694033573220894f, -0.29028467725446211f);
        case 36: return emul(a, -0.92387953251128685f, -0.38268343236508967f);
        case 37: return emul(a, -0.88192126434835505f, -0.47139673682599764f);
        case 38: return emul(a, -0.83146961230254546f, -0.55557023301960196f);
        case 39: return emul(a, -0.7730104533627371f, -0.63439328416364527f);
        case 40: return emul(a, -0.70710678118654768f, -0.70710678118654746f);
        case 41: return emul(a, -0.63439328416364593f, -0.77301045336273666f);
        case 42: return emul(a, -0.55557023301960218f, -0.83146961230254524f);
        case 43: return emul(a, -0.47139673682599786f, -0.88192126434835494f);
        case 44: return emul(a, -0.38268343236509034f, -0.92387953251128652f);
        case 45: return emul(a, -0.29028467725446244f, -0.95694033573220882f);
        case 46: return emul(a, -0.19509032201612866f, -0.98078528040323032f);
        case 47: return emul(a, -0.098017140329560451f, -0.99518472667219693f);
        case 48: return make_float2(a.y, -a.x);
        case 49: return emul(a, 0.09801714032956009f, -0.99518472667219693f);
        case 50: return emul(a, 0.1950903220161283f, -0.98078528040323043f);
        case 51: return emul(a, 0.29028467725446205f, -0.95694033573220894f);
        case 52: return emul(a, 0.38268343236509f, -0.92387953251128663f);
        case 53: return emul(a, 0.47139673682599759f, -0.88192126434835505f);
        case 54: return emul(a, 0.55557023301960184f, -0.83146961230254546f);
        case 55: return emul(a, 0.6343932841636456f, -0.77301045336273688f);
        case 56: return emul(a, 0.70710678118654735f, -0.70710678118654768f);
        case 57: return emul(a, 0.77301045336273666f, -0.63439328416364593f);
        case 58: return emul(a, 0.83146961230254524f, -0.55557023301960218f);
        case 59: return emul(a, 0.88192126434835483f, -0.47139673682599792f);
        case 60: return emul(a, 0.92387953251128652f, -0.38268343236509039f);
        case 61: return emul(a, 0.95694033573220882f, -0.2902846772544625f);
        case 62: return emul(a, 0.98078528040323032f, -0.19509032201612872f);
        case 63: return emul(a, 0.99518472667219693f, -0.098017140329560506f);
    }
    return a;
}

// In-register inverse DFT of R = 2^LOGR points, decimation in frequency: on return x[i] = Y[brev(i)],
// Y[m'] = sum_m x[m] exp(+2 pi i m m' / R).
template <typename E, int LOGR, bool PACKED = true>
__device__ __forceinline__ void bfly(E* x) {
    constexpr int R = 1 << LOGR;
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int blk = 0; blk < R; blk += 2 * half) {
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const E a = x[blk + j], b = x[blk + j + half];
                x[blk + j] = PACKED ? eadd(a, b) : sadd(a, b);
                x[blk + j + half] = mul_w32(PACKED ? esub(a, b) : ssub(a, b), j * (16 / half));
            }
        }
    }
}

// ---- occupancy masks -----------------------------------------------------------------------------------------
// Storage (FFT-native) tile coordinates.  class_mask[(k nt + tx) 8 + c]: bit m set <=> tile (ty = c + 8 m, tx) of
// plane k holds visibilities (the R0 inputs of pass 1a's butterflies on the rows of class c = (row mod 256) / 32).
// band_mask[k 8 + tx / 32]: bit tx % 32 set <=> some tile of column band tx of plane k does.
// Two sets are kept: set 0 for the mesh as the header describes it ([k][v][u]), set 1 for a mesh stored transposed
// ([k][u][v]: the roles of tx and ty swap).  A WS_GRID_SPARSE mesh is private to this library, so the gridder stores
// it in whichever orientation leaves fewer bands to transform (ctrl[2]): the uv tracks of an east-west-ish array are
// squeezed in v by sin(dec), and a band costs 2 N x 256 B of traffic in pass 1b and pass 2.
// Buffer: ctrl[8] = {bands of set 0, bands of set 1, transposed, ...} | set 0 | set 1; set = class masks, band masks,
// band list.  band list: the k nt + tx of the non-empty bands, in the order they were first marked (ctrl[set] of
// them): the column passes walk that list instead of testing every band of every plane.
// Masks are OR-ed into (chunked gridding accumulates); ws_fft_masks_clear zeroes them.
constexpr int MASK_CTRL = WS_MASK_CTRL;
// Words per class mask (one bit per input of pass 1a's radix-R0 butterfly: R0 = 64 for N = 16384 needs two) and band
// words per plane (one bit per 32-column band: 512 bands for N = 16384).
__host__ __device__ constexpr int class_words(int r0) { return r0 > 32 ? 2 : 1; }
__host__ __device__ constexpr int band_words(int nt) { return nt > 256 ? nt / 32 : 8; }
__device__ __forceinline__ const uint32_t* mask_set(const uint32_t* __restrict__ masks, uint32_t set_words) {
    return masks + MASK_CTRL + (masks[2] ? set_words : 0u);
}
__global__ void __launch_bounds__(256)
k_fft_masks(const uint32_t* __restrict__ rec_start, int nt, int r0, uint32_t n_classes, uint32_t set_words,
            uint32_t* __restrict__ masks) {
    const uint32_t id = blockIdx.x * 256u + threadIdx.x;      // (k nt + band) 8 + c
    if (id >= n_classes) return;
    const int set = blockIdx.y, cw = class_words(r0), bw = band_words(nt);
    uint32_t* class_mask = masks + MASK_CTRL + set * set_words;
    uint32_t* band_mask = class_mask + (size_t)n_classes * cw;
    const int c = id & 7;
    const uint32_t kb = id >> 3;
    const int bs = kb % nt, k = kb / nt;
    const int bl = (bs + nt / 2) & (nt - 1);                  // logical tile coordinate of the band
    uint32_t mask[2] = {0u, 0u};
    for (int m = 0; m < r0; ++m) {
        const int ol = (c + 8 * m + nt / 2) & (nt - 1);       // the other coordinate: ty (set 0) or tx (set 1)
        const uint32_t bin = set == 0 ? ((uint32_t)k * nt + ol) * nt + bl : ((uint32_t)k * nt + bl) * nt + ol;
        if (rec_start[bin + 1] > rec_start[bin]) mask[m >> 5] |= 1u << (m & 31);
    }
    if (mask[0] | mask[1]) {
        for (int i = 0; i < cw; ++i)
            if (mask[i]) atomicOr(class_mask + (size_t)id * cw + i, mask[i]);
        const uint32_t bit = 1u << (bs & 31);
        if (!(atomicOr(band_mask + k * bw + (bs >> 5), bit) & bit)) {
            uint32_t* band_list = band_mask + (n_classes >> 3) / nt * bw;
            band_list[atomicAdd(masks + set, 1u)] = kb;
        }
    }
}
// Degridding (ws_degrid.cu): the planes are DENSE on the way in (rows of the model image times the w screen, transformed
// along u) and only the column bands that hold visibilities -- or border on one that does: a footprint reaches S / 2
// cells into the neighbour tile -- are wanted on the way out.  Such a band gets every class bit, all others none:
// passes 1a / 1b then transform exactly those bands, whole.  bin_start: home counts per (plane, ty, tx), logical tiles.
// As for a WS_GRID_SPARSE mesh the planes are private to the library and are laid out ([k][v][u] or [k][u][v]) so that
// fewer bands are wanted.
__global__ void __launch_bounds__(256)
k_fft_masks_degrid(const uint32_t* __restrict__ bin_start, int nt, int r0, uint32_t n_kb, uint32_t set_words,
                   uint32_t* __restrict__ masks) {
    const uint32_t kb = blockIdx.x * 256u + threadIdx.x;      // k nt + band (storage order)
    if (kb >= n_kb) return;
    const int set = blockIdx.y, cw = class_words(r0), bw = band_words(nt);   // set 0: planes [k][v][u], a band is 32 adjacent u; 1: [k][u][v]
    const int bs = kb % nt, k = kb / nt;
    const int bl = (bs + nt / 2) & (nt - 1);                  // logical tile coordinate of the band
    bool any = false;
    for (int d = -1; d <= 1 && !any; ++d) {
        const int x = bl + d;
        if (x < 0 || x >= nt) continue;
        for (int o = 0; o < nt && !any; ++o) {
            const uint32_t bin = set == 0 ? ((uint32_t)k * nt + o) * nt + x : ((uint32_t)k * nt + x) * nt + o;
            any = bin_start[bin + 1] > bin_start[bin];
        }
    }
    if (!any) return;
    uint32_t* class_mask = masks + MASK_CTRL + set * set_words;
    uint32_t* band_mask = class_mask + (size_t)n_kb * 8u * cw;
    for (int c = 0; c < 8; ++c)
        for (int i = 0; i < cw; ++i) {
            const int left = r0 - 32 * i;
            class_mask[((size_t)kb * 8u + c) * cw + i] = left >= 32 ? 0xFFFFFFFFu : (1u << left) - 1u;
        }
    atomicOr(band_mask + k * bw + (bs >> 5), 1u << (bs & 31));
    uint32_t* band_list = band_mask + n_kb / nt * bw;
    band_list[atomicAdd(masks + set, 1u)] = kb;
}

// the orientation of a WS_GRID_SPARSE mesh: transposed iff that leaves fewer bands (allow = 0: as the header says)
__global__ void k_fft_orient(uint32_t* __restrict__ masks, int allow) { masks[2] = allow && masks[1] < masks[0] ? 1u : 0u; }

// ---- pass 1b: the 256-point column transforms -------------------------------------------------------------------
// Item = (plane, column band tx, block m0 of 256 rows).  Warp w, lane = column.  Stage 1: j in {w, w + 8}, rows
// j + 16 m; stage 2: blocks b in {w, w + 8}, rows 16 b + m; frequency f = b + 16 m' is stored at row 256 m0 + f.
// bit c of the result: class c of the band holds data (0: nothing to do)
template <int LOGN>
__device__ __forceinline__ uint32_t band_classes(const uint32_t* __restrict__ class_mask, uint32_t ktx) {
    constexpr int CW = class_words(1 << (LOGN - 8));
    if (!class_mask) return 0xFFu;
    uint32_t cmask = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        uint32_t any = class_mask[(ktx * 8 + c) * CW];
        if (CW > 1) any |= class_mask[(ktx * 8 + c) * CW + 1];
        cmask |= (any != 0 ? 1u : 0u) << c;
    }
    return cmask;
}
template <int LOGN>
__device__ __forceinline__ void colB_item(float2* __restrict__ grid, const float2* __restrict__ tw, float2* __restrict__ blk,
                                          uint32_t cmask, uint32_t ktx, uint32_t m0) {
    constexpr int N = 1 << LOGN, NT = N / 32;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t tx = ktx % NT, k = ktx / NT;
    float2* p = grid + ((size_t)k * N + m0 * 256) * N + tx * 32 + lane;
    float2 x[32];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int j = w + 8 * i;
#pragma unroll
        for (int m = 0; m < 16; ++m)
            x[i * 16 + m] = (cmask >> (m >> 1)) & 1 ? __ldcs(p + (size_t)(j + 16 * m) * N) : make_float2(0.f, 0.f);
    }
    __syncthreads();          // the previous item's second stage has read `blk`
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int j = w + 8 * i;
        bfly<float2, 4, false>(x + i * 16);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            float2 v = x[i * 16 + r];
            if (r) {
                const float2 tv = __ldg(tw + (brev(r, 4) - 1) * 16 + j);
                v = emul(v, tv.x, tv.y);
            }
            blk[(j + 16 * brev(r, 4)) * 32 + lane] = v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int b = w + 8 * i;
#pragma unroll
        for (int m = 0; m < 16; ++m) x[i * 16 + m] = blk[(16 * b + m) * 32 + lane];
        bfly<float2, 4, false>(x + i * 16);
#pragma unroll
        for (int r = 0; r < 16; ++r) __stcs(p + (size_t)(b + 16 * brev(r, 4)) * N, x[i * 16 + r]);   // read next by pass 2, long after
    }
}

template <int LOGN>
__global__ void __launch_bounds__(CT, 2)
k_fft_colB(float2* __restrict__ grid, const float2* __restrict__ tw, const uint32_t* __restrict__ masks,
           uint32_t set_words, uint32_t n_items) {
    constexpr int R0 = 1 << (LOGN - 8);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2* blk = (float2*)smem_raw;          // [256 rows][32 columns]
    if (!masks) {
        for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x)
            colB_item<LOGN>(grid, tw, blk, 0xFFu, item / R0, item % R0);
        return;
    }
    const uint32_t* class_mask = mask_set(masks, set_words);
    const uint32_t* band_list = class_mask + (set_words - n_items / R0);    // the non-empty (plane, band) pairs
    const uint32_t n_list = masks[masks[2] ? 1 : 0] * R0;
    for (uint32_t item = blockIdx.x; item < n_list; item += gridDim.x) {
        const uint32_t m0 = item % R0, ktx = band_list[item / R0];
        const uint32_t cmask = band_classes<LOGN>(class_mask, ktx);
        if (cmask == 0) continue;
        colB_item<LOGN>(grid, tw, blk, cmask, ktx, m0);
    }
}

// ---- passes 1a + 1b of the listed bands in ONE launch ---------------------------------------------------------------
// Two launches move a band's intermediate (the classes pass 1a writes: 10.8 GB on Large) out to DRAM and back in.  Here
// the items of both passes are handed out from ONE queue (an atomic counter) in an order that puts pass 1b of a band
// LAG bands (COL_LAG_ITEMS items) behind its pass 1a: round r = the IA items of pass 1a of band r, then the IB items of
// pass 1b of band r - LAG.
// A pass-1b item waits until the band's IA pass-1a items have signalled (sync[1 + band]); by then they were handed out at
// least LAG (IA + IB) items ago, so the wait is a formality, and what they wrote (a few bands x 2 MB) is still in L2: DRAM
// sees the occupied tiles once on the way in and the band once on the way out.  No deadlock: only pass-1b items wait, and
// only for items that were handed out earlier, i.e. to CTAs that are running.  sync[] is zeroed before the launch.
constexpr uint32_t COL_LAG_ITEMS = 768;      // in items of 64 KB (8-warp CTAs: x 8 / W for W warps).  Measured on Large (bands of 2 MB, 64 such
                                             // items) with 8-warp CTAs: 6 bands 6.55 ms, 10-16 bands 5.8, 24: 5.9, 48: 6.7 (L2 overflows);
                                             // Extreme (4 MB, 128 items): 2 bands 20.4 ms, 4-6: 16.1, 12: 16.5, 24: 18.8
                                             // With 4-warp CTAs: Large 10-12 bands 5.26 ms, 16: 5.30, 20: 5.43; Extreme 3: 15.3, 4: 14.5, 6: 14.4, 8: 14.6, 10: 15.0
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__host__ __device__ constexpr bool cols_fused(int logn) { return logn >= 9 && logn <= 14; }
constexpr int COLS_W = 4;                 // warps per CTA of k_fft_cols
// CTAs of W = 4 warps, four per SM (128 registers per thread either way), with items to match -- pass 1a: W rows j of the band
// (N = 16384: W / 2 rows, two warps each: one forms a + b and leaves the even outputs of the radix-64 step, the other
// (a - b) W_64^m and the odd ones, so that a thread holds 32 points, not 64; both read all 64 inputs, the second read hits L1,
// and the barrier keeps the in-place stores of one behind the loads of the other); pass 1b: 256 rows x 4 W columns.  Every
// item is a load phase, a compute phase and a store phase with barriers between them; four small CTAs whose phases fall at
// different times keep an SM busier than two large ones (measured, Large / Extreme: W = 8: 5.74 / 16.0 ms, W = 4: 5.26 / 14.2,
// W = 2: 5.87 / 15.6 -- 64-byte row segments).
template <int LOGN, int W>
__device__ __forceinline__ void colsA_item(float2* __restrict__ grid, const float2* __restrict__ tw,
                                           const uint32_t* __restrict__ class_mask, uint32_t ktx, uint32_t jq) {
    constexpr int N = 1 << LOGN, LR0 = LOGN - 8, R0 = 1 << LR0, NT = N / 32;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t tx = ktx % NT, k = ktx / NT;
    if constexpr (LOGN == 14) {
        const int h = w / (W / 2), j = (int)jq * (W / 2) + (w % (W / 2));
        float2* p = grid + ((size_t)k * N + j) * N + tx * 32 + lane;
        const uint32_t cls = jq / (64 / W);
        const uint32_t m_lo = class_mask ? class_mask[(ktx * 8 + cls) * 2] : 0xFFFFFFFFu;      // (NULL: a dense mesh)
        const uint32_t m_hi = class_mask ? class_mask[(ktx * 8 + cls) * 2 + 1] : 0xFFFFFFFFu;
        if ((m_lo | m_hi) == 0) return;                   // (the whole CTA: one class)
        float2 x[32];
#pragma unroll
        for (int m = 0; m < 32; ++m) x[m] = (m_lo >> m) & 1 ? __ldcs(p + (size_t)m * 256 * N) : make_float2(0.f, 0.f);
#pragma unroll
        for (int m = 0; m < 32; ++m) {
            const float2 b = (m_hi >> m) & 1 ? __ldcs(p + (size_t)(m + 32) * 256 * N) : make_float2(0.f, 0.f);
            x[m] = h ? mul_w64(ssub(x[m], b), m) : sadd(x[m], b);
        }
        __syncthreads();
        bfly<float2, 5, false>(x);
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const int f = 2 * brev(r, 5) + h;
            if (f) {
                const float2 tv = __ldg(tw + (f - 1) * 256 + j);
                x[r] = emul(x[r], tv.x, tv.y);
            }
        }
#pragma unroll
        for (int r = 0; r < 32; ++r) p[(size_t)(2 * brev(r, 5) + h) * 256 * N] = x[r];
    } else {
        const int j = (int)jq * W + w;
        float2* p = grid + ((size_t)k * N + j) * N + tx * 32 + lane;
        const uint32_t mask = class_mask ? class_mask[ktx * 8 + jq / (32 / W)] : 0xFFFFFFFFu;
        if (mask == 0) return;
        float2 x[R0];
#pragma unroll
        for (int m = 0; m < R0; ++m) x[m] = (mask >> m) & 1 ? __ldcs(p + (size_t)m * 256 * N) : make_float2(0.f, 0.f);
        bfly<float2, LR0, false>(x);
#pragma unroll
        for (int r = 1; r < R0; ++r) {
            const float2 tv = __ldg(tw + (brev(r, LR0) - 1) * 256 + j);
            x[r] = emul(x[r], tv.x, tv.y);
        }
#pragma unroll
        for (int r = 0; r < R0; ++r) p[(size_t)brev(r, LR0) * 256 * N] = x[r];
    }
}
// pass 1b of 4 W columns of a band block: lane = (column c, jj), warp w: rows j = (32 / COLS) w + jj + 8 i, i < 2, as in colB_item;
// the rows were written by other CTAs of the SAME launch: read them past L1 (ld.global.cg), which may hold the lines as they
// were when a pass-1a item on this SM read them
template <int LOGN, int W>
__device__ __forceinline__ void colsB_item(float2* __restrict__ grid, const float2* __restrict__ tw, float2* __restrict__ blk,
                                           uint32_t cmask, uint32_t ktx, uint32_t item) {
    constexpr int N = 1 << LOGN, NT = N / 32, COLS = 4 * W, JPW = 32 / COLS, PARTS = 32 / COLS;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, c = lane & (COLS - 1), jj = lane / COLS;
    const uint32_t tx = ktx % NT, k = ktx / NT, m0 = item / PARTS, h = item % PARTS;
    float2* p = grid + ((size_t)k * N + m0 * 256) * N + tx * 32 + h * COLS + c;
    float2 x[32];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int j = JPW * w + jj + 8 * i;
#pragma unroll
        for (int m = 0; m < 16; ++m)
            x[i * 16 + m] = (cmask >> (m >> 1)) & 1 ? __ldcg(p + (size_t)(j + 16 * m) * N) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int j = JPW * w + jj + 8 * i;
        bfly<float2, 4, false>(x + i * 16);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            float2 v = x[i * 16 + r];
            if (r) {
                const float2 tv = __ldg(tw + (brev(r, 4) - 1) * 16 + j);
                v = emul(v, tv.x, tv.y);
            }
            blk[(j + 16 * brev(r, 4)) * COLS + c] = v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int b = JPW * w + jj + 8 * i;
#pragma unroll
        for (int m = 0; m < 16; ++m) x[i * 16 + m] = blk[(16 * b + m) * COLS + c];
        bfly<float2, 4, false>(x + i * 16);
#pragma unroll
        for (int r = 0; r < 16; ++r) __stcs(p + (size_t)(b + 16 * brev(r, 4)) * N, x[i * 16 + r]);
    }
}

template <int LOGN, int W>
__global__ void __launch_bounds__(32 * W, 16 / W)
k_fft_cols(float2* __restrict__ grid, const float2* __restrict__ tw_a, const float2* __restrict__ tw_b,
            const uint32_t* __restrict__ masks, uint32_t set_words, uint32_t n_kb, uint32_t* __restrict__ sync) {
    constexpr uint32_t R0 = 1u << (LOGN - 8), IA = (LOGN == 14 ? 512 : 256) / W, IB = R0 * 8 / W, PER = IA + IB, LAG = (8 / W) * COL_LAG_ITEMS / PER;
    // masks == NULL: a dense mesh, every band of every plane in storage order
    const uint32_t* class_mask = masks ? mask_set(masks, set_words) : nullptr;
    const uint32_t* band_list = masks ? class_mask + (set_words - n_kb) : nullptr;
    const uint32_t n = masks ? masks[masks[2] ? 1 : 0] : n_kb;       // listed bands
    const uint32_t lag = n < LAG ? n : LAG;
    const uint32_t head = lag * IA, body = (n - lag) * PER, total = n * PER;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2* blk = (float2*)smem_raw;          // [256 rows][4 W columns]
    __shared__ uint32_t s_q[2];               // the item in hand and the next one, by the parity of the iteration
    uint32_t next = 0;
    if (threadIdx.x == 0) s_q[0] = atomicAdd(sync, 1u);
    __syncthreads();
    for (uint32_t it = 0;; ++it) {
        const uint32_t q = s_q[it & 1];
        if (q >= total) break;
        if (threadIdx.x == 0) next = atomicAdd(sync, 1u);
        bool pass_a;
        uint32_t band, item;
        if (q < head) {
            pass_a = true, band = q / IA, item = q % IA;
        } else if (q < head + body) {
            const uint32_t r = (q - head) / PER, rem = (q - head) % PER;
            pass_a = rem < IA;
            band = pass_a ? lag + r : r;
            item = pass_a ? rem : rem - IA;
        } else {
            pass_a = false, band = n - lag + (q - head - body) / IB, item = (q - head - body) % IB;
        }
        const uint32_t ktx = band_list ? band_list[band] : band;
        if (pass_a) {
            colsA_item<LOGN, W>(grid, tw_a, class_mask, ktx, item);
            __syncthreads();
            if (threadIdx.x == 0) {
                __threadfence();
                atomicAdd(sync + 1 + band, 1u);
            }
        } else {
            const uint32_t cmask = band_classes<LOGN>(class_mask, ktx);
            if (cmask != 0) {
                if (threadIdx.x == 0)
                    while (ld_acquire(sync + 1 + band) < IA) __nanosleep(200);
                __syncthreads();
                colsB_item<LOGN, W>(grid, tw_b, blk, cmask, ktx, item);
            }
        }
        if (threadIdx.x == 0) s_q[(it + 1) & 1] = next;
        __syncthreads();
    }
}

// ---- TMA bulk copy + mbarrier (PTX) ------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- pass 2: rows + fused w-correction -------------------------------------------------------------------------
// A CTA owns "super-row" sr = 8192 contiguous points = 8192 / N whole row positions of every plane; row position
// `pos` holds v-frequency (pos >> 8) + R0 (pos & 255) (pass 1b).  Planes are visited from the top one down so that
// the phase screen is applied by Horner's rule: h <- h r + P_k, r = exp(2 pi i dw t); every WC_SPAN planes the
// chain is closed with the exactly evaluated phase of its lowest plane and restarted.
//
// 512 threads x 16 points.  Stage s, radix R: butterfly b takes the points base + m Q (Q = L / R, base =
// (b / Q) L + b mod Q) and leaves Y[m'] W_L^(j m') at base + m' Q: in place.  For N >= 4096 the CTA is two groups
// of 8 warps that share nothing but the landing buffer, each with its own named barrier, so that one group's
// exchanges overlap the other's arithmetic: N = 4096: a group per row; N = 8192: the first stage is radix 32 with
// each butterfly split over the two groups by the parity of its outputs (both read its 32 inputs; the even half
// is the 16-point transform of a + b, the odd half that of (a - b) W_32^m), after which the blocks of even and
// odd first digit are separate problems.
// band_mask (or NULL = dense): only the non-empty 32-column bands of a plane are copied in, as maximal runs; a
// band that is empty now but was filled by the previous copy is cleared first; a plane without any is skipped.
template <int BW>
__device__ __forceinline__ bool any_band_of(const uint32_t* __restrict__ band_mask, int k, int nt) {
    uint32_t o = 0;
#pragma unroll
    for (int i = 0; i < BW; ++i) {
        const int lo = 32 * i;
        const uint32_t full = nt >= lo + 32 ? 0xFFFFFFFFu : (nt > lo ? (1u << (nt - lo)) - 1u : 0u);
        o |= band_mask ? (band_mask[k * BW + i] & full) : full;
    }
    return o != 0;
}
template <int LOGN>
struct RowCfg {
    static constexpr int N = 1 << LOGN, NT = N / 32, R0 = 1 << (LOGN - 8);
    static constexpr int LAND = N > PTS ? N : PTS;    // points the landing buffer holds: whole rows, at least 8192 points
    static constexpr int ROWS = LAND / N;
    static constexpr int S = n_stages(LOGN);
    static constexpr bool GROUPED = LOGN >= 12;       // two independent 8-warp groups
    static constexpr bool SPLIT32 = LOGN == 13;       // first stage: radix 32 split over the groups
    static constexpr bool SPLIT64 = LOGN == 14;       // first stage: radix 64 split over the groups of TWO CTAs (by output parity)
    static constexpr int ITEMS_PER_ROW = SPLIT64 ? 2 : 1;
    static constexpr int BW = band_words(NT);
    static constexpr int NBUF = 1;                    // landing buffers (2 works where the shared memory allows it; see tw_factored)
    static constexpr int LRL = log2r(LOGN, S - 1);    // last stage
};

// butterfly i of thread u in stage s (s >= 1, or any stage when not SPLIT32)
template <int LOGN>
__device__ __forceinline__ int bfly_id(int u, int i) {
    if constexpr (RowCfg<LOGN>::SPLIT32 || RowCfg<LOGN>::SPLIT64) return (((u & 255) >> 4) << 5) | ((u >> 8) << 4) | (u & 15);   // first digit parity = group
    return u + FT * i;
}
template <int LOGL, int LOGR>
__device__ __forceinline__ int stage_base(int b) {
    constexpr int LOGQ = LOGL - LOGR;
    return ((b >> LOGQ) << LOGL) + (b & ((1 << LOGQ) - 1));
}

// generic stage on the padded work buffer (or, FIRST, from the unpadded landing buffer): load, butterfly, and unless
// LAST twiddle + store.  After the LAST stage x[i R + r] is position (bfly_id(u, i) << LOGR) + brev(r).
template <int LOGN, int STAGE, bool FIRST, bool LAST>
__device__ __forceinline__ void row_stage(float2* x, const float2* __restrict__ src, float2* __restrict__ work,
                                          const float2* __restrict__ tw, int u) {
    constexpr int LOGL = log2l(LOGN, STAGE), LOGR = log2r(LOGN, STAGE), LOGQ = LOGL - LOGR, R = 1 << LOGR, Q = 1 << LOGQ;
#pragma unroll
    for (int i = 0; i < EPT / R; ++i) {
        const int b = bfly_id<LOGN>(u, i), base = stage_base<LOGL, LOGR>(b);
        float2* xi = x + i * R;
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const int p = base + (m << LOGQ);
            xi[m] = src[FIRST ? p : pad(p)];
        }
    }
    if constexpr (!FIRST) {  // (FIRST: the caller releases the landing buffer before the arithmetic)
#pragma unroll
    for (int i = 0; i < EPT / R; ++i) {
        const int b = bfly_id<LOGN>(u, i), base = stage_base<LOGL, LOGR>(b);
        float2* xi = x + i * R;
        bfly<float2, LOGR>(xi);
        if (!LAST) {
            const int j = b & (Q - 1);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float2 v = xi[r];
                if (r) {
                    const float2 w = tw[tw_offset(LOGN, STAGE) + (brev(r, LOGR) - 1) * Q + j];
                    v = emul(v, w.x, w.y);
                }
                work[pad(base + (brev(r, LOGR) << LOGQ))] = v;
            }
        }
    }
    }
}
// arithmetic + store of a first stage whose inputs are already in x[]
template <int LOGN>
__device__ __forceinline__ void first_stage_finish(float2* x, float2* __restrict__ work, const float2* __restrict__ tw, int u) {
    constexpr int LOGL = LOGN, LOGR = log2r(LOGN, 0), LOGQ = LOGL - LOGR, R = 1 << LOGR, Q = 1 << LOGQ;
    static_assert(R == EPT, "first stage: one radix-16 butterfly per thread");
    const int b = u, base = stage_base<LOGL, LOGR>(b), j = b & (Q - 1);
    bfly<float2, LOGR>(x);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        float2 v = x[r];
        if (r) {
            const float2 w = tw[(brev(r, LOGR) - 1) * Q + j];
            v = emul(v, w.x, w.y);
        }
        work[pad(base + (brev(r, LOGR) << LOGQ))] = v;
    }
}

// row (within the super-row) and frequency of register slot `slot` after the last stage
template <int LOGN>
__device__ __forceinline__ int final_pos(int slot, int u);
template <int LOGN>
__device__ __forceinline__ int slot_row(int slot, int u) {
    if constexpr (LOGN >= 13) return 0;
    else if constexpr (LOGN == 12) return u >> 8;
    else return final_pos<LOGN>(slot, u) >> LOGN;
}
// (par: N = 16384 only, the parity of the output frequencies this CTA computes)
template <int LOGN>
__device__ __forceinline__ int slot_freq(int slot, int u, int par) {
    const int ug = u & 255, g = u >> 8;
    if constexpr (LOGN == 14) return (2 * (2 * (ug >> 4) + g) + par) + 64 * (ug & 15) + 1024 * brev(slot, 4);
    else if constexpr (LOGN == 13) return (2 * (ug >> 4) + g) + 32 * (ug & 15) + 512 * brev(slot, 4);
    else if constexpr (LOGN == 12) return (ug >> 4) + 16 * (ug & 15) + 256 * brev(slot, 4);
    else return freq_of<LOGN>(final_pos<LOGN>(slot, u) & ((1 << LOGN) - 1));
}
// CTA position of register slot `slot` after the last stage (generic path)
template <int LOGN>
__device__ __forceinline__ int final_pos(int slot, int u) {
    constexpr int LRL = RowCfg<LOGN>::LRL, R = 1 << LRL;
    return (bfly_id<LOGN>(u, slot / R) << LRL) + brev(slot % R, LRL);
}

// ---- the two-group path (N = 4096, 8192) with every shared-memory address in the form base + constant ---------
// Padded index of position blk * 256 + x (x < 256) is blk * 272 + x + (x >> 4).  Group g, thread ug < 256:
//   first stage   j = ug: 32 (N = 8192) or 16 (N = 4096, row g) inputs j + 256 m from `landing`; output digit d goes
//                 to block d (N = 8192: d = 2 brev(r) + g; N = 4096: block 16 g + brev(r)) at x = j;
//   second stage  block blk = (N = 8192: 2 (ug >> 4) + g; N = 4096: 16 g + (ug >> 4)), jj = ug & 15, points jj + 16 m;
//   third stage   points 16 jj + m of the same block: they were written by the 16 lanes that share blk, so the
//                 exchange between the last two stages needs a warp barrier only.
template <int LOGN>
struct Grouped {
    static constexpr bool SPLIT32 = LOGN == 13, SPLIT64 = LOGN == 14, SPLIT = SPLIT32 || SPLIT64;
    __device__ static __forceinline__ int blk(int ug, int g) { return SPLIT ? 2 * (ug >> 4) + g : 16 * g + (ug >> 4); }
    // N = 16384, first stage radix 64, m' = m + 16 t: output digit d = 4 d' + q gets
    //   Y[d] = sum_m [ (sum_t x[m + 16 t] i^(t q)) W_64^(m q) ] W_16^(m d'),
    // so a thread that wants the outputs of ONE q (= 2 g + parity of the CTA) forms z[m] from four inputs and runs
    // the 16-point butterfly over m.
    template <int Q>
    __device__ static __forceinline__ void load_first64(float2* x, const float2* __restrict__ in) {
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            const float2 x0 = in[256 * m], x1 = in[256 * m + 4096], x2 = in[256 * m + 8192], x3 = in[256 * m + 12288];
            float2 z;
            if (Q == 0) z = eadd(eadd(x0, x2), eadd(x1, x3));
            else if (Q == 1) z = eadd(esub(x0, x2), emul_i(esub(x1, x3)));
            else if (Q == 2) z = esub(eadd(x0, x2), eadd(x1, x3));
            else z = esub(esub(x0, x2), emul_i(esub(x1, x3)));
            x[m] = mul_w64(z, Q * m);
        }
    }
    __device__ static __forceinline__ void load_first(float2* x, const float2* __restrict__ landing, int ug, int g, int par) {
        if constexpr (SPLIT64) {
            const float2* in = landing + ug;
            switch (2 * g + par) {                 // warp-uniform
                case 0: load_first64<0>(x, in); break;
                case 1: load_first64<1>(x, in); break;
                case 2: load_first64<2>(x, in); break;
                default: load_first64<3>(x, in); break;
            }
        } else if constexpr (SPLIT32) {
            const float2* in = landing + ug;
            if (g == 0) {
#pragma unroll
                for (int m = 0; m < 16; ++m) x[m] = eadd(in[256 * m], in[256 * (m + 16)]);
            } else {
#pragma unroll
                for (int m = 0; m < 16; ++m) x[m] = mul_w32(esub(in[256 * m], in[256 * (m + 16)]), m);
            }
        } else {
            const float2* in = landing + g * 4096 + ug;
#pragma unroll
            for (int m = 0; m < 16; ++m) x[m] = in[256 * m];
        }
    }
    // tw_factored (N = 16384): no room for the whole first-stage table (63 x 256 entries) beside the 128 KB landing buffer.  A
    // thread's outputs are the digits d = M p + q, p = 4 a + b < 16 (M = 4, q = 2 g + parity of the CTA), and
    // W_N^(ug d) = W_N^(ug (M b + q)) W_N^(4 M a ug): two factors from two small tables in shared memory (8 + 3 x 256 entries
    // per CTA, 7 loads per thread and plane instead of 15; two roundings instead of one).  As register constants they spilled.
    __device__ static __forceinline__ void finish_first(float2* x, float2* __restrict__ work, const float2* __restrict__ tw,
                                                        int ug, int g) {
        bfly<float2, 4>(x);
        if constexpr (SPLIT && tw_factored(LOGN)) {
            float2* out = work + g * 272 + ug + (ug >> 4);
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                constexpr int n1 = tw_entries(LOGN) - tw_offset(LOGN, 1);
                const float2 tb = tw[n1 + 768 + (g * 4 + b) * 256 + ug];                  // W_N^(ug (M b + q))
#pragma unroll
                for (int a = 0; a < 4; ++a) {
                    const int pq = 4 * a + b, r = brev(pq, 4);
                    float2 v = emul(x[r], tb.x, tb.y);
                    if (a) {
                        const float2 pa = tw[n1 + (a - 1) * 256 + ug];                     // W_N^(4 M a ug)
                        v = emul(v, pa.x, pa.y);
                    }
                    out[pq * 544] = v;
                }
            }
        } else if constexpr (SPLIT32) {
            float2* out = work + g * 272 + ug + (ug >> 4);
            const float2* t = tw + ug + (g - 1) * 256;              // tw[(d - 1) 256 + j], d = 2 brev(r) + g
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                float2 v = x[r];
                if (r) {
                    const float2 w = t[brev(r, 4) * 512];
                    v = emul(v, w.x, w.y);
                } else if (g) {
                    const float2 w = t[0];
                    v = emul(v, w.x, w.y);
                }
                out[brev(r, 4) * 544] = v;
            }
        } else {
            float2* out = work + g * (16 * 272) + ug + (ug >> 4);
            const float2* t = tw + ug - 256;                        // tw[(m' - 1) 256 + j]
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                float2 v = x[r];
                if (r) {
                    const float2 w = t[brev(r, 4) * 256];
                    v = emul(v, w.x, w.y);
                }
                out[brev(r, 4) * 272] = v;
            }
        }
    }
    __device__ static __forceinline__ void second_third(float2* x, float2* __restrict__ work, const float2* __restrict__ tw,
                                                        int ug, int g) {
        const int jj = ug & 15;
        float2* b1 = work + blk(ug, g) * 272 + jj;
        const float2* t = tw + tw_smem_off1(LOGN) + jj - 16;        // tw1[(m' - 1) 16 + jj]
#pragma unroll
        for (int m = 0; m < 16; ++m) x[m] = b1[17 * m];
        bfly<float2, 4>(x);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            float2 v = x[r];
            if (r) {
                const float2 w = t[brev(r, 4) * 16];
                v = emul(v, w.x, w.y);
            }
            b1[17 * brev(r, 4)] = v;
        }
        __syncwarp();
        const float2* b2 = work + blk(ug, g) * 272 + 17 * jj;
#pragma unroll
        for (int m = 0; m < 16; ++m) x[m] = b2[m];
        bfly<float2, 4>(x);
    }
};

// Work item -> super-row.  For N = 8192 (one row position per super-row) items are taken in the order of the
// FREQUENCY the row position holds, pos = (F mod R0) 256 + F / R0, so that the CTAs running side by side own adjacent
// lines of the image: when the mesh is transposed their 8-byte pixels share 32-byte sectors and meet in L2.
// N = 16384: two items per row (even / odd output frequencies), taken by neighbouring CTAs at the same time, so that the
// second reader of the row finds it in L2.
template <int LOGN>
__device__ __forceinline__ uint32_t super_row_of(uint32_t item) {
    constexpr int LR0 = LOGN - 8;
    if constexpr (RowCfg<LOGN>::SPLIT64) item >>= 1;
    if constexpr (RowCfg<LOGN>::ROWS == 1) return ((item & ((1u << LR0) - 1u)) << 8) | (item >> LR0);
    else return item;
}

// ---- producer warp of the row kernels: clears the bands of a landing buffer that the last copy filled and the next one
// will not, then brings the non-empty bands of the next plane in.  Lane wi < BW owns mask word wi (32 bands = 8 KB per row)
// and issues one bulk copy per maximal run of set bits.
template <int LOGN>
__device__ __forceinline__ void rows_producer(float2* landing0, uint64_t* full, uint64_t* empty, const uint32_t* s_any,
                                              const uint32_t* __restrict__ band_mask, const float2* __restrict__ planes, int nw,
                                              uint32_t item_lo, uint32_t n_super, int lane) {
    using C = RowCfg<LOGN>;
    constexpr int N = C::N, ROWS = C::ROWS, NT = C::NT, LAND = C::LAND, BW = C::BW, NBUF = C::NBUF;
    const size_t plane_elems = (size_t)N * N;
    uint32_t was[NBUF], seq = 0;                      // seq: planes copied so far; plane seq lands in buffer seq % NBUF
#pragma unroll
    for (int i = 0; i < NBUF; ++i) was[i] = 0;
    for (uint32_t it = item_lo + blockIdx.x; it < n_super; it += gridDim.x) {
        const uint32_t sr = super_row_of<LOGN>(it);
        for (int k = nw - 1; k >= 0; --k) {
            if (!((s_any[k >> 5] >> (k & 31)) & 1u)) continue;
            uint32_t now = 0;
            if (lane < BW) {
                const int lo = 32 * lane;
                const uint32_t fullw = NT >= lo + 32 ? 0xFFFFFFFFu : (NT > lo ? (1u << (NT - lo)) - 1u : 0u);
                now = band_mask ? (__ldg(band_mask + k * BW + lane) & fullw) : fullw;
            }
            // what needs neither `landing` nor the barrier happens before the wait for the consumers
            uint32_t n_bands = __popc(now);
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) n_bands += __shfl_xor_sync(0xffffffffu, n_bands, d);
            const uint32_t buf = seq % NBUF, use = seq / NBUF;       // this buffer's use-th filling
            float2* landing = landing0 + buf * LAND;
            const uint32_t stale = (NBUF == 2 && buf ? was[NBUF - 1] : was[0]) & ~now;
            const bool any_stale = __any_sync(0xffffffffu, stale != 0);
            if (use > 0) {
                while (!mbar_try_wait(empty + buf, (use - 1) & 1u)) {}
            }
            // stale bands are cleared BEFORE the arrive: its release then orders the zeroing stores ahead of the
            // consumers' reads (they acquire `full`), whatever the bulk copies' timing
            if (any_stale) {
#pragma unroll
                for (int wi = 0; wi < BW; ++wi) {
                    uint32_t z = __shfl_sync(0xffffffffu, stale, wi);
                    while (z) {
                        const int b = wi * 32 + __ffs(z) - 1;
                        z &= z - 1;
                        for (int r = 0; r < ROWS; ++r) landing[r * N + b * 32 + lane] = make_float2(0.f, 0.f);
                    }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            }
            __syncwarp();
            if (lane == 0) mbar_expect_tx(full + buf, n_bands * 256u * ROWS);     // (the previous phase is complete now)
            __syncwarp();
            const char* src = (const char*)(planes + (size_t)k * plane_elems + (size_t)sr * LAND);
            uint32_t m = now;
            while (m) {
                const int b0 = __ffs(m) - 1;
                const uint32_t inv = ~(m >> b0);
                const int len = inv ? __ffs(inv) - 1 : 32;
                m &= ~((len == 32 ? 0xFFFFFFFFu : (1u << len) - 1u) << b0);
                const size_t off = (size_t)(lane * 32 + b0) * 256;
                for (int r = 0; r < ROWS; ++r)
                    bulk_g2s((char*)landing + (size_t)r * N * 8 + off, src + (size_t)r * N * 8 + off, len * 256, full + buf);
            }
            if (NBUF == 2 && buf) was[NBUF - 1] = now;
            else was[0] = now;
            ++seq;
        }
    }
}

template <int LOGN>
__global__ void __launch_bounds__(FT + PT, 1)
k_fft_rows(const __grid_constant__ WcParams prm, const float2* __restrict__ planes, float2* __restrict__ image,
           float* __restrict__ dirty, int accumulate, const float2* __restrict__ tw_g, const float2* __restrict__ tc_g,
           const uint32_t* __restrict__ masks, uint32_t set_words, uint32_t item_lo, uint32_t n_super) {
    using C = RowCfg<LOGN>;
    constexpr int N = C::N, ROWS = C::ROWS, NT = C::NT, R0 = C::R0, LAND = C::LAND, BW = C::BW, NBUF = C::NBUF;
    // occupancy: the band masks of the orientation the mesh is stored in; transposed: the mesh is [k][u][v], i.e. a
    // row position is a u-frequency and the image comes out transposed (the phase screen is symmetric in l and m)
    const uint32_t* band_mask =
        masks ? mask_set(masks, set_words) + (uint32_t)prm.n_wplanes * (uint32_t)(NT * 8 * class_words(R0)) : nullptr;
    const bool transposed = masks && masks[2];
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2* landing0 = (float2*)smem_raw;                               // NBUF buffers of LAND points
    float2* work = landing0 + NBUF * LAND;
    float2* tw = work + PAD_PTS;
    uint64_t* full = (uint64_t*)(tw + ((tw_smem_entries(LOGN) + 1) & ~1));   // [NBUF] the copy of a plane has landed
    uint64_t* empty = full + NBUF;                                      // [NBUF] every group has consumed it
    uint32_t* s_any = (uint32_t*)(empty + NBUF);                        // bit k: plane k has a non-empty band
    const int u = threadIdx.x, g = u >> 8;
    const int par = C::SPLIT64 ? (int)(blockIdx.x & 1u) : 0;           // (the grid is even: every item of a CTA has its parity)
    const int nw = prm.n_wplanes;
    if constexpr (tw_factored(LOGN)) {
        constexpr int n1 = tw_entries(LOGN) - tw_offset(LOGN, 1);
        for (int i = u; i < n1; i += FT + PT) tw[i] = tw_g[i];
        for (int i = u; i < 768; i += FT + PT) tw[n1 + i] = tc_g[16 * 256 + i];
        for (int i = u; i < 2048; i += FT + PT)        // [g][b][ug] <- [q = 2 g + par][b][ug]
            tw[n1 + 768 + i] = tc_g[((2 * (i >> 10) + par) * 4 + ((i >> 8) & 3)) * 256 + (i & 255)];
    } else {
        for (int i = u; i < tw_smem_entries(LOGN); i += FT + PT) tw[i] = tw_g[i];
    }
    for (int i = u; i < NBUF * LAND; i += FT + PT) landing0[i] = make_float2(0.f, 0.f);
    for (int k0 = 0; k0 < nw; k0 += FT + PT) {       // (FT + PT is a multiple of 32: one ballot per mask word)
        const int k = k0 + u;
        bool any = false;
        if (k < nw) any = any_band_of<BW>(band_mask, k, NT);
        const uint32_t bits = __ballot_sync(0xffffffffu, any);
        if ((u & 31) == 0 && k < nw) s_any[k >> 5] = bits;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (u == 0) {
        for (int i = 0; i < NBUF; ++i) {
            mbar_init(full + i, 1);
            mbar_init(empty + i, C::GROUPED ? 2 : 1);
        }
    }
    __syncthreads();
    if (item_lo + blockIdx.x >= n_super) return;       // items [item_lo, n_super) belong to this launch

    if (u >= FT) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (u >= FT + 32) return;
        rows_producer<LOGN>(landing0, full, empty, s_any, band_mask, planes, nw, item_lo, n_super, u & 31);
        return;
    }

    // ---- the 16 compute warps (they take over the registers the producer's warpgroup gave back: the pool is the CTA's
    // launch allocation, 640 x 96 registers, so 112 is the most that 512 threads can take; asking for more blocks forever.
    // ptxas honours the raised budget in this region -- without setmaxnreg, 544 threads compile to 96 registers and spill)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
    auto cta_sync = [&]() { asm volatile("bar.sync 3, %0;" ::"r"(FT) : "memory"); };     // (the producer is not part of it)
    auto group_sync = [&]() {
        if (C::GROUPED) asm volatile("bar.sync %0, %1;" ::"r"(1 + g), "r"(GT) : "memory");
        else cta_sync();
    };
    uint32_t seq = 0;                      // planes consumed so far (the producer's count, same order)
    const int top_span_lo = ((nw - 1) / WC_SPAN) * WC_SPAN;
    for (uint32_t it = item_lo + blockIdx.x; it < n_super; it += gridDim.x) {
        const uint32_t sr = super_row_of<LOGN>(it);
        float2 rot[EPT], h[EPT];
#pragma unroll
        for (int s = 0; s < EPT; ++s) {
            const int pos = (int)sr * ROWS + slot_row<LOGN>(s, u);
            const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
            const int p = (slot_freq<LOGN>(s, u, par) + N / 2) & (N - 1);
            bool inside;
            const double tt = ws_n_minus_1(prm, q, p, &inside);
            rot[s] = ws_expi_turns(prm.dw * tt);
            h[s] = make_float2(0.f, 0.f);
        }
        for (int k = nw - 1; k >= 0; --k) {
            float2 x[EPT];
            if ((s_any[k >> 5] >> (k & 31)) & 1u) {      // CTA-uniform: the plane has data, its copy is under way
                const uint32_t buf = seq % NBUF, use = seq / NBUF;
                const float2* landing = landing0 + buf * LAND;
                while (!mbar_try_wait(full + buf, use & 1u)) {}
                ++seq;
                // ---- first stage: inputs from the landing buffer
                if constexpr (C::GROUPED) Grouped<LOGN>::load_first(x, landing, u & 255, g, par);
                else row_stage<LOGN, 0, true, false>(x, landing, work, tw, u);
                group_sync();          // this group is done with `landing` (and with last plane's reads of `work`)
                if ((u & 255) == 0 && (C::GROUPED || g == 0))
                    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(empty + buf)) : "memory");
                // ---- arithmetic, twiddles, exchanges
                if constexpr (C::GROUPED) {
                    Grouped<LOGN>::finish_first(x, work, tw, u & 255, g);
                    group_sync();
                    Grouped<LOGN>::second_third(x, work, tw, u & 255, g);
                } else {
                    first_stage_finish<LOGN>(x, work, tw, u);
                    group_sync();
                    if constexpr (C::S == 3) {
                        row_stage<LOGN, 1, false, false>(x, work, work, tw, u);
                        group_sync();
                    }
                    row_stage<LOGN, C::S - 1, false, true>(x, work, work, tw, u);
                }
#pragma unroll
                for (int s = 0; s < EPT; ++s) h[s] = ws_horner(h[s], rot[s], x[s].x, x[s].y);
            } else {                          // empty plane: P_k = 0
#pragma unroll
                for (int s = 0; s < EPT; ++s) h[s] = ws_cmul(h[s], rot[s]);
            }
            if (k % WC_SPAN != 0) continue;
            // close the chain: x <- E h, E = exp(2 pi i (w0 + k dw) t) evaluated exactly
#pragma unroll
            for (int s = 0; s < EPT; ++s) {
                const int pos = (int)sr * ROWS + slot_row<LOGN>(s, u);
                const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
                const int p = (slot_freq<LOGN>(s, u, par) + N / 2) & (N - 1);
                bool inside;
                const double tt = ws_n_minus_1(prm, q, p, &inside);
                x[s] = ws_cmul(h[s], ws_expi_turns((prm.w0 + (double)k * prm.dw) * tt));
                if (!inside) x[s] = make_float2(0.f, 0.f);
                h[s] = make_float2(0.f, 0.f);
            }
            if (transposed) {      // pixel (row position, frequency) belongs at image[frequency][row position]
#pragma unroll
                for (int s = 0; s < EPT; ++s) {
                    const int pos = (int)sr * ROWS + slot_row<LOGN>(s, u);
                    const int a = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
                    const int b = (slot_freq<LOGN>(s, u, par) + N / 2) & (N - 1);
                    const size_t o = (size_t)b * N + a;
                    float2 v = x[s];
                    if (accumulate || k != top_span_lo) {
                        const float2 old = image[o];
                        v.x += old.x; v.y += old.y;
                    }
                    image[o] = v;
                    if (dirty && k == 0) dirty[o] = v.x;
                }
                continue;
            }
            // un-permute through `work`: natural order along the rows of the centred image (both groups)
            cta_sync();
            if constexpr (C::SPLIT64) {
                // this CTA holds every second pixel of the line (those of its parity): work[i] = pixel 2 i + par
#pragma unroll
                for (int s = 0; s < EPT; ++s) work[pad(((slot_freq<LOGN>(s, u, par) + N / 2) & (N - 1)) >> 1)] = x[s];
                cta_sync();
                const int pos = (int)sr;
                const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
#pragma unroll
                for (int i = 0; i < EPT; ++i) {
                    const int e = u + FT * i;
                    float2 v = work[pad(e)];
                    const size_t o = (size_t)q * N + 2 * e + par;
                    if (accumulate || k != top_span_lo) {
                        const float2 old = image[o];
                        v.x += old.x; v.y += old.y;
                    }
                    image[o] = v;
                    if (dirty && k == 0) dirty[o] = v.x;
                }
            } else {
#pragma unroll
                for (int s = 0; s < EPT; ++s)
                    work[pad(slot_row<LOGN>(s, u) * N + ((slot_freq<LOGN>(s, u, par) + N / 2) & (N - 1)))] = x[s];
                cta_sync();
#pragma unroll
                for (int i = 0; i < EPT / 2; ++i) {
                    const int e = (u + FT * i) * 2;
                    const float2 a = work[pad(e)], b = work[pad(e) + 1];
                    float4 v = make_float4(a.x, a.y, b.x, b.y);
                    const int pos = (int)sr * ROWS + (e >> LOGN);
                    const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
                    const size_t o = (size_t)q * N + (e & (N - 1));
                    if (accumulate || k != top_span_lo) {
                        const float4 old = *(const float4*)(image + o);
                        v.x += old.x; v.y += old.y; v.z += old.z; v.w += old.w;
                    }
                    *(float4*)(image + o) = v;
                    if (dirty && k == 0) *(float2*)(dirty + o) = make_float2(v.x, v.z);
                }
            }
            cta_sync();            // `work` is free again before the next plane's first stage stores into it
        }
    }
}


// ---- host side ---------------------------------------------------------------------------------------------
template <int LOGN>
size_t rows_smem() {
    return (size_t)RowCfg<LOGN>::NBUF * RowCfg<LOGN>::LAND * sizeof(float2) + (size_t)PAD_PTS * sizeof(float2) +
           (size_t)((tw_smem_entries(LOGN) + 1) & ~1) * sizeof(float2) + 16 * RowCfg<LOGN>::NBUF + MAX_PLANES / 8;
}

float2 unit(long long e, long long L) {      // exp(+2 pi i e / L), fp64 -> fp32
    const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)(e % L) / (double)L;
    return make_float2((float)cos(a), (float)sin(a));
}

// Table = [pass 2: every stage but the last, (R-1) Q entries W_L^(j m') each (N = 16384: stage 1 only) | pass 1a:
// (R0-1) x 256 entries W_N^(j m') | pass 1b: 15 x 16 entries W_256^(j m') | N >= 8192: the first-stage register constants
// of the row kernel, [q][b][ug] = W_N^(ug (M b + q)) (4 x 4 x 256) then [a][ug] = W_N^(4 M a ug), a = 1..3]
template <int LOGN>
int init_n(ws_plan* plan) {
    constexpr int N = 1 << LOGN, R0 = N / 256;
    std::vector<float2> tw;
    for (int s = tw_factored(LOGN) ? 1 : 0; s + 1 < n_stages(LOGN); ++s) {
        const int L = 1 << log2l(LOGN, s), R = 1 << log2r(LOGN, s), Q = L / R;
        for (int m = 1; m < R; ++m)
            for (int j = 0; j < Q; ++j) tw.push_back(unit((long long)j * m, L));
    }
    plan->tw_off_a = tw.size();
    for (int m = 1; m < R0; ++m)
        for (int j = 0; j < 256; ++j) tw.push_back(unit((long long)j * m, N));
    plan->tw_off_b = tw.size();
    for (int m = 1; m < 16; ++m)
        for (int j = 0; j < 16; ++j) tw.push_back(unit((long long)j * m, 256));
    plan->tw_off_c = tw.size();
    if (tw_factored(LOGN)) {
        const int M = LOGN == 14 ? 4 : 2;          // first-stage digits of one thread: d = M p + q, q < M
        for (int q = 0; q < 4; ++q)
            for (int b = 0; b < 4; ++b)
                for (int ug = 0; ug < 256; ++ug) tw.push_back(unit((long long)ug * (M * b + (q % M)), N));
        for (int a = 1; a < 4; ++a)
            for (int ug = 0; ug < 256; ++ug) tw.push_back(unit((long long)ug * 4 * M * a, N));
    }
    const size_t n_class = (size_t)plan->prm.n_wplanes * (N / 32) * 8 * class_words(R0),
                 n_band = (size_t)plan->prm.n_wplanes * band_words(N / 32);
    plan->mask_set_words = n_class + n_band + (size_t)plan->prm.n_wplanes * (N / 32);      // + the band list
    plan->mask_class_words = class_words(R0);
    plan->mask_band_words = band_words(N / 32);
    plan->mask_words = MASK_CTRL + 2 * plan->mask_set_words + 8 + (size_t)plan->prm.n_wplanes * (N / 32);   // + k_fft_cols' queue and signals
    if (cudaMalloc((void**)&plan->d_twiddles, tw.size() * sizeof(float2)) != cudaSuccess ||
        cudaMalloc((void**)&plan->d_masks, plan->mask_words * sizeof(uint32_t)) != cudaSuccess)
        return WS_ERR_CUDA;
    if (cudaMemcpy(plan->d_twiddles, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(plan->d_masks, 0, plan->mask_words * sizeof(uint32_t)) != cudaSuccess)
        return WS_ERR_CUDA;
    if (cudaFuncSetAttribute(k_fft_rows<LOGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rows_smem<LOGN>()) !=
            cudaSuccess ||
        cudaFuncSetAttribute(k_fft_colB<LOGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 256 * 32 * 8) != cudaSuccess)
        return WS_ERR_CUDA;
    if constexpr (cols_fused(LOGN)) {
        if (cudaFuncSetAttribute(k_fft_cols<LOGN, COLS_W>, cudaFuncAttributeMaxDynamicSharedMemorySize, 256 * 4 * COLS_W * 8) != cudaSuccess)
            return WS_ERR_CUDA;
    }
    return WS_OK;
}

template <int LOGN>
int launch_cols_n(ws_plan* plan, float2* grid, bool sparse, cudaStream_t st) {
    constexpr int N = 1 << LOGN, R0 = N / 256, NT = N / 32;
    const float2* tw = (const float2*)plan->d_twiddles;
    const uint32_t* cm = sparse ? (const uint32_t*)plan->d_masks : nullptr;
    const uint32_t sw = (uint32_t)plan->mask_set_words;
    const uint32_t nw = (uint32_t)plan->prm.n_wplanes;
    int launches = 0;
    if constexpr (cols_fused(LOGN)) {
        if (plan->d_masks) {   // both passes from one queue, the intermediate stays in L2 (cm == NULL: every band)
            uint32_t* sync = (uint32_t*)plan->d_masks + MASK_CTRL + 2 * plan->mask_set_words;
            if (cudaMemsetAsync(sync, 0, (size_t)(1 + nw * NT) * sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;
            k_fft_cols<LOGN, COLS_W><<<(uint32_t)plan->sm_count * (16u / COLS_W), 32 * COLS_W, 256 * 4 * COLS_W * 8, st>>>(
                grid, tw + plan->tw_off_a, tw + plan->tw_off_b, cm, sw, nw * NT, sync);
            return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
        }
    }
    if (R0 > 1) return WS_ERR_UNSUPPORTED;          // (N >= 512 always goes through k_fft_cols: the plan owns the masks buffer)
    const uint32_t n_items = nw * NT * (uint32_t)R0;
    const uint32_t ctas = n_items < (uint32_t)plan->sm_count * 2u ? n_items : (uint32_t)plan->sm_count * 2u;
    k_fft_colB<LOGN><<<ctas, CT, 256 * 32 * 8, st>>>(grid, tw + plan->tw_off_b, cm, sw, n_items);
    ++launches;
    return cudaGetLastError() == cudaSuccess ? launches : WS_ERR_CUDA;
}

// part / n_parts: the launch covers that share of the image lines (items are ordered by the line they produce), so
// that a caller can start copying finished lines out while the rest is computed; 0 / 1: everything
template <int LOGN>
int launch_rows_n(ws_plan* plan, const float2* grid, float2* image, float* dirty, int accumulate, bool sparse,
                  int part, int n_parts, cudaStream_t st) {
    constexpr int N = 1 << LOGN;
    const ws_params& P = plan->prm;
    WcParams prm;
    prm.n_pix = P.n_pix;
    prm.n_wplanes = P.n_wplanes;
    prm.cell = P.cell_rad;
    prm.dw = (P.w_max - P.w_min) / (double)P.n_wplanes;
    prm.w0 = P.w_min + 0.5 * prm.dw;
    const uint32_t n_all = (uint32_t)(((size_t)N * N) / RowCfg<LOGN>::LAND) * RowCfg<LOGN>::ITEMS_PER_ROW;
    if (n_parts < 1 || part < 0 || part >= n_parts || n_all % (uint32_t)(2 * n_parts) != 0) return WS_ERR_INVALID_ARG;
    const uint32_t lo = n_all / (uint32_t)n_parts * (uint32_t)part, hi = lo + n_all / (uint32_t)n_parts, n_items = hi - lo;
    uint32_t ctas = n_items < (uint32_t)plan->sm_count ? n_items : (uint32_t)plan->sm_count;
    if (RowCfg<LOGN>::ITEMS_PER_ROW == 2) ctas &= ~1u;      // even grid (and even item_lo): a CTA keeps the parity of its first item
    const uint32_t* bm = sparse ? (const uint32_t*)plan->d_masks : nullptr;
    k_fft_rows<LOGN><<<ctas, FT + PT, rows_smem<LOGN>(), st>>>(prm, grid, image, dirty, accumulate,
                                                          (const float2*)plan->d_twiddles,
                                                          (const float2*)plan->d_twiddles + plan->tw_off_c, bm,
                                                          (uint32_t)plan->mask_set_words, lo, hi);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}

int logn_of(int n_pix) {
    for (int l = 8; l <= 14; ++l)
        if (n_pix == (1 << l)) return l;
    return 0;
}

}  // namespace

#define WS_FFT_DISPATCH(fn, ...)                     \
    switch (logn_of(plan->prm.n_pix)) {              \
        case 8: return fn<8>(__VA_ARGS__);           \
        case 9: return fn<9>(__VA_ARGS__);           \
        case 10: return fn<10>(__VA_ARGS__);         \
        case 11: return fn<11>(__VA_ARGS__);         \
        case 12: return fn<12>(__VA_ARGS__);         \
        case 13: return fn<13>(__VA_ARGS__);         \
        case 14: return fn<14>(__VA_ARGS__);         \
    }                                                \
    return WS_ERR_UNSUPPORTED;

bool ws_fft_own_supported(int n_pix, int n_wplanes) { return logn_of(n_pix) != 0 && n_wplanes <= MAX_PLANES; }

int ws_fft_own_init(ws_plan* plan) { WS_FFT_DISPATCH(init_n, plan) }

int ws_launch_fft_cols(ws_plan* plan, float2* grid, bool sparse, cudaStream_t st) {
    WS_FFT_DISPATCH(launch_cols_n, plan, grid, sparse, st)
}

int ws_launch_fft_rows(ws_plan* plan, const float2* grid, float2* image, float* dirty, int accumulate, bool sparse,
                       int part, int n_parts, cudaStream_t st) {
    WS_FFT_DISPATCH(launch_rows_n, plan, grid, image, dirty, accumulate, sparse, part, n_parts, st)
}

int ws_launch_fft_masks_clear(ws_plan* plan, cudaStream_t st) {
    if (!plan->d_masks) return 0;
    return cudaMemsetAsync(plan->d_masks, 0, plan->mask_words * sizeof(uint32_t), st) == cudaSuccess ? 0 : WS_ERR_CUDA;
}

// OR the occupancy of the bins (rec_start of ws_bin.cu, logical tile coordinates) into the plan's masks (both
// orientations); decide: 1 = choose the orientation of the mesh (WS_GRID_SPARSE), 0 = as the header says, -1 = keep
int ws_launch_fft_masks(ws_plan* plan, const uint32_t* rec_start, int decide, cudaStream_t st) {
    if (!plan->d_masks) return 0;
    const int nt = plan->geom.nt, r0 = plan->prm.n_pix / 256;
    const uint32_t n_classes = (uint32_t)plan->prm.n_wplanes * (uint32_t)nt * 8u;     // (class masks: class_words(r0) words each)
    uint32_t* m = (uint32_t*)plan->d_masks;
    k_fft_masks<<<dim3((n_classes + 255) / 256, 2), 256, 0, st>>>(rec_start, nt, r0, n_classes, (uint32_t)plan->mask_set_words, m);
    int launches = 1;
    if (decide >= 0) {
        k_fft_orient<<<1, 1, 0, st>>>(m, decide && !(plan->prm.flags & WS_FLAG_NO_TRANSPOSE));
        ++launches;
    }
    return cudaGetLastError() == cudaSuccess ? launches : WS_ERR_CUDA;
}

// masks for the column passes of a degridding call (cleared first), for both orientations of the planes, and the choice
int ws_launch_fft_masks_degrid(ws_plan* plan, const uint32_t* bin_start, cudaStream_t st) {
    if (!plan->d_masks) return WS_ERR_UNSUPPORTED;
    if (cudaMemsetAsync(plan->d_masks, 0, plan->mask_words * sizeof(uint32_t), st) != cudaSuccess) return WS_ERR_CUDA;
    const int nt = plan->geom.nt, r0 = plan->prm.n_pix / 256;
    const uint32_t n_kb = (uint32_t)plan->prm.n_wplanes * (uint32_t)nt;
    k_fft_masks_degrid<<<dim3((n_kb + 255) / 256, 2), 256, 0, st>>>(bin_start, nt, r0, n_kb, (uint32_t)plan->mask_set_words,
                                                                   (uint32_t*)plan->d_masks);
    k_fft_orient<<<1, 1, 0, st>>>((uint32_t*)plan->d_masks, !(plan->prm.flags & WS_FLAG_NO_TRANSPOSE));   // fewer bands wins
    return cudaGetLastError() == cudaSuccess ? 2 : WS_ERR_CUDA;
}

WsMaskView ws_fft_mask_view(const ws_plan* plan) {
    return WsMaskView{(const uint32_t*)plan->d_masks, (uint32_t)plan->mask_set_words, plan->d_masks ? plan->mask_class_words : 1};
}

const uint32_t* ws_fft_orientation_flag(const ws_plan* plan) { return plan->d_masks ? (const uint32_t*)plan->d_masks + 2 : nullptr; }
