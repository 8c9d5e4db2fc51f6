// a3 + a4: the per-plane un-normalised inverse 2-D FFT written for this path, with the
// phase correction and the reduction over the w-planes (Eq. 2) fused into its last pass.
//
// The paper leaves the FFT to FFTW on the CPU (55-80 % of its GPU runs) and names a GPU FFT as
// future work (:459).  A library 2-D FFT of an 8192^2 plane reads and writes the mesh three times (rows, and the
// columns in two steps), and a4 reads it a fourth time.  Here, for N = R0 * 256 (N = 2^8 .. 2^13):
//   pass 1a k_fft_colA   columns, first radix-R0 step across the N/R0-spaced rows, in registers: a warp = 32
//                        adjacent columns, so every access is a whole 256-byte row segment; twiddles are
//                        warp-uniform; no shared memory;
//   pass 1b k_fft_colB   columns, the remaining 256-point transforms: a CTA holds a [256 rows x 32 columns] block
//                        (lane = column: conflict-free, coalesced), radix 16 x 16, in place.  Row position
//                        256 m0 + f of the mesh then holds v-frequency m0 + R0 f;
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

constexpr int FT = 256;            // threads per CTA
constexpr int EPT = 32;            // points per thread
constexpr int PTS = FT * EPT;      // points per CTA
constexpr int WC_SPAN = 64;        // planes per Horner chain of the fused w-correction (exact restart between chains)

// ---- stage plan: N = prod R_s ------------------------------------------------------------------------------
__host__ __device__ constexpr int n_stages(int logn) { return logn <= 10 ? 2 : 3; }
__host__ __device__ constexpr int log2r(int logn, int s) {
    switch (logn) {
        case 8: return s < 2 ? 4 : 0;                       // 16 16
        case 9: return s == 0 ? 5 : (s == 1 ? 4 : 0);       // 32 16
        case 10: return s < 2 ? 5 : 0;                      // 32 32
        case 11: return s < 2 ? 4 : (s == 2 ? 3 : 0);       // 16 16 8
        case 12: return s < 3 ? 4 : 0;                      // 16 16 16
        case 13: return s == 0 ? 5 : (s < 3 ? 4 : 0);       // 32 16 16
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
__device__ __forceinline__ float2 eadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 esub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
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

// In-register inverse DFT of R = 2^LOGR points, decimation in frequency: on return x[i] = Y[brev(i)],
// Y[m'] = sum_m x[m] exp(+2 pi i m m' / R).
template <typename E, int LOGR>
__device__ __forceinline__ void bfly(E* x) {
    constexpr int R = 1 << LOGR;
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int blk = 0; blk < R; blk += 2 * half) {
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const E a = x[blk + j], b = x[blk + j + half];
                x[blk + j] = eadd(a, b);
                x[blk + j + half] = mul_w32(esub(a, b), j * (16 / half));
            }
        }
    }
}

// ---- one stage of the CTA-wide transform -------------------------------------------------------------------
// Stage with sub-transform length L = 2^LOGL and radix R = 2^LOGR (Q = L / R): butterfly b of the CTA
// (b = t + 256 i, i < 32 / R) takes the points base + m Q, m < R, base = (b / Q) L + (b mod Q), and leaves
// Y[m'] W_L^(j m') at base + m' Q (j = b mod Q): in place, so consecutive stages need one barrier only.
template <int LOGL, int LOGR>
__device__ __forceinline__ int stage_base(int b) {
    constexpr int LOGQ = LOGL - LOGR;
    return ((b >> LOGQ) << LOGL) + (b & ((1 << LOGQ) - 1));
}

template <typename E, int LOGL, int LOGR, bool PADDED>
__device__ __forceinline__ void stage_load(E* x, const E* __restrict__ src, int t) {
    constexpr int R = 1 << LOGR, LOGQ = LOGL - LOGR;
#pragma unroll
    for (int i = 0; i < EPT / R; ++i) {
        const int base = stage_base<LOGL, LOGR>(t + FT * i);
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const int p = base + (m << LOGQ);
            x[i * R + m] = src[PADDED ? pad(p) : p];
        }
    }
}

template <typename E, int LOGL, int LOGR>
__device__ __forceinline__ void stage_compute(E* x, const float2* __restrict__ tw, int t) {
    constexpr int R = 1 << LOGR, LOGQ = LOGL - LOGR, Q = 1 << LOGQ;
#pragma unroll
    for (int i = 0; i < EPT / R; ++i) {
        bfly<E, LOGR>(x + i * R);
        if (LOGQ > 0) {
            const int j = (t + FT * i) & (Q - 1);
#pragma unroll
            for (int r = 1; r < R; ++r) {
                const float2 w = tw[(brev(r, LOGR) - 1) * Q + j];
                x[i * R + r] = emul(x[i * R + r], w.x, w.y);
            }
        }
    }
}

template <typename E, int LOGL, int LOGR>
__device__ __forceinline__ void stage_store(const E* x, E* __restrict__ dst, int t) {
    constexpr int R = 1 << LOGR, LOGQ = LOGL - LOGR;
#pragma unroll
    for (int i = 0; i < EPT / R; ++i) {
        const int base = stage_base<LOGL, LOGR>(t + FT * i);
#pragma unroll
        for (int r = 0; r < R; ++r) dst[pad(base + (brev(r, LOGR) << LOGQ))] = x[i * R + r];
    }
}

// Stages 1 .. S-1 on the padded work buffer; the first stage's results must already be in `work` (not yet
// synchronised).  On return x[] holds the transform: register i*R + r of thread t is position
// ((t + 256 i) R + brev(r)) of the CTA, R the radix of the last stage.
template <typename E, int LOGN>
__device__ __forceinline__ void later_stages(E* x, E* work, const float2* tw, int t) {
    constexpr int S = n_stages(LOGN);
    __syncthreads();
    if (S == 3) {
        constexpr int L1 = log2l(LOGN, 1), R1 = log2r(LOGN, 1);
        stage_load<E, L1, R1, true>(x, work, t);
        stage_compute<E, L1, R1>(x, tw + tw_offset(LOGN, 1), t);
        stage_store<E, L1, R1>(x, work, t);
        __syncthreads();
    }
    constexpr int LL = log2l(LOGN, S - 1), RL = log2r(LOGN, S - 1);
    static_assert(LL == RL, "last stage must have Q = 1");
    stage_load<E, LL, RL, true>(x, work, t);
    stage_compute<E, LL, RL>(x, tw, t);
}

// CTA position of register slot `slot` after later_stages()
template <int LOGN>
__device__ __forceinline__ int final_pos(int slot, int t) {
    constexpr int RL = log2r(LOGN, n_stages(LOGN) - 1), R = 1 << RL;
    return ((t + FT * (slot / R)) << RL) + brev(slot % R, RL);
}

__device__ __forceinline__ void load_twiddles(float2* tw_s, const float2* __restrict__ tw_g, int n, int t) {
    for (int i = t; i < n; i += FT) tw_s[i] = tw_g[i];
}


// ---- occupancy masks -----------------------------------------------------------------------------------------
// Storage (FFT-native) tile coordinates.  class_mask[(k nt + tx) 8 + c]: bit m set <=> tile (ty = c + 8 m, tx) of
// plane k holds visibilities (the R0 inputs of pass 1a's butterflies on the rows of class c = (row mod 256) / 32).
// band_mask[k 8 + tx / 32]: bit tx % 32 set <=> some tile of column band tx of plane k does.
// Masks are OR-ed into (chunked gridding accumulates); ws_fft_masks_clear zeroes them.
__global__ void __launch_bounds__(256)
k_fft_masks(const uint32_t* __restrict__ rec_start, int nt, int r0, uint32_t n_classes, uint32_t* __restrict__ class_mask,
            uint32_t* __restrict__ band_mask) {
    const uint32_t id = blockIdx.x * 256u + threadIdx.x;      // (k nt + txs) 8 + c
    if (id >= n_classes) return;
    const int c = id & 7;
    const uint32_t ktx = id >> 3;
    const int txs = ktx % nt, k = ktx / nt;
    const int tx = (txs + nt / 2) & (nt - 1);
    uint32_t mask = 0;
    for (int m = 0; m < r0; ++m) {
        const int ty = (c + 8 * m + nt / 2) & (nt - 1);
        const uint32_t bin = ((uint32_t)k * nt + ty) * nt + tx;
        if (rec_start[bin + 1] > rec_start[bin]) mask |= 1u << m;
    }
    if (mask) {
        atomicOr(class_mask + id, mask);
        atomicOr(band_mask + k * 8 + (txs >> 5), 1u << (txs & 31));
    }
}

// ---- pass 1a: first radix-R0 step of the column transforms ------------------------------------------------------
// Thread = (column, row j of the first 256-row block): x[m] = row j + 256 m, m < R0; Y[m'] W_N^(j m') goes back to
// row j + 256 m'.  A warp = 32 adjacent columns at one j, a CTA = 8 consecutive j.
template <int LOGN>
__global__ void __launch_bounds__(FT)
k_fft_colA(float2* __restrict__ grid, const float2* __restrict__ tw, const uint32_t* __restrict__ class_mask,
           uint32_t n_items) {
    constexpr int N = 1 << LOGN, LR0 = LOGN - 8, R0 = 1 << LR0, NT = N / 32;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const uint32_t jb = item & 31, ktx = item >> 5;            // 32 groups of 8 rows per (plane, band)
        const uint32_t tx = ktx % NT, k = ktx / NT;
        const uint32_t mask = class_mask ? class_mask[ktx * 8 + (jb >> 2)] : 0xFFFFFFFFu;
        if (mask == 0) continue;
        const int j = (int)jb * 8 + w;
        float2* p = grid + ((size_t)k * N + j) * N + tx * 32 + lane;
        float2 x[R0];
#pragma unroll
        for (int m = 0; m < R0; ++m)
            x[m] = (mask >> m) & 1 ? __ldcs(p + (size_t)m * 256 * N) : make_float2(0.f, 0.f);
        bfly<float2, LR0>(x);
#pragma unroll
        for (int r = 1; r < R0; ++r) {
            const float2 tv = __ldg(tw + (brev(r, LR0) - 1) * 256 + j);
            x[r] = emul(x[r], tv.x, tv.y);
        }
#pragma unroll
        for (int r = 0; r < R0; ++r) p[(size_t)brev(r, LR0) * 256 * N] = x[r];
    }
}

// ---- pass 1b: the 256-point column transforms -------------------------------------------------------------------
// Item = (plane, column band tx, block m0 of 256 rows).  Warp w, lane = column.  Stage 1: j in {w, w + 8}, rows
// j + 16 m; stage 2: blocks b in {w, w + 8}, rows 16 b + m; frequency f = b + 16 m' is stored at row 256 m0 + f.
template <int LOGN>
__global__ void __launch_bounds__(FT, 2)
k_fft_colB(float2* __restrict__ grid, const float2* __restrict__ tw, const uint32_t* __restrict__ class_mask,
           uint32_t n_items) {
    constexpr int N = 1 << LOGN, R0 = 1 << (LOGN - 8), NT = N / 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2* blk = (float2*)smem_raw;          // [256 rows][32 columns]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const uint32_t m0 = item % R0, ktx = item / R0;
        const uint32_t tx = ktx % NT, k = ktx / NT;
        uint32_t cmask = 0xFFu;
        if (class_mask) {
            cmask = 0;
#pragma unroll
            for (int c = 0; c < 8; ++c) cmask |= (class_mask[ktx * 8 + c] != 0 ? 1u : 0u) << c;
        }
        if (cmask == 0) continue;
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
            bfly<float2, 4>(x + i * 16);
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
            bfly<float2, 4>(x + i * 16);
#pragma unroll
            for (int r = 0; r < 16; ++r) p[(size_t)(b + 16 * brev(r, 4)) * N] = x[i * 16 + r];
        }
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
// band_mask (or NULL = dense): only the non-empty 32-column bands of a plane are copied in, as maximal runs; a
// band that is empty now but was filled by the previous copy is cleared by the CTA; a plane without any is skipped.
struct BandMask {
    uint32_t w[8];
};
__device__ __forceinline__ BandMask load_bands(const uint32_t* __restrict__ band_mask, int k, int nt) {
    BandMask b;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int lo = 32 * i;
        const uint32_t full = nt >= lo + 32 ? 0xFFFFFFFFu : (nt > lo ? (1u << (nt - lo)) - 1u : 0u);
        b.w[i] = band_mask ? (__ldg(band_mask + k * 8 + i) & full) : full;
    }
    return b;
}
__device__ __forceinline__ bool any_band(const BandMask& b) {
    uint32_t o = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) o |= b.w[i];
    return o != 0;
}

template <int LOGN>
__global__ void __launch_bounds__(FT, 1)
k_fft_rows(const __grid_constant__ WcParams prm, const float2* __restrict__ planes, float2* __restrict__ image,
           float* __restrict__ dirty, int accumulate, const float2* __restrict__ tw_g,
           const uint32_t* __restrict__ band_mask, uint32_t n_super) {
    constexpr int N = 1 << LOGN, ROWS = PTS / N, NT = N / 32, R0 = 1 << (LOGN - 8);
    constexpr int L0 = LOGN, LR0 = log2r(LOGN, 0);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2* landing = (float2*)smem_raw;
    float2* work = landing + PTS;
    float2* tw = work + PAD_PTS;
    uint64_t* bar = (uint64_t*)(tw + ((tw_entries(LOGN) + 1) & ~1));
    const int t = threadIdx.x;
    const int nw = prm.n_wplanes;
    const size_t plane_elems = (size_t)N * N;
    load_twiddles(tw, tw_g, tw_entries(LOGN), t);
#pragma unroll
    for (int i = 0; i < EPT; ++i) landing[t + FT * i] = make_float2(0.f, 0.f);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (t == 0) mbar_init(bar, 1);
    __syncthreads();
    if (blockIdx.x >= n_super) return;

    // Lane 0 of warp w brings the non-empty bands of word w (32 bands, 8 KB per row) of super-row sr of plane k into
    // `landing`, one bulk copy per maximal run; thread 0 posts the byte count (the copies of the other warps may
    // complete before it does: the phase cannot, it needs this arrival).
    auto issue = [&](uint32_t sr, int k, const BandMask& bm) {
        if (t & 31) return;
        if (t == 0) {
            uint32_t n_bands = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) n_bands += __popc(bm.w[i]);
            mbar_expect_tx(bar, n_bands * 256u * ROWS);
        }
        const char* src = (const char*)(planes + (size_t)k * plane_elems + (size_t)sr * PTS);
        uint32_t m = 0;
#pragma unroll
        for (int wi = 0; wi < 8; ++wi) m = (t >> 5) == wi ? bm.w[wi] : m;
        while (m) {
            const int b0 = __ffs(m) - 1;
            const uint32_t inv = ~(m >> b0);
            const int len = inv ? __ffs(inv) - 1 : 32;
            m &= ~((len == 32 ? 0xFFFFFFFFu : (1u << len) - 1u) << b0);
            const size_t off = (size_t)((t >> 5) * 32 + b0) * 256;
            for (int r = 0; r < ROWS; ++r)
                bulk_g2s((char*)landing + (size_t)r * N * 8 + off, src + (size_t)r * N * 8 + off, len * 256, bar);
        }
    };
    // first plane (from the top) of this CTA's super-row that has data; -1 if none
    auto next_plane = [&](int k, BandMask& bm) {
        for (; k >= 0; --k) {
            bm = load_bands(band_mask, k, NT);
            if (any_band(bm)) return k;
        }
        return -1;
    };

    BandMask cur, nxt;                 // invariant: the non-zero bands of `landing` are a subset of `cur`
    int k_cur = next_plane(nw - 1, cur);
    uint32_t sr_cur = blockIdx.x;
    if (k_cur >= 0) issue(blockIdx.x, k_cur, cur);
    uint32_t parity = 0;
    const int top_span_lo = ((nw - 1) / WC_SPAN) * WC_SPAN;

    for (uint32_t sr = blockIdx.x; sr < n_super; sr += gridDim.x) {
        float2 rot[EPT], h[EPT];
#pragma unroll
        for (int s = 0; s < EPT; ++s) {
            const int P = final_pos<LOGN>(s, t);
            const int pos = (int)sr * ROWS + (P >> LOGN);
            const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
            const int p = (freq_of<LOGN>(P & (N - 1)) + N / 2) & (N - 1);
            bool inside;
            const double tt = ws_n_minus_1(prm, q, p, &inside);
            rot[s] = ws_expi_turns(prm.dw * tt);
            h[s] = make_float2(0.f, 0.f);
        }
        for (int k = nw - 1; k >= 0; --k) {
            float2 x[EPT];
            if (k == k_cur && sr == sr_cur) { // CTA-uniform: this plane has data and its copy is in flight
                while (!mbar_try_wait(bar, parity)) {}
                parity ^= 1u;
                stage_load<float2, L0, LR0, false>(x, landing, t);
                __syncthreads();       // landing consumed (and the previous plane's last stage has read `work`)
                // next copy: the next non-empty plane of this super-row, else the first one of the next super-row
                int k_nxt = next_plane(k - 1, nxt);
                uint32_t sr_nxt = sr;
                if (k_nxt < 0 && sr + gridDim.x < n_super) {
                    sr_nxt = sr + gridDim.x;
                    k_nxt = next_plane(nw - 1, nxt);
                }
                if (k_nxt >= 0) {
                    uint32_t stale = 0;                    // bands the last copy filled and the next one will not
#pragma unroll
                    for (int i = 0; i < 8; ++i) stale |= cur.w[i] & ~nxt.w[i];
                    if (stale) {
#pragma unroll
                        for (int i = 0; i < EPT; ++i) {
                            const int wi = ((8 * i) & (NT - 1)) >> 5;      // band of point t + 256 i: (t >> 5) + 8 i
                            const int bit = ((t >> 5) + 8 * i) & 31;
                            if (((cur.w[wi] & ~nxt.w[wi]) >> bit) & 1u) landing[t + FT * i] = make_float2(0.f, 0.f);
                        }
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    }
                    issue(sr_nxt, k_nxt, nxt);
                }
                cur = nxt;
                k_cur = k_nxt;
                sr_cur = sr_nxt;
                stage_compute<float2, L0, LR0>(x, tw, t);
                stage_store<float2, L0, LR0>(x, work, t);
                later_stages<float2, LOGN>(x, work, tw, t);
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
                const int P = final_pos<LOGN>(s, t);
                const int pos = (int)sr * ROWS + (P >> LOGN);
                const int q = ((pos >> 8) + R0 * (pos & 255) + N / 2) & (N - 1);
                const int p = (freq_of<LOGN>(P & (N - 1)) + N / 2) & (N - 1);
                bool inside;
                const double tt = ws_n_minus_1(prm, q, p, &inside);
                x[s] = ws_cmul(h[s], ws_expi_turns((prm.w0 + (double)k * prm.dw) * tt));
                if (!inside) x[s] = make_float2(0.f, 0.f);
                h[s] = make_float2(0.f, 0.f);
            }
            // un-permute through `work`: natural order along the rows of the centred image
            __syncthreads();
#pragma unroll
            for (int s = 0; s < EPT; ++s) {
                const int P = final_pos<LOGN>(s, t);
                work[pad((P & ~(N - 1)) + ((freq_of<LOGN>(P & (N - 1)) + N / 2) & (N - 1)))] = x[s];
            }
            __syncthreads();
#pragma unroll
            for (int i = 0; i < EPT / 2; ++i) {
                const int e = (t + FT * i) * 2;
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
            __syncthreads();       // `work` is free again before the next plane's first stage stores into it
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int LOGN>
size_t rows_smem() {
    return (size_t)PTS * sizeof(float2) + (size_t)PAD_PTS * sizeof(float2) +
           (size_t)((tw_entries(LOGN) + 1) & ~1) * sizeof(float2) + 16;
}

float2 unit(long long e, long long L) {      // exp(+2 pi i e / L), fp64 -> fp32
    const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)(e % L) / (double)L;
    return make_float2((float)cos(a), (float)sin(a));
}

// Table = [pass 2: every stage but the last, (R-1) Q entries W_L^(j m') each | pass 1a: (R0-1) x 256 entries
// W_N^(j m') | pass 1b: 15 x 16 entries W_256^(j m')]
template <int LOGN>
int init_n(ws_plan* plan) {
    constexpr int N = 1 << LOGN, R0 = N / 256;
    std::vector<float2> tw;
    for (int s = 0; s + 1 < n_stages(LOGN); ++s) {
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
    const size_t n_class = (size_t)plan->prm.n_wplanes * (N / 32) * 8, n_band = (size_t)plan->prm.n_wplanes * 8;
    plan->mask_words = n_class + n_band;
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
    return WS_OK;
}

template <int LOGN>
int launch_cols_n(ws_plan* plan, float2* grid, bool sparse, cudaStream_t st) {
    constexpr int N = 1 << LOGN, R0 = N / 256, NT = N / 32;
    const float2* tw = (const float2*)plan->d_twiddles;
    const uint32_t* cm = sparse ? (const uint32_t*)plan->d_masks : nullptr;
    const uint32_t nw = (uint32_t)plan->prm.n_wplanes;
    int launches = 0;
    if (R0 > 1) {
        const uint32_t n_items = nw * NT * 32u;
        const uint32_t ctas = n_items < (uint32_t)plan->sm_count * 8u ? n_items : (uint32_t)plan->sm_count * 8u;
        k_fft_colA<LOGN><<<ctas, FT, 0, st>>>(grid, tw + plan->tw_off_a, cm, n_items);
        ++launches;
    }
    const uint32_t n_items = nw * NT * (uint32_t)R0;
    const uint32_t ctas = n_items < (uint32_t)plan->sm_count * 2u ? n_items : (uint32_t)plan->sm_count * 2u;
    k_fft_colB<LOGN><<<ctas, FT, 256 * 32 * 8, st>>>(grid, tw + plan->tw_off_b, cm, n_items);
    ++launches;
    return cudaGetLastError() == cudaSuccess ? launches : WS_ERR_CUDA;
}

template <int LOGN>
int launch_rows_n(ws_plan* plan, const float2* grid, float2* image, float* dirty, int accumulate, bool sparse,
                  cudaStream_t st) {
    constexpr int N = 1 << LOGN;
    const ws_params& P = plan->prm;
    WcParams prm;
    prm.n_pix = P.n_pix;
    prm.n_wplanes = P.n_wplanes;
    prm.cell = P.cell_rad;
    prm.dw = (P.w_max - P.w_min) / (double)P.n_wplanes;
    prm.w0 = P.w_min + 0.5 * prm.dw;
    const uint32_t n_super = (uint32_t)(((size_t)N * N) / PTS);
    const uint32_t ctas = n_super < (uint32_t)plan->sm_count ? n_super : (uint32_t)plan->sm_count;
    const uint32_t* bm = sparse ? (const uint32_t*)plan->d_masks + (size_t)P.n_wplanes * (N / 32) * 8 : nullptr;
    k_fft_rows<LOGN><<<ctas, FT, rows_smem<LOGN>(), st>>>(prm, grid, image, dirty, accumulate,
                                                          (const float2*)plan->d_twiddles, bm, n_super);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}

int logn_of(int n_pix) {
    for (int l = 8; l <= 13; ++l)
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
    }                                                \
    return WS_ERR_UNSUPPORTED;

bool ws_fft_own_supported(int n_pix) { return logn_of(n_pix) != 0; }

int ws_fft_own_init(ws_plan* plan) { WS_FFT_DISPATCH(init_n, plan) }

int ws_launch_fft_cols(ws_plan* plan, float2* grid, bool sparse, cudaStream_t st) {
    WS_FFT_DISPATCH(launch_cols_n, plan, grid, sparse, st)
}

int ws_launch_fft_rows(ws_plan* plan, const float2* grid, float2* image, float* dirty, int accumulate, bool sparse,
                       cudaStream_t st) {
    WS_FFT_DISPATCH(launch_rows_n, plan, grid, image, dirty, accumulate, sparse, st)
}

int ws_launch_fft_masks_clear(ws_plan* plan, cudaStream_t st) {
    if (!plan->d_masks) return 0;
    return cudaMemsetAsync(plan->d_masks, 0, plan->mask_words * sizeof(uint32_t), st) == cudaSuccess ? 0 : WS_ERR_CUDA;
}

// OR the occupancy of the bins (rec_start of ws_bin.cu, logical tile coordinates) into the plan's masks
int ws_launch_fft_masks(ws_plan* plan, const uint32_t* rec_start, cudaStream_t st) {
    if (!plan->d_masks) return 0;
    const int nt = plan->geom.nt, r0 = plan->prm.n_pix / 256;
    const uint32_t n_classes = (uint32_t)plan->prm.n_wplanes * (uint32_t)nt * 8u;
    uint32_t* cm = (uint32_t*)plan->d_masks;
    k_fft_masks<<<(n_classes + 255) / 256, 256, 0, st>>>(rec_start, nt, r0, n_classes, cm, cm + n_classes);
    return cudaGetLastError() == cudaSuccess ? 1 : WS_ERR_CUDA;
}
