/*
 * wstack_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU statement of what the w-stacking hot path computes, written from
 * /root/reference/PAPER.md (arxiv 2301.06061) and the readings listed in DESIGN.md section 3.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * build, load or call it.  It shares no code, header, table or constant generator with the CUDA
 * library under paper_2301_06061_b200/csrc/ and never includes anything from there.
 *
 * The method is an approximation scheme (convolutional gridding + nearest-w-plane), so the oracle
 * is the algorithm itself, step by step, in the paper's order:
 *
 *   orc_positions      PAPER.md:66  "visibilities are mapped to the closest w-plane"
 *                      (a visibility is convolved onto the mesh around its (u,v)).  Position rule,
 *                      drop rule and bin key = DESIGN.md readings R4-R6 (the paper is silent).
 *   orc_bins           PAPER.md:78, :144-150: the per-region lists of visibilities ("bucketing"),
 *                      here as a stable counting sort by (w-plane, uv-tile) key.
 *   orc_grid           PAPER.md:80 Eq. 3,  V~(u_i,v_j,w_k) = sum_m V_m G(...), Gaussian G with a
 *                      7-cell support (:82), weights per measurement (:74) -- no binning, no tiling.
 *   orc_dft2_naive     PAPER.md:84, :152 "each w plane is Fourier transformed separately": the 2-D
 *                      inverse DFT written out as two 1-D sums (O(N^3) per plane).
 *   orc_fft2           the same transform by a textbook radix-2 FFT (the paper uses FFTW, :84);
 *                      pinned against orc_dft2_naive and numpy in tests/test_oracle_pins.py.
 *   orc_wcorrect       PAPER.md:68 Eq. 2 / :86 "phase shift and reduction of the w-planes":
 *                      D(l,m) = sum_k exp(2 pi i w_k (sqrt(1-l^2-m^2)-1)) P_k(l,m).
 *   orc_kernel1d       the 1-D convolution function: the paper's Gaussian or the Kaiser-Bessel
 *                      window the paper names as the production kernel and as its next step (:82, :459),
 *                      I0 by its power series; unit integral (reading R2 / R28).
 *   orc_taper1d        the continuous Fourier transform of that function (closed forms), i.e. the image-plane
 *                      response the convolution leaves behind ("aliasing response in image space", :82).
 *   orc_sum_weights    sum of the weights of the kept visibilities (the normalisation of the direct sum).
 *   orc_dirty          PAPER.md:68 Eq. 2 solved for I: the factor n = sqrt(1-l^2-m^2) of its left side, the
 *                      division by the taper and by the sum of weights (readings R12 / R29).
 *   orc_wscreen_fwd    degridding, step 1 ("the degridding procedure (transforming from the image to
 *                      the visibility space)"; Eq. 1 at :59): model image times exp(-2 pi i w_k (n-1)).
 *   orc_degrid         degridding, step 3: every visibility reads its S x S footprint of the forward-transformed
 *                      plane k through the same convolution function (the transpose of Eq. 3, :80).
 *                      Step 2, the forward DFT, is conj(orc_dft2(conj(.))) in oracle/wstack_oracle.py.
 *   orc_image_samples  the composition orc_grid -> DFT -> orc_wcorrect evaluated at single pixels
 *                      with the order of the (finite, linear) sums exchanged: visibility outermost.
 *                      Used where a full fp64 plane stack would not fit; pinned against the chain.
 *
 * Layout everywhere: logical, centred.  Mesh cell (j,i) <-> (v,u) = ((j-N/2) du, (i-N/2) du);
 * image pixel (q,p) <-> (m,l) = ((q-N/2) cell, (p-N/2) cell); u / l fastest.
 *
 * Every oracle function is pinned by tests/test_oracle_pins.py; none is
 * "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build_oracle.py).
 * -ffp-contract=off matters: the position rule is a fixed sequence of correctly rounded binary64
 * operations (explicit fma()), and the bin keys derived from it are compared bit for bit.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_C_LIGHT 299792458.0
#define ORC_PI 3.14159265358979323846264338327950288

typedef struct {
    int32_t n_pix;      /* N: mesh / image side (even)                         */
    int32_t n_wplanes;  /* N_w                                                 */
    int32_t support;    /* S: odd kernel size in cells (paper: 7) */
    int32_t tile;       /* T: uv-tile side used by the bin key                 */
    double sigma;       /* Gaussian sigma in cells (reading R1)                */
    double cell_rad;    /* image pixel size, radians                           */
    double w_min;       /* w range covered by the planes, wavelengths (R6)     */
    double w_max;
    int32_t kernel_type; /* 0: Gaussian, `sigma` = sigma in cells; 1: Kaiser-Bessel, `sigma` = beta (R28) */
    int32_t pad_;
} orc_params;

/* ---- O1: per-channel scalar constants (O1) ------------------------- */
/* su: cells per stored-uvw unit; sw: planes per stored-uvw unit; ow: plane offset.          */
void orc_channel_constants(const orc_params *p, const double *freq_hz, int32_t n_chan,
                           double *su, double *sw, double *ow) {
    double dw = (p->w_max - p->w_min) / (double)p->n_wplanes;
    for (int c = 0; c < n_chan; ++c) {
        if (freq_hz) {
            su[c] = (freq_hz[c] / ORC_C_LIGHT) * ((double)p->n_pix * p->cell_rad);
            sw[c] = (freq_hz[c] / ORC_C_LIGHT) / dw;
        } else {
            su[c] = (double)p->n_pix * p->cell_rad;
            sw[c] = 1.0 / dw;
        }
    }
    *ow = -p->w_min / dw;
}

/* ---- O2-O4: position, plane, drop rule, key of ONE visibility --------------------------- */
/* Returns 1 if kept.  Each arithmetic line is one correctly rounded binary64 operation.     */
static int orc_place(const orc_params *p, double u, double v, double w, double su, double sw, double ow,
                     int32_t *i0, int32_t *j0, int32_t *k, double *fu, double *fv) {
    const double half = (double)(p->n_pix / 2);
    const int h = (p->support - 1) / 2;
    double pu = fma(u, su, half);
    double pv = fma(v, su, half);
    double pw = fma(w, sw, ow);
    double ci = floor(pu + 0.5);          /* nearest cell centre, ties up (R4) */
    double cj = floor(pv + 0.5);
    double ck = floor(pw);                /* N_w equal bins over [w_min, w_max] (R6) */
    if (ck < 0.0) ck = 0.0;
    if (ck > (double)(p->n_wplanes - 1)) ck = (double)(p->n_wplanes - 1);
    *k = pw == pw ? (int32_t)ck : 0;
    /* drop rule O3 (R5): the whole S x S footprint must lie on the mesh; a NaN coordinate drops too (R33) */
    if (!(ci >= (double)h && ci <= (double)(p->n_pix - 1 - h) &&
          cj >= (double)h && cj <= (double)(p->n_pix - 1 - h) && pw == pw)) {
        *i0 = *j0 = -1; *fu = *fv = 0.0;
        return 0;
    }
    *i0 = (int32_t)ci; *j0 = (int32_t)cj;
    *fu = pu - ci;                         /* exact in binary64, in [-1/2, 1/2) */
    *fv = pv - cj;
    return 1;
}

static inline uint32_t orc_key_of(const orc_params *p, int32_t i0, int32_t j0, int32_t k) {
    uint32_t nt = (uint32_t)(p->n_pix / p->tile);
    return ((uint32_t)k * nt + (uint32_t)(j0 / p->tile)) * nt + (uint32_t)(i0 / p->tile);
}

/* Per-visibility outputs, flat index = row * n_chan + c.  Any output pointer may be NULL.   */
void orc_positions(const orc_params *p, const float *uvw, int64_t n_rows, int32_t n_chan,
                   const double *freq_hz, int32_t *i0, int32_t *j0, int32_t *k,
                   double *fu, double *fv, uint32_t *key) {
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
    for (int64_t r = 0; r < n_rows; ++r) {
        double u = (double)uvw[3 * r], v = (double)uvw[3 * r + 1], w = (double)uvw[3 * r + 2];
        for (int c = 0; c < n_chan; ++c) {
            int32_t a, b, kk; double x, y;
            int kept = orc_place(p, u, v, w, su[c], sw[c], ow, &a, &b, &kk, &x, &y);
            int64_t m = r * n_chan + c;
            if (i0) i0[m] = a;
            if (j0) j0[m] = b;
            if (k) k[m] = kk;
            if (fu) fu[m] = x;
            if (fv) fv[m] = y;
            if (key) key[m] = kept ? orc_key_of(p, a, b, kk) : 0xFFFFFFFFu;
        }
    }
    free(su); free(sw);
}

/* ---- O4: stable counting sort of the keys ------------------------------------------------ */
/* bin_start[b] = number of kept visibilities with key < b (b = 0..n_bins); perm lists the     */
/* kept flat indices by ascending key, ties by ascending index.  Returns n_dropped.            */
int64_t orc_bins(const uint32_t *key, int64_t n_vis, int64_t n_bins, uint32_t *bin_start, uint32_t *perm) {
    int64_t dropped = 0;
    memset(bin_start, 0, sizeof(uint32_t) * (size_t)(n_bins + 1));
    for (int64_t m = 0; m < n_vis; ++m) {
        if (key[m] == 0xFFFFFFFFu) ++dropped; else ++bin_start[key[m] + 1];
    }
    for (int64_t b = 0; b < n_bins; ++b) bin_start[b + 1] += bin_start[b];
    if (perm) {
        uint32_t *cur = malloc(sizeof(uint32_t) * (size_t)n_bins);
        memcpy(cur, bin_start, sizeof(uint32_t) * (size_t)n_bins);
        for (int64_t m = 0; m < n_vis; ++m)
            if (key[m] != 0xFFFFFFFFu) perm[cur[key[m]]++] = (uint32_t)m;
        free(cur);
    }
    return dropped;
}

/* ---- O5: 1-D convolution function, unit integral (readings R1, R2, R28) ------------------- */
/* Modified Bessel function of the first kind, order 0, by its defining power series            */
/* I0(x) = sum_k (x^2/4)^k / (k!)^2 (all terms positive: no cancellation).                       */
double orc_i0(double x) {
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    return sum;
}

/* Gaussian: g(x) = exp(-x^2 / (2 sigma^2)) / (sigma sqrt(2 pi)).                  */
/* Kaiser-Bessel (Jackson et al. 1991), width S cells, shape beta:             */
/*   g(x) = I0(beta sqrt(1 - (2x/S)^2)) * beta / (S sinh(beta))   for |x| <= S/2, else 0,         */
/* whose integral over [-S/2, S/2] is 1 because int_{-1}^{1} I0(beta sqrt(1-t^2)) dt = 2 sinh(beta)/beta. */
double orc_kernel1d(const orc_params *p, double x) {
    if (p->kernel_type == 1) {
        const double S = (double)p->support, beta = p->sigma;
        double y = 1.0 - (2.0 * x / S) * (2.0 * x / S);
        if (y < 0.0) return 0.0;
        return orc_i0(beta * sqrt(y)) * beta / (S * sinh(beta));
    }
    return exp(-(x * x) / (2.0 * p->sigma * p->sigma)) / (p->sigma * sqrt(2.0 * ORC_PI));
}

/* Continuous Fourier transform ghat(xi) = int g(x) e^{2 pi i x xi} dx, xi in cycles per cell.    */
/* Gaussian (untruncated): exp(-2 pi^2 sigma^2 xi^2).  Kaiser-Bessel: with a = pi S xi,            */
/* (beta / sinh beta) sinh(sqrt(beta^2 - a^2)) / sqrt(beta^2 - a^2), continued as sin(.)/. for a > beta. */
double orc_taper1d(const orc_params *p, double xi) {
    if (p->kernel_type == 1) {
        const double beta = p->sigma, a = ORC_PI * (double)p->support * xi;
        const double d = beta * beta - a * a;
        double f;
        if (d > 1e-12) { double r = sqrt(d); f = sinh(r) / r; }
        else if (d < -1e-12) { double r = sqrt(-d); f = sin(r) / r; }
        else f = 1.0;
        return f * beta / sinh(beta);
    }
    return exp(-2.0 * ORC_PI * ORC_PI * p->sigma * p->sigma * xi * xi);
}

/* ---- O6: gridding, Eq. 3 ------------------------------------------------------------------ */
/* Adds every kept visibility whose plane k lies in [plane_lo, plane_hi) onto                  */
/* G[(k - plane_lo)][j][i] (interleaved re,im doubles).  Visibilities are visited in input     */
/* order; with OpenMP each thread owns whole planes, which leaves that order unchanged.        */
void orc_grid(const orc_params *p, const float *uvw, const float *vis /* re,im */, const float *wt,
              const double *freq_hz, int64_t n_rows, int32_t n_chan,
              int32_t plane_lo, int32_t plane_hi, double *G) {
    const int N = p->n_pix, S = p->support, h = (S - 1) / 2;
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
#pragma omp parallel for schedule(static, 1)
    for (int kp = plane_lo; kp < plane_hi; ++kp) {
        double *Gk = G + (size_t)(kp - plane_lo) * (size_t)N * (size_t)N * 2;
        double gu[32], gv[32];
        for (int64_t r = 0; r < n_rows; ++r) {
            double u = (double)uvw[3 * r], v = (double)uvw[3 * r + 1], w = (double)uvw[3 * r + 2];
            for (int c = 0; c < n_chan; ++c) {
                int32_t i0, j0, k; double fu, fv;
                if (!orc_place(p, u, v, w, su[c], sw[c], ow, &i0, &j0, &k, &fu, &fv) || k != kp) continue;
                int64_t m = r * n_chan + c;
                double vr = (double)wt[m] * (double)vis[2 * m], vi = (double)wt[m] * (double)vis[2 * m + 1];
                for (int a = -h; a <= h; ++a) {
                    gu[a + h] = orc_kernel1d(p, (double)a - fu);
                    gv[a + h] = orc_kernel1d(p, (double)a - fv);
                }
                for (int b = -h; b <= h; ++b)
                    for (int a = -h; a <= h; ++a) {
                        double t = gu[a + h] * gv[b + h];
                        size_t cell = ((size_t)(j0 + b) * (size_t)N + (size_t)(i0 + a)) * 2;
                        Gk[cell] += vr * t;
                        Gk[cell + 1] += vi * t;
                    }
            }
        }
    }
    free(su); free(sw);
}

/* ---- O7: per-plane un-normalised inverse 2-D DFT, centred indices ------------------------- */
/* P[q][p] = sum_j sum_i G[j][i] exp(+2 pi i ((i-N/2)(p-N/2) + (j-N/2)(q-N/2)) / N)            */
void orc_dft2_naive(int32_t N, const double *G, double *P) {
    double *E = malloc(sizeof(double) * 2 * (size_t)N);       /* E[m] = exp(2 pi i m / N) */
    double *A = malloc(sizeof(double) * 2 * (size_t)N * (size_t)N);
    for (int m = 0; m < N; ++m) {
        E[2 * m] = cos(2.0 * ORC_PI * (double)m / (double)N);
        E[2 * m + 1] = sin(2.0 * ORC_PI * (double)m / (double)N);
    }
    const int64_t H = N / 2;
#pragma omp parallel for
    for (int j = 0; j < N; ++j)           /* A[j][p] = sum_i G[j][i] e(i,p) */
        for (int pp = 0; pp < N; ++pp) {
            double sr = 0.0, si = 0.0;
            for (int i = 0; i < N; ++i) {
                int64_t m = (((int64_t)i - H) * ((int64_t)pp - H)) % N; if (m < 0) m += N;
                double gr = G[2 * ((size_t)j * N + i)], gi = G[2 * ((size_t)j * N + i) + 1];
                sr += gr * E[2 * m] - gi * E[2 * m + 1];
                si += gr * E[2 * m + 1] + gi * E[2 * m];
            }
            A[2 * ((size_t)j * N + pp)] = sr; A[2 * ((size_t)j * N + pp) + 1] = si;
        }
#pragma omp parallel for
    for (int q = 0; q < N; ++q)           /* P[q][p] = sum_j A[j][p] e(j,q) */
        for (int pp = 0; pp < N; ++pp) {
            double sr = 0.0, si = 0.0;
            for (int j = 0; j < N; ++j) {
                int64_t m = (((int64_t)j - H) * ((int64_t)q - H)) % N; if (m < 0) m += N;
                double ar = A[2 * ((size_t)j * N + pp)], ai = A[2 * ((size_t)j * N + pp) + 1];
                sr += ar * E[2 * m] - ai * E[2 * m + 1];
                si += ar * E[2 * m + 1] + ai * E[2 * m];
            }
            P[2 * ((size_t)q * N + pp)] = sr; P[2 * ((size_t)q * N + pp) + 1] = si;
        }
    free(E); free(A);
}

/* Textbook iterative radix-2 decimation-in-time, sign +, no scaling, length n = 2^lg,          */
/* tw[m] = exp(2 pi i m / n) for m < n/2.                                                       */
static void orc_fft1(double *x, int n, int lg, const double *tw) {
    for (int i = 0; i < n; ++i) {          /* bit reversal */
        int r = 0;
        for (int b = 0; b < lg; ++b) r |= ((i >> b) & 1) << (lg - 1 - b);
        if (r > i) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * r]; x[2 * i + 1] = x[2 * r + 1];
            x[2 * r] = tr; x[2 * r + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int s = 0; s < n; s += len)
            for (int m = 0; m < half; ++m) {
                double wr = tw[2 * (m * step)], wi = tw[2 * (m * step) + 1];
                double *a = x + 2 * (s + m), *b = x + 2 * (s + m + half);
                double br = b[0] * wr - b[1] * wi, bi = b[0] * wi + b[1] * wr;
                b[0] = a[0] - br; b[1] = a[1] - bi;
                a[0] += br; a[1] += bi;
            }
    }
}

static void orc_transpose(int N, double *X) {
    const int B = 32;
#pragma omp parallel for schedule(dynamic)
    for (int jb = 0; jb < N; jb += B)
        for (int ib = jb; ib < N; ib += B)
            for (int j = jb; j < jb + B && j < N; ++j)
                for (int i = (ib == jb ? j + 1 : ib); i < ib + B && i < N; ++i) {
                    size_t a = 2 * ((size_t)j * N + i), b = 2 * ((size_t)i * N + j);
                    double tr = X[a], ti = X[a + 1];
                    X[a] = X[b]; X[a + 1] = X[b + 1]; X[b] = tr; X[b + 1] = ti;
                }
}

/* In place, N a power of two.  P = cb * IFFT(cb * G), cb[j][i] = (-1)^(i+j): the centred        */
/* transform of orc_dft2_naive expressed through the ordinary (origin-at-0) one; the two           */
/* e^{i pi N/2} factors of the two axes multiply to 1 for even N.  Returns 0, or -1 if N is not   */
/* a power of two.                                                                                */
int orc_fft2(int32_t N, double *X) {
    int lg = 0; while ((1 << lg) < N) ++lg;
    if ((1 << lg) != N || N < 2) return -1;
    double *tw = malloc(sizeof(double) * (size_t)N);
    for (int m = 0; m < N / 2; ++m) {
        tw[2 * m] = cos(2.0 * ORC_PI * (double)m / (double)N);
        tw[2 * m + 1] = sin(2.0 * ORC_PI * (double)m / (double)N);
    }
    for (int pass = 0; pass < 2; ++pass) {
#pragma omp parallel for
        for (int j = 0; j < N; ++j) {
            double *row = X + 2 * (size_t)j * N;
            if (pass == 0)                      /* cb on the way in */
                for (int i = 0; i < N; ++i) if ((i + j) & 1) { row[2 * i] = -row[2 * i]; row[2 * i + 1] = -row[2 * i + 1]; }
            orc_fft1(row, N, lg, tw);
        }
        orc_transpose(N, X);
    }
#pragma omp parallel for
    for (int j = 0; j < N; ++j) {               /* cb on the way out */
        double *row = X + 2 * (size_t)j * N;
        for (int i = 0; i < N; ++i) if ((i + j) & 1) { row[2 * i] = -row[2 * i]; row[2 * i + 1] = -row[2 * i + 1]; }
    }
    free(tw);
    return 0;
}

/* ---- O8: w-correction and reduction over planes, Eq. 2 ------------------------------------- */
/* D[q][p] += sum_{k in [plane_lo, plane_hi)} exp(2 pi i w_k t) P[(k - plane_lo)][q][p],         */
/* t = n - 1 = -r^2 / (1 + sqrt(1 - r^2)), w_k = w_min + (k + 1/2) dw; pixels with r^2 >= 1      */
/* receive nothing (R14).                                                                        */
void orc_wcorrect(const orc_params *p, const double *P, int32_t plane_lo, int32_t plane_hi, double *D) {
    const int N = p->n_pix;
    const double dw = (p->w_max - p->w_min) / (double)p->n_wplanes;
#pragma omp parallel for
    for (int q = 0; q < N; ++q)
        for (int pp = 0; pp < N; ++pp) {
            double l = (double)(pp - N / 2) * p->cell_rad, m = (double)(q - N / 2) * p->cell_rad;
            double r2 = l * l + m * m;
            if (r2 >= 1.0) continue;
            double t = -r2 / (1.0 + sqrt(1.0 - r2));
            double sr = 0.0, si = 0.0;
            for (int k = plane_lo; k < plane_hi; ++k) {
                double wk = p->w_min + ((double)k + 0.5) * dw;
                double ph = 2.0 * ORC_PI * wk * t;
                double c = cos(ph), s = sin(ph);
                size_t idx = 2 * (((size_t)(k - plane_lo) * N + q) * N + pp);
                sr += c * P[idx] - s * P[idx + 1];
                si += s * P[idx] + c * P[idx + 1];
            }
            D[2 * ((size_t)q * N + pp)] += sr;
            D[2 * ((size_t)q * N + pp) + 1] += si;
        }
}

/* ---- the chain at single pixels, visibility-outermost ------------------------------------- */
/* D(q,p) = sum_vis wt V e^{2 pi i w_k t} [sum_a gu[a] e^{2 pi i (i0+a-N/2)(p-N/2)/N}]            */
/*                                         [sum_b gv[b] e^{2 pi i (j0+b-N/2)(q-N/2)/N}]            */
/* i.e. O6 -> O7 -> O8 with the three finite sums re-ordered; no mesh is formed.                  */
void orc_image_samples(const orc_params *p, const float *uvw, const float *vis, const float *wt,
                       const double *freq_hz, int64_t n_rows, int32_t n_chan,
                       int32_t n_samp, const int32_t *sq, const int32_t *sp, double *D /* re,im per sample */) {
    const int N = p->n_pix, S = p->support, h = (S - 1) / 2, Nw = p->n_wplanes;
    const double dw = (p->w_max - p->w_min) / (double)Nw;
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
    /* per sample and plane: the w phase; per sample: nothing else is shared */
    double *wph = malloc(sizeof(double) * 2 * (size_t)n_samp * Nw);
    for (int s = 0; s < n_samp; ++s) {
        double l = (double)(sp[s] - N / 2) * p->cell_rad, m = (double)(sq[s] - N / 2) * p->cell_rad;
        double r2 = l * l + m * m;
        for (int k = 0; k < Nw; ++k) {
            if (r2 >= 1.0) { wph[2 * ((size_t)s * Nw + k)] = 0.0; wph[2 * ((size_t)s * Nw + k) + 1] = 0.0; continue; }
            double t = -r2 / (1.0 + sqrt(1.0 - r2));
            double ph = 2.0 * ORC_PI * (p->w_min + ((double)k + 0.5) * dw) * t;
            wph[2 * ((size_t)s * Nw + k)] = cos(ph); wph[2 * ((size_t)s * Nw + k) + 1] = sin(ph);
        }
    }
    double *E = malloc(sizeof(double) * 2 * (size_t)N);       /* E[m] = exp(2 pi i m / N) */
    for (int m = 0; m < N; ++m) {
        E[2 * m] = cos(2.0 * ORC_PI * (double)m / (double)N);
        E[2 * m + 1] = sin(2.0 * ORC_PI * (double)m / (double)N);
    }
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    double *part = calloc((size_t)nthreads * 2 * n_samp, sizeof(double));
#pragma omp parallel
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *acc = part + (size_t)tid * 2 * n_samp;
        double gu[32], gv[32];
#pragma omp for schedule(static)
        for (int64_t r = 0; r < n_rows; ++r) {
            double u = (double)uvw[3 * r], v = (double)uvw[3 * r + 1], w = (double)uvw[3 * r + 2];
            for (int c = 0; c < n_chan; ++c) {
                int32_t i0, j0, k; double fu, fv;
                if (!orc_place(p, u, v, w, su[c], sw[c], ow, &i0, &j0, &k, &fu, &fv)) continue;
                int64_t mi = r * n_chan + c;
                double vr = (double)wt[mi] * (double)vis[2 * mi], vi = (double)wt[mi] * (double)vis[2 * mi + 1];
                for (int a = -h; a <= h; ++a) {
                    gu[a + h] = orc_kernel1d(p, (double)a - fu);
                    gv[a + h] = orc_kernel1d(p, (double)a - fv);
                }
                for (int s = 0; s < n_samp; ++s) {
                    double xr = 0, xi = 0, yr = 0, yi = 0;
                    for (int a = -h; a <= h; ++a) {
                        int64_t mx = (((int64_t)(i0 + a) - N / 2) * ((int64_t)sp[s] - N / 2)) % N; if (mx < 0) mx += N;
                        int64_t my = (((int64_t)(j0 + a) - N / 2) * ((int64_t)sq[s] - N / 2)) % N; if (my < 0) my += N;
                        xr += gu[a + h] * E[2 * mx]; xi += gu[a + h] * E[2 * mx + 1];
                        yr += gv[a + h] * E[2 * my]; yi += gv[a + h] * E[2 * my + 1];
                    }
                    double fr = xr * yr - xi * yi, fi = xr * yi + xi * yr;           /* footprint's DFT  */
                    double cr = wph[2 * ((size_t)s * Nw + k)], ci = wph[2 * ((size_t)s * Nw + k) + 1];
                    double gr = fr * cr - fi * ci, gi = fr * ci + fi * cr;           /* x w screen       */
                    acc[2 * s] += vr * gr - vi * gi;
                    acc[2 * s + 1] += vr * gi + vi * gr;
                }
            }
        }
    }
    for (int s = 0; s < n_samp; ++s) {
        double sr = 0, si = 0;
        for (int t = 0; t < nthreads; ++t) { sr += part[(size_t)t * 2 * n_samp + 2 * s]; si += part[(size_t)t * 2 * n_samp + 2 * s + 1]; }
        D[2 * s] = sr; D[2 * s + 1] = si;
    }
    free(part); free(wph); free(E); free(su); free(sw);
}

/* ---- degridding: image -> visibilities (Eq. 1 :59 discretised; reading R30) ---------- */
/* Step 1: Q[q][p] = M[q][p] exp(-2 pi i w_k t), t = n - 1 as in O8; pixels with r^2 >= 1 give 0 (R14).   */
void orc_wscreen_fwd(const orc_params *p, const double *M, int32_t k, double *Q) {
    const int N = p->n_pix;
    const double dw = (p->w_max - p->w_min) / (double)p->n_wplanes;
    const double wk = p->w_min + ((double)k + 0.5) * dw;
#pragma omp parallel for
    for (int q = 0; q < N; ++q)
        for (int pp = 0; pp < N; ++pp) {
            size_t idx = 2 * ((size_t)q * N + pp);
            double l = (double)(pp - N / 2) * p->cell_rad, m = (double)(q - N / 2) * p->cell_rad;
            double r2 = l * l + m * m;
            if (r2 >= 1.0) { Q[idx] = 0.0; Q[idx + 1] = 0.0; continue; }
            double t = -r2 / (1.0 + sqrt(1.0 - r2));
            double ph = -2.0 * ORC_PI * wk * t;
            double c = cos(ph), s = sin(ph);
            Q[idx] = c * M[idx] - s * M[idx + 1];
            Q[idx + 1] = s * M[idx] + c * M[idx + 1];
        }
}

/* Step 3: V_m = sum_{a,b} g(a - fu) g(b - fv) H[(k - plane_lo)][j0 + b][i0 + a] for every kept visibility   */
/* whose plane lies in [plane_lo, plane_hi); others are left untouched (the caller starts from zeros, so a    */
/* dropped visibility predicts 0).  H: forward-transformed planes, logical centred layout.  out: re,im.       */
void orc_degrid(const orc_params *p, const float *uvw, const double *freq_hz, int64_t n_rows, int32_t n_chan,
                int32_t plane_lo, int32_t plane_hi, const double *H, double *out) {
    const int N = p->n_pix, S = p->support, h = (S - 1) / 2;
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
#pragma omp parallel for
    for (int64_t r = 0; r < n_rows; ++r) {
        double gu[32], gv[32];
        double u = (double)uvw[3 * r], v = (double)uvw[3 * r + 1], w = (double)uvw[3 * r + 2];
        for (int c = 0; c < n_chan; ++c) {
            int32_t i0, j0, k; double fu, fv;
            if (!orc_place(p, u, v, w, su[c], sw[c], ow, &i0, &j0, &k, &fu, &fv) || k < plane_lo || k >= plane_hi) continue;
            const double *Hk = H + (size_t)(k - plane_lo) * (size_t)N * (size_t)N * 2;
            for (int a = -h; a <= h; ++a) {
                gu[a + h] = orc_kernel1d(p, (double)a - fu);
                gv[a + h] = orc_kernel1d(p, (double)a - fv);
            }
            double sr = 0.0, si = 0.0;
            for (int b = -h; b <= h; ++b)
                for (int a = -h; a <= h; ++a) {
                    double t = gu[a + h] * gv[b + h];
                    size_t cell = ((size_t)(j0 + b) * (size_t)N + (size_t)(i0 + a)) * 2;
                    sr += t * Hk[cell];
                    si += t * Hk[cell + 1];
                }
            out[2 * (r * n_chan + c)] = sr;
            out[2 * (r * n_chan + c) + 1] = si;
        }
    }
    free(su); free(sw);
}

/* The degridding chain at single visibilities for a SPARSE model (n_src non-zero pixels (sq, sp) with values sval):   */
/* V_m = sum_s val_s e^{-2 pi i w_k t_s} [sum_a gu[a] e^{-2 pi i (i0+a-N/2)(p_s-N/2)/N}] [sum_b gv[b] e^{-2 pi i (j0+b-N/2)(q_s-N/2)/N}] */
/* i.e. steps 1-3 with the finite sums re-ordered (visibility outermost); no plane is formed.  Used at sizes where the   */
/* fp64 plane stack cannot be transformed in reasonable time; pinned against the chain.  samp: flat indices row*n_chan+c. */
void orc_predict_samples(const orc_params *p, const float *uvw, const double *freq_hz, int32_t n_chan,
                         int32_t n_src, const int32_t *sq, const int32_t *sp, const double *sval,
                         int64_t n_samp, const int64_t *samp, double *out) {
    const int N = p->n_pix, S = p->support, h = (S - 1) / 2, Nw = p->n_wplanes;
    const double dw = (p->w_max - p->w_min) / (double)Nw;
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
    double *E = malloc(sizeof(double) * 2 * (size_t)N);       /* E[m] = exp(-2 pi i m / N) */
    for (int m = 0; m < N; ++m) {
        E[2 * m] = cos(2.0 * ORC_PI * (double)m / (double)N);
        E[2 * m + 1] = -sin(2.0 * ORC_PI * (double)m / (double)N);
    }
    double *ts = malloc(sizeof(double) * n_src);              /* n - 1 per source pixel; NaN marks r^2 >= 1 */
    for (int s = 0; s < n_src; ++s) {
        double l = (double)(sp[s] - N / 2) * p->cell_rad, m = (double)(sq[s] - N / 2) * p->cell_rad;
        double r2 = l * l + m * m;
        ts[s] = r2 < 1.0 ? -r2 / (1.0 + sqrt(1.0 - r2)) : NAN;
    }
#pragma omp parallel for
    for (int64_t n = 0; n < n_samp; ++n) {
        double gu[32], gv[32];
        int64_t r = samp[n] / n_chan; int c = (int)(samp[n] % n_chan);
        int32_t i0, j0, k; double fu, fv;
        out[2 * n] = 0.0; out[2 * n + 1] = 0.0;
        if (!orc_place(p, (double)uvw[3 * r], (double)uvw[3 * r + 1], (double)uvw[3 * r + 2], su[c], sw[c], ow,
                       &i0, &j0, &k, &fu, &fv)) continue;
        for (int a = -h; a <= h; ++a) {
            gu[a + h] = orc_kernel1d(p, (double)a - fu);
            gv[a + h] = orc_kernel1d(p, (double)a - fv);
        }
        const double wk = p->w_min + ((double)k + 0.5) * dw;
        double vr = 0.0, vi = 0.0;
        for (int s = 0; s < n_src; ++s) {
            if (isnan(ts[s])) continue;
            double xr = 0, xi = 0, yr = 0, yi = 0;
            for (int a = -h; a <= h; ++a) {
                int64_t mx = (((int64_t)(i0 + a) - N / 2) * ((int64_t)sp[s] - N / 2)) % N; if (mx < 0) mx += N;
                int64_t my = (((int64_t)(j0 + a) - N / 2) * ((int64_t)sq[s] - N / 2)) % N; if (my < 0) my += N;
                xr += gu[a + h] * E[2 * mx]; xi += gu[a + h] * E[2 * mx + 1];
                yr += gv[a + h] * E[2 * my]; yi += gv[a + h] * E[2 * my + 1];
            }
            double fr = xr * yr - xi * yi, fi = xr * yi + xi * yr;
            double ph = -2.0 * ORC_PI * wk * ts[s];
            double cr = cos(ph), ci = sin(ph);
            double gr = fr * cr - fi * ci, gi = fr * ci + fi * cr;
            vr += sval[2 * s] * gr - sval[2 * s + 1] * gi;
            vi += sval[2 * s] * gi + sval[2 * s + 1] * gr;
        }
        out[2 * n] = vr; out[2 * n + 1] = vi;
    }
    free(su); free(sw); free(E); free(ts);
}

/* ---- normalisation of the image (Eq. 2 solved for I; readings R12, R29) ------------------- */
/* Sum of the weights of the kept visibilities (O3), in input order.                             */
double orc_sum_weights(const orc_params *p, const float *uvw, const float *wt, const double *freq_hz,
                       int64_t n_rows, int32_t n_chan) {
    double *su = malloc(sizeof(double) * n_chan), *sw = malloc(sizeof(double) * n_chan), ow, sum = 0.0;
    orc_channel_constants(p, freq_hz, n_chan, su, sw, &ow);
    for (int64_t r = 0; r < n_rows; ++r) {
        double u = (double)uvw[3 * r], v = (double)uvw[3 * r + 1], w = (double)uvw[3 * r + 2];
        for (int c = 0; c < n_chan; ++c) {
            int32_t i0, j0, k; double fu, fv;
            if (orc_place(p, u, v, w, su[c], sw[c], ow, &i0, &j0, &k, &fu, &fv)) sum += (double)wt[r * n_chan + c];
        }
    }
    free(su); free(sw);
    return sum;
}

/* dirty[q][p] = Re D[q][p] * f, f the product of the factors `flags` selects:                    */
/*   1 (SUMWT): 1 / sum_wt        -- the direct sum I = sum wt V e^{..} becomes a weighted mean    */
/*   2 (N):     n = sqrt(1-l^2-m^2) -- the 1/n on the left side of Eq. 2              */
/*   4 (TAPER): 1 / (ghat(xi_p) ghat(xi_q)), xi = (p - N/2)/N -- undoes the image-plane response    */
/*              of the convolution function.  Pixels with l^2+m^2 >= 1 stay 0 (R14).                */
void orc_dirty(const orc_params *p, const double *D, uint32_t flags, double sum_wt, double *dirty) {
    const int N = p->n_pix;
    for (int q = 0; q < N; ++q)
        for (int pp = 0; pp < N; ++pp) {
            double f = 1.0;
            double l = (double)(pp - N / 2) * p->cell_rad, m = (double)(q - N / 2) * p->cell_rad;
            double r2 = l * l + m * m;
            if (flags & 1u) f /= sum_wt;
            if (flags & 2u) f *= r2 < 1.0 ? sqrt(1.0 - r2) : 0.0;
            if (flags & 4u)
                f /= orc_taper1d(p, (double)(pp - N / 2) / (double)N) * orc_taper1d(p, (double)(q - N / 2) / (double)N);
            dirty[(size_t)q * N + pp] = D[2 * ((size_t)q * N + pp)] * f;
        }
}

int32_t orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
