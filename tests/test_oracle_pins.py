"""Pins for the fp64 oracle (CPU only): what the paper and the mathematics fix, written
independently of oracle/wstack_oracle.c (numpy / fractions here, never the oracle's own formulae
re-called).  DESIGN.md section 5 lists which plausible mistake each pin catches.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from synth import get_config, make_dataset, make_random_dataset
from synth.interferometer import C_LIGHT

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _prm(oracle, d, tile=32, **kw):
    return oracle.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad,
                               w_min=d.w_min, w_max=d.w_max, sigma=d.sigma_cells, tile=tile, **kw)


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


def _small(seed=7, n_rows=300, n_chan=1, n_pix=64, n_w=4, support=7, **kw):
    return make_random_dataset(seed, n_rows, n_chan, n_pix, n_w, support, **kw)


def _independent_positions(d, n_chan):
    """pu, pv, pw per visibility by plain numpy fp64 (not fma): independent of orc_place."""
    uvw = d.uvw.numpy().astype(np.float64)
    sc = d.chan_scale()
    N, dw = d.n_pix, (d.w_max - d.w_min) / d.n_wplanes
    pu = np.multiply.outer(uvw[:, 0], sc * N * d.cell_rad) + N / 2
    pv = np.multiply.outer(uvw[:, 1], sc * N * d.cell_rad) + N / 2
    pw = (np.multiply.outer(uvw[:, 2], sc) - d.w_min) / dw
    return pu.ravel(), pv.ravel(), pw.ravel()


def _gauss(x, sigma):
    return np.exp(-0.5 * (x / sigma) ** 2) / (sigma * math.sqrt(2 * math.pi))


# --------------------------------------------------------------------------- paper-printed numbers
def test_golden_footprint_is_full_square(oracle):
    """PAPER.md:380 / Table 3: 26.65 G additions for 0.54 G visibilities = 49 = 7 x 7 per visibility:
    the footprint is the full S x S square (reading R3), not a disc."""
    vals = {}
    for line in open(os.path.join(GOLDEN, "paper_numbers.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    S = int(vals["kernel_support_cells"])
    assert round(vals["giga_grid_point_additions_medium"] / vals["n_visibilities_medium_giga"]) == S * S
    d = _small(n_rows=1, n_w=1, support=S, fill=0.5)
    G = oracle.grid(_prm(oracle, d), *_np(d))
    assert np.count_nonzero(G) == S * S
    jj, ii = np.nonzero(G[0])
    assert jj.max() - jj.min() == S - 1 and ii.max() - ii.min() == S - 1


# --------------------------------------------------------------------------- P9: bins, exact
def test_p9_positions_and_keys_exact_rational(oracle):
    """Keys recomputed with exact rational arithmetic: Fraction(u)*Fraction(su)+N/2 rounded once to
    binary64 is, by definition, the IEEE fma.  Sample includes visibilities close to cell borders."""
    d = _small(seed=11, n_rows=400, n_chan=3, n_pix=128, n_w=5, wavelengths=False, fill=1.05)
    prm = _prm(oracle, d, tile=32)
    pos = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)
    N, T, h, Nw = d.n_pix, 32, 3, d.n_wplanes
    dw = (d.w_max - d.w_min) / Nw
    uvw = d.uvw.numpy()
    n_checked = n_dropped = 0
    for r in range(d.n_rows):
        for c in range(d.n_chan):
            su = (d.freqs_hz[c] / C_LIGHT) * (N * d.cell_rad)
            sw = (d.freqs_hz[c] / C_LIGHT) / dw
            ow = -d.w_min / dw
            pu = float(Fraction(float(uvw[r, 0])) * Fraction(su) + N // 2)
            pv = float(Fraction(float(uvw[r, 1])) * Fraction(su) + N // 2)
            pw = float(Fraction(float(uvw[r, 2])) * Fraction(sw) + Fraction(ow))
            i0, j0 = math.floor(pu + 0.5), math.floor(pv + 0.5)
            k = min(max(math.floor(pw), 0), Nw - 1)
            m = r * d.n_chan + c
            if h <= i0 <= N - 1 - h and h <= j0 <= N - 1 - h:
                key = (k * (N // T) + j0 // T) * (N // T) + i0 // T
                assert (pos["i0"][m], pos["j0"][m], pos["k"][m]) == (i0, j0, k)
                assert pos["fu"][m] == pu - i0 and pos["fv"][m] == pv - j0
                assert -0.5 <= pos["fu"][m] < 0.5
            else:
                key = 0xFFFFFFFF
                n_dropped += 1
            assert pos["key"][m] == key
            n_checked += 1
    assert n_checked == d.n_vis and 0 < n_dropped < d.n_vis // 4


def test_nan_coordinates_are_dropped(oracle):
    """DESIGN.md R33: a visibility with a NaN in u, v or w is dropped (key 0xFFFFFFFF, no contribution); +-Inf in w
    clamps into the first / last plane like any w outside [w_min, w_max] (R6).  Pinned by construction: the mesh of the
    data with such rows inserted equals the mesh of the data without them (+ the clamped ones added by hand)."""
    d = _small(seed=15, n_rows=300, n_chan=2, n_pix=128, n_w=4, fill=0.8)
    prm = _prm(oracle, d, tile=32)
    uvw, vis, wt = d.uvw.numpy().copy(), d.vis.numpy(), d.weights.numpy()
    clean = oracle.grid(prm, uvw, vis, wt, d.freqs_hz)
    bad = uvw.copy()
    bad[3, 0] = np.nan
    bad[7, 1] = np.nan
    bad[11, 2] = np.nan
    bad[20, 2] = np.inf
    bad[21, 2] = -np.inf
    pos = oracle.positions(prm, bad, d.n_chan, d.freqs_hz)
    key = pos["key"].reshape(d.n_rows, d.n_chan)
    assert np.all(key[[3, 7, 11]] == 0xFFFFFFFF)
    assert np.all(pos["k"].reshape(d.n_rows, d.n_chan)[20] == prm.n_wplanes - 1) and np.all(pos["k"].reshape(d.n_rows, d.n_chan)[21] == 0)
    ok = np.ones(d.n_rows, bool)
    ok[[3, 7, 11]] = False
    ref_uvw = uvw[ok].copy()
    sel = np.flatnonzero(ok)
    ref_uvw[np.searchsorted(sel, 20), 2] = 1e30          # far beyond w_max: clamps into the last plane
    ref_uvw[np.searchsorted(sel, 21), 2] = -1e30
    want = oracle.grid(prm, ref_uvw, vis[ok], wt[ok], d.freqs_hz)
    got = oracle.grid(prm, bad, vis, wt, d.freqs_hz)
    assert np.array_equal(got, want) and not np.array_equal(got, clean)
    assert oracle.sum_weights(prm, bad, wt, d.freqs_hz) == pytest.approx(float(wt[ok].astype(np.float64).sum()), rel=1e-12)


def test_p9_bins_are_a_stable_counting_sort(oracle):
    d = _small(seed=12, n_rows=5000, n_chan=2, n_pix=128, n_w=3, fill=1.02)
    prm = _prm(oracle, d, tile=32)
    key = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)["key"]
    bin_start, perm, dropped = oracle.bins(prm, key)
    kept = np.flatnonzero(key != 0xFFFFFFFF)
    assert dropped == key.size - kept.size and dropped > 0
    order = kept[np.argsort(key[kept], kind="stable")]          # numpy's stable sort: independent routine
    assert np.array_equal(perm, order.astype(np.uint32))
    assert np.array_equal(bin_start, np.searchsorted(key[order], np.arange(prm.n_bins + 1)).astype(np.uint32))
    assert bin_start[0] == 0 and bin_start[-1] == kept.size and np.all(np.diff(bin_start.astype(np.int64)) >= 0)


def test_plane_assignment_is_closest_midpoint(oracle):
    """PAPER.md:66 'mapped to the closest w-plane': plane k has value w_min+(k+1/2)dw (R6); the assigned
    plane must be the one whose value is nearest to w."""
    d = _small(seed=13, n_rows=2000, n_w=7, w_span=300.0)
    prm = _prm(oracle, d)
    k = oracle.positions(prm, d.uvw.numpy(), 1)["k"]
    dw = (d.w_max - d.w_min) / d.n_wplanes
    mid = d.w_min + (np.arange(d.n_wplanes) + 0.5) * dw
    w = d.uvw.numpy()[:, 2].astype(np.float64)
    nearest = np.abs(w[:, None] - mid[None, :]).argmin(1)
    far_from_border = np.abs(((w - d.w_min) / dw) % 1.0 - 0.5) < 0.499
    assert np.array_equal(k[far_from_border], nearest[far_from_border])
    assert k.min() == 0 and k.max() == d.n_wplanes - 1        # w_max clamps into the last plane


# --------------------------------------------------------------------------- P4 / P3: mass
def test_p4_mass_per_plane(oracle):
    """Sum of a plane = sum over its visibilities of wt V Ku Kv, tap sums computed here independently."""
    d = _small(seed=21, n_rows=500, n_chan=2, n_pix=96, n_w=3, wavelengths=False)
    prm = _prm(oracle, d)
    G = oracle.grid(prm, *_np(d))
    pu, pv, pw = _independent_positions(d, d.n_chan)
    i0, j0 = np.floor(pu + 0.5), np.floor(pv + 0.5)
    k = np.clip(np.floor(pw), 0, d.n_wplanes - 1).astype(int)
    h = 3
    keep = (i0 >= h) & (i0 <= d.n_pix - 1 - h) & (j0 >= h) & (j0 <= d.n_pix - 1 - h)
    a = np.arange(-h, h + 1)
    Ku = _gauss(a[None, :] - (pu - i0)[:, None], d.sigma_cells).sum(1)
    Kv = _gauss(a[None, :] - (pv - j0)[:, None], d.sigma_cells).sum(1)
    val = (d.weights.numpy().ravel().astype(np.float64) * d.vis.numpy().ravel().astype(np.complex128)) * Ku * Kv
    for kk in range(d.n_wplanes):
        ref = val[keep & (k == kk)].sum()
        assert abs(G[kk].sum() - ref) <= 1e-12 * max(1.0, abs(ref))
    # kernel normalisation (R2): unit-integral Gaussian, truncated at +-3.5 sigma
    assert 0.9990 < Ku.min() and Ku.max() < 0.9998


def test_p3_centre_pixel_is_total_mass(oracle):
    d = _small(seed=22, n_rows=400, n_pix=64, n_w=4)
    prm = _prm(oracle, d)
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    c = d.n_pix // 2
    assert abs(D[c, c] - G.sum()) <= 1e-12 * abs(G.sum())


# --------------------------------------------------------------------------- P6: textbook reduction
def test_p6_delta_kernel_reduces_to_numpy_ifft2(oracle):
    """N_w = 1, w = 0, S = 1, uvw on cell centres: the chain is the inverse DFT of the sample histogram."""
    N, n = 64, 200
    rng = np.random.default_rng(31)
    cell = 1e-3
    ii, jj = rng.integers(0, N, n), rng.integers(0, N, n)
    du = 1.0 / (N * cell)
    uvw = np.stack([(ii - N // 2) * du, (jj - N // 2) * du, np.zeros(n)], 1).astype(np.float32)
    # float32 rounding moves samples off the centres by < 1e-4 cells: still the same nearest cell
    vis = (rng.standard_normal(n) + 1j * rng.standard_normal(n)).astype(np.complex64)[:, None]
    wt = rng.uniform(0.5, 1.5, (n, 1)).astype(np.float32)
    prm = oracle.OracleParams(n_pix=N, n_wplanes=1, support=1, cell_rad=cell, w_min=-1.0, w_max=1.0, sigma=1.0)
    hist = np.zeros((N, N), np.complex128)
    np.add.at(hist, (jj, ii), wt[:, 0].astype(np.float64) * vis[:, 0].astype(np.complex128))
    G = oracle.grid(prm, uvw, vis, wt)
    g0 = 1.0 / math.sqrt(2 * math.pi)
    assert np.allclose(G[0], hist * g0 * g0, rtol=1e-6, atol=1e-9)       # fu ~ 1e-5: g(fu) ~ g(0)(1 - 5e-11)
    D = oracle.dirty_image(prm, uvw, vis, wt)
    ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(G[0]))) * N * N   # w-screen is e^{2 pi i * 0 * t} = 1
    assert np.abs(D - ref).max() <= 1e-11 * np.abs(ref).max()


@pytest.mark.parametrize("N", [2, 4, 8, 16, 32, 64, 128, 256, 512])
def test_fft_matches_naive_dft_and_numpy(oracle, N):
    rng = np.random.default_rng(100 + N)
    x = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    f = oracle.fft2(x)
    ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(x))) * N * N
    assert np.abs(f - ref).max() <= 1e-12 * np.abs(ref).max()
    if N <= 128 or N == 512:
        nv = oracle.dft2_naive(x)
        assert np.abs(nv - ref).max() <= 1e-11 * np.abs(ref).max()


def test_naive_dft_non_power_of_two_and_asymmetry(oracle):
    """A single off-centre cell must give the phase ramp with the + sign in BOTH axes (R10) and the
    axes not transposed: catches a conjugated or transposed transform."""
    N = 12
    x = np.zeros((N, N), np.complex128)
    j, i = 8, 3                       # v-offset +2, u-offset -3
    x[j, i] = 1.0
    P = oracle.dft2_naive(x)
    q, p = np.meshgrid(np.arange(N) - N // 2, np.arange(N) - N // 2, indexing="ij")
    ref = np.exp(2j * np.pi * ((i - N // 2) * p + (j - N // 2) * q) / N)
    assert np.abs(P - ref).max() < 1e-13
    with pytest.raises(ValueError):
        oracle.fft2(x)


# --------------------------------------------------------------------------- P1: closed form, no mesh, no DFT
def _closed_form_image(d, tap=None):
    """D(l,m) per visibility with numpy: wt V e^{2 pi i w_k t} [sum_a gu e^{2 pi i (i0+a-N/2) du l}] [same in v].
    `tap`: the 1-D convolution function (default: the Gaussian of PAPER.md:82)."""
    tap = tap or (lambda x: _gauss(x, d.sigma_cells))
    N, h = d.n_pix, (d.support - 1) // 2
    pu, pv, pw = _independent_positions(d, d.n_chan)
    i0, j0 = np.floor(pu + 0.5), np.floor(pv + 0.5)
    k = np.clip(np.floor(pw), 0, d.n_wplanes - 1)
    keep = (i0 >= h) & (i0 <= N - 1 - h) & (j0 >= h) & (j0 <= N - 1 - h)
    val = d.weights.numpy().ravel().astype(np.float64) * d.vis.numpy().ravel().astype(np.complex128)
    dw = (d.w_max - d.w_min) / d.n_wplanes
    wk = d.w_min + (k + 0.5) * dw
    x = (np.arange(N) - N // 2) * d.cell_rad
    l, m = np.meshgrid(x, x, indexing="xy")        # l varies along the last axis
    r2 = l * l + m * m
    t = np.where(r2 < 1, np.sqrt(np.clip(1 - r2, 0, None)) - 1.0, 0.0)   # n - 1 by subtraction: fine in fp64 here
    du = 1.0 / (N * d.cell_rad)
    D = np.zeros((N, N), np.complex128)
    a = np.arange(-h, h + 1)
    for n in np.flatnonzero(keep):
        gu = tap(a - (pu[n] - i0[n]))
        gv = tap(a - (pv[n] - j0[n]))
        fx = (gu[:, None] * np.exp(2j * np.pi * np.outer((i0[n] + a - N // 2) * du, x))).sum(0)   # [N] over l
        fy = (gv[:, None] * np.exp(2j * np.pi * np.outer((j0[n] + a - N // 2) * du, x))).sum(0)   # [N] over m
        D += val[n] * np.exp(2j * np.pi * wk[n] * t) * np.outer(fy, fx)
    D[r2 >= 1] = 0
    return D


def test_p1_closed_form_whole_chain(oracle):
    d = _small(seed=41, n_rows=60, n_chan=2, n_pix=64, n_w=4, wavelengths=False, fill=1.0, w_span=40.0,
               cell_rad=6e-3)     # FoV 0.38 rad: the w-screen is far from 1
    prm = _prm(oracle, d)
    D = oracle.dirty_image(prm, *_np(d))
    ref = _closed_form_image(d)
    err = np.linalg.norm(D - ref) / np.linalg.norm(ref)
    assert err < 1e-12, err
    # the FFT route of O7 gives the same image
    D2 = oracle.dirty_image(prm, *_np(d), naive_max=0)
    assert np.linalg.norm(D2 - ref) / np.linalg.norm(ref) < 1e-12


def test_image_samples_equal_the_chain(oracle):
    d = _small(seed=42, n_rows=500, n_chan=3, n_pix=128, n_w=6, wavelengths=False, w_span=80.0, cell_rad=3e-3)
    prm = _prm(oracle, d)
    D = oracle.dirty_image(prm, *_np(d))
    rng = np.random.default_rng(1)
    q, p = rng.integers(0, d.n_pix, 40), rng.integers(0, d.n_pix, 40)
    q[:3], p[:3] = [0, 64, 127], [127, 64, 0]
    s = oracle.image_samples(prm, *_np(d), q, p)
    assert np.abs(s - D[q, p]).max() <= 1e-11 * np.abs(D).max()


# --------------------------------------------------------------------------- P2: brute-force direct DFT
def _model_dataset(n_w, seed=51, n_pix=64):
    """Noise-free visibilities of 3 asymmetric point sources (Eq. 1 without 1/n) on random uvw."""
    d = _small(seed=seed, n_rows=1500, n_pix=n_pix, n_w=n_w, fill=0.85, w_span=60.0, cell_rad=4e-3,
               unit_weights=True)
    l = np.array([0.031, -0.052, 0.012]); m = np.array([-0.043, 0.018, 0.066]); f = np.array([1.0, 0.7, 0.5])
    nm1 = np.sqrt(1 - l * l - m * m) - 1
    uvw = d.uvw.numpy().astype(np.float64)
    ph = uvw[:, :1] * l + uvw[:, 1:2] * m + uvw[:, 2:3] * nm1
    import torch
    d.vis = torch.from_numpy((np.exp(-2j * np.pi * ph) @ f).astype(np.complex64)[:, None])
    return d, (l, m, f)


def _direct_dft(d, w_used):
    """I(l,m) = sum wt V e^{+2 pi i (u l + v m + w (n-1))} at every pixel (north_star's brute force)."""
    N = d.n_pix
    uvw = d.uvw.numpy().astype(np.float64)
    val = d.weights.numpy()[:, 0].astype(np.float64) * d.vis.numpy()[:, 0].astype(np.complex128)
    x = (np.arange(N) - N // 2) * d.cell_rad
    I = np.zeros((N, N), np.complex128)
    for q in range(N):
        nm1 = np.sqrt(1 - x * x - x[q] ** 2) - 1
        ph = np.outer(uvw[:, 0], x) + (uvw[:, 1] * x[q])[:, None] + np.outer(w_used, nm1)
        I[q] = (val[:, None] * np.exp(2j * np.pi * ph)).sum(0)
    return I


def test_p2_direct_dft_with_snapped_w(oracle):
    """D / (ghat(xi_l) ghat(xi_m)) ~ I when w is snapped to the plane midpoints; ghat = e^{-2 pi^2 sigma^2 xi^2}.
    Bound: few 1e-3 of the peak in the inner half for S = 7, sigma = 1.
    Catches: sign of the transform or of the w-term, u/v transposition, wrong w_k, wrong cell scale."""
    d, (ls, ms, fs) = _model_dataset(n_w=8)
    prm = _prm(oracle, d)
    D = oracle.dirty_image(prm, *_np(d))
    k = oracle.positions(prm, d.uvw.numpy(), 1)["k"]
    dw = (d.w_max - d.w_min) / d.n_wplanes
    I = _direct_dft(d, d.w_min + (k + 0.5) * dw)
    N = d.n_pix
    xi = (np.arange(N) - N // 2) / N
    gh = np.exp(-2 * np.pi ** 2 * d.sigma_cells ** 2 * xi ** 2)
    C = D / np.outer(gh, gh)
    inner = slice(N // 4, 3 * N // 4)
    err = np.abs(C[inner, inner] - I[inner, inner]).max() / np.abs(I).max()
    assert err < 5e-3, err
    # the brightest pixel sits on the brightest source (l -> column, m -> row)
    q, p = np.unravel_index(np.abs(C[inner, inner]).argmax(), (N // 2, N // 2))
    assert (p + N // 4 - N // 2, q + N // 4 - N // 2) == (round(ls[0] / d.cell_rad), round(ms[0] / d.cell_rad))
    # a mirrored / conjugated chain would put it elsewhere: the model is asymmetric
    assert np.abs(C[N // 2 - (q + N // 4 - N // 2), N // 2 - (p + N // 4 - N // 2)]) < 0.6 * np.abs(C[inner, inner]).max()


def test_p2_plane_quantisation_error_falls_with_n_wplanes(oracle):
    """Against the un-snapped direct DFT the extra error is <= 2 pi (dw/2) |n-1| and must fall ~ 1/N_w."""
    errs = []
    for n_w in (2, 8, 32):
        d, _ = _model_dataset(n_w=n_w)
        D = oracle.dirty_image(_prm(oracle, d), *_np(d))
        I = _direct_dft(d, d.uvw.numpy()[:, 2].astype(np.float64))
        N = d.n_pix
        xi = (np.arange(N) - N // 2) / N
        gh = np.exp(-2 * np.pi ** 2 * xi ** 2)
        inner = slice(N // 4, 3 * N // 4)
        errs.append(np.abs((D / np.outer(gh, gh))[inner, inner] - I[inner, inner]).max() / np.abs(I).max())
    assert errs[0] > 2.5 * errs[1] and errs[1] > errs[2] and errs[2] < 6e-3, errs


# --------------------------------------------------------------------------- P5 / P7 / P8
def test_p5_point_source_at_phase_centre(oracle):
    d = _small(seed=61, n_rows=800, n_pix=64, n_w=4, w_span=30.0, cell_rad=5e-3)
    import torch
    d.vis = torch.ones_like(d.vis)
    prm = _prm(oracle, d)
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    c = d.n_pix // 2
    assert np.abs(D).argmax() == c * d.n_pix + c
    assert abs(D[c, c].imag) < 1e-9 and D[c, c].real > 0
    assert abs(D[c, c] - G.sum()) < 1e-9
    assert np.all(G.imag == 0) and np.all(G.real >= 0)


def test_p7_hermitian_consistency(oracle):
    """Appending (-u,-v,-w, V*) with a symmetric plane range makes the mesh Hermitian and the image real."""
    d = _small(seed=71, n_rows=400, n_pix=64, n_w=6, fill=0.8, w_span=50.0, cell_rad=5e-3)
    uvw, vis, wt, _ = _np(d)
    uvw2 = np.concatenate([uvw, -uvw]); vis2 = np.concatenate([vis, vis.conj()]); wt2 = np.concatenate([wt, wt])
    W = float(np.abs(uvw[:, 2]).max()) * 1.01
    prm = oracle.OracleParams(n_pix=d.n_pix, n_wplanes=6, support=7, cell_rad=d.cell_rad, w_min=-W, w_max=W)
    D, G = oracle.dirty_image(prm, uvw2, vis2, wt2, return_grid=True)
    Dh = oracle.dirty_image(prm, uvw, vis, wt)
    N = d.n_pix
    mirrored = np.conj(G[::-1, ::-1, ::-1])                 # G[Nw-1-k][N-1-j][N-1-i]
    assert np.abs(G[:, 1:, 1:] - mirrored[:, :-1, :-1]).max() <= 1e-12 * np.abs(G).max()   # (N-j, N-i) for i,j >= 1
    assert np.abs(D.imag).max() <= 1e-12 * np.abs(D).max()
    assert np.abs(D.real - 2 * Dh.real).max() <= 1e-12 * np.abs(D).max()


def test_p8_linearity_and_chunking(oracle):
    d = _small(seed=81, n_rows=600, n_chan=2, n_pix=64, n_w=3, wavelengths=False)
    prm = _prm(oracle, d)
    uvw, vis, wt, fr = _np(d)
    G = oracle.grid(prm, uvw, vis, wt, fr)
    Gc = oracle.grid(prm, uvw[:250], vis[:250], wt[:250], fr)
    oracle.grid(prm, uvw[250:], vis[250:], wt[250:], fr, out=Gc)
    assert np.abs(G - Gc).max() <= 1e-13 * np.abs(G).max()
    G3 = oracle.grid(prm, uvw, (3.0 * vis).astype(np.complex64), wt, fr)
    assert np.abs(G3 - 3 * G).max() <= 1e-6 * np.abs(G).max()      # complex64 rounding of 3 V
    # plane ranges tile the stack
    parts = [oracle.grid(prm, uvw, vis, wt, fr, k, k + 1)[0] for k in range(3)]
    assert np.array_equal(np.stack(parts), G)


def test_wcorrect_special_values(oracle):
    """t = n - 1: zero at the phase centre, -r^2/2 for small r; pixels outside the unit circle get nothing (R14).
    Catches a wrong sign of the screen (R11) and w_k off by half a plane."""
    N, cell = 16, 0.2                 # corner r^2 = 2 * (8*0.2)^2 > 1
    prm = oracle.OracleParams(n_pix=N, n_wplanes=2, support=7, cell_rad=cell, w_min=10.0, w_max=14.0)
    P = np.ones((2, N, N), np.complex128)
    D = oracle.wcorrect(prm, P)
    c = N // 2
    assert D[c, c] == 2.0
    assert D[0, 0] == 0 and D[0, N - 1] == 0
    l = cell
    n1 = math.sqrt(1 - l * l) - 1
    ref = np.exp(2j * np.pi * 11.0 * n1) + np.exp(2j * np.pi * 13.0 * n1)     # plane midpoints 11 and 13
    assert abs(D[c, c + 1] - ref) < 1e-13 and abs(D[c + 1, c] - ref) < 1e-13
    assert D[c, c + 1].imag < 0       # n - 1 < 0 and w > 0: negative phase for the + sign of Eq. 2


def test_tiny_config_runs_in_seconds(oracle):
    """configs[0] end to end: the oracle plus its invariants on the real Tiny workload."""
    d = make_dataset(get_config("tiny"))
    prm = _prm(oracle, d)
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    c = d.n_pix // 2
    assert abs(D[c, c] - G.sum()) <= 1e-11 * abs(G.sum())
    key = oracle.positions(prm, d.uvw.numpy(), 1)["key"]
    bin_start, perm, dropped = oracle.bins(prm, key)
    assert bin_start[-1] + dropped == d.n_vis
    # the five model sources stand out of the dirty image near their positions
    peak = np.unravel_index(np.abs(D.real).argmax(), D.shape)
    dist = np.hypot((peak[1] - c) * d.cell_rad - d.src_l, (peak[0] - c) * d.cell_rad - d.src_m)
    assert dist.min() < 2 * d.cell_rad
