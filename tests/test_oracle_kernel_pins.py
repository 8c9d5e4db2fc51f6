"""Pins for the oracle's convolution functions and image normalisation (CPU only).

Nothing here re-types the oracle's formulae: Bessel functions come from scipy / numpy, integrals from
scipy.integrate.quad, and the calibrated image is checked against north_star's brute-force direct DFT.
"""
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.special

from tests.test_oracle_pins import _closed_form_image, _direct_dft, _model_dataset, _np, _prm, _small, _independent_positions

KB = 1


def _kb_beta(S, alpha=2.0):
    """Shape parameter for a window of S cells and an image that is cropped to 1/alpha of the field (Beatty et al.)."""
    return math.pi * math.sqrt((S / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8)


def _kb_scipy(x, S, beta):
    y = 1.0 - (2.0 * np.asarray(x, dtype=np.float64) / S) ** 2
    return np.where(y >= 0, scipy.special.i0(beta * np.sqrt(np.clip(y, 0, None))), 0.0) * beta / (S * math.sinh(beta))


def test_i0_matches_scipy_and_numpy(oracle):
    """Catches a wrong series (x/2 vs x^2/4, k! vs (k!)^2) or an early truncation."""
    for x in [0.0, 1e-3, 0.5, 1.0, 3.75, 7.0, 12.0, 16.25, 21.0, 30.0]:
        ref = float(scipy.special.i0(x))
        assert abs(oracle.i0(x) - ref) <= 4e-15 * ref, x
        assert abs(oracle.i0(x) - float(np.i0(x))) <= 1e-12 * ref, x


@pytest.mark.parametrize("S,beta", [(7, _kb_beta(7)), (9, _kb_beta(9)), (5, 4.0), (3, 2.5)])
def test_kaiser_bessel_is_numpy_kaiser_window_with_unit_integral(oracle, S, beta):
    """Shape = numpy.kaiser (library routine) resampled on [-S/2, S/2]; integral = 1; zero outside; even.
    Catches a wrong width (S vs S/2), a missing square root, a wrong normalisation."""
    prm = oracle.OracleParams(n_pix=64, n_wplanes=1, support=S, cell_rad=1e-3, w_min=-1, w_max=1, sigma=beta, kernel_type=KB)
    M = 41
    win = np.kaiser(M, beta)
    xs = (np.arange(M) - (M - 1) / 2) * S / (M - 1)
    g = np.array([oracle.kernel1d(prm, x) for x in xs])
    assert np.abs(g / oracle.kernel1d(prm, 0.0) - win).max() < 1e-12
    integral, _ = scipy.integrate.quad(lambda x: oracle.kernel1d(prm, x), -S / 2, S / 2, epsabs=1e-13, epsrel=1e-13)
    assert abs(integral - 1.0) < 1e-10
    assert oracle.kernel1d(prm, S / 2 + 1e-9) == 0.0 and oracle.kernel1d(prm, -S / 2 - 1e-9) == 0.0
    assert oracle.kernel1d(prm, 1.3) == oracle.kernel1d(prm, -1.3)
    assert abs(oracle.kernel1d(prm, 0.7) - float(_kb_scipy(0.7, S, beta))) < 1e-14


@pytest.mark.parametrize("S,beta", [(7, _kb_beta(7)), (5, 4.0), (3, 1.5)])
def test_kaiser_bessel_taper_is_the_fourier_integral_of_the_kernel(oracle, S, beta):
    """ghat(xi) = int g(x) cos(2 pi x xi) dx by quadrature of the oracle's own g, on both branches
    (pi S xi below and above beta).  Catches a wrong argument scale, a missing 1/sinh, a wrong continuation."""
    prm = oracle.OracleParams(n_pix=64, n_wplanes=1, support=S, cell_rad=1e-3, w_min=-1, w_max=1, sigma=beta, kernel_type=KB)
    seen_upper = False
    for xi in [0.0, 0.05, 0.2, 0.35, 0.5, beta / (math.pi * S), 0.9, 1.7]:
        num, _ = scipy.integrate.quad(lambda x: oracle.kernel1d(prm, x) * math.cos(2 * math.pi * x * xi), -S / 2, S / 2,
                                      epsabs=1e-13, epsrel=1e-12, limit=400)
        assert abs(oracle.taper1d(prm, xi) - num) < 2e-10, (xi, oracle.taper1d(prm, xi), num)
        seen_upper |= math.pi * S * xi > beta
    assert seen_upper


def test_gaussian_taper_is_the_fourier_integral_of_the_kernel(oracle):
    for sigma in (1.0, 0.7):
        prm = oracle.OracleParams(n_pix=64, n_wplanes=1, support=7, cell_rad=1e-3, w_min=-1, w_max=1, sigma=sigma)
        for xi in (0.0, 0.1, 0.25, 0.5):
            num, _ = scipy.integrate.quad(lambda x: oracle.kernel1d(prm, x) * math.cos(2 * math.pi * x * xi), -12, 12,
                                          epsabs=1e-13, epsrel=1e-12, limit=400)
            assert abs(oracle.taper1d(prm, xi) - num) < 1e-10


def test_p1_closed_form_whole_chain_kaiser_bessel(oracle):
    """The per-visibility closed form of the chain (no mesh, no DFT) with scipy's I0 as the tap function."""
    d = _small(seed=43, n_rows=50, n_chan=2, n_pix=64, n_w=4, wavelengths=False, fill=1.0, w_span=40.0, cell_rad=6e-3)
    beta = _kb_beta(7)
    prm = _prm(oracle, d, kernel_type=KB)
    prm.sigma = beta
    D = oracle.dirty_image(prm, *_np(d))
    ref = _closed_form_image(d, tap=lambda x: _kb_scipy(x, 7, beta))
    assert np.linalg.norm(D - ref) / np.linalg.norm(ref) < 1e-12
    s = oracle.image_samples(prm, *_np(d), [5, 32, 60], [40, 32, 3])
    assert np.abs(s - D[[5, 32, 60], [40, 32, 3]]).max() <= 1e-11 * np.abs(D).max()


def test_sum_weights_counts_kept_visibilities_only(oracle):
    d = _small(seed=44, n_rows=400, n_chan=3, n_pix=64, n_w=4, wavelengths=False, fill=1.15)   # some fall off the mesh
    prm = _prm(oracle, d)
    pu, pv, _ = _independent_positions(d, d.n_chan)
    h, N = 3, d.n_pix
    i0, j0 = np.floor(pu + 0.5), np.floor(pv + 0.5)
    keep = (i0 >= h) & (i0 <= N - 1 - h) & (j0 >= h) & (j0 <= N - 1 - h)
    assert 0 < keep.sum() < keep.size
    ref = d.weights.numpy().ravel().astype(np.float64)[keep].sum()
    assert abs(oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy(), d.freqs_hz) - ref) < 1e-9 * ref


@pytest.mark.parametrize("kernel", ["kaiser_bessel", "gaussian"])
def test_p2_calibrated_image_equals_the_direct_dft(oracle, kernel):
    """All normalisation flags on: dirty = Re D n / (sum_wt ghat ghat) against n Re(I) / sum_wt with I the
    brute-force direct DFT (w snapped to the plane midpoints), inner half of the field.  With the Kaiser-Bessel
    window the two agree to 1e-7 of the peak (measured 1.1e-7; SURVEY 8(f) NEXT-1 asks for 1e-4); the Gaussian of PAPER.md:82 only to a few
    1e-3 ("high aliasing response").  Catches a wrong taper, xi scale, a missing n or weight sum."""
    d, _ = _model_dataset(n_w=8)
    prm = _prm(oracle, d)
    if kernel == "kaiser_bessel":
        prm.kernel_type, prm.sigma = KB, _kb_beta(7)
    D = oracle.dirty_image(prm, *_np(d))
    k = oracle.positions(prm, d.uvw.numpy(), 1)["k"]
    dw = (d.w_max - d.w_min) / d.n_wplanes
    I = _direct_dft(d, d.w_min + (k + 0.5) * dw)
    sw = oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy())
    N = d.n_pix
    x = (np.arange(N) - N // 2) * d.cell_rad
    n = np.sqrt(1 - x[None, :] ** 2 - x[:, None] ** 2)
    ref = n * I.real / sw
    out = oracle.dirty(prm, D, oracle.NORM_SUMWT | oracle.NORM_N | oracle.NORM_TAPER, sw)
    inner = slice(N // 4, 3 * N // 4)
    err = np.abs(out[inner, inner] - ref[inner, inner]).max() / np.abs(ref).max()
    assert err < (2e-6 if kernel == "kaiser_bessel" else 5e-3), err
    # each flag is one factor: exact relations between the partially normalised images
    d0 = oracle.dirty(prm, D, 0)
    assert np.array_equal(d0, D.real)
    assert np.allclose(oracle.dirty(prm, D, oracle.NORM_SUMWT, sw) * sw, d0, rtol=1e-14, atol=0)
    assert np.allclose(oracle.dirty(prm, D, oracle.NORM_N), d0 * n, rtol=1e-14, atol=0)
    tap = oracle.dirty(prm, D, oracle.NORM_TAPER)
    assert np.abs(tap[inner, inner] - I.real[inner, inner]).max() / np.abs(I).max() < (2e-6 if kernel == "kaiser_bessel" else 5e-3)
