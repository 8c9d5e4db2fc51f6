"""Pins for the oracle's degridding chain (CPU only).

Degridding with unit weights is the adjoint of the imaging chain that tests/test_oracle_pins.py pins, and for point
sources on pixel centres it must reproduce Eq. 1 evaluated directly -- neither check re-types the
oracle's loops.
"""
import math

import numpy as np
import pytest
import scipy.special

from tests.test_oracle_pins import _np, _prm, _small, _independent_positions

KB = 1


def _kb_beta(S, alpha=2.0):
    return math.pi * math.sqrt((S / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8)


def test_forward_transform_is_numpy_fft2(oracle):
    rng = np.random.default_rng(3)
    for N in (8, 12, 64, 1024):
        x = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        ref = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(x)))
        got = oracle.transform_fwd(x)
        assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max(), N


@pytest.mark.parametrize("kernel", ["gaussian", "kaiser_bessel"])
def test_degridding_is_the_adjoint_of_imaging(oracle, kernel):
    """<predict(M), y> = <M, image(y)> for random complex M and y (unit weights), to rounding.
    Catches any sign, index, conjugation, screen or tap mistake in the degridding chain: the imaging side is pinned."""
    d = _small(seed=81, n_rows=400, n_chan=2, n_pix=64, n_w=5, wavelengths=False, fill=1.04, w_span=40.0, cell_rad=7e-3,
               unit_weights=True)
    prm = _prm(oracle, d)
    if kernel == "kaiser_bessel":
        prm.kernel_type, prm.sigma = KB, _kb_beta(7)
    rng = np.random.default_rng(5)
    M = rng.standard_normal((64, 64)) + 1j * rng.standard_normal((64, 64))
    uvw, y, wt, fr = _np(d)
    pred = oracle.predict(prm, M, uvw, d.n_chan, fr)
    D = oracle.dirty_image(prm, uvw, y, wt, fr)
    # pixels outside the unit circle take no part on either side (R14)
    x = (np.arange(64) - 32) * d.cell_rad
    inside = (x[None, :] ** 2 + x[:, None] ** 2) < 1
    lhs = np.vdot(pred, y.astype(np.complex128))
    rhs = np.vdot(M[inside], D[inside])
    assert abs(lhs - rhs) <= 1e-12 * abs(rhs), (lhs, rhs)
    # the FFT route gives the same prediction; dropped visibilities predict exactly 0
    pred2 = oracle.predict(prm, M, uvw, d.n_chan, fr, naive_max=0)
    assert np.abs(pred2 - pred).max() <= 1e-11 * np.abs(pred).max()
    key = oracle.positions(prm, uvw, d.n_chan, fr)["key"].reshape(pred.shape)
    assert (key == 0xFFFFFFFF).any() and not np.any(pred[key == 0xFFFFFFFF]) and np.all(pred[key != 0xFFFFFFFF] != 0)


@pytest.mark.parametrize("kernel,tol", [("kaiser_bessel", 2e-6), ("gaussian", 5e-3)])
def test_predicted_visibilities_of_point_sources_equal_eq1(oracle, kernel, tol):
    """Sources on pixel centres of the inner half, model = flux / (ghat ghat) there: the prediction must equal
    V = sum_s F_s exp(-2 pi i (u l_s + v m_s + w_k (n_s - 1))) (Eq. 1 without 1/n, w snapped to the plane midpoints).
    Independent of the imaging chain: numpy + scipy only on the reference side."""
    d = _small(seed=83, n_rows=600, n_pix=64, n_w=8, fill=0.85, w_span=60.0, cell_rad=4e-3)
    prm = _prm(oracle, d)
    beta = _kb_beta(7)
    N = d.n_pix
    xi = lambda i: (i - N // 2) / N
    if kernel == "kaiser_bessel":
        prm.kernel_type, prm.sigma = KB, beta
        def ghat(x):
            r = np.sqrt(beta ** 2 - (math.pi * 7 * x) ** 2)
            return beta / math.sinh(beta) * np.sinh(r) / r
    else:
        ghat = lambda x: np.exp(-2 * math.pi ** 2 * d.sigma_cells ** 2 * x ** 2)
    src = [(40, 25, 1.0), (22, 44, 0.6), (33, 30, 0.3)]            # (q, p, flux): asymmetric
    M = np.zeros((N, N), np.complex128)
    for q, p, f in src:
        M[q, p] = f / (ghat(xi(p)) * ghat(xi(q)))
    uvw = d.uvw.numpy()
    pred = oracle.predict(prm, M, uvw, 1)[:, 0]
    k = oracle.positions(prm, uvw, 1)["k"]
    dw = (d.w_max - d.w_min) / d.n_wplanes
    wk = d.w_min + (k + 0.5) * dw
    u64 = uvw.astype(np.float64)
    ref = np.zeros(len(u64), np.complex128)
    for q, p, f in src:
        l, m = (p - N // 2) * d.cell_rad, (q - N // 2) * d.cell_rad
        ref += f * np.exp(-2j * np.pi * (u64[:, 0] * l + u64[:, 1] * m + wk * (math.sqrt(1 - l * l - m * m) - 1)))
    err = np.abs(pred - ref).max() / sum(f for _, _, f in src)
    assert err < tol, err


def test_predict_samples_equal_the_chain(oracle):
    """The sampled, re-ordered form used at full size against the plane-by-plane chain, both kernels, with drops."""
    d = _small(seed=85, n_rows=300, n_chan=3, n_pix=128, n_w=6, wavelengths=False, fill=1.04, w_span=30.0, cell_rad=0.012)
    rng = np.random.default_rng(2)
    N = d.n_pix
    sq, sp = rng.integers(0, N, 25), rng.integers(0, N, 25)
    sq[:2], sp[:2] = [0, 64], [0, 64]                     # a corner outside the unit circle (ignored), the centre
    val = rng.standard_normal(25) + 1j * rng.standard_normal(25)
    M = np.zeros((N, N), np.complex128)
    np.add.at(M, (sq, sp), val)
    for kt, par in ((0, 1.0), (KB, _kb_beta(7))):
        prm = _prm(oracle, d, kernel_type=kt)
        prm.sigma = par
        full = oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz).ravel()
        samp = rng.choice(full.size, 200, replace=False)
        # duplicate source pixels add up in M: give predict_samples the same list
        got = oracle.predict_samples(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz, sq, sp, val, samp)
        assert np.abs(got - full[samp]).max() <= 1e-11 * np.abs(full).max()
        assert (0.012 * 64) ** 2 * 2 >= 1 and np.any(full[samp] == 0)      # the corner is outside; some samples are dropped
