"""Property pins for the oracle over randomly drawn shapes (hypothesis; CPU only): whatever the support, kernel, mesh
size, plane count or frequency set-up, (i) the mass of the mesh equals the weighted visibilities times the tap sums
evaluated with scipy / numpy (north_star's invariant), (ii) degridding is the adjoint of imaging, (iii) the image is
linear in the visibilities.  None of these re-types an oracle loop."""
import math

import numpy as np
import scipy.special
from hypothesis import given, settings, strategies as st

from synth import make_random_dataset

KB = 1


def _tap(kernel, param, S):
    if kernel == KB:
        def f(x):
            y = 1.0 - (2.0 * np.asarray(x, dtype=np.float64) / S) ** 2
            return np.where(y >= 0, scipy.special.i0(param * np.sqrt(np.clip(y, 0, None))), 0.0) * param / (S * math.sinh(param))
        return f
    return lambda x: np.exp(-0.5 * (np.asarray(x, dtype=np.float64) / param) ** 2) / (param * math.sqrt(2 * math.pi))


shapes = st.tuples(st.sampled_from([1, 3, 5, 7, 9]), st.sampled_from([0, KB]), st.floats(0.6, 1.5), st.floats(2.0, 20.0),
                   st.sampled_from([32, 48, 64]), st.integers(1, 5), st.integers(1, 3), st.booleans(), st.integers(0, 10 ** 6))


@settings(max_examples=20, deadline=None)
@given(shapes)
def test_mass_adjoint_and_linearity(oracle, shape):
    S, kernel, sigma, beta, N, n_w, n_chan, metres, seed = shape
    d = make_random_dataset(seed, 40, n_chan, N, n_w, S, wavelengths=not metres, fill=1.05, w_span=25.0, cell_rad=0.4 / N,
                            unit_weights=True)
    param = beta if kernel == KB else sigma
    prm = oracle.OracleParams(n_pix=N, n_wplanes=n_w, support=S, cell_rad=d.cell_rad, w_min=d.w_min, w_max=d.w_max,
                              sigma=param, tile=16, kernel_type=kernel)
    uvw, vis, wt, fr = d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz
    pos = oracle.positions(prm, uvw, n_chan, fr)
    kept = pos["key"] != 0xFFFFFFFF
    # (i) mass
    G = oracle.grid(prm, uvw, vis, wt, fr)
    h = (S - 1) // 2
    a = np.arange(-h, h + 1)
    tap = _tap(kernel, param, S)
    Ku = tap(a[None, :] - pos["fu"][:, None]).sum(1)
    Kv = tap(a[None, :] - pos["fv"][:, None]).sum(1)
    ref = (vis.ravel().astype(np.complex128) * Ku * Kv)[kept].sum()
    assert abs(G.sum() - ref) <= 1e-11 * max(1.0, np.abs(vis).sum())
    # (ii) adjoint
    rng = np.random.default_rng(seed)
    M = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    D = oracle.dirty_image(prm, uvw, vis, wt, fr)
    pred = oracle.predict(prm, M, uvw, n_chan, fr)
    lhs, rhs = np.vdot(pred, vis.astype(np.complex128)), np.vdot(M, D)
    assert abs(lhs - rhs) <= 1e-11 * (np.linalg.norm(pred) * np.linalg.norm(vis) + 1e-30)
    # (iii) linearity
    D2 = oracle.dirty_image(prm, uvw, (2.5 - 1.5j) * vis.astype(np.complex128), wt, fr)
    assert np.abs(D2 - (2.5 - 1.5j) * D).max() <= 1e-5 * max(np.abs(D).max(), 1e-30)      # vis are rounded to complex64 on the way in
