"""Pins of the oracle's screen pre-processing: Eq. 4 and the aperture-footprint smoothing (R24)."""
import numpy as np
from scipy import ndimage

from oracle import oracle as O


def test_footprint_weights_by_hand():
    K = O.footprint_weights(1.0, 1.0, 2.5, -10.0)
    assert K.shape == (5, 5) and np.isclose(K.sum(), 1.0)
    # corners (r^2 = 8 >= 6.25) lie outside the aperture, (2, 1) (r^2 = 5) inside
    assert K[0, 0] == 0 and K[4, 4] == 0 and K[0, 1] > 0
    # Gaussian: 10 dB down in amplitude at the rim means a factor 10^(-0.5 r^2 / R^2)
    assert np.isclose(K[2, 3] / K[2, 2], 10 ** (-0.5 * 1.0 / 6.25))
    assert np.isclose(K[0, 1] / K[2, 2], 10 ** (-0.5 * 5.0 / 6.25))
    assert np.allclose(K, K[::-1, :]) and np.allclose(K, K[:, ::-1]) and np.allclose(K, K.T)
    # no taper: a uniform disc; anisotropic grid: radii follow R / dx and R / dy
    K0 = O.footprint_weights(1.0, 1.0, 2.5, 0.0)
    assert np.allclose(K0[K0 > 0], 1.0 / 21.0)
    assert O.footprint_weights(0.5, 2.0, 2.5, -10.0).shape == (3, 11)
    # r = R_tel itself is outside (strict inequality of Eq. 2)
    assert O.footprint_weights(1.0, 1.0, 2.0, -10.0)[2, 0] == 0


def test_smoothing_against_scipy_and_invariants():
    rng = np.random.default_rng(0)
    epl = rng.normal(0.0, 0.3, (37, 53))
    got = O.screen_line_of_sight(epl, 0.7, 0.9, 3.0, -11.0, 1.2)
    K = O.footprint_weights(0.7, 0.9, 3.0, -11.0)
    want = 1.2 + ndimage.correlate(epl, K, mode="wrap") / 6.587
    assert np.allclose(got, want, rtol=0, atol=1e-13)
    # unit-sum kernel: the mean is kept, a flat screen stays flat, fluctuations shrink
    assert np.isclose(got.mean(), 1.2 + epl.mean() / 6.587, atol=1e-13)
    assert np.allclose(O.screen_line_of_sight(np.full((8, 9), 2.0), 0.7, 0.9, 3.0, -11.0, 0.5), 0.5 + 2.0 / 6.587)
    assert got.std() < epl.std() / 6.587
    # an aperture smaller than a pixel leaves Eq. 4 alone
    assert np.allclose(O.screen_line_of_sight(epl, 0.7, 0.9, 0.5, -11.0, 1.2), 1.2 + epl / 6.587)
    # a single spike returns the (flipped = same, symmetric) kernel, wrapped around the edges
    spike = np.zeros((16, 16)); spike[0, 0] = 6.587
    out = O.screen_line_of_sight(spike, 1.0, 1.0, 2.5, -10.0, 0.0)
    Kk = O.footprint_weights(1.0, 1.0, 2.5, -10.0)
    assert np.isclose(out[0, 0], Kk[2, 2]) and np.isclose(out[15, 1], Kk[1, 3]) and np.isclose(out[2, 14], Kk[4, 0] if Kk[4, 0] else 0.0)
