"""Pins of the oracle's source pre-processing: far field (Eq. 2-3) and beam convolution (Eq. 1), R25."""
import numpy as np
from scipy import ndimage, special

from oracle import oracle as O

ARCSEC = np.pi / 180 / 3600


def test_uniform_aperture_gives_the_airy_pattern():
    nu, R = 350e9, 5.0
    lam = 299792458.0 / nu
    rho = np.array([0.0, 3.0, 7.5, 12.0, 21.0, 40.0]) * ARCSEC
    x = 2 * np.pi * R * rho / lam
    airy = np.ones_like(x)
    airy[1:] = (2 * special.j1(x[1:]) / x[1:]) ** 2
    assert np.allclose(O.far_field(rho, nu, R, 0.0), airy, rtol=1e-9, atol=1e-14)
    # first null of the Airy disc at 1.2197 lambda / D
    assert O.far_field([1.2197 * lam / (2 * R)], nu, R, 0.0)[0] < 1e-8


def test_strong_taper_tends_to_the_gaussian_beam():
    """With the rim 100 dB down the truncation does not matter: A = exp(-k r^2) transforms to exp(-(pi rho / lambda)^2 / k),
    squared for power."""
    nu, R, t = 300e9, 5.0, -100.0
    lam = 299792458.0 / nu
    k = 100.0 / 20.0 * np.log(10.0) / R ** 2
    rho = np.array([0.0, 5.0, 10.0, 20.0]) * ARCSEC
    want = np.exp(-2 * (np.pi * rho / lam) ** 2 / k)
    assert np.allclose(O.far_field(rho, nu, R, t), want, rtol=1e-4)
    # taper broadens the main lobe: -10 dB is wider than uniform at the uniform half-power point
    hp = 0.5145 * lam / (2 * R)
    assert O.far_field([hp], nu, R, -10.0)[0] > O.far_field([hp], nu, R, 0.0)[0] > 0.49


def test_convolution_against_scipy_and_point_source():
    rng = np.random.default_rng(2)
    n_el, n_az, r = 9, 11, 3
    nu = np.array([250e9, 400e9])
    d = 6.0 * ARCSEC
    I = rng.random((n_el, n_az, 2))
    el_first = np.deg2rad(60.0)
    got = O.source_power(I, nu, d, 1.5 * d, el_first, r, 5.0, -10.0)
    for f in range(2):
        W = O.beam_weights(nu[f], d, 1.5 * d, r, 5.0, -10.0)
        src = I[:, :, f] * np.cos(el_first + 1.5 * d * np.arange(n_el))[:, None]
        want = np.pi * 25.0 * d * 1.5 * d * ndimage.convolve(src, W, mode="constant", cval=0.0)
        assert np.allclose(got[:, :, f], want, rtol=1e-12)
        assert W[r, r] == 1.0 and np.allclose(W, W[::-1]) and np.allclose(W, W[:, ::-1])
    # a point source returns the beam, scaled by A_p cos(theta) dOmega
    P = np.zeros((n_el, n_az, 1)); P[4, 5, 0] = 2.0
    out = O.source_power(P, nu[:1], d, d, 0.3, r, 5.0, -10.0)[:, :, 0]
    W = O.beam_weights(nu[0], d, d, r, 5.0, -10.0)
    assert np.allclose(out[1:8, 2:9], 2.0 * np.pi * 25.0 * d * d * np.cos(0.3 + 4 * d) * W, rtol=1e-12)
    assert out[0, 0] == 0
