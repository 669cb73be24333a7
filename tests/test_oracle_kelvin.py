"""Pins of the oracle's brightness-temperature output (R22): the simulated skydip and the
per-channel linear map T_b = a + b P_KID."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2604_23305_b200 import workloads as W

H, KB = 6.62607015e-34, 1.380649e-23


def _w(seed=3, **kw):
    w = W.random_workload(seed, n_samples=8, n_spaxel=2, n_chan=10, n_freq=64, **kw)
    return w.replace(output_unit=1, skydip_n=9, skydip_pwv_lo_mm=0.4, skydip_pwv_hi_mm=1.6)


def test_skydip_sweep_is_even_in_pwv_and_brightens():
    w = _w()
    P, T, pwv = O.Oracle(w).skydip()
    assert P.shape == T.shape == (9, w.n_chan)
    assert np.allclose(pwv, np.linspace(0.4, 1.6, 9), rtol=0, atol=1e-12)
    # more water: a warmer line of sight and (T_atm > T_cmb) more power on every detector
    assert np.all(np.diff(T, axis=0) > 0) and np.all(np.diff(P, axis=0) > 0)
    assert np.all(T > w.T_cmb_K) and np.all(T < w.T_atm_K)


def test_map_is_the_least_squares_line():
    """Against numpy.polyfit (a library routine) and the normal equations."""
    o = O.Oracle(_w(5))
    P, T, _ = o.skydip()
    a, b = o.kelvin_map()
    for c in range(P.shape[1]):
        s = P[:, c].mean()
        b1, a1 = np.polyfit(P[:, c] / s, T[:, c], 1)
        assert np.isclose(b[c] * s, b1, rtol=1e-9) and np.isclose(a[c], a1, rtol=1e-8, atol=1e-9 * T.max())
    r = a + b * P - T
    assert np.all(np.abs(r.sum(axis=0)) < 1e-9 * np.abs(T).sum(axis=0))
    assert np.all(np.abs((r * P).sum(axis=0)) < 1e-9 * np.abs(T * P).sum(axis=0))
    assert np.all(b > 0)
    # the map is nearly linear over a skydip: residual far below the span of T_b
    assert np.max(np.abs(r)) < 0.02 * (T.max() - T.min())


def test_single_frequency_channels_closed_form():
    """No optics, no CMB, one frequency per channel: P_KID = dnu Fm (1 - eta) B(nu, T_atm) and T_b = (1 - eta) T_atm
    are proportional, so a = 0 and b = T_atm / (dnu Fm B(nu, T_atm)) exactly."""
    w = _w(7)
    idx = np.array([3, 17, 40, 63])
    filt = np.zeros((4, w.n_freq), dtype=np.float32)
    filt[np.arange(4), idx] = np.float32([0.1, 0.2, 0.05, 0.3])
    w = w.replace(stages=[], eta_front_nu=None, T_cmb_K=0.0, filt=filt, f_center_hz=w.nu_hz[idx], dnu_eff_hz=None)
    a, b = O.Oracle(w).kelvin_map()
    nu = w.nu_hz[idx]
    B_atm = H * nu / np.expm1(H * nu / (KB * w.T_atm_K))
    want_b = w.T_atm_K / (w.dnu_hz * filt[np.arange(4), idx].astype(np.float64) * B_atm)
    assert np.allclose(b, want_b, rtol=1e-9)
    assert np.all(np.abs(a) < 1e-9 * w.T_atm_K)


def test_T_b_from_the_lookup_table_by_hand():
    """PWV values on LUT rows: eta_z is the LUT row interpolated in frequency (numpy.interp), raised to the
    airmass; T_b is its filter-weighted mean temperature."""
    w = _w(9)
    n_pwv = np.asarray(w.atm_lut).shape[0]
    lo, hi = w.lut_pwv0_mm, w.lut_pwv0_mm + w.lut_dpwv_mm * (n_pwv - 1)
    w = w.replace(skydip_n=n_pwv, skydip_pwv_lo_mm=lo, skydip_pwv_hi_mm=hi)
    _, T, pwv = O.Oracle(w).skydip()
    nu_lut = w.lut_nu0_hz + w.lut_dnu_hz * np.arange(np.asarray(w.atm_lut).shape[1])
    F = np.asarray(w.filt, dtype=np.float64)
    for k in range(n_pwv):
        eta_z = np.interp(w.nu_hz, nu_lut, np.asarray(w.atm_lut, dtype=np.float64)[k])
        eta = eta_z ** (1.0 / np.sin(w.el0_rad))
        want = F @ ((1 - eta) * w.T_atm_K + eta * w.T_cmb_K) / F.sum(axis=1)
        assert np.allclose(T[k], want, rtol=1e-9)
