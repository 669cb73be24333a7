"""Pins of the oracle's common-mode subtraction (Eq. 25-26): three spaxels by hand, the invariant the
step exists for (a pure-atmosphere TOD is removed exactly), the on-source limit, and the lookup-table transmission
against scipy's interpolator."""
import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

from oracle import oracle as O
from paper_2604_23305_b200 import workloads as W

ARCSEC = np.pi / 180 / 3600


def test_three_spaxels_by_hand():
    """One sample, one channel, spaxels at 0", 250", 300" with r_out = 200": S = (0, 1, 1), N_out = 2."""
    Tb = np.array([[[30.0], [20.0], [22.0]]])
    eta_z = np.array([0.8])
    csc = np.array([[1.25, 1.30, 1.35]])
    daz = np.array([0.0, 250.0, 0.0]) * ARCSEC
    de = np.array([0.0, 0.0, -300.0]) * ARCSEC
    out, S, common = O.common_mode_subtract(Tb, eta_z, csc, daz, de, 200 * ARCSEC)
    e0, e1, e2 = 0.8 ** 1.25, 0.8 ** 1.30, 0.8 ** 1.35
    cm = 20.0 / (1 - e1) + 22.0 / (1 - e2)
    assert list(S) == [0.0, 1.0, 1.0]
    assert common[0, 0] == pytest.approx(cm, rel=1e-15)
    assert out[0, 0, 0] == pytest.approx(30.0 / e0 - (1 - e0) / (e0 * 2) * cm, rel=1e-14)
    assert out[0, 1, 0] == pytest.approx(20.0 / e1 - (1 - e1) / (e1 * 2) * cm, rel=1e-14)
    # the radius test is strict (Eq. 26 ">"): a spaxel exactly on r_out is not used
    _, S2, _ = O.common_mode_subtract(Tb, eta_z, csc, np.array([0.0, 200.0, 0.0]) * ARCSEC, de, 200 * ARCSEC)
    assert list(S2) == [0.0, 0.0, 1.0]
    with pytest.raises(ValueError):
        O.common_mode_subtract(Tb, eta_z, csc, daz, de, 1000 * ARCSEC)


def test_pure_atmosphere_is_removed_and_a_source_is_recovered():
    """T_b,j = (1 - eta_j) T_atm for every spaxel (blank sky seen through the atmosphere): the common mode is T_atm and
    Eq. 25 returns 0.  A source T_src behind the atmosphere in an on-source spaxel (T_b += eta T_src) comes back as T_src."""
    rng = np.random.default_rng(3)
    n_t, n_s, n_c = 7, 9, 5
    eta_z = rng.uniform(0.3, 0.95, n_c)
    csc = rng.uniform(1.1, 1.6, (n_t, n_s))
    eta = eta_z[None, None, :] ** csc[:, :, None]
    T_atm = 265.0
    Tb = (1 - eta) * T_atm
    r = np.concatenate([[0.0, 50.0], rng.uniform(210, 400, n_s - 2)]) * ARCSEC
    ang = rng.uniform(0, 2 * np.pi, n_s)
    daz, de = r * np.cos(ang), r * np.sin(ang)
    out, S, _ = O.common_mode_subtract(Tb, eta_z, csc, daz, de, 200 * ARCSEC)
    assert S.sum() == n_s - 2
    assert np.max(np.abs(out)) < 1e-10 * T_atm
    T_src = rng.uniform(0.1, 2.0, (n_t, n_c))
    Tb2 = Tb.copy()
    Tb2[:, 0, :] += eta[:, 0, :] * T_src
    out2, _, _ = O.common_mode_subtract(Tb2, eta_z, csc, daz, de, 200 * ARCSEC)
    np.testing.assert_allclose(out2[:, 0, :], T_src, rtol=1e-10)
    assert np.max(np.abs(out2[:, 1:, :])) < 1e-10 * T_atm
    # linear in T_b
    out3, _, _ = O.common_mode_subtract(3.0 * Tb2, eta_z, csc, daz, de, 200 * ARCSEC)
    np.testing.assert_allclose(out3, 3.0 * out2, rtol=1e-12, atol=1e-9)


def test_zenith_transmission_against_scipy():
    w = W.random_workload(5, n_chan=9)
    n_pwv, n_nu = w.atm_lut.shape
    pw = w.lut_pwv0_mm + w.lut_dpwv_mm * np.arange(n_pwv)
    nu = w.lut_nu0_hz + w.lut_dnu_hz * np.arange(n_nu)
    rgi = RegularGridInterpolator((pw, nu), w.atm_lut.astype(np.float64), method="linear")
    for pwv in (pw[0], 0.5 * (pw[2] + pw[3]), pw[-1] - 1e-3):
        got = O.eta_zenith_at(w, w.f_center_hz, pwv)
        np.testing.assert_allclose(got, rgi(np.stack([np.full(9, pwv), w.f_center_hz], axis=1)), rtol=1e-13)
    # clamped outside the table (R13), nodes returned at nodes
    np.testing.assert_allclose(O.eta_zenith_at(w, nu[3:5], pw[-1] + 5.0), w.atm_lut[-1, 3:5], rtol=1e-7)
    np.testing.assert_allclose(O.eta_zenith_at(w, nu[3:5], pw[0] - 5.0), w.atm_lut[0, 3:5], rtol=1e-7)
