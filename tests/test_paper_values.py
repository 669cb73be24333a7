"""Pins of the input generators (workloads.py) to the values the paper prints; the fixture
tests/golden/paper_values.txt carries one citation per value."""
from pathlib import Path

import numpy as np
import pytest

from paper_2604_23305_b200 import workloads as W

GOLD = {}
for line in (Path(__file__).parent / "golden" / "paper_values.txt").read_text().splitlines():
    if line.strip() and not line.startswith("#"):
        name, value, tol, cite = [x.strip() for x in line.split("|")]
        GOLD[name] = (float(value), float(tol), cite)


def check(name, got):
    want, tol, cite = GOLD[name]
    assert abs(got - want) <= tol * abs(want) + 1e-300, f"{name}: got {got}, paper prints {want} ({cite})"


def test_fixture_is_complete_and_cited():
    assert len(GOLD) == 12 and all("PAPER.md:" in c for _, _, c in GOLD.values())


def test_readout_rate_and_constants():
    check("f_sample_hz", W.F_SAMPLE_DESHIMA)
    check("kid_cutoff_ghz", 2 * 188e-6 * 1.602176634e-19 / W.H_PLANCK / 1e9)


def test_hexagon_and_channel_count():
    daz, de = W.hex_spaxels(3, 8 * W.ARCSEC)
    check("hex_spaxels_R3", daz.size)
    assert [W.hex_spaxels(r, 1.0)[0].size for r in (0, 1, 4)] == [1, 7, 61]          # 1 + 3R(R+1): the configs' counts
    check("channels_90_180_R20", W.channel_count_half_power(90e9, 180e9, 20))
    assert W.channel_count_half_power(220e9, 440e9, 500) == 347                        # BASELINE.json configs
    # nearest neighbours of the packed hexagon are one pitch apart
    d = np.hypot(daz[:, None] - daz[None, :], de[:, None] - de[None, :])
    np.fill_diagonal(d, np.inf)
    assert np.allclose(d.min(axis=1), 8 * W.ARCSEC, rtol=1e-12)


def test_cascade_helpers():
    check("ohmic_loss_at_840ghz", 1.0 - float(W.eta_ohmic(np.array([840e9]))[0]))
    check("surface_eta_n3p41", W.eta_dielectric_surface(3.41))
    # Eq. 14 has no loss for tan(delta) = 0 and Eq. 13 scales as sqrt(nu)
    assert np.all(W.eta_dielectric_bulk(np.array([3e11]), 4e-3, 3.41, 0.0) == 1.0)
    assert np.isclose((1 - W.eta_ohmic(np.array([210e9]))[0]) / 0.0025, 0.5)


def test_daisy_scan_closed_form_and_bounds():
    r, om, ratio = GOLD["daisy_r_arcsec"][0], GOLD["daisy_omega_hz"][0], GOLD["daisy_Omega_ratio"][0]
    az, el = W.scan_daisy(4000, 160.0)
    t = np.arange(4000) / 160.0
    w, Wm = 2 * np.pi * om, 2 * np.pi * om / ratio
    assert np.allclose(az, r * W.ARCSEC * np.cos(Wm * t) * np.sin(w * t), rtol=0, atol=1e-18)     # Eq. 8 :129-133
    assert np.allclose(el, r * W.ARCSEC * np.sin(Wm * t) * np.sin(w * t), rtol=0, atol=1e-18)
    assert np.hypot(az, el).max() <= r * W.ARCSEC * (1 + 1e-12)


def test_filterbank_peak_and_front_end_constants():
    nu = np.array([300e9])
    check("eta_peak_filter", float(W.lorentzian_filterbank(nu, nu, 500)[0, 0]))
    # half power at nu = f (1 +- 1/(2R)) (FWHM = f/R, reading R1)
    half = W.lorentzian_filterbank(np.array([300e9 * (1 + 1 / 1000)]), nu, 500)[0, 0]
    assert np.isclose(half, 0.08, rtol=1e-6)
    w = W.make_workload("C2", n_samples=16)
    check("t_cmb_K", w.T_cmb_K)
    ef = W.eta_front_aste(np.array([1e9]))[0]                                                      # Ruze term -> 1 at low nu
    assert np.isclose(ef / 0.85, GOLD["eta_pol"][0], rtol=1e-5)          # the Ruze factor at 1 GHz is 1 - 3e-6


def test_filterbank_with_upstream_absorption_eq7():
    """Eq. 7 against its closed form: with a common peak height the recursion telescopes to
    eta_k = eta_peak L_k prod_{f_j > f_k} (1 - L_j), L = 1 / (1 + 4 R^2 (nu/f - 1)^2)."""
    nu = np.linspace(200e9, 460e9, 1500)
    fc = W.channel_centres_log(40)
    R, pk = 300.0, 0.16
    got = W.filterbank_upstream_absorption(nu, fc, R, pk).astype(np.float64)
    L = 1.0 / (1.0 + 4.0 * R * R * (nu[None, :] / fc[:, None] - 1.0) ** 2)
    want = np.empty_like(L)
    for k in range(fc.size):
        up = fc > fc[k]
        want[k] = pk * L[k] * np.prod(1.0 - L[up], axis=0)
    assert np.allclose(got, want, rtol=2e-6, atol=1e-12)
    # the highest-frequency channel is fed first: it is the isolated Lorentzian of Eq. 6
    top = np.argmax(fc)
    assert np.allclose(got[top], W.lorentzian_filterbank(nu, fc[top:top + 1], R, pk)[0], rtol=1e-6)
    # no frequency is absorbed more than once: the total never exceeds the peak height, and every downstream
    # channel is below its isolated Lorentzian
    assert np.all(got.sum(axis=0) <= pk * (1 + 1e-6))
    assert np.all(got <= W.lorentzian_filterbank(nu, fc, R, pk).astype(np.float64) * (1 + 1e-6) + 1e-12)
    # row order follows f_c_hz whatever its order
    perm = np.random.default_rng(0).permutation(fc.size)
    assert np.array_equal(W.filterbank_upstream_absorption(nu, fc[perm], R, pk), W.filterbank_upstream_absorption(nu, fc, R, pk)[perm])
