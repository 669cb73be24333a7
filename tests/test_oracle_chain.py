"""Pins for the oracle's signal chain (steps 0-6a): physical invariants, closed forms,
library interpolators and an independent literal NumPy transcription of Eqs. 9-12, 16.

Each test is chosen so that a plausible mistake (a dropped term, a wrong sign or index, a
transposed operand) fails at least one of them.
"""
import math

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator
from scipy.ndimage import map_coordinates

from oracle import oracle as O
from paper_2604_23305_b200 import workloads as W

H, KB = 6.62607015e-34, 1.380649e-23
ARCSEC = W.ARCSEC


def B(nu, T):
    nu = np.asarray(nu, dtype=np.float64)
    return np.zeros_like(nu) if T <= 0 else H * nu / np.expm1(H * nu / (KB * T))


# --------------------------------------------------------------------------------------
# third implementation: literal NumPy float64 transcription straight from the paper
# --------------------------------------------------------------------------------------
def numpy_chain(w, n, s):
    """Eqs. 9-12 and 16 for one row, written directly from PAPER.md with literal tan/sin
    of the summed angles (not the addition formulas the oracle uses)."""
    nu = w.nu_hz
    t = n / w.f_sample_hz
    a, e = w.az_rad[n] + w.daz_rad[s], w.el_rad[n] + w.del_rad[s]
    ny, nx = w.screen.shape
    x = w.h_column_m * math.tan(a) + w.wind_mps * t                      # Eq. 9
    y = w.h_column_m * math.tan(e)
    u, v = x / w.dx_m + nx / 2, y / w.dy_m + ny / 2
    iu, iv = math.floor(u), math.floor(v)
    fu, fv = u - iu, v - iv
    scr = w.screen.astype(np.float64)
    g = lambda j, i: scr[j % ny, i % nx]
    pwv = ((1 - fv) * ((1 - fu) * g(iv, iu) + fu * g(iv, iu + 1))
           + fv * ((1 - fu) * g(iv + 1, iu) + fu * g(iv + 1, iu + 1))) + w.pwv0_a_mm + w.pwv0_b_mm_per_s * t
    # LUT bilinear in (pwv, nu) via scipy on the LUT's own grid, PWV clamped
    n_pwv, n_nl = w.atm_lut.shape
    pg = w.lut_pwv0_mm + w.lut_dpwv_mm * np.arange(n_pwv)
    ng = w.lut_nu0_hz + w.lut_dnu_hz * np.arange(n_nl)
    lut = RegularGridInterpolator((pg, ng), w.atm_lut.astype(np.float64), method="linear")
    eta_z = lut(np.stack([np.full_like(nu, min(max(pwv, pg[0]), pg[-1])), nu], axis=1))
    eta_atm = eta_z ** (1.0 / math.sin(w.el0_rad + e))                   # Eq. 10
    # source
    S = np.zeros_like(nu)
    if w.cube is not None:
        n_el, n_az, _ = w.cube.shape
        ag = w.az_min_rad + w.daz_grid_rad * np.arange(n_az)
        eg = w.el_min_rad + w.del_grid_rad * np.arange(n_el)
        us, vs = (a - ag[0]) / w.daz_grid_rad, (e - eg[0]) / w.del_grid_rad
        if 0 <= us <= n_az - 1 and 0 <= vs <= n_el - 1:
            ju, jv = min(math.floor(us), n_az - 2), min(math.floor(vs), n_el - 2)
            gu, gv = us - ju, vs - jv
            c = w.cube.astype(np.float64)
            S = ((1 - gv) * ((1 - gu) * c[jv, ju] + gu * c[jv, ju + 1])
                 + gv * ((1 - gu) * c[jv + 1, ju] + gu * c[jv + 1, ju + 1]))
    front = 1.0 if w.eta_front_nu is None else w.eta_front_nu.astype(np.float64)
    P = front * S + B(nu, w.T_cmb_K)                                     # Eq. 11
    P = eta_atm * P + (1 - eta_atm) * B(nu, w.T_atm_K)                   # Eq. 12, k = 0
    for st in w.stages:                                                  # Eq. 12, k >= 1
        eta = np.asarray(st.eta, dtype=np.float64)
        J = ((1 - eta_atm) * B(nu, w.T_atm_K) + eta_atm * B(nu, w.T_cmb_K)) if st.couple_atmosphere \
            else B(nu, st.T_K)
        P = eta * P + (1 - eta) * J
    pk = w.dnu_hz * (w.filt.astype(np.float64) @ P)                      # Eq. 16
    return dict(pwv=pwv, eta_atm=eta_atm, S=S, P=P, pkid=pk, fu=fu, fv=fv, iu=iu % nx, iv=iv % ny)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_end_to_end_vs_literal_numpy_transcription(seed):
    w = W.random_workload(seed, n_samples=24, n_spaxel=3, n_chan=7, n_freq=33)
    o = O.Oracle(w)
    r = o.simulate(want=("pkid", "pwv"))
    geo = o.geometry()
    inside = 0
    for n in range(w.n_samples):
        for s in range(w.n_spaxel):
            ref = numpy_chain(w, n, s)
            np.testing.assert_allclose(r["pkid"][n, s], ref["pkid"], rtol=2e-12)
            assert r["pwv"][n, s] == pytest.approx(ref["pwv"], rel=1e-12)
            # canonical (addition-formula) geometry agrees with the literal tan/sin
            assert (geo[n, s]["iu0"], geo[n, s]["iv0"]) == (ref["iu"], ref["iv"])
            assert geo[n, s]["fu"] == pytest.approx(ref["fu"], abs=1e-8)
            inside += geo[n, s]["ju"] >= 0
            P, eta, S = o.row_spectrum(n, s, intermediates=True)
            np.testing.assert_allclose(P, ref["P"], rtol=2e-12)
            np.testing.assert_allclose(eta, ref["eta_atm"], rtol=2e-12)
            np.testing.assert_allclose(S, ref["S"], rtol=1e-12, atol=1e-40)
    assert 0 < inside < w.n_samples * w.n_spaxel          # both branches exercised


def test_brute_force_tiny_C1():
    """Config 1 shrunk to 8 samples x 4 channels x 16 frequencies."""
    w = W.make_workload("C1", n_samples=8, n_chan=4, n_freq=16)
    r = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    for n in range(8):
        np.testing.assert_allclose(r[n, 0], numpy_chain(w, n, 0)["pkid"], rtol=1e-12)


def test_canonical_trig_matches_literal():
    """tan(a+b), sin(E+b) from the addition formulas vs the literal functions: 1e-13."""
    w = W.make_workload("C4", n_samples=4000, n_freq=8, n_chan=2, screen_n=64, cube_n=8)
    g = O.Oracle(w).geometry()
    n, s = np.meshgrid(np.arange(w.n_samples), np.arange(w.n_spaxel), indexing="ij")
    csc = 1.0 / np.sin(w.el0_rad + w.el_rad[n] + w.del_rad[s])
    np.testing.assert_allclose(g["csc"], csc, rtol=1e-13)
    a = w.az_rad[n] + w.daz_rad[s]
    u = (w.h_column_m * np.tan(a) + w.wind_mps * n / w.f_sample_hz) / w.dx_m + 32.0
    np.testing.assert_allclose(g["fu"], u - np.floor(u), atol=1e-7)
    assert np.array_equal(g["iu0"], np.floor(u).astype(np.int64) % 64)


# --------------------------------------------------------------------------------------
# invariants of the cascade (Eq. 12)
# --------------------------------------------------------------------------------------
def _row_normalised(filt, dnu):
    f = filt.astype(np.float64)
    return (f / (f.sum(axis=1, keepdims=True) * dnu)).astype(np.float32)


@pytest.mark.parametrize("variant", ["no_source", "source_is_blackbody"])
def test_thermal_equilibrium(variant):
    """Everything at one temperature T returns B(nu, T) whatever the efficiencies."""
    T = 77.0
    w = W.random_workload(5, n_samples=12, n_spaxel=2, n_chan=6, n_freq=40, couple=(variant == "no_source"))
    stages = [W.Stage(s.eta, T, s.couple_atmosphere) for s in w.stages]
    if variant == "no_source":
        w = w.replace(cube=None, T_cmb_K=T, T_atm_K=T, stages=stages)
    else:
        nu = w.nu_hz
        cube = np.broadcast_to(B(nu, T), w.cube.shape).astype(np.float32)
        w = w.replace(cube=cube, eta_front_nu=None, T_cmb_K=0.0, T_atm_K=T, stages=stages,
                      az_rad=np.zeros(12), el_rad=np.zeros(12))           # stay on the cube
    filt = _row_normalised(w.filt, w.dnu_hz)
    w = w.replace(filt=filt)
    o = O.Oracle(w)
    Bnu = B(w.nu_hz, T)
    for n in (0, 5, 11):
        rtol = 1e-12 if variant == "no_source" else 1e-7      # cube is stored in fp32
        np.testing.assert_allclose(o.row_spectrum(n, 1), Bnu, rtol=rtol)
    pk = o.simulate(want=("pkid",))["pkid"]
    expect = w.dnu_hz * (filt.astype(np.float64) @ Bnu)
    np.testing.assert_allclose(pk, np.broadcast_to(expect, pk.shape), rtol=1e-7)


def test_transparent_limit_returns_filtered_source():
    w = W.random_workload(6, n_samples=10, n_spaxel=2, n_chan=5, n_freq=30)
    w = w.replace(stages=[W.Stage(1.0, 300.0), W.Stage(np.ones(30, np.float32), 50.0, True)],
                  atm_lut=np.ones_like(w.atm_lut), T_cmb_K=0.0, eta_front_nu=None,
                  az_rad=np.linspace(-20, 20, 10) * ARCSEC, el_rad=np.linspace(15, -15, 10) * ARCSEC)
    o = O.Oracle(w)
    pk = o.simulate(want=("pkid",))["pkid"]
    for n in range(10):
        for s in range(2):
            S = numpy_chain(w, n, s)["S"]
            assert S.max() > 0
            np.testing.assert_allclose(pk[n, s], w.dnu_hz * (w.filt.astype(np.float64) @ S), rtol=1e-12)


def test_delta_filter_reproduces_spectrum():
    w = W.random_workload(7, n_samples=6, n_spaxel=2, n_chan=30, n_freq=30)
    filt = (np.eye(30) / w.dnu_hz).astype(np.float32)
    w = w.replace(filt=filt)
    o = O.Oracle(w)
    pk = o.simulate(want=("pkid",))["pkid"]
    for n in range(6):
        P = o.row_spectrum(n, 1)
        np.testing.assert_allclose(pk[n, 1], P * (w.dnu_hz * filt.astype(np.float64).diagonal()), rtol=1e-14)
        np.testing.assert_allclose(pk[n, 1], P, rtol=1e-6)               # 1/dnu rounded to fp32


def test_single_stage_by_hand():
    """One grey stage, grey atmosphere, no source, no CMB: two applications of Eq. 12."""
    w = W.random_workload(8, n_samples=3, n_spaxel=1, n_chan=2, n_freq=5)
    lut = np.full_like(w.atm_lut, 0.8)
    w = w.replace(cube=None, T_cmb_K=0.0, T_atm_K=250.0, atm_lut=lut, stages=[W.Stage(0.6, 100.0)],
                  el0_rad=math.pi / 2, el_rad=np.zeros(3), del_rad=np.zeros(1))
    P = O.Oracle(w).row_spectrum(1, 0)
    nu = w.nu_hz
    expect = 0.6 * ((1 - 0.8) * B(nu, 250.0)) + 0.4 * B(nu, 100.0)
    np.testing.assert_allclose(P, expect, rtol=1e-7)                      # 0.8 stored as fp32


def test_coupled_stage_term():
    """J_k = (1 - eta_atm) B(T_atm) + eta_atm B(T_cmb)."""
    w = W.random_workload(9, n_samples=2, n_spaxel=1, n_chan=2, n_freq=6)
    base = dict(cube=None, T_cmb_K=2.725, T_atm_K=260.0, el0_rad=math.pi / 2,
                el_rad=np.zeros(2), del_rad=np.zeros(1))
    w1 = w.replace(stages=[W.Stage(0.85, 999.0, True)], **base)
    o = O.Oracle(w1)
    P, eta, _ = o.row_spectrum(0, 0, intermediates=True)
    nu = w.nu_hz
    sky = eta * B(nu, 2.725) + (1 - eta) * B(nu, 260.0)
    np.testing.assert_allclose(P, 0.85 * sky + 0.15 * sky, rtol=1e-12)    # sky seen both ways


# --------------------------------------------------------------------------------------
# samplers
# --------------------------------------------------------------------------------------
def test_screen_sampler_vs_scipy_grid_wrap():
    w = W.random_workload(10, n_samples=200, n_spaxel=3, n_chan=2, n_freq=4, screen_n=16)
    w = w.replace(wind_mps=37.0, pwv0_a_mm=0.0, pwv0_b_mm_per_s=0.0)      # many wrap-arounds
    pwv = O.Oracle(w).simulate(want=("pwv",))["pwv"]
    n, s = np.meshgrid(np.arange(200), np.arange(3), indexing="ij")
    x = w.h_column_m * np.tan(w.az_rad[n] + w.daz_rad[s]) + w.wind_mps * n / w.f_sample_hz
    y = w.h_column_m * np.tan(w.el_rad[n] + w.del_rad[s])
    u, v = x / w.dx_m + 8.0, y / w.dy_m + 8.0
    ref = map_coordinates(w.screen.astype(np.float64), [v.ravel(), u.ravel()], order=1, mode="grid-wrap")
    np.testing.assert_allclose(pwv.ravel(), ref, rtol=1e-9)
    assert (u.max() - u.min()) > 3 * 16                                    # really wrapped


def test_screen_sampler_exact_on_affine_field_and_periodic_shift():
    n = 32
    jj, ii = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    w = W.random_workload(11, n_samples=50, n_spaxel=2, n_chan=2, n_freq=4, screen_n=n)
    w = w.replace(screen=(1.0 + 0.01 * ii + 0.003 * jj).astype(np.float32), wind_mps=0.0,
                  pwv0_a_mm=0.0, pwv0_b_mm_per_s=0.0,
                  az_rad=np.linspace(-100, 100, 50) * ARCSEC, el_rad=np.linspace(80, -80, 50) * ARCSEC)
    o = O.Oracle(w)
    g = o.geometry()
    pwv = o.simulate(want=("pwv",))["pwv"]
    u = g["iu0"] + g["fu"]
    v = g["iv0"] + g["fv"]
    assert u.min() > 1 and u.max() < n - 2 and v.min() > 1 and v.max() < n - 2      # no wrap here
    scr64 = w.screen.astype(np.float64)
    a, b, c = scr64[0, 0], scr64[0, 1] - scr64[0, 0], scr64[1, 0] - scr64[0, 0]
    np.testing.assert_allclose(pwv, a + b * u + c * v, rtol=1e-6)          # fp32 field values
    # shifting the scan by exactly one screen period in x changes nothing (R7)
    shift = math.atan(n * w.dx_m / w.h_column_m)
    w2 = w.replace(az_rad=np.zeros(50), daz_rad=np.array([0.0, shift]), del_rad=np.zeros(2))
    p2 = O.Oracle(w2).simulate(want=("pwv",))["pwv"]
    np.testing.assert_allclose(p2[:, 0], p2[:, 1], rtol=1e-9)


def test_source_sampler_vs_scipy_and_outside_rule():
    w = W.random_workload(12, n_samples=300, n_spaxel=2, n_chan=2, n_freq=5)
    o = O.Oracle(w)
    n_el, n_az, _ = w.cube.shape
    ag = w.az_min_rad + w.daz_grid_rad * np.arange(n_az)
    eg = w.el_min_rad + w.del_grid_rad * np.arange(n_el)
    rgi = RegularGridInterpolator((eg, ag), w.cube.astype(np.float64), method="linear",
                                  bounds_error=False, fill_value=0.0)
    n_out = 0
    for n in range(0, 300, 7):
        for s in range(2):
            a, e = w.az_rad[n] + w.daz_rad[s], w.el_rad[n] + w.del_rad[s]
            _, _, S = o.row_spectrum(n, s, intermediates=True)
            np.testing.assert_allclose(S, rgi([[e, a]])[0], rtol=1e-9, atol=1e-40)
            out = not (ag[0] <= a <= ag[-1] and eg[0] <= e <= eg[-1])
            n_out += out
            if out:
                assert np.all(S == 0.0)
    assert n_out > 3


def test_source_nodes_and_upper_edge():
    """Node values at integer coordinates; the upper edge belongs to the grid (R12)."""
    w = W.random_workload(13, n_samples=4, n_spaxel=1, n_chan=2, n_freq=5)
    n_el, n_az, _ = w.cube.shape
    ag = w.az_min_rad + w.daz_grid_rad * np.arange(n_az)
    eg = w.el_min_rad + w.del_grid_rad * np.arange(n_el)
    w = w.replace(az_rad=np.array([ag[2], ag[-1], ag[0], ag[-1] + 1e-9]),
                  el_rad=np.array([eg[3], eg[-1], eg[0], eg[1]]), daz_rad=np.zeros(1), del_rad=np.zeros(1))
    o = O.Oracle(w)
    c = w.cube.astype(np.float64)
    for n, (j, i) in enumerate([(3, 2), (n_el - 1, n_az - 1), (0, 0)]):
        np.testing.assert_allclose(o.row_spectrum(n, 0, True)[2], c[j, i], rtol=1e-9)
    assert np.all(o.row_spectrum(3, 0, True)[2] == 0.0)


def test_lut_vs_scipy_and_pwv_clamp():
    w = W.random_workload(14, n_samples=40, n_spaxel=2, n_chan=2, n_freq=23)
    w = w.replace(pwv0_a_mm=-1.0, pwv0_b_mm_per_s=10.0)          # PWV sweeps through and past the LUT
    o = O.Oracle(w)
    g = o.geometry()
    pwv_hi = w.lut_pwv0_mm + w.lut_dpwv_mm * (w.atm_lut.shape[0] - 1)
    assert (g["pwv_mm"] > pwv_hi).any() and (g["pwv_mm"] < w.lut_pwv0_mm).any()    # rows clamped both ways
    assert g["ip"].min() == 0 and g["ip"].max() == w.atm_lut.shape[0] - 2
    assert ((g["fp"] >= 0) & (g["fp"] <= 1)).all()
    for n in (0, 13, 20, 39):
        ref = numpy_chain(w, n, 1)
        np.testing.assert_allclose(o.row_spectrum(n, 1, True)[1], ref["eta_atm"], rtol=1e-12)


def test_airmass_closed_form():
    """Synthetic LUT exp(-tau pwv) with pwv on a LUT node and nu on LUT nodes:
    eta_atm = exp(-tau pwv csc(el)); el = 90 deg returns the zenith value."""
    lut, lnu0, ldnu, lp0, ldp = W.atm_lut()
    nf = 50
    nu0, dnu = lnu0 + 100 * ldnu, 20 * ldnu                     # grid frequencies on LUT nodes
    w = W.random_workload(15, n_samples=2, n_spaxel=1, n_chan=2, n_freq=nf)
    pwv_node = lp0 + 18 * ldp                                    # 1.0 mm
    w = w.replace(nu0_hz=nu0, dnu_hz=dnu, atm_lut=lut, lut_nu0_hz=lnu0, lut_dnu_hz=ldnu,
                  lut_pwv0_mm=lp0, lut_dpwv_mm=ldp, screen=np.full((8, 8), pwv_node, np.float32),
                  pwv0_a_mm=0.0, pwv0_b_mm_per_s=0.0, cube=None,
                  stages=[W.Stage(s.eta if np.ndim(s.eta) == 0 else 0.9, s.T_K, s.couple_atmosphere) for s in w.stages],
                  eta_front_nu=None, el_rad=np.zeros(2), del_rad=np.zeros(1), el0_rad=np.deg2rad(47.8))
    eta = O.Oracle(w).row_spectrum(0, 0, True)[1]
    tau = W.tau_per_mm(w.nu_hz)
    np.testing.assert_allclose(eta, np.exp(-tau * pwv_node / math.sin(np.deg2rad(47.8))), rtol=2e-6)
    eta90 = O.Oracle(w.replace(el0_rad=math.pi / 2)).row_spectrum(0, 0, True)[1]
    np.testing.assert_allclose(eta90, np.exp(-tau * pwv_node), rtol=1e-6)


# --------------------------------------------------------------------------------------
# noise through the chain
# --------------------------------------------------------------------------------------
def test_photon_noise_variance_through_chain():
    """Stare at a flat screen: Var_t(tod[c]) = sigma_c^2 (Eq. 18)."""
    nt = 20000
    w = W.random_workload(16, n_samples=8, n_spaxel=1, n_chan=6, n_freq=20, photon_noise=True)
    w = w.replace(n_samples=nt, az_rad=np.zeros(nt), el_rad=np.zeros(nt), wind_mps=0.0, pwv0_b_mm_per_s=0.0)
    o = O.Oracle(w)
    r = o.simulate(want=("tod", "pkid"))
    pk = r["pkid"][0, 0]
    assert np.abs(r["pkid"] - pk).max() <= 1e-12 * pk.max()
    d = o.dnu_eff()
    for c in range(w.n_chan):
        sig = O.photon_sigma(pk[c], w.f_center_hz[c], d[c], w.f_sample_hz)
        var = np.var(r["tod"][:, 0, c] - pk[c])
        assert var / sig ** 2 == pytest.approx(1.0, abs=4 * math.sqrt(2 / nt))
        assert abs(np.mean(r["tod"][:, 0, c] - pk[c])) < 4 * sig / math.sqrt(nt)


def test_simulate_is_sum_of_its_parts_and_chunk_invariant():
    """Eq. 21: tod = (P_KID + wn) + pn, and a window equals the same rows of a full run."""
    w = W.random_workload(17, n_samples=48, n_spaxel=2, n_chan=5, n_freq=16, photon_noise=True, pink_noise=True)
    o = O.Oracle(w)
    full = o.simulate(want=("tod", "pkid"))
    t_idx, s_idx = np.meshgrid(np.arange(48), np.arange(2), indexing="ij")
    pk, wn = o.simulate_rows(t_idx.ravel(), s_idx.ravel(), noise=True)
    assert np.array_equal(pk.reshape(48, 2, 5), full["pkid"])
    ss, cc = np.meshgrid(np.arange(2), np.arange(5), indexing="ij")
    pn = o.pink_series(ss.ravel(), cc.ravel(), 0, 48).reshape(2, 5, 48).transpose(2, 0, 1)
    assert np.array_equal(full["tod"], (full["pkid"] + wn.reshape(48, 2, 5)) + pn)
    part = o.simulate(t_begin=19, t_count=20, want=("tod",))["tod"]
    assert np.array_equal(part, full["tod"][19:39])
    # noise terms are switched independently
    quiet = O.Oracle(w.replace(photon_noise=False, pink_noise=False)).simulate(want=("tod",))["tod"]
    assert np.array_equal(quiet, full["pkid"])
    assert np.abs(wn).max() > 0 and np.abs(pn).max() > 0


def test_photon_noise_counter_layout():
    """wn of row (n, s), channel c uses normal (c div 32) mod 4 of Philox(counter = (n, s, 32 (c div 128) + c mod 32, 0),
    key = seed) (R19; the block and normal are written out per channel here)."""
    w = W.random_workload(18, n_samples=5, n_spaxel=2, n_chan=131, n_freq=8, photon_noise=True)
    o = O.Oracle(w)
    pk, wn = o.simulate_rows([4, 2], [1, 0], noise=True)
    d = o.dnu_eff()
    where = {0: (0, 0), 2: (2, 0), 33: (1, 1), 70: (6, 2), 100: (4, 3), 127: (31, 3), 128: (32, 0), 130: (34, 0)}
    for r, (n, s) in enumerate([(4, 1), (2, 0)]):
        for c, (blk, k) in where.items():
            z0 = O.normals4(w.seed, n, s, blk, 0)[k]
            sig = O.photon_sigma(pk[r, c], w.f_center_hz[c], d[c], w.f_sample_hz)
            assert wn[r, c] == pytest.approx(sig * z0, rel=1e-14)
