"""Pins for the oracle's elementary pieces: each is checked against something other than
the oracle itself (closed forms, the vendor's Philox, distribution tests, exact PSDs)."""
import math
import shutil
import subprocess
from pathlib import Path

import numpy as np
import pytest
from scipy import signal, stats

from oracle import oracle as O
from paper_2604_23305_b200 import workloads as W

H, KB = 6.62607015e-34, 1.380649e-23
GOLDEN = Path(__file__).resolve().parent / "golden"


# ---------------------------------------------------------------- P^JN
def test_planck_rayleigh_jeans_limit():
    # h nu << k T:  B = k T (1 - x/2 + x^2/12 - ...)
    nu, T = 1e9, 300.0
    x = H * nu / (KB * T)
    assert O.planck(nu, T) == pytest.approx(KB * T * (1 - x / 2 + x * x / 12), rel=1e-14)


def test_planck_wien_tail_and_zero():
    nu, T = 400e9, 2.0          # x ~ 9.6
    x = H * nu / (KB * T)
    # exact form via exp; and the Wien tail B -> h nu e^-x within e^-x relative
    assert O.planck(nu, T) == pytest.approx(H * nu / (math.exp(x) - 1.0), rel=1e-13)
    assert O.planck(nu, T) == pytest.approx(H * nu * math.exp(-x), rel=2 * math.exp(-x))
    assert O.planck(nu, 0.0) == 0.0
    assert O.planck(300e9, 273.0) == pytest.approx(3.5697e-21, rel=1e-3)   # ~ k T (1 - x/2)


def test_planck_monotone_in_T():
    v = [O.planck(350e9, T) for T in (2.725, 4.0, 77.0, 273.0, 290.0)]
    assert all(a < b for a, b in zip(v, v[1:]))


# ---------------------------------------------------------------- Philox4x32-10
@pytest.mark.skipif(shutil.which("nvcc") is None, reason="needs nvcc for the vendor header")
def test_philox_matches_curand_host_implementation(tmp_path):
    """Known answers from NVIDIA's curand_philox4x32_x.h compiled for the host."""
    exe = tmp_path / "curand_philox_host"
    subprocess.check_call(["nvcc", "-O1", "-Wno-deprecated-gpu-targets", "-o", str(exe),
                           str(GOLDEN / "curand_philox_host.cu")])
    rng = np.random.default_rng(11)
    cases = [[0] * 6, [0xffffffff] * 6, [1, 0, 0, 0, 0, 0], [0, 0, 0, 0, 1, 0], [0, 0, 0, 1, 0, 0]]
    cases += [list(map(int, rng.integers(0, 2 ** 32, 6))) for _ in range(200)]
    inp = "\n".join(" ".join(f"{v:x}" for v in c) for c in cases) + "\n"
    out = subprocess.run([str(exe)], input=inp, capture_output=True, text=True, check=True).stdout
    ref = [[int(t, 16) for t in line.split()] for line in out.strip().splitlines()]
    assert len(ref) == len(cases)
    for c, r in zip(cases, ref):
        assert O.philox4x32_10(c[:4], c[4:]) == r


def test_philox_is_a_bijection_on_a_small_slice():
    outs = {tuple(O.philox4x32_10([i, 0, 0, 0], [5, 6])) for i in range(2000)}
    assert len(outs) == 2000


def test_uniform_is_open_interval_and_fp32_exact():
    for w in (0, 1, 511, 512, 2 ** 31, 2 ** 32 - 1):
        u = O.uniform01(w)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                 # exactly representable in binary32
    assert O.uniform01(0) == 0.5 / 2 ** 23
    assert O.uniform01(2 ** 32 - 1) == 1.0 - 0.5 / 2 ** 23


def test_normals_box_muller_definition():
    seed, ctr = 0x1234567890abcdef, (7, 3, 5, 1)
    w = O.philox4x32_10(ctr, [seed & 0xffffffff, seed >> 32])
    u = [((x >> 9) + 0.5) / 2 ** 23 for x in w]
    z = O.normals4(seed, *ctr)
    r0, r1 = math.sqrt(-2 * math.log(u[0])), math.sqrt(-2 * math.log(u[2]))
    exp = [r0 * math.cos(2 * math.pi * u[1]), r0 * math.sin(2 * math.pi * u[1]),
           r1 * math.cos(2 * math.pi * u[3]), r1 * math.sin(2 * math.pi * u[3])]
    np.testing.assert_allclose(z, exp, rtol=1e-13, atol=1e-15)


def test_normals_distribution():
    z = O.normals_bulk(seed=42, c0_begin=0, count=500_000, c1=1, c2=2, c3=0).ravel()   # 2e6 draws
    n = z.size
    assert abs(z.mean()) < 4 / math.sqrt(n)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs(stats.kurtosis(z)) < 4 * math.sqrt(24 / n)
    assert abs(stats.skew(z)) < 4 * math.sqrt(6 / n)
    assert stats.kstest(z[:200_000], "norm").pvalue > 1e-3
    assert np.abs(z).max() <= math.sqrt(2 * 24 * math.log(2)) + 1e-9        # U >= 2^-24
    # the four outputs of a block are uncorrelated
    c = np.corrcoef(z.reshape(-1, 4).T)
    assert np.abs(c - np.eye(4)).max() < 5 / math.sqrt(n / 4)


def test_photon_normal_channel_mapping():
    """R19: one stream-0 block serves the four channels b + 128 q + {0, 32, 64, 96}.  Checked without the formula's own
    index arithmetic: every channel of a 300-channel row must find its normal among the four of exactly one of the
    blocks 0..95 of that (n, s), each (block, normal) pair is used by exactly one channel, and the table below lists the
    expected (block, normal) of hand-picked channels."""
    seed, n, s = 0xfeedfacecafe, 1234, 17
    blocks = np.array([O.normals4(seed, n, s, b, 0) for b in range(96)])          # [block][normal]
    used = {}
    for ch in range(300):
        z = O.photon_normal(seed, n, s, ch)
        hit = np.argwhere(blocks == z)
        assert len(hit) == 1
        used[ch] = tuple(int(v) for v in hit[0])
    assert len(set(used.values())) == 300
    by_hand = {0: (0, 0), 31: (31, 0), 32: (0, 1), 63: (31, 1), 64: (0, 2), 97: (1, 3), 127: (31, 3),
               128: (32, 0), 160: (32, 1), 255: (63, 3), 256: (64, 0), 299: (75, 1)}
    for ch, bk in by_hand.items():
        assert used[ch] == bk
    # other samples, spaxels and seeds give other values
    z0 = O.photon_normal(seed, n, s, 5)
    assert len({z0, O.photon_normal(seed, n + 1, s, 5), O.photon_normal(seed, n, s + 1, 5), O.photon_normal(seed + 1, n, s, 5)}) == 4


def test_photon_normals_of_a_row_are_independent_standard_normals():
    """The four channels that share a block use the cosine and sine branches of two Box-Muller pairs: jointly independent
    N(0,1).  Moments over 347 channels x 3000 samples, and the correlation between the channels of a block."""
    seed, s, nc, ns = 99, 3, 347, 3000
    z = np.array([[O.photon_normal(seed, n, s, ch) for ch in range(nc)] for n in range(ns)])
    m = z.size
    assert abs(z.mean()) < 4 / math.sqrt(m)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / m)
    assert abs(stats.kurtosis(z.ravel())) < 4 * math.sqrt(24 / m)
    assert stats.kstest(z.ravel()[:200_000], "norm").pvalue > 1e-3
    c = np.corrcoef(z[:, [5, 37, 69, 101, 133, 6]].T)             # channels 5, 37, 69, 101 share block 5
    assert np.abs(c - np.eye(6)).max() < 5 / math.sqrt(ns)
    q = np.corrcoef((z[:, [5, 37, 69, 101]] ** 2).T)               # and their squares (radius shared by cos / sin branches)
    assert np.abs(q - np.eye(4)).max() < 5 / math.sqrt(ns)


# ---------------------------------------------------------------- photon noise (Eq. 17-19)
def test_photon_sigma_formula_and_limits():
    P, fc, dn, fs = 1.3e-13, 300e9, 1.9e9, 160.0
    s = O.photon_sigma(P, fc, dn, fs)
    assert s == pytest.approx(math.sqrt((2 * H * fc * P + 2 * P * P / dn) * fs / 2), rel=1e-14)
    # shot-noise limit (P -> 0): sigma^2 -> h f P f_s ; bunching limit: sigma -> P sqrt(f_s/dnu)
    assert O.photon_sigma(1e-22, fc, dn, fs) ** 2 == pytest.approx(H * fc * 1e-22 * fs, rel=1e-5)
    assert O.photon_sigma(1e-6, fc, dn, fs) == pytest.approx(1e-6 * math.sqrt(fs / dn), rel=1e-5)
    assert O.photon_sigma(0.0, fc, dn, fs) == 0.0


def test_dnu_eff_default_is_lorentzian_equivalent_width():
    # an isolated Lorentzian on a wide fine grid: (int F)^2 / int F^2 = pi f / R
    f0, R = 300e9, 500.0
    nu = np.linspace(f0 - 150e9, f0 + 150e9, 60001)
    w = W.random_workload(1, n_chan=1, n_freq=nu.size)
    w = w.replace(nu0_hz=float(nu[0]), dnu_hz=float(nu[1] - nu[0]),
                  filt=W.lorentzian_filterbank(nu, np.array([f0]), R), f_center_hz=np.array([f0]),
                  eta_front_nu=None, cube=None,
                  stages=[], lut_nu0_hz=float(nu[0]) - 1e9,
                  lut_dnu_hz=(nu[-1] - nu[0] + 2e9) / (w.atm_lut.shape[1] - 1))
    d = O.Oracle(w).dnu_eff()[0]
    assert d == pytest.approx(math.pi * f0 / R, rel=1e-2)


# ---------------------------------------------------------------- AR(1) cascade pink noise
def _pink_workload(J=4, n_samples=1 << 15, n_chan=64):
    w = W.random_workload(3, n_samples=8, n_spaxel=1, n_chan=n_chan, pink_noise=True, J=J)
    n = w.n_spaxel * w.n_chan
    return w.replace(n_samples=n_samples, az_rad=np.zeros(n_samples), el_rad=np.zeros(n_samples),
                     pink_A=np.full(n, 2.5e-34), pink_alpha=np.full(n, 1.0))


def test_pink_coefficients_closed_form():
    w = _pink_workload()
    phi, g = O.Oracle(w).pink_coeffs(0, 5)
    fj = w.pink_f_corner_hz
    np.testing.assert_allclose(phi, np.exp(-2 * np.pi * fj / w.f_sample_hz), rtol=1e-15)
    # alpha = 1: g_j^2 = A ln(10)
    np.testing.assert_allclose(g ** 2, 2.5e-34 * math.log(10.0) * np.ones(4), rtol=1e-12)


def test_pink_stage_statistics_and_psd():
    """Unit-variance stationary stages: total variance = sum g_j^2; Welch PSD averaged over
    detectors matches the exact discrete-time AR(1) sum, and follows A/f mid-band."""
    w = _pink_workload()
    o = O.Oracle(w)
    nd = w.n_chan
    x = o.pink_series(np.zeros(nd, np.int32), np.arange(nd, dtype=np.int32), 0, w.n_samples)
    phi, g = o.pink_coeffs(0, 0)
    var_exact = float(np.sum(g ** 2))
    # slow stages decorrelate slowly: compare the ensemble variance at fixed times
    v = x[:, ::4096].var(axis=0).mean()
    assert v == pytest.approx(var_exact, rel=0.25)
    fs = w.f_sample_hz
    f, pxx = signal.welch(x, fs=fs, nperseg=4096, axis=1)
    pxx = pxx.mean(axis=0)
    exact = sum(gj ** 2 * (2 / fs) * (1 - p * p) / (1 - 2 * p * np.cos(2 * np.pi * f / fs) + p * p)
                for gj, p in zip(g, phi))
    band = (f > 0.2) & (f < 60)
    n_avg = nd * (w.n_samples // 2048 - 1)
    assert np.abs(pxx[band] / exact[band] - 1).max() < 6 / math.sqrt(n_avg) + 0.03
    # stated approximation of A f^-alpha: holds between the lowest and the highest corner
    # (0.002-2 Hz here); above the top corner the cascade rolls off as f^-2 (R18)
    mid = (f > 0.04) & (f < 2.0)
    ratio = exact[mid] / (2.5e-34 / f[mid])
    assert 0.85 < ratio.min() and ratio.max() < 1.1


def test_pink_lag1_autocorrelation_single_stage():
    w = _pink_workload(J=1, n_samples=1 << 14, n_chan=32)
    o = O.Oracle(w)
    x = o.pink_series(np.zeros(32, np.int32), np.arange(32, dtype=np.int32), 0, w.n_samples)
    phi, g = o.pink_coeffs(0, 0)
    r1 = np.mean(x[:, 1:] * x[:, :-1]) / np.mean(x * x)
    assert r1 == pytest.approx(phi[0], abs=0.01)
    assert np.mean(x * x) == pytest.approx(g[0] ** 2, rel=0.05)


def test_pink_series_windows_are_consistent():
    """A window starting at t_begin equals the same samples of a run from 0 (chunk seams)."""
    w = _pink_workload(n_samples=600, n_chan=4)
    o = O.Oracle(w)
    s, c = np.zeros(4, np.int32), np.arange(4, dtype=np.int32)
    full = o.pink_series(s, c, 0, 600)
    part = o.pink_series(s, c, 217, 300)
    assert np.array_equal(full[:, 217:517], part)


# ---- the J > 4 branch: stages 4-7 draw from Philox stream 2 (gateau_oracle.cpp pink_series, R19) ----
def _pink8_workload(n_samples, n_chan):
    """Eight corners an octave apart, 16 ... 0.125 Hz: every stage carries power inside the Welch band, so a slip
    in the second stream (stages 4-7 re-using stream 1, or the wrong normals of stream 2) shows in the PSD."""
    w = _pink_workload(J=8, n_samples=n_samples, n_chan=n_chan)
    return w.replace(pink_f_corner_hz=16.0 * 2.0 ** (-np.arange(8, dtype=np.float64)))


def test_pink_eight_stages_psd_and_variance():
    """Welch PSD of the J = 8 cascade against the exact discrete-time sum of EIGHT independent unit-variance AR(1)
    spectra, and the ensemble variance against sum g_j^2.  Correlated stages (x_{j+4} driven by the innovations of
    x_j) would add the cross spectra 2 g_j g_{j+4} Re(H_j H*_{j+4}): tens of per cent here."""
    w = _pink8_workload(1 << 16, 128)
    o = O.Oracle(w)
    nd, fs = w.n_chan, w.f_sample_hz
    x = o.pink_series(np.zeros(nd, np.int32), np.arange(nd, dtype=np.int32), 0, w.n_samples)
    phi, g = o.pink_coeffs(0, 0)
    assert phi.shape == (8,) and g.shape == (8,)
    np.testing.assert_allclose(phi, np.exp(-2 * np.pi * w.pink_f_corner_hz / fs), rtol=1e-15)
    np.testing.assert_allclose(g ** 2, 2.5e-34 * math.log(2.0) * np.ones(8), rtol=1e-12)     # alpha = 1, rho = 2
    f, pxx = signal.welch(x, fs=fs, nperseg=4096, axis=1)
    pxx = pxx.mean(axis=0)

    def H2(p):
        return (2 / fs) * (1 - p * p) / (1 - 2 * p * np.cos(2 * np.pi * f / fs) + p * p)

    exact = sum(gj ** 2 * H2(p) for gj, p in zip(g, phi))
    band = (f > 0.2) & (f < 60)
    n_avg = nd * (w.n_samples // 2048 - 1)
    tol = 6 / math.sqrt(n_avg) + 0.03
    assert np.abs(pxx[band] / exact[band] - 1).max() < tol
    # what the test would see if stages j and j+4 shared their innovations: far outside the tolerance
    z = np.exp(-2j * np.pi * f / fs)
    shared = exact + sum(2 * g[j] * g[j + 4] * (2 / fs) * math.sqrt((1 - phi[j] ** 2) * (1 - phi[j + 4] ** 2))
                         * np.real(1 / ((1 - phi[j] * z) * np.conj(1 - phi[j + 4] * z))) for j in range(4))
    assert np.abs(shared[band] / exact[band] - 1).min() > 3 * tol
    # every stage is stationary with unit variance from n = 0 on: ensemble variance at fixed times
    v = x[:, ::1024].var(axis=0).mean()
    assert v == pytest.approx(float(np.sum(g ** 2)), rel=0.08)


def test_pink_eight_stages_two_streams_by_hand():
    """The series rebuilt from the pinned Philox normals: stages 0-3 take the four normals of stream 1, stages 4-7
    those of stream 2, initial states from counter 0xFFFFFFFF (R19).  The two halves are also uncorrelated."""
    w = _pink8_workload(4096, 3)
    o = O.Oracle(w)
    n, ch = w.n_samples, 2
    got = o.pink_series(np.zeros(1, np.int32), np.array([ch], dtype=np.int32), 0, n)[0]
    phi, g = o.pink_coeffs(0, ch)
    z = np.concatenate([O.normals_bulk(w.seed, 0, n, 0, ch, 1), O.normals_bulk(w.seed, 0, n, 0, ch, 2)], axis=1)
    x = np.concatenate([O.normals4(w.seed, 0xFFFFFFFF, 0, ch, 1), O.normals4(w.seed, 0xFFFFFFFF, 0, ch, 2)])
    xs = np.empty((n, 8))
    for i in range(n):
        x = phi * x + np.sqrt(1 - phi * phi) * z[i]
        xs[i] = x
    np.testing.assert_allclose(got, xs @ g, rtol=0, atol=1e-12 * np.abs(got).max())
    # innovations of the two streams are independent draws
    c = np.corrcoef(z.T)
    assert np.abs(c[:4, 4:]).max() < 5 / math.sqrt(n)


# ---- Timmer & Koenig pink noise (the paper's own method; R21) ----
def _tk_workload(n_samples, n_chan=6, alpha=1.0, seed=5):
    from paper_2604_23305_b200 import workloads as W
    w = W.random_workload(seed, n_samples=n_samples, n_spaxel=2, n_chan=n_chan, n_freq=8, pink_noise=True)
    return w.replace(pink_method=1, pink_A=np.full(2 * n_chan, 3e-34), pink_alpha=np.full(2 * n_chan, alpha))


@pytest.mark.parametrize("N", [1000, 1001])
def test_tk_series_spectrum_roundtrip_and_parseval(N):
    """rfft of the series gives back exactly the drawn coefficients (X_0 = 0, Hermitian extension), so the
    periodogram IS the requested PSD times the squared normals; mean zero; Parseval."""
    w = _tk_workload(N)
    o = O.Oracle(w)
    s_idx, c_idx = np.array([0, 1, 1], dtype=np.int32), np.array([0, 3, 5], dtype=np.int32)
    x = o.pink_tk_series(s_idx, c_idx)
    assert x.shape == (3, N) and np.all(np.abs(x.mean(axis=1)) < 1e-12 * np.abs(x).max())
    K = N // 2
    fk = np.arange(K + 1) * w.f_sample_hz / N
    for i, (s, c) in enumerate(zip(s_idx, c_idx)):
        X = np.fft.rfft(x[i])
        z = O.normals_bulk(w.seed, 0, K + 1, int(s), int(c), 3)
        P = 3e-34 / fk[1:]
        top = K if N % 2 == 1 else K - 1
        want = np.sqrt(P[:top] * w.f_sample_hz * N / 4.0) * (z[1:top + 1, 0] + 1j * z[1:top + 1, 1])
        assert np.allclose(X[1:top + 1], want, rtol=1e-9, atol=1e-12 * np.abs(want).max())
        assert abs(X[0]) < 1e-9 * np.abs(want).max()
        if N % 2 == 0:
            assert np.isclose(X[K].real, np.sqrt(P[K - 1] * w.f_sample_hz * N) * z[K, 0], rtol=1e-9)
        # Parseval: sum x^2 = (1/N) (2 sum |X_k|^2 + |X_{N/2}|^2)
        rhs = (2 * np.sum(np.abs(X[1:top + 1]) ** 2) + (abs(X[K]) ** 2 if N % 2 == 0 else 0.0)) / N
        assert np.isclose(np.sum(x[i] ** 2), rhs, rtol=1e-10)


@pytest.mark.parametrize("alpha", [1.0, 1.5])
def test_tk_average_periodogram_follows_the_power_law(alpha):
    """One-sided periodogram (2 / (f_s N)) |X_k|^2 averaged over many detectors = A f^-alpha."""
    N, n_chan = 512, 200
    w = _tk_workload(N, n_chan=n_chan, alpha=alpha)
    o = O.Oracle(w)
    s_idx = np.repeat(np.arange(2), n_chan).astype(np.int32)
    c_idx = np.tile(np.arange(n_chan), 2).astype(np.int32)
    x = o.pink_tk_series(s_idx, c_idx)
    S = 2.0 / (w.f_sample_hz * N) * np.abs(np.fft.rfft(x, axis=1)[:, 1:N // 2]) ** 2
    fk = np.arange(1, N // 2) * w.f_sample_hz / N
    ratio = S.mean(axis=0) / (3e-34 * fk ** (-alpha))
    # each |X_k|^2 / (2 sigma^2) is chi^2_2 / 2: the mean over 400 detectors has relative std 1/20
    assert abs(ratio.mean() - 1.0) < 0.02 and np.all(np.abs(ratio - 1.0) < 0.25)


@pytest.mark.parametrize("N", [16, 17])
def test_tk_series_is_the_direct_fourier_sum(N):
    """Tiny N, the definition written out as cosines and sines (no FFT): x_n = (2/N) sum_{0<k<N/2} sigma_k
    (z0 cos(2 pi k n / N) - z1 sin(2 pi k n / N)) + (1/N) sqrt(P f_s N) z0 (-1)^n, sigma_k = sqrt(P(f_k) f_s N / 4)."""
    w = _tk_workload(N, alpha=1.3)
    o = O.Oracle(w)
    x = o.pink_tk_series(np.array([1], dtype=np.int32), np.array([2], dtype=np.int32))[0]
    K = N // 2
    z = O.normals_bulk(w.seed, 0, K + 1, 1, 2, 3)
    want = np.zeros(N)
    for n in range(N):
        acc = 0.0
        for k in range(1, K + 1):
            fk = k * w.f_sample_hz / N
            P = 3e-34 * fk ** (-1.3)
            if 2 * k == N:
                acc += np.sqrt(P * w.f_sample_hz * N) * z[k, 0] * (-1.0) ** n / N
            else:
                ph = 2.0 * np.pi * k * n / N
                acc += 2.0 / N * np.sqrt(P * w.f_sample_hz * N / 4.0) * (z[k, 0] * np.cos(ph) - z[k, 1] * np.sin(ph))
        want[n] = acc
    assert np.allclose(x, want, rtol=1e-10, atol=1e-12 * np.abs(want).max())


def test_tk_slope_variance_and_independence():
    """Fitted log-log slope of the averaged periodogram is -alpha; the series variance is the integral of the
    one-sided PSD over the resolved band, sum_k P(f_k) f_s / N; different detectors / seeds are uncorrelated."""
    N, n_chan, alpha = 1024, 150, 1.2
    w = _tk_workload(N, n_chan=n_chan, alpha=alpha)
    o = O.Oracle(w)
    s_idx = np.repeat(np.arange(2), n_chan).astype(np.int32)
    c_idx = np.tile(np.arange(n_chan), 2).astype(np.int32)
    x = o.pink_tk_series(s_idx, c_idx)
    S = (2.0 / (w.f_sample_hz * N) * np.abs(np.fft.rfft(x, axis=1)[:, 1:N // 2]) ** 2).mean(axis=0)
    fk = np.arange(1, N // 2) * w.f_sample_hz / N
    slope = np.polyfit(np.log(fk), np.log(S), 1)[0]
    assert abs(slope + alpha) < 0.03
    fall = np.arange(1, N // 2 + 1) * w.f_sample_hz / N
    var_want = np.sum(3e-34 * fall ** (-alpha)) * w.f_sample_hz / N
    assert abs(x.var(axis=1).mean() / var_want - 1.0) < 0.1
    # whitened coefficients of different detectors are uncorrelated unit normals (1022 of them per detector)
    X = np.fft.rfft(x, axis=1)[:, 1:N // 2] / np.sqrt(3e-34 * fk ** (-alpha) * w.f_sample_hz * N / 4.0)
    g = np.concatenate([X.real, X.imag], axis=1)
    assert abs(g.mean()) < 0.01 and abs(g.var() - 1.0) < 0.01
    cc = g @ g.T / g.shape[1]
    np.fill_diagonal(cc, 0.0)
    assert np.abs(cc).max() < 6.0 / np.sqrt(g.shape[1])
    x2 = O.Oracle(w.replace(seed=w.seed + 1)).pink_tk_series(s_idx[:4], c_idx[:4])
    assert np.abs(x2 - x[:4]).max() > 0.5 * np.abs(x[:4]).max()
