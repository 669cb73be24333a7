"""Pins of the oracle's exact photon-noise NEP, Eq. 17 (R23)."""
import numpy as np

from oracle import oracle as O
from paper_2604_23305_b200 import workloads as W

H = 6.62607015e-34
GAP = 188e-6 * 1.602176634e-19


def test_single_frequency_by_hand():
    F = np.array([[0.0, 0.2, 0.0], [0.0, 0.0, 0.5]])
    P = np.array([1e-22, 3e-22, 5e-22])
    nu = np.array([3e11, 3.1e11, 3.2e11])
    got = O.nep2_exact(F, P, nu, 1e8, GAP, 0.4)
    for c, i in ((0, 1), (1, 2)):
        x = F[c, i] * P[i]
        assert np.isclose(got[c], 2 * 1e8 * x * (H * nu[i] + x + 2 * GAP / 0.4), rtol=1e-14)


def test_flat_spectrum_reduces_to_the_three_named_terms():
    """P_nu = P0: NEP^2 = 2 P0 sum F h nu dnu (shot) + 2 P0^2 sum F^2 dnu (bunching) + (4 Delta / eta_pb) P0 sum F dnu (GR);
    in terms of P_KID = P0 sum F dnu and dnu_c = (sum F dnu)^2 / sum F^2 dnu the bunching term is 2 P_KID^2 / dnu_c,
    north_star's form (R17)."""
    rng = np.random.default_rng(0)
    nu = 3e11 + 1e8 * np.arange(400)
    F = 0.3 * rng.random((5, 400)) ** 3
    P0, dnu = 2.5e-22, 1e8
    got = O.nep2_exact(F, np.full(400, P0), nu, dnu, GAP, 0.4)
    pk = P0 * F.sum(axis=1) * dnu
    dnu_c = (F.sum(axis=1) * dnu) ** 2 / ((F ** 2).sum(axis=1) * dnu)
    shot = 2 * P0 * dnu * (F * H * nu).sum(axis=1)
    want = shot + 2 * pk ** 2 / dnu_c + 4 * GAP / 0.4 * pk
    assert np.allclose(got, want, rtol=1e-12)
    # without the GR term and for a filter narrow against nu: within the filter's fractional width of R17's formula
    Fn = np.zeros((1, 400)); Fn[0, 195:205] = 0.2
    got = O.nep2_exact(Fn, np.full(400, P0), nu, dnu, 0.0, 0.4)
    pk = P0 * Fn.sum() * dnu
    nb = 2 * H * nu[199:201].mean() * pk + 2 * pk ** 2 / (10 * dnu)
    assert np.isclose(got[0], nb, rtol=1e-5)


def test_limits_and_scaling():
    rng = np.random.default_rng(1)
    nu = 2.5e11 + 2e8 * np.arange(200)
    F = 0.2 * rng.random((3, 200))
    P = 1e-22 * (1 + rng.random(200))
    full = O.nep2_exact(F, P, nu, 2e8, GAP, 0.4)
    # GR term is linear in the gap, and proportional to P_KID
    no_gr = O.nep2_exact(F, P, nu, 2e8, 0.0, 0.4)
    assert np.allclose(full - no_gr, 4 * GAP / 0.4 * 2e8 * (F @ P), rtol=1e-10)
    # Poisson limit: at vanishing power only the terms linear in P survive
    tiny = O.nep2_exact(F, 1e-12 * P, nu, 2e8, 0.0, 0.4)
    assert np.allclose(tiny, 2 * 2e8 * (F * H * nu) @ (1e-12 * P), rtol=1e-9)
    # bunching term quadruples when the power doubles
    b1 = no_gr - 2 * 2e8 * (F * H * nu) @ P
    b2 = O.nep2_exact(F, 2 * P, nu, 2e8, 0.0, 0.4) - 2 * 2e8 * (F * H * nu) @ (2 * P)
    assert np.allclose(b2, 4 * b1, rtol=1e-9)
    assert np.isclose(2 * GAP / H / 1e9, 90.9, rtol=2e-3)      # the 90 GHz pair-breaking cutoff of PAPER.md:103


def test_rows_exact_uses_the_chain_and_the_same_normals():
    w = W.random_workload(13, n_samples=12, n_spaxel=2, n_chan=6, n_freq=40, photon_noise=True).replace(photon_mode=1)
    o = O.Oracle(w)
    t_idx, s_idx = np.array([0, 5, 11]), np.array([1, 0, 1])
    pk, wn = o.simulate_rows_exact(t_idx, s_idx)
    pk0, wn0 = o.simulate_rows(t_idx, s_idx, noise=True)             # narrow-band mode: same P_KID, same z
    assert np.allclose(pk, pk0, rtol=1e-12)
    z0 = wn0 / np.array([[O.photon_sigma(pk0[i, c], w.f_center_hz[c], o.dnu_eff()[c], w.f_sample_hz)
                          for c in range(w.n_chan)] for i in range(3)])
    nep2 = np.array([O.nep2_exact(w.filt, o.row_spectrum(int(n), int(s)), w.nu_hz, w.dnu_hz, w.kid_gap_J, w.eta_pb)
                     for n, s in zip(t_idx, s_idx)])
    assert np.allclose(wn / np.sqrt(nep2 * w.f_sample_hz / 2), z0, rtol=1e-9)
    assert np.all(nep2 > 0)
