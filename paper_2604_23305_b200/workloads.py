"""Seeded synthetic inputs for the gateau hot path (arXiv 2604.23305).

This module only *makes inputs*: frequency grids, filterbank matrices, PWV screens,
transmission lookup tables, source cubes, cascade stage lists, spaxel layouts and scan
patterns, with the shapes, sizes and value ranges of the paper's DESHIMA-2.0 and IFU
workloads and of BASELINE.json's five configs.
It holds none of the signal chain (no screen/LUT/cube sampling, no cascade, no
contraction, no noise): both the CPU oracle (oracle/) and the CUDA path are fed the very
same arrays made here, and neither is imported here.

The paper's real inputs (ARIS screens, the ATM table, radiobear/JPL Uranus models,
MockSZ cubes, DESHIMA 2.0 data) are not available; these inputs stand in for them
("Input recipe").  Everything is float64 NumPy math from `default_rng(seed)`,
stored as float32 where the boundary takes float32.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import List, Optional, Tuple, Union

import numpy as np

H_PLANCK = 6.62607015e-34
K_BOLTZ = 1.380649e-23
C_LIGHT = 299792458.0
ARCSEC = np.pi / 180.0 / 3600.0

F_SAMPLE_DESHIMA = 2e9 / 2 ** 19 / 24      # PAPER.md:243, ~158.9457 Hz (configs use 160 Hz)


# --------------------------------------------------------------------------------------
# containers
# --------------------------------------------------------------------------------------
@dataclass
class Stage:
    """One optical stage k >= 1 of the cascade (Eq. 12)."""
    eta: Union[float, np.ndarray]          # scalar or float32 [n_freq]
    T_K: float
    couple_atmosphere: bool = False
    name: str = ""


@dataclass
class Workload:
    name: str
    # frequency grid
    n_freq: int
    nu0_hz: float
    dnu_hz: float
    # sampling / scan
    n_samples: int
    f_sample_hz: float
    az_rad: np.ndarray
    el_rad: np.ndarray
    el0_rad: float
    # spaxels
    daz_rad: np.ndarray
    del_rad: np.ndarray
    # source cube [n_el][n_az][n_freq] (None = blank sky)
    cube: Optional[np.ndarray]
    az_min_rad: float
    daz_grid_rad: float
    el_min_rad: float
    del_grid_rad: float
    # front end
    eta_front_nu: Optional[np.ndarray]
    T_cmb_K: float
    # screen
    screen: np.ndarray
    dx_m: float
    dy_m: float
    h_column_m: float
    wind_mps: float
    pwv0_a_mm: float
    pwv0_b_mm_per_s: float
    # LUT
    atm_lut: np.ndarray
    lut_nu0_hz: float
    lut_dnu_hz: float
    lut_pwv0_mm: float
    lut_dpwv_mm: float
    T_atm_K: float
    # cascade
    stages: List[Stage]
    # filterbank
    filt: np.ndarray
    f_center_hz: np.ndarray
    dnu_eff_hz: Optional[np.ndarray] = None
    # noise
    seed: int = 0
    photon_noise: bool = False
    pink_noise: bool = False
    # 0: north_star's narrow-band photon noise (R17); 1: the paper's Eq. 17 with the generation-
    # recombination term 2 Delta_Al / eta_pb (Delta_Al = 188 micro-eV, eta_pb = 0.4) (R23)
    photon_mode: int = 0
    kid_gap_J: float = 188e-6 * 1.602176634e-19
    eta_pb: float = 0.4
    pink_method: int = 0                   # 0: AR(1) cascade (north_star), 1: Timmer & Koenig FFT
    pink_A: Optional[np.ndarray] = None
    pink_alpha: Optional[np.ndarray] = None
    pink_f_corner_hz: Optional[np.ndarray] = None
    # output unit: 0 = detected power [W], 1 = brightness temperature [K] through the linear map of a
    # simulated skydip over skydip_n PWV values in [skydip_pwv_lo_mm, skydip_pwv_hi_mm] (R22)
    output_unit: int = 0
    skydip_n: int = 16
    skydip_pwv_lo_mm: float = 0.5
    skydip_pwv_hi_mm: float = 1.5
    # streaming
    chunk_samples: int = 0
    # global index of spaxel 0 when the workload holds a sub-range of an instrument's spaxels (RNG counter word 1)
    spaxel_index_base: int = 0

    # derived sizes
    @property
    def n_spaxel(self) -> int:
        return int(self.daz_rad.shape[0])

    @property
    def n_chan(self) -> int:
        return int(self.filt.shape[0])

    @property
    def nu_hz(self) -> np.ndarray:
        return self.nu0_hz + self.dnu_hz * np.arange(self.n_freq)

    def replace(self, **kw) -> "Workload":
        return dataclasses.replace(self, **kw)

    def detector_samples(self) -> int:
        return self.n_samples * self.n_spaxel * self.n_chan


# --------------------------------------------------------------------------------------
# instrument pieces
# --------------------------------------------------------------------------------------
def frequency_grid(n_freq: int, lo_hz: float = 200e9, hi_hz: float = 460e9) -> Tuple[float, float]:
    """Uniform grid, both ends included; wider than the channels so that the Lorentzian
    tails are covered, as the paper does."""
    return lo_hz, (hi_hz - lo_hz) / (n_freq - 1)


def channel_centres_log(n_chan: int, f_lo_hz: float = 220e9, octaves: float = 1.0) -> np.ndarray:
    """f_c = f_lo * 2^(c/(n_chan-1)) (log-spaced over `octaves`)."""
    if n_chan == 1:
        return np.array([f_lo_hz])
    return f_lo_hz * 2.0 ** (octaves * np.arange(n_chan) / (n_chan - 1))


def channel_count_half_power(f_lo_hz: float, f_hi_hz: float, R: float) -> int:
    """Number of channels when adjacent Lorentzians overlap at half power, f_{c+1} =
    f_c (1 + 1/R) (90-180 GHz, R = 20 -> 15 channels)."""
    return int(np.ceil(np.log(f_hi_hz / f_lo_hz) / np.log1p(1.0 / R)))


def lorentzian_filterbank(nu_hz: np.ndarray, f_c_hz: np.ndarray, R: float,
                          eta_peak: float = 0.16) -> np.ndarray:
    """Eq. 6 with the '1 +' restored in the denominator (reading R1):
    eta_filt(f, nu) = eta_peak / (1 + 4 R^2 (nu/f - 1)^2); FWHM = f/R."""
    x = nu_hz[None, :] / f_c_hz[:, None] - 1.0
    return (eta_peak / (1.0 + 4.0 * R * R * x * x)).astype(np.float32)


def filterbank_upstream_absorption(nu_hz: np.ndarray, f_c_hz: np.ndarray, R: float,
                                   eta_peak: Union[float, np.ndarray] = 0.16) -> np.ndarray:
    """Eq. 7: channels on a common transmission line, highest frequency first; a channel sees
    the signal from which the channels upstream (f_bar > f) have already absorbed their share:
        eta_filt(f, nu) = (eta_peak(f) - sum_{f_bar > f} eta_filt(f_bar, nu)) / (1 + 4 R^2 (nu/f - 1)^2)
    (the '1 +' restored as in Eq. 6, reading R1).  Evaluated literally, in descending order of f; rows are
    returned in the order of `f_c_hz`.  The hot path only sees the resulting matrix."""
    f_c_hz = np.asarray(f_c_hz, dtype=np.float64)
    peak = np.broadcast_to(np.asarray(eta_peak, dtype=np.float64), f_c_hz.shape)
    order = np.argsort(-f_c_hz, kind="stable")
    out = np.zeros((f_c_hz.size, nu_hz.size), dtype=np.float64)
    absorbed = np.zeros(nu_hz.size, dtype=np.float64)              # sum over the channels upstream
    for k in order:
        x = nu_hz / f_c_hz[k] - 1.0
        out[k] = (peak[k] - absorbed) / (1.0 + 4.0 * R * R * x * x)
        absorbed = absorbed + out[k]
    return out.astype(np.float32)


def hex_spaxels(R_hex: int, pitch_rad: float) -> Tuple[np.ndarray, np.ndarray]:
    """Packed hexagon of circumradius R_hex spaxels: 1 + 3R(R+1)
    offsets, axial coordinates (j outer, i inner), one lattice axis along azimuth."""
    daz, de = [], []
    for j in range(-R_hex, R_hex + 1):
        for i in range(-R_hex, R_hex + 1):
            if abs(i + j) <= R_hex:
                daz.append(pitch_rad * (i + 0.5 * j))
                de.append(pitch_rad * (np.sqrt(3.0) / 2.0) * j)
    return np.asarray(daz, dtype=np.float64), np.asarray(de, dtype=np.float64)


# --------------------------------------------------------------------------------------
# cascade helpers (plan-time efficiencies, Sect. 2.3/2.5)
# --------------------------------------------------------------------------------------
def eta_ruze(nu_hz: np.ndarray, rms_m: float) -> np.ndarray:
    """Eq. 5 read as exp(-(4 pi rho / lambda)^2) (reading R2)."""
    lam = C_LIGHT / nu_hz
    return np.exp(-(4.0 * np.pi * rms_m / lam) ** 2)


def eta_ohmic(nu_hz: np.ndarray, eps_ref: float = 0.0025, nu_ref_hz: float = 840e9) -> np.ndarray:
    """Eq. 13, aluminium reflector."""
    return 1.0 - eps_ref * np.sqrt(nu_hz / nu_ref_hz)


def eta_dielectric_bulk(nu_hz: np.ndarray, d_m: float, n: float, tan_delta: float) -> np.ndarray:
    """Eq. 14."""
    lam = C_LIGHT / nu_hz
    return np.exp(-2.0 * np.pi * d_m * n * tan_delta / lam)


def eta_dielectric_surface(n: float) -> float:
    """Eq. 15."""
    return 1.0 - ((1.0 - n) / (1.0 + n)) ** 2


def refractive_stage(nu_hz, d_m, n, tan_delta, T_K, T_ambient_K=None, ar_coated=False, name=""):
    """A refractive stage = surface, bulk, surface applications of Eq. 12;
    AR coating drops the two surface stages."""
    bulk = Stage(eta_dielectric_bulk(nu_hz, d_m, n, tan_delta).astype(np.float32), T_K, False, name + ":bulk")
    if ar_coated:
        return [bulk]
    Ta = T_K if T_ambient_K is None else T_ambient_K
    surf = eta_dielectric_surface(n)
    return [Stage(surf, Ta, False, name + ":in"), bulk, Stage(surf, Ta, False, name + ":out")]


def cascade_tiny() -> List[Stage]:
    """Config 1: eta 0.9 / 0.95 / 0.8 at 270 / 280 / 4 K."""
    return [Stage(0.9, 270.0), Stage(0.95, 280.0), Stage(0.8, 4.0)]


def cascade_deshima8(nu_hz: np.ndarray) -> List[Stage]:
    """Eight optical stages after PAPER.md Table 1 (:259-274)."""
    ohm = eta_ohmic(nu_hz).astype(np.float32)
    st = [
        Stage(0.99, 273.0, False, "primary spillover"),
        Stage(ohm, 273.0, False, "primary Ohmic-Al"),
        Stage(ohm.copy(), 273.0, False, "secondary Ohmic-Al"),
        Stage(0.85, 273.0, True, "secondary spillover -> atmosphere"),
        Stage(0.99, 290.0, False, "warm optics spillover"),
    ]
    st += refractive_stage(nu_hz, 4e-3, 3.41, 1e-4, 290.0, ar_coated=True, name="cryostat window")
    st += [Stage(0.65, 4.0, False, "low-pass filterstack"), Stage(0.7, 4.0, False, "leaky lens")]
    return st


def eta_front_aste(nu_hz: np.ndarray, eta_t=0.85, rms_m=42e-6, eta_pol=0.5) -> np.ndarray:
    """eta_t * eta_surf * eta_pol of Eq. 11."""
    return (eta_t * eta_ruze(nu_hz, rms_m) * eta_pol).astype(np.float32)


# --------------------------------------------------------------------------------------
# atmosphere
# --------------------------------------------------------------------------------------
def kolmogorov_screen(n: int, seed: int, mean_mm: float = 1.0, rms_frac: float = 0.01) -> np.ndarray:
    """Periodic n x n PWV screen: FFT of seeded white noise shaped by k^(-11/6) (k = 0
    removed), normalised to zero mean / unit std g, PWV = mean (1 + rms_frac g).
    Stands in for an ARIS screen."""
    rng = np.random.default_rng(seed)
    white = rng.standard_normal((n, n))
    k1 = np.fft.fftfreq(n)
    kk = np.hypot(k1[:, None], k1[None, :])
    kk[0, 0] = 1.0
    amp = kk ** (-11.0 / 6.0)
    amp[0, 0] = 0.0
    g = np.fft.ifft2(np.fft.fft2(white) * amp).real
    g = (g - g.mean()) / g.std()
    return (mean_mm * (1.0 + rms_frac * g)).astype(np.float32)


ATM_LINES_GHZ = (183.0, 325.0, 380.0, 448.0, 557.0)
ATM_LINE_STRENGTH = (2.0, 1.5, 20.0, 10.0, 500.0)
ATM_LINE_GAMMA_GHZ = 3.0


def tau_per_mm(nu_hz: np.ndarray) -> np.ndarray:
    """Made-up but plausible zenith opacity per mm PWV: a nu^2 continuum plus Lorentzian
    water lines at 183/325/380/448/557 GHz (BASELINE.json config 3)."""
    g = nu_hz / 1e9
    tau = 0.05 * (g / 300.0) ** 2
    for f0, s in zip(ATM_LINES_GHZ, ATM_LINE_STRENGTH):
        tau = tau + s * ATM_LINE_GAMMA_GHZ ** 2 / ((g - f0) ** 2 + ATM_LINE_GAMMA_GHZ ** 2)
    return tau


def atm_lut(nu_lo_hz=190e9, nu_step_hz=0.1e9, n_nu=2801, pwv_lo=0.1, pwv_step=0.05, n_pwv=79):
    """eta_atm,z(nu, PWV) = exp(-tau(nu) PWV) on a (PWV, nu) grid; stands in for the ATM
    table.  Returns (lut[n_pwv][n_nu] float32, nu0, dnu, pwv0, dpwv)."""
    nu = nu_lo_hz + nu_step_hz * np.arange(n_nu)
    pwv = pwv_lo + pwv_step * np.arange(n_pwv)
    lut = np.exp(-tau_per_mm(nu)[None, :] * pwv[:, None]).astype(np.float32)
    return lut, nu_lo_hz, nu_step_hz, pwv_lo, pwv_step


# --------------------------------------------------------------------------------------
# sources
# --------------------------------------------------------------------------------------
def _jn_power(nu_hz, T_K):
    """h nu / expm1(h nu / k T): used only to give synthetic cubes a thermal spectrum."""
    with np.errstate(over="ignore", divide="ignore", invalid="ignore"):
        x = H_PLANCK * nu_hz / (K_BOLTZ * np.maximum(T_K, 1e-300))
        out = H_PLANCK * nu_hz / np.expm1(x)
    return np.where(T_K > 0, out, 0.0)


def blob_cube(nu_hz, n_pix, half_extent_rad, n_blob, seed, sigma_range_rad, peak_range_K,
              clip_K=50.0, pol_factor=2.0):
    """[n_pix][n_pix][n_freq] cube: T_b(az, el) = sum of seeded Gaussian blobs (clipped),
    cube value pol_factor * JN(nu, T_b) (beam filling)."""
    rng = np.random.default_rng(seed)
    ax = np.linspace(-half_extent_rad, half_extent_rad, n_pix)
    cx = rng.uniform(-0.8 * half_extent_rad, 0.8 * half_extent_rad, n_blob)
    cy = rng.uniform(-0.8 * half_extent_rad, 0.8 * half_extent_rad, n_blob)
    sg = rng.uniform(sigma_range_rad[0], sigma_range_rad[1], n_blob)
    pk = rng.uniform(peak_range_K[0], peak_range_K[1], n_blob)
    Tb = np.zeros((n_pix, n_pix))
    for b in range(n_blob):
        r2 = (ax[None, :] - cx[b]) ** 2 + (ax[:, None] - cy[b]) ** 2
        Tb += pk[b] * np.exp(-0.5 * r2 / sg[b] ** 2)
    Tb = np.minimum(Tb, clip_K)
    cube = np.empty((n_pix, n_pix, nu_hz.size), dtype=np.float32)
    for j in range(n_pix):                                  # row by row: bounded temporaries
        cube[j] = (pol_factor * _jn_power(nu_hz[None, :], Tb[j][:, None])).astype(np.float32)
    grid0 = -half_extent_rad
    dgrid = 2.0 * half_extent_rad / (n_pix - 1)
    return cube, grid0, dgrid


def single_blob_cube(nu_hz, n_pix=16, half_extent_rad=60 * ARCSEC, T_b=20.0, sigma_rad=20 * ARCSEC):
    """Config 1: one centred Gaussian blob."""
    ax = np.linspace(-half_extent_rad, half_extent_rad, n_pix)
    Tb = T_b * np.exp(-0.5 * (ax[None, :] ** 2 + ax[:, None] ** 2) / sigma_rad ** 2)
    cube = _jn_power(nu_hz[None, None, :], Tb[:, :, None]).astype(np.float32)
    return cube, -half_extent_rad, 2.0 * half_extent_rad / (n_pix - 1)


def uranus_cube(nu_hz, n_pix=55, half_extent_rad=70 * ARCSEC, T_disk=120.0,
                disk_diam_rad=3.5 * ARCSEC, dish_m=10.0):
    """Configs 2/3: a 120 K disk already convolved with a Gaussian beam of FWHM
    1.2 lambda / D on a 0 K sky (PAPER.md:307-312 grid): both polarisations, RJ law."""
    ax = np.linspace(-half_extent_rad, half_extent_rad, n_pix)
    rho2 = ax[None, :] ** 2 + ax[:, None] ** 2
    fwhm = 1.2 * (C_LIGHT / nu_hz) / dish_m
    omega_a = np.pi * fwhm ** 2 / (4.0 * np.log(2.0))
    omega_d = np.pi * (0.5 * disk_diam_rad) ** 2
    peak = 2.0 * K_BOLTZ * T_disk * omega_d / omega_a
    cube = (peak[None, None, :] * np.exp(-4.0 * np.log(2.0) * rho2[:, :, None] / fwhm[None, None, :] ** 2))
    return cube.astype(np.float32), -half_extent_rad, 2.0 * half_extent_rad / (n_pix - 1)


# --------------------------------------------------------------------------------------
# scan patterns (relative to the scan centre)
# --------------------------------------------------------------------------------------
def scan_stare(n: int):
    return np.zeros(n), np.zeros(n)


def scan_daisy(n: int, f_s: float, r_petal_rad=65 * ARCSEC, omega=2 * np.pi * 1.54, Omega=None):
    """Eq. 8 with the parameters of PAPER.md:312."""
    Omega = omega / 50.0 if Omega is None else Omega
    t = np.arange(n, dtype=np.float64) / f_s
    return (r_petal_rad * np.cos(Omega * t) * np.sin(omega * t),
            r_petal_rad * np.sin(Omega * t) * np.sin(omega * t))


def scan_raster(n: int, f_s: float, half_rad=60 * ARCSEC, period_s=2.0):
    """Config 1: azimuth triangle wave +-half with the given period, elevation ramp
    -half -> +half over the observation."""
    t = np.arange(n, dtype=np.float64) / f_s
    ph = (t / period_s) % 1.0
    az = half_rad * (4.0 * np.abs(ph - 0.5) - 1.0)
    el = half_rad * (2.0 * np.arange(n) / max(n - 1, 1) - 1.0)
    return az, el


def scan_chop_nod(n: int, throw_rad=240 * ARCSEC, chop_samples=8, nod_samples=9600):
    """Config 2: ON-OFF.  chop state (n // 8) & 1 (10 Hz at 160 Hz), nod state
    (n // 9600) & 1 flips the throw sign."""
    idx = np.arange(n, dtype=np.int64)
    chop = (idx // chop_samples) & 1
    nod = (idx // nod_samples) & 1
    az = throw_rad * chop * np.where(nod == 1, -1.0, 1.0)
    return az.astype(np.float64), np.zeros(n)


# --------------------------------------------------------------------------------------
# pink-noise levels
# --------------------------------------------------------------------------------------
def pink_levels(n_det: int, seed: int, f_knee_hz=0.1, alpha=1.0, nep_ref=8e-18):
    """A_d = NEP_d^2 f_knee^alpha with a seeded per-detector NEP_d = nep_ref (0.5 + u),
    nep_ref ~ photon NEP of a DESHIMA-like channel (PAPER.md:243 takes A, alpha from
    measurements that are not available here)."""
    rng = np.random.default_rng(seed + 7919)
    nep = nep_ref * (0.5 + rng.random(n_det))
    return nep ** 2 * f_knee_hz ** alpha, np.full(n_det, alpha)


PINK_CORNERS_DEFAULT = np.array([2.0, 0.2, 0.02, 0.002])


# --------------------------------------------------------------------------------------
# the five configs of BASELINE.json
# --------------------------------------------------------------------------------------
_SCREEN_CACHE = {}


def _screen(n, seed):
    key = (n, seed)
    if key not in _SCREEN_CACHE:
        _SCREEN_CACHE[key] = kolmogorov_screen(n, seed)
    return _SCREEN_CACHE[key]


def make_workload(cfg: str, n_samples: Optional[int] = None, n_freq: Optional[int] = None,
                  n_chan: Optional[int] = None, screen_n: Optional[int] = None,
                  cube_n: Optional[int] = None, photon_noise: Optional[bool] = None,
                  pink_noise: Optional[bool] = None) -> Workload:
    """Build config "C1".."C5" (BASELINE.json configs[0..4]).  The optional arguments
    shrink a config for tests; None keeps the configured size."""
    cfg = cfg.upper()
    f_s = 160.0
    lut, lnu0, ldnu, lp0, ldp = atm_lut()
    common = dict(f_sample_hz=f_s, dx_m=0.2, dy_m=0.2, h_column_m=1537.0, wind_mps=10.0,
                  pwv0_a_mm=0.0, pwv0_b_mm_per_s=0.0, atm_lut=lut, lut_nu0_hz=lnu0,
                  lut_dnu_hz=ldnu, lut_pwv0_mm=lp0, lut_dpwv_mm=ldp, T_atm_K=273.0)

    if cfg == "C1":
        nf = n_freq or 512; nc = n_chan or 64; nt = n_samples or 1000
        nu0, dnu = frequency_grid(nf); nu = nu0 + dnu * np.arange(nf)
        fc = channel_centres_log(nc)
        cube, g0, dg = single_blob_cube(nu, n_pix=cube_n or 16)
        az, el = scan_raster(nt, f_s)
        daz, de = hex_spaxels(0, 8 * ARCSEC)
        return Workload(name="C1", n_freq=nf, nu0_hz=nu0, dnu_hz=dnu, n_samples=nt, az_rad=az, el_rad=el,
                        el0_rad=np.deg2rad(60.0), daz_rad=daz, del_rad=de, cube=cube, az_min_rad=g0,
                        daz_grid_rad=dg, el_min_rad=g0, del_grid_rad=dg, eta_front_nu=None, T_cmb_K=0.0,
                        screen=_screen(screen_n or 256, 0), stages=cascade_tiny(),
                        filt=lorentzian_filterbank(nu, fc, 300.0), f_center_hz=fc, seed=0,
                        photon_noise=bool(photon_noise), pink_noise=bool(pink_noise), **common)

    nc = n_chan or 347
    fc = channel_centres_log(nc)
    if cfg in ("C2", "C3"):
        nf = n_freq or 3000
        nu0, dnu = frequency_grid(nf); nu = nu0 + dnu * np.arange(nf)
        cube, g0, dg = uranus_cube(nu, n_pix=cube_n or 55)
        if cfg == "C2":
            nt = n_samples or 96000
            az, el = scan_chop_nod(nt)
            daz, de = hex_spaxels(0, 8 * ARCSEC)
            seed, ph, pk = 1, False, False
        else:
            nt = n_samples or 576000
            az, el = scan_daisy(nt, f_s)
            daz, de = hex_spaxels(1, 8 * ARCSEC)
            seed, ph, pk = 2, True, False
    elif cfg in ("C4", "C5"):
        nf = n_freq or 4000
        nu0, dnu = frequency_grid(nf); nu = nu0 + dnu * np.arange(nf)
        if cfg == "C4":
            nt = n_samples or 160000
            npx = cube_n or 128
            half = 0.5 * (npx - 1) * 3.5 * ARCSEC
            cube, g0, dg = blob_cube(nu, npx, half, 32, 1, (5 * ARCSEC, 30 * ARCSEC), (0.0, 50.0))
            daz, de = hex_spaxels(4, 8 * ARCSEC)
            seed = 3
        else:
            nt = n_samples or 576000
            cube, g0, dg = blob_cube(nu, cube_n or 61, 210 * ARCSEC, 32, 1,
                                     (5 * ARCSEC, 30 * ARCSEC), (0.0, 50.0))
            daz, de = hex_spaxels(3, 8 * ARCSEC)
            seed = 4
            common.update(pwv0_a_mm=-0.5, pwv0_b_mm_per_s=1.0 / 3600.0)
            common["chunk_samples"] = 9600          # 60 s chunks
        az, el = scan_daisy(nt, f_s)
        ph, pk = True, True
    else:
        raise ValueError(f"unknown config {cfg!r}")

    ph = ph if photon_noise is None else photon_noise
    pk = pk if pink_noise is None else pink_noise
    pink = {}
    if pk:
        A, alpha = pink_levels(daz.size * nc, seed)
        pink = dict(pink_A=A, pink_alpha=alpha, pink_f_corner_hz=PINK_CORNERS_DEFAULT.copy())
    return Workload(name=cfg, n_freq=nf, nu0_hz=nu0, dnu_hz=dnu, n_samples=nt, az_rad=az, el_rad=el,
                    el0_rad=np.deg2rad(47.8), daz_rad=daz, del_rad=de, cube=cube, az_min_rad=g0,
                    daz_grid_rad=dg, el_min_rad=g0, del_grid_rad=dg, eta_front_nu=eta_front_aste(nu),
                    T_cmb_K=2.725, screen=_screen(screen_n or 4096, 0), stages=cascade_deshima8(nu),
                    filt=lorentzian_filterbank(nu, fc, 500.0), f_center_hz=fc, seed=seed,
                    photon_noise=ph, pink_noise=pk, **pink, **common)


# --------------------------------------------------------------------------------------
# small random workloads for parity / invariant tests
# --------------------------------------------------------------------------------------
def random_workload(seed: int, n_samples=64, n_spaxel=3, n_chan=24, n_freq=96, n_stage=4,
                    screen_n=32, cube_n=6, n_pwv=7, n_nu_lut=41, couple=True,
                    with_cube=True, photon_noise=False, pink_noise=False, J=4) -> Workload:
    """Unstructured random inputs with valid ranges: exercises every term of the chain
    (per-frequency and scalar stages, an atmosphere-coupled stage, rows inside and
    outside the cube, PWV inside and outside the LUT, screen wrap-around)."""
    rng = np.random.default_rng(seed)
    nu0, dnu = 210e9, 230e9 / max(n_freq - 1, 1)
    nu = nu0 + dnu * np.arange(n_freq)
    lnu0 = nu0 - 3.3e9
    ldnu = (nu[-1] + 2.9e9 - lnu0) / (n_nu_lut - 1)
    lp0, ldp = 0.3, 0.25
    tau = 0.05 + 1.5 * rng.random(n_nu_lut)
    lut = np.exp(-tau[None, :] * (lp0 + ldp * np.arange(n_pwv))[:, None]).astype(np.float32)
    screen = (1.0 + 0.5 * rng.random((screen_n, screen_n))).astype(np.float32)   # 1..1.5 mm
    half = 40 * ARCSEC
    cube = None
    if with_cube:
        cube = (K_BOLTZ * 40.0 * rng.random((cube_n, cube_n, n_freq))).astype(np.float32)
    az = rng.uniform(-1.4 * half, 1.4 * half, n_samples)      # some rows leave the cube
    el = rng.uniform(-1.4 * half, 1.4 * half, n_samples)
    daz = rng.uniform(-10 * ARCSEC, 10 * ARCSEC, n_spaxel)
    de = rng.uniform(-10 * ARCSEC, 10 * ARCSEC, n_spaxel)
    stages = []
    for k in range(n_stage):
        eta = (0.6 + 0.4 * rng.random(n_freq)).astype(np.float32) if k % 2 else float(0.6 + 0.4 * rng.random())
        stages.append(Stage(eta, float(rng.uniform(3.0, 300.0)), bool(couple and k == 1)))
    fc = np.linspace(nu[0] + 10 * dnu, nu[-1] - 10 * dnu, n_chan)
    filt = (0.3 * rng.random((n_chan, n_freq)) ** 3).astype(np.float32)
    pink = {}
    if pink_noise:
        pink = dict(pink_A=1e-34 * (0.5 + rng.random(n_spaxel * n_chan)),
                    pink_alpha=rng.uniform(0.8, 1.3, n_spaxel * n_chan),
                    pink_f_corner_hz=2.0 * 10.0 ** (-np.arange(J, dtype=np.float64)))
    return Workload(name=f"rand{seed}", n_freq=n_freq, nu0_hz=nu0, dnu_hz=dnu, n_samples=n_samples,
                    f_sample_hz=160.0, az_rad=az, el_rad=el, el0_rad=np.deg2rad(55.0), daz_rad=daz,
                    del_rad=de, cube=cube, az_min_rad=-half, daz_grid_rad=2 * half / (cube_n - 1),
                    el_min_rad=-half, del_grid_rad=2 * half / (cube_n - 1),
                    eta_front_nu=(0.3 + 0.2 * rng.random(n_freq)).astype(np.float32), T_cmb_K=2.725,
                    screen=screen, dx_m=0.2, dy_m=0.25, h_column_m=1537.0, wind_mps=10.0,
                    pwv0_a_mm=-0.2, pwv0_b_mm_per_s=2.0, atm_lut=lut, lut_nu0_hz=lnu0, lut_dnu_hz=ldnu,
                    lut_pwv0_mm=lp0, lut_dpwv_mm=ldp, T_atm_K=273.0, stages=stages, filt=filt,
                    f_center_hz=fc, seed=seed * 1000003 + 17, photon_noise=photon_noise,
                    pink_noise=pink_noise, **pink)
