"""ctypes wrapper of the CPU ORACLE (oracle/gateau_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: imported only by tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs.  Nothing here touches the CUDA
path; it marshals a `Workload` (the shared seeded inputs) into the oracle's own struct.

The options of SURVEY rows f1-f4 are written here in NumPy, in double precision, each from the passage it cites
and each pinned in tests/test_oracle_*.py: Timmer & Koenig pink noise (pink_tk_series, R21),
the skydip and its Kelvin map (skydip, kelvin_map, R22), the exact NEP of Eq. 17 (nep2_exact, simulate_rows_exact,
R23), the screen and source pre-processing (footprint_weights, screen_line_of_sight, R24; far_field, beam_weights,
source_power, R25).  Parity unpinned: only the absolute physical realism of the synthetic inputs (out of scope).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gateau_oracle.cpp"
_LIB = _HERE / "libgateau_oracle.so"

CXXFLAGS = ["-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
            "-Wall", "-Wextra", "-shared", "-fPIC"]


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (building the checker is not using it)."""
    hdr = _HERE / "gateau_oracle.h"
    stale = (not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime
             or _LIB.stat().st_mtime < hdr.stat().st_mtime)
    if force or stale:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["g++", *CXXFLAGS, str(_SRC), "-o", str(tmp)])
        os.replace(tmp, _LIB)
    return _LIB


class GoStage(C.Structure):
    _fields_ = [("eta_nu", C.c_void_p), ("eta_scalar", C.c_double), ("T_K", C.c_double),
                ("couple_atmosphere", C.c_int32)]


class GoConfig(C.Structure):
    _fields_ = [
        ("n_freq", C.c_int32), ("nu0_hz", C.c_double), ("dnu_hz", C.c_double),
        ("n_samples", C.c_int64), ("f_sample_hz", C.c_double),
        ("az_rad", C.c_void_p), ("el_rad", C.c_void_p), ("el0_rad", C.c_double),
        ("n_spaxel", C.c_int32), ("daz_rad", C.c_void_p), ("del_rad", C.c_void_p),
        ("cube", C.c_void_p), ("n_az", C.c_int32), ("n_el", C.c_int32),
        ("az_min_rad", C.c_double), ("daz_grid_rad", C.c_double),
        ("el_min_rad", C.c_double), ("del_grid_rad", C.c_double),
        ("eta_front_nu", C.c_void_p), ("T_cmb_K", C.c_double),
        ("screen", C.c_void_p), ("nx", C.c_int32), ("ny", C.c_int32),
        ("dx_m", C.c_double), ("dy_m", C.c_double), ("h_column_m", C.c_double),
        ("wind_mps", C.c_double), ("pwv0_a_mm", C.c_double), ("pwv0_b_mm_per_s", C.c_double),
        ("atm_lut", C.c_void_p), ("n_pwv", C.c_int32), ("n_nu_lut", C.c_int32),
        ("lut_nu0_hz", C.c_double), ("lut_dnu_hz", C.c_double), ("lut_pwv0_mm", C.c_double),
        ("lut_dpwv_mm", C.c_double), ("T_atm_K", C.c_double),
        ("n_stage", C.c_int32), ("stages", C.c_void_p),
        ("n_chan", C.c_int32), ("filt", C.c_void_p),
        ("f_center_hz", C.c_void_p), ("dnu_eff_hz", C.c_void_p),
        ("seed", C.c_uint64), ("photon_noise", C.c_int32), ("pink_noise", C.c_int32),
        ("pink_A", C.c_void_p), ("pink_alpha", C.c_void_p),
        ("pink_n_stage", C.c_int32), ("pink_f_corner_hz", C.c_void_p),
    ]


GEOREC_DTYPE = np.dtype([
    ("n", "<i8"), ("iu0", "<i4"), ("iv0", "<i4"), ("ju", "<i4"), ("jv", "<i4"), ("ip", "<i4"),
    ("pad_", "<i4"), ("fu", "<f8"), ("fv", "<f8"), ("gu", "<f8"), ("gv", "<f8"), ("fp", "<f8"),
    ("pwv_mm", "<f8"), ("csc", "<f8")])

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.go_planck.restype = C.c_double
        L.go_planck.argtypes = [C.c_double, C.c_double]
        L.go_uniform.restype = C.c_double
        L.go_uniform.argtypes = [C.c_uint32]
        L.go_photon_sigma.restype = C.c_double
        L.go_photon_sigma.argtypes = [C.c_double] * 4
        L.go_philox4x32_10.restype = None
        L.go_normals4.restype = None
        L.go_photon_normal.restype = C.c_double
        L.go_photon_normal.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.go_normals4.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        for name in ("go_geometry", "go_row_spectrum", "go_simulate", "go_simulate_rows",
                     "go_pink_series", "go_num_threads"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


class Oracle:
    """The oracle bound to one Workload.  Keeps the marshalled arrays alive."""

    def __init__(self, w):
        self.w = w
        self.L = lib()
        k = self._keep = {}
        c = self.cfg = GoConfig()

        def ptr(name, arr):
            k[name] = arr
            return arr.ctypes.data

        c.n_freq, c.nu0_hz, c.dnu_hz = w.n_freq, w.nu0_hz, w.dnu_hz
        c.n_samples, c.f_sample_hz = w.n_samples, w.f_sample_hz
        c.az_rad, c.el_rad, c.el0_rad = ptr("az", _f64(w.az_rad)), ptr("el", _f64(w.el_rad)), w.el0_rad
        c.n_spaxel = w.n_spaxel
        c.daz_rad, c.del_rad = ptr("daz", _f64(w.daz_rad)), ptr("del", _f64(w.del_rad))
        if w.cube is not None:
            cube = _f32(w.cube)
            c.cube, c.n_el, c.n_az = ptr("cube", cube), cube.shape[0], cube.shape[1]
            assert cube.shape[2] == w.n_freq
        else:
            c.cube, c.n_el, c.n_az = None, 0, 0
        c.az_min_rad, c.daz_grid_rad = w.az_min_rad, w.daz_grid_rad
        c.el_min_rad, c.del_grid_rad = w.el_min_rad, w.del_grid_rad
        c.eta_front_nu = ptr("front", _f32(w.eta_front_nu)) if w.eta_front_nu is not None else None
        c.T_cmb_K = w.T_cmb_K
        scr = _f32(w.screen)
        c.screen, c.ny, c.nx = ptr("screen", scr), scr.shape[0], scr.shape[1]
        c.dx_m, c.dy_m, c.h_column_m, c.wind_mps = w.dx_m, w.dy_m, w.h_column_m, w.wind_mps
        c.pwv0_a_mm, c.pwv0_b_mm_per_s = w.pwv0_a_mm, w.pwv0_b_mm_per_s
        lut = _f32(w.atm_lut)
        c.atm_lut, c.n_pwv, c.n_nu_lut = ptr("lut", lut), lut.shape[0], lut.shape[1]
        c.lut_nu0_hz, c.lut_dnu_hz = w.lut_nu0_hz, w.lut_dnu_hz
        c.lut_pwv0_mm, c.lut_dpwv_mm, c.T_atm_K = w.lut_pwv0_mm, w.lut_dpwv_mm, w.T_atm_K
        st = (GoStage * max(len(w.stages), 1))()
        for i, s in enumerate(w.stages):
            if np.ndim(s.eta) == 0:
                st[i].eta_nu, st[i].eta_scalar = None, float(s.eta)
            else:
                st[i].eta_nu, st[i].eta_scalar = ptr(f"stage{i}", _f32(s.eta)), 0.0
            st[i].T_K, st[i].couple_atmosphere = float(s.T_K), int(bool(s.couple_atmosphere))
        k["stages"] = st
        c.n_stage, c.stages = len(w.stages), C.cast(st, C.c_void_p)
        filt = _f32(w.filt)
        assert filt.shape == (w.n_chan, w.n_freq)
        c.n_chan, c.filt = filt.shape[0], ptr("filt", filt)
        c.f_center_hz = ptr("fc", _f64(w.f_center_hz))
        c.dnu_eff_hz = ptr("dnueff", _f64(w.dnu_eff_hz)) if w.dnu_eff_hz is not None else None
        c.seed, c.photon_noise, c.pink_noise = int(w.seed), int(w.photon_noise), int(w.pink_noise)
        if w.pink_noise:
            c.pink_A, c.pink_alpha = ptr("pA", _f64(w.pink_A)), ptr("palpha", _f64(w.pink_alpha))
            fcn = _f64(w.pink_f_corner_hz)
            c.pink_n_stage, c.pink_f_corner_hz = fcn.size, ptr("pfc", fcn)
        else:
            c.pink_A = c.pink_alpha = c.pink_f_corner_hz = None
            c.pink_n_stage = 0

    def _chk(self, rc, what):
        if rc != 0:
            raise RuntimeError(f"oracle {what} failed with code {rc}")

    # ---- the path ----
    def geometry(self, t_begin=0, t_count=None):
        t_count = self.w.n_samples - t_begin if t_count is None else t_count
        out = np.zeros(t_count * self.w.n_spaxel, dtype=GEOREC_DTYPE)
        self._chk(self.L.go_geometry(C.byref(self.cfg), C.c_int64(t_begin), C.c_int64(t_count),
                                     C.c_void_p(out.ctypes.data)), "geometry")
        return out.reshape(t_count, self.w.n_spaxel)

    def row_spectrum(self, n, spaxel, intermediates=False):
        P = np.zeros(self.w.n_freq)
        eta = np.zeros(self.w.n_freq)
        S = np.zeros(self.w.n_freq)
        self._chk(self.L.go_row_spectrum(C.byref(self.cfg), C.c_int64(n), C.c_int32(spaxel),
                                         C.c_void_p(P.ctypes.data), C.c_void_p(eta.ctypes.data),
                                         C.c_void_p(S.ctypes.data)), "row_spectrum")
        return (P, eta, S) if intermediates else P

    def simulate(self, t_begin=0, t_count=None, want=("tod",)):
        """Returns a dict with the requested arrays among tod, pkid, pwv (float64)."""
        w = self.w
        t_count = w.n_samples - t_begin if t_count is None else t_count
        out = {}
        if "tod" in want:
            out["tod"] = np.zeros((t_count, w.n_spaxel, w.n_chan))
        if "pkid" in want:
            out["pkid"] = np.zeros((t_count, w.n_spaxel, w.n_chan))
        if "pwv" in want:
            out["pwv"] = np.zeros((t_count, w.n_spaxel))
        p = lambda key: C.c_void_p(out[key].ctypes.data) if key in out else None
        self._chk(self.L.go_simulate(C.byref(self.cfg), C.c_int64(t_begin), C.c_int64(t_count),
                                     p("tod"), p("pkid"), p("pwv")), "simulate")
        return out

    def simulate_rows(self, t_idx, s_idx, noise=False):
        t_idx = np.ascontiguousarray(t_idx, dtype=np.int64)
        s_idx = np.ascontiguousarray(s_idx, dtype=np.int32)
        pk = np.zeros((t_idx.size, self.w.n_chan))
        wn = np.zeros((t_idx.size, self.w.n_chan)) if noise else None
        self._chk(self.L.go_simulate_rows(C.byref(self.cfg), C.c_int64(t_idx.size),
                                          C.c_void_p(t_idx.ctypes.data), C.c_void_p(s_idx.ctypes.data),
                                          C.c_void_p(pk.ctypes.data),
                                          C.c_void_p(wn.ctypes.data) if noise else None), "simulate_rows")
        return (pk, wn) if noise else pk

    def pink_series(self, s_idx, c_idx, t_begin, t_count):
        s_idx = np.ascontiguousarray(s_idx, dtype=np.int32)
        c_idx = np.ascontiguousarray(c_idx, dtype=np.int32)
        out = np.zeros((s_idx.size, t_count))
        self._chk(self.L.go_pink_series(C.byref(self.cfg), C.c_int64(s_idx.size),
                                        C.c_void_p(s_idx.ctypes.data), C.c_void_p(c_idx.ctypes.data),
                                        C.c_int64(t_begin), C.c_int64(t_count),
                                        C.c_void_p(out.ctypes.data)), "pink_series")
        return out

    def pink_tk_series(self, s_idx, c_idx):
        """Pink noise by the method the paper itself uses (Timmer & Koenig 1995; R21):
        for detector (s, c) with one-sided PSD P(f) = A f^-alpha and N = n_samples, f_k = k f_s / N,
            X_0 = 0,  X_k = sqrt(P(f_k) f_s N / 4) (z0 + i z1)  (0 < k < N/2),  X_{N/2} = sqrt(P f_s N) z0  (N even),
        (z0, z1) = normals 0, 1 of Philox(seed; c0 = k, c1 = s, c2 = c, c3 = 3), and the series is the inverse real
        FFT x_n = irfft(X) (numpy convention, 1/N).  Returns [len(s_idx)][n_samples] in double."""
        w = self.w
        N = int(w.n_samples)
        K = N // 2
        out = np.zeros((len(s_idx), N))
        fk = np.arange(K + 1, dtype=np.float64) * (w.f_sample_hz / N)
        for i, (s, c) in enumerate(zip(s_idx, c_idx)):
            d = int(s) * w.n_chan + int(c)
            z = normals_bulk(w.seed, 0, K + 1, int(s), int(c), 3)
            X = np.zeros(K + 1, dtype=np.complex128)
            if K >= 1:
                P = np.zeros(K + 1)
                P[1:] = float(w.pink_A[d]) * fk[1:] ** (-float(w.pink_alpha[d]))
                X[1:] = np.sqrt(P[1:] * w.f_sample_hz * N / 4.0) * (z[1:, 0] + 1j * z[1:, 1])
                if N % 2 == 0:
                    X[K] = np.sqrt(P[K] * w.f_sample_hz * N) * z[K, 0]
            out[i] = np.fft.irfft(X, n=N) if N > 1 else 0.0
        return out

    # ---- exact photon noise, Eq. 17-19 (R23) ----
    def simulate_rows_exact(self, t_idx, s_idx):
        """For the rows (t_idx[i], s_idx[i]): noiseless P_KID [i][c] (Eq. 16) and the white-noise draw
        P_wn = sigma z [i][c], sigma from Eq. 17-18 on the row's own spectrum, z = normal 0 of
        Philox(seed; n, spaxel, channel, 0) as in the narrow-band mode."""
        w = self.w
        F = np.asarray(w.filt, dtype=np.float64)
        nu = w.nu_hz
        pk = np.zeros((len(t_idx), w.n_chan))
        wn = np.zeros((len(t_idx), w.n_chan))
        for i, (n, s) in enumerate(zip(t_idx, s_idx)):
            P_nu = self.row_spectrum(int(n), int(s))
            pk[i] = w.dnu_hz * (F @ P_nu)
            nep2 = nep2_exact(F, P_nu, nu, w.dnu_hz, w.kid_gap_J, w.eta_pb)
            sigma = np.sqrt(nep2 * 0.5 * w.f_sample_hz)                                  # Eq. 18
            z = np.array([photon_normal(w.seed, int(n), int(s), c) for c in range(w.n_chan)])
            wn[i] = sigma * z                                                            # Eq. 19
        return pk, wn

    # ---- brightness-temperature output (R22) ----
    def skydip(self):
        """The simulated skydip: a blank-sky stare of one on-axis detector row at the boresight elevation while
        the PWV takes skydip_n evenly spaced values in [lo, hi] (a flat zero screen plus the drift a + b t carries
        them), simulated noiseless with this oracle's own chain.  Returns (P_KID [k][c] in W, T_b [k][c] in K,
        pwv [k]);  T_b = sum_nu Fm T_los / sum_nu Fm,  T_los = (1 - eta_atm) T_atm + eta_atm T_cmb."""
        w = self.w
        K = int(w.skydip_n)
        step = (w.skydip_pwv_hi_mm - w.skydip_pwv_lo_mm) / (K - 1)
        sd = w.replace(n_samples=K, az_rad=np.zeros(K), el_rad=np.zeros(K), daz_rad=np.zeros(1), del_rad=np.zeros(1),
                       cube=None, screen=np.zeros((2, 2), dtype=np.float32), pwv0_a_mm=w.skydip_pwv_lo_mm,
                       pwv0_b_mm_per_s=step * w.f_sample_hz, photon_noise=False, pink_noise=False, output_unit=0,
                       pink_A=None, pink_alpha=None, pink_f_corner_hz=None, chunk_samples=0)
        o = Oracle(sd)
        res = o.simulate(want=("pkid", "pwv"))
        P = res["pkid"][:, 0, :]
        F = np.asarray(w.filt, dtype=np.float64)
        T = np.zeros((K, w.n_chan))
        for k in range(K):
            _, eta, _ = o.row_spectrum(k, 0, intermediates=True)
            T_los = (1.0 - eta) * w.T_atm_K + eta * w.T_cmb_K
            T[k] = (F @ T_los) / F.sum(axis=1)
        return P, T, res["pwv"][:, 0]

    def kelvin_map(self):
        """Least-squares line T_b = a_c + b_c P_KID per channel over the skydip ('a linear mapping
        is set up between P_KID^tot and T_b')."""
        P, T, _ = self.skydip()
        Pm, Tm = P.mean(axis=0), T.mean(axis=0)
        b = ((P - Pm) * (T - Tm)).sum(axis=0) / ((P - Pm) ** 2).sum(axis=0)
        a = Tm - b * Pm
        return a, b

    def dnu_eff(self):
        out = np.zeros(self.w.n_chan)
        self.L.go_dnu_eff(C.byref(self.cfg), C.c_void_p(out.ctypes.data))
        return out

    def pink_coeffs(self, spaxel, chan):
        J = self.cfg.pink_n_stage
        phi, g = np.zeros(J), np.zeros(J)
        self.L.go_pink_coeffs(C.byref(self.cfg), C.c_int32(spaxel), C.c_int32(chan),
                              C.c_void_p(phi.ctypes.data), C.c_void_p(g.ctypes.data))
        return phi, g


# ---- elementary pieces ----
def planck(nu_hz, T_K):
    return lib().go_planck(float(nu_hz), float(T_K))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xffffffff for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xffffffff for x in key])
    o = (C.c_uint32 * 4)()
    lib().go_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def uniform01(w):
    return lib().go_uniform(int(w) & 0xffffffff)


def normals4(seed, c0, c1, c2, c3):
    z = np.zeros(4)
    lib().go_normals4(int(seed), int(c0) & 0xffffffff, int(c1), int(c2), int(c3), C.c_void_p(z.ctypes.data))
    return z


def photon_normal(seed, n, s, ch):
    """The photon-noise normal of (sample n, spaxel s, channel ch) (R19): normal (ch div 32) mod 4 of the
    Philox block with counter (n, s, 32 (ch div 128) + ch mod 32, stream 0)."""
    return lib().go_photon_normal(int(seed), int(n) & 0xffffffff, int(s), int(ch))


def normals_bulk(seed, c0_begin, count, c1=0, c2=0, c3=0):
    z = np.zeros((count, 4))
    f = lib().go_normals_bulk
    f.restype = None
    f(C.c_uint64(int(seed)), C.c_uint32(int(c0_begin)), C.c_int64(count), C.c_uint32(c1),
      C.c_uint32(c2), C.c_uint32(c3), C.c_void_p(z.ctypes.data))
    return z


def photon_sigma(P_W, f_center_hz, dnu_eff_hz, f_sample_hz):
    return lib().go_photon_sigma(float(P_W), float(f_center_hz), float(dnu_eff_hz), float(f_sample_hz))


def nep2_exact(F, P_nu, nu_hz, dnu_hz, kid_gap_J, eta_pb):
    """Eq. 17, rectangle rule on the uniform grid (R16):
    NEP^2[c] = 2 sum_nu Fm[c][nu] P_nu (h nu + Fm[c][nu] P_nu + 2 Delta_Al / eta_pb) dnu."""
    h = 6.62607015e-34
    F = np.asarray(F, dtype=np.float64)
    FP = F * np.asarray(P_nu, dtype=np.float64)[None, :]
    return 2.0 * dnu_hz * np.sum(FP * (h * np.asarray(nu_hz)[None, :] + FP + 2.0 * kid_gap_J / eta_pb), axis=1)


def footprint_weights(dx_m, dy_m, R_tel_m, t_edge_db):
    """Aperture footprint on the screen grid (PAPER.md:92 with the illumination of Eq. 2 :76, R24):
    A(r) = 10^(-|t_edge| / 20 * r^2 / R_tel^2) inside r < R_tel (Gaussian, |t_edge| dB down at the rim), 0 outside,
    sampled at (i dx, j dy), normalised to unit sum.  Returns K[j + ry][i + rx]."""
    rx, ry = int(np.floor(R_tel_m / dx_m)), int(np.floor(R_tel_m / dy_m))
    K = np.zeros((2 * ry + 1, 2 * rx + 1))
    for j in range(-ry, ry + 1):
        for i in range(-rx, rx + 1):
            r2 = (i * dx_m) ** 2 + (j * dy_m) ** 2
            if r2 < R_tel_m ** 2:
                K[j + ry, i + rx] = 10.0 ** (-abs(t_edge_db) / 20.0 * r2 / R_tel_m ** 2)
    return K / K.sum()


def screen_line_of_sight(epl, dx_m, dy_m, R_tel_m, t_edge_db, pwv0_mm):
    """Eq. 4 and the footprint smoothing (:92) on a periodic screen (R7):
    PWV[y][x] = PWV_0 + (1 / 6.587) sum_{i,j} K[j][i] EPL[(y + j) mod ny][(x + i) mod nx]."""
    epl = np.asarray(epl, dtype=np.float64)
    K = footprint_weights(dx_m, dy_m, R_tel_m, t_edge_db)
    ry, rx = K.shape[0] // 2, K.shape[1] // 2
    acc = np.zeros_like(epl)
    for j in range(-ry, ry + 1):
        for i in range(-rx, rx + 1):
            if K[j + ry, i + rx] != 0.0:
                acc += K[j + ry, i + rx] * np.roll(epl, (-j, -i), axis=(0, 1))
    return pwv0_mm + acc / 6.587


def far_field(rho_rad, nu_hz, R_tel_m, t_edge_db):
    """Eq. 2-3 (R25): far-field power pattern of the circular aperture with the Gaussian
    illumination A(r) = 10^(-|t_edge|/20 r^2/R^2), r < R_tel, normalised to 1 on axis.  The 2-D Fourier transform of
    a circularly symmetric A is the Hankel transform: F(rho) = |int_0^R A(r) J0(2 pi r rho / lambda) r dr|^2 / F(0)."""
    from scipy import integrate, special
    lam = 299792458.0 / nu_hz
    k = abs(t_edge_db) / 20.0 * np.log(10.0) / R_tel_m ** 2
    g = lambda rho: integrate.quad(lambda r: np.exp(-k * r * r) * special.j0(2 * np.pi * r * rho / lam) * r,
                                   0.0, R_tel_m, epsabs=1e-13 * R_tel_m ** 2, epsrel=1e-11, limit=400)[0]
    g0 = g(0.0)
    rho = np.atleast_1d(np.asarray(rho_rad, dtype=np.float64))
    return np.array([(g(x) / g0) ** 2 for x in rho.ravel()]).reshape(rho.shape)


def beam_weights(nu_hz, daz_rad, del_rad, r_pix, R_tel_m, t_edge_db):
    """F sampled at the cube's pixel offsets (i daz, j del), |i|, |j| <= r_pix: W[j + r][i + r]."""
    off = np.arange(-r_pix, r_pix + 1)
    rho = np.hypot(off[None, :] * daz_rad, off[:, None] * del_rad)
    u, inv = np.unique(np.round(rho / 1e-15).astype(np.int64), return_inverse=True)
    return far_field(u * 1e-15, nu_hz, R_tel_m, t_edge_db)[inv].reshape(rho.shape)


def source_power(I_cube, nu_hz, daz_rad, del_rad, el_first_rad, r_pix, R_tel_m, t_edge_db):
    """Eq. 1 on the cube's grid, rectangle rule, zero intensity outside the cube (:137):
    P[j][i][nu] = A_p sum_{j',i'} I[j'][i'][nu] F_nu((i - i') daz, (j - j') del) cos(theta_j') daz del,
    A_p = pi R_tel^2, theta_j' = el_first + j' del, offsets limited to |i - i'|, |j - j'| <= r_pix."""
    I = np.asarray(I_cube, dtype=np.float64)
    n_el, n_az, n_f = I.shape
    cosw = np.cos(el_first_rad + del_rad * np.arange(n_el))[:, None]
    out = np.zeros_like(I)
    for f in range(n_f):
        W = beam_weights(nu_hz[f], daz_rad, del_rad, r_pix, R_tel_m, t_edge_db)
        src = I[:, :, f] * cosw
        pad = np.zeros((n_el + 2 * r_pix, n_az + 2 * r_pix))
        pad[r_pix:r_pix + n_el, r_pix:r_pix + n_az] = src
        acc = np.zeros((n_el, n_az))
        for dj in range(-r_pix, r_pix + 1):
            for di in range(-r_pix, r_pix + 1):
                # pixel (j, i) receives source pixel (j - dj, i - di) through F(di daz, dj del)
                acc += W[dj + r_pix, di + r_pix] * pad[r_pix - dj:r_pix - dj + n_el, r_pix - di:r_pix - di + n_az]
        out[:, :, f] = np.pi * R_tel_m ** 2 * daz_rad * del_rad * acc
    return out


def eta_zenith_at(w, f_hz, pwv_mm):
    """Zenith transmission eta_atm,z(f) of the workload's lookup table at frequencies f_hz and one PWV: bilinear on the
    table's own grid, PWV clamped to the table (R13) -- the per-channel transmission Eq. 25 starts from (PAPER.md:366:
    "the zenith PWV ... averaged over the entire observation and used to calculate eta_atm,z(f)")."""
    lut = np.asarray(w.atm_lut, dtype=np.float64)
    n_pwv, n_nu = lut.shape
    q = min(max((pwv_mm - w.lut_pwv0_mm) / w.lut_dpwv_mm, 0.0), n_pwv - 1.0)
    ip = min(int(np.floor(q)), n_pwv - 2)
    fp = q - ip
    r = (np.asarray(f_hz, dtype=np.float64) - w.lut_nu0_hz) / w.lut_dnu_hz
    ir = np.clip(np.floor(r).astype(int), 0, n_nu - 2)
    fr = r - ir
    row0 = (1 - fr) * lut[ip, ir] + fr * lut[ip, ir + 1]
    row1 = (1 - fr) * lut[ip + 1, ir] + fr * lut[ip + 1, ir + 1]
    return (1 - fp) * row0 + fp * row1


def common_mode_subtract(T_b, eta_z, csc, daz_rad, del_rad, r_out_rad):
    """Eq. 25-26, literally, in double.  T_b [t][spaxel][chan] brightness temperature, eta_z [chan]
    zenith transmission, csc [t][spaxel] = 1 / sin(elevation) (Eq. 10: eta_j(t,f) = eta_z(f)^csc_j(t)), spaxel offsets
    daz, del [spaxel]:
        S_j = 1 if sqrt(daz_j^2 + del_j^2) > r_out else 0,   N_out = sum_j S_j,
        T*_a,i = T_b,i / eta_i - (1 - eta_i) / (eta_i N_out) sum_j S_j T_b,j / (1 - eta_j).
    Returns (T*_a, S, common) with common[t][chan] = sum_j S_j T_b,j / (1 - eta_j)."""
    T_b = np.asarray(T_b, dtype=np.float64)
    eta = np.asarray(eta_z, dtype=np.float64)[None, None, :] ** np.asarray(csc, dtype=np.float64)[:, :, None]
    S = (np.sqrt(np.asarray(daz_rad, dtype=np.float64) ** 2 + np.asarray(del_rad, dtype=np.float64) ** 2) > r_out_rad).astype(np.float64)
    n_out = S.sum()
    if n_out < 1:
        raise ValueError("Eq. 25: no spaxel lies outside r_out")
    common = (S[None, :, None] * T_b / (1.0 - eta)).sum(axis=1)
    return T_b / eta - (1.0 - eta) / (eta * n_out) * common[:, None, :], S, common


def num_threads():
    return lib().go_num_threads()
