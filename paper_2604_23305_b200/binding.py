"""Thin ctypes binding of the C ABI in include/gateau_b200.h (libgateau_b200.so).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.
PyTorch is used for device memory and streams.  There is no CPU fallback: if the library
is missing it is built with nvcc, and if that fails, or no CUDA device is present, the
calls raise.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

GT_OK = 0
STATUS_NAMES = {0: "GT_OK", 1: "GT_ERR_NULL", 2: "GT_ERR_SHAPE", 3: "GT_ERR_VALUE", 4: "GT_ERR_RANGE",
                5: "GT_ERR_OOM", 6: "GT_ERR_CUDA", 7: "GT_ERR_UNSUPPORTED"}
VARIANT_DEFAULT, VARIANT_FP32, VARIANT_TENSOR, VARIANT_TENSOR_FULL = 0, 1, 2, 3

EXPORTS = ("gt_plan_create", "gt_simulate", "gt_plan_destroy", "gt_last_error", "gt_debug_geometry",
           "gt_debug_philox", "gt_debug_pkid", "gt_launch_count", "gt_variant_name", "gt_last_fused_ms",
           "gt_debug_kelvin_map", "gt_prepare_screen", "gt_prepare_source", "gt_plan_counters",
           "gt_pink_state_export", "gt_pink_state_import", "gt_debug_chunking", "gt_debug_timeline",
           "gt_measure_fp32_fma", "gt_common_mode_partial", "gt_common_mode_apply", "gt_release_cached_memory",
           "gt_common_mode_static", "gt_debug_corrections")


COMMON_MODE_STATIC_MAX = 2097152      # GT_COMMON_MODE_STATIC_MAX: floats of static device scratch (t_count * n_chan per call)


class GtStage(C.Structure):
    _fields_ = [("eta_nu", C.c_void_p), ("eta_scalar", C.c_double), ("T_K", C.c_double),
                ("couple_atmosphere", C.c_int32)]


class GtConfig(C.Structure):
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
        ("chunk_samples", C.c_int64),
        ("variant", C.c_int32),
        ("pink_method", C.c_int32),
        ("output_unit", C.c_int32), ("skydip_n", C.c_int32),
        ("skydip_pwv_lo_mm", C.c_double), ("skydip_pwv_hi_mm", C.c_double),
        ("photon_mode", C.c_int32), ("kid_gap_J", C.c_double), ("eta_pb", C.c_double),
        ("spaxel_index_base", C.c_int32),
    ]


GEOREC_DTYPE = np.dtype([
    ("n", "<i8"), ("iu0", "<i4"), ("iv0", "<i4"), ("ju", "<i4"), ("jv", "<i4"), ("ip", "<i4"),
    ("pad_", "<i4"), ("fu", "<f8"), ("fv", "<f8"), ("gu", "<f8"), ("gv", "<f8"), ("fp", "<f8"),
    ("pwv_mm", "<f8"), ("csc", "<f8")])

_lib = None


class GateauError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


def lib() -> C.CDLL:
    """Loads (building first if stale or missing) libgateau_b200.so.  Raises if it cannot."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        L.gt_plan_create.restype = C.c_int
        L.gt_plan_create.argtypes = [C.POINTER(GtConfig), C.c_void_p, C.POINTER(C.c_void_p)]
        L.gt_simulate.restype = C.c_int
        L.gt_simulate.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gt_debug_pkid.restype = C.c_int
        L.gt_debug_pkid.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        L.gt_plan_destroy.restype = C.c_int
        L.gt_plan_destroy.argtypes = [C.c_void_p]
        L.gt_last_error.restype = C.c_char_p
        L.gt_last_error.argtypes = [C.c_void_p]
        L.gt_debug_geometry.restype = C.c_int
        L.gt_debug_geometry.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
        L.gt_debug_philox.restype = C.c_int
        L.gt_debug_philox.argtypes = [C.c_uint64, C.c_uint32, C.c_int64, C.c_uint32, C.c_uint32, C.c_uint32,
                                      C.c_void_p]
        L.gt_launch_count.restype = C.c_int64
        L.gt_launch_count.argtypes = [C.c_void_p]
        L.gt_variant_name.restype = C.c_char_p
        L.gt_variant_name.argtypes = [C.c_void_p]
        L.gt_last_fused_ms.restype = C.c_double
        L.gt_last_fused_ms.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.gt_prepare_screen.restype = C.c_int
        L.gt_prepare_screen.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.gt_prepare_source.restype = C.c_int
        L.gt_prepare_source.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p]
        L.gt_debug_kelvin_map.restype = C.c_int
        L.gt_debug_kelvin_map.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.gt_plan_counters.restype = C.c_int
        L.gt_plan_counters.argtypes = [C.c_void_p] + [C.POINTER(C.c_int64)] * 4
        L.gt_debug_timeline.restype = C.c_int
        L.gt_debug_timeline.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_void_p]
        L.gt_measure_fp32_fma.restype = C.c_int
        L.gt_measure_fp32_fma.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.gt_common_mode_partial.restype = C.c_int
        L.gt_common_mode_partial.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double, C.c_double, C.c_void_p,
                                             C.POINTER(C.c_int32), C.c_void_p]
        L.gt_common_mode_apply.restype = C.c_int
        L.gt_common_mode_apply.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double, C.c_void_p, C.c_int32, C.c_void_p]
        L.gt_common_mode_static.restype = C.c_int
        L.gt_common_mode_static.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double, C.c_double,
                                            C.POINTER(C.c_int32), C.c_void_p]
        L.gt_debug_corrections.restype = C.c_int
        L.gt_debug_corrections.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.gt_release_cached_memory.restype = C.c_int
        L.gt_release_cached_memory.argtypes = []
        L.gt_debug_chunking.restype = C.c_int
        L.gt_debug_chunking.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.gt_pink_state_export.restype = C.c_int
        L.gt_pink_state_export.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
        L.gt_pink_state_import.restype = C.c_int
        L.gt_pink_state_import.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def fill_config(w, dev: dict, keep: dict, variant: int = VARIANT_DEFAULT, chunk_samples: Optional[int] = None) -> GtConfig:
    """Marshals a Workload into gt_config.  `dev` maps names to device pointers of the large
    fp32 arrays (cube, screen, atm_lut, filt, eta_front, stage<k>); `keep` receives the
    host arrays that must stay alive until gt_plan_create returns."""
    c = GtConfig()

    def hp(name, arr):
        keep[name] = arr
        return arr.ctypes.data

    c.n_freq, c.nu0_hz, c.dnu_hz = w.n_freq, w.nu0_hz, w.dnu_hz
    c.n_samples, c.f_sample_hz = w.n_samples, w.f_sample_hz
    c.az_rad, c.el_rad, c.el0_rad = hp("az", _f64(w.az_rad)), hp("el", _f64(w.el_rad)), w.el0_rad
    c.n_spaxel = w.n_spaxel
    c.daz_rad, c.del_rad = hp("daz", _f64(w.daz_rad)), hp("del", _f64(w.del_rad))
    if w.cube is not None:
        c.cube, c.n_el, c.n_az = dev["cube"], w.cube.shape[0], w.cube.shape[1]
    else:
        c.cube, c.n_el, c.n_az = None, 0, 0
    c.az_min_rad, c.daz_grid_rad = w.az_min_rad, w.daz_grid_rad
    c.el_min_rad, c.del_grid_rad = w.el_min_rad, w.del_grid_rad
    c.eta_front_nu = dev.get("eta_front") if w.eta_front_nu is not None else None
    c.T_cmb_K = w.T_cmb_K
    c.screen, c.ny, c.nx = dev["screen"], w.screen.shape[0], w.screen.shape[1]
    c.dx_m, c.dy_m, c.h_column_m, c.wind_mps = w.dx_m, w.dy_m, w.h_column_m, w.wind_mps
    c.pwv0_a_mm, c.pwv0_b_mm_per_s = w.pwv0_a_mm, w.pwv0_b_mm_per_s
    c.atm_lut, c.n_pwv, c.n_nu_lut = dev["atm_lut"], w.atm_lut.shape[0], w.atm_lut.shape[1]
    c.lut_nu0_hz, c.lut_dnu_hz = w.lut_nu0_hz, w.lut_dnu_hz
    c.lut_pwv0_mm, c.lut_dpwv_mm, c.T_atm_K = w.lut_pwv0_mm, w.lut_dpwv_mm, w.T_atm_K
    st = (GtStage * max(len(w.stages), 1))()
    for i, s in enumerate(w.stages):
        if np.ndim(s.eta) == 0:
            st[i].eta_nu, st[i].eta_scalar = None, float(s.eta)
        else:
            st[i].eta_nu, st[i].eta_scalar = dev[f"stage{i}"], 0.0
        st[i].T_K, st[i].couple_atmosphere = float(s.T_K), int(bool(s.couple_atmosphere))
    keep["stages"] = st
    c.n_stage, c.stages = len(w.stages), C.cast(st, C.c_void_p)
    c.n_chan, c.filt = w.n_chan, dev["filt"]
    c.f_center_hz = hp("fc", _f64(w.f_center_hz))
    c.dnu_eff_hz = hp("dnueff", _f64(w.dnu_eff_hz)) if w.dnu_eff_hz is not None else None
    c.seed, c.photon_noise, c.pink_noise = int(w.seed), int(w.photon_noise), int(w.pink_noise)
    if w.pink_noise:
        c.pink_A, c.pink_alpha = hp("pA", _f64(w.pink_A)), hp("palpha", _f64(w.pink_alpha))
        fcn = _f64(w.pink_f_corner_hz)
        c.pink_n_stage, c.pink_f_corner_hz = fcn.size, hp("pfc", fcn)
    else:
        c.pink_A = c.pink_alpha = c.pink_f_corner_hz = None
        c.pink_n_stage = 0
    c.chunk_samples = int(w.chunk_samples if chunk_samples is None else chunk_samples)
    c.variant = int(variant)
    c.pink_method = int(getattr(w, "pink_method", 0))
    c.output_unit = int(getattr(w, "output_unit", 0))
    c.skydip_n = int(getattr(w, "skydip_n", 16))
    c.skydip_pwv_lo_mm = float(getattr(w, "skydip_pwv_lo_mm", 0.5))
    c.skydip_pwv_hi_mm = float(getattr(w, "skydip_pwv_hi_mm", 1.5))
    c.photon_mode = int(getattr(w, "photon_mode", 0))
    c.kid_gap_J = float(getattr(w, "kid_gap_J", 188e-6 * 1.602176634e-19))
    c.eta_pb = float(getattr(w, "eta_pb", 0.4))
    c.spaxel_index_base = int(getattr(w, "spaxel_index_base", 0))
    return c


class Plan:
    """gt_plan bound to one Workload.  Uploads the workload's large arrays with torch (device
    memory only) and keeps them alive for the plan's lifetime."""

    def __init__(self, w, variant: int = VARIANT_DEFAULT, chunk_samples: Optional[int] = None, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise GateauError(6, "no CUDA device: the gateau_b200 path has no CPU fallback")
        self.torch = torch
        self.w = w
        self.L = lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._dev = {}
        ptrs = {}

        import time
        t_start = time.perf_counter()

        def up(name, arr):
            # a torch tensor (e.g. pinned host memory) is copied as it is; NumPy arrays go through from_numpy
            if isinstance(arr, torch.Tensor):
                t = arr.to(device=self.device, dtype=torch.float32, non_blocking=True).contiguous()
            else:
                t = torch.from_numpy(np.ascontiguousarray(arr, dtype=np.float32)).to(self.device)
            self._dev[name] = t
            ptrs[name] = t.data_ptr()

        if w.cube is not None:
            up("cube", w.cube)
        up("screen", w.screen)
        up("atm_lut", w.atm_lut)
        up("filt", w.filt)
        if w.eta_front_nu is not None:
            up("eta_front", w.eta_front_nu)
        for i, s in enumerate(w.stages):
            if np.ndim(s.eta) != 0:
                up(f"stage{i}", s.eta)
        torch.cuda.synchronize()
        t_up = time.perf_counter()
        keep = {}
        cfg = fill_config(w, ptrs, keep, variant, chunk_samples)
        self.handle = C.c_void_p()
        st = self.L.gt_plan_create(C.byref(cfg), None, C.byref(self.handle))
        if st != GT_OK:
            raise GateauError(st, self.L.gt_last_error(None).decode())
        self.upload_ms, self.create_ms = 1e3 * (t_up - t_start), 1e3 * (time.perf_counter() - t_up)

    # ---- helpers ----
    def _check(self, st):
        if st != GT_OK:
            raise GateauError(st, self.L.gt_last_error(self.handle).decode())

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream().cuda_stream)

    @property
    def variant_name(self) -> str:
        return self.L.gt_variant_name(self.handle).decode()

    @property
    def launch_count(self) -> int:
        return int(self.L.gt_launch_count(self.handle))

    def last_fused_ms(self):
        n = C.c_int32(0)
        ms = self.L.gt_last_fused_ms(self.handle, C.byref(n))
        return float(ms), int(n.value)

    def kelvin_map(self):
        """gt_debug_kelvin_map: (a [n_chan], b [n_chan]) of T_b = a + b P_KID, float64."""
        a, b = np.zeros(self.w.n_chan), np.zeros(self.w.n_chan)
        self._check(self.L.gt_debug_kelvin_map(self.handle, C.c_void_p(a.ctypes.data), C.c_void_p(b.ctypes.data)))
        return a, b

    def chunking(self):
        """gt_debug_chunking: (samples per launch for host output, for device output)."""
        h, d = C.c_int64(0), C.c_int64(0)
        self._check(self.L.gt_debug_chunking(self.handle, C.byref(h), C.byref(d)))
        return int(h.value), int(d.value)

    def timeline(self, capacity=4096):
        """gt_debug_timeline: [n_chunks, 4] ms = compute begin, compute end, copy begin, copy end of the last host-output call."""
        n = C.c_int32(0)
        ms = np.zeros((capacity, 4), dtype=np.float64)
        self._check(self.L.gt_debug_timeline(self.handle, capacity, C.byref(n), C.c_void_p(ms.ctypes.data)))
        return ms[:int(n.value)].copy()

    def common_mode_partial(self, tod_K, pwv_mean_mm, r_out_rad, t_begin=0):
        """gt_common_mode_partial: (partial [t, chan] CUDA tensor, this plan's N_out)."""
        t_count = int(tod_K.shape[0])
        partial = self.torch.empty((t_count, self.w.n_chan), dtype=self.torch.float32, device=self.device)
        n = C.c_int32(0)
        self._check(self.L.gt_common_mode_partial(self.handle, t_begin, t_count, _ptr(tod_K), float(pwv_mean_mm), float(r_out_rad),
                                                  _ptr(partial), C.byref(n), self._stream()))
        return partial, int(n.value)

    def common_mode_apply(self, tod_K, pwv_mean_mm, total, n_out_total, t_begin=0):
        """gt_common_mode_apply: tod_K <- T*_a (Eq. 25) in place."""
        self._check(self.L.gt_common_mode_apply(self.handle, t_begin, int(tod_K.shape[0]), _ptr(tod_K), float(pwv_mean_mm),
                                                _ptr(total), int(n_out_total), self._stream()))
        return tod_K

    def common_mode_static(self, tod_K, pwv_mean_mm, r_out_rad, t_begin=0):
        """gt_common_mode_static: tod_K <- T*_a (Eq. 25) in place, partial sums in the library's static device array
        (no allocation; t_count * n_chan <= COMMON_MODE_STATIC_MAX).  Returns (tod_K, N_out)."""
        n = C.c_int32(0)
        self._check(self.L.gt_common_mode_static(self.handle, t_begin, int(tod_K.shape[0]), _ptr(tod_K), float(pwv_mean_mm),
                                                 float(r_out_rad), C.byref(n), self._stream()))
        return tod_K, int(n.value)

    def corrections(self):
        """gt_debug_corrections: (blocks, blocks that skip the split's correction MMAs)."""
        a, b = C.c_int64(0), C.c_int64(0)
        self._check(self.L.gt_debug_corrections(self.handle, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def counters(self) -> dict:
        """gt_plan_counters: rows processed, rows outside the cube, PWV clamps below / above the LUT."""
        v = [C.c_int64(0) for _ in range(4)]
        self._check(self.L.gt_plan_counters(self.handle, *[C.byref(x) for x in v]))
        return dict(zip(("rows", "rows_outside_cube", "pwv_below_lut", "pwv_above_lut"), (int(x.value) for x in v)))

    def pink_state_export(self):
        """gt_pink_state_export: (state [n_spaxel * n_chan, J] float32, next_t)."""
        J = int(np.size(self.w.pink_f_corner_hz))
        st = np.zeros((self.w.n_spaxel * self.w.n_chan, J), dtype=np.float32)
        nt = C.c_int64(0)
        self._check(self.L.gt_pink_state_export(self.handle, C.c_void_p(st.ctypes.data), C.byref(nt)))
        return st, int(nt.value)

    def pink_state_import(self, state, next_t):
        st = np.ascontiguousarray(state, dtype=np.float32)
        self._check(self.L.gt_pink_state_import(self.handle, C.c_void_p(st.ctypes.data), int(next_t)))

    # ---- the three calls ----
    def simulate(self, t_begin=0, t_count=None, out=None, pwv_out=None, device_out=True, want_pwv=False):
        """gt_simulate.  `out`: a torch CUDA tensor, a pinned/pageable torch CPU tensor or a
        NumPy array of shape [t_count, n_spaxel, n_chan] float32; allocated when None."""
        torch, w = self.torch, self.w
        t_count = w.n_samples - t_begin if t_count is None else t_count
        if out is None:
            out = torch.empty((t_count, w.n_spaxel, w.n_chan), dtype=torch.float32,
                              device=self.device if device_out else "cpu", pin_memory=not device_out)
        if want_pwv and pwv_out is None:
            pwv_out = torch.empty((t_count, w.n_spaxel), dtype=torch.float32,
                                  device=self.device if device_out else "cpu", pin_memory=not device_out)
        self._check(self.L.gt_simulate(self.handle, t_begin, t_count, _ptr(out), _ptr(pwv_out), self._stream()))
        return (out, pwv_out) if want_pwv else out

    def pkid(self, t_begin=0, t_count=None, out=None):
        """gt_debug_pkid: noiseless Eq. 16 power for the same range."""
        torch, w = self.torch, self.w
        t_count = w.n_samples - t_begin if t_count is None else t_count
        if out is None:
            out = torch.empty((t_count, w.n_spaxel, w.n_chan), dtype=torch.float32, device=self.device)
        self._check(self.L.gt_debug_pkid(self.handle, t_begin, t_count, _ptr(out), self._stream()))
        return out

    def geometry(self, t_begin=0, t_count=None):
        w = self.w
        t_count = w.n_samples - t_begin if t_count is None else t_count
        rec = np.zeros(t_count * w.n_spaxel, dtype=GEOREC_DTYPE)
        self._check(self.L.gt_debug_geometry(self.handle, t_begin, t_count, C.c_void_p(rec.ctypes.data)))
        return rec.reshape(t_count, w.n_spaxel)

    def destroy(self):
        if getattr(self, "handle", None) is not None and self.handle.value:
            self.L.gt_plan_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()


def _ptr(x):
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        assert x.dtype == np.float32 and x.flags.c_contiguous
        return C.c_void_p(x.ctypes.data)
    assert x.is_contiguous()
    return C.c_void_p(x.data_ptr())


def release_cached_memory() -> None:
    """gt_release_cached_memory: returns the plan pool's cached device memory to the driver."""
    st = lib().gt_release_cached_memory()
    if st != GT_OK:
        raise GateauError(st, lib().gt_last_error(None).decode())


def measure_fp32_fma() -> float:
    """gt_measure_fp32_fma: FP32 FMA peak of the current device, TFLOP/s."""
    v = C.c_double(0.0)
    st = lib().gt_measure_fp32_fma(None, C.byref(v))
    if st != GT_OK:
        raise GateauError(st, lib().gt_last_error(None).decode())
    return float(v.value)


def debug_philox(seed, c0_begin, count, c1=0, c2=0, c3=0) -> np.ndarray:
    out = np.zeros((count, 4), dtype=np.uint32)
    st = lib().gt_debug_philox(int(seed), int(c0_begin) & 0xffffffff, int(count), int(c1), int(c2), int(c3),
                               C.c_void_p(out.ctypes.data))
    if st != GT_OK:
        raise GateauError(st, lib().gt_last_error(None).decode())
    return out


# names of the C ABI, re-exported (same names as include/gateau_b200.h)
def gt_plan_create(cfg: GtConfig, stream=None):
    h = C.c_void_p()
    st = lib().gt_plan_create(C.byref(cfg), stream, C.byref(h))
    return st, h


def gt_simulate(handle, t_begin, t_count, tod_out, pwv_out=None, stream=None):
    return lib().gt_simulate(handle, t_begin, t_count, _ptr(tod_out), _ptr(pwv_out), stream)


def gt_plan_destroy(handle):
    return lib().gt_plan_destroy(handle)


def gt_last_error(handle=None) -> str:
    return lib().gt_last_error(handle).decode()


def gt_prepare_screen(epl, dx_m, dy_m, R_tel_m, t_edge_db, pwv0_mm, out=None):
    """gt_prepare_screen: `epl` a contiguous float32 CUDA tensor [ny][nx]; returns the PWV screen (a new CUDA tensor
    unless `out` is given).  Argument marshalling only."""
    import torch
    if not (epl.is_cuda and epl.dtype == torch.float32 and epl.dim() == 2 and epl.is_contiguous()):
        raise ValueError("epl must be a contiguous float32 CUDA tensor [ny][nx]")
    out = torch.empty_like(epl) if out is None else out
    st = lib().gt_prepare_screen(_ptr(epl), int(epl.shape[1]), int(epl.shape[0]), float(dx_m), float(dy_m),
                                 float(R_tel_m), float(t_edge_db), float(pwv0_mm), _ptr(out),
                                 C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != GT_OK:
        raise GateauError(st, lib().gt_last_error(None).decode())
    return out


def gt_prepare_source(I_cube, nu0_hz, dnu_hz, daz_rad, del_rad, el_first_rad, R_tel_m, t_edge_db, r_pix, out=None):
    """gt_prepare_source: `I_cube` a contiguous float32 CUDA tensor [n_el][n_az][n_freq]; returns P_nu,src (a new CUDA
    tensor unless `out` is given).  Argument marshalling only."""
    import torch
    if not (I_cube.is_cuda and I_cube.dtype == torch.float32 and I_cube.dim() == 3 and I_cube.is_contiguous()):
        raise ValueError("I_cube must be a contiguous float32 CUDA tensor [n_el][n_az][n_freq]")
    out = torch.empty_like(I_cube) if out is None else out
    n_el, n_az, n_freq = (int(x) for x in I_cube.shape)
    st = lib().gt_prepare_source(_ptr(I_cube), n_az, n_el, n_freq, float(nu0_hz), float(dnu_hz), float(daz_rad),
                                 float(del_rad), float(el_first_rad), float(R_tel_m), float(t_edge_db), int(r_pix),
                                 _ptr(out), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != GT_OK:
        raise GateauError(st, lib().gt_last_error(None).decode())
    return out
