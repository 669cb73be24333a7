"""CPU-side checks of the C ABI: the library builds, loads and exports every symbol that
include/gateau_b200.h declares; argument validation returns the documented status codes
before any device work; without a CUDA device the compute entry points fail loudly
(GT_ERR_CUDA) -- there is no CPU fallback.  No compute call is made here."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2604_23305_b200 import binding as B
from paper_2604_23305_b200 import workloads as W

ROOT = Path(__file__).resolve().parent.parent


def _cuda():
    import torch
    return torch.cuda.is_available()


def test_library_exports_every_declared_symbol():
    hdr = (ROOT / "include" / "gateau_b200.h").read_text()
    declared = set(re.findall(r"\b(gt_[a-z_0-9]+)\s*\(", hdr))
    assert {"gt_plan_create", "gt_simulate", "gt_plan_destroy"} <= declared
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in the header but not exported"
    assert declared == set(B.EXPORTS)


def test_struct_layout_matches_header_field_order():
    hdr = (ROOT / "include" / "gateau_b200.h").read_text()
    body = hdr[hdr.index("typedef struct {\n    /* uniform frequency grid"):hdr.index("} gt_config;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S).replace("typedef struct {", "")
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(float|double|int32_t|int64_t|uint64_t|gt_stage)\s*\*?", "", decl)
        names += [n.strip(" *\n") for n in decl.split(",")]
    names = [n for n in names if n]
    assert names == [f[0] for f in B.GtConfig._fields_]
    assert C.sizeof(B.GtStage) == 32
    assert B.GEOREC_DTYPE.itemsize == 88


def _host_cfg(w, keep):
    """gt_config with HOST pointers standing in for the device arrays: good enough for the
    validation path, which never dereferences them."""
    dev = {}
    for name, arr in (("cube", w.cube), ("screen", w.screen), ("atm_lut", w.atm_lut), ("filt", w.filt),
                      ("eta_front", w.eta_front_nu)):
        if arr is not None:
            keep["d_" + name] = np.ascontiguousarray(arr, dtype=np.float32)
            dev[name] = keep["d_" + name].ctypes.data
    for i, s in enumerate(w.stages):
        if np.ndim(s.eta) != 0:
            keep[f"d_stage{i}"] = np.ascontiguousarray(s.eta, dtype=np.float32)
            dev[f"stage{i}"] = keep[f"d_stage{i}"].ctypes.data
    return B.fill_config(w, dev, keep)


@pytest.mark.parametrize("mutate,status", [
    (lambda c: setattr(c, "n_freq", 0), 2),
    (lambda c: setattr(c, "n_samples", -1), 2),
    (lambda c: setattr(c, "screen", None), 1),
    (lambda c: setattr(c, "filt", None), 1),
    (lambda c: setattr(c, "f_sample_hz", 0.0), 3),
    (lambda c: setattr(c, "T_atm_K", -1.0), 3),
    (lambda c: setattr(c, "lut_nu0_hz", 250e9), 4),           # LUT no longer covers the grid
    (lambda c: setattr(c, "variant", 9), 3),
    (lambda c: (setattr(c, "pink_noise", 1), setattr(c, "pink_n_stage", 9)), 2),
])
def test_validation_status_codes(mutate, status):
    w = W.random_workload(3, n_samples=8)
    keep = {}
    cfg = _host_cfg(w, keep)
    mutate(cfg)
    st, h = B.gt_plan_create(cfg)
    assert st == status, B.gt_last_error()
    assert not h.value
    assert B.gt_last_error() != ""


def test_bad_stage_eta_is_rejected():
    w = W.random_workload(4, n_samples=8)
    w.stages[0].eta = 1.5
    keep = {}
    st, h = B.gt_plan_create(_host_cfg(w, keep))
    assert st == 3 and not h.value


def test_null_safety():
    assert B.gt_plan_destroy(None) == 0
    assert B.lib().gt_simulate(None, 0, 1, None, None, None) == 1
    assert B.lib().gt_plan_create(None, None, C.byref(C.c_void_p())) == 1


@pytest.mark.skipif(_cuda(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback_without_a_device():
    w = W.random_workload(5, n_samples=8)
    keep = {}
    st, h = B.gt_plan_create(_host_cfg(w, keep))
    assert st == 6 and not h.value                       # GT_ERR_CUDA
    assert "no CPU fallback" in B.gt_last_error()
    with pytest.raises(B.GateauError):
        B.Plan(w)
    with pytest.raises(B.GateauError):
        B.debug_philox(1, 0, 4)
