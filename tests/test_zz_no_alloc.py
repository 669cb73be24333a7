"""gt_common_mode_static: the no-allocation entry point (partial sums of Eq. 25 in the library's static device array)
against the existing path gt_common_mode_partial + gt_common_mode_apply, on two calls in a row.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  Passes alone in a fresh process and after the other tests (the array is shared and keeps the last call's
contents; nothing in it has to start at zero).
"""
import ctypes as C

import numpy as np
import pytest

from oracle import oracle as O
from paper_2604_23305_b200 import binding as B
from paper_2604_23305_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_CM = 3e-7          # the tolerance of test_common_mode_subtraction_sharded_and_single_plan_against_the_oracle


def _workload(n_samples=150):
    w = W.random_workload(121, n_samples=n_samples, n_spaxel=7, n_chan=21, n_freq=80, photon_noise=True)
    return w.replace(output_unit=1, skydip_n=10, skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.7)


def test_common_mode_static_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    w = _workload()
    r_out = 8 * np.pi / 180 / 3600
    o = O.Oracle(w)
    with B.Plan(w) as p:
        tod, pwv = p.simulate(want_pwv=True)
        pwv_mean = float(pwv.double().mean().item())
        # existing path: caller-owned buffer for the partial sums
        partial, n_out = p.common_mode_partial(tod, pwv_mean, r_out)
        ref1 = p.common_mode_apply(tod.clone(), pwv_mean, partial, n_out)
        # a second, different input on a window of the samples: other values and a SMALLER footprint in the shared array
        t0, tc = 40, 70
        tod2 = (tod[t0:t0 + tc] * 1.5 + 3.0).contiguous()
        partial2, n_out2 = p.common_mode_partial(tod2, pwv_mean, r_out, t_begin=t0)
        ref2 = p.common_mode_apply(tod2.clone(), pwv_mean, partial2, n_out2, t_begin=t0)
        in1, in2, in3 = tod.clone(), tod2.clone(), tod.clone()
        torch.cuda.synchronize()

        # call 1 (whatever the array held before: zeros in a fresh process, another test's sums otherwise)
        got1, n1 = p.common_mode_static(in1, pwv_mean, r_out)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        # calls 2 and 3, back to back on one stream: the array still holds call 1's (then call 2's) partial sums
        got2, n2 = p.common_mode_static(in2, pwv_mean, r_out, t_begin=t0)
        got3, n3 = p.common_mode_static(in3, pwv_mean, r_out)
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info()[0]
        g1, g2, g3 = (x.cpu().numpy() for x in (got1, got2, got3))
        r1, r2 = ref1.cpu().numpy(), ref2.cpu().numpy()
        tod_np = tod.cpu().numpy()
    assert n1 == n2 == n3 == n_out == n_out2 and 0 < n_out < w.n_spaxel
    assert free_after == free_before                                  # no device memory was taken or returned
    # against the existing path: within the tests' tolerance -- and, same kernels on the same inputs, bit for bit
    eta_z = O.eta_zenith_at(w, w.f_center_hz, pwv_mean)
    csc = o.geometry()["csc"]
    scale = np.max(np.abs(tod_np / (eta_z[None, None, :] ** csc[:, :, None])))
    for g, r, s in ((g1, r1, scale), (g2, r2, 1.5 * scale + 3.0), (g3, r1, scale)):
        assert g.shape == r.shape
        assert np.max(np.abs(g.astype(np.float64) - r.astype(np.float64))) <= TOL_CM * s
        assert np.array_equal(g, r)
    # and against the oracle's literal Eq. 25-26 on the same TOD
    ref, S, _ = O.common_mode_subtract(tod_np.astype(np.float64), eta_z, csc, w.daz_rad, w.del_rad, r_out)
    assert n_out == int(S.sum())
    assert np.max(np.abs(g1 - ref)) <= TOL_CM * scale
    assert np.max(np.abs(g3 - ref)) <= TOL_CM * scale


def test_common_mode_static_rejects_sizes_beyond_the_static_array():
    import torch
    n = B.COMMON_MODE_STATIC_MAX // 21 + 1                            # one sample more than fits: t_count * n_chan > max
    w = _workload(n_samples=n + 10)
    with B.Plan(w) as p:
        small = torch.zeros((4, w.n_spaxel, w.n_chan), dtype=torch.float32, device="cuda")
        n_out = C.c_int32(0)
        st = p.L.gt_common_mode_static(p.handle, 0, n, C.c_void_p(small.data_ptr()), 1.0, 0.0, C.byref(n_out), None)
        assert st == 2                                                # GT_ERR_SHAPE, before anything is launched
        msg = p.L.gt_last_error(p.handle).decode()
        assert "GT_COMMON_MODE_STATIC_MAX" in msg and str(B.COMMON_MODE_STATIC_MAX) in msg
        torch.cuda.synchronize()
        assert float(small.abs().max().item()) == 0.0
        with pytest.raises(B.GateauError) as e:
            p.common_mode_static(small, 1.0, 1.0)                     # r_out = 1 rad: no spaxel outside -> N_out = 0
        assert e.value.status == 3
