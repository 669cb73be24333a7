"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.

Gates (BASELINE.json north_star): geometry integers and Philox words bit-exact; noiseless
channel power max relative error <= 1e-5; noisy TOD <= 2e-5 relative to
max(|oracle|, 1e-3 * median|oracle|).
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2604_23305_b200 import binding as B
from paper_2604_23305_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_PKID = 1e-5
TOL_TOD = 2e-5
VARIANTS = [B.VARIANT_FP32, B.VARIANT_TENSOR]
VARIANT_IDS = ["fp32", "tensor"]


def rel_err(got, ref):
    ref = np.asarray(ref, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    floor = 1e-3 * np.median(np.abs(ref))
    return np.max(np.abs(got - ref) / np.maximum(np.abs(ref), floor))


def _plan(w, variant, **kw):
    try:
        return B.Plan(w, variant=variant, **kw)
    except B.GateauError as e:
        if e.status == 7:
            pytest.skip(f"variant not available: {e}")
        raise


# --------------------------------------------------------------------------------------
# bit-exact integer work
# --------------------------------------------------------------------------------------
def test_philox_words_bit_exact():
    for seed, c0, c1, c2, c3 in [(0, 0, 0, 0, 0), (0x0123456789ABCDEF, 4294967290, 60, 346, 2), (3, 12345, 7, 11, 1)]:
        got = B.debug_philox(seed, c0, 64, c1, c2, c3)
        key = (seed & 0xffffffff, seed >> 32)
        for i in range(64):
            assert list(got[i]) == O.philox4x32_10(((c0 + i) & 0xffffffff, c1, c2, c3), key)


INT_FIELDS = ("n", "iu0", "iv0", "ju", "jv", "ip")
FRAC_FIELDS = ("fu", "fv", "gu", "gv", "fp", "csc", "pwv_mm")


def _check_geometry(w, t_begin=0, t_count=None):
    with B.Plan(w, variant=B.VARIANT_FP32) as p:
        got = p.geometry(t_begin, t_count)
    ref = O.Oracle(w).geometry(t_begin, t_count)
    for f in INT_FIELDS:
        assert np.array_equal(got[f], ref[f]), f"geometry field {f} differs"
    for f in FRAC_FIELDS:
        assert np.array_equal(got[f], ref[f]), f"geometry field {f} is not bit-identical"


@pytest.mark.parametrize("seed", [1, 2])
def test_geometry_bit_exact_random(seed):
    _check_geometry(W.random_workload(seed, n_samples=700, n_spaxel=5))


def test_geometry_bit_exact_C1():
    _check_geometry(W.make_workload("C1"))


def test_geometry_bit_exact_C5_window_late_in_the_scan():
    # wind drift has carried the boresight 3.4e5 screen cells away; PWV drifts through LUT rows
    w = W.make_workload("C5", n_chan=8, n_freq=64, cube_n=9, screen_n=512)
    _check_geometry(w, t_begin=w.n_samples - 3000, t_count=3000)


# --------------------------------------------------------------------------------------
# noiseless channel power (steps 0-5)
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("seed,kw", [
    (11, dict(n_samples=67, n_spaxel=3, n_chan=24, n_freq=96)),               # ragged row tile
    (12, dict(n_samples=150, n_spaxel=2, n_chan=70, n_freq=333, n_stage=6)),  # ragged everything
    (13, dict(n_samples=40, n_spaxel=7, n_chan=347, n_freq=530)),             # full channel width
    (14, dict(n_samples=33, n_spaxel=1, n_chan=5, n_freq=17, with_cube=False)),
])
def test_pkid_random(variant, seed, kw):
    w = W.random_workload(seed, **kw)
    ref = O.Oracle(w).simulate(want=("pkid", "pwv"))
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
        tod, pwv = p.simulate(want_pwv=True)
    assert rel_err(got, ref["pkid"]) <= TOL_PKID
    assert np.array_equal(tod.cpu().numpy(), got)           # noise off => TOD is the noiseless power
    assert np.max(np.abs(pwv.cpu().numpy() - ref["pwv"])) <= 1e-6


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("n_chan,n_freq", [(32, 256), (130, 300), (256, 520), (400, 288), (800, 100)])
def test_pkid_channel_group_layouts(variant, n_chan, n_freq):
    """Tensor kernel: 1, 2 and 3 column groups per tile, and more than 384 channels (several channel groups
    per row tile); n_freq spans several accumulation segments with a ragged last slab."""
    w = W.random_workload(70 + n_chan, n_samples=90, n_spaxel=3, n_chan=n_chan, n_freq=n_freq)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_pkid_C1_full(variant):
    w = W.make_workload("C1")
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("cfg", ["C2", "C3", "C4", "C5"])
def test_pkid_configs_window(variant, cfg):
    """Full channel/frequency sizes of each config, several row tiles and a ragged tail."""
    w = W.make_workload(cfg, n_samples=4000 if cfg == "C2" else 2000, screen_n=1024,
                        photon_noise=False, pink_noise=False)
    T = 333 // w.n_spaxel + 3
    t0 = w.n_samples - T
    ref = O.Oracle(w).simulate(t0, T, want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid(t0, T).cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


# --------------------------------------------------------------------------------------
# invariants that hold at any size, through the CUDA path
# --------------------------------------------------------------------------------------
def _planck(nu, T):
    h, kb = 6.62607015e-34, 1.380649e-23
    return h * nu / np.expm1(h * nu / (kb * T))


def _row_normalised(filt, dnu):
    f = filt.astype(np.float64)
    return (f / (f.sum(axis=1, keepdims=True) * dnu)).astype(np.float32)


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("case", ["no_source", "source_is_blackbody"])
def test_thermal_equilibrium_on_gpu(variant, case):
    """Everything at one temperature T returns B(nu, T) in every channel whatever the efficiencies (Eq. 12,
    PAPER.md:165), with the ROW-NORMALISED filter (sum Fm dnu = 1, values ~1e-10) exactly as the
    oracle-side pin builds it (tests/test_oracle_chain.py test_thermal_equilibrium), both variants of the pin."""
    T = 77.0
    w = W.random_workload(21, n_samples=50, n_spaxel=2, n_chan=40, n_freq=200, couple=(case == "no_source"))
    stages = [W.Stage(s.eta, T, s.couple_atmosphere) for s in w.stages]
    if case == "no_source":
        w = w.replace(cube=None, T_cmb_K=T, T_atm_K=T, stages=stages)
    else:
        cube = np.broadcast_to(_planck(w.nu_hz, T), w.cube.shape).astype(np.float32)
        w = w.replace(cube=cube, eta_front_nu=None, T_cmb_K=0.0, T_atm_K=T, stages=stages,
                      az_rad=np.zeros(w.n_samples), el_rad=np.zeros(w.n_samples))      # stay on the cube
    filt = _row_normalised(w.filt, w.dnu_hz)
    assert filt.max() < 1e-8
    w = w.replace(filt=filt)
    expect = w.dnu_hz * (filt.astype(np.float64) @ _planck(w.nu_hz, T))
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, np.broadcast_to(expect, got.shape)) <= TOL_PKID


# --------------------------------------------------------------------------------------
# operand range of the contraction: the tensor kernel multiplies fp16 pairs, so
# north_star's own invariants -- filters and spectra of any magnitude -- must come through at the same gates
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_delta_filter_reproduces_the_spectrum_on_gpu(variant):
    """north_star: "a delta filter must reproduce the spectrum" -- one-hot rows 1/dnu (1e-9 here) return the
    oracle's own row_spectrum at that frequency (rectangle rule, R16; SURVEY 8c.4 "Contraction")."""
    w = W.random_workload(22, n_samples=70, n_spaxel=2, n_chan=130, n_freq=333)
    hot = np.linspace(0, w.n_freq - 1, w.n_chan).astype(int)               # first and last frequency included
    filt = np.zeros((w.n_chan, w.n_freq), dtype=np.float32)
    filt[np.arange(w.n_chan), hot] = 1.0 / w.dnu_hz
    w = w.replace(filt=filt, f_center_hz=w.nu_hz[hot], dnu_eff_hz=None)
    o = O.Oracle(w)
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, o.simulate(want=("pkid",))["pkid"]) <= TOL_PKID
    for n, s in ((0, 0), (33, 1), (69, 0)):
        spec = o.row_spectrum(n, s)[hot]
        assert np.max(np.abs(got[n, s] / (np.float32(1.0 / w.dnu_hz) * w.dnu_hz) - spec) / spec) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("peak", [1e-12, 1e-6, 1.0, 3e4])
def test_filter_magnitude_does_not_matter(variant, peak):
    """Lorentzian channels of peak 1e-12 ... 3e4 (a transmission is <= 1; the contraction is linear and the ABI
    sets no range): every channel carries its own power-of-two scale."""
    w = W.random_workload(23, n_samples=60, n_spaxel=2, n_chan=96, n_freq=700)
    fc = np.geomspace(w.nu_hz[20], w.nu_hz[-20], w.n_chan)
    w = w.replace(filt=W.lorentzian_filterbank(w.nu_hz, fc, 300.0, peak), f_center_hz=fc, dnu_eff_hz=None)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_filterbank_of_eq7_with_negative_rows(variant):
    """Eq. 7 with unequal peak efficiencies: where the channels upstream have absorbed more than a
    channel's own eta_peak its row goes negative (a quarter of the matrix here, half of the channel powers are
    negative).  Cancellation is mild (sum |Fm| P <= 1.15 |sum Fm P|), so the plain 1e-5 gate applies."""
    w = W.random_workload(78, n_samples=40, n_spaxel=2, n_chan=64, n_freq=600)
    fc = w.nu_hz[40] * (1 + 1 / 120.0) ** np.arange(64)
    F = W.filterbank_upstream_absorption(w.nu_hz, fc, 40.0, np.where(np.arange(64) % 2 == 0, 0.3, 0.05))
    assert (F < 0).mean() > 0.2
    w = w.replace(filt=F, f_center_hz=fc, dnu_eff_hz=None)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    assert (ref < 0).mean() > 0.3
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert np.max(np.abs(got - ref) / np.abs(ref)) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("gain", [1e-6, 1e3, 1e12])
def test_spectrum_magnitude_does_not_matter(variant, gain):
    """A source 1e3 x brighter than the synthetic one (30 x the atmosphere: a planet on axis), 1e12 x brighter
    (nothing else left), and a faint one: the plan scales the spectrum from max |Xn|, max |G| max |cube|."""
    w = W.random_workload(24, n_samples=90, n_spaxel=3, n_chan=50, n_freq=300)
    w = w.replace(cube=(w.cube.astype(np.float64) * gain).astype(np.float32))
    if gain > 1e6:
        # rows that leave the cube would see a sky 1e-12 of the plan's brightest element: below the stated
        # dynamic range of the operand pairs (include/gateau_b200.h "Value ranges"); stay on the source
        w = w.replace(az_rad=0.5 * w.az_rad, el_rad=0.5 * w.el_rad)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


def test_narrow_channels_on_the_edges_of_accumulation_segments():
    """Tensor kernel: the accumulators truncate, so a segment loses about one ulp of its running
    sum per chained MMA -- all of it for a narrow channel in the FIRST slab of a segment, nothing for one in the
    LAST.  Channels three frequency points wide centred on every slab of a 27-slab grid (segments of 12, 12 and 3
    slabs, staggered between the three column groups: every group meets first, last and short-tail positions),
    on a spectrum and a filter scale that keep every other error small."""
    n_kb = 27
    w = W.random_workload(25, n_samples=140, n_spaxel=2, n_chan=300, n_freq=64 * n_kb)
    c = np.arange(w.n_chan)
    idx = 64 * (c % n_kb) + 5 + (c * 7) % 54
    fc = w.nu_hz[idx]
    filt = np.stack([W.lorentzian_filterbank(w.nu_hz, fc[i:i + 1], fc[i] / (3 * w.dnu_hz), 0.16)[0] for i in range(w.n_chan)])
    filt[np.abs(np.arange(w.n_freq)[None, :] - idx[:, None]) > 40] = 0.0       # no tails: the mass sits in one slab (or two)
    w = w.replace(filt=filt, f_center_hz=fc, dnu_eff_hz=None)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, B.VARIANT_TENSOR) as p:
        got = p.pkid().cpu().numpy()
    err = (got - ref) / ref
    by_slab = np.array([np.abs(err[:, :, (c % n_kb) == k]).max() for k in range(n_kb)])
    print("max |rel err| per centre slab:", np.array2string(by_slab, precision=2))
    print("mean rel err per centre slab:", np.array2string(np.array([err[:, :, (c % n_kb) == k].mean() for k in range(n_kb)]), precision=2))
    assert np.abs(err).max() <= TOL_PKID
    assert np.abs(err).max() <= 0.6 * TOL_PKID, "the per-segment compensation is off: recalibrate kTcTruncUlp"


def test_banded_corrections_skip_only_what_the_plan_can_bound():
    """Tensor kernel, DESIGN.md section 6 "Banded corrections": the correction products A_lo.Fm_hi and A_hi.Fm_lo of a
    (column group, slab) block are not issued where the plan bounds them -- worst case over the spectra it can produce,
    all skipped products of a channel together -- below 1e-6 of the channel's power.  On the C4 shape (R = 500
    Lorentzians, a quiet sky) about half of them go; with a PWV screen 40 x rougher (rows spread over several table
    rows: a wider range of spectra) fewer; with filter rows that change sign none; parity holds in every case."""
    w = W.make_workload("C4", n_samples=256)
    n_kb = -(-w.n_freq // 64)
    rows_t, rows_s = [0, 77, 131, 255], [0, 20, 41, 60]
    counts = []
    for rough in (1.0, 40.0):
        scr = np.asarray(w.screen, dtype=np.float64)
        wr = w if rough == 1.0 else w.replace(screen=(scr.mean() + rough * (scr - scr.mean())).astype(np.float32))
        assert wr.screen.min() + wr.pwv0_a_mm > wr.lut_pwv0_mm
        ref = O.Oracle(wr).simulate_rows(rows_t, rows_s, noise=False)
        with _plan(wr, B.VARIANT_TENSOR) as p:
            products, skipped = p.corrections()
            banded = p.pkid()
        with _plan(wr, B.VARIANT_TENSOR_FULL) as p:          # the same kernel issuing every correction product
            assert p.corrections() == (products, 0) and p.variant_name.endswith("-full")
            full = p.pkid()
        assert products == 2 * 3 * n_kb                      # one channel group of three column groups, two products each
        assert rel_err(banded.cpu().numpy()[rows_t, rows_s], ref) <= TOL_PKID
        # the claim itself, on every element of the window (5.4e6 values): what the skipped products were worth is inside
        # the plan's worst-case budget (measured 4-5e-7 at most, 7e-8 rms, truncation-path differences included)
        d = ((banded.double() - full.double()) / full.double()).abs()
        print(f"screen x {rough:g}: {skipped} of {products} skipped, max |banded/full - 1| = {float(d.max()):.2e}")
        assert float(d.max()) <= 1e-6
        counts.append(skipped)
    assert 0.35 * 6 * n_kb <= counts[0] <= 0.75 * 6 * n_kb
    assert 0 < counts[1] < counts[0]
    # a source 1e3 x brighter (its spectrum dominates some rows and not others: a wide bracket per frequency)
    wb = w.replace(cube=(np.asarray(w.cube, dtype=np.float64) * 1e3).astype(np.float32))
    with _plan(wb, B.VARIANT_TENSOR) as p:
        skipped_b = p.corrections()[1]
        banded = p.pkid(0, 128)
    with _plan(wb, B.VARIANT_TENSOR_FULL) as p:
        full = p.pkid(0, 128)
    d = ((banded.double() - full.double()) / full.double()).abs()
    print(f"cube x 1e3: {skipped_b} skipped, max |banded/full - 1| = {float(d.max()):.2e}")
    assert float(d.max()) <= 1e-6 and skipped_b <= counts[0]
    with _plan(w, B.VARIANT_FP32) as p:
        assert p.corrections() == (0, 0)
    # filter rows that change sign (Eq. 7): a share of the channel's power bounds nothing
    w7 = W.random_workload(78, n_samples=40, n_spaxel=2, n_chan=64, n_freq=600)
    fc = w7.nu_hz[40] * (1 + 1 / 120.0) ** np.arange(64)
    F = W.filterbank_upstream_absorption(w7.nu_hz, fc, 40.0, np.where(np.arange(64) % 2 == 0, 0.3, 0.05))
    with _plan(w7.replace(filt=F, f_center_hz=fc, dnu_eff_hz=None), B.VARIANT_TENSOR) as p:
        products, skipped = p.corrections()
    assert products > 0 and skipped == 0


@pytest.mark.parametrize("n_chan,n_freq,R,drift,gain", [(420, 1920, 500.0, 2.0, 0.0), (420, 4000, 150.0, 2.0, 1.0),
                                                       (347, 4000, 500.0, 2.0, 1.0), (130, 1920, 2000.0, 0.05, 1e3)])
def test_banded_corrections_stay_inside_their_budget_on_random_inputs(n_chan, n_freq, R, drift, gain):
    """Random cascades, screens and cubes with Lorentzian filterbanks (two channel groups included, PWV drifting through
    the whole table, a source 1e3 x brighter): the banded kernel against the one that issues every product, every element."""
    w = W.random_workload(1003, n_samples=96, n_spaxel=3, n_chan=n_chan, n_freq=n_freq)
    fc = np.linspace(w.nu_hz[8], w.nu_hz[-8], n_chan)
    w = w.replace(filt=W.lorentzian_filterbank(w.nu_hz, fc, R, 0.3), f_center_hz=fc, dnu_eff_hz=None,
                  pwv0_a_mm=0.2, pwv0_b_mm_per_s=drift, cube=(w.cube.astype(np.float64) * gain).astype(np.float32))
    with _plan(w, B.VARIANT_TENSOR) as p:
        products, skipped = p.corrections()
        banded = p.pkid().double()
    with _plan(w, B.VARIANT_TENSOR_FULL) as p:
        full = p.pkid().double()
    assert skipped > 0
    assert float(((banded - full) / full).abs().max()) <= 1e-6
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    assert rel_err(banded.cpu().numpy(), ref) <= TOL_PKID


def test_non_finite_inputs_and_lines_of_sight_below_the_horizon_are_refused():
    w = W.random_workload(26, n_samples=20)
    bad_cube = np.array(w.cube, copy=True); bad_cube[2, 3, 7] = np.nan
    bad_screen = np.array(w.screen, copy=True); bad_screen[5, 6] = np.inf
    bad_filt = np.array(w.filt, copy=True); bad_filt[1, 2] = np.nan
    for ww in (w.replace(cube=bad_cube), w.replace(screen=bad_screen), w.replace(filt=bad_filt),
               w.replace(el0_rad=1e-5), w.replace(el_rad=w.el_rad + np.pi)):
        for variant in VARIANTS:
            with pytest.raises(B.GateauError) as e:
                B.Plan(ww, variant=variant)
            assert e.value.status == 3, str(e.value)


def test_plan_counters():
    """gt_plan_counters: rows outside the cube and PWV clamps, against the oracle's geometry records."""
    w = W.random_workload(27, n_samples=300, n_spaxel=3)
    geo = O.Oracle(w).geometry()
    q = (geo["pwv_mm"] - w.lut_pwv0_mm) / w.lut_dpwv_mm
    with B.Plan(w) as p:
        p.simulate()
        got = p.counters()
        p.pkid(10, 50)
        again = p.counters()
    assert got == dict(rows=w.n_samples * w.n_spaxel, rows_outside_cube=int((geo["ju"] < 0).sum()),
                       pwv_below_lut=int((q < 0).sum()), pwv_above_lut=int((q > w.atm_lut.shape[0] - 1).sum()))
    assert got["rows_outside_cube"] > 0 and got["pwv_above_lut"] + got["pwv_below_lut"] > 0
    assert again["rows"] == got["rows"] + 50 * w.n_spaxel


def test_pink_state_export_import_resumes_a_run():
    """Checkpoint at call granularity: a second plan of the same configuration, given the exported
    AR(1) state, continues the TOD bit for bit."""
    w = W.random_workload(28, n_samples=700, n_spaxel=2, n_chan=20, n_freq=48, photon_noise=True, pink_noise=True, J=6)
    with B.Plan(w) as p:
        whole = p.simulate().cpu().numpy()
        p.simulate(0, 333)
        state, nt = p.pink_state_export()
    assert nt == 333 and state.shape == (40, 6)
    with B.Plan(w) as p2:
        with pytest.raises(B.GateauError):
            p2.simulate(333, 10)                              # no state yet: out of order
        p2.pink_state_import(state, nt)
        rest = p2.simulate(333, 367).cpu().numpy()
    assert np.array_equal(rest, whole[333:])
    with B.Plan(w.replace(pink_noise=False)) as p3:
        with pytest.raises(B.GateauError) as e:
            p3.pink_state_export()
        assert e.value.status == 7


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("pink_method", [0, 1])
def test_spaxel_shard_reproduces_the_full_plan(variant, pink_method):
    """gt_config.spaxel_index_base: a plan holding spaxels [3, 7) of an instrument gives bit for bit the TOD those
    spaxels have in the plan that holds all of them (photon, pink noise keyed by the GLOBAL spaxel index)."""
    w = W.random_workload(29, n_samples=200, n_spaxel=7, n_chan=21, n_freq=80, photon_noise=True, pink_noise=True)
    w = w.replace(pink_method=pink_method)
    lo, hi = 3, 7
    nc = w.n_chan
    shard = w.replace(daz_rad=w.daz_rad[lo:hi], del_rad=w.del_rad[lo:hi], spaxel_index_base=lo,
                      pink_A=w.pink_A[lo * nc:hi * nc], pink_alpha=w.pink_alpha[lo * nc:hi * nc])
    with _plan(w, variant) as p, _plan(shard, variant) as ps:
        full = p.simulate().cpu().numpy()
        part = ps.simulate().cpu().numpy()
    assert np.array_equal(part, full[:, lo:hi])


# --------------------------------------------------------------------------------------
# noise (steps 6a, 6b) and Eq. 21
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_tod_photon_noise(variant):
    w = W.random_workload(31, n_samples=130, n_spaxel=3, n_chan=50, n_freq=128, photon_noise=True)
    ref = O.Oracle(w).simulate(want=("tod", "pkid"))
    with _plan(w, variant) as p:
        got = p.simulate().cpu().numpy()
    assert rel_err(got, ref["tod"]) <= TOL_TOD
    assert np.std(got - ref["pkid"]) > 0                    # the noise is really there


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("J", [1, 4, 6, 8])
def test_tod_photon_and_pink_noise(variant, J):
    w = W.random_workload(40 + J, n_samples=300, n_spaxel=2, n_chan=33, n_freq=64, photon_noise=True,
                          pink_noise=True, J=J)
    ref = O.Oracle(w).simulate(want=("tod",))["tod"]
    with _plan(w, variant) as p:
        got = p.simulate().cpu().numpy()
    assert rel_err(got, ref) <= TOL_TOD


def test_pink_noise_is_carried_across_calls_and_chunks():
    """Contiguous calls continue the AR(1) state; chunked host streaming gives the same values."""
    w = W.random_workload(51, n_samples=1000, n_spaxel=2, n_chan=20, n_freq=48, photon_noise=True, pink_noise=True)
    ref = O.Oracle(w).simulate(want=("tod",))["tod"]
    with B.Plan(w, variant=B.VARIANT_FP32, chunk_samples=97) as p:
        whole = p.simulate().cpu().numpy()
        parts = np.concatenate([p.simulate(0, 333).cpu().numpy(), p.simulate(333, 500).cpu().numpy(),
                                p.simulate(833, 167).cpu().numpy()])
        host = p.simulate(device_out=False).numpy()
        with pytest.raises(B.GateauError) as ei:
            p.simulate(500, 10)                               # out of order with pink noise on
        assert ei.value.status == 3
    assert rel_err(whole, ref) <= TOL_TOD
    assert rel_err(parts, ref) <= TOL_TOD
    assert np.array_equal(host, whole)


def test_pink_only_series_matches_oracle_tightly():
    """TOD minus noiseless power with photon noise off isolates P_pn."""
    w = W.random_workload(52, n_samples=2000, n_spaxel=1, n_chan=16, n_freq=32, pink_noise=True)
    o = O.Oracle(w)
    ref = o.pink_series(np.zeros(16, dtype=np.int32), np.arange(16, dtype=np.int32), 0, w.n_samples)   # [det][t]
    ref_pk = o.simulate(want=("pkid",))["pkid"][:, 0, :]
    with B.Plan(w, variant=B.VARIANT_FP32) as p:
        got = p.simulate().cpu().numpy()[:, 0, :].astype(np.float64)
        base = p.pkid().cpu().numpy()[:, 0, :].astype(np.float64)    # the fp32 value the pink kernels added to
    assert rel_err(base, ref_pk) <= TOL_PKID
    pn = (got - base).T
    scale = np.std(ref)
    # two fp32 read-modify-writes of the TOD (<= 1 ulp = 1.2e-7 |P| together) dominate; the series
    # itself must agree with the oracle's recurrence to ~1e-3 of its rms
    assert np.max(np.abs(pn - ref)) <= 2e-3 * scale + 1.3e-7 * np.max(np.abs(base))


# --------------------------------------------------------------------------------------
# boundary behaviour
# --------------------------------------------------------------------------------------
def test_host_streaming_equals_device_output_and_pwv():
    w = W.random_workload(61, n_samples=500, n_spaxel=3, n_chan=40, n_freq=64, photon_noise=True)
    with B.Plan(w, variant=B.VARIANT_FP32, chunk_samples=64) as p:
        dev, pwv_d = p.simulate(want_pwv=True)
        host, pwv_h = p.simulate(device_out=False, want_pwv=True)
        pageable = np.empty((w.n_samples, w.n_spaxel, w.n_chan), dtype=np.float32)
        p.simulate(out=pageable)
        sub = p.simulate(123, 200).cpu().numpy()              # photon noise only: any range is legal
    assert np.array_equal(dev.cpu().numpy(), host.numpy())
    assert np.array_equal(dev.cpu().numpy(), pageable)
    assert np.array_equal(pwv_d.cpu().numpy(), pwv_h.numpy())
    assert np.array_equal(sub, dev.cpu().numpy()[123:323])


def test_empty_and_out_of_range_calls():
    w = W.random_workload(62, n_samples=16)
    with B.Plan(w, variant=B.VARIANT_FP32) as p:
        n0 = p.launch_count                                   # plan creation ran its own kernels (input statistics)
        out = p.simulate(0, 0)
        assert out.shape[0] == 0
        with pytest.raises(B.GateauError) as ei:
            p.simulate(10, 7)
        assert ei.value.status == 4
        assert p.launch_count == n0


def test_rows_outside_the_cube_are_blank_sky():
    """A scan that leaves the cube returns exactly the blank-sky value."""
    w = W.random_workload(63, n_samples=64, n_spaxel=1, n_chan=12, n_freq=40)
    far = w.replace(az_rad=w.az_rad + 1e-2)                   # ~2000 arcsec away: every row outside
    blank = w.replace(cube=None)
    with B.Plan(far, variant=B.VARIANT_FP32) as p1, B.Plan(blank, variant=B.VARIANT_FP32) as p2:
        g = p1.geometry()
        assert np.all(g["ju"] == -1)
        a = p1.pkid().cpu().numpy()
        # same geometry except the pointing offset changes the screen position: compare with the oracle instead
    ref = O.Oracle(far).simulate(want=("pkid",))["pkid"]
    assert rel_err(a, ref) <= TOL_PKID


# --------------------------------------------------------------------------------------
# full-size configuration, sampled
# --------------------------------------------------------------------------------------
def test_C2_full_size_sampled_rows():
    """BASELINE.json configs[1] at full size in the launch configuration bench.py uses,
    checked on sampled rows the oracle computes one by one."""
    w = W.make_workload("C2", photon_noise=True)
    rng = np.random.default_rng(5)
    t_idx = np.sort(rng.choice(w.n_samples, 96, replace=False)).astype(np.int64)
    t_idx[:4] = [0, 1, w.n_samples - 2, w.n_samples - 1]
    s_idx = np.zeros_like(t_idx, dtype=np.int32)
    pk, wn = O.Oracle(w).simulate_rows(t_idx, s_idx, noise=True)
    with B.Plan(w) as p:
        tod = p.simulate()
        pkid = p.pkid()
        got_t = tod[t_idx].cpu().numpy()[:, 0, :]
        got_p = pkid[t_idx].cpu().numpy()[:, 0, :]
    assert rel_err(got_p, pk) <= TOL_PKID
    assert rel_err(got_t, pk + wn) <= TOL_TOD


def _sampled_tiles(w, launch, rng, frac, extra_t=()):
    """Rows for a full-size check, following SURVEY 8d: (i) at least `frac` of all rows as seeded random kernel tiles
    (128 consecutive samples of one spaxel, aligned to the launches of `launch` samples the plan really makes);
    (ii) the samples on both sides of EVERY launch seam, for a random spaxel each; (iii) the last tile block of a few
    launches for every spaxel (the last, partial wave of the persistent kernel's CTA pairs); (iv) the first and last
    samples; (v) `extra_t`.  Returns sorted unique (t_idx, s_idx)."""
    n_t, n_s = w.n_samples, w.n_spaxel
    rows = set()
    starts = np.arange(0, n_t, launch)
    n_tiles = int(np.ceil(frac * n_t * n_s / 128.0))
    for _ in range(n_tiles):
        l0 = int(rng.choice(starts))
        len_l = min(launch, n_t - l0)
        tb = int(rng.integers(0, (len_l + 127) // 128))
        s = int(rng.integers(0, n_s))
        for t in range(l0 + 128 * tb, min(l0 + 128 * tb + 128, l0 + len_l)):
            rows.add((t, s))
    for l0 in starts[1:]:
        s = int(rng.integers(0, n_s))
        rows.update({(int(l0) - 1, s), (int(l0), s)})
    for l0 in rng.choice(starts, min(3, starts.size), replace=False):
        len_l = min(launch, n_t - int(l0))
        t_last = int(l0) + 128 * ((len_l - 1) // 128)
        for s in range(n_s):
            rows.update({(t_last, s), (int(l0) + len_l - 1, s)})
    rows.update({(0, 0), (1, n_s - 1), (n_t - 2, 0), (n_t - 1, n_s - 1)})
    rows.update((int(t), int(rng.integers(0, n_s))) for t in extra_t)
    arr = np.array(sorted(rows), dtype=np.int64)
    return arr[:, 0].copy(), arr[:, 1].astype(np.int32)


def _pink_on(o, w, s_idx, chans, t_idx):
    """The oracle's pink series (run from sample 0) of detectors (s_idx[i], chans[j]) at t_idx[i]: [rows][chans]."""
    pairs = sorted({(int(s), int(c)) for s in np.unique(s_idx) for c in chans})
    ss = np.array([p[0] for p in pairs], dtype=np.int32)
    cc = np.array([p[1] for p in pairs], dtype=np.int32)
    series = o.pink_series(ss, cc, 0, w.n_samples)                               # [pair][t]
    where = {p: i for i, p in enumerate(pairs)}
    out = np.empty((t_idx.size, len(chans)))
    for j, c in enumerate(chans):
        rows = np.array([where[(int(s), int(c))] for s in s_idx])
        out[:, j] = series[rows, t_idx]
    return out


def test_C4_bench_configuration_full_size_sampled():
    """BASELINE.json configs[3] (the bench.py workload) at full size and in bench.py's launch configuration (default
    variant, device output, launches of gt_debug_chunking()'s device chunk): noiseless power on >= 1 % of all rows taken
    as whole kernel tiles plus every launch seam and last waves, and the noisy TOD (photon + pink) on the
    same rows for channels on both sides of every column-group seam, whose pink series the oracle runs from sample 0."""
    w = W.make_workload("C4")
    assert w.photon_noise and w.pink_noise and w.n_samples == 160000 and w.n_spaxel == 61 and w.n_chan == 347
    rng = np.random.default_rng(11)
    chans = np.array([0, 1, 63, 64, 127, 128, 255, 256, 346], dtype=np.int32)
    o = O.Oracle(w)
    with B.Plan(w) as p:
        assert p.variant_name.startswith("tcgen05")
        _, launch = p.chunking()
        assert 0 < launch < w.n_samples                       # several launches: there are seams to look at
        t_idx, s_idx = _sampled_tiles(w, launch, rng, 0.0105)
        assert t_idx.size >= 0.01 * w.n_samples * w.n_spaxel
        tod = p.simulate()
        got_t = tod[t_idx, s_idx.astype(np.int64)].cpu().numpy()
        del tod
        pkid = p.pkid()
        got_p = pkid[t_idx, s_idx.astype(np.int64)].cpu().numpy()
        del pkid
    pk, wn = o.simulate_rows(t_idx, s_idx, noise=True)                          # [row][chan]
    assert rel_err(got_p, pk) <= TOL_PKID
    # pink noise: a fixed set of spaxels (their rows only), all t they were sampled at
    sel = np.isin(s_idx, [0, 17, 30, 44, 60])
    pn = _pink_on(o, w, s_idx[sel], chans, t_idx[sel])
    assert rel_err(got_t[sel][:, chans], (pk + wn)[sel][:, chans] + pn) <= TOL_TOD
    # everywhere else the TOD carries the same photon noise plus its own pink noise (a few 1e-4 of P)
    assert rel_err(got_t, pk + wn) <= 1e-2


def test_C5_long_survey_streamed_in_60s_chunks():
    """BASELINE.json configs[4] at full size the way the config describes it: the TOD of the 1 h, 37-spaxel
    survey is produced in 60 s chunks (9600 samples) into ONE reused pinned host buffer by consecutive
    gt_simulate calls (the pink-noise state carries over).  Compared with the oracle: >= 1 % of all rows as whole
    kernel tiles, +-128 samples around 12 chunk seams, every chunk seam itself, pink noise included on a
    fixed set of detectors."""
    import torch
    w = W.make_workload("C5")
    assert w.n_samples == 576000 and w.n_spaxel == 37 and w.photon_noise and w.pink_noise
    chunk = 9600
    n_chunks = w.n_samples // chunk
    rng = np.random.default_rng(23)
    seams = rng.choice(np.arange(1, n_chunks), 12, replace=False) * chunk
    around = np.concatenate([np.arange(sm - 128, sm + 128) for sm in seams])
    t_idx, s_idx = _sampled_tiles(w, chunk, rng, 0.0105, extra_t=around)
    assert t_idx.size >= 0.01 * w.n_samples * w.n_spaxel
    chans = np.array([0, 127, 128, 255, 256, 346], dtype=np.int32)
    got = np.empty((t_idx.size, w.n_chan), dtype=np.float32)
    buf = torch.empty((chunk, w.n_spaxel, w.n_chan), dtype=torch.float32, pin_memory=True)
    with B.Plan(w, chunk_samples=chunk) as p:
        assert p.chunking()[0] == chunk
        for k in range(n_chunks):
            p.simulate(k * chunk, chunk, out=buf)                      # blocking: returns after the D2H copies
            sel = np.nonzero((t_idx >= k * chunk) & (t_idx < (k + 1) * chunk))[0]
            if sel.size:
                got[sel] = buf[torch.from_numpy(t_idx[sel] - k * chunk), torch.from_numpy(s_idx[sel].astype(np.int64))].numpy()
    o = O.Oracle(w)
    pk, wn = o.simulate_rows(t_idx, s_idx, noise=True)
    sel = np.isin(s_idx, [0, 18, 36])
    pn = _pink_on(o, w, s_idx[sel], chans, t_idx[sel])
    assert rel_err(got[sel][:, chans], (pk + wn)[sel][:, chans] + pn) <= TOL_TOD
    assert rel_err(got, pk + wn) <= 1e-2
    # the pink term is a few 1e-4 of P: on the noiseless scale every sampled row is right to that level, and the
    # mean over the sampled rows (pink noise averages out) to the parity gate
    assert abs(np.mean(got / (pk + wn)) - 1.0) <= 1e-4


def test_C3_full_size_sampled_rows():
    """BASELINE.json configs[2] (7-spaxel IFU, 1 h daisy scan, photon noise) at full size: >= 1 % of all rows as
    whole kernel tiles, every launch seam, last waves."""
    w = W.make_workload("C3")
    assert w.n_samples == 576000 and w.n_spaxel == 7 and w.photon_noise and not w.pink_noise
    rng = np.random.default_rng(7)
    with B.Plan(w) as p:
        _, launch = p.chunking()
        t_idx, s_idx = _sampled_tiles(w, launch, rng, 0.0105)
        assert t_idx.size >= 0.01 * w.n_samples * w.n_spaxel
        tod = p.simulate()
        got_t = tod[t_idx, s_idx.astype(np.int64)].cpu().numpy()
        del tod
        pkid = p.pkid()
        got_p = pkid[t_idx, s_idx.astype(np.int64)].cpu().numpy()
        del pkid
    pk, wn = O.Oracle(w).simulate_rows(t_idx, s_idx, noise=True)
    assert rel_err(got_p, pk) <= TOL_PKID
    assert rel_err(got_t, pk + wn) <= TOL_TOD


def test_C4_slice_tensor_against_fp32_kernel_every_element():
    """Two independent kernels (tcgen05 tensor path, FP32 CUDA-core path) on a C4 slice of more than two launches,
    compared on the device over EVERY element: a sporadic bad tile (a race in the tile pipeline) that the sampled
    oracle rows could miss shows here.  Each kernel is within 1e-5 of the oracle, so they agree to 2e-5."""
    import torch
    w = W.make_workload("C4", photon_noise=False, pink_noise=False)
    with B.Plan(w, variant=B.VARIANT_TENSOR) as pt:
        _, launch = pt.chunking()
    n = 2 * launch + 1000                                      # two full launches and a ragged third
    w = w.replace(n_samples=n, az_rad=w.az_rad[:n], el_rad=w.el_rad[:n])
    with B.Plan(w, variant=B.VARIANT_TENSOR) as pt, B.Plan(w, variant=B.VARIANT_FP32) as pf:
        assert pt.chunking()[1] == launch
        a = pt.pkid()
        b = pf.pkid()
        err = ((a - b).abs() / b.abs()).max().item()
        worst = int(((a - b).abs() / b.abs()).argmax().item())
    print("tensor vs fp32 kernel, max rel diff over", a.numel(), "elements:", err, "at flat index", worst)
    assert err <= 2e-5


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("kw", [
    dict(n_samples=1, n_spaxel=1, n_chan=1, n_freq=1),          # the smallest legal problem
    dict(n_samples=2, n_spaxel=1, n_chan=3, n_freq=5, with_cube=False),
    dict(n_samples=129, n_spaxel=1, n_chan=33, n_freq=65),      # one sample past a 128-sample row tile, one past a slab
    dict(n_samples=3, n_spaxel=130, n_chan=2, n_freq=64),       # more spaxels than rows in a tile
], ids=["1x1x1x1", "blank-2x1x3x5", "129x1x33x65", "3x130x2x64"])
def test_degenerate_sizes(variant, kw):
    w = W.random_workload(90, photon_noise=True, **kw)
    ref = O.Oracle(w).simulate(want=("tod", "pkid"))
    with _plan(w, variant) as p:
        got_p = p.pkid().cpu().numpy()
        got_t = p.simulate().cpu().numpy()
    assert rel_err(got_p, ref["pkid"]) <= TOL_PKID
    assert rel_err(got_t, ref["tod"]) <= TOL_TOD


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_pkid_with_the_filterbank_model_of_eq7(variant):
    """The paper's filterbank model (Eq. 7, upstream absorption) as the dispersive element: the hot path only
    sees the matrix."""
    w = W.random_workload(77, n_samples=140, n_spaxel=2, n_chan=96, n_freq=700)
    filt = W.filterbank_upstream_absorption(w.nu_hz, w.f_center_hz, 300.0, 0.16)
    w = w.replace(filt=filt, dnu_eff_hz=None)
    ref = O.Oracle(w).simulate(want=("pkid",))["pkid"]
    with _plan(w, variant) as p:
        got = p.pkid().cpu().numpy()
    assert rel_err(got, ref) <= TOL_PKID


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("n_samples", [600, 601, 1])
def test_tod_with_timmer_koenig_pink_noise(variant, n_samples):
    """The paper's own pink-noise method (R21): series drawn in the Fourier domain with
    PSD A f^-alpha, inverse real FFT (cuFFT) at plan creation; any sample range can then be simulated."""
    w = W.random_workload(81, n_samples=n_samples, n_spaxel=2, n_chan=20, n_freq=48, photon_noise=True, pink_noise=True)
    w = w.replace(pink_method=1, pink_A=w.pink_A * 3e3)                  # pink rms ~ 1e-3 of P: visible at the 2e-5 gate
    o = O.Oracle(w.replace(pink_noise=False))
    base = o.simulate(want=("tod",))["tod"]                              # (P + wn), Eq. 21 order
    s_idx = np.repeat(np.arange(w.n_spaxel), w.n_chan).astype(np.int32)
    c_idx = np.tile(np.arange(w.n_chan), w.n_spaxel).astype(np.int32)
    tk = O.Oracle(w).pink_tk_series(s_idx, c_idx).T.reshape(n_samples, w.n_spaxel, w.n_chan)
    ref = base + tk
    with _plan(w, variant) as p:
        got = p.simulate().cpu().numpy()
        if n_samples > 100:
            part = p.simulate(313, 200).cpu().numpy()                    # no recurrence: any range, any order
            assert np.array_equal(part, got[313:513])
    assert rel_err(got, ref) <= TOL_TOD
    if n_samples > 100:
        # the pink series itself, isolated with the GPU's own photon-noise TOD
        with _plan(w.replace(pink_noise=False), variant) as p0:
            nop = p0.simulate().cpu().numpy().astype(np.float64)
        pn = got.astype(np.float64) - nop
        assert np.max(np.abs(pn - tk)) <= 2e-4 * np.std(tk) + 1.3e-7 * np.max(np.abs(nop))


# --------------------------------------------------------------------------------------
# brightness-temperature output (R22)
def _kelvin_workload(seed=91, **kw):
    w = W.random_workload(seed, n_samples=300, n_spaxel=3, n_chan=37, n_freq=144, photon_noise=True, pink_noise=True, **kw)
    return w.replace(output_unit=1, skydip_n=12, skydip_pwv_lo_mm=0.4, skydip_pwv_hi_mm=1.7)


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_kelvin_output_through_the_skydip_map(variant):
    """tod_K = a_c + b_c (P_KID + wn + pn): the skydip runs in double on the GPU at plan creation, the map is
    applied to the finished TOD.  Tolerance: the 2e-5 gate of the noisy TOD carried through the map, i.e.
    2e-5 |b tod_W|, plus fp32 rounding of the two terms of the line."""
    w = _kelvin_workload()
    o = O.Oracle(w)
    a, b = o.kelvin_map()
    tod_w = o.simulate(want=("tod",))["tod"]
    ref = a + b * tod_w
    with _plan(w, variant) as p:
        ga, gb = p.kelvin_map()
        got = p.simulate().cpu().numpy().astype(np.float64)
        host = p.simulate(device_out=False)
        pk = p.pkid().cpu().numpy()                                   # the noiseless hook stays in W
    assert np.max(np.abs(gb / b - 1.0)) <= 1e-6 and np.max(np.abs(ga - a)) <= 1e-6 * np.max(np.abs(ref))
    tol = 2e-5 * np.abs(b * tod_w) + 3e-7 * (np.abs(a) + np.abs(b * tod_w))
    assert np.all(np.abs(got - ref) <= tol)
    assert np.array_equal(np.asarray(host, dtype=np.float64), got)
    assert rel_err(pk, o.simulate(want=("pkid",))["pkid"]) <= TOL_PKID
    # the brightness scale is sensible: between the CMB and the atmosphere's physical temperature
    assert ref.min() > 0 and np.median(got) < w.T_atm_K


def test_kelvin_output_rejects_what_it_cannot_calibrate():
    w = _kelvin_workload()
    for bad, status in ((dict(skydip_n=1), 2), (dict(skydip_pwv_hi_mm=0.4), 3), (dict(output_unit=2), 3)):
        with pytest.raises(B.GateauError) as e:
            B.Plan(w.replace(**bad), variant=B.VARIANT_FP32)
        assert e.value.status == status
    filt = np.array(w.filt, copy=True)
    filt[5] = 0.0
    with pytest.raises(B.GateauError) as e:
        B.Plan(w.replace(filt=filt), variant=B.VARIANT_FP32)
    assert e.value.status == 3 and "channel 5" in str(e.value)
    with _plan(w.replace(output_unit=0), B.VARIANT_FP32) as p:
        with pytest.raises(B.GateauError):
            p.kelvin_map()


# --------------------------------------------------------------------------------------
# exact photon noise, Eq. 17 (R23)
@pytest.mark.parametrize("case", ["random", "lorentzian", "nocube"])
def test_exact_photon_noise_eq17(case):
    """photon_mode = 1: sigma from the full Eq. 17 on each row's own spectrum (three contractions through the
    tensor kernel), same normals as the narrow-band mode.  The TOD meets the 2e-5 gate; sigma itself, isolated
    with the GPU's own noiseless power, agrees with the oracle's to 1e-3 (it only scales a noise draw)."""
    if case == "random":
        w = W.random_workload(101, n_samples=260, n_spaxel=3, n_chan=37, n_freq=144, photon_noise=True)
    elif case == "nocube":
        w = W.random_workload(102, n_samples=131, n_spaxel=2, n_chan=20, n_freq=70, photon_noise=True, with_cube=False)
    else:
        w = W.random_workload(103, n_samples=200, n_spaxel=2, n_chan=30, n_freq=512, photon_noise=True)
        fc = np.linspace(w.nu_hz[40], w.nu_hz[-40], 30)
        w = w.replace(filt=W.lorentzian_filterbank(w.nu_hz, fc, 200.0, 0.16), f_center_hz=fc, dnu_eff_hz=None)
    w = w.replace(photon_mode=1)
    o = O.Oracle(w)
    t_idx = np.repeat(np.arange(w.n_samples), w.n_spaxel)
    s_idx = np.tile(np.arange(w.n_spaxel), w.n_samples)
    pk, wn = o.simulate_rows_exact(t_idx, s_idx)
    ref = (pk + wn).reshape(w.n_samples, w.n_spaxel, w.n_chan)
    with _plan(w, B.VARIANT_TENSOR) as p:
        got = p.simulate().cpu().numpy().astype(np.float64)
        nop = p.pkid().cpu().numpy().astype(np.float64)
        part = p.simulate(57, 40).cpu().numpy()
    assert rel_err(got, ref) <= TOL_TOD
    assert np.array_equal(part, got[57:97].astype(np.float32))
    wn_g = (got - nop).reshape(-1, w.n_chan)
    big = np.abs(wn) > 0.3 * np.abs(wn).std()                       # ratios are meaningful where the draw is not ~0
    ratio = wn_g[big] / wn[big]
    assert np.max(np.abs(ratio - 1.0)) <= 1e-3 + 4e-7 * np.max(np.abs(pk)) / np.min(np.abs(wn[big]))
    # and it is not the narrow-band sigma: the generation-recombination term raises it
    _, wn0 = o.simulate_rows(t_idx, s_idx, noise=True)
    assert np.median(np.abs(wn[big] / wn0[big])) > 1.02


def test_exact_photon_noise_needs_the_tensor_variant():
    w = W.random_workload(104, n_samples=8, n_spaxel=1, n_chan=4, n_freq=16, photon_noise=True).replace(photon_mode=1)
    with pytest.raises(B.GateauError) as e:
        B.Plan(w, variant=B.VARIANT_FP32)
    assert e.value.status == 7
    with pytest.raises(B.GateauError) as e:
        B.Plan(w.replace(eta_pb=0.0), variant=B.VARIANT_TENSOR)
    assert e.value.status == 3


def test_C2_full_size_exact_photon_noise_and_kelvin():
    """BASELINE.json configs[1] at full size with the paper's own options switched on: Eq. 17 photon noise (R23) and
    brightness-temperature output (R22), on sampled rows."""
    w = W.make_workload("C2").replace(photon_noise=True, photon_mode=1, output_unit=1,
                                      skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.4)
    rng = np.random.default_rng(11)
    t_idx = np.sort(rng.choice(w.n_samples, 64, replace=False)).astype(np.int64)
    t_idx[0] = 0; t_idx[-1] = w.n_samples - 1
    s_idx = rng.integers(0, w.n_spaxel, t_idx.size).astype(np.int32)
    o = O.Oracle(w)
    pk, wn = o.simulate_rows_exact(t_idx, s_idx)
    a, b = o.kelvin_map()
    ref = a + b * (pk + wn)
    with B.Plan(w) as p:
        tod = p.simulate()
        got = tod[t_idx, s_idx.astype(np.int64)].cpu().numpy().astype(np.float64)
        del tod
    tol = 2e-5 * np.abs(b * (pk + wn)) + 3e-7 * (np.abs(a) + np.abs(b * (pk + wn)))
    assert np.all(np.abs(got - ref) <= tol)


# --------------------------------------------------------------------------------------
# screen pre-processing (R24)
@pytest.mark.parametrize("shape,dx,dy,R,taper", [((37, 53), 0.7, 0.9, 3.0, -11.0), ((200, 131), 0.25, 0.25, 5.0, -10.0),
                                                 ((5, 4), 1.0, 1.0, 7.5, -3.0), ((64, 64), 2.0, 2.0, 1.0, -10.0),
                                                 ((96, 160), 0.5, 1.0, 30.0, -12.0)])
def test_screen_preprocessing(shape, dx, dy, R, taper):
    """Eq. 4 + footprint smoothing through gt_prepare_screen against the oracle: ragged tiles, a screen smaller than
    the footprint (wraps several times), a footprint of one pixel, an anisotropic grid, a 60-pixel radius."""
    import torch
    rng = np.random.default_rng(5)
    epl = rng.normal(0.0, 0.4, shape).astype(np.float32)
    ref = O.screen_line_of_sight(epl, dx, dy, R, taper, 1.1)
    got = B.gt_prepare_screen(torch.from_numpy(epl).cuda(), dx, dy, R, taper, 1.1).cpu().numpy()
    assert got.dtype == np.float32 and got.shape == shape
    assert np.max(np.abs(got - ref)) <= 3e-7 * 1.1 + 2e-6 * np.max(np.abs(ref - 1.1))


def test_screen_preprocessing_rejects_bad_arguments():
    import torch
    epl = torch.zeros((8, 8), dtype=torch.float32, device="cuda")
    for args, status in (((0.0, 1.0, 2.0, -10.0, 1.0), 3), ((1.0, 1.0, -2.0, -10.0, 1.0), 3), ((0.01, 1.0, 2.0, -10.0, 1.0), 7)):
        with pytest.raises(B.GateauError) as e:
            B.gt_prepare_screen(epl, *args)
        assert e.value.status == status
    with pytest.raises(B.GateauError) as e:
        B.gt_prepare_screen(epl, 1.0, 1.0, 2.0, -10.0, 1.0, out=epl)
    assert e.value.status == 3


# --------------------------------------------------------------------------------------
# source pre-processing: far field + beam convolution (R25)
@pytest.mark.parametrize("n_el,n_az,n_freq,r,taper,pitch", [(9, 11, 5, 3, -10.0, 6.0), (20, 7, 130, 2, 0.0, 4.0),
                                                           (3, 4, 3, 6, -14.0, 3.5), (6, 6, 2, 0, -10.0, 5.0)])
def test_source_preprocessing(n_el, n_az, n_freq, r, taper, pitch):
    """gt_prepare_source against the oracle: Hankel-transform far field (Simpson on the GPU, adaptive quadrature in
    the oracle) and the direct convolution with zero intensity outside the cube; kernels wider than the cube, more
    than one frequency block, no taper (Airy), r_pix = 0 (beam = on-axis value only)."""
    import torch
    rng = np.random.default_rng(8)
    I = (1e-18 * rng.random((n_el, n_az, n_freq))).astype(np.float32)
    nu0, dnu = 230e9, 1.7e9
    nu = nu0 + dnu * np.arange(n_freq)
    d = pitch * np.pi / 180 / 3600
    el_first = np.deg2rad(58.0)
    f_idx = np.unique(np.linspace(0, n_freq - 1, 4).astype(int))          # the oracle's quadrature is slow: sampled frequencies
    ref = O.source_power(I[:, :, f_idx], nu[f_idx], d, 1.25 * d, el_first, r, 5.0, taper)
    got = B.gt_prepare_source(torch.from_numpy(I).cuda(), nu0, dnu, d, 1.25 * d, el_first, 5.0, taper, r).cpu().numpy()
    assert got.shape == I.shape and got.dtype == np.float32
    assert np.max(np.abs(got[:, :, f_idx] - ref)) <= 5e-7 * np.max(np.abs(ref))


def test_source_preprocessing_rejects_bad_arguments():
    import torch
    I = torch.zeros((4, 4, 4), dtype=torch.float32, device="cuda")
    for kw, status in ((dict(r_pix=65), 2), (dict(R_tel_m=0.0), 3), (dict(daz_rad=-1e-5), 3)):
        a = dict(nu0_hz=2e11, dnu_hz=1e9, daz_rad=2e-5, del_rad=2e-5, el_first_rad=1.0, R_tel_m=5.0, t_edge_db=-10.0, r_pix=2)
        a.update(kw)
        with pytest.raises(B.GateauError) as e:
            B.gt_prepare_source(I, **a)
        assert e.value.status == status


def test_common_mode_subtraction_sharded_and_single_plan_against_the_oracle():
    """Eq. 25-26 on the Kelvin TOD: one plan holding every spaxel, and three plans holding spaxel
    sub-ranges whose partial sums are added (the all-reduce of a sharded run), against the oracle's literal formula
    evaluated on the same TOD.  The shards' TODs are bit-identical slices of the full plan's."""
    import torch
    from paper_2604_23305_b200 import shard
    w = W.random_workload(121, n_samples=150, n_spaxel=7, n_chan=21, n_freq=80, photon_noise=True)
    w = w.replace(output_unit=1, skydip_n=10, skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.7)
    r_out = 8 * np.pi / 180 / 3600                                  # offsets are +-10 arcsec: some spaxels inside, some outside
    o = O.Oracle(w)
    with B.Plan(w) as p:
        tod, pwv = p.simulate(want_pwv=True)
        pwv_mean = float(pwv.double().mean().item())
        partial, n_out = p.common_mode_partial(tod, pwv_mean, r_out)
        got = p.common_mode_apply(tod.clone(), pwv_mean, partial, n_out).cpu().numpy().astype(np.float64)
        tod_np = tod.cpu().numpy()
    eta_z = O.eta_zenith_at(w, w.f_center_hz, pwv_mean)
    csc = o.geometry()["csc"]
    ref, S, common = O.common_mode_subtract(tod_np.astype(np.float64), eta_z, csc, w.daz_rad, w.del_rad, r_out)
    assert 0 < S.sum() < w.n_spaxel and n_out == int(S.sum())
    scale = np.max(np.abs(tod_np / (eta_z[None, None, :] ** csc[:, :, None])))
    assert np.max(np.abs(partial.cpu().numpy() - common)) <= 3e-7 * np.max(np.abs(common))
    assert np.max(np.abs(got - ref)) <= 3e-7 * scale
    # spaxel shards: partial sums and counts added over the plans, then each finishes its own slab
    parts = shard.partition_spaxels(w.n_spaxel, 3)
    plans = [B.Plan(shard.shard_workload(w, b, e)) for b, e in parts]
    try:
        tods = [q.simulate() for q in plans]
        for (b, e), t in zip(parts, tods):
            assert np.array_equal(t.cpu().numpy(), tod_np[:, b:e])
        ps = [q.common_mode_partial(t, pwv_mean, r_out) for q, t in zip(plans, tods)]
        total = torch.stack([x[0] for x in ps]).sum(dim=0)
        n_tot = sum(x[1] for x in ps)
        assert n_tot == n_out
        outs = [q.common_mode_apply(t, pwv_mean, total, n_tot).cpu().numpy() for q, t in zip(plans, tods)]
    finally:
        for q in plans:
            q.destroy()
    assert np.max(np.abs(np.concatenate(outs, axis=1) - ref)) <= 3e-7 * scale
    with B.Plan(w) as p:
        with pytest.raises(B.GateauError) as e:
            p.common_mode_apply(tod, pwv_mean, partial, 0)
        assert e.value.status == 3


def test_common_mode_subtraction_over_a_wide_elevation_range():
    """The common-mode kernels form eta = eta_z^csc from its value at the boresight airmass and a short fp32 polynomial
    in x = (csc - csc0) ln eta_z, with the library functions beyond |x| = 0.05 (csrc/gt_common_mode.cuh).  A scan over
    +-9 degrees of elevation puts |x| on both sides of that switch (0 ... 0.3); same oracle, same 3e-7."""
    w = W.random_workload(122, n_samples=200, n_spaxel=5, n_chan=33, n_freq=80, photon_noise=True)
    w = w.replace(output_unit=1, skydip_n=10, skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.7,
                  el_rad=np.linspace(-0.16, 0.16, 200))
    r_out = 8 * np.pi / 180 / 3600
    o = O.Oracle(w)
    with B.Plan(w) as p:
        tod, pwv = p.simulate(want_pwv=True)
        pwv_mean = float(pwv.double().mean().item())
        partial, n_out = p.common_mode_partial(tod, pwv_mean, r_out)
        got = p.common_mode_apply(tod.clone(), pwv_mean, partial, n_out).cpu().numpy().astype(np.float64)
        got_static, n_static = p.common_mode_static(tod.clone(), pwv_mean, r_out)
        tod_np = tod.cpu().numpy()
    eta_z = O.eta_zenith_at(w, w.f_center_hz, pwv_mean)
    csc = o.geometry()["csc"]
    x = (csc - 1.0 / np.sin(w.el0_rad))[:, :, None] * np.log(eta_z)[None, None, :]
    assert np.abs(x).min() < 1e-3 and (np.abs(x) > 0.05).mean() > 0.2 and (np.abs(x) < 0.05).mean() > 0.2
    ref, S, common = O.common_mode_subtract(tod_np.astype(np.float64), eta_z, csc, w.daz_rad, w.del_rad, r_out)
    assert 0 < S.sum() and n_out == int(S.sum()) == n_static
    scale = np.max(np.abs(tod_np / (eta_z[None, None, :] ** csc[:, :, None])))
    assert np.max(np.abs(partial.cpu().numpy() - common)) <= 3e-7 * np.max(np.abs(common))
    assert np.max(np.abs(got - ref)) <= 3e-7 * scale
    assert np.array_equal(got_static.cpu().numpy(), got.astype(np.float32))


def test_measurement_hooks_and_plan_pool():
    """gt_debug_timeline (per-chunk compute / copy events of a host-output call: every copy starts after its chunk's
    kernels and ends after it started), gt_measure_fp32_fma (tens of TFLOP/s on a B200), gt_release_cached_memory
    (plans created after the pool was trimmed still work and give the same TOD)."""
    w = W.random_workload(131, n_samples=400, n_spaxel=3, n_chan=40, n_freq=64, photon_noise=True)
    with B.Plan(w, chunk_samples=64) as p:
        host = p.simulate(device_out=False).numpy().copy()
        tl = p.timeline()
        assert p.chunking()[0] == 64
    assert tl.shape == (7, 4)                                   # 400 samples in chunks of 64
    assert np.all(tl[:, 1] >= tl[:, 0]) and np.all(tl[:, 2] >= tl[:, 1]) and np.all(tl[:, 3] >= tl[:, 2])
    assert np.all(np.diff(tl[:, 0]) >= 0) and np.all(np.diff(tl[:, 3]) >= 0)
    B.release_cached_memory()
    with B.Plan(w, chunk_samples=64) as p:
        again = p.simulate(device_out=False).numpy()
    assert np.array_equal(host, again)
    assert 20.0 < B.measure_fp32_fma() < 100.0


def test_all_paper_options_together_streamed():
    """The paper's own choices at once -- Eq. 7 filterbank, Eq. 17 photon noise, Timmer & Koenig pink noise, Kelvin
    output -- streamed to host memory in ragged chunks; device and host outputs are identical."""
    w = W.random_workload(111, n_samples=333, n_spaxel=2, n_chan=24, n_freq=160, photon_noise=True, pink_noise=True)
    fc = np.geomspace(w.nu_hz[30], w.nu_hz[-30], 24)
    w = w.replace(filt=W.filterbank_upstream_absorption(w.nu_hz, fc, 80.0, 0.16), f_center_hz=fc, dnu_eff_hz=None,
                  photon_mode=1, pink_method=1, pink_A=w.pink_A * 3e3, output_unit=1,
                  skydip_pwv_lo_mm=0.5, skydip_pwv_hi_mm=1.6, chunk_samples=64)
    o = O.Oracle(w)
    t_idx = np.repeat(np.arange(w.n_samples), w.n_spaxel)
    s_idx = np.tile(np.arange(w.n_spaxel), w.n_samples)
    pk, wn = o.simulate_rows_exact(t_idx, s_idx)
    d_s = np.repeat(np.arange(w.n_spaxel), w.n_chan).astype(np.int32)
    d_c = np.tile(np.arange(w.n_chan), w.n_spaxel).astype(np.int32)
    tk = o.pink_tk_series(d_s, d_c).T.reshape(w.n_samples, w.n_spaxel, w.n_chan)
    a, b = o.kelvin_map()
    tod_w = (pk + wn).reshape(w.n_samples, w.n_spaxel, w.n_chan) + tk
    ref = a + b * tod_w
    with _plan(w, B.VARIANT_TENSOR) as p:
        dev = p.simulate().cpu().numpy()
        host = np.asarray(p.simulate(device_out=False))
    assert np.array_equal(dev, host)
    tol = 2e-5 * np.abs(b * tod_w) + 3e-7 * (np.abs(a) + np.abs(b * tod_w))
    assert np.all(np.abs(dev.astype(np.float64) - ref) <= tol)
