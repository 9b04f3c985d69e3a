"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, on the same seeded inputs.

Bars (BASELINE.json north_star): integer / index work bit-exact; fp64 field relative L2 <= 1e-10
(complex, no global-phase removal); mixed mode <= 1e-4.
"""
import math

import numpy as np
import pytest
import torch

import gen
import oracle

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
TOLMIX = 1e-4
# Figure of merit (peak-normalised intensity I = |E|^2/|E0|^2 against Airy): a field within TOL64 of the peak per pixel
# and an on-axis value within TOL64 move I by at most 2 |E| dE/|E0|^2 + 2 I dE0/|E0| <= 4 TOL64 in absolute terms, and
# the RMS / maximum of (I - Airy) by no more than that.
ATOL_METRIC = 4 * TOL64
# What the kernels actually use of that bound (B200, round 3; the tests print it): RMS values deviate from the oracle's
# by <= 2.8e-13, the maximum of |I - Airy| by 5.9e-12; two algorithms on the GPU differ by <= 1.2e-12 in the RMS values.
# The asserted bars are min(derived bound, 10 x measured), so a regression of the per-term accuracy shows here first:
ATOL_RMS = min(ATOL_METRIC, 3e-12)          # RMS figures of merit against the oracle
ATOL_MAXDIFF = min(ATOL_METRIC, 6e-11)      # max |I - Airy| against the oracle
ATOL_RMS_ALGOS = min(ATOL_METRIC, 1.5e-11)  # GPU against GPU, different algorithms (direct / recurrence / separable)
RTOL_SAME_ALGO = 1e-9                       # GPU against GPU, the same kernels through another call path


@pytest.fixture(scope="module")
def G():
    from paper_2404_12454_b200 import build
    build.build()
    import paper_2404_12454_b200 as g
    g.load_library()
    return g


def rel_l2(a, b):
    a = np.asarray(a).astype(np.complex128)
    b = np.asarray(b).astype(np.complex128)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def max_pixel_err(a, b):
    """Largest single-pixel deviation, relative to the peak of the reference field."""
    a = np.asarray(a).astype(np.complex128)
    b = np.asarray(b).astype(np.complex128)
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b))) if b.size else 0.0


def deep_word(b):
    """The device word by which the pre-pass of the last gbd_eval_field call on `b` told the table kernels which of the
    gated pair runs (0: the fast kernel on detector-coordinate records; 1: its beamlet-centred twin).  It sits behind
    the two record regions of the workspace (gbd_api.cu: [n][16] and [n][14] doubles, each rounded up to 256 bytes),
    second int of the gate block."""
    up = lambda x: (x + 255) // 256 * 256
    off = up(b.n * 16 * 8) + up(b.n * 14 * 8) + 4
    torch.cuda.synchronize()
    return int(b._ws[off:off + 4].view(torch.int32).item())


def assert_field_close(got, ref, tol, what=None):
    """The bar of BASELINE.json (relative L2 over the compared pixels) AND a bound on every single pixel:
    |got - ref| <= tol * max|ref| ("per-pixel bound"), so that no pixel can hide in the norm."""
    e2, epx = rel_l2(got, ref), max_pixel_err(got, ref)
    assert np.all(np.isfinite(np.asarray(got).view(np.float64 if np.asarray(got).dtype == np.complex128
                                                   else np.float32))), what
    assert e2 < tol, (what, "rel-L2", e2)
    assert epx <= tol, (what, "worst pixel / peak", epx)


FULL_GRID_CORES = 8     # host threads from which the minute-long full-grid oracle comparisons run unthinned


def _report_thinning(step, what):
    """A comparison that had to be thinned (few host cores) passed on what it compared, but must not look like
    the full-grid one in the log: it is reported as SKIPPED with the reason."""
    if step != 1:
        pytest.skip(f"PARTIAL COMPARISON (passed): only every {step}th of the {what} was compared, because the "
                    f"host has {oracle.num_threads()} < {FULL_GRID_CORES} oracle threads")


def oracle_run(w, rows=None):
    return oracle.run_workload(w, gen.make_inputs, rows=rows)


# ----------------------------------------------------------------------------- a1

@pytest.mark.parametrize("n", [1, 2, 11, 51, 64, 101, 201])
def test_lattice_bit_exact(G, n):
    ref = oracle.lattice(n, 25.4)
    b = G.beamlets_create(n, 25.4, 1.5, 0.6328e-3)
    assert b.n == ref.shape[1]
    got = b.positions.cpu().numpy()
    assert np.array_equal(got, ref)
    assert b.waist == oracle.waist(1.5, 25.4 / n)


# ----------------------------------------------------------------------------- a2

def param_err(got, ref):
    scale = np.maximum(np.abs(ref), np.max(np.abs(ref), axis=0, keepdims=True) * 1e-3 + 1e-300)
    return float(np.max(np.abs(got - ref) / scale))


@pytest.mark.parametrize("idx", [0, 1, 3, 4])
def test_parameter_records_match_oracle(G, idx):
    w = gen.workload(idx)
    if idx == 3:
        w = gen.Workload(**{**w.__dict__, "n_across": 61})
    r = oracle_run(w, rows=(0, 1, 1))
    g = G.run_workload(w, gen.make_inputs)
    got = g["params"].cpu().numpy()
    # amplitude compared as a complex number, the rest column by column
    assert param_err(got[:, :11], r["rec"][:, :11]) < 1e-11
    amp_g = got[:, 11] + 1j * got[:, 12]
    amp_r = r["rec"][:, 11] + 1j * r["rec"][:, 12]
    assert np.max(np.abs(amp_g - amp_r) / np.abs(amp_r)) < 1e-12
    # the optical path must agree to a tiny fraction of a wavelength (it is the 1e5-turn term)
    assert np.max(np.abs(got[:, 4] - r["rec"][:, 4])) < 1e-12 * w.wavelength * 1e3


# ----------------------------------------------------------------------------- a3 + a4, full configs

def test_field_c0(G):
    w = gen.workload(0)
    r = oracle_run(w)
    g = G.run_workload(w, gen.make_inputs)
    assert_field_close(g["field"].cpu().numpy(), r["field"], TOL64)


def test_field_c1(G):
    w = gen.workload(1)
    r = oracle_run(w)
    g = G.run_workload(w, gen.make_inputs)
    assert_field_close(g["field"].cpu().numpy(), r["field"], TOL64)


@pytest.mark.parametrize("n,of", [(11, 1.0), (31, 3.0), (61, 1.5), (101, 2.25)])
def test_field_c2_sweep_members(G, n, of):
    w = gen.workload(2, n, of)
    r = oracle_run(w, rows=(0, 256, 4))
    g = G.run_workload(w, gen.make_inputs)
    got = g["field"].cpu().numpy()
    assert_field_close(got[0:256:4], r["field"][0:256:4], TOL64)


def test_field_c3_sampled_rows_full_size(G):
    """Full-size C3 in the launch configuration bench.py times; the oracle does 12 of 1024 rows
    (centre, corners and a spread), every pixel of those rows compared."""
    w = gen.workload(3)
    g = G.run_workload(w, gen.make_inputs)
    got = g["field"].cpu().numpy()
    rows = [0, 1, 255, 256, 511, 512, 513, 700, 767, 1000, 1022, 1023]
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    rd = oracle.to_detector(rec, inp["detector"])
    ref = np.zeros((1024, 1024), dtype=np.complex128)
    for v in rows:
        oracle.field_rows(rd, inp["detector"], w.wavelength, v, v + 1, 1, out=ref)
    assert_field_close(got[rows], ref[rows], TOL64)


def test_field_c4_tilted_full(G):
    """BASELINE.json configs[4] at full size, every pixel of every row (2.1e9 terms: seconds of oracle time)."""
    w = gen.workload(4)
    r = oracle_run(w)
    g = G.run_workload(w, gen.make_inputs)
    assert_field_close(g["field"].cpu().numpy(), r["field"], TOL64)


# ----------------------------------------------------------------------------- edge cases

def small_case(G, n_u, n_v, n_across=9, tilt=False, cull_tau=0.0, precision=0, algo=0):
    w = gen.workload(0)
    xy = oracle.lattice(n_across, w.pupil_diameter)
    w0 = oracle.waist(1.5, w.pupil_diameter / n_across)
    abcd = gen.ideal_lens_abcd(w.focal_length, 0.3).reshape(16)
    rng = np.random.default_rng(n_u * 1000 + n_v)
    wt = rng.standard_normal((2, xy.shape[1]))
    base = np.stack([rng.uniform(-1e-4, 1e-4, xy.shape[1]), rng.uniform(-1e-4, 1e-4, xy.shape[1]),
                     rng.uniform(-1e-3, 1e-3, xy.shape[1])])
    det = dict(n_u=n_u, n_v=n_v, du=0.9e-3, dv=1.1e-3, origin=[2e-3, -1e-3, 0.0],
               e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    if tilt:
        t = 0.2
        det.update(origin=[2e-3, -1e-3, 5e-3], e_u=[math.cos(t), 0.0, -math.sin(t)], e_v=[0.0, 1.0, 0.0])
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, 100.3, base, wt)
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength, cull_tau)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, 100.3, base, wt)
    got = G.eval_field(b, det, precision=precision, algo=algo, cull_tau=cull_tau).cpu().numpy()
    return got, ref


@pytest.mark.parametrize("n_u,n_v", [(1, 1), (1, 37), (37, 1), (31, 5), (33, 7), (64, 64), (65, 3),
                                     (127, 9), (129, 2), (300, 11), (1000, 3)])
def test_ragged_detectors(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v)
    assert got.shape == ref.shape == (n_v, n_u)
    assert_field_close(got, ref, TOL64)


@pytest.mark.parametrize("n_across", [1, 2, 3, 13])
def test_few_beamlets(G, n_across):
    got, ref = small_case(G, 50, 20, n_across=n_across)
    assert_field_close(got, ref, TOL64)


def test_tilted_small(G):
    got, ref = small_case(G, 70, 33, tilt=True)
    assert_field_close(got, ref, TOL64)


def test_zero_beamlets_gives_zero_field(G):
    xy = np.zeros((2, 0))
    b = G.beamlets_custom(xy, 1.0, 1e-3)
    G.propagate_q(b, 1, gen.ideal_lens_abcd(100.0).reshape(16), 100.0)
    det = dict(n_u=17, n_v=5, du=1e-3, dv=1e-3, origin=[0, 0, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    out = torch.full((5, 17), 3.0 + 1j, dtype=torch.complex128, device="cuda:0")
    G.eval_field(b, det, out=out)
    assert torch.count_nonzero(out).item() == 0


def test_zero_weight_beamlets_vanish(G):
    w = gen.workload(0)
    xy = oracle.lattice(7, w.pupil_diameter)
    wt = np.ones((2, xy.shape[1]))
    wt[:, ::2] = 0.0
    abcd = gen.ideal_lens_abcd(100.0).reshape(16)
    det = dict(n_u=40, n_v=12, du=1e-3, dv=1e-3, origin=[0, 0, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    rec = oracle.propagate(xy, 2.0, w.wavelength, 1, abcd, 100.0, None, wt)
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
    b = G.beamlets_custom(xy, 2.0, w.wavelength)
    G.propagate_q(b, 1, abcd, 100.0, None, wt)
    got = G.eval_field(b, det).cpu().numpy()
    assert_field_close(got, ref, TOL64)


def test_zero_weight_beamlets_on_the_table_kernels(G):
    """An apodised pupil with exact zeros (a spider / central obscuration mask) at a size that takes the table kernels
    (2,053 beamlets x 256 x 256 px = 1.3e8 terms): the zero-weight beamlets contribute nothing, and they do not push
    the launch off the fast path (their detector-coordinate record is a constant 2^-1000)."""
    w = gen.workload(1)
    ref_run = G.run_workload(w, gen.make_inputs)
    inp, b = ref_run["inputs"], ref_run["beamlets"]
    xy = np.asarray(inp["xy"])
    wt = np.ones((2, b.n))
    wt[1] = 0.0
    r = np.hypot(xy[0], xy[1])
    mask = (r < 0.33 * 0.5 * w.pupil_diameter) | (np.abs(xy[0]) < 0.02 * w.pupil_diameter) | (np.abs(xy[1]) < 0.02 * w.pupil_diameter)
    wt[:, mask] = 0.0
    assert 100 < mask.sum() < b.n - 100
    G.propagate_q(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], wt)
    det = inp["detector"]
    rec = oracle.propagate(xy, b.waist, w.wavelength, inp["abcd_mode"], np.asarray(inp["abcd"]), inp["l0"], inp["base"], wt)
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
    for algo in (0, 1, 2):
        got = G.eval_field(b, det, algo=algo).cpu().numpy()
        if algo == 0:
            assert deep_word(b) == 0                           # the zero weights did not push the launch off the fast path
        assert_field_close(got, ref, TOL64, algo)
    # the same pupil without the masked beamlets at all
    keep = ~mask
    b2 = G.beamlets_custom(xy[:, keep], b.waist, w.wavelength)
    base2 = None if inp["base"] is None else np.asarray(inp["base"])[:, keep]
    G.propagate_q(b2, inp["abcd_mode"], inp["abcd"], inp["l0"], base2, wt[:, keep])
    got2 = G.eval_field(b2, det).cpu().numpy()
    assert_field_close(got2, ref, TOL64, "masked beamlets removed")


def test_cull_matches_oracle_threshold(G):
    """Out-of-focus plane (beamlets much narrower than the detector): most terms are culled."""
    w = gen.workload(1)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    w0 = oracle.waist(1.5, w.pupil_diameter / 21)
    det = dict(n_u=96, n_v=64, du=0.13, dv=0.2, origin=[0, 0, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    rd = oracle.to_detector(rec, det)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f / 2)
    for tau in (1e-18, 1e-6):
        ref = oracle.field(rd, det, w.wavelength, tau)
        got = G.eval_field(b, det, cull_tau=tau).cpu().numpy()
        amp = np.hypot(rd[:, 11], rd[:, 12])
        # boundary-rounding disagreements change a pixel by at most tau*|amp| per term (R-14)
        assert np.max(np.abs(got - ref)) <= 4 * tau * amp.max() + 1e-10 * np.max(np.abs(ref))
    ref0 = oracle.field(rd, det, w.wavelength, 0.0)
    got0 = G.eval_field(b, det).cpu().numpy()
    assert_field_close(got0, ref0, TOL64)
    # a wide detector: most (beamlet, strip) pairs are skipped as a whole by the strip-level test
    det2 = dict(n_u=1024, n_v=48, du=0.0125, dv=0.26, origin=[0.3, -0.2, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    rd2 = oracle.to_detector(rec, det2)
    for tau in (1e-18, 1e-3):
        ref = oracle.field(rd2, det2, w.wavelength, tau)
        got = G.eval_field(b, det2, cull_tau=tau).cpu().numpy()
        assert np.max(np.abs(got - ref)) <= 4 * tau * amp.max() + 1e-10 * np.max(np.abs(ref))
        gm = G.eval_field(b, det2, cull_tau=tau, precision=G.PRECISION_MIXED).cpu().numpy()
        assert_field_close(gm, ref, 2e-3 if tau > 1e-6 else TOLMIX)


def test_bitwise_reproducible(G):
    w = gen.workload(1)
    g = G.run_workload(w, gen.make_inputs)
    a = g["field"].clone()
    b2 = G.eval_field(g["beamlets"], g["inputs"]["detector"])
    assert torch.equal(a.view(torch.float64), b2.view(torch.float64))


def test_host_call_equals_device_path(G):
    w = gen.workload(0)
    g = G.run_workload(w, gen.make_inputs)
    b, inp = g["beamlets"], g["inputs"]
    need = G.host_workspace_bytes(b, inp["detector"], inp["abcd_mode"])
    ws = torch.empty(need, dtype=torch.uint8, device="cuda:0")
    h_xy = torch.as_tensor(inp["xy"]).contiguous().pin_memory()
    h_abcd = torch.as_tensor(inp["abcd"]).contiguous().pin_memory()
    h_field = torch.empty((64, 64), dtype=torch.complex128).pin_memory()
    G.eval_field_host(b, h_xy, inp["abcd_mode"], h_abcd, inp["l0"], None, None, inp["detector"],
                      h_field, ws)
    assert torch.equal(h_field.view(torch.float64), g["field"].cpu().view(torch.float64))


def test_errors_are_loud(G):
    w = gen.workload(0)
    b = G.beamlets_create(w.n_across, w.pupil_diameter, 1.5, w.wavelength)
    det = gen.detector_dict(w)
    with pytest.raises(G.GbdError):
        G.eval_field(b, det, params=torch.zeros((b.n, 13), dtype=torch.float64, device="cuda:0"))


# ----------------------------------------------------------------------------- mixed precision

@pytest.mark.parametrize("idx", [0, 1, 4])
def test_mixed_mode_small_configs(G, idx):
    w = gen.workload(idx)
    if idx == 4:
        w = gen.Workload(**{**w.__dict__, "det_n": 128})
    r = oracle_run(w)
    g = G.run_workload(w, gen.make_inputs, precision=G.PRECISION_MIXED)
    assert g["field"].dtype == torch.complex64
    assert_field_close(g["field"].cpu().numpy(), r["field"], TOLMIX)


def test_mixed_mode_c3_sampled_rows(G):
    w = gen.workload(3)
    g = G.run_workload(w, gen.make_inputs, precision=G.PRECISION_MIXED)
    got = g["field"].cpu().numpy()
    rows = [0, 300, 511, 512, 800, 1023]
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    rd = oracle.to_detector(rec, inp["detector"])
    ref = np.zeros((1024, 1024), dtype=np.complex128)
    for v in rows:
        oracle.field_rows(rd, inp["detector"], w.wavelength, v, v + 1, 1, out=ref)
    assert_field_close(got[rows], ref[rows], TOLMIX)


@pytest.mark.parametrize("n_u,n_v", [(1, 1), (33, 7), (129, 2), (300, 11)])
def test_mixed_ragged(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v, precision=1)
    assert_field_close(got, ref, TOLMIX)


def test_mixed_cull(G):
    got, ref = small_case(G, 100, 40, precision=1, cull_tau=1e-6)
    assert_field_close(got, ref, TOLMIX)


# ----------------------------------------------------------------------------- recurrence (algo = 1)

@pytest.mark.parametrize("idx", [0, 1, 4])
def test_recurrence_configs(G, idx):
    w = gen.workload(idx)
    r = oracle_run(w, rows=(0, w.det_n, 4))
    g = G.run_workload(w, gen.make_inputs, algo=G.ALGO_RECURRENCE)
    got = g["field"].cpu().numpy()
    assert_field_close(got[0:w.det_n:4], r["field"][0:w.det_n:4], TOL64)


def test_recurrence_c3_sampled_rows(G):
    w = gen.workload(3)
    g = G.run_workload(w, gen.make_inputs, algo=G.ALGO_RECURRENCE)
    got = g["field"].cpu().numpy()
    rows = [0, 1, 256, 511, 512, 640, 1000, 1023]
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    rd = oracle.to_detector(rec, inp["detector"])
    ref = np.zeros((1024, 1024), dtype=np.complex128)
    for v in rows:
        oracle.field_rows(rd, inp["detector"], w.wavelength, v, v + 1, 1, out=ref)
    assert_field_close(got[rows], ref[rows], TOL64)
    # and against the direct algorithm on every pixel
    gd = G.eval_field(g["beamlets"], g["inputs"]["detector"]).cpu().numpy()
    assert rel_l2(got, gd) < 1e-11


@pytest.mark.parametrize("n_u,n_v", [(65, 3), (127, 9), (129, 2), (300, 11), (513, 4), (1000, 3), (1100, 2)])
def test_recurrence_ragged(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v, algo=1)
    assert_field_close(got, ref, TOL64)


def test_recurrence_tilted(G):
    got, ref = small_case(G, 300, 33, tilt=True, algo=1)
    assert_field_close(got, ref, TOL64)


def test_recurrence_narrow_beams_fall_back_to_direct(G):
    """Beamlets ~0.45 mm wide on a 128 mm wide detector: the envelope exponent is far below -900 at the
    ends of a thread's run, where the multiplicative recurrence would start from a flushed value."""
    w = gen.workload(1)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    w0 = oracle.waist(1.5, w.pupil_diameter / 21)
    det = dict(n_u=1024, n_v=24, du=0.0125, dv=0.5, origin=[0.3, -0.2, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f / 2)
    got = G.eval_field(b, det, algo=G.ALGO_RECURRENCE).cpu().numpy()
    assert_field_close(got, ref, TOL64)
    det2 = dict(det, du=0.125)                     # 128 mm wide: exponents reach -1e5
    ref2 = oracle.field(oracle.to_detector(rec, det2), det2, w.wavelength)
    got2 = G.eval_field(b, det2, algo=G.ALGO_RECURRENCE).cpu().numpy()
    assert_field_close(got2, ref2, TOL64)


# ----------------------------------------------------------------------------- figure of merit, sweep

def test_psf_metrics_match_oracle(G):
    w = gen.workload(2, 31, 1.25)
    w = gen.Workload(**{**w.__dict__, "det_n": 200, "det_halfwidth_lfn": 15.0})
    r = oracle_run(w)
    det = r["inputs"]["detector"]
    e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
    ref = oracle.psf_metrics(r["field"], det, w.wavelength * w.f_number, e0)
    g = G.run_workload(w, gen.make_inputs)
    e0g = G.eval_field(g["beamlets"], dict(det, n_u=1, n_v=1))
    assert abs(complex(e0g.cpu().numpy()[0, 0]) - e0) < 1e-11 * abs(e0)
    got = G.psf_metrics(g["field"], det, w.wavelength * w.f_number, e0g).cpu().numpy()
    assert np.array_equal(got[4:8], ref[4:8])                      # zone membership: bit exact
    print(f"psf_metrics vs oracle: max |RMS dev| {np.max(np.abs(got[:4] - ref[:4])):.2e}, |max-diff dev| "
          f"{abs(got[8] - ref[8]):.2e} (bounds {ATOL_RMS:.1e} / {ATOL_MAXDIFF:.1e})")
    np.testing.assert_allclose(got[:4], ref[:4], rtol=0, atol=ATOL_RMS)
    np.testing.assert_allclose(got[8], ref[8], rtol=0, atol=ATOL_MAXDIFF)
    # mixed-precision field through the same metric
    gm = G.eval_field(g["beamlets"], det, precision=G.PRECISION_MIXED)
    gotm = G.psf_metrics(gm, det, w.wavelength * w.f_number, e0g).cpu().numpy()
    np.testing.assert_allclose(gotm[:4], ref[:4], rtol=2e-3)


def test_c2_sweep_all_90_runs(G):
    """The whole C2 sweep on the GPU (90 runs, 1.84e10 terms); oracle metrics on a spread of 4 runs;
    the paper's trend: more beamlets -> lower RMS."""
    from paper_2404_12454_b200 import sweep
    ws = gen.sweep_workloads()
    w0 = ws[0]
    det = gen.detector_dict(w0)
    runs = [(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength) for w in ws]
    res = sweep.airy_sweep(runs, gen.ideal_lens_abcd(w0.focal_length).reshape(16), w0.focal_length, det,
                           w0.wavelength * w0.f_number).numpy()
    assert res.shape == (90, 10)
    counts = {11: 97, 21: 349, 31: 749, 41: 1313, 51: 2053, 61: 2933, 71: 3969, 81: 5169, 91: 6509, 101: 8021}
    for i, w in enumerate(ws):
        assert res[i, 9] == counts[w.n_across]
    dev = 0.0
    for i in (0, 17, 44, 89):
        w = ws[i]
        r = oracle_run(w)
        e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
        ref = oracle.psf_metrics(r["field"], det, w.wavelength * w.f_number, e0)
        dev = max(dev, float(np.max(np.abs(res[i, :4] - ref[:4]))))
        np.testing.assert_allclose(res[i, :4], ref[:4], rtol=0, atol=ATOL_RMS)
    print(f"C2 sweep metrics vs oracle (runs 0, 17, 44, 89): max |RMS dev| {dev:.2e} (bound {ATOL_RMS:.1e})")
    rms = res[:, 0].reshape(10, 9)                   # [N index][OF index]
    of15 = 2                                          # OF = 1.5
    assert rms[0, of15] > rms[2, of15] > rms[5, of15] > rms[9, of15]
    # the run-by-run driver (three basic calls + 1x1 on-axis evaluation) agrees with the batched call
    res1 = sweep.airy_sweep_per_run(runs[40:50], gen.ideal_lens_abcd(w0.focal_length).reshape(16),
                                    w0.focal_length, det, w0.wavelength * w0.f_number).numpy()
    print(f"C2 sweep, GPU vs GPU: per-run driver vs batched {np.max(np.abs(res1[:, :4] - res[40:50, :4])):.2e}")
    np.testing.assert_allclose(res1[:, :4], res[40:50, :4], rtol=RTOL_SAME_ALGO, atol=0)
    assert np.array_equal(res1[:, 4:8], res[40:50, 4:8]) and np.array_equal(res1[:, 9], res[40:50, 9])
    # the separable evaluation gives the same figure of merit
    res3 = sweep.airy_sweep(runs, gen.ideal_lens_abcd(w0.focal_length).reshape(16), w0.focal_length, det,
                            w0.wavelength * w0.f_number, algo=G.ALGO_SEPARABLE).numpy()
    print(f"C2 sweep, GPU vs GPU: separable vs direct {np.max(np.abs(res3[:, :4] - res[:, :4])):.2e}")
    np.testing.assert_allclose(res3[:, :4], res[:, :4], rtol=0, atol=ATOL_RMS_ALGOS)
    assert np.array_equal(res3[:, 4:8], res[:, 4:8]) and np.array_equal(res3[:, 9], res[:, 9])
    # the recurrence algorithm gives the same figure of merit
    res2 = sweep.airy_sweep(runs[40:50], gen.ideal_lens_abcd(w0.focal_length).reshape(16), w0.focal_length,
                            det, w0.wavelength * w0.f_number, algo=G.ALGO_RECURRENCE).numpy()
    print(f"C2 sweep, GPU vs GPU: recurrence vs direct {np.max(np.abs(res2[:, :4] - res[40:50, :4])):.2e}")
    np.testing.assert_allclose(res2[:, :4], res[40:50, :4], rtol=0, atol=ATOL_RMS_ALGOS)


@pytest.mark.parametrize("precision,algo,n_px", [(0, 0, 64), (0, 0, 100), (0, 1, 160), (1, 0, 100), (1, 1, 100),
                                                  (0, 2, 100), (0, 2, 200), (1, 2, 200)])
def test_grouped_sweep_fields_match_oracle(G, precision, algo, n_px):
    """gbd_airy_sweep evaluates all runs in ONE grouped stream-K launch: every run's field (ragged
    detector, shares cut across run boundaries) against the oracle, and the figure of merit."""
    import torch
    specs = [(11, 1.0), (3, 2.0), (21, 1.5), (1, 1.0), (31, 2.75), (17, 1.25), (41, 1.5)]
    ws = [gen.Workload(**{**gen.workload(2, n, of).__dict__, "det_n": n_px}) for n, of in specs]
    det = gen.detector_dict(ws[0])
    runs = [(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength) for w in ws]
    dtype = torch.complex128 if precision == 0 else torch.complex64
    fields = torch.zeros((len(ws), n_px, n_px), dtype=dtype, device="cuda:0")
    res = G.airy_sweep(runs, gen.ideal_lens_abcd(ws[0].focal_length).reshape(16), ws[0].focal_length, det,
                       ws[0].wavelength * ws[0].f_number, precision=precision, algo=algo, fields=fields)
    res = res.cpu().numpy()
    fields = fields.cpu().numpy()
    for i, w in enumerate(ws):
        r = oracle_run(w)
        assert res[i, 9] == r["rec"].shape[0]
        assert_field_close(fields[i], r["field"], TOL64 if precision == 0 else TOLMIX)
        e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
        ref = oracle.psf_metrics(r["field"], det, w.wavelength * w.f_number, e0)
        np.testing.assert_allclose(res[i, :4], ref[:4], rtol=0 if precision == 0 else 5e-3, atol=ATOL_METRIC)
        assert np.array_equal(res[i, 4:8], ref[4:8])
    # without a caller buffer the fields live in the workspace: same metrics, bit for bit
    res_b = G.airy_sweep(runs, gen.ideal_lens_abcd(ws[0].focal_length).reshape(16), ws[0].focal_length, det,
                         ws[0].wavelength * ws[0].f_number, precision=precision, algo=algo).cpu().numpy()
    assert np.array_equal(res_b, res)


# ----------------------------------------------------------------------------- a0 differential ray trace

def _trace_both(G, w):
    import torch
    b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength)
    xy = b.positions.cpu().numpy()
    spec = gen.trace_spec(w, xy)
    abcd, base = G.trace_mirrors(b, spec, spec["p_in"], spec["opl0"])
    torch.cuda.synchronize()
    ref_abcd, ref_base = oracle.trace_mirrors(xy, spec, spec["p_in"], spec["opl0"], wavelength=w.wavelength)
    return abcd.cpu().numpy(), base.cpu().numpy(), ref_abcd, ref_base, spec, xy


# Tolerances of a0 ("a0 tolerance").  The kernel traces in double-double arithmetic (~106 bits)
# and rounds every output to double once; the oracle's tracer works in extended precision (64-bit significand) from
# its own formulation and rounds once as well.  So |kernel - oracle| is the ORACLE's rounding: a chain of ~10
# extended-precision operations per mirror on numbers up to L (the longest optical path of the trace = the largest
# number it handles), eps_x = 2^-63, plus one unit in the last place of the output itself (the two final roundings):
#   * ray coordinates on the evaluation plane          -> C_X * eps_x * L + ulp(q)
#   * the path, reduced modulo lambda on both sides (R-24) -> C_X * eps_x * L + ulp(lambda), compared modulo lambda
#   * direction cosines (numbers <= 1)                 -> C_X * eps_x + ulp(p)
#   * ABCD entries, differences of two rays over the step h -> 2 C_X eps_x L / h + ulp (q rows), 2 C_X eps_x / h + ulp (p rows)
C_X = 8.0
EPS_X = 2.0 ** -63


def _trace_scale(xy, spec):
    """L: the longest optical path of the trace, from the oracle's unreduced trace (without the pupil's own opl0)."""
    _, full = oracle.trace_mirrors(xy, spec, spec["p_in"], None)
    return float(np.max(np.abs(full[4])))


@pytest.mark.parametrize("idx", [4, 5])
def test_trace_mirrors_matches_oracle(G, idx):
    """gbd_trace_mirrors (paraboloid with field + Zernike tilts; the paper's two-mirror telescope) against the
    oracle's tracer, which is written independently (direct conic quadratic from the current point, both roots,
    sheet selection by the sign of dF/dz', unnormalised-gradient reflection, long double throughout).  The bound
    is the oracle's extended-precision rounding plus the final rounding to double (constants above)."""
    w = gen.workload(idx)
    abcd, base, ref_abcd, ref_base, spec, xy = _trace_both(G, w)
    L = _trace_scale(xy, spec)
    ulp = lambda a: np.spacing(np.abs(a))
    dpath = np.abs(base[4] - ref_base[4])
    dpath = np.minimum(dpath, np.abs(dpath - w.wavelength))           # representatives may differ by one lambda
    assert np.all(np.abs(base[4]) < w.wavelength)
    eq = np.max((np.abs(base[:2] - ref_base[:2]) - ulp(ref_base[:2])) / (EPS_X * L))
    eo = np.max((dpath - np.spacing(w.wavelength)) / (EPS_X * L))
    ep = np.max((np.abs(base[2:4] - ref_base[2:4]) - ulp(ref_base[2:4])) / EPS_X)
    d = ((np.abs(abcd - ref_abcd) - ulp(ref_abcd))).reshape(-1, 4, 4)
    ea = max(np.max(d[:, :2, :2]) * spec["dq"], np.max(d[:, :2, 2:]) * spec["dp"]) / (EPS_X * L)
    ec = max(np.max(d[:, 2:, :2]) * spec["dq"], np.max(d[:, 2:, 2:]) * spec["dp"]) / EPS_X
    print(f"trace C{idx}: L = {L:.1f} mm; errors beyond one ulp of the output, in units of the bound's scale "
          f"(2^-63 L etc.): q {eq:.2f}, path mod lambda {eo:.2f} (= {2 * math.pi * np.max(dpath) / w.wavelength:.1e} rad), "
          f"p {ep:.2f}, AB rows {ea:.2f}, CD rows {ec:.2f}")
    assert eq <= C_X and eo <= C_X and ep <= C_X
    assert ea <= 2 * C_X and ec <= 2 * C_X


def test_trace_path_is_reduced_before_it_is_rounded(G):
    """R-24 with exactly representable numbers: no mirror, 2^14 of free space along the axis, lambda = 2^-11, a
    pupil path of 2^-45.  The optical path 2^14 + 2^-45 does not fit a double (it would round to 2^14 and the phase
    of 2^-45 -- 2e-10 turns -- would be lost); reduced modulo lambda first, it is 2^-45 exactly.  Same for a
    negative path (fmod keeps the sign).  Both sides must return exactly that."""
    lam, L, tiny = 2.0 ** -11, 2.0 ** 14, 2.0 ** -45
    b = G.beamlets_create(3, 1.0, 1.5, lam)
    xy = b.positions.cpu().numpy()
    spec = dict(mirrors=[], z_pupil=0.0, dir_sign=1.0, origin=[0.0, 0.0, L], e_x=[1.0, 0.0, 0.0],
                e_y=[0.0, 1.0, 0.0], dq=1e-4, dp=1e-6, p_common=[0.0, 0.0], p_in=None, opl0=None)
    for Lz, opl0, want in ((L, tiny, tiny), (2.0 ** 4, -2.0 ** 5 - tiny, -tiny), (L, 3 * lam / 4, 3 * lam / 4),
                           (L, 0.0, 0.0)):
        spec["origin"] = [0.0, 0.0, Lz]
        o = np.full(b.n, opl0)
        _, base = G.trace_mirrors(b, spec, None, o)
        _, ref = oracle.trace_mirrors(xy, spec, None, o, wavelength=lam)
        assert np.array_equal(ref[4], np.full(b.n, want)), (opl0, ref[4])
        assert np.array_equal(base.cpu().numpy()[4], ref[4]), (opl0, base.cpu().numpy()[4])
        assert np.array_equal(base.cpu().numpy()[:4], ref[:4])            # straight rays: q = (x, y), p = 0, exactly


def _gpu_field_from_traced(G, w, abcd, base, **kw):
    b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength)
    G.propagate_q(b, 0, abcd, 0.0, base, None)
    return b, G.eval_field(b, gen.detector_dict(w), **kw).cpu().numpy()


def test_field_c5_hst_like_same_traced_rays(G):
    """NEXT-1 workload C5 (Table 2-3), steps a2-a4 at full size (8,021 beamlets x 512 x 512 px, every
    pixel): the SAME traced rays (the oracle's, handed over as inputs) go through each side's parameters,
    re-expansion and field sum."""
    w = gen.workload(5)
    xy = oracle.lattice(w.n_across, w.pupil_diameter)
    spec = gen.trace_spec(w, xy)
    abcd, base = oracle.trace_mirrors(xy, spec)
    det = gen.detector_dict(w)
    rec = oracle.propagate(xy, oracle.waist(w.overlap_factor, w.pitch), w.wavelength, 0, abcd, 0.0, base, None)
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
    b, got = _gpu_field_from_traced(G, w, abcd, base)
    assert_field_close(got, ref, TOL64)
    for algo in (G.ALGO_RECURRENCE, G.ALGO_SEPARABLE):
        assert_field_close(G.eval_field(b, det, algo=algo).cpu().numpy(), ref, TOL64)
    assert_field_close(G.eval_field(b, det, precision=G.PRECISION_MIXED).cpu().numpy(), ref, TOLMIX)


def _own_trace_tol(w, xy, spec):
    """Each side traces for itself, and both hand on the path already reduced modulo lambda (R-24): the paths then
    differ by the oracle's extended-precision rounding, <= C_X 2^-63 L, and a path error dL is a phase error
    2 pi dL / lambda of that beamlet (16 m at 551 nm: 1.6e-10 rad); the ABCD differences move Q^-1 and the amplitude
    by less."""
    return TOL64 + 2 * math.pi * C_X * EPS_X * _trace_scale(xy, spec) / w.wavelength


def test_field_c5_hst_like_own_trace_each_side(G):
    """C5 end to end, each side deriving the ABCD with its OWN ray tracer; full size, every pixel.  The tolerance
    is the one the a0 bound implies for the field (see _own_trace_tol), 2.6e-10 here; the 1e-10 bar of the
    field sum itself is test_field_c5_hst_like_same_traced_rays."""
    w = gen.workload(5)
    g = G.run_workload(w, gen.make_inputs)
    r = oracle_run(w)
    tol = _own_trace_tol(w, r["inputs"]["xy"], r["inputs"]["trace"])
    err = rel_l2(g["field"].cpu().numpy(), r["field"])
    print(f"C5 own trace each side: rel-L2 {err:.3e} (bound {tol:.3e})")
    assert err < tol and tol < 3e-10


def test_field_c4_own_trace_each_side(G):
    """C4 with the generator's numpy ray trace replaced by each side's own tracer (small version)."""
    w = gen.Workload(**{**gen.workload(4).__dict__, "n_across": 31, "det_n": 96, "trace_on_side": True})
    g = G.run_workload(w, gen.make_inputs)
    r = oracle_run(w)
    tol = _own_trace_tol(w, r["inputs"]["xy"], r["inputs"]["trace"])
    err = rel_l2(g["field"].cpu().numpy(), r["field"])
    print(f"C4 own trace each side: rel-L2 {err:.3e} (bound {tol:.3e})")
    assert err < tol and tol < 1.1e-10


# ----------------------------------------------------------------------------- mixed-precision recurrence

@pytest.mark.parametrize("idx", [0, 1, 4])
def test_mixed_recurrence_configs(G, idx):
    """precision 1 + algo 1: fp64 phase at every restart, fp32 recurrence in between; <= 1e-4 like mixed."""
    w = gen.workload(idx)
    if idx == 4:
        w = gen.Workload(**{**w.__dict__, "n_across": 51, "det_n": 256})
    r = oracle_run(w, rows=(0, w.det_n, 4))
    g = G.run_workload(w, gen.make_inputs, precision=G.PRECISION_MIXED, algo=G.ALGO_RECURRENCE)
    got = g["field"].cpu().numpy()
    assert got.dtype == np.complex64
    assert_field_close(got[0:w.det_n:4], r["field"][0:w.det_n:4], TOLMIX)


def test_mixed_recurrence_c3_against_fp64_direct(G):
    w = gen.workload(3)
    g = G.run_workload(w, gen.make_inputs, precision=G.PRECISION_MIXED, algo=G.ALGO_RECURRENCE)
    gd = G.eval_field(g["beamlets"], g["inputs"]["detector"]).cpu().numpy()     # fp64 direct: parity-tested above
    assert_field_close(g["field"].cpu().numpy(), gd, TOLMIX)


@pytest.mark.parametrize("n_u,n_v", [(16, 5), (33, 7), (129, 2), (300, 11), (1000, 3)])
def test_mixed_recurrence_ragged(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v, precision=1, algo=1)
    assert_field_close(got, ref, TOLMIX)


def test_mixed_recurrence_tilted_and_narrow_beams(G):
    got, ref = small_case(G, 300, 33, tilt=True, precision=1, algo=1)
    assert_field_close(got, ref, TOLMIX)
    # beams far narrower than a thread's run (same set-up as the fp64 narrow-beam test): the start value of
    # most (beamlet, thread) pairs would be flushed in fp32, those pairs take the direct path
    w = gen.workload(1)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    w0 = oracle.waist(1.5, w.pupil_diameter / 21)
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f / 2)
    for du in (0.0125, 0.125):
        det = dict(n_u=1024, n_v=24, du=du, dv=0.5, origin=[0.3, -0.2, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
        ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
        got = G.eval_field(b, det, precision=1, algo=1).cpu().numpy()
        assert_field_close(got, ref, TOLMIX)


# ----------------------------------------------------------------------------- large detector

@pytest.mark.parametrize("precision,algo", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_large_detector_sampled_pixels(G, precision, algo):
    """4096 x 4097 px (16.8 M pixels, 268 MB of complex128; 64-bit pixel indexing, ragged last tile) with a
    handful of beamlets: 4000 random pixels and the four corners against the oracle, one by one."""
    w = gen.workload(0)
    n_u, n_v = 4096, 4097
    xy = oracle.lattice(5, w.pupil_diameter)
    w0 = oracle.waist(1.5, w.pupil_diameter / 5)
    abcd = gen.ideal_lens_abcd(w.focal_length, 0.05).reshape(16)
    det = dict(n_u=n_u, n_v=n_v, du=2.0e-5, dv=2.0e-5, origin=[1e-3, 2e-3, 0.0], e_u=[1.0, 0.0, 0.0],
               e_v=[0.0, 1.0, 0.0])
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, 100.05)
    rd = oracle.to_detector(rec, det)
    rng = np.random.default_rng(11)
    iu = np.concatenate([rng.integers(0, n_u, 4000), [0, n_u - 1, 0, n_u - 1]])
    iv = np.concatenate([rng.integers(0, n_v, 4000), [0, 0, n_v - 1, n_v - 1]])
    ref = oracle.field_pixels(rd, det, w.wavelength, iu, iv)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, 100.05)
    got = G.eval_field(b, det, precision=precision, algo=algo)
    got = got[torch.as_tensor(iv, device=got.device), torch.as_tensor(iu, device=got.device)].cpu().numpy()
    assert_field_close(got, ref, TOL64 if precision == 0 else TOLMIX)


# ----------------------------------------------------------------------------- separable evaluation (algo 2)

@pytest.mark.parametrize("idx", [0, 1, 4, 5])
def test_separable_configs(G, idx):
    """algo 2: C0/C1 have no cross terms (rank-1 kernel runs); C4/C5 have them (the gate routes the call to the
    recurrence kernel, bit for bit the algo-1 result)."""
    w = gen.workload(idx)
    if idx in (4, 5):
        w = gen.Workload(**{**w.__dict__, "n_across": 41, "det_n": 200})
    r = oracle_run(w, rows=(0, w.det_n, 4))
    g = G.run_workload(w, gen.make_inputs, algo=G.ALGO_SEPARABLE)
    got = g["field"].cpu().numpy()
    # C5: each side traces its own rays, so the field bar is the one the a0 bound implies (_own_trace_tol)
    tol = TOL64 if idx != 5 else _own_trace_tol(w, r["inputs"]["xy"], r["inputs"]["trace"])
    assert_field_close(got[0:w.det_n:4], r["field"][0:w.det_n:4], tol)
    rec = G.eval_field(g["beamlets"], g["inputs"]["detector"], algo=G.ALGO_RECURRENCE).cpu().numpy()
    if idx in (4, 5):
        assert np.array_equal(got, rec)
    else:
        assert not np.array_equal(got, rec) and rel_l2(got, rec) < 1e-11


def test_separable_c3_sampled_rows(G):
    w = gen.workload(3)
    g = G.run_workload(w, gen.make_inputs, algo=G.ALGO_SEPARABLE)
    got = g["field"].cpu().numpy()
    rows = [0, 1, 63, 64, 511, 512, 640, 1000, 1023]
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    rd = oracle.to_detector(rec, inp["detector"])
    ref = np.zeros((1024, 1024), dtype=np.complex128)
    for v in rows:
        oracle.field_rows(rd, inp["detector"], w.wavelength, v, v + 1, 1, out=ref)
    assert_field_close(got[rows], ref[rows], TOL64)
    gd = G.eval_field(g["beamlets"], g["inputs"]["detector"]).cpu().numpy()
    assert rel_l2(got, gd) < 1e-11
    again = G.eval_field(g["beamlets"], g["inputs"]["detector"], algo=G.ALGO_SEPARABLE).cpu().numpy()
    assert np.array_equal(got, again)                              # fixed summation order


@pytest.mark.parametrize("n_u,n_v", [(1, 1), (7, 9), (16, 5), (33, 7), (127, 65), (129, 2), (300, 130), (1000, 3), (130, 1000)])
def test_separable_ragged(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v, algo=2)
    assert_field_close(got, ref, TOL64)


def test_separable_tilted_and_narrow_beams(G):
    got, ref = small_case(G, 300, 33, tilt=True, algo=2)           # tilt about y: cross terms -> fallback
    assert_field_close(got, ref, TOL64)
    w = gen.workload(1)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    w0 = oracle.waist(1.5, w.pupil_diameter / 21)
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f / 2)
    for du in (0.0125, 0.125):                                     # beams far narrower than an edge run
        det = dict(n_u=1024, n_v=24, du=du, dv=0.5, origin=[0.3, -0.2, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
        ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
        got = G.eval_field(b, det, algo=2).cpu().numpy()
        assert_field_close(got, ref, TOL64)


@pytest.mark.parametrize("idx", [0, 1, 3, 4])
def test_mixed_separable_configs(G, idx):
    """precision 1 + algo 2: fp32 rank-1 updates, edge values started from the fp64 phase; C4 takes the gated
    mixed-recurrence fallback.  C3 at full size against the fp64 direct field (itself parity-tested)."""
    w = gen.workload(idx)
    if idx == 4:
        w = gen.Workload(**{**w.__dict__, "n_across": 41, "det_n": 200})
    g = G.run_workload(w, gen.make_inputs, precision=G.PRECISION_MIXED, algo=G.ALGO_SEPARABLE)
    got = g["field"].cpu().numpy()
    assert got.dtype == np.complex64
    if idx == 3:
        ref = G.eval_field(g["beamlets"], g["inputs"]["detector"]).cpu().numpy()
        assert_field_close(got, ref, TOLMIX)
    else:
        r = oracle_run(w, rows=(0, w.det_n, 4))
        assert_field_close(got[0:w.det_n:4], r["field"][0:w.det_n:4], TOLMIX)


@pytest.mark.parametrize("n_u,n_v", [(1, 1), (7, 9), (16, 5), (127, 65), (300, 130), (130, 1000)])
def test_mixed_separable_ragged(G, n_u, n_v):
    got, ref = small_case(G, n_u, n_v, precision=1, algo=2)
    assert_field_close(got, ref, TOLMIX)


# ----------------------------------------------------------------------------- streams

def test_side_streams_give_the_same_field(G):
    """The calls enqueue on the caller's stream and never synchronise: two field sums on two side streams
    (own handles, own workspaces) equal the default-stream results bit for bit."""
    w = gen.workload(1)
    ref = G.run_workload(w, gen.make_inputs)
    ref_r = G.eval_field(ref["beamlets"], ref["inputs"]["detector"], algo=G.ALGO_SEPARABLE)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    inp = ref["inputs"]
    outs = []
    for st, algo in ((s1, G.ALGO_DIRECT), (s2, G.ALGO_SEPARABLE)):
        with torch.cuda.stream(st):
            b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, stream=st)
            b.xy[:, : b.n] = torch.as_tensor(inp["xy"], device=b.device)
            G.propagate_q(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"], stream=st)
            outs.append((b, G.eval_field(b, inp["detector"], algo=algo, stream=st)))
    s1.synchronize()
    s2.synchronize()
    assert torch.equal(outs[0][1], ref["field"]) and torch.equal(outs[1][1], ref_r)


# ----------------------------------------------------------------------------- randomised cases

def _random_symplectic_abcd(rng):
    """Product of free spaces, thin lenses and a rotated cylindrical lens: a general astigmatic system
    (P:62-82); every factor is symplectic, so the product is."""
    def space(d):
        m = np.eye(4); m[0, 2] = d; m[1, 3] = d; return m
    def lens(fx, fy):
        m = np.eye(4); m[2, 0] = -1.0 / fx; m[3, 1] = -1.0 / fy; return m
    def rot(t):
        c, s_ = math.cos(t), math.sin(t)
        r = np.array([[c, s_], [-s_, c]]); m = np.zeros((4, 4)); m[:2, :2] = r; m[2:, 2:] = r; return m
    t = rng.uniform(0, math.pi)
    m = space(rng.uniform(5, 40)) @ lens(rng.uniform(60, 200), rng.uniform(60, 200))
    if rng.random() < 0.6:                                       # cross terms
        m = m @ rot(-t) @ lens(rng.uniform(150, 600), 1e12) @ rot(t)
    return space(rng.uniform(20, 120)) @ m


@pytest.mark.parametrize("seed", range(12))
def test_random_systems_all_algorithms(G, seed):
    """Random astigmatic ABCD, beamlet positions / tilts / OPD / complex weights, waist, wavelength, detector size,
    pitch, offset and (every third case) tilt: every algorithm and precision against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(3, 400))
    lam = float(rng.uniform(0.4e-3, 1.6e-3))
    w0 = float(rng.uniform(0.2, 1.5))
    xy = rng.uniform(-8, 8, (2, n))
    base = np.stack([rng.uniform(-2e-4, 2e-4, n), rng.uniform(-2e-4, 2e-4, n), rng.uniform(-2e-3, 2e-3, n)])
    wt = rng.standard_normal((2, n))
    abcd = _random_symplectic_abcd(rng)
    l0 = float(rng.uniform(50, 400))
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), l0, base, wt)
    c = rec[:, :2].mean(axis=0)
    spread = float(np.abs(rec[:, :2] - c).max()) + 5 * lam * 100 / w0
    n_u, n_v = int(rng.integers(16, 300)), int(rng.integers(1, 90))
    det = dict(n_u=n_u, n_v=n_v, du=2 * spread / n_u * rng.uniform(0.3, 1.0), dv=2 * spread / max(n_v, 8) * rng.uniform(0.3, 1.0),
               origin=[float(c[0]), float(c[1]), 0.0], e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    if seed % 3 == 2:
        t = float(rng.uniform(-0.3, 0.3))
        det.update(e_u=[math.cos(t), 0.0, -math.sin(t)], origin=[float(c[0]), float(c[1]), float(rng.uniform(-0.5, 0.5))])
    ref = oracle.field(oracle.to_detector(rec, det), det, lam)
    assert np.linalg.norm(ref) > 0
    b = G.beamlets_custom(xy, w0, lam)
    G.propagate_q(b, 1, abcd.reshape(16), l0, base, wt)
    for precision in (0, 1):
        for algo in (0, 1, 2):
            got = G.eval_field(b, det, precision=precision, algo=algo).cpu().numpy()
            assert_field_close(got, ref, TOL64 if precision == 0 else TOLMIX, (seed, precision, algo))


@pytest.mark.parametrize("seed", range(8))
def test_random_systems_at_table_kernel_size(G, seed):
    """The same randomised astigmatic systems, sized so that the direct launches take the table kernels (1.6e7 - 5e7
    terms: field_fold_kernel / field_mixed_tab_kernel or, when the pre-pass does not clear the launch, their twins):
    cross terms, decentred and tilted beamlets, complex weights, detector offsets and (every other case) a tilted
    detector; fp64 and mixed, direct algorithm, plus the mode-factor kernel on the untilted cases."""
    rng = np.random.default_rng(5000 + seed)
    n = int(rng.integers(500, 1500))
    lam = float(rng.uniform(0.4e-3, 1.6e-3))
    w0 = float(rng.uniform(0.2, 1.5))
    xy = rng.uniform(-8, 8, (2, n))
    base = np.stack([rng.uniform(-2e-4, 2e-4, n), rng.uniform(-2e-4, 2e-4, n), rng.uniform(-2e-3, 2e-3, n)])
    wt = rng.standard_normal((2, n))
    abcd = _random_symplectic_abcd(rng)
    l0 = float(rng.uniform(50, 400))
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), l0, base, wt)
    c = rec[:, :2].mean(axis=0)
    spread = float(np.abs(rec[:, :2] - c).max()) + 5 * lam * 100 / w0
    n_u, n_v = 256, 128
    det = dict(n_u=n_u, n_v=n_v, du=2 * spread / n_u * rng.uniform(0.3, 1.0), dv=2 * spread / n_v * rng.uniform(0.3, 1.0),
               origin=[float(c[0]), float(c[1]), 0.0], e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    tilted = seed % 2 == 1
    if tilted:
        t = float(rng.uniform(-0.3, 0.3))
        det.update(e_u=[math.cos(t), 0.0, -math.sin(t)], origin=[float(c[0]), float(c[1]), float(rng.uniform(-0.5, 0.5))])
    rd = oracle.to_detector(rec, det)
    ref = oracle.field(rd, det, lam)
    assert np.linalg.norm(ref) > 0 and n * n_u * n_v >= 1.0e7
    b = G.beamlets_custom(xy, w0, lam)
    G.propagate_q(b, 1, abcd.reshape(16), l0, base, wt)
    assert_field_close(G.eval_field(b, det).cpu().numpy(), ref, TOL64, (seed, "fp64"))
    assert_field_close(G.eval_field(b, det, precision=G.PRECISION_MIXED).cpu().numpy(), ref, TOLMIX, (seed, "mixed"))
    if not tilted:
        mw = rng.standard_normal((12, n))
        ref_m = oracle.field_modes(rd, oracle.hg_modes(n, w0, lam, 1, abcd.reshape(16), mw), det, lam)
        got_m = G.eval_field_modes(b, G.hg_modes(b, 1, abcd.reshape(16), mw), det).cpu().numpy()
        assert_field_close(got_m, ref_m, TOL64, (seed, "modes"))


# ----------------------------------------------------------------------------- row sharding (multi-GPU layout)

@pytest.mark.parametrize("world,algo", [(2, 0), (3, 1), (8, 2)])
def test_row_bands_reassemble_the_field(G, world, algo):
    """rank r evaluates its band of detector rows from the same records, no collective.
    Here the `world` bands are evaluated one after the other on this GPU and stitched: they reproduce the
    oracle field of the full detector (tilted C4 detector, uneven split)."""
    from paper_2404_12454_b200 import sharding
    w = gen.Workload(**{**gen.workload(4).__dict__, "n_across": 31, "det_n": 101})
    r = oracle_run(w)
    g = G.run_workload(w, gen.make_inputs)
    det = g["inputs"]["detector"]
    got = np.zeros((w.det_n, w.det_n), dtype=np.complex128)
    rows = 0
    for rank in range(world):
        band = sharding.row_band(det, rank, world)
        f = G.eval_field(g["beamlets"], {k: band[k] for k in ("n_u", "n_v", "du", "dv", "origin", "e_u", "e_v")},
                         algo=algo).cpu().numpy()
        got[band["row_offset"]:band["row_offset"] + band["n_v"]] = f
        rows += band["n_v"]
    assert rows == w.det_n
    assert_field_close(got, r["field"], TOL64)


# ----------------------------------------------------------------------------- CUDA graph capture

@pytest.mark.parametrize("algo,idx", [(0, 0), (1, 0), (2, 0), (0, 2)])
def test_whole_path_captures_into_a_cuda_graph(G, algo, idx):
    """No call of the path synchronises or allocates, so a1 + a2 + a3 + a4 can be captured once and replayed
    (launch-bound small configs: C0 is 5-7 kernels of a few microseconds each).  The replayed field equals the
    eagerly computed one bit for bit; after the inputs changed in place (new weights) it follows them.
    (0, 2): a C2 member with 1.3e8 terms, i.e. the table kernel with its memset node and device-side loop choice."""
    w = gen.workload(idx)
    inp = gen.make_inputs(w, oracle.lattice(w.n_across, w.pupil_diameter))
    det = inp["detector"]
    dev = torch.device("cuda:0")
    abcd = torch.as_tensor(inp["abcd"], device=dev)
    n = G.lattice_count(w.n_across, w.pupil_diameter)
    weight = torch.ones((2, n), dtype=torch.float64, device=dev)
    weight[1] = 0.0
    params = torch.empty((n, 13), dtype=torch.float64, device=dev)
    field = torch.zeros((det["n_v"], det["n_u"]), dtype=torch.complex128, device=dev)
    keep = {}

    def step():
        b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, device=dev)
        keep["b"] = b
        if "ws" not in keep:
            keep["ws"] = torch.empty(G.eval_workspace_bytes(b, det), dtype=torch.uint8, device=dev)
        G.propagate_q(b, 1, abcd, inp["l0"], None, weight, out=params)
        G.eval_field(b, det, out=field, workspace=keep["ws"], algo=algo)

    step()                                           # eager reference (also allocates the workspace)
    torch.cuda.synchronize()
    eager = field.clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        step()                                       # warm-up on the capture stream
        side.synchronize()
        with torch.cuda.graph(graph, stream=side):
            step()
    field.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(field, eager)
    assert_field_close(field.cpu().numpy(), oracle_run(w)["field"], TOL64)
    weight[0] *= 2.0                                 # same graph, new inputs
    graph.replay()
    torch.cuda.synchronize()
    assert rel_l2(field.cpu().numpy(), 2.0 * eager.cpu().numpy()) < 1e-13   # |A| enters through log2: not bitwise


# ----------------------------------------------------------------------------- C3, every pixel

def test_field_c3_full_grid_all_variants(G):
    """BASELINE.json configs[3] at full size (31,757 beamlets x 1024 x 1024 px = 3.33e10 terms), EVERY pixel
    against the oracle (about a minute of oracle time on the GPU box's host cores), for all six variants of
    gbd_eval_field in the launch configuration bench.py times."""
    w = gen.workload(3)
    step = 1 if oracle.num_threads() >= FULL_GRID_CORES else 4   # few host cores: every 4th row (8.3e9 terms)
    r = oracle_run(w, rows=(0, w.det_n, step))
    ref = r["field"][::step]
    g = G.run_workload(w, gen.make_inputs)
    det = g["inputs"]["detector"]
    errs = {}
    for precision in (0, 1):
        for algo in (0, 1, 2):
            got = G.eval_field(g["beamlets"], det, precision=precision, algo=algo).cpu().numpy()
            errs[(precision, algo)] = (rel_l2(got[::step], ref), max_pixel_err(got[::step], ref))
    print("C3 full-grid (rel-L2, worst pixel / peak):", {k: f"{v[0]:.2e}, {v[1]:.2e}" for k, v in errs.items()})
    for (precision, algo), e in errs.items():
        assert max(e) < (TOL64 if precision == 0 else TOLMIX), (precision, algo, e)
    _report_thinning(step, "rows of C3")


def test_c2_all_90_runs_fields_and_metrics_against_oracle(G):
    """BASELINE.json configs[2] in full: every pixel of every one of the 90 runs (1.84e10 terms, about half a
    minute of oracle time) and the per-run figure of merit, from ONE gbd_airy_sweep call (separable evaluation;
    the direct and recurrence sweeps are compared with it in test_c2_sweep_all_90_runs)."""
    ws = gen.sweep_workloads()
    w0 = ws[0]
    det = gen.detector_dict(w0)
    runs = [(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength) for w in ws]
    fields = torch.zeros((len(ws), det["n_v"], det["n_u"]), dtype=torch.complex128, device="cuda:0")
    res = G.airy_sweep(runs, gen.ideal_lens_abcd(w0.focal_length).reshape(16), w0.focal_length, det,
                       w0.wavelength * w0.f_number, algo=G.ALGO_SEPARABLE, fields=fields).cpu().numpy()
    fields = fields.cpu().numpy()
    worst = 0.0
    stride = 1 if oracle.num_threads() >= FULL_GRID_CORES else 3   # few host cores: every 3rd run
    for i, w in list(enumerate(ws))[::stride]:
        r = oracle_run(w)
        worst = max(worst, rel_l2(fields[i], r["field"]), max_pixel_err(fields[i], r["field"]))
        e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
        ref = oracle.psf_metrics(r["field"], det, w.wavelength * w.f_number, e0)
        np.testing.assert_allclose(res[i, :4], ref[:4], rtol=0, atol=ATOL_METRIC)
        assert np.array_equal(res[i, 4:8], ref[4:8]) and res[i, 9] == r["rec"].shape[0]
    assert worst < TOL64
    _report_thinning(stride, "runs of C2")


# ----------------------------------------------------------------------------- plane away from focus

def test_defocused_plane_all_variants(G):
    """Half-way to focus every beamlet covers a small part of the detector: the recurrence kernel skips the runs
    a beamlet does not reach and walks runs that cross the edge of a footprint backwards, the separable kernel
    fills dead edge runs with zeros and skips beamlets that do not reach a tile, the direct kernel culls.  8,021
    beamlets x 640 x 512 px, 6000 random pixels + corners against the oracle, pixel by pixel."""
    w = gen.workload(1)
    f = w.focal_length
    xy = oracle.lattice(101, w.pupil_diameter)
    w0 = oracle.waist(1.6, w.pupil_diameter / 101)
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    n_u, n_v = 640, 512
    L = 0.55 * w.pupil_diameter / 2
    det = dict(n_u=n_u, n_v=n_v, du=2 * L / n_u, dv=2 * L / n_v, origin=[0.05, -0.02, 0.0], e_u=[1.0, 0.0, 0.0],
               e_v=[0.0, 1.0, 0.0])
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    rd = oracle.to_detector(rec, det)
    rng = np.random.default_rng(5)
    iu = np.concatenate([rng.integers(0, n_u, 6000), [0, n_u - 1, 0, n_u - 1]])
    iv = np.concatenate([rng.integers(0, n_v, 6000), [0, 0, n_v - 1, n_v - 1]])
    ref = oracle.field_pixels(rd, det, w.wavelength, iu, iv)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f / 2)
    tiu, tiv = torch.as_tensor(iu, device="cuda:0"), torch.as_tensor(iv, device="cuda:0")
    for precision in (0, 1):
        for algo, tau in ((0, 0.0), (0, 1e-18), (1, 0.0), (2, 0.0)):
            got = G.eval_field(b, det, precision=precision, algo=algo, cull_tau=tau)[tiv, tiu].cpu().numpy()
            assert np.all(np.isfinite(got))
            assert_field_close(got, ref, TOL64 if precision == 0 else TOLMIX)


# ----------------------------------------------------------------------------- point-evaluation baseline

def _pointwise_both(G, w, rows=None, det=None, n_across=None):
    """gbd_eval_field_pointwise and the oracle's gbdo_field_pointeval on the same generator inputs."""
    if n_across is not None:
        w = gen.Workload(**{**w.__dict__, "n_across": n_across})
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    det = inp["detector"] if det is None else det
    w0 = oracle.waist(w.overlap_factor, w.pitch)
    ref = oracle.field_pointeval(inp["xy"], w0, w.wavelength, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"],
                                 inp["weight"], det, rows=rows)
    b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength)
    b.xy[:, : b.n] = torch.as_tensor(inp["xy"], device=b.device)
    got = G.eval_field_pointwise(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"], det)
    return got.cpu().numpy(), ref, b, inp


@pytest.mark.parametrize("idx", [0, 1, 4])
def test_pointwise_baseline_matches_oracle(G, idx):
    """The point-evaluation kernel against the oracle's step-by-step version: C0 in full, C1 (jittered
    positions, 1.3e8 pairs) on every 4th row, C4 (per-beamlet ray-traced ABCD, Zernike tilts, 5-degree tilted detector,
    41 beamlets across x 128^2 px) in full."""
    w = gen.workload(idx)
    rows = None
    if idx == 1:
        rows = (0, w.det_n, 4)
    if idx == 4:
        w = gen.Workload(**{**w.__dict__, "n_across": 41, "det_n": 128})
    got, ref, _, _ = _pointwise_both(G, w, rows=rows)
    sel = slice(None) if rows is None else slice(rows[0], rows[1], rows[2])
    assert_field_close(got[sel], ref[sel], TOL64)


@pytest.mark.parametrize("n_u,n_v,n_across", [(1, 1, 11), (37, 3, 5), (130, 129, 3), (5, 700, 21), (64, 64, 1)])
def test_pointwise_baseline_ragged(G, n_u, n_v, n_across):
    """Ragged detectors and beamlet counts around the shared-memory stage (32) and split sizes."""
    w = gen.workload(0)
    det = dict(gen.detector_dict(w), n_u=n_u, n_v=n_v, origin=[1e-3, -2e-3, 0.0])
    got, ref, _, _ = _pointwise_both(G, w, det=det, n_across=n_across)
    assert_field_close(got, ref, TOL64)


def test_pointwise_baseline_zero_beamlets_and_reproducible(G):
    w = gen.workload(0)
    det = gen.detector_dict(w)
    b = G.beamlets_custom(np.zeros((2, 0)), 1.0, w.wavelength)
    z = G.eval_field_pointwise(b, 1, gen.ideal_lens_abcd(100.0).reshape(16), 100.0, None, None, det).cpu().numpy()
    assert z.shape == (64, 64) and not np.any(z)
    got, _, b, inp = _pointwise_both(G, w)
    again = G.eval_field_pointwise(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"],
                                   inp["detector"]).cpu().numpy()
    assert np.array_equal(got, again)


def test_pointwise_and_plane_evaluation_agree_to_the_obliquity(G):
    """Both algorithms on the GPU, C2 member N = 51 (256^2 px): the fields differ by the normalisation per unit
    area normal to each ray vs per unit area of the plane (<= |p|^2/4 per beamlet) and the parabasal residual --
    the paper's Fig. 5 comparison on synthetic optics."""
    w = gen.workload(2, 51, 1.5)
    g = G.run_workload(w, gen.make_inputs)
    inp = g["inputs"]
    pw = G.eval_field_pointwise(g["beamlets"], inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"],
                                inp["detector"]).cpu().numpy()
    pl = g["field"].cpu().numpy()
    d = np.max(np.abs(pw - pl)) / np.max(np.abs(pl))
    assert 1e-5 < d < 0.5 * (0.5 / w.f_number) ** 2


# ----------------------------------------------------------------------------- Hermite-Gaussian beamlets

def _hg_case(G, w, n_across, det, seed, mode_weight="random"):
    """gbd_hg_modes + gbd_eval_field_modes against gbdo_hg_modes + gbdo_field_rows_modes on the same inputs."""
    w = gen.Workload(**{**w.__dict__, "n_across": n_across})
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    n = xy0.shape[1]
    rng = np.random.default_rng(seed)
    mw = None
    if mode_weight == "random":
        mw = rng.standard_normal((12, n))
    elif mode_weight == "hg10":
        mw = np.zeros((12, n))
        mw[2] = 1.0
    w0 = oracle.waist(w.overlap_factor, w.pitch)
    rec = oracle.propagate(inp["xy"], w0, w.wavelength, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"],
                           inp["weight"])
    modes_ref = oracle.hg_modes(n, w0, w.wavelength, inp["abcd_mode"], inp["abcd"], mw)
    ref = oracle.field_modes(oracle.to_detector(rec, det), modes_ref, det, w.wavelength)
    b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength)
    b.xy[:, : b.n] = torch.as_tensor(inp["xy"], device=b.device)
    G.propagate_q(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    modes = G.hg_modes(b, inp["abcd_mode"], inp["abcd"], mw)
    got = G.eval_field_modes(b, modes, det).cpu().numpy()
    return got, ref, modes.cpu().numpy(), modes_ref, b, modes


@pytest.mark.parametrize("idx,n_across,n_px", [(0, 11, 64), (1, 51, 256), (3, 201, 512), (4, 41, 96)])
def test_hg_beamlets_match_oracle(G, idx, n_across, n_px):
    """Hermite-Gaussian beamlets of orders m+n <= 2 with six random complex weights per beamlet: mode factors and field,
    every pixel.  C0 (polynomial kernel: small launch), C1 and C3 optics with 201 across x 512^2 px (table kernel,
    8.3e9 terms), C4 optics (per-beamlet ray-traced ABCD: a different M1^-1 for every beamlet) on an untilted plane."""
    w = gen.workload(idx)
    det = dict(gen.detector_dict(gen.Workload(**{**w.__dict__, "tilt_deg": 0.0})), n_u=n_px, n_v=n_px)
    if idx == 4:
        c = gen.workloads.c4_chief_intercept(w)
        det["origin"] = [float(c[0]), float(c[1]), 0.0]
    if idx == 3:
        det["du"] *= 2
        det["dv"] *= 2
    got, ref, modes, modes_ref, _, _ = _hg_case(G, w, n_across, det, seed=idx)
    assert np.max(np.abs(modes - modes_ref)) <= 1e-12 * np.max(np.abs(modes_ref))
    assert_field_close(got, ref, TOL64)


def test_hg_beamlets_off_the_fast_path(G):
    """A table-size mode launch the pre-pass does NOT clear for the detector-coordinate kernel: a quarter of the way
    out of focus the beamlet centres spread over millimetres, so the monomials of the expansion about the detector centre
    exceed the gate (and the envelope exponents leave the unclamped range): the beamlet-centred twin must run and match
    the oracle (2,053 beamlets x 512 x 64 px = 6.7e7 terms)."""
    w = gen.workload(1)
    f = w.focal_length
    xy0 = oracle.lattice(51, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    n = xy0.shape[1]
    abcd = gen.ideal_lens_abcd(f, -f / 4).reshape(16)
    mw = np.random.default_rng(3).standard_normal((12, n))
    w0 = oracle.waist(w.overlap_factor, w.pitch)
    det = dict(n_u=512, n_v=64, du=0.02, dv=0.02, origin=[0.3, -0.2, 0.0], e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    rec = oracle.propagate(inp["xy"], w0, w.wavelength, 1, abcd, f - f / 4, None, None)
    rd = oracle.to_detector(rec, det)
    assert np.abs(4 * rd[:, 2] / w.wavelength * rd[:, 0]).max() > 2040.0          # |tu cu| beyond the gate
    ref = oracle.field_modes(rd, oracle.hg_modes(n, w0, w.wavelength, 1, abcd, mw), det, w.wavelength)
    b = G.beamlets_custom(inp["xy"], w0, w.wavelength)
    G.propagate_q(b, 1, abcd, f - f / 4)
    got = G.eval_field_modes(b, G.hg_modes(b, 1, abcd, mw), det).cpu().numpy()
    assert_field_close(got, ref, TOL64)


@pytest.mark.parametrize("n_u,n_v", [(1, 1), (33, 7), (300, 11), (129, 130)])
def test_hg_beamlets_ragged(G, n_u, n_v):
    w = gen.workload(0)
    det = dict(gen.detector_dict(w), n_u=n_u, n_v=n_v, origin=[2e-3, -1e-3, 0.0])
    got, ref, _, _, _, _ = _hg_case(G, w, 9, det, seed=n_u)
    assert_field_close(got, ref, TOL64)


def test_hg_fundamental_weights_reproduce_eval_field_and_tilt_is_refused(G):
    """mode_weight = NULL (w00 = 1) must give the fundamental field of gbd_eval_field; a tilted detector is refused
    loudly (the mode law is stated for planes orthogonal to the axis)."""
    w = gen.workload(1)
    det = gen.detector_dict(w)
    got, ref, _, _, b, modes = _hg_case(G, w, 31, det, seed=0, mode_weight=None)
    base = G.eval_field(b, det).cpu().numpy()
    # two table evaluations with different remainder intervals (nearest / floor index of the exponent table), each
    # within the 1.3e-11 of its 2-term polynomial: they agree to twice that, not to rounding
    assert_field_close(got, base, 3e-11)
    assert_field_close(got, ref, TOL64)
    t = math.radians(5.0)
    tilted = dict(det, e_v=[0.0, math.cos(t), math.sin(t)])
    with pytest.raises(G.GbdError, match="untilted"):
        G.eval_field_modes(b, modes, tilted)


def test_table_kernel_extreme_exponents_take_the_clamped_path(G):
    """The table kernel's unclamped loop needs every envelope exponent inside [-1000, 1000]; the pre-pass decides on
    the device.  Half-way to focus with a 410 mm wide detector the exponents reach -5e6 (beyond the +-2^22 range of
    the exponent word): the launch (8,021 beamlets x 1024 x 8 px = 6.6e7 terms, table kernel) must take the clamped
    loop and still match the oracle; and a focal-plane launch of the same size must match too (unclamped loop)."""
    w = gen.workload(1)
    f = w.focal_length
    xy = oracle.lattice(101, w.pupil_diameter)
    w0 = oracle.waist(1.5, w.pupil_diameter / 101)
    b = G.beamlets_custom(xy, w0, w.wavelength)
    for delta, du in ((-f / 2, 0.4), (0.0, gen.detector_dict(w)["du"])):
        abcd = gen.ideal_lens_abcd(f, delta).reshape(16)
        det = dict(n_u=1024, n_v=8, du=du, dv=du, origin=[0.01, -0.02, 0.0], e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
        rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f + delta)
        rd = oracle.to_detector(rec, det)
        if delta != 0.0:
            k = 2 * math.pi / w.wavelength
            gmin = 0.5 * k * rd[0, 6] * (204.0 + abs(rd[:, 0]).max()) ** 2 * math.log2(math.e)
            assert gmin < -4.3e6                       # the case does leave the exponent word's range
        ref = oracle.field(rd, det, w.wavelength)
        G.propagate_q(b, 1, abcd, f + delta)
        got = G.eval_field(b, det).cpu().numpy()
        assert deep_word(b) == (1 if delta != 0.0 else 0)
        assert_field_close(got, ref, TOL64, delta)


@pytest.mark.parametrize("tilt,expect_fast", [(1e-3, True), (1e-2, True), (2e-2, True), (3e-2, False), (0.1, False)])
def test_table_kernel_detector_coordinate_records_and_their_gate(G, tilt, expect_fast):
    """The fast table kernel evaluates the two quadratics expanded about the detector centre (no Du = u - cu per term);
    the pre-pass allows that only while the monomials of the expansion stay below 2040 quarter turns (4096 log2 units
    for the envelope) on the detector, else the beamlet-centred twin runs.  Wide collimated beamlets (w0 = 6 mm, so that
    the envelope exponents stay far inside the unclamped range and only this gate decides) after 200 mm of free space
    with base-ray tilts up to `tilt`: the linear phase across the detector grows with the tilt and crosses that limit;
    the field must match the oracle on both sides of the gate (600 beamlets x 512 x 128 px = 3.9e7 terms: table
    kernels).  The bound is recomputed here from the oracle's records to make sure both sides are exercised."""
    rng = np.random.default_rng(77)
    n, lam, w0, d = 600, 1.0e-3, 6.0, 200.0
    xy = rng.uniform(-4, 4, (2, n))
    base = np.stack([rng.uniform(-tilt, tilt, n), rng.uniform(-tilt, tilt, n), rng.uniform(-2e-3, 2e-3, n)])
    wt = rng.standard_normal((2, n))
    abcd = np.eye(4); abcd[0, 2] = d; abcd[1, 3] = d
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), d, base, wt)
    c = rec[:, :2].mean(axis=0)
    half = float(np.abs(rec[:, :2] - c).max()) + 3.0
    det = dict(n_u=512, n_v=128, du=2 * half / 512, dv=2 * half / 128, origin=[float(c[0]), float(c[1]), 0.0],
               e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    rd = oracle.to_detector(rec, det)
    # the gate's bound (phase part; the envelope part is far smaller here): monomials of the expansion about the
    # detector centre, at the beamlet centre and at the detector corner
    cu, cv, pu, pv = rd[:, 0], rd[:, 1], rd[:, 2], rd[:, 3]
    tu, tv = -4 * pu / lam, -4 * pv / lam
    tuu, tuv, tvv = -2 * rd[:, 5] / lam, -2 * rd[:, 7] / lam, -2 * rd[:, 9] / lam
    U, V = 0.5 * 511 * det["du"], 0.5 * 127 * det["dv"]
    Tu, Tv = tu - 2 * tuu * cu - tuv * cv, tv - 2 * tvv * cv - tuv * cu
    big = np.maximum(abs(tu * cu) + abs(tv * cv) + abs(tuu) * cu**2 + abs(tuv * cu * cv) + abs(tvv) * cv**2,
                     abs(Tu) * U + abs(Tv) * V + abs(tuu) * U**2 + abs(tuv) * U * V + abs(tvv) * V**2).max()
    assert (big + 4.0 < 2040.0) if expect_fast else (big > 2040.0), big      # GBD_FOLD_T_LIMIT
    ref = oracle.field(rd, det, lam)
    b = G.beamlets_custom(xy, w0, lam)
    G.propagate_q(b, 1, abcd.reshape(16), d, base, wt)
    got = G.eval_field(b, det).cpu().numpy()
    assert deep_word(b) == (0 if expect_fast else 1)          # the path the device actually took
    assert_field_close(got, ref, TOL64, (tilt, big))


@pytest.mark.parametrize("tilt,lam,expect_fast", [(2e-2, 1.0e-3, True), (0.3, 1.0e-3, True), (0.3, 1.0e-4, False)])
def test_mixed_table_kernel_and_its_gate(G, tilt, lam, expect_fast):
    """Mixed precision, table-kernel size (600 beamlets x 512 x 128 px): cis from the fp32 shared-memory table and the
    phase quadratic in detector coordinates (field_mixed_tab_kernel), allowed by the pre-pass while no monomial of the
    expansion exceeds 2^20 quarter turns; beyond that the MUFU twin runs.  Both must meet the mixed bar against the
    oracle; the bound is recomputed here so that both sides of the gate are exercised."""
    rng = np.random.default_rng(78)
    n, w0, d = 600, 6.0, 200.0
    xy = rng.uniform(-4, 4, (2, n))
    base = np.stack([rng.uniform(-tilt, tilt, n), rng.uniform(-tilt, tilt, n), rng.uniform(-2e-3, 2e-3, n)])
    wt = rng.standard_normal((2, n))
    abcd = np.eye(4); abcd[0, 2] = d; abcd[1, 3] = d
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), d, base, wt)
    c = rec[:, :2].mean(axis=0)
    half = float(np.abs(rec[:, :2] - c).max()) + 3.0
    det = dict(n_u=512, n_v=128, du=2 * half / 512, dv=2 * half / 128, origin=[float(c[0]), float(c[1]), 0.0],
               e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    rd = oracle.to_detector(rec, det)
    cu, cv, pu, pv = rd[:, 0], rd[:, 1], rd[:, 2], rd[:, 3]
    tu, tv = -4 * pu / lam, -4 * pv / lam
    tuu, tuv, tvv = -2 * rd[:, 5] / lam, -2 * rd[:, 7] / lam, -2 * rd[:, 9] / lam
    U, V = 0.5 * 511 * det["du"], 0.5 * 127 * det["dv"]
    Tu, Tv = tu - 2 * tuu * cu - tuv * cv, tv - 2 * tvv * cv - tuv * cu
    big = np.maximum(abs(tu * cu) + abs(tv * cv) + abs(tuu) * cu**2 + abs(tuv * cu * cv) + abs(tvv) * cv**2,
                     abs(Tu) * U + abs(Tv) * V + abs(tuu) * U**2 + abs(tuv) * U * V + abs(tvv) * V**2).max()
    assert (big + 4.0 < 2.0**20) if expect_fast else (big > 2.0**20), big
    ref = oracle.field(rd, det, lam)
    b = G.beamlets_custom(xy, w0, lam)
    G.propagate_q(b, 1, abcd.reshape(16), d, base, wt)
    got = G.eval_field(b, det, precision=G.PRECISION_MIXED).cpu().numpy()
    assert got.dtype == np.complex64
    assert deep_word(b) == (0 if expect_fast else 1)          # the path the device actually took
    assert_field_close(got, ref, TOLMIX, (tilt, lam, big))


# ----------------------------------------------------------------------------- boundary behaviour (round 2)

def test_nonfinite_weight_poisons_the_field_instead_of_vanishing(G):
    """A beamlet with a NaN or Inf weight must not silently disappear: every pixel becomes non-finite on
    both sides; a weight of exactly zero still contributes nothing.  Both the polynomial and the table kernel."""
    w = gen.workload(1)
    for n_across, n_px in ((9, 64), (101, 128)):              # 3e5 terms (polynomial), 1.3e8 terms (table kernel)
        xy = oracle.lattice(n_across, w.pupil_diameter)
        n = xy.shape[1]
        w0 = oracle.waist(1.5, w.pupil_diameter / n_across)
        abcd = gen.ideal_lens_abcd(w.focal_length).reshape(16)
        det = dict(gen.detector_dict(w), n_u=n_px, n_v=n_px)
        for bad in (float("nan"), float("inf")):
            wt = np.ones((2, n))
            wt[1] = 0.0
            wt[0, n // 2] = bad
            rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, w.focal_length, None, wt)
            ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
            b = G.beamlets_custom(xy, w0, w.wavelength)
            G.propagate_q(b, 1, abcd, w.focal_length, None, wt)
            for algo in (0, 1, 2):
                got = G.eval_field(b, det, algo=algo).cpu().numpy()
                assert not np.all(np.isfinite(got.view(np.float64))), (n_across, bad, algo)
            got = G.eval_field(b, det).cpu().numpy()
            bad_px = ~np.isfinite(got.view(np.float64)).reshape(n_px, n_px, 2).all(axis=2)
            ref_bad = ~np.isfinite(ref.view(np.float64)).reshape(n_px, n_px, 2).all(axis=2)
            assert bad_px.all() and ref_bad.all(), (n_across, bad)


def test_lattice_many_ctas_bit_exact_and_count(G):
    """The multi-CTA lattice kernel: positions bit-identical to the oracle's for sizes around its row blocking
    (8 rows per CTA, at most 296 CTAs -> several row blocks per CTA from N = 2369), odd and even N."""
    for n in (7, 8, 9, 16, 17, 127, 200, 301, 2400):
        ref = oracle.lattice(n, 31.7)
        b = G.beamlets_create(n, 31.7, 1.5, 1e-3)
        assert b.n == ref.shape[1] == G.lattice_count(n, 31.7)
        assert np.array_equal(b.positions.cpu().numpy(), ref), n


def test_sweep_refuses_graph_capture_and_debug_sync_mode(G):
    """gbd_airy_sweep uploads host tables through a process-wide staging buffer and says so: on a capturing stream
    it returns GBD_ESTATE instead of recording a copy that would replay stale tables.  GBD_DEBUG_SYNC=1
    in a fresh process: the calls synchronise, the device lattice count is compared with the host's, results agree."""
    import os
    import subprocess
    import sys
    ws = gen.sweep_workloads()[:3]
    det = gen.detector_dict(ws[0])
    runs = [(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength) for w in ws]
    abcd = torch.as_tensor(gen.ideal_lens_abcd(ws[0].focal_length).reshape(16), device="cuda:0")
    res = G.airy_sweep(runs, abcd, ws[0].focal_length, det, ws[0].wavelength * ws[0].f_number)
    torch.cuda.synchronize()
    out2 = torch.empty_like(res)
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    err = None
    with torch.cuda.stream(side):
        side.synchronize()
        try:
            with torch.cuda.graph(graph, stream=side):
                try:
                    G.airy_sweep(runs, abcd, ws[0].focal_length, det, ws[0].wavelength * ws[0].f_number,
                                 out=out2, workspace=res._keep[1], stream=side)
                except G.GbdError as e:
                    err = str(e)
        except Exception:
            pass
    assert err is not None and "captur" in err
    code = ("import numpy as np, gen, oracle, paper_2404_12454_b200 as G\n"
            "w = gen.workload(0)\n"
            "g = G.run_workload(w, gen.make_inputs)\n"
            "ref = oracle.run_workload(w, gen.make_inputs)['field']\n"
            "got = g['field'].cpu().numpy()\n"
            "assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 1e-10\n"
            "print('debug-sync ok', g['beamlets'].n)\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, GBD_DEBUG_SYNC="1"),
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and "debug-sync ok 97" in out.stdout, out.stderr[-2000:]


def test_psf_metrics_accepts_a_complex64_on_axis_value(G):
    """A 1x1 mixed-precision field (complex64) as e0: the binding must not drop its imaginary part."""
    w = gen.workload(2, 21, 1.5)
    g = G.run_workload(w, gen.make_inputs)
    det = g["inputs"]["detector"]
    e64 = G.eval_field(g["beamlets"], dict(det, n_u=1, n_v=1))
    e32 = G.eval_field(g["beamlets"], dict(det, n_u=1, n_v=1), precision=G.PRECISION_MIXED)
    assert e32.dtype == torch.complex64 and abs(e32.cpu().numpy()[0, 0].imag) > 1e-3 * abs(e32.cpu().numpy()[0, 0])
    a = G.psf_metrics(g["field"], det, w.wavelength * w.f_number, e64).cpu().numpy()
    b = G.psf_metrics(g["field"], det, w.wavelength * w.f_number, e32).cpu().numpy()
    np.testing.assert_allclose(b[:4], a[:4], rtol=1e-4)


# ----------------------------------------------------------------------------- properties that hold at any size

@pytest.mark.parametrize("algo,precision", [(0, 0), (1, 0), (2, 0), (0, 1)])
def test_properties_of_the_gpu_field_at_bench_size(G, algo, precision):
    """Properties that need no oracle and therefore hold at the full size bench.py times (C3: 31,757 beamlets x
    1024 x 1024 px, table kernel for algo 0): (i) the C3 inputs are symmetric under x -> -x and y -> -y only through
    the lattice, not the random weights, so instead: linearity -- the field of weights W1 + 2 W2 equals E(W1) + 2 E(W2)
    (SURVEY 4(iv)); (ii) shifting the detector origin by m pixels shifts the output array by m pixels; (iii) an
    untilted detector through the general tilted-plane path (origin z = 1e-300) equals the untilted shortcut."""
    w = gen.workload(3)
    tol = 1e-11 if precision == 0 else 3e-5        # each fp64 field is within ~1e-12 of the exact sum (bar: 1e-10)
    b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength)
    inp = gen.make_inputs(w, b.positions.cpu().numpy())
    det = inp["detector"]
    rng = np.random.default_rng(11)
    W1 = inp["weight"]
    W2 = np.stack([rng.standard_normal(b.n), rng.standard_normal(b.n)])

    def field(weight, d=det):
        G.propagate_q(b, 1, inp["abcd"], inp["l0"], None, weight)
        return G.eval_field(b, d, algo=algo, precision=precision).cpu().numpy().astype(np.complex128)
    E1, E2, E12 = field(W1), field(W2), field(W1 + 2.0 * W2)
    scale = np.max(np.abs(E12))
    assert np.max(np.abs(E12 - (E1 + 2.0 * E2))) <= (tol if precision == 0 else 1e-4) * scale          # (i)
    m_u, m_v = 37, -11
    shifted = dict(det, origin=[m_u * det["du"], m_v * det["dv"], 0.0])
    Es = field(W1, shifted)
    # pixel (iu, iv) of the shifted detector is pixel (iu + m_u, iv + m_v) of the original one
    a = Es[max(0, -m_v):1024 - max(0, m_v), 0:1024 - m_u]
    c = E1[max(0, -m_v) + m_v:1024 - max(0, m_v) + m_v, m_u:1024]
    assert a.shape == c.shape and np.max(np.abs(a - c)) <= 50 * tol * np.max(np.abs(E1))                # (ii)
    if algo != 2:            # the separable kernel needs the untilted shortcut's exact zeros in the cross terms
        Et = field(W1, dict(det, origin=[0.0, 0.0, 1e-300]))
        assert np.max(np.abs(Et - E1)) <= 50 * tol * np.max(np.abs(E1))                                 # (iii)


def test_d4_symmetry_of_the_gpu_field(G):
    """C2 member (uniform weights, centred lattice, square detector): E(u,v) = E(-u,v) = E(u,-v) = E(v,u) on the GPU
    output itself, all three fp64 algorithms (the table kernel included: 1.3e8 terms)."""
    w = gen.workload(2, 51, 1.75)
    g = G.run_workload(w, gen.make_inputs)
    for algo in (0, 1, 2):
        E = G.eval_field(g["beamlets"], g["inputs"]["detector"], algo=algo).cpu().numpy()
        s = np.max(np.abs(E))
        for other in (E[:, ::-1], E[::-1, :], E.T):
            assert np.max(np.abs(E - other)) < 1e-11 * s, algo
