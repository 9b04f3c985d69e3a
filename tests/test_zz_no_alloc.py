"""gbd_psf_metrics_static: the one call of libgbd that takes no workspace.

Who it is for: code that needs the figure of merit at a point where it cannot get device memory -- a stage running
inside an application whose own arena holds all of HBM (no allocator handle, nothing left for cudaMalloc), a loop that
may not take the driver's allocation lock, a long job that must not depend on what the heap looks like by then.  Its
scratch is a fixed array inside libgbd.so (GBD_STATIC_METRICS_ROWS rows of 9 doubles per GPU), shared by every call and
never cleared, so what has to hold is: (1) the same numbers as gbd_psf_metrics, the path with a caller's workspace;
(2) still the same numbers on the next call, when the array is full of the previous call's partial sums -- including
a call that uses fewer rows than the one before; (3) a loud refusal, with nothing launched, beyond the array's size.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  The GPU test passes alone in a fresh process (its first call is then the one that
resolves the array's device address) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import gen

# the bars of tests/test_parity_gpu.py for this metric: zone counts bit-exact, RMS / maximum within 4 x 1e-10
ATOL_METRIC = 4e-10


@pytest.fixture(scope="module")
def G():
    from paper_2404_12454_b200 import build
    build.build()
    import paper_2404_12454_b200 as g
    g.load_library()
    return g


def _fields_and_e0(G, n_acrosses, det_n):
    """Fields of a few members of the C2 search on one detector, stacked, and their on-axis values (n, 2)."""
    fields, e0s, det, lfn = [], [], None, None
    for n in n_acrosses:
        w = gen.workload(2, n, 1.25)
        w = gen.Workload(**{**w.__dict__, "det_n": det_n, "det_halfwidth_lfn": 15.0})
        g = G.run_workload(w, gen.make_inputs)
        det = g["inputs"]["detector"]
        lfn = w.wavelength * w.f_number
        fields.append(g["field"])
        e0 = G.eval_field(g["beamlets"], dict(det, n_u=1, n_v=1))
        e0s.append(torch.view_as_real(e0).reshape(2))
    return torch.stack(fields).contiguous(), torch.stack(e0s).contiguous(), det, lfn


def _existing_path(G, fields, e0, det, lfn):
    """gbd_psf_metrics, one call per field, each with its own freshly allocated workspace."""
    return np.stack([G.psf_metrics(fields[i], det, lfn, e0[i]).cpu().numpy() for i in range(fields.shape[0])])


def _assert_same(got, ref):
    assert got.shape == ref.shape
    assert np.array_equal(got[:, 4:8], ref[:, 4:8])                               # pixels per zone
    np.testing.assert_allclose(got[:, :4], ref[:, :4], rtol=0, atol=ATOL_METRIC)  # RMS per zone
    np.testing.assert_allclose(got[:, 8], ref[:, 8], rtol=0, atol=ATOL_METRIC)    # max |I - Airy|
    assert np.all(np.isfinite(got))


@pytest.mark.gpu
def test_static_scratch_metrics_match_the_workspace_path_on_two_calls_in_a_row(G):
    fields, e0, det, lfn = _fields_and_e0(G, (31, 21, 41), 200)        # 3 x 157 block rows of the array
    ref = _existing_path(G, fields, e0, det, lfn)
    assert ref[0, 0] != ref[1, 0] != ref[2, 0]                          # three different answers to tell apart

    out = torch.full((3, 9), float("nan"), dtype=torch.float64, device=fields.device)
    before = G.launch_count()
    got1 = G.psf_metrics_static(fields, det, lfn, e0, out=out)
    assert got1.data_ptr() == out.data_ptr()
    assert G.launch_count() - before == 2                               # libgbd's own kernels ran, both of them
    _assert_same(got1.cpu().numpy(), ref)

    # second call straight after, same stream: the array now holds the first call's sums for (31, 21, 41); ask for
    # the fields in another order, so that stale rows could not pass for fresh ones
    perm = [2, 0, 1]
    got2 = G.psf_metrics_static(fields[perm].contiguous(), det, lfn, e0[perm].contiguous())
    _assert_same(got2.cpu().numpy(), ref[perm])

    # third: fewer rows than the array already holds (one smaller field: 40 rows), in mixed precision, then the first
    # request again -- the leftovers beyond row 40 belong to nobody and must not show up anywhere
    small, e0s, det_s, lfn_s = _fields_and_e0(G, (21,), 100)
    ref_s = _existing_path(G, small, e0s, det_s, lfn_s)
    _assert_same(G.psf_metrics_static(small[0], det_s, lfn_s, e0s).cpu().numpy(), ref_s)
    small32 = small.to(torch.complex64)
    ref_s32 = _existing_path(G, small32, e0s, det_s, lfn_s)
    _assert_same(G.psf_metrics_static(small32, det_s, lfn_s, e0s).cpu().numpy(), ref_s32)
    _assert_same(G.psf_metrics_static(fields, det, lfn, e0).cpu().numpy(), ref)


@pytest.mark.gpu
def test_static_scratch_refuses_more_rows_than_it_has(G):
    """Full-size fields take 592 rows each: 8 fit, 9 do not.  The refusal comes before any launch, so handing it a
    buffer that is too short for 9 fields is safe."""
    det = dict(n_u=1024, n_v=1024, du=1e-3, dv=1e-3, origin=[0, 0, 0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    assert 8 * 592 == G.STATIC_METRICS_ROWS
    lib = G.load_library()
    d = G.Detector.from_dict(det)
    buf = torch.zeros(1024, dtype=torch.float64, device="cuda:0")
    before = G.launch_count()
    rc = lib.gbd_psf_metrics_static(C.c_void_p(buf.data_ptr()), 9, 0, C.byref(d), 1.0,
                                    C.c_void_p(buf.data_ptr()), C.c_void_p(buf.data_ptr()), None)
    assert rc == 2                                                      # GBD_ECAPACITY
    msg = lib.gbd_last_error().decode()
    assert "5328" in msg and "4736" in msg
    assert G.launch_count() == before
    # exactly at the limit it runs (8 full-size fields), and agrees with the workspace path on the first and last
    fields = torch.randn((8, 1024, 1024), dtype=torch.complex128, device="cuda:0")
    e0 = torch.ones((8, 2), dtype=torch.float64, device="cuda:0")
    got = G.psf_metrics_static(fields, det, 0.05, e0).cpu().numpy()
    for i in (0, 7):
        ref = G.psf_metrics(fields[i], det, 0.05, e0[i]).cpu().numpy()
        assert np.array_equal(got[i, 4:8], ref[4:8])
        np.testing.assert_allclose(got[i, [0, 1, 2, 3, 8]], ref[[0, 1, 2, 3, 8]], rtol=1e-12)


def test_static_scratch_limit_is_checked_on_the_host():
    """No GPU needed: the size check precedes every CUDA call, so it can be seen from a CPU-only box.  (The pointers
    are never dereferenced on this path.)"""
    from paper_2404_12454_b200 import build, gbd
    build.build()
    lib = gbd.load_library()
    d = gbd.Detector.from_dict(dict(n_u=128, n_v=128, du=1e-3, dv=1e-3, origin=[0, 0, 0],
                                    e_u=[1, 0, 0], e_v=[0, 1, 0]))                 # 64 rows per field
    fake = C.c_void_p(4096)
    assert lib.gbd_psf_metrics_static(fake, 75, 0, C.byref(d), 1.0, fake, fake, None) == 2
    assert b"4800" in lib.gbd_last_error() and b"4736" in lib.gbd_last_error()
    assert lib.gbd_psf_metrics_static(fake, 0, 0, C.byref(d), 1.0, fake, fake, None) == 1
    assert lib.gbd_psf_metrics_static(None, 1, 0, C.byref(d), 1.0, fake, fake, None) == 1
    assert lib.gbd_psf_metrics_static(fake, 1, 2, C.byref(d), 1.0, fake, fake, None) == 1
