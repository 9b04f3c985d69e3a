"""CPU-side checks of the boundary: libgbd.so builds, loads, exports every symbol include/gbd.h
declares, and validates arguments without touching a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2404_12454_b200 import build, gbd
    build.build()
    return gbd.load_library()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "gbd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gbd_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2404_12454_b200 import gbd
    syms = header_symbols()
    assert len(syms) >= 14
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in gbd.h but not exported"
    assert sorted(gbd.EXPORTS) == syms


def test_record_size_and_error_string(lib):
    assert lib.gbd_record_doubles() == 13
    assert isinstance(lib.gbd_last_error(), bytes)


def test_argument_validation_without_gpu(lib):
    from paper_2404_12454_b200.gbd import Detector
    h = C.c_void_p()
    assert lib.gbd_beamlets_create_custom(C.byref(h), 5, 0.0, 1e-3) == 1        # waist must be > 0
    assert b"waist" in lib.gbd_last_error()
    assert lib.gbd_beamlets_create_custom(C.byref(h), 5, 0.3, 1e-3) == 0
    assert lib.gbd_beamlets_count(h) == 5
    assert lib.gbd_params_bytes(h) == 5 * 13 * 8
    det = Detector.from_dict(dict(n_u=64, n_v=64, du=1e-3, dv=1e-3, origin=[0, 0, 0],
                                  e_u=[1, 0, 0], e_v=[0, 1, 0]))
    assert lib.gbd_eval_workspace_bytes(h, C.byref(det), 0) > 0
    # eval before propagate -> GBD_ESTATE; null pointers -> GBD_EINVAL
    assert lib.gbd_eval_field(h, None, C.byref(det), 0, 0, 0.0, None, None, 0, None) == 1
    bad = Detector.from_dict(dict(n_u=64, n_v=64, du=1e-3, dv=1e-3, origin=[0, 0, 0],
                                  e_u=[1, 0, 0], e_v=[0.5, 1, 0]))
    assert lib.gbd_eval_workspace_bytes(h, C.byref(bad), 0) == 0                 # not orthonormal
    lib.gbd_beamlets_destroy(h)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2404_12454_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt
                assert "gbd_oracle" not in txt
    osrc = open(os.path.join(ROOT, "oracle", "gbd_oracle.c")).read()
    assert "#include \"../" not in osrc and "gbd.h" not in osrc.replace("gbd.h\"", "")


def test_host_lattice_count_matches_oracle_lattice(lib):
    """gbd_lattice_count (host arithmetic the batched sweep plans with) against the oracle's lattice,
    including diameters for which lattice points fall on or next to the clipping circle."""
    import oracle
    for d in (25.4, 50.0, 2.4, 1.0, 10.0, 7.77):
        for n in list(range(1, 66)) + [100, 101, 128, 201, 500, 999, 1000]:
            assert lib.gbd_lattice_count(n, d) == oracle.lattice(n, d).shape[1], (n, d)
    assert lib.gbd_lattice_count(0, 1.0) == -1


def test_trace_and_sweep_argument_validation_without_gpu(lib):
    """The newer entry points reject bad arguments on the host, before any launch."""
    from paper_2404_12454_b200.gbd import Detector, TraceSystem, SweepRun
    h = C.c_void_p()
    assert lib.gbd_beamlets_create_custom(C.byref(h), 5, 0.3, 1e-3) == 0
    spec = dict(mirrors=[dict(curvature=0.01, conic=-1.0, z_vertex=0.0)], z_pupil=50.0, dir_sign=-1.0,
                origin=[0, 0, 50.0], e_x=[1, 0, 0], e_y=[0, 1, 0], dq=1e-4, dp=1e-6)
    t = TraceSystem.from_dict(spec)
    fake = C.c_void_p(0x1000)                    # never dereferenced: validation fails first
    assert lib.gbd_trace_mirrors(h, None, 5, None, None, C.byref(t), fake, fake, None) == 1      # null d_xy
    t_bad = TraceSystem.from_dict(dict(spec, dir_sign=0.5))
    assert lib.gbd_trace_mirrors(h, fake, 5, None, None, C.byref(t_bad), fake, fake, None) == 1
    assert b"dir_sign" in lib.gbd_last_error()
    t_bad = TraceSystem.from_dict(dict(spec, e_y=[0.6, 1, 0]))
    assert lib.gbd_trace_mirrors(h, fake, 5, None, None, C.byref(t_bad), fake, fake, None) == 1
    assert lib.gbd_trace_mirrors(h, fake, 3, None, None, C.byref(t), fake, fake, None) == 1      # xy_stride < n
    lib.gbd_beamlets_destroy(h)

    det = Detector.from_dict(dict(n_u=64, n_v=64, du=1e-3, dv=1e-3, origin=[0, 0, 0],
                                  e_u=[1, 0, 0], e_v=[0, 1, 0]))
    runs = (SweepRun * 2)(SweepRun(11, 25.4, 1.5, 6e-4), SweepRun(21, 25.4, 2.0, 6e-4))
    need = lib.gbd_airy_sweep_workspace_bytes(runs, 2, C.byref(det), 0, 1)
    assert need > (97 + 349) * 13 * 8 + 2 * 64 * 64 * 16
    assert lib.gbd_airy_sweep_workspace_bytes(runs, 2, C.byref(det), 0, 0) < need            # caller-owned fields
    bad = (SweepRun * 1)(SweepRun(0, 25.4, 1.5, 6e-4))
    assert lib.gbd_airy_sweep_workspace_bytes(bad, 1, C.byref(det), 0, 1) == 0
    assert lib.gbd_airy_sweep(runs, 2, fake, 100.0, C.byref(det), 1e-3, 0, 7, fake, None, fake, need, None) == 1
    assert b"algo" in lib.gbd_last_error()
    assert lib.gbd_airy_sweep(runs, 2, fake, 100.0, C.byref(det), 1e-3, 0, 0, fake, None, fake, 16, None) == 2
    assert b"workspace" in lib.gbd_last_error()
