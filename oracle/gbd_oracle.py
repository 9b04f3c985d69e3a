"""ctypes/numpy front end of oracle/gbd_oracle.c (argument marshalling only -- all arithmetic is in C).

TEST INFRASTRUCTURE, not the product; see the header of gbd_oracle.c.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

NREC = 13
_lib = None


class _Det(C.Structure):
    _fields_ = [("n_u", C.c_int), ("n_v", C.c_int), ("du", C.c_double), ("dv", C.c_double),
                ("origin", C.c_double * 3), ("e_u", C.c_double * 3), ("e_v", C.c_double * 3)]


class _Mirror(C.Structure):
    _fields_ = [("curvature", C.c_double), ("conic", C.c_double), ("z_vertex", C.c_double)]


def _det(d: dict) -> _Det:
    return _Det(int(d["n_u"]), int(d["n_v"]), float(d["du"]), float(d["dv"]),
                (C.c_double * 3)(*d["origin"]), (C.c_double * 3)(*d["e_u"]),
                (C.c_double * 3)(*d["e_v"]))


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        lib.gbdo_lattice.restype = C.c_long
        lib.gbdo_lattice.argtypes = [C.c_int, C.c_double, dp, dp, C.c_long]
        lib.gbdo_waist.restype = C.c_double
        lib.gbdo_waist.argtypes = [C.c_double, C.c_double]
        lib.gbdo_propagate.restype = C.c_int
        lib.gbdo_propagate.argtypes = [C.c_long, dp, dp, C.c_double, C.c_double, C.c_int, dp,
                                       C.c_double, dp, dp, dp]
        lib.gbdo_to_detector.restype = C.c_int
        lib.gbdo_to_detector.argtypes = [C.c_long, dp, C.POINTER(_Det), dp]
        lib.gbdo_field_rows.restype = C.c_int
        lib.gbdo_field_rows.argtypes = [C.c_long, dp, C.POINTER(_Det), C.c_double, C.c_double,
                                        C.c_int, C.c_int, C.c_int, dp]
        lib.gbdo_field_pixels.restype = C.c_int
        lib.gbdo_field_pixels.argtypes = [C.c_long, dp, C.POINTER(_Det), C.c_double, C.c_double,
                                          C.c_long, ip, ip, dp]
        lib.gbdo_field_points.restype = C.c_int
        lib.gbdo_field_points.argtypes = [C.c_long, dp, C.c_double, C.c_double, C.c_long, dp, dp, dp]
        lib.gbdo_psf_metrics.restype = C.c_int
        lib.gbdo_psf_metrics.argtypes = [dp, C.POINTER(_Det), C.c_double, dp, dp]
        lib.gbdo_trace_mirrors.restype = C.c_int
        lib.gbdo_trace_mirrors.argtypes = [C.c_long, dp, dp, dp, dp, dp, C.c_double, C.c_double, dp, C.c_int,
                                           C.POINTER(_Mirror), dp, dp, dp, C.c_double, C.c_double, C.c_double,
                                           dp, dp]
        lib.gbdo_field_pointeval.restype = C.c_int
        lib.gbdo_field_pointeval.argtypes = [C.c_long, dp, dp, C.c_double, C.c_double, C.c_int, dp, C.c_double, dp, dp,
                                             C.POINTER(_Det), C.c_int, C.c_int, C.c_int, dp]
        lib.gbdo_hg_modes.restype = C.c_int
        lib.gbdo_hg_modes.argtypes = [C.c_long, C.c_double, C.c_double, C.c_int, dp, dp, dp]
        lib.gbdo_field_rows_modes.restype = C.c_int
        lib.gbdo_field_rows_modes.argtypes = [C.c_long, dp, dp, C.POINTER(_Det), C.c_double, C.c_int, C.c_int,
                                              C.c_int, dp]
        lib.gbdo_num_threads.restype = C.c_int
        lib.gbdo_set_num_threads.argtypes = [C.c_int]
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_load().gbdo_num_threads())


def set_num_threads(t: int) -> None:
    _load().gbdo_set_num_threads(int(t))


def lattice(n_across: int, diameter: float) -> np.ndarray:
    """a1.  Returns xy (2,n)."""
    lib = _load()
    cap = n_across * n_across
    x = np.empty(cap)
    y = np.empty(cap)
    n = lib.gbdo_lattice(n_across, diameter, _p(x), _p(y), cap)
    return np.ascontiguousarray(np.stack([x[:n], y[:n]]))


def waist(overlap_factor: float, pitch: float) -> float:
    return float(_load().gbdo_waist(overlap_factor, pitch))


def propagate(xy, w0, wavelength, abcd_mode, abcd, l0=0.0, base=None, weight=None) -> np.ndarray:
    """a2.  Returns records (n,13) on the nominal plane."""
    lib = _load()
    xy = _f64(xy)
    n = xy.shape[1]
    x, y = np.ascontiguousarray(xy[0]), np.ascontiguousarray(xy[1])
    abcd, base, weight = _f64(abcd), _f64(base), _f64(weight)
    assert abcd.size == (16 if abcd_mode == 1 else 16 * n)
    if base is not None:
        assert base.shape == ((3, n) if abcd_mode == 1 else (5, n))
    if weight is not None:
        assert weight.shape == (2, n)
    rec = np.empty((n, NREC))
    rc = lib.gbdo_propagate(n, _p(x), _p(y), w0, wavelength, abcd_mode, _p(abcd), l0, _p(base),
                            _p(weight), _p(rec))
    if rc:
        raise ValueError("gbdo_propagate: invalid arguments")
    return rec


def to_detector(rec, detector: dict) -> np.ndarray:
    """a3.  Nominal-plane records -> detector-coordinate records (n,13)."""
    lib = _load()
    rec = _f64(rec)
    out = np.empty_like(rec)
    d = _det(detector)
    if lib.gbdo_to_detector(rec.shape[0], _p(rec), C.byref(d), _p(out)):
        raise ValueError("gbdo_to_detector: invalid arguments")
    return out


def field_rows(rec_det, detector, wavelength, v0, v1, vstep=1, cull_tau=0.0, out=None):
    """a4 on rows v0:v1:vstep; returns the full (n_v,n_u) complex array (unvisited rows = 0)."""
    lib = _load()
    rec_det = _f64(rec_det)
    d = _det(detector)
    if out is None:
        out = np.zeros((detector["n_v"], detector["n_u"]), dtype=np.complex128)
    buf = out.view(np.float64)
    if lib.gbdo_field_rows(rec_det.shape[0], _p(rec_det), C.byref(d), wavelength, cull_tau,
                           int(v0), int(v1), int(vstep), _p(buf)):
        raise ValueError("gbdo_field_rows: invalid arguments")
    return out


def field(rec_det, detector, wavelength, cull_tau=0.0) -> np.ndarray:
    """a4 on the whole detector: (n_v, n_u) complex128."""
    return field_rows(rec_det, detector, wavelength, 0, detector["n_v"], 1, cull_tau)


def field_pixels(rec_det, detector, wavelength, iu, iv, cull_tau=0.0) -> np.ndarray:
    lib = _load()
    rec_det = _f64(rec_det)
    d = _det(detector)
    iu = np.ascontiguousarray(iu, dtype=np.int32)
    iv = np.ascontiguousarray(iv, dtype=np.int32)
    out = np.empty(iu.size, dtype=np.complex128)
    ip = C.POINTER(C.c_int)
    if lib.gbdo_field_pixels(rec_det.shape[0], _p(rec_det), C.byref(d), wavelength, cull_tau,
                             iu.size, iu.ctypes.data_as(ip), iv.ctypes.data_as(ip),
                             _p(out.view(np.float64))):
        raise ValueError("gbdo_field_pixels: invalid arguments")
    return out


def field_points(rec_det, wavelength, u, v, cull_tau=0.0) -> np.ndarray:
    lib = _load()
    rec_det = _f64(rec_det)
    u, v = _f64(np.atleast_1d(u)), _f64(np.atleast_1d(v))
    out = np.empty(u.size, dtype=np.complex128)
    if lib.gbdo_field_points(rec_det.shape[0], _p(rec_det), wavelength, cull_tau, u.size, _p(u),
                             _p(v), _p(out.view(np.float64))):
        raise ValueError("gbdo_field_points: invalid arguments")
    return out


def field_pointeval(xy, w0, wavelength, abcd_mode, abcd, l0, base, weight, detector, rows=None) -> np.ndarray:
    """The point-evaluation algorithm (P:88-100 steps 1-6) on the whole detector or rows=(v0, v1, vstep):
    (n_v, n_u) complex128 (unvisited rows = 0).  Inputs as for propagate()."""
    lib = _load()
    xy = _f64(xy)
    n = xy.shape[1]
    x, y = np.ascontiguousarray(xy[0]), np.ascontiguousarray(xy[1])
    abcd, base, weight = _f64(abcd), _f64(base), _f64(weight)
    assert abcd.size == (16 if abcd_mode == 1 else 16 * n)
    d = _det(detector)
    v0, v1, vs = (0, detector["n_v"], 1) if rows is None else rows
    out = np.zeros((detector["n_v"], detector["n_u"]), dtype=np.complex128)
    if lib.gbdo_field_pointeval(n, _p(x), _p(y), w0, wavelength, abcd_mode, _p(abcd), l0, _p(base), _p(weight),
                                C.byref(d), int(v0), int(v1), int(vs), _p(out.view(np.float64))):
        raise ValueError("gbdo_field_pointeval: invalid arguments")
    return out


def hg_modes(n, w0, wavelength, abcd_mode, abcd, mode_weight=None) -> np.ndarray:
    """Mode factors (complex polynomial of degree <= 2 in D) of Hermite-Gaussian beamlets of orders m+n <= 2 (R-23):
    (n, 12).  mode_weight: (12, n) = Re, Im of w00, w10, w01, w20, w11, w02."""
    lib = _load()
    abcd, mode_weight = _f64(abcd), _f64(mode_weight)
    assert abcd.size == (16 if abcd_mode == 1 else 16 * n)
    if mode_weight is not None:
        assert mode_weight.shape == (12, n)
    out = np.empty((n, 12))
    if lib.gbdo_hg_modes(n, w0, wavelength, abcd_mode, _p(abcd), _p(mode_weight), _p(out)):
        raise ValueError("gbdo_hg_modes: invalid arguments")
    return out


def field_modes(rec_det, modes, detector, wavelength, rows=None) -> np.ndarray:
    """Field sum with the mode factors on an untilted detector: (n_v, n_u) complex128."""
    lib = _load()
    rec_det, modes = _f64(rec_det), _f64(modes)
    d = _det(detector)
    v0, v1, vs = (0, detector["n_v"], 1) if rows is None else rows
    out = np.zeros((detector["n_v"], detector["n_u"]), dtype=np.complex128)
    if lib.gbdo_field_rows_modes(rec_det.shape[0], _p(rec_det), _p(modes), C.byref(d), wavelength, int(v0), int(v1),
                                 int(vs), _p(out.view(np.float64))):
        raise ValueError("gbdo_field_rows_modes: invalid arguments (untilted detectors only)")
    return out


def psf_metrics(fld, detector, lambda_fnum, e0) -> np.ndarray:
    """RMS difference to the Airy pattern: [rms_all, rms_0_5, rms_5_10, rms_10_15, 4 counts, max|d|]."""
    lib = _load()
    fld = np.ascontiguousarray(fld, dtype=np.complex128)
    d = _det(detector)
    e = np.array([complex(e0).real, complex(e0).imag])
    out = np.empty(9)
    if lib.gbdo_psf_metrics(_p(fld.view(np.float64)), C.byref(d), float(lambda_fnum), _p(e), _p(out)):
        raise ValueError("gbdo_psf_metrics: invalid arguments")
    return out


def trace_mirrors(xy, spec: dict, p_in=None, opl0=None, wavelength=None):
    """Differential ray trace (5 rays per beamlet) through the conic mirrors of `spec` (see
    gen.trace_spec): returns (abcd (n,16), base (5,n)).  wavelength: the OPL row is reduced modulo it in
    extended precision before it is rounded to double (R-24); None: the full path."""
    lib = _load()
    xy = _f64(xy)
    n = xy.shape[1]
    x, y = np.ascontiguousarray(xy[0]), np.ascontiguousarray(xy[1])
    p_in = _f64(p_in)
    px = None if p_in is None else np.ascontiguousarray(p_in[0])
    py = None if p_in is None else np.ascontiguousarray(p_in[1])
    pc = _f64(spec.get("p_common", [0.0, 0.0]))
    opl0 = _f64(opl0)
    mirrors = spec["mirrors"]
    arr = (_Mirror * max(1, len(mirrors)))(*[_Mirror(float(m["curvature"]), float(m["conic"]),
                                                     float(m["z_vertex"])) for m in mirrors])
    o, ex, ey = _f64(spec["origin"]), _f64(spec["e_x"]), _f64(spec["e_y"])
    abcd = np.empty((n, 16))
    base = np.empty((5, n))
    rc = lib.gbdo_trace_mirrors(n, _p(x), _p(y), _p(px), _p(py), _p(pc), float(spec["dir_sign"]),
                                float(spec["z_pupil"]), _p(opl0), len(mirrors), arr, _p(o), _p(ex), _p(ey),
                                float(spec["dq"]), float(spec["dp"]),
                                0.0 if wavelength is None else float(wavelength), _p(abcd), _p(base))
    if rc:
        raise ValueError("gbdo_trace_mirrors: invalid arguments")
    return abcd, base


def run_workload(w, make_inputs, rows=None):
    """Whole path a1..a4 for a gen.Workload.  `make_inputs` is gen.make_inputs (passed in so this
    module imports nothing but numpy).  rows=(v0,v1,vstep) restricts the field to those rows.
    Returns dict(xy, inputs, rec, rec_det, field)."""
    xy0 = lattice(w.n_across, w.pupil_diameter)
    inp = make_inputs(w, xy0)
    w0 = waist(w.overlap_factor, w.pupil_diameter / w.n_across)
    if inp.get("trace") is not None:                  # ABCD by this side's own differential ray trace
        inp["abcd"], inp["base"] = trace_mirrors(inp["xy"], inp["trace"], inp["trace"].get("p_in"),
                                                 inp["trace"].get("opl0"), wavelength=w.wavelength)
    rec = propagate(inp["xy"], w0, w.wavelength, inp["abcd_mode"], inp["abcd"], inp["l0"],
                    inp["base"], inp["weight"])
    rec_det = to_detector(rec, inp["detector"])
    if rows is None:
        fld = field(rec_det, inp["detector"], w.wavelength)
    else:
        fld = field_rows(rec_det, inp["detector"], w.wavelength, *rows)
    return dict(xy0=xy0, inputs=inp, w0=w0, rec=rec, rec_det=rec_det, field=fld)
