"""Thin ctypes binding of libgbd.so (include/gbd.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; torch is used for device memory and
streams.  There is NO CPU fallback: if libgbd.so is missing or no CUDA device is present, the
calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgbd.so")

PRECISION_FP64, PRECISION_MIXED = 0, 1
ALGO_DIRECT, ALGO_RECURRENCE, ALGO_SEPARABLE = 0, 1, 2
NREC = 13
NMODE = 12

EXPORTS = [
    "gbd_last_error", "gbd_record_doubles", "gbd_beamlets_create", "gbd_beamlets_create_custom",
    "gbd_beamlets_destroy", "gbd_beamlets_count", "gbd_beamlets_waist", "gbd_beamlets_wavelength",
    "gbd_propagate_q", "gbd_params_bytes", "gbd_eval_field", "gbd_eval_workspace_bytes",
    "gbd_eval_field_host", "gbd_host_workspace_bytes", "gbd_probe_dfma", "gbd_launch_count",
    "gbd_set_profile_events", "gbd_psf_metrics", "gbd_psf_metrics_workspace_bytes",
    "gbd_airy_sweep", "gbd_airy_sweep_workspace_bytes", "gbd_lattice_count", "gbd_trace_mirrors",
    "gbd_eval_field_pointwise", "gbd_pointeval_workspace_bytes", "gbd_hg_modes", "gbd_eval_field_modes",
    "gbd_eval_modes_workspace_bytes", "gbd_psf_metrics_static",
]


class GbdError(RuntimeError):
    pass


class Detector(C.Structure):
    _fields_ = [("n_u", C.c_int), ("n_v", C.c_int), ("du", C.c_double), ("dv", C.c_double),
                ("origin", C.c_double * 3), ("e_u", C.c_double * 3), ("e_v", C.c_double * 3)]

    @classmethod
    def from_dict(cls, d) -> "Detector":
        if isinstance(d, cls):
            return d
        return cls(int(d["n_u"]), int(d["n_v"]), float(d["du"]), float(d["dv"]),
                   (C.c_double * 3)(*d["origin"]), (C.c_double * 3)(*d["e_u"]),
                   (C.c_double * 3)(*d["e_v"]))


MAX_MIRRORS = 8


class ConicMirror(C.Structure):
    _fields_ = [("curvature", C.c_double), ("conic", C.c_double), ("z_vertex", C.c_double)]


class TraceSystem(C.Structure):
    _fields_ = [("n_mirrors", C.c_int), ("mirrors", ConicMirror * MAX_MIRRORS), ("z_pupil", C.c_double),
                ("dir_sign", C.c_double), ("p_common", C.c_double * 2), ("origin", C.c_double * 3),
                ("e_x", C.c_double * 3), ("e_y", C.c_double * 3), ("dq", C.c_double), ("dp", C.c_double)]

    @classmethod
    def from_dict(cls, d) -> "TraceSystem":
        if isinstance(d, cls):
            return d
        mirrors = list(d["mirrors"])
        if len(mirrors) > MAX_MIRRORS:
            raise GbdError(f"at most {MAX_MIRRORS} mirrors")
        t = cls()
        t.n_mirrors = len(mirrors)
        for i, m in enumerate(mirrors):
            t.mirrors[i] = ConicMirror(float(m["curvature"]), float(m["conic"]), float(m["z_vertex"]))
        t.z_pupil, t.dir_sign = float(d["z_pupil"]), float(d["dir_sign"])
        t.p_common = (C.c_double * 2)(*d.get("p_common", (0.0, 0.0)))
        t.origin = (C.c_double * 3)(*d["origin"])
        t.e_x = (C.c_double * 3)(*d["e_x"])
        t.e_y = (C.c_double * 3)(*d["e_y"])
        t.dq, t.dp = float(d["dq"]), float(d["dp"])
        return t


class SweepRun(C.Structure):
    _fields_ = [("n_across", C.c_int), ("pupil_diameter", C.c_double), ("overlap_factor", C.c_double),
                ("wavelength", C.c_double)]


_lib = None


def load_library():
    """dlopen the in-tree libgbd.so and declare prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GbdError(f"{LIB_PATH} not found: build it with `python -m paper_2404_12454_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp, lp = C.c_void_p, C.c_void_p, C.POINTER(C.c_long)
    det = C.POINTER(Detector)
    lib.gbd_last_error.restype = C.c_char_p
    lib.gbd_record_doubles.restype = C.c_int
    lib.gbd_launch_count.restype = C.c_long
    lib.gbd_beamlets_create.restype = C.c_int
    lib.gbd_beamlets_create.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, C.c_double,
                                        C.c_double, dp, C.c_long, lp, vp]
    lib.gbd_beamlets_create_custom.restype = C.c_int
    lib.gbd_beamlets_create_custom.argtypes = [C.POINTER(vp), C.c_long, C.c_double, C.c_double]
    lib.gbd_beamlets_destroy.argtypes = [vp]
    lib.gbd_beamlets_destroy.restype = None
    lib.gbd_beamlets_count.restype = C.c_long
    lib.gbd_beamlets_count.argtypes = [vp]
    lib.gbd_beamlets_waist.restype = C.c_double
    lib.gbd_beamlets_waist.argtypes = [vp]
    lib.gbd_beamlets_wavelength.restype = C.c_double
    lib.gbd_beamlets_wavelength.argtypes = [vp]
    lib.gbd_propagate_q.restype = C.c_int
    lib.gbd_propagate_q.argtypes = [vp, dp, C.c_long, C.c_int, dp, C.c_double, dp, dp, dp, vp]
    lib.gbd_params_bytes.restype = C.c_size_t
    lib.gbd_params_bytes.argtypes = [vp]
    lib.gbd_eval_field.restype = C.c_int
    lib.gbd_eval_field.argtypes = [vp, dp, det, C.c_int, C.c_int, C.c_double, vp, vp, C.c_size_t, vp]
    lib.gbd_eval_workspace_bytes.restype = C.c_size_t
    lib.gbd_eval_workspace_bytes.argtypes = [vp, det, C.c_int]
    lib.gbd_eval_field_host.restype = C.c_int
    lib.gbd_eval_field_host.argtypes = [vp, dp, C.c_int, dp, C.c_double, dp, dp, det, C.c_int,
                                        C.c_int, C.c_double, vp, vp, C.c_size_t, vp]
    lib.gbd_host_workspace_bytes.restype = C.c_size_t
    lib.gbd_host_workspace_bytes.argtypes = [vp, det, C.c_int, C.c_int]
    lib.gbd_eval_field_pointwise.restype = C.c_int
    lib.gbd_eval_field_pointwise.argtypes = [vp, dp, C.c_long, C.c_int, dp, C.c_double, dp, dp, det, vp, vp,
                                             C.c_size_t, vp]
    lib.gbd_pointeval_workspace_bytes.restype = C.c_size_t
    lib.gbd_pointeval_workspace_bytes.argtypes = [vp, det]
    lib.gbd_hg_modes.restype = C.c_int
    lib.gbd_hg_modes.argtypes = [vp, C.c_int, dp, dp, dp, vp]
    lib.gbd_eval_field_modes.restype = C.c_int
    lib.gbd_eval_field_modes.argtypes = [vp, dp, dp, det, vp, vp, C.c_size_t, vp]
    lib.gbd_eval_modes_workspace_bytes.restype = C.c_size_t
    lib.gbd_eval_modes_workspace_bytes.argtypes = [vp, det]
    lib.gbd_set_profile_events.restype = None
    lib.gbd_set_profile_events.argtypes = [vp, vp]
    lib.gbd_psf_metrics.restype = C.c_int
    lib.gbd_psf_metrics.argtypes = [vp, C.c_int, det, C.c_double, dp, dp, vp, C.c_size_t, vp]
    lib.gbd_psf_metrics_workspace_bytes.restype = C.c_size_t
    lib.gbd_psf_metrics_workspace_bytes.argtypes = [det]
    lib.gbd_psf_metrics_static.restype = C.c_int
    lib.gbd_psf_metrics_static.argtypes = [vp, C.c_int, C.c_int, det, C.c_double, dp, dp, vp]
    lib.gbd_trace_mirrors.restype = C.c_int
    lib.gbd_trace_mirrors.argtypes = [vp, dp, C.c_long, dp, dp, C.POINTER(TraceSystem), dp, dp, vp]
    runs = C.POINTER(SweepRun)
    lib.gbd_airy_sweep.restype = C.c_int
    lib.gbd_airy_sweep.argtypes = [runs, C.c_int, dp, C.c_double, det, C.c_double, C.c_int, C.c_int, dp, vp,
                                   vp, C.c_size_t, vp]
    lib.gbd_airy_sweep_workspace_bytes.restype = C.c_size_t
    lib.gbd_airy_sweep_workspace_bytes.argtypes = [runs, C.c_int, det, C.c_int, C.c_int]
    lib.gbd_lattice_count.restype = C.c_long
    lib.gbd_lattice_count.argtypes = [C.c_int, C.c_double]
    lib.gbd_probe_dfma.restype = C.c_int
    lib.gbd_probe_dfma.argtypes = [dp, C.c_long, C.POINTER(C.c_double), vp]
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load_library().gbd_last_error().decode(errors="replace")
        raise GbdError(f"{what} failed (status {rc}): {msg}")


def _stream_ptr(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _dev_f64(t, device):
    if t is None:
        return None
    if not torch.is_tensor(t):
        t = torch.as_tensor(t, dtype=torch.float64)
    return t.to(device=device, dtype=torch.float64).contiguous()


def set_profile_events(ev_start=None, ev_stop=None) -> None:
    """Record the two torch.cuda.Event objects around the field-sum kernel of later eval_field calls."""
    lib = load_library()
    if ev_start is None or ev_stop is None:
        lib.gbd_set_profile_events(None, None)
    else:
        for ev in (ev_start, ev_stop):           # torch creates the cudaEvent_t lazily, on first record
            if not ev.cuda_event:
                ev.record()
        lib.gbd_set_profile_events(C.c_void_p(ev_start.cuda_event), C.c_void_p(ev_stop.cuda_event))


def launch_count() -> int:
    return int(load_library().gbd_launch_count())


class Beamlets:
    """Handle + device positions of one pupil decomposition (gbd_beamlets_create, a1)."""

    def __init__(self, handle, xy, n, device):
        self._h, self.xy, self.n, self.device = handle, xy, n, device
        self.params = None

    def __del__(self):
        try:
            if self._h:
                load_library().gbd_beamlets_destroy(self._h)
                self._h = None
        except Exception:
            pass

    @property
    def waist(self) -> float:
        return float(load_library().gbd_beamlets_waist(self._h))

    @property
    def wavelength(self) -> float:
        return float(load_library().gbd_beamlets_wavelength(self._h))

    @property
    def positions(self) -> torch.Tensor:
        """(2, n) view of the device positions."""
        return self.xy[:, : self.n]


def beamlets_create(n_across, pupil_diameter, overlap_factor, wavelength, waist=0.0,
                    device="cuda:0", stream=None) -> Beamlets:
    lib = load_library()
    device = torch.device(device)
    cap = int(n_across) * int(n_across)
    xy = torch.empty((2, cap), dtype=torch.float64, device=device)
    h = C.c_void_p()
    n = C.c_long(0)
    with torch.cuda.device(device):
        _check(lib.gbd_beamlets_create(C.byref(h), int(n_across), float(pupil_diameter),
                                       float(overlap_factor), float(waist), float(wavelength),
                                       _ptr(xy), cap, C.byref(n), _stream_ptr(stream)),
               "gbd_beamlets_create")
    return Beamlets(h, xy, int(n.value), device)


def beamlets_custom(xy, waist, wavelength, device="cuda:0") -> Beamlets:
    lib = load_library()
    device = torch.device(device)
    xy = _dev_f64(xy, device)
    h = C.c_void_p()
    _check(lib.gbd_beamlets_create_custom(C.byref(h), int(xy.shape[1]), float(waist),
                                          float(wavelength)), "gbd_beamlets_create_custom")
    return Beamlets(h, xy, int(xy.shape[1]), device)


def trace_mirrors(b: Beamlets, system, p_in=None, opl0=None, stream=None):
    """a0 (gbd_trace_mirrors): 5-ray differential trace of every beamlet through the conic mirrors of
    `system` (dict or TraceSystem).  Returns device tensors (abcd (n,16), base (5,n)) for propagate_q mode 0."""
    lib = load_library()
    sysm = TraceSystem.from_dict(system)
    p_in = _dev_f64(p_in, b.device)
    opl0 = _dev_f64(opl0, b.device)
    n = b.n
    if p_in is not None and tuple(p_in.shape) != (2, n):
        raise GbdError("trace_mirrors: p_in must be (2, n)")
    if opl0 is not None and opl0.numel() != n:
        raise GbdError("trace_mirrors: opl0 must have n elements")
    abcd = torch.empty((n, 16), dtype=torch.float64, device=b.device)
    base = torch.empty((5, n), dtype=torch.float64, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_trace_mirrors(b._h, _ptr(b.xy), int(b.xy.shape[1]), _ptr(p_in), _ptr(opl0),
                                     C.byref(sysm), _ptr(abcd), _ptr(base), _stream_ptr(stream)),
               "gbd_trace_mirrors")
    b._trace_keep = (p_in, opl0)
    return abcd, base


def propagate_q(b: Beamlets, abcd_mode, abcd, l0=0.0, base=None, weight=None, out=None,
                stream=None) -> torch.Tensor:
    """a2: returns the device parameter records (n, 13)."""
    lib = load_library()
    abcd = _dev_f64(abcd, b.device)
    base = _dev_f64(base, b.device)
    weight = _dev_f64(weight, b.device)
    n = b.n
    if abcd.numel() != (16 if abcd_mode == 1 else 16 * n):
        raise GbdError("propagate_q: abcd has the wrong size")
    if base is not None and tuple(base.shape) != ((3, n) if abcd_mode == 1 else (5, n)):
        raise GbdError("propagate_q: base has the wrong shape")
    if weight is not None and tuple(weight.shape) != (2, n):
        raise GbdError("propagate_q: weight has the wrong shape")
    if out is None:
        out = torch.empty((n, NREC), dtype=torch.float64, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_propagate_q(b._h, _ptr(b.xy), int(b.xy.shape[1]), int(abcd_mode), _ptr(abcd),
                                   float(l0), _ptr(base), _ptr(weight), _ptr(out),
                                   _stream_ptr(stream)), "gbd_propagate_q")
    b.params = out
    b._keep = (abcd, base, weight)
    return out


def eval_workspace_bytes(b: Beamlets, detector, precision=PRECISION_FP64) -> int:
    det = Detector.from_dict(detector)
    return int(load_library().gbd_eval_workspace_bytes(b._h, C.byref(det), int(precision)))


def eval_field(b: Beamlets, detector, precision=PRECISION_FP64, algo=ALGO_DIRECT, cull_tau=0.0,
               params=None, out=None, workspace=None, stream=None) -> torch.Tensor:
    """a3-a5: returns the device field (n_v, n_u), complex128 (precision 0) or complex64 (1)."""
    lib = load_library()
    det = Detector.from_dict(detector)
    params = b.params if params is None else params
    if params is None:
        raise GbdError("eval_field: call propagate_q first")
    dtype = torch.complex128 if precision == PRECISION_FP64 else torch.complex64
    if out is None:
        out = torch.empty((det.n_v, det.n_u), dtype=dtype, device=b.device)
    need = int(lib.gbd_eval_workspace_bytes(b._h, C.byref(det), int(precision)))
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_eval_field(b._h, _ptr(params), C.byref(det), int(precision), int(algo),
                                  float(cull_tau), _ptr(out), _ptr(workspace), workspace.numel(),
                                  _stream_ptr(stream)), "gbd_eval_field")
    b._ws = workspace
    return out


def eval_field_pointwise(b: Beamlets, abcd_mode, abcd, l0, base, weight, detector, out=None, workspace=None,
                         stream=None) -> torch.Tensor:
    """The point-evaluation baseline (gbd_eval_field_pointwise): returns the device field
    (n_v, n_u) complex128.  Inputs as for propagate_q."""
    lib = load_library()
    det = Detector.from_dict(detector)
    abcd = _dev_f64(abcd, b.device)
    base = _dev_f64(base, b.device)
    weight = _dev_f64(weight, b.device)
    n = b.n
    if abcd.numel() != (16 if abcd_mode == 1 else 16 * n):
        raise GbdError("eval_field_pointwise: abcd has the wrong size")
    if base is not None and tuple(base.shape) != ((3, n) if abcd_mode == 1 else (5, n)):
        raise GbdError("eval_field_pointwise: base has the wrong shape")
    if weight is not None and tuple(weight.shape) != (2, n):
        raise GbdError("eval_field_pointwise: weight has the wrong shape")
    if out is None:
        out = torch.empty((det.n_v, det.n_u), dtype=torch.complex128, device=b.device)
    need = int(lib.gbd_pointeval_workspace_bytes(b._h, C.byref(det)))
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_eval_field_pointwise(b._h, _ptr(b.xy), int(b.xy.shape[1]), int(abcd_mode), _ptr(abcd),
                                            float(l0), _ptr(base), _ptr(weight), C.byref(det), _ptr(out),
                                            _ptr(workspace), workspace.numel(), _stream_ptr(stream)),
               "gbd_eval_field_pointwise")
    b._pe_keep = (abcd, base, weight, workspace)
    return out


def hg_modes(b: Beamlets, abcd_mode, abcd, mode_weight=None, stream=None) -> torch.Tensor:
    """Mode factors of Hermite-Gaussian beamlets of orders m+n <= 2 (gbd_hg_modes): device tensor (n, 12).
    mode_weight: (12, n) = Re, Im of w00, w10, w01, w20, w11, w02, or None (fundamental beamlets)."""
    lib = load_library()
    abcd = _dev_f64(abcd, b.device)
    mode_weight = _dev_f64(mode_weight, b.device)
    n = b.n
    if abcd.numel() != (16 if abcd_mode == 1 else 16 * n):
        raise GbdError("hg_modes: abcd has the wrong size")
    if mode_weight is not None and tuple(mode_weight.shape) != (NMODE, n):
        raise GbdError(f"hg_modes: mode_weight must be ({NMODE}, n)")
    out = torch.empty((n, NMODE), dtype=torch.float64, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_hg_modes(b._h, int(abcd_mode), _ptr(abcd), _ptr(mode_weight), _ptr(out), _stream_ptr(stream)),
               "gbd_hg_modes")
    b._hg_keep = (abcd, mode_weight)
    return out


def eval_field_modes(b: Beamlets, modes, detector, params=None, out=None, workspace=None, stream=None) -> torch.Tensor:
    """gbd_eval_field_modes: the field sum with every term multiplied by its beamlet's mode factor (untilted
    detectors, fp64): device tensor (n_v, n_u) complex128."""
    lib = load_library()
    det = Detector.from_dict(detector)
    params = b.params if params is None else params
    if params is None:
        raise GbdError("eval_field_modes: call propagate_q first")
    if tuple(modes.shape) != (b.n, NMODE) or modes.dtype != torch.float64 or not modes.is_contiguous():
        raise GbdError(f"eval_field_modes: modes must be a contiguous float64 (n, {NMODE}) tensor")
    if out is None:
        out = torch.empty((det.n_v, det.n_u), dtype=torch.complex128, device=b.device)
    need = int(lib.gbd_eval_modes_workspace_bytes(b._h, C.byref(det)))
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=b.device)
    with torch.cuda.device(b.device):
        _check(lib.gbd_eval_field_modes(b._h, _ptr(params), _ptr(modes), C.byref(det), _ptr(out), _ptr(workspace),
                                        workspace.numel(), _stream_ptr(stream)), "gbd_eval_field_modes")
    b._ws_modes = (workspace, modes)
    return out


def host_workspace_bytes(b: Beamlets, detector, abcd_mode, precision=PRECISION_FP64) -> int:
    det = Detector.from_dict(detector)
    return int(load_library().gbd_host_workspace_bytes(b._h, C.byref(det), int(abcd_mode),
                                                       int(precision)))


def eval_field_host(b: Beamlets, h_xy, abcd_mode, h_abcd, l0, h_base, h_weight, detector, h_field,
                    workspace, precision=PRECISION_FP64, algo=ALGO_DIRECT, cull_tau=0.0,
                    stream=None) -> None:
    """End-to-end call with HOST tensors (pinned for full speed); synchronises the stream."""
    lib = load_library()
    det = Detector.from_dict(detector)
    for t in (h_xy, h_abcd, h_base, h_weight, h_field):
        if t is not None and (t.is_cuda or not t.is_contiguous()):
            raise GbdError("eval_field_host: host tensors must be contiguous CPU tensors")
    with torch.cuda.device(b.device):
        _check(lib.gbd_eval_field_host(b._h, _ptr(h_xy), int(abcd_mode), _ptr(h_abcd), float(l0),
                                       _ptr(h_base), _ptr(h_weight), C.byref(det), int(precision),
                                       int(algo), float(cull_tau), _ptr(h_field), _ptr(workspace),
                                       workspace.numel(), _stream_ptr(stream)),
               "gbd_eval_field_host")


def probe_dfma(iters=4096, device="cuda:0", stream=None) -> float:
    """Launch the DFMA-chain probe once; returns the number of thread-level DFMAs it executes."""
    lib = load_library()
    device = torch.device(device)
    sink = torch.zeros(2, dtype=torch.float64, device=device)
    cnt = C.c_double(0.0)
    with torch.cuda.device(device):
        _check(lib.gbd_probe_dfma(_ptr(sink), int(iters), C.byref(cnt), _stream_ptr(stream)),
               "gbd_probe_dfma")
    return float(cnt.value)


def psf_metrics(field, detector, lambda_fnum, e0, out=None, workspace=None, stream=None) -> torch.Tensor:
    """Device figure of merit (gbd_psf_metrics): returns a device tensor of 9 doubles
    [rms_all, rms_0_5, rms_5_10, rms_10_15, n_all, n_0_5, n_5_10, n_10_15, max_abs_diff]."""
    lib = load_library()
    det = Detector.from_dict(detector)
    precision = PRECISION_FP64 if field.dtype == torch.complex128 else PRECISION_MIXED
    dev = field.device
    e0 = e0.reshape(-1)
    if e0.is_complex():                      # complex64 (a 1x1 mixed-precision field) or complex128
        e0 = torch.view_as_real(e0.to(torch.complex128)).reshape(-1)
    e0 = e0.to(device=dev, dtype=torch.float64).contiguous()
    if e0.numel() != 2:
        raise GbdError("psf_metrics: e0 must be one complex number (or its (re, im) pair)")
    if out is None:
        out = torch.empty(9, dtype=torch.float64, device=dev)
    need = int(lib.gbd_psf_metrics_workspace_bytes(C.byref(det)))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    with torch.cuda.device(dev):
        _check(lib.gbd_psf_metrics(_ptr(field), precision, C.byref(det), float(lambda_fnum), _ptr(e0),
                                   _ptr(out), _ptr(workspace), workspace.numel(), _stream_ptr(stream)),
               "gbd_psf_metrics")
    out._keep = (e0, workspace, field)        # stream-ordered work still reads them
    return out


STATIC_METRICS_ROWS = 4736      # GBD_STATIC_METRICS_ROWS of gbd.h


def psf_metrics_static(fields, detector, lambda_fnum, e0, out=None, stream=None) -> torch.Tensor:
    """gbd_psf_metrics_static: the figure of merit of `fields` ((n_fields, n_v, n_u) or (n_v, n_u), complex128 or
    complex64, contiguous, on the GPU) without a workspace, for code that cannot get device memory where it needs the
    metric -- a stage inside an application whose arena owns all of HBM, a loop that must not take the driver's
    allocation lock, a job that must not depend on the state of the heap.  The partial sums go to a 341 kB array built
    into libgbd.so (present on every GPU the library is used on), which bounds the batch: n_fields x blocks(detector)
    <= STATIC_METRICS_ROWS, else GbdError (status 2) and nothing is launched.

    `e0`: device float64 (n_fields, 2), the (re, im) on-axis value of each field.  `out`: device float64
    (n_fields, 9); pass it to keep this wrapper allocation-free as well (it is created with torch.empty otherwise).
    Same values as psf_metrics, field by field.  All calls on one GPU share the array: keep them on one stream.  The
    first call on a GPU resolves the array's device address; make it at start-up, before any stream capture."""
    lib = load_library()
    det = Detector.from_dict(detector)
    if not fields.is_cuda or not fields.is_contiguous() or fields.dtype not in (torch.complex128, torch.complex64):
        raise GbdError("psf_metrics_static: fields must be a contiguous complex CUDA tensor")
    n_fields = 1 if fields.dim() == 2 else int(fields.shape[0])
    if fields.dim() not in (2, 3) or tuple(fields.shape[-2:]) != (det.n_v, det.n_u):
        raise GbdError("psf_metrics_static: fields must be (n_fields, n_v, n_u) or (n_v, n_u)")
    precision = PRECISION_FP64 if fields.dtype == torch.complex128 else PRECISION_MIXED
    dev = fields.device
    if e0.device != dev or e0.dtype != torch.float64 or not e0.is_contiguous() or e0.numel() != 2 * n_fields:
        raise GbdError("psf_metrics_static: e0 must be a contiguous float64 tensor (n_fields, 2) on the fields' GPU")
    if out is None:
        out = torch.empty((n_fields, 9), dtype=torch.float64, device=dev)
    elif out.device != dev or out.dtype != torch.float64 or not out.is_contiguous() or out.numel() != 9 * n_fields:
        raise GbdError("psf_metrics_static: out must be a contiguous float64 tensor (n_fields, 9) on the fields' GPU")
    with torch.cuda.device(dev):
        _check(lib.gbd_psf_metrics_static(_ptr(fields), n_fields, precision, C.byref(det), float(lambda_fnum),
                                          _ptr(e0), _ptr(out), _stream_ptr(stream)), "gbd_psf_metrics_static")
    out._keep = (e0, fields)                  # stream-ordered work still reads them
    return out


def lattice_count(n_across, pupil_diameter) -> int:
    """Number of beamlets gbd_beamlets_create keeps (host arithmetic, no GPU needed)."""
    return int(load_library().gbd_lattice_count(int(n_across), float(pupil_diameter)))


def airy_sweep(runs, abcd, l0, detector, lambda_fnum, precision=PRECISION_FP64, algo=ALGO_DIRECT,
               fields=None, out=None, workspace=None, device="cuda:0", stream=None) -> torch.Tensor:
    """gbd_airy_sweep: the whole beamlet-parameter search in one call.  runs: iterable of
    (n_across, pupil_diameter, overlap_factor, wavelength).  Returns a device tensor (n_runs, 10):
    the 9 values of psf_metrics and the beamlet count.  `fields` (optional, (n_runs, n_v, n_u) complex)
    receives the fields."""
    lib = load_library()
    device = torch.device(device)
    det = Detector.from_dict(detector)
    runs = list(runs)
    arr = (SweepRun * len(runs))(*[SweepRun(int(n), float(d), float(of), float(lam)) for n, d, of, lam in runs])
    abcd = _dev_f64(abcd, device).reshape(16)
    if out is None:
        out = torch.empty((len(runs), 10), dtype=torch.float64, device=device)
    need = int(lib.gbd_airy_sweep_workspace_bytes(arr, len(runs), C.byref(det), int(precision),
                                                  0 if fields is not None else 1))
    if need == 0:
        raise GbdError("airy_sweep: bad runs or detector")
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=device)
    with torch.cuda.device(device):
        _check(lib.gbd_airy_sweep(arr, len(runs), _ptr(abcd), float(l0), C.byref(det), float(lambda_fnum),
                                  int(precision), int(algo), _ptr(out), _ptr(fields), _ptr(workspace),
                                  workspace.numel(), _stream_ptr(stream)), "gbd_airy_sweep")
    out._keep = (abcd, workspace)         # stream-ordered work still reads them
    return out


def run_workload(w, make_inputs, precision=PRECISION_FP64, algo=ALGO_DIRECT, cull_tau=0.0,
                 device="cuda:0"):
    """Whole path a1..a4 for a gen.Workload on the GPU (`make_inputs` = gen.make_inputs).
    Returns dict(beamlets, inputs, params, field) with device tensors."""
    b = beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, device=device)
    inp = make_inputs(w, b.positions.cpu().numpy())
    b.xy[:, : b.n] = torch.as_tensor(inp["xy"], device=b.device)          # C1 jitter, in place
    if inp.get("trace") is not None:                 # ABCD from the library's own differential ray trace
        inp["abcd"], inp["base"] = trace_mirrors(b, inp["trace"], inp["trace"].get("p_in"),
                                                 inp["trace"].get("opl0"))
    params = propagate_q(b, inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    fld = eval_field(b, inp["detector"], precision=precision, algo=algo, cull_tau=cull_tau)
    return dict(beamlets=b, inputs=inp, params=params, field=fld)
