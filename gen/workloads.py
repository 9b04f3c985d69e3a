"""Workload descriptions C0..C4 (BASELINE.json `configs`) and their seeded inputs.

Everything here is INPUT generation.  The hot path (lattice, Q^-1 propagation,
amplitude, tilt re-expansion, field sum) is implemented twice elsewhere --
`oracle/` (CPU, plain C) and `paper_2404_12454_b200/csrc/` (CUDA) -- and neither of
those imports the other; both consume the arrays produced here.

Conventions:
  * lengths in mm;
  * phase-space coordinates on a plane are (q, p) = (in-plane position, in-plane
    components of the unit direction vector), refractive index 1;
  * a 4x4 ray-transfer matrix is stored row-major as [[A, B], [C, D]] acting on
    (q_x, q_y, p_x, p_y) (Eq. 23 layout);
  * random draws: numpy.random.default_rng(SEED_BASE + config index); the draw
    order is stated in each function.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SEED_BASE = 240412454


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    index: int
    wavelength: float          # mm
    pupil_diameter: float      # mm
    n_across: int              # beamlets across the pupil diameter (PAPER.md:245 N_g)
    overlap_factor: float      # PAPER.md:245 Eq. 24
    optics: str                # "ideal_lens" | "paraboloid" | "rc_telescope"
    focal_length: float        # mm
    det_n: int                 # detector is det_n x det_n
    det_halfwidth_lfn: float   # half-width in units of lambda * F#
    jitter: bool = False       # C1: +-1% of pitch, uniform, seeded
    weights: str = "unit"      # "unit" | "apodised_random"
    zernike_rms_waves: float = 0.0
    field_deg: float = 0.0
    tilt_deg: float = 0.0
    seed: int = SEED_BASE
    trace_on_side: bool = False  # True: each side (oracle / CUDA) derives ABCD with its OWN ray tracer

    @property
    def f_number(self) -> float:
        return self.focal_length / self.pupil_diameter

    @property
    def pitch(self) -> float:
        return self.pupil_diameter / self.n_across

    @property
    def det_halfwidth(self) -> float:
        return self.det_halfwidth_lfn * self.wavelength * self.f_number

    @property
    def abcd_mode(self) -> int:
        """1: one shared 4x4 for all beamlets; 0: one 4x4 per beamlet."""
        return 1 if self.optics == "ideal_lens" else 0


_LAM_HENE = 0.6328e-3


def workload(index: int, n_across: Optional[int] = None,
             overlap_factor: Optional[float] = None) -> Workload:
    """BASELINE.json configs[index].  For index 2 (the sweep) pass n_across/overlap_factor."""
    if index == 0:
        return Workload("C0 airy-smoke", 0, _LAM_HENE, 25.4, 11, 1.5, "ideal_lens", 100.0,
                        64, 5.0, seed=SEED_BASE + 0)
    if index == 1:
        return Workload("C1 airy-medium", 1, _LAM_HENE, 25.4, 51, 1.75, "ideal_lens", 100.0,
                        256, 8.0, jitter=True, seed=SEED_BASE + 1)
    if index == 2:
        n = 51 if n_across is None else int(n_across)
        of = 1.5 if overlap_factor is None else float(overlap_factor)
        return Workload(f"C2 sweep N={n} OF={of:g}", 2, _LAM_HENE, 25.4, n, of, "ideal_lens",
                        100.0, 256, 8.0, seed=SEED_BASE + 2)
    if index == 3:
        return Workload("C3 large-focal-plane", 3, _LAM_HENE, 25.4, 201, 2.0, "ideal_lens",
                        4.0 * 25.4, 1024, 16.0, weights="apodised_random", seed=SEED_BASE + 3)
    if index == 4:
        return Workload("C4 paraboloid-tilted", 4, 1.0e-3, 50.0, 101, 1.5, "paraboloid", 50.0,
                        512, 12.0, zernike_rms_waves=0.5, field_deg=0.5, tilt_deg=5.0,
                        seed=SEED_BASE + 4)
    if index == 5:
        # NEXT-1 second workload: the paper's HST-like Ritchey-Chretien telescope, unobscured, on axis
        # (prescription PAPER.md:324-327 Table 2; simulation parameters PAPER.md:345-351
        # Table 3: 551 nm, EPD 2.4 m, EFL 57.6 m, 512 x 512 px of 2.8 mas).  Lengths in mm.
        lam, epd, efl = 551.0e-6, 2400.0, 57600.0
        pixel = efl * math.radians(2.8e-3 / 3600.0)
        half_lfn = 256.0 * pixel / (lam * efl / epd)
        return Workload("C5 hst-like-rc", 5, lam, epd, 101 if n_across is None else int(n_across),
                        1.5 if overlap_factor is None else float(overlap_factor), "rc_telescope", efl,
                        512, half_lfn, seed=SEED_BASE + 5, trace_on_side=True)
    raise ValueError(f"no such config: {index}")


def sweep_workloads():
    """The 90 runs of C2: N in {11,21,...,101} x OF in {1.0,1.25,...,3.0} (N-major order)."""
    out = []
    for n in range(11, 102, 10):
        for iof in range(9):
            out.append(workload(2, n, 1.0 + 0.25 * iof))
    return out


# --------------------------------------------------------------------------- optics inputs

def ideal_lens_abcd(f: float, delta: float = 0.0) -> np.ndarray:
    """PAPER.md:181 Eq. 23: free space (f+delta) after a paraxial thin lens f.  Returns (4,4)."""
    lens = np.eye(4)
    lens[2, 0] = -1.0 / f
    lens[3, 1] = -1.0 / f
    space = np.eye(4)
    space[0, 2] = f + delta
    space[1, 3] = f + delta
    return space @ lens


def jitter_positions(xy: np.ndarray, pitch: float, seed: int) -> np.ndarray:
    """C1: x_j += U(-0.01,0.01)*pitch, y_j likewise.  Draw order: all x offsets, then all y."""
    rng = np.random.default_rng(seed)
    n = xy.shape[1]
    jx = rng.uniform(-0.01, 0.01, n)
    jy = rng.uniform(-0.01, 0.01, n)
    out = np.array(xy, dtype=np.float64, copy=True)
    out[0] += jx * pitch
    out[1] += jy * pitch
    return out


def apodised_random_weights(xy: np.ndarray, pupil_diameter: float, seed: int) -> np.ndarray:
    """C3: W_j = exp(-|r_j|^2/(D/2)^2) * (1 + 0.1*xi_j), xi ~ N(0,1), real.  Returns (2,n) re,im."""
    rng = np.random.default_rng(seed)
    n = xy.shape[1]
    xi = rng.standard_normal(n)
    r2 = xy[0] ** 2 + xy[1] ** 2
    w = np.exp(-r2 / (0.5 * pupil_diameter) ** 2) * (1.0 + 0.1 * xi)
    return np.stack([w, np.zeros(n)]).astype(np.float64)


# Noll Zernike Z4..Z11 on the unit disk in Cartesian form (x, y = r/(D/2)); unit RMS each.
def _zern_terms(x, y):
    r2 = x * x + y * y
    s3, s5, s6, s8 = math.sqrt(3.0), math.sqrt(5.0), math.sqrt(6.0), math.sqrt(8.0)
    return [
        s3 * (2.0 * r2 - 1.0),                               # Z4 defocus
        s6 * (2.0 * x * y),                                  # Z5 rho^2 sin2t
        s6 * (x * x - y * y),                                # Z6 rho^2 cos2t
        s8 * (3.0 * r2 - 2.0) * y,                           # Z7 (3r^3-2r) sin t
        s8 * (3.0 * r2 - 2.0) * x,                           # Z8 (3r^3-2r) cos t
        s8 * (3.0 * x * x * y - y ** 3),                     # Z9 rho^3 sin3t
        s8 * (x ** 3 - 3.0 * x * y * y),                     # Z10 rho^3 cos3t
        s5 * (6.0 * r2 * r2 - 6.0 * r2 + 1.0),               # Z11 spherical
    ]


def _zern_grads(x, y):
    r2 = x * x + y * y
    s3, s5, s6, s8 = math.sqrt(3.0), math.sqrt(5.0), math.sqrt(6.0), math.sqrt(8.0)
    return [
        (s3 * 4.0 * x, s3 * 4.0 * y),
        (s6 * 2.0 * y, s6 * 2.0 * x),
        (s6 * 2.0 * x, -s6 * 2.0 * y),
        (s8 * 6.0 * x * y, s8 * (3.0 * r2 - 2.0 + 6.0 * y * y)),
        (s8 * (3.0 * r2 - 2.0 + 6.0 * x * x), s8 * 6.0 * x * y),
        (s8 * 6.0 * x * y, s8 * (3.0 * x * x - 3.0 * y * y)),
        (s8 * (3.0 * x * x - 3.0 * y * y), -s8 * 6.0 * x * y),
        (s5 * (24.0 * r2 - 12.0) * x, s5 * (24.0 * r2 - 12.0) * y),
    ]


def zernike_coefficients(rms_waves: float, seed: int) -> np.ndarray:
    """c_4..c_11 ~ N(0,1) (one draw of 8), rescaled to sqrt(sum c^2) = rms_waves."""
    rng = np.random.default_rng(seed)
    c = rng.standard_normal(8)
    return c * (rms_waves / math.sqrt(float(np.sum(c * c))))


def zernike_opd(xy: np.ndarray, pupil_diameter: float, coeff_waves: np.ndarray,
                wavelength: float) -> np.ndarray:
    """OPD(r) = lambda * sum_n c_n Z_n(r/(D/2)) in mm."""
    x = xy[0] / (0.5 * pupil_diameter)
    y = xy[1] / (0.5 * pupil_diameter)
    t = _zern_terms(x, y)
    w = sum(c * z for c, z in zip(coeff_waves, t))
    return wavelength * w


def zernike_opd_grad(xy: np.ndarray, pupil_diameter: float, coeff_waves: np.ndarray,
                     wavelength: float) -> np.ndarray:
    """grad OPD in (mm/mm), shape (2,n)."""
    a = 0.5 * pupil_diameter
    x = xy[0] / a
    y = xy[1] / a
    g = _zern_grads(x, y)
    gx = sum(c * gg[0] for c, gg in zip(coeff_waves, g))
    gy = sum(c * gg[1] for c, gg in zip(coeff_waves, g))
    return np.stack([wavelength * gx / a, wavelength * gy / a])


class ParaboloidSystem:
    """C4 optics: concave paraboloid z = r^2/(4f), vertex at the origin, focus at (0,0,f).

    The pupil plane is z = z_pupil; light arrives travelling towards -z, reflects, and is
    evaluated where it crosses the nominal plane z = z_eval (normal +z; light now travels +z).
    Rays are exact (non-paraxial) and n = 1.  The ABCD of each beamlet is a forward finite
    difference of base + 4 differential rays in in-plane (q, p) at both ends
    ("5 parabasal rays", PAPER.md:98 step 4).
    """

    def __init__(self, f: float, z_pupil: float, z_eval: float,
                 dq: float = 1.0e-4, dp: float = 1.0e-6):
        self.f, self.z_pupil, self.z_eval, self.dq, self.dp = f, z_pupil, z_eval, dq, dp

    def trace(self, q: np.ndarray, p: np.ndarray, z_eval=None, plane=None):
        """Trace rays from the pupil plane.  q, p: (2,n).

        Returns (q_out (2,n), p_out (2,n), path (n,), dir3 (3,n), hit3 (3,n)).
        With plane=(origin3, e_u, e_v) the rays are intersected with that plane instead and
        q_out/p_out are in-plane coordinates/direction components in its (e_u, e_v) basis.
        """
        f = self.f
        x0, y0 = q[0], q[1]
        dx, dy = p[0], p[1]
        dz = -np.sqrt(1.0 - dx * dx - dy * dy)
        a = (dx * dx + dy * dy) / (4.0 * f)
        b = (2.0 * (x0 * dx + y0 * dy)) / (4.0 * f) - dz
        c = (x0 * x0 + y0 * y0) / (4.0 * f) - self.z_pupil
        t1 = (-2.0 * c) / (b + np.sqrt(b * b - 4.0 * a * c))
        hx, hy, hz = x0 + t1 * dx, y0 + t1 * dy, self.z_pupil + t1 * dz
        nx, ny, nz = -hx / (2.0 * f), -hy / (2.0 * f), np.ones_like(hx)
        nn = np.sqrt(nx * nx + ny * ny + nz * nz)
        nx, ny, nz = nx / nn, ny / nn, nz / nn
        dn = dx * nx + dy * ny + dz * nz
        rx, ry, rz = dx - 2.0 * dn * nx, dy - 2.0 * dn * ny, dz - 2.0 * dn * nz
        if plane is None:
            ze = self.z_eval if z_eval is None else z_eval
            t2 = (ze - hz) / rz
            ex, ey, ez = hx + t2 * rx, hy + t2 * ry, hz + t2 * rz
            q_out = np.stack([ex, ey])
            p_out = np.stack([rx, ry])
        else:
            o, eu, ev = (np.asarray(v, dtype=np.float64) for v in plane)
            nrm = np.cross(eu, ev)
            num = (o[0] - hx) * nrm[0] + (o[1] - hy) * nrm[1] + (o[2] - hz) * nrm[2]
            den = rx * nrm[0] + ry * nrm[1] + rz * nrm[2]
            t2 = num / den
            ex, ey, ez = hx + t2 * rx, hy + t2 * ry, hz + t2 * rz
            wx, wy, wz = ex - o[0], ey - o[1], ez - o[2]
            q_out = np.stack([wx * eu[0] + wy * eu[1] + wz * eu[2],
                              wx * ev[0] + wy * ev[1] + wz * ev[2]])
            p_out = np.stack([rx * eu[0] + ry * eu[1] + rz * eu[2],
                              rx * ev[0] + ry * ev[1] + rz * ev[2]])
        return q_out, p_out, t1 + t2, np.stack([rx, ry, rz]), np.stack([ex, ey, ez])

    def differential_abcd(self, q: np.ndarray, p: np.ndarray, plane=None):
        """Base + 4 differential rays -> per-beamlet ABCD (n,16), base rays (q_out, p_out, path)."""
        n = q.shape[1]
        qb, pb, path, _, _ = self.trace(q, p, plane=plane)
        m = np.zeros((n, 4, 4))
        for k in range(4):
            dq = np.zeros((2, 1))
            dpp = np.zeros((2, 1))
            if k < 2:
                dq[k, 0] = self.dq
                h = self.dq
            else:
                dpp[k - 2, 0] = self.dp
                h = self.dp
            qk, pk, _, _, _ = self.trace(q + dq, p + dpp, plane=plane)
            m[:, 0:2, k] = ((qk - qb) / h).T
            m[:, 2:4, k] = ((pk - pb) / h).T
        return m.reshape(n, 16), qb, pb, path


def c4_system(w: Workload) -> ParaboloidSystem:
    return ParaboloidSystem(w.focal_length, z_pupil=w.focal_length, z_eval=w.focal_length)


def c4_chief_intercept(w: Workload) -> np.ndarray:
    """Chief ray (pupil centre, field direction, no aberration) on the nominal plane."""
    sysm = c4_system(w)
    p_field = np.array([[0.0], [math.sin(math.radians(w.field_deg))]])
    qc, _, _, _, _ = sysm.trace(np.zeros((2, 1)), p_field)
    return qc[:, 0]


# PAPER.md:324-327 Table 2 (metres there, mm here): RoC, conic constant, distance to the next surface.
HST_TABLE2 = dict(m1_roc=-11040.0, m1_conic=-1.00230, m1_to_m2=-4906.07,
                  m2_roc=1358.0, m2_conic=-1.49686, m2_to_focus=6406.20)


def trace_spec(w: Workload, xy: np.ndarray) -> dict:
    """Description of the optics for the sides' own ray tracers (gbd_trace_mirrors / the oracle's
    gbdo_trace_mirrors): reflecting conics c(x^2+y^2+(1+k)z'^2) - 2z' = 0 with c signed along +z, the
    pupil plane z = z_pupil (light starts towards dir_sign * z), the evaluation frame (origin, e_x, e_y;
    the light arrives along e_x x e_y), finite-difference steps, and the per-beamlet start direction
    p_in (2,n) / start path opl0 (n,) (None -> p_common / 0)."""
    n = xy.shape[1]
    if w.optics == "paraboloid":
        f = w.focal_length
        coeff = zernike_coefficients(w.zernike_rms_waves, w.seed)
        p_field = np.array([0.0, math.sin(math.radians(w.field_deg))])
        grad = zernike_opd_grad(xy, w.pupil_diameter, coeff, w.wavelength)
        opd = zernike_opd(xy, w.pupil_diameter, coeff, w.wavelength)
        return dict(mirrors=[dict(curvature=1.0 / (2.0 * f), conic=-1.0, z_vertex=0.0)],
                    z_pupil=f, dir_sign=-1.0, origin=[0.0, 0.0, f], e_x=[1.0, 0.0, 0.0], e_y=[0.0, 1.0, 0.0],
                    dq=1.0e-4, dp=1.0e-6, p_common=[float(p_field[0]), float(p_field[1])],
                    p_in=np.ascontiguousarray(p_field[:, None] + grad),
                    opl0=np.ascontiguousarray(p_field[0] * xy[0] + p_field[1] * xy[1] + opd))
    if w.optics == "rc_telescope":
        t = HST_TABLE2
        # Table 2's sign convention: negative RoC = concave.  Here the light first travels towards -z, M1
        # (vertex z = 0) opens towards +z, M2 sits at z = +4906.07 with its centre of curvature beyond it,
        # and the focus lies 6406.20 behind M2, i.e. at z = -1500.13 (behind M1); the light arrives
        # travelling -z, so the evaluation frame is (x, -y) with normal -z.
        z_m2 = -t["m1_to_m2"]
        z_focus = z_m2 - t["m2_to_focus"]
        return dict(mirrors=[dict(curvature=-1.0 / t["m1_roc"], conic=t["m1_conic"], z_vertex=0.0),
                             dict(curvature=1.0 / t["m2_roc"], conic=t["m2_conic"], z_vertex=z_m2)],
                    z_pupil=z_m2 + 100.0, dir_sign=-1.0, origin=[0.0, 0.0, z_focus],
                    e_x=[1.0, 0.0, 0.0], e_y=[0.0, -1.0, 0.0], dq=1.0e-2, dp=1.0e-6,
                    p_common=[0.0, 0.0], p_in=None, opl0=None)
    raise ValueError(f"no ray-trace description for optics {w.optics!r}")


# --------------------------------------------------------------------------- detector

def detector_dict(w: Workload) -> dict:
    """Detector descriptor in the nominal-plane frame (X, Y in-plane, Z = normal, z = 0 on it).

    Cell-centred grid (reading A12): pixel (iu, iv) sits at
    origin + (iu-(n_u-1)/2)*du*e_u + (iv-(n_v-1)/2)*dv*e_v, du = 2L/n.
    """
    n = w.det_n
    h = 2.0 * w.det_halfwidth / n
    if w.tilt_deg == 0.0:
        origin = [0.0, 0.0, 0.0]
        e_u = [1.0, 0.0, 0.0]
        e_v = [0.0, 1.0, 0.0]
    else:
        c = c4_chief_intercept(w) if w.optics == "paraboloid" else np.zeros(2)
        t = math.radians(w.tilt_deg)
        origin = [float(c[0]), float(c[1]), 0.0]
        e_u = [1.0, 0.0, 0.0]
        e_v = [0.0, math.cos(t), math.sin(t)]          # rotation about x
    return dict(n_u=n, n_v=n, du=h, dv=h, origin=origin, e_u=e_u, e_v=e_v)


# --------------------------------------------------------------------------- assembled inputs

def make_inputs(w: Workload, xy: np.ndarray) -> dict:
    """All inputs of gbd_propagate_q / gbd_eval_field for workload `w`.

    `xy` (2,n) are the lattice positions produced by step a1 of whichever side is being
    run (oracle or CUDA); this function never builds the lattice itself.
    Returned dict: xy (2,n; jittered for C1), abcd_mode, abcd ((16,) or (n,16)), l0,
    base (None | (3,n) mode 1 | (5,n) mode 0), weight (None | (2,n)), detector (dict).
    """
    xy = np.ascontiguousarray(xy, dtype=np.float64)
    n = xy.shape[1]
    out = dict(abcd_mode=w.abcd_mode, detector=detector_dict(w), l0=0.0, base=None, weight=None)
    if w.jitter:
        xy = jitter_positions(xy, w.pitch, w.seed)
    out["xy"] = xy
    if w.weights == "apodised_random":
        out["weight"] = apodised_random_weights(xy, w.pupil_diameter, w.seed)
    if w.optics == "ideal_lens":
        out["abcd"] = ideal_lens_abcd(w.focal_length).reshape(16).copy()
        out["l0"] = float(w.focal_length)
    elif w.optics == "paraboloid":
        sysm = c4_system(w)
        coeff = zernike_coefficients(w.zernike_rms_waves, w.seed)
        p_field = np.array([0.0, math.sin(math.radians(w.field_deg))])
        opd = zernike_opd(xy, w.pupil_diameter, coeff, w.wavelength)
        grad = zernike_opd_grad(xy, w.pupil_diameter, coeff, w.wavelength)
        p_in = p_field[:, None] + grad
        abcd, qb, pb, path = sysm.differential_abcd(xy, p_in)
        opl = p_field[0] * xy[0] + p_field[1] * xy[1] + opd + path
        out["abcd"] = np.ascontiguousarray(abcd)
        out["base"] = np.ascontiguousarray(np.stack([qb[0], qb[1], pb[0], pb[1], opl]))
        out["zernike_coeff_waves"] = coeff
        assert out["base"].shape == (5, n)
    elif w.optics == "rc_telescope":
        out["abcd"] = None
        out["trace"] = trace_spec(w, xy)
    else:
        raise ValueError(w.optics)
    if w.trace_on_side and w.optics == "paraboloid":
        out["abcd"], out["base"] = None, None
        out["trace"] = trace_spec(w, xy)
    return out
