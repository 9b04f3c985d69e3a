"""Pins of the CPU oracle against things other than itself (all CPU; `-m "not gpu"`).

Each test states which part of oracle/gbd_oracle.c it pins and the passage / mathematics that
fixes the expected value.  "P:n" = /root/reference/PAPER.md line n.  None of the expected values
comes from the oracle or from the CUDA path: they are closed forms, brute-force quadrature of the
paper's Collins integral written out in numpy here, scipy's Bessel function, or ray traces.
"""
import json
import math
import os

import numpy as np
import pytest
from scipy.special import j1

import gen
import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
X3, Y3 = [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]


def flat_detector(n=8, h=1e-3, origin=(0.0, 0.0, 0.0)):
    return dict(n_u=n, n_v=n, du=h, dv=h, origin=list(origin), e_u=X3, e_v=Y3)


def single_beamlet_field(abcd, l0, lam, w0, r1m, th1, pts, opd=0.0, weight=None):
    """Oracle field of ONE beamlet (shared-ABCD mode) at in-plane points pts (2,m)."""
    xy = np.array(r1m, dtype=float).reshape(2, 1)
    base = np.array([[th1[0]], [th1[1]], [opd]])
    rec = oracle.propagate(xy, w0, lam, 1, np.asarray(abcd).reshape(16), l0, base, weight)
    rec_det = oracle.to_detector(rec, flat_detector())
    return oracle.field_points(rec_det, lam, pts[0], pts[1]), rec


# ----------------------------------------------------------------------------- a1 lattice

@pytest.mark.parametrize("n,count", [(11, 97), (21, 349), (31, 749), (41, 1313), (51, 2053),
                                     (61, 2933), (71, 3969), (81, 5169), (91, 6509), (101, 8021),
                                     (201, 31757)])
def test_lattice_matches_bruteforce_count(n, count):
    """evenly spaced beamlets, N_g across width W; BASELINE.json: N=11 -> '~97',
    N=51 -> '~2,040', N=201 -> '~31,700', N=101 -> '~8,000'.  Brute force with exact rational
    arithmetic on integers: keep (2i-(N-1))^2 + (2j-(N-1))^2 <= N^2."""
    xy = oracle.lattice(n, 25.4)
    i = 2 * np.arange(n) - (n - 1)
    keep = (i[None, :] ** 2 + i[:, None] ** 2) <= n * n
    assert xy.shape[1] == int(keep.sum()) == count
    # order: iy slow, ix fast; cell-centred coordinates
    jj, ii = np.nonzero(keep)
    pitch = 25.4 / n
    np.testing.assert_allclose(xy[0], (ii - (n - 1) / 2) * pitch, rtol=0, atol=1e-13)
    np.testing.assert_allclose(xy[1], (jj - (n - 1) / 2) * pitch, rtol=0, atol=1e-13)
    assert np.all(np.hypot(xy[0], xy[1]) <= 12.7)


def test_waist_from_overlap_factor():
    """P:245 Eq. 24: OF = N_g * 2 w0 / W."""
    n, width, of = 51, 25.4, 1.75
    w0 = oracle.waist(of, width / n)
    assert abs(n * 2 * w0 / width - of) < 1e-15


# ----------------------------------------------------------------------------- P1 closed forms

def test_focused_gaussian_closed_form():
    """Pins Q2^-1 (Eq. 22), amplitude and its branch (Eq. 21), sign of Q1^-1.
    Single on-axis beamlet, ideal lens f, evaluated at z = f (Eq. 23):
    Q^-1 = 1/f - i zR/f^2, amplitude = +i zR/f, |E(r)| = (w0/wf) exp(-r^2/wf^2), wf = lambda f/(pi w0)
    (BASELINE.json north_star check 1)."""
    lam, f, w0 = 0.6328e-3, 100.0, 1.7
    zr = math.pi * w0 ** 2 / lam
    wf = lam * f / (math.pi * w0)
    r = np.linspace(0, 3 * wf, 7)
    pts = np.stack([r * math.cos(0.3), r * math.sin(0.3)])
    E, rec = single_beamlet_field(gen.ideal_lens_abcd(f), f, lam, w0, (0, 0), (0, 0), pts)
    rec = rec[0]
    assert abs(rec[5] - 1 / f) < 1e-12 / f and abs(rec[9] - 1 / f) < 1e-12 / f
    assert abs(rec[6] + zr / f ** 2) < 1e-13 * zr / f ** 2
    assert abs(rec[7]) < 1e-18 and abs(rec[8]) < 1e-18
    amp = complex(rec[11], rec[12])
    assert abs(amp - 1j * zr / f) < 1e-13 * zr / f
    np.testing.assert_allclose(np.abs(E), (w0 / wf) * np.exp(-r ** 2 / wf ** 2), rtol=2e-13)
    # phase on axis: exp(-ik f) * (+i) with k f taken modulo 2 pi exactly
    ph = np.exp(-2j * math.pi * math.fmod(f, lam) / lam) * 1j
    assert abs(E[0] / abs(E[0]) - ph) < 1e-12


@pytest.mark.parametrize("delta", [-3.0, -0.4, 0.0, 0.05, 1.0, 7.0])
def test_gaussian_beam_through_focus_textbook(delta):
    """Scalar ABCD law q2 = (A q1 + B)/(C q1 + D) with q1 = i zR and the textbook on-axis field
    sqrt-free form E(0) = 1/(A + B/q1) (Siegman, cited at P:388): pins Eq. 21/22 and the
    continuity of the amplitude branch through focus (reading R-5: Gouy phase runs 0 -> -pi)."""
    lam, f, w0 = 1.0e-3, 100.0, 3.0
    zr = math.pi * w0 ** 2 / lam
    z = f + delta
    A, B, Cc, D = 1 - z / f, z, -1 / f, 1.0
    q1 = 1j * zr
    q2 = (A * q1 + B) / (Cc * q1 + D)
    E, rec = single_beamlet_field(gen.ideal_lens_abcd(f, delta), 0.0, lam, w0, (0, 0), (0, 0),
                                  np.zeros((2, 1)))
    assert abs(complex(rec[0][5], rec[0][6]) - 1 / q2) < 1e-12 * abs(1 / q2)
    # 2-D isotropic: amplitude = 1/(A + B/q1) exactly (no square root, no branch)
    assert abs(E[0] - 1 / (A + B / q1)) < 1e-12 * abs(E[0])
    # beam radius from Im(Q^-1) = -lambda/(pi w^2) vs textbook w(z)
    wz = w0 * math.sqrt((1 - z / f) ** 2 + (z / zr) ** 2)
    assert abs(-lam / (math.pi * rec[0][6]) - wz ** 2) < 1e-11 * wz ** 2


# ----------------------------------------------------------------------------- P2 Collins quadrature

def collins_quadrature(abcd, l0, lam, w0, r1m, th1, r2, half=6.4, npts=1201):
    """Brute-force trapezoid quadrature of P:82 Eq. 13 with K of P:62 Eq. 6 (n1 = 1):
       E2(r2) = i/(lambda sqrt(det B)) e^{-i k l0} Int E1(r1)
                exp(-(ik/2)[r2^T D B^-1 r2 + r1^T B^-1 A r1 - 2 r1^T B^-1 r2]) d^2 r1
    for E1 = exp(-|r1-r1M|^2/w0^2) exp(-i k th1.(r1-r1M))  (a decentred, tilted Gaussian)."""
    M = np.asarray(abcd, dtype=float).reshape(4, 4)
    A, B, D = M[:2, :2], M[:2, 2:], M[2:, 2:]
    Bi = np.linalg.inv(B)
    S, T = Bi @ A, D @ Bi
    k = 2 * math.pi / lam
    g = np.linspace(-half * w0, half * w0, npts)
    h = g[1] - g[0]
    dx, dy = np.meshgrid(g, g, indexing="xy")
    x1, y1 = dx + r1m[0], dy + r1m[1]
    E1 = np.exp(-(dx ** 2 + dy ** 2) / w0 ** 2) * np.exp(-1j * k * (th1[0] * dx + th1[1] * dy))
    q11 = S[0, 0] * x1 * x1 + (S[0, 1] + S[1, 0]) * x1 * y1 + S[1, 1] * y1 * y1
    K = 1j / (lam * np.sqrt(np.linalg.det(B) + 0j)) * np.exp(-2j * math.pi * math.fmod(l0, lam) / lam)
    out = []
    for x2, y2 in zip(*r2):
        q22 = T[0, 0] * x2 * x2 + (T[0, 1] + T[1, 0]) * x2 * y2 + T[1, 1] * y2 * y2
        bx = Bi[0, 0] * x2 + Bi[0, 1] * y2
        by = Bi[1, 0] * x2 + Bi[1, 1] * y2
        ph = q22 + q11 - 2 * (x1 * bx + y1 * by)
        out.append(K * np.sum(E1 * np.exp(-0.5j * k * ph)) * h * h)
    return np.array(out)


def test_collins_quadrature_paper_section_4_1():
    """The paper's own validation: decentred Gaussian through a lens, 1 mm past focus.
    Pins the whole per-term expression: centre (Eq. 28), linear phase (Eq. 29 / the cross term of
    Eq. 19), constant phase (Eq. 17), Q2^-1, amplitude, and reading R-4 (envelope centred on r2M)."""
    g = json.load(open(os.path.join(GOLD, "paper_sec4_1_decentred_gaussian.json")))
    f, w0, lam, z = g["focal_length"], g["waist_radius"], g["wavelength"], g["propagation_distance"]
    abcd = gen.ideal_lens_abcd(f, z - f)
    r1m = g["decentre"]
    zr = math.pi * w0 ** 2 / lam
    wz = w0 * math.sqrt((1 - z / f) ** 2 + (z / zr) ** 2)
    c = (1 - z / f) * np.array(r1m)                      # Eq. 28 with theta = 0
    assert np.allclose(c, [0.0, -0.1], atol=1e-12) and abs(wz - 0.0319) < 1e-4
    pts = c[:, None] + wz * np.array([[0.0, 0.7, -0.5, 1.2, 0.0], [0.0, 0.2, 0.9, -0.6, -1.5]])
    E, rec = single_beamlet_field(abcd, z, lam, w0, r1m, (0, 0), pts)
    np.testing.assert_allclose(rec[0][:2], c, atol=1e-13)
    ref = collins_quadrature(abcd, z, lam, w0, r1m, (0, 0), pts)
    assert np.max(np.abs(E / ref - 1)) < 1e-11
    # the literal Eq. 19-20 form (envelope centred on r2 = 0) would be ~0 here: make sure we are not
    assert abs(E[0]) > 0.99 * w0 / wz * 0.999 and abs(E[0]) < 1.01 * w0 / wz


def rotated_cyl_system():
    """free 5 -> cylindrical lens pair (f=100 along an axis at 0.4 rad, f=140 across) -> free 60."""
    def free(d):
        m = np.eye(4)
        m[0, 2] = m[1, 3] = d
        return m
    c, s = math.cos(0.4), math.sin(0.4)
    R = np.array([[c, -s], [s, c]])
    P = R @ np.diag([1 / 100.0, 1 / 140.0]) @ R.T
    lens = np.eye(4)
    lens[2:, :2] = -P
    return free(60.0) @ lens @ free(5.0), 65.0


def test_collins_quadrature_astigmatic_decentred_tilted():
    """General nonorthogonal ABCD (Eq. 6 'nonorthogonal optical systems'), decentre AND tilt:
    pins matrix ordering in Eq. 22 / Eq. 28-29 (a transposed or swapped operand fails), the
    Q_xy + Q_yx cross term, the theta.r term of the constant phase (R-8)."""
    abcd, l0 = rotated_cyl_system()
    J = np.block([[np.zeros((2, 2)), np.eye(2)], [-np.eye(2), np.zeros((2, 2))]])
    assert np.max(np.abs(abcd.T @ J @ abcd - J)) < 1e-14           # P:70-78 Eq. 8-12
    lam, w0 = 1.0e-3, 0.5
    r1m, th1 = (1.3, -0.7), (2e-3, -1e-3)
    M = abcd
    c = M[:2, :2] @ np.array(r1m) + M[:2, 2:] @ np.array(th1)
    pts = c[:, None] + np.array([[0.0, 0.05, -0.08, 0.02], [0.0, 0.03, 0.04, -0.09]])
    E, rec = single_beamlet_field(abcd, l0, lam, w0, r1m, th1, pts)
    ref = collins_quadrature(abcd, l0, lam, w0, r1m, th1, pts)
    assert np.max(np.abs(E / ref - 1)) < 1e-11
    # symplectic ABCD -> Q symmetric (so the record's Q_xy+Q_yx loses nothing)
    assert abs(rec[0][7]) > 1e-6                                    # cross term is exercised


# ----------------------------------------------------------------------------- P3 Airy, P3' lattice

def airy(r, lam_fnum):
    x = math.pi * np.asarray(r) / lam_fnum
    out = np.ones_like(x)
    nz = x != 0
    out[nz] = (2 * j1(x[nz]) / x[nz]) ** 2
    return out


def psf_rms_vs_airy(w):
    res = oracle.run_workload(w, gen.make_inputs)
    det = res["inputs"]["detector"]
    E0 = oracle.field_points(res["rec_det"], w.wavelength, 0.0, 0.0)[0]
    I = np.abs(res["field"]) ** 2 / abs(E0) ** 2
    u = (np.arange(det["n_u"]) - (det["n_u"] - 1) / 2) * det["du"]
    uu, vv = np.meshgrid(u, u, indexing="xy")
    ref = airy(np.hypot(uu, vv), w.wavelength * w.f_number)
    return float(np.sqrt(np.mean((I - ref) ** 2))), float(np.max(np.abs(I - ref)))


def test_airy_pattern_c0_and_trend():
    """GBD of a uniformly lit circular pupil targets the Airy pattern
    (2 J1(x)/x)^2 (BASELINE.json check 3).  GBD is not exact: loose bound + the paper's trend
    'more beamlets -> lower RMS'."""
    rms0, max0 = psf_rms_vs_airy(gen.workload(0))
    assert rms0 < 1e-2 and max0 < 5e-2
    rms = []
    for n in (11, 21, 41):
        w = gen.workload(2, n, 1.5)
        w = gen.Workload(**{**w.__dict__, "det_n": 64})
        rms.append(psf_rms_vs_airy(w)[0])
    assert rms[0] > rms[1] > rms[2]
    assert rms[2] < 1e-3


def test_c2_detector_matches_paper_geometry():
    """The C2 stand-in (256 px over +-8 lambda F#) has the shape of the paper's timed workload:
    256 px at 2.8 mas, EPD 2.4 m, 551 nm -> +-7.57 lambda/D."""
    g = json.load(open(os.path.join(GOLD, "paper_table2_table3.json")))
    t3 = g["table3"]
    lam_over_d_mas = t3["wavelength_nm"] * 1e-9 / t3["epd_m"] * 180 / math.pi * 3600e3
    half = g["fig7"]["npix"] / 2 * g["fig7"]["pixelscale_mas"] / lam_over_d_mas
    w = gen.workload(2, 51, 1.5)
    assert abs(half - 7.57) < 0.01 and abs(w.det_halfwidth_lfn / half - 1) < 0.06
    assert w.det_n == g["fig7"]["npix"]


def test_unclipped_lattice_dirichlet_closed_form():
    """Unclipped N x N lattice, unit weights, focus: every beamlet has c = 0, the same Q^-1 and
    amplitude, p_j = -r_j/f, so the sum is a product of Dirichlet kernels:
      E(u,v) = amp * exp(-ik f) exp(-(ik/2) Q (u^2+v^2)) D_N(k pitch u/f) D_N(k pitch v/f),
      D_N(t) = sin(N t/2)/sin(t/2).
    Pins the SUM (indexing, the sign of the linear term p.Delta) sharply."""
    lam, f, n, pitch, w0 = 0.6328e-3, 100.0, 9, 2.0, 1.4
    i = (np.arange(n) - (n - 1) / 2) * pitch
    xx, yy = np.meshgrid(i, i, indexing="xy")
    xy = np.stack([xx.ravel(), yy.ravel()])
    rec = oracle.propagate(xy, w0, lam, 1, gen.ideal_lens_abcd(f).reshape(16), f)
    rec_det = oracle.to_detector(rec, flat_detector())
    u = np.array([0.0, 1.3e-3, -2.2e-3, 4.0e-3, 7.7e-3])
    v = np.array([0.0, -0.4e-3, 3.1e-3, 5.0e-3, -6.1e-3])
    E = oracle.field_points(rec_det, lam, u, v)
    k = 2 * math.pi / lam
    zr = math.pi * w0 ** 2 / lam
    Q = 1 / f - 1j * zr / f ** 2
    amp = 1j * zr / f

    def dirichlet(t):
        t = np.asarray(t, dtype=float)
        out = np.full_like(t, float(n))
        nz = np.abs(np.sin(t / 2)) > 1e-12
        out[nz] = np.sin(n * t[nz] / 2) / np.sin(t[nz] / 2)
        return out
    ref = (amp * np.exp(-2j * math.pi * math.fmod(f, lam) / lam)
           * np.exp(-0.5j * k * Q * (u ** 2 + v ** 2))
           * dirichlet(k * pitch * u / f) * dirichlet(k * pitch * v / f))
    assert np.max(np.abs(E - ref)) < 1e-11 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------- P4 symmetry, power

def test_d4_symmetry_c0():
    """C0 inputs are symmetric under x -> -x and x <-> y, so E(u,v) = E(-u,v) = E(v,u): pins the
    output layout [n_v][n_u] and pixel-coordinate indexing (BASELINE.json check 4)."""
    E = oracle.run_workload(gen.workload(0), gen.make_inputs)["field"]
    s = np.max(np.abs(E))
    assert np.max(np.abs(E - E[:, ::-1])) < 1e-12 * s
    assert np.max(np.abs(E - E[::-1, :])) < 1e-12 * s
    assert np.max(np.abs(E - E.T)) < 1e-12 * s


def test_field_layout_is_v_slow_u_fast():
    """One off-axis beamlet displaced along +u only: the bright column must be at high iu."""
    lam, f = 1e-3, 100.0
    abcd = gen.ideal_lens_abcd(f, 1.0)
    xy = np.array([[-10.0], [0.0]])                     # A = -0.01 -> centre at u = +0.1
    rec = oracle.propagate(xy, 3.0, lam, 1, abcd.reshape(16), 101.0)
    det = dict(n_u=16, n_v=4, du=0.02, dv=0.02, origin=[0, 0, 0], e_u=X3, e_v=Y3)
    E = oracle.field(oracle.to_detector(rec, det), det, lam)
    assert E.shape == (4, 16)
    assert np.argmax(np.abs(E).sum(axis=0)) in (12, 13)


def test_power_invariant_general_abcd():
    """Collins propagation conserves power (standard Gaussian law): for one beamlet
    Int |E|^2 d^2r = pi w0^2/2 |W|^2.  Checked two ways: from the record (closed-form Gaussian
    integral) and by summing the oracle's field on a grid (pins the envelope the sum produces)."""
    abcd, l0 = rotated_cyl_system()
    lam, w0 = 1.0e-3, 0.5
    W = np.array([[0.6], [-0.8]])
    xy = np.array([[0.4], [0.2]])
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), l0, None, W)
    k = 2 * math.pi / lam
    r = rec[0]
    amp2 = r[11] ** 2 + r[12] ** 2
    imq = np.array([[r[6], r[8] / 2], [r[8] / 2, r[10]]])
    closed = amp2 * math.pi / (k * math.sqrt(np.linalg.det(-imq)))
    assert abs(closed / (math.pi * w0 ** 2 / 2) - 1) < 1e-12
    n, h = 900, 4.0e-3
    det = dict(n_u=n, n_v=n, du=h, dv=h, origin=[r[0], r[1], 0.0], e_u=X3, e_v=Y3)
    E = oracle.field(oracle.to_detector(rec, det), det, lam)
    assert abs(np.sum(np.abs(E) ** 2) * h * h / (math.pi * w0 ** 2 / 2) - 1) < 1e-9


# ----------------------------------------------------------------------------- P5 tilted plane (a3)

def test_tilt_zero_general_path_equals_untilted():
    """R-T with s -> 0 and e_u = X, e_v = Y must reproduce the nominal-plane records.  The general
    path is forced by origin z = 1e-300 (the untilted shortcut needs z == 0 exactly)."""
    w = gen.workload(4)
    xy = oracle.lattice(21, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    rec = oracle.propagate(inp["xy"], 0.5, w.wavelength, 0, inp["abcd"], 0.0, inp["base"])
    o = inp["detector"]["origin"]
    a = oracle.to_detector(rec, flat_detector(origin=(o[0], o[1], 0.0)))
    b = oracle.to_detector(rec, flat_detector(origin=(o[0], o[1], 1e-300)))
    scale = np.maximum(np.abs(a), 1e-3)
    assert np.max(np.abs(a - b) / scale) < 1e-12


def test_plane_shift_equals_extra_free_space_on_axis():
    """Detector plane shifted by dz along the axis, on-axis beamlet: must equal Eq. 22/21 with the
    ABCD of P:181 Eq. 23 with delta_f = dz.  Pins s, M(I+sM)^-1, amplitude/sqrt det(I+sM) and
    opl' = opl + s in gbdo_to_detector."""
    lam, f, w0 = 1e-3, 100.0, 3.0
    xy = np.zeros((2, 1))
    for dz in (0.7, -0.3, 2.5):
        rec0 = oracle.propagate(xy, w0, lam, 1, gen.ideal_lens_abcd(f, 0.0).reshape(16), f)
        a = oracle.to_detector(rec0, flat_detector(origin=(0, 0, dz)))[0]
        rec1 = oracle.propagate(xy, w0, lam, 1, gen.ideal_lens_abcd(f, dz).reshape(16), f + dz)
        b = oracle.to_detector(rec1, flat_detector())[0]
        # opl compared modulo lambda
        d_opl = (a[4] - b[4]) / lam
        assert abs(d_opl - round(d_opl)) < 1e-9
        np.testing.assert_allclose(a[5:], b[5:], rtol=1e-10, atol=1e-14)


def test_inplane_rotation_of_detector_axes_is_invariant():
    """Rotating (e_u, e_v) about the plane normal changes coordinates, not the field: the field at
    the same physical points must agree.  Pins P' / P0 handling in R-T."""
    w = gen.workload(4)
    xy = oracle.lattice(15, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    rec = oracle.propagate(inp["xy"], 0.6, w.wavelength, 0, inp["abcd"], 0.0, inp["base"])
    o = inp["detector"]["origin"]
    al = 0.3
    ca, sa = math.cos(al), math.sin(al)
    d0 = dict(n_u=4, n_v=4, du=1e-3, dv=1e-3, origin=[o[0], o[1], 1e-300], e_u=X3, e_v=Y3)
    d1 = dict(d0, e_u=[ca, sa, 0.0], e_v=[-sa, ca, 0.0])
    u = np.array([0.0, 3e-3, -5e-3, 8e-3])
    v = np.array([0.0, -2e-3, 6e-3, 1e-3])
    E0 = oracle.field_points(oracle.to_detector(rec, d0), w.wavelength, u, v)
    u1, v1 = ca * u + sa * v, -sa * u + ca * v                      # same physical points
    E1 = oracle.field_points(oracle.to_detector(rec, d1), w.wavelength, u1, v1)
    assert np.max(np.abs(E0 - E1)) < 1e-9 * np.max(np.abs(E0))


def _route_b_records(w, xy, plane, w0):
    """Trace base + differential rays DIRECTLY onto the tilted plane (longdouble, central
    differences) and build in-plane ABCD there; then Eq. 21/22 on that plane, no tilt formulas."""
    sysm = gen.workloads.c4_system(w)
    coeff = gen.workloads.zernike_coefficients(w.zernike_rms_waves, w.seed)
    ld = np.longdouble
    p_field = np.array([0.0, math.sin(math.radians(w.field_deg))])
    grad = gen.zernike_opd_grad(xy, w.pupil_diameter, coeff, w.wavelength)
    opd = gen.zernike_opd(xy, w.pupil_diameter, coeff, w.wavelength)
    q = xy.astype(ld)
    p = (p_field[:, None] + grad).astype(ld)
    n = xy.shape[1]

    def jac(pl):
        qb, pb, path, _, _ = sysm.trace(q, p, plane=pl)
        m = np.zeros((n, 4, 4), dtype=ld)
        for kk in range(4):
            h = ld(1e-5) if kk < 2 else ld(1e-6)
            dq = np.zeros((2, 1), dtype=ld)
            dp = np.zeros((2, 1), dtype=ld)
            (dq if kk < 2 else dp)[kk % 2, 0] = h
            qp, pp, _, _, _ = sysm.trace(q + dq, p + dp, plane=pl)
            qm, pm, _, _, _ = sysm.trace(q - dq, p - dp, plane=pl)
            m[:, 0:2, kk] = ((qp - qm) / (2 * h)).T
            m[:, 2:4, kk] = ((pp - pm) / (2 * h)).T
        opl = p_field[0] * xy[0] + p_field[1] * xy[1] + opd + path.astype(float)
        base = np.stack([qb[0], qb[1], pb[0], pb[1], opl]).astype(float)
        return m.reshape(n, 16).astype(float), base
    abcd_n, base_n = jac(None)                                     # nominal plane (accurate ABCD)
    abcd_t, base_t = jac(plane)                                    # tilted plane, its own frame
    rec_n = oracle.propagate(xy, w0, w.wavelength, 0, abcd_n, 0.0, base_n)
    rec_t = oracle.propagate(xy, w0, w.wavelength, 0, abcd_t, 0.0, base_t)
    return rec_n, rec_t


def test_tilted_plane_route_a_equals_direct_trace_route_b():
    """R-T pinned by physics it does not use: (A) records on the nominal plane re-expanded onto the
    5-degree tilted detector by gbdo_to_detector, versus (B) ABCD obtained by ray tracing straight
    onto the tilted plane and Eq. 21/22 applied there.  In-plane (q,p) are canonical on any plane,
    so both must give the same centre, tilt, path, curvature and amplitude."""
    w = gen.workload(4)
    det = gen.detector_dict(w)
    xy = oracle.lattice(9, w.pupil_diameter)
    w0 = 0.4
    plane = ([det["origin"][0], det["origin"][1], w.focal_length + det["origin"][2]],
             det["e_u"], det["e_v"])
    rec_n, rec_t = _route_b_records(w, xy, plane, w0)
    a = oracle.to_detector(rec_n, det)                             # route A
    b = rec_t                                                      # route B (already in (u,v))
    assert np.max(np.abs(a[:, 0:2] - b[:, 0:2])) < 1e-12           # centres (mm)
    assert np.max(np.abs(a[:, 2:4] - b[:, 2:4])) < 1e-13           # direction cosines
    d = (a[:, 4] - b[:, 4]) / w.wavelength
    assert np.max(np.abs(d - np.round(d))) < 1e-8                  # path modulo lambda
    qscale = np.max(np.abs(b[:, 5:11]))
    assert np.max(np.abs(a[:, 5:11] - b[:, 5:11])) < 2e-7 * qscale  # curvature
    amp_a = a[:, 11] + 1j * a[:, 12]
    amp_b = b[:, 11] + 1j * b[:, 12]
    assert np.max(np.abs(amp_a / amp_b - 1)) < 2e-7                # amplitude incl. branch


# ----------------------------------------------------------------------------- P6 generator sanity

def test_paraboloid_generator_on_axis_and_symplectic():
    """Inputs, not oracle: a paraboloid images an on-axis collimated beam perfectly: every base
    ray hits (0,0,f) with path z_pupil + f; finite-difference ABCD is symplectic to O(step)."""
    w = gen.workload(4)
    sysm = gen.workloads.c4_system(w)
    xy = oracle.lattice(21, w.pupil_diameter)
    q, p, path, _, _ = sysm.trace(xy, np.zeros_like(xy))
    assert np.max(np.abs(q)) < 1e-12 and np.max(np.abs(path - 100.0)) < 1e-12
    inp = gen.make_inputs(w, xy)
    J = np.block([[np.zeros((2, 2)), np.eye(2)], [-np.eye(2), np.zeros((2, 2))]])
    M = inp["abcd"].reshape(-1, 4, 4)
    res = np.max(np.abs(np.einsum("nji,jk,nkl->nil", M, J, M) - J))
    assert res < 2e-5
    c = gen.workloads.c4_chief_intercept(w)
    assert abs(c[0]) < 1e-12 and abs(c[1] - 50.0 * math.tan(math.radians(0.5))) < 2e-4


def test_zernike_terms_orthonormal_and_gradients():
    """Noll Z4..Z11 have unit RMS on the unit disk and are mutually orthogonal; analytic gradient
    matches central differences."""
    rng = np.random.default_rng(1)
    r = np.sqrt(rng.uniform(0, 1, 400000))
    t = rng.uniform(0, 2 * math.pi, r.size)
    x, y = r * np.cos(t), r * np.sin(t)
    Z = np.array(gen.workloads._zern_terms(x, y))
    G = Z @ Z.T / r.size
    assert np.max(np.abs(G - np.eye(8))) < 0.02
    xy = np.stack([x[:50], y[:50]]) * 25.0
    c = gen.workloads.zernike_coefficients(0.5, 7)
    assert abs(math.sqrt(np.sum(c ** 2)) - 0.5) < 1e-15
    h = 1e-5
    g = gen.zernike_opd_grad(xy, 50.0, c, 1e-3)
    for ax in range(2):
        d = np.zeros((2, 1))
        d[ax] = h
        num = (gen.zernike_opd(xy + d, 50.0, c, 1e-3) - gen.zernike_opd(xy - d, 50.0, c, 1e-3)) / (2 * h)
        assert np.max(np.abs(num - g[ax])) < 1e-11


# ----------------------------------------------------------------------------- P7 linearity, shift, cull

def test_linearity_in_weights_and_detector_shift():
    w = gen.workload(0)
    xy = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    det = inp["detector"]
    w0 = oracle.waist(w.overlap_factor, w.pitch)
    rng = np.random.default_rng(5)
    W1 = rng.standard_normal((2, xy.shape[1]))
    W2 = rng.standard_normal((2, xy.shape[1]))

    def fld(W, d=det):
        rec = oracle.propagate(xy, w0, w.wavelength, 1, inp["abcd"], inp["l0"], None, W)
        return oracle.field(oracle.to_detector(rec, d), d, w.wavelength)
    E1, E2, E12 = fld(W1), fld(W2), fld(2.0 * W1 - 0.5 * W2)
    assert np.max(np.abs(E12 - (2.0 * E1 - 0.5 * E2))) < 1e-12 * np.max(np.abs(E12))
    m = 3
    d2 = dict(det, origin=[m * det["du"], -2 * det["dv"], 0.0])
    Es = fld(W1, d2)
    s = np.max(np.abs(E1))
    assert np.max(np.abs(Es[2:, :-m] - E1[:-2, m:])) < 1e-11 * s


def test_cull_threshold_bound():
    """R-14: dropping terms with envelope < tau changes the field by at most sum_j tau |amp_j|,
    and actually drops terms on an out-of-focus plane (C1 optics, plane at z = f/2)."""
    w = gen.workload(1)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    abcd = gen.ideal_lens_abcd(f, -f / 2).reshape(16)
    w0 = oracle.waist(1.5, w.pupil_diameter / 21)
    rec = oracle.propagate(xy, w0, w.wavelength, 1, abcd, f / 2)
    det = dict(n_u=32, n_v=32, du=0.4, dv=0.4, origin=[0, 0, 0], e_u=X3, e_v=Y3)
    rd = oracle.to_detector(rec, det)
    tau = 1e-18
    E0 = oracle.field(rd, det, w.wavelength)
    Ec = oracle.field(rd, det, w.wavelength, cull_tau=tau)
    amp = np.hypot(rd[:, 11], rd[:, 12])
    assert np.max(np.abs(E0 - Ec)) <= tau * amp.sum()
    # the beamlets are ~0.45 mm wide here and the detector spans 12.8 mm: most terms are culled,
    # so a huge tau must change the result while tau = 1e-18 must not (beyond the bound)
    Ebig = oracle.field(rd, det, w.wavelength, cull_tau=0.5)
    assert np.max(np.abs(E0 - Ebig)) > 1e-3 * np.max(np.abs(E0))


# ----------------------------------------------------------------------------- figure of merit

def test_psf_metrics_closed_cases():
    """gbdo_psf_metrics against scipy's J1 written out here: (i) a field that IS the Airy amplitude
    gives zero everywhere; (ii) a constant field gives RMS = sqrt(mean((1-airy)^2)) per zone, with
    zone membership by r/(lambda F#) in [0,5), [5,10), [10,15); (iii) zero at the first dark
    ring x = 3.8317 (textbook)."""
    n, lfn = 96, 0.0025
    h = 2 * 16 * lfn / n
    det = dict(n_u=n, n_v=n, du=h, dv=h, origin=[0, 0, 0], e_u=X3, e_v=Y3)
    u = (np.arange(n) - (n - 1) / 2) * h
    uu, vv = np.meshgrid(u, u, indexing="xy")
    rl = np.hypot(uu, vv) / lfn
    x = math.pi * rl
    amp = np.where(x == 0, 1.0, 2 * j1(x) / np.where(x == 0, 1, x))
    m = oracle.psf_metrics(amp.astype(complex) * (0.3 - 0.4j), det, lfn, 0.3 - 0.4j)
    assert np.all(m[:4] < 1e-15) and m[8] < 1e-15
    m = oracle.psf_metrics(np.ones((n, n), dtype=complex), det, lfn, 2.0)   # I = 1/4 everywhere
    d2 = (0.25 - amp ** 2) ** 2
    zones = [np.ones_like(rl, bool), rl < 5, (rl >= 5) & (rl < 10), (rl >= 10) & (rl < 15)]
    for k, z in enumerate(zones):
        assert m[4 + k] == z.sum()
        assert abs(m[k] - math.sqrt(d2[z].mean())) < 1e-14
    assert abs(m[8] - np.sqrt(d2).max()) < 1e-15
    assert abs(2 * j1(3.8317059702075125) / 3.8317059702075125) < 1e-15


def test_psf_metrics_on_c2_member_and_zone_trend():
    """more beamlets -> lower RMS in every zone (first order)."""
    res = []
    for nn in (11, 31):
        w = gen.workload(2, nn, 1.5)
        w = gen.Workload(**{**w.__dict__, "det_n": 96, "det_halfwidth_lfn": 15.0})
        r = oracle.run_workload(w, gen.make_inputs)
        e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
        res.append(oracle.psf_metrics(r["field"], r["inputs"]["detector"], w.wavelength * w.f_number, e0))
    assert np.all(res[1][:4] < res[0][:4])
    assert res[0][4] == 96 * 96 and res[0][5] > 0 and res[0][6] > 0 and res[0][7] > 0


# ----------------------------------------------------------------------------- a0 differential ray trace

def _spec(mirrors, z_pupil, dir_sign, origin, e_x=X3, e_y=Y3, dq=1e-4, dp=1e-6, p_common=(0.0, 0.0)):
    return dict(mirrors=mirrors, z_pupil=z_pupil, dir_sign=dir_sign, origin=list(origin), e_x=list(e_x),
                e_y=list(e_y), dq=dq, dp=dp, p_common=list(p_common))


def test_trace_conic_focus_property():
    """Pins the conic intersection / normal / reflection / path of gbdo_trace_mirrors, (1+k) terms included:
    a ray through one geometric focus of a conic mirror reflects through (or, for a hyperboloid, away from)
    the other; foci at z' = R/(1 +- e), e = sqrt(-k); the path via the mirror is the same for every ray
    (textbook property of conic sections).  Ellipsoid, hyperboloid (the Table-2 secondary) and sphere."""
    rng = np.random.default_rng(7)
    for R, k in ((800.0, -0.36), (1358.0, -1.49686), (500.0, 0.0)):
        e = math.sqrt(-k)
        f1 = R / (1.0 + e)
        f2 = R / (1.0 - e) if e != 1.0 else None
        n = 40
        p_in = rng.uniform(-0.3, 0.3, (2, n))
        xy = np.zeros((2, n))                       # every ray starts AT the near focus, heading to the mirror
        spec = _spec([dict(curvature=1.0 / R, conic=k, z_vertex=0.0)], z_pupil=f1, dir_sign=-1.0,
                     origin=(0.0, 0.0, f2))
        _, base = oracle.trace_mirrors(xy, spec, p_in)
        assert np.max(np.abs(base[:2])) < 1e-9 * abs(f2), (R, k)     # all rays pass through the far focus
        assert np.ptp(base[4]) < 1e-12 * abs(f2), (R, k)             # |PF1| +- |PF2| = const


def test_trace_paraboloid_stigmatic_and_matches_independent_numpy_trace():
    """Paraboloid: collimated on-axis rays meet at (0,0,f) with equal path z_pupil + f (closed form).
    C4 (off-axis field + Zernike tilts): base rays and finite-difference ABCD against gen's numpy
    ParaboloidSystem, which solves the intersection by a different (direct quadratic) formula."""
    w = gen.workload(4)
    xy = oracle.lattice(21, w.pupil_diameter)
    f = w.focal_length
    spec = _spec([dict(curvature=1.0 / (2 * f), conic=-1.0, z_vertex=0.0)], z_pupil=f, dir_sign=-1.0,
                 origin=(0.0, 0.0, f))
    abcd, base = oracle.trace_mirrors(xy, spec)
    assert np.max(np.abs(base[:2])) < 1e-12 and np.max(np.abs(base[4] - 2 * f)) < 1e-12
    w21 = gen.Workload(**{**w.__dict__, "n_across": 21})
    inp = gen.make_inputs(w21, xy)                               # numpy trace (generator)
    ts = gen.trace_spec(w21, xy)
    abcd2, base2 = oracle.trace_mirrors(xy, ts, ts["p_in"], ts["opl0"])
    assert np.max(np.abs(base2 - inp["base"])) < 1e-12
    assert np.max(np.abs(abcd2 - inp["abcd"])) < 1e-7             # 1e-14 coordinate noise / dp = 1e-6


def test_trace_hst_prescription_reproduces_paper_efl_and_focus():
    """The paper's Table 2 prescription traced on axis: the finite-difference B block is the
    effective focal length of Table 3, 57.6 m, A ~ 0 at the Table-2 focus, the on-axis image
    is far smaller than one lambda F# (Ritchey-Chretien: no spherical aberration), the ABCD is symplectic
    (Eq. 8-12)."""
    gold = json.load(open(os.path.join(GOLD, "paper_table2_table3.json")))
    t2 = gold["table2"]
    assert gen.HST_TABLE2["m1_roc"] == t2["M1"]["roc_m"] * 1e3 and gen.HST_TABLE2["m2_conic"] == t2["M2"]["conic"]
    assert abs(gen.HST_TABLE2["m2_to_focus"] - t2["M2"]["distance_m"] * 1e3) < 1e-9
    w = gen.workload(5)
    assert w.wavelength == gold["table3"]["wavelength_nm"] * 1e-6 and w.pupil_diameter == gold["table3"]["epd_m"] * 1e3
    xy = oracle.lattice(21, w.pupil_diameter)
    spec = gen.trace_spec(w, xy)
    abcd, base = oracle.trace_mirrors(xy, spec)
    M = abcd.reshape(-1, 4, 4)
    efl = gold["table3"]["efl_m"] * 1e3
    assert np.max(np.abs(M[:, 0, 2] / efl - 1)) < 2e-5 and np.max(np.abs(M[:, 1, 3] / (-efl) - 1)) < 2e-5
    assert np.max(np.abs(M[:, :2, :2])) < 1e-4                    # at focus A = 0
    lfn = w.wavelength * w.f_number
    assert np.max(np.hypot(base[0], base[1])) < 0.25 * lfn        # geometric spot << Airy core
    assert np.ptp(base[4]) < 0.1 * w.wavelength                   # equal paths to < lambda/10
    # symplectic in balanced units (q -> q/L, p -> p L keeps dq ^ dp; L^2 ~ |B|/|D| makes the blocks O(1-10))
    J = np.block([[np.zeros((2, 2)), np.eye(2)], [-np.eye(2), np.zeros((2, 2))]])
    T = np.diag([84.0, 84.0, 1 / 84.0, 1 / 84.0])
    Mb = np.linalg.inv(T) @ M @ T
    assert np.max(np.abs(np.einsum("nji,jk,nkl->nil", Mb, J, Mb) - J)) < 1e-5


def test_hst_psf_approaches_airy():
    """GBD of the unobscured HST-like telescope against the Airy pattern (oracle trace ->
    parameters -> field); small version (41 beamlets across, 96 px)."""
    w = gen.Workload(**{**gen.workload(5, 41, 1.7).__dict__, "det_n": 96})
    r = oracle.run_workload(w, gen.make_inputs)
    det = r["inputs"]["detector"]
    e0 = oracle.field_points(r["rec_det"], w.wavelength, 0.0, 0.0)[0]
    m = oracle.psf_metrics(r["field"], det, w.wavelength * w.f_number, e0)
    assert m[0] < 3e-3 and m[8] < 3e-2


# ----------------------------------------------------------------------------- round-2 pins

def test_field_pixels_indexing_against_dirichlet_closed_form():
    """Pins the (iu, iv) plumbing of gbdo_field_pixels and the [n_v][n_u] layout / pixel coordinates of
    gbdo_field_rows on a NON-SQUARE detector (n_u != n_v, du != dv) against the Dirichlet-kernel closed form of
    an unclipped lattice (see test_unclipped_lattice_dirichlet_closed_form), which is neither symmetric under
    u <-> v here (different pitches in x and y) nor under index reversal (off-centre origin)."""
    lam, f, w0 = 0.6328e-3, 100.0, 1.4
    nx, ny, px, py = 7, 5, 2.0, 2.6
    xx, yy = np.meshgrid((np.arange(nx) - (nx - 1) / 2) * px, (np.arange(ny) - (ny - 1) / 2) * py, indexing="xy")
    xy = np.stack([xx.ravel(), yy.ravel()])
    rec = oracle.propagate(xy, w0, lam, 1, gen.ideal_lens_abcd(f).reshape(16), f)
    det = dict(n_u=13, n_v=6, du=0.9e-3, dv=1.7e-3, origin=[2.1e-3, -1.3e-3, 0.0], e_u=X3, e_v=Y3)
    rd = oracle.to_detector(rec, det)
    k = 2 * math.pi / lam
    zr = math.pi * w0 ** 2 / lam
    Q, amp = 1 / f - 1j * zr / f ** 2, 1j * zr / f

    def dirichlet(n, t):
        return np.sin(n * t / 2) / np.sin(t / 2)

    def closed(iu, iv):
        # pixel (iu, iv) sits at origin + (iu-(n_u-1)/2) du e_u + (iv-(n_v-1)/2) dv e_v  (gbd.h / R-12)
        x = det["origin"][0] + (np.asarray(iu) - (det["n_u"] - 1) / 2) * det["du"]
        y = det["origin"][1] + (np.asarray(iv) - (det["n_v"] - 1) / 2) * det["dv"]
        return (amp * np.exp(-2j * math.pi * math.fmod(f, lam) / lam) * np.exp(-0.5j * k * Q * (x * x + y * y))
                * dirichlet(nx, k * px * x / f) * dirichlet(ny, k * py * y / f))
    iu = np.array([0, 12, 3, 7, 12, 0, 5, 11])
    iv = np.array([0, 0, 5, 2, 5, 4, 1, 3])
    ref = closed(iu, iv)
    s = np.max(np.abs(ref))
    assert np.max(np.abs(oracle.field_pixels(rd, det, lam, iu, iv) - ref)) < 1e-11 * s
    # a swapped (iu, iv), a transposed layout or reversed index would miss by O(1):
    assert np.max(np.abs(closed(iv, iu % det["n_v"]) - ref)) > 1e-2 * s
    IU, IV = np.meshgrid(np.arange(det["n_u"]), np.arange(det["n_v"]), indexing="xy")
    full = oracle.field(rd, det, lam)
    assert full.shape == (det["n_v"], det["n_u"])
    assert np.max(np.abs(full - closed(IU, IV))) < 1e-11 * s


def _eikonal_3d(rec_nominal, X):
    """Complex eikonal (phase / k) of ONE parabasal astigmatic Gaussian beamlet at 3-D points X (m,3), built
    from its nominal-plane record WITHOUT any transversal basis: the base ray starts at c3 = (c_x, c_y, 0)
    along k^ = (p_x, p_y, sqrt(1-|p|^2)); H is the unique symmetric 3x3 matrix whose in-plane block is the
    record's curvature M and which annihilates k^ (a wavefront curvature has no component along the ray):
        H = [[M, -M p/p_z], [-(M p)^T/p_z, p^T M p/p_z^2]];
    with w = X - c3, s = k^.w and xi = w - s k^ (3-vector transverse offset),
        psi(X) = opl + s + 1/2 xi^T H (I + s H)^-1 xi
    (free-space propagation of a complex curvature matrix, the 3x3 form of P:176 Eq. 22 with A = I, B = s I,
    C = 0, D = I)."""
    r = rec_nominal
    p = np.array([r[2], r[3]])
    pz = math.sqrt(1.0 - p @ p)
    khat = np.array([p[0], p[1], pz])
    M = np.array([[complex(r[5], r[6]), 0.5 * complex(r[7], r[8])],
                  [0.5 * complex(r[7], r[8]), complex(r[9], r[10])]])
    Mp = M @ p
    H = np.zeros((3, 3), dtype=complex)
    H[:2, :2] = M
    H[:2, 2] = H[2, :2] = -Mp / pz
    H[2, 2] = (p @ Mp) / pz ** 2
    assert np.max(np.abs(H @ khat)) < 1e-12 * np.max(np.abs(H))
    w = np.asarray(X, dtype=float) - np.array([r[0], r[1], 0.0])
    s = w @ khat
    xi = w - s[:, None] * khat[None, :]
    out = np.empty(len(s), dtype=complex)
    for i in range(len(s)):
        Hs = H @ np.linalg.inv(np.eye(3) + s[i] * H)
        out[i] = r[4] + s[i] + 0.5 * xi[i] @ Hs @ xi[i]
    return out


@pytest.mark.parametrize("tilt", ["x5", "y-12", "x20_y8_dz", "x-9_spin"])
def test_tilted_plane_records_are_value_gradient_hessian_of_the_3d_eikonal(tilt):
    """Pin P5(ii) of SURVEY 8c / DESIGN R-T: on the detector plane the re-expanded record is the second-order
    Taylor expansion of the beamlet's 3-D complex eikonal about the base-ray intercept,
        psi(X(u,v)) = opl' + p'.D + 1/2 D^T M' D + O(D^3),  X(u,v) = origin + u e_u + v e_v,  D = (u,v) - c'.
    The 3-D eikonal is written above in coordinate-free 3x3 form (no t1/t2 basis, no P0, no P'); its value,
    gradient and Hessian on the plane are taken by 4th-order central differences.  Pins s, c', opl', p' and M' of
    gbdo_to_detector for tilts about x, about y, both with an axial offset, and with in-plane spin."""
    w = gen.workload(4)
    xy = oracle.lattice(9, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    rec = oracle.propagate(inp["xy"], 0.4, w.wavelength, 0, inp["abcd"], 0.0, inp["base"])
    o = gen.detector_dict(w)["origin"]

    def rot(axis, deg):
        a = math.radians(deg)
        c, s = math.cos(a), math.sin(a)
        return {"x": np.array([[1, 0, 0], [0, c, -s], [0, s, c]]), "y": np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]]),
                "z": np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]])}[axis]
    R, dz = {"x5": (rot("x", 5), 0.0), "y-12": (rot("y", -12), 0.0),
             "x20_y8_dz": (rot("x", 20) @ rot("y", 8), 0.04),
             "x-9_spin": (rot("x", -9) @ rot("z", 33), -0.02)}[tilt]
    det = dict(n_u=4, n_v=4, du=1e-3, dv=1e-3, origin=[o[0], o[1], dz], e_u=list(R[:, 0]), e_v=list(R[:, 1]))
    out = oracle.to_detector(rec, det)
    origin, eu, ev = np.array(det["origin"]), R[:, 0], R[:, 1]
    h = 2.0e-3                                                   # mm; beam radius here is ~0.04 mm
    st = np.array([-2, -1, 0, 1, 2])
    c1 = np.array([1, -8, 0, 8, -1]) / 12.0                       # f'  (4th order)
    c2 = np.array([-1, 16, -30, 16, -1]) / 12.0                   # f'' (4th order)
    worst = np.zeros(5)
    for j in (0, 7, 23, 40, len(rec) - 1):
        cu, cv = out[j, 0], out[j, 1]
        uu, vv = np.meshgrid(cu + st * h, cv + st * h, indexing="ij")
        X = origin[None, :] + uu.reshape(-1, 1) * eu[None, :] + vv.reshape(-1, 1) * ev[None, :]
        psi = _eikonal_3d(rec[j], X).reshape(5, 5)
        # the point (c'_u, c'_v) of the plane lies on the base ray
        wv = origin + cu * eu + cv * ev - np.array([rec[j, 0], rec[j, 1], 0.0])
        kh = np.array([rec[j, 2], rec[j, 3], math.sqrt(1 - rec[j, 2] ** 2 - rec[j, 3] ** 2)])
        worst[0] = max(worst[0], np.linalg.norm(np.cross(wv, kh)))
        worst[1] = max(worst[1], abs(psi[2, 2] - out[j, 4]))                                     # opl' = opl + s
        gu, gv = (c1 @ psi[:, 2]) / h, (c1 @ psi[2, :]) / h
        worst[2] = max(worst[2], abs(gu - out[j, 2]), abs(gv - out[j, 3]))                       # p'
        huu, hvv = (c2 @ psi[:, 2]) / h ** 2, (c2 @ psi[2, :]) / h ** 2
        huv = (c1 @ psi @ c1) / h ** 2
        Mq = np.array([complex(out[j, 5], out[j, 6]), complex(out[j, 7], out[j, 8]), complex(out[j, 9], out[j, 10])])
        scale = np.max(np.abs(Mq))
        worst[3] = max(worst[3], abs(huu - Mq[0]) / scale, abs(2 * huv - Mq[1]) / scale, abs(hvv - Mq[2]) / scale)
        # amplitude: along the ray |amp|^2 scales with 1/|det(I + s M_perp)|, times the obliquity ratio
        # (pinned separately by power below); here the branch-free square: amp'^2 det3(I + sH) cos/cos' = amp^2
        s = wv @ kh
        r = rec[j]
        p = np.array([r[2], r[3]])
        M = np.array([[complex(r[5], r[6]), 0.5 * complex(r[7], r[8])], [0.5 * complex(r[7], r[8]), complex(r[9], r[10])]])
        H = np.zeros((3, 3), dtype=complex)
        H[:2, :2] = M
        H[:2, 2] = H[2, :2] = -(M @ p) / kh[2]
        H[2, 2] = (p @ M @ p) / kh[2] ** 2
        a2 = complex(out[j, 11], out[j, 12]) ** 2 * np.linalg.det(np.eye(3) + s * H) * kh[2] / (kh @ np.cross(eu, ev))
        worst[4] = max(worst[4], abs(a2 / complex(r[11], r[12]) ** 2 - 1))
    assert worst[0] < 1e-13 and worst[1] < 1e-13 and worst[2] < 1e-9 and worst[3] < 1e-7 and worst[4] < 1e-11, worst


@pytest.mark.parametrize("tx,ty,dz", [(20.0, 0.0, 0.0), (0.0, -20.0, 0.0), (12.0, 15.0, 0.3), (-20.0, 7.0, -0.2)])
def test_power_through_tilted_plane_pins_obliquity_factor(tx, ty, dz):
    """The sqrt((k^.n')/(k^.Z)) factor of DESIGN R-T, by an invariant that does not use route B: Eq. 21 normalises
    a beamlet so that Int |E|^2 d(in-plane area) = pi w0^2/2 |W|^2 on whatever plane Eq. 21-22 are applied
    (test_power_invariant_general_abcd; Collins propagation in canonical in-plane coordinates is unitary), so the
    record re-expanded onto a tilted, axially shifted plane must carry the same integral in (u, v).  One oblique
    beamlet (decentred in the pupil of an ideal lens, slightly defocused), tilts about x and y up to 20 degrees;
    checked from the record (closed-form Gaussian integral) and by summing the oracle's field on the tilted
    detector.  Without the factor the integral is off by (k^.Z)/(k^.n') - 1, 1 to 8 % here."""
    lam, f, w0 = 1.0e-3, 100.0, 2.0
    xy = np.array([[14.0], [-9.0]])                      # p = -r/f = (-0.14, 0.09): 9.6 degrees oblique
    W = np.array([[0.6], [-0.8]])
    rec = oracle.propagate(xy, w0, lam, 1, gen.ideal_lens_abcd(f, 0.8).reshape(16), f + 0.8, None, W)
    ax, ay = math.radians(tx), math.radians(ty)
    Rx = np.array([[1, 0, 0], [0, math.cos(ax), -math.sin(ax)], [0, math.sin(ax), math.cos(ax)]])
    Ry = np.array([[math.cos(ay), 0, math.sin(ay)], [0, 1, 0], [-math.sin(ay), 0, math.cos(ay)]])
    R = Rx @ Ry
    det0 = dict(n_u=2, n_v=2, du=1e-3, dv=1e-3, origin=[rec[0, 0], rec[0, 1], dz], e_u=list(R[:, 0]), e_v=list(R[:, 1]))
    r = oracle.to_detector(rec, det0)[0]
    k = 2 * math.pi / lam
    imq = np.array([[r[6], r[8] / 2], [r[8] / 2, r[10]]])
    closed = (r[11] ** 2 + r[12] ** 2) * math.pi / (k * math.sqrt(np.linalg.det(-imq)))
    target = math.pi * w0 ** 2 / 2 * float(W[0, 0] ** 2 + W[1, 0] ** 2)
    assert abs(closed / target - 1) < 1e-12
    kh = np.array([rec[0, 2], rec[0, 3], math.sqrt(1 - rec[0, 2] ** 2 - rec[0, 3] ** 2)])
    assert abs(kh[2] / (kh @ np.cross(R[:, 0], R[:, 1])) - 1) > 0.01           # the factor matters in this geometry
    # grid sum on the tilted detector, centred on the beamlet (r[0], r[1] are its centre in detector coordinates)
    wbeam = math.sqrt(lam / (math.pi * min(-np.linalg.eigvalsh(imq))))
    n = 600
    hpx = 10.0 * wbeam / n
    c3 = np.array(det0["origin"]) + r[0] * R[:, 0] + r[1] * R[:, 1]
    det = dict(n_u=n, n_v=n, du=hpx, dv=hpx, origin=list(c3), e_u=list(R[:, 0]), e_v=list(R[:, 1]))
    E = oracle.field(oracle.to_detector(rec, det), det, lam)
    assert abs(np.sum(np.abs(E) ** 2) * hpx * hpx / target - 1) < 1e-9


def test_large_path_enters_modulo_wavelength_exactly():
    """Reading R-9: the optical path enters only through fmod(OPL, lambda).  With lambda = 2^-10 mm and
    OPL = 1e5 lambda + 2^-12 mm (both exact in fp64) the field of a beamlet must equal the one with OPL = 2^-12 mm
    to rounding of the SMALL phase (1e-15), for per-beamlet paths (abcd_mode 0) and for the shared path l0
    (abcd_mode 1); and the on-axis phase is exp(-i 2 pi 2^-12/2^-10) = -i times the amplitude's phase.  A naive
    k*OPL (argument ~6e5 rad, rounding 1e-10 rad) misses this bar by four orders."""
    lam, f, w0 = 2.0 ** -10, 100.0, 1.5
    big, small = 1.0e5 * lam + 2.0 ** -12, 2.0 ** -12
    assert big - 1.0e5 * lam == small                               # exact inputs
    abcd = gen.ideal_lens_abcd(f).reshape(16)
    xy = np.array([[0.0, 3.0], [0.0, -2.0]])
    u, v = np.array([0.0, 1e-3, -2e-3]), np.array([0.0, 2e-3, 1e-3])
    E = {}
    for tag, opl in (("big", big), ("small", small)):
        base = np.array([[0.0, 0.0], [0.0, 0.0], [0.0, -0.03], [0.0, 0.02], [opl, opl]])
        rec0 = oracle.propagate(xy, w0, lam, 0, np.tile(abcd, (2, 1)), 0.0, base)
        E["m0" + tag] = oracle.field_points(oracle.to_detector(rec0, flat_detector()), lam, u, v)
        rec1 = oracle.propagate(xy, w0, lam, 1, abcd, opl)
        E["m1" + tag] = oracle.field_points(oracle.to_detector(rec1, flat_detector()), lam, u, v)
    for m in ("m0", "m1"):
        assert np.max(np.abs(E[m + "big"] - E[m + "small"])) < 4e-15 * np.max(np.abs(E[m + "small"])), m
    rec = oracle.propagate(xy[:, :1], w0, lam, 0, abcd[None, :], 0.0, np.array([[0.0], [0.0], [0.0], [0.0], [big]]))
    E0 = oracle.field_points(oracle.to_detector(rec, flat_detector()), lam, 0.0, 0.0)[0]
    amp = complex(rec[0, 11], rec[0, 12])
    assert abs(E0 / amp - (-1j)) < 1e-15


def test_trace_takes_the_mirror_sheet_through_the_vertex():
    """Sequential tracing intersects the mirror, not the rest of the quadric (DESIGN R-20): a ray parallel to the
    axis that starts BEYOND the whole surface (z' = 5R; a sphere or ellipsoid is crossed on its far side first)
    must land on the sheet through the vertex, at the standard sag z' = c h^2/(1 + sqrt(1 - (1+k) c^2 h^2))
    (sphere, prolate and oblate ellipsoid, the Table-2 hyperboloid).  The hit point is read off the reflected base
    ray (its line through two evaluation planes must pass through (h, 0, sag)) and off the path length."""
    for R, kc in ((500.0, 0.0), (800.0, -0.36), (1358.0, -1.49686), (600.0, 0.7)):
        c = 1.0 / R
        hgt = np.array([0.0, 40.0, 150.0, 0.3 * R])
        sag = c * hgt ** 2 / (1 + np.sqrt(1 - (1 + kc) * c * c * hgt ** 2))
        xy = np.stack([hgt, np.zeros_like(hgt)])
        zp = 5.0 * R
        hits = []
        for z_eval in (0.25 * R, 0.4 * R):
            spec = _spec([dict(curvature=c, conic=kc, z_vertex=0.0)], z_pupil=zp, dir_sign=-1.0,
                         origin=(0.0, 0.0, z_eval))
            _, base = oracle.trace_mirrors(xy, spec)
            hits.append((base[0].copy(), base[2].copy(), base[4].copy(), z_eval))
        (q1, p1, l1, z1), (q2, p2, l2, z2) = hits
        # reflected line in the x-z plane: x(z) = q1 + (z - z1) * slope, slope from the two planes
        slope = (q2 - q1) / (z2 - z1)
        x_at_sag = q1 + (sag - z1) * slope
        assert np.max(np.abs(x_at_sag - hgt)) < 1e-9 * R, (R, kc)
        # path = (z_pupil - sag) + distance from the hit to the plane z1 along the reflected ray
        pz = np.sqrt(1 - p1 ** 2)
        assert np.max(np.abs(l1 - ((zp - sag) + (z1 - sag) / pz))) < 1e-9 * R, (R, kc)


# ----------------------------------------------------------------------------- point evaluation

def _pointeval_one(abcd, l0, lam, w0, r1m, th1, det, weight=None, opd=0.0):
    xy = np.array(r1m, dtype=float).reshape(2, 1)
    base = np.array([[th1[0]], [th1[1]], [opd]])
    return oracle.field_pointeval(xy, w0, lam, 1, np.asarray(abcd).reshape(16), l0, base, weight, det)


def test_pointeval_equals_plane_evaluation_for_a_beamlet_along_the_axis():
    """P:88-100 steps 2-5 for a beamlet whose base ray is the axis (p = 0): the transversal plane through any
    pixel of an untilted detector IS the evaluation plane (t = 0, P0 = Pd = I), so the point-evaluation field must
    equal the plane-evaluation field (itself pinned by closed forms and quadrature) to rounding -- through focus,
    astigmatic, with a complex weight; and on an axially shifted plane it must equal Eq. 23 with that delta_f
    (pins t and the A' = A + t C, B' = B + t D update)."""
    lam, w0 = 1.0e-3, 0.5
    abcd, l0 = rotated_cyl_system()
    W = np.array([[0.3], [-1.1]])
    det = dict(n_u=7, n_v=5, du=0.021, dv=0.017, origin=[0.004, -0.003, 0.0], e_u=X3, e_v=Y3)
    rec = oracle.propagate(np.zeros((2, 1)), w0, lam, 1, abcd.reshape(16), l0, None, W)
    ref = oracle.field(oracle.to_detector(rec, det), det, lam)
    got = _pointeval_one(abcd, l0, lam, w0, (0.0, 0.0), (0.0, 0.0), det, W)
    assert np.max(np.abs(got - ref)) < 1e-12 * np.max(np.abs(ref))
    f, lam2 = 100.0, 2.0 ** -10                        # f + dz and the path modulo lambda are then exact in fp64
    for dz in (0.625, -0.25):
        det_z = dict(det, origin=[0.0, 0.0, dz], du=0.004, dv=0.003)
        got = _pointeval_one(gen.ideal_lens_abcd(f), f, lam2, 3.0, (0.0, 0.0), (0.0, 0.0), det_z)
        rec = oracle.propagate(np.zeros((2, 1)), 3.0, lam2, 1, gen.ideal_lens_abcd(f, dz).reshape(16), f + dz)
        ref = oracle.field(oracle.to_detector(rec, dict(det_z, origin=[0.0, 0.0, 0.0])), det_z, lam2)
        assert np.max(np.abs(got - ref)) < 1e-12 * np.max(np.abs(ref)), dz


def test_pointeval_oblique_beamlet_against_the_3d_beam_field():
    """One oblique, astigmatic, decentred and tilted beamlet: the point-evaluation value at a 3-D point R is the
    beamlet's parabasal 3-D field there, written independently of the algorithm's steps (no transversal frame, no
    P0 / Pd, no rebuilt ABCD):  E(R) = amp / sqrt(p_z det3(I + s H)) exp(-ik psi(R)),  psi and H from the
    coordinate-free 3x3 form of _eikonal_3d, s = (R - c3).k^, amp = the nominal-plane amplitude of Eq. 21;
    1/sqrt(p_z) is the change from power per unit area of the evaluation plane to per unit area normal to the ray.
    Points on a tilted, axially shifted detector (s up to ~0.1 mm).  Pins steps 2-5 of gbdo_field_pointeval."""
    abcd, l0 = rotated_cyl_system()
    lam, w0 = 1.0e-3, 0.5
    r1m, th1 = (9.0, -6.0), (-8e-2, 5e-2)
    W = np.array([[0.8], [0.5]])
    xy = np.array(r1m).reshape(2, 1)
    base = np.array([[th1[0]], [th1[1]], [2.5e-4]])
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), l0, base, W)[0]
    assert math.hypot(rec[2], rec[3]) > 0.05                        # genuinely oblique
    a = math.radians(11.0)
    R = np.array([[1, 0, 0], [0, math.cos(a), -math.sin(a)], [0, math.sin(a), math.cos(a)]])
    det = dict(n_u=6, n_v=5, du=0.03, dv=0.025, origin=[rec[0] + 0.01, rec[1] - 0.02, 0.05], e_u=list(R[:, 0]),
               e_v=list(R[:, 1]))
    got = oracle.field_pointeval(xy, w0, lam, 1, abcd.reshape(16), l0, base, W, det)
    uu, vv = np.meshgrid((np.arange(6) - 2.5) * 0.03, (np.arange(5) - 2.0) * 0.025, indexing="xy")
    X = (np.array(det["origin"])[None, :] + uu.reshape(-1, 1) * R[:, 0][None, :] + vv.reshape(-1, 1) * R[:, 1][None, :])
    psi = _eikonal_3d(rec, X)
    p = np.array([rec[2], rec[3]])
    pz = math.sqrt(1 - p @ p)
    kh = np.array([p[0], p[1], pz])
    M = np.array([[complex(rec[5], rec[6]), 0.5 * complex(rec[7], rec[8])],
                  [0.5 * complex(rec[7], rec[8]), complex(rec[9], rec[10])]])
    H = np.zeros((3, 3), dtype=complex)
    H[:2, :2] = M
    H[:2, 2] = H[2, :2] = -(M @ p) / pz
    H[2, 2] = (p @ M @ p) / pz ** 2
    s = (X - np.array([rec[0], rec[1], 0.0])) @ kh
    assert 0.02 < np.max(np.abs(s)) < 0.2
    det3 = np.array([np.linalg.det(np.eye(3) + si * H) for si in s])
    k = 2 * math.pi / lam
    ref = complex(rec[11], rec[12]) / np.sqrt(pz * det3) * np.exp(-1j * k * psi)    # |arg det3| small: principal root
    assert np.max(np.abs(np.angle(det3))) < 1.0
    assert np.max(np.abs(got.ravel() - ref)) < 1e-10 * np.max(np.abs(ref))


def test_pointeval_and_plane_evaluation_agree_to_the_obliquity_of_the_beamlets():
    """the two algorithms produce the same PSF up to small differences.  What separates them here is
    known: the normalisation per unit area normal to each ray vs per unit area of the plane, 1/sqrt(p_z) - 1 <=
    |p|^2/4 per beamlet, plus the third-order (parabasal) residual.  C0 (f/3.9: |p| <= 0.127) -> a few 1e-3;
    the paper's f/24 telescope (C5 optics, small version) -> a few 1e-5."""
    w = gen.workload(0)
    r = oracle.run_workload(w, gen.make_inputs)
    inp = r["inputs"]
    Ep = oracle.field_pointeval(inp["xy"], r["w0"], w.wavelength, inp["abcd_mode"], inp["abcd"], inp["l0"],
                                inp["base"], inp["weight"], inp["detector"])
    d0 = np.max(np.abs(Ep - r["field"])) / np.max(np.abs(r["field"]))
    pmax = 0.5 / w.f_number
    assert 1e-4 < d0 < 0.5 * pmax ** 2
    w5 = gen.Workload(**{**gen.workload(5, 21, 1.7).__dict__, "det_n": 48})
    r5 = oracle.run_workload(w5, gen.make_inputs)
    i5 = r5["inputs"]
    Ep5 = oracle.field_pointeval(i5["xy"], r5["w0"], w5.wavelength, 0, i5["abcd"], 0.0, i5["base"], None, i5["detector"])
    d5 = np.max(np.abs(Ep5 - r5["field"])) / np.max(np.abs(r5["field"]))
    assert d5 < 0.5 * (0.5 / w5.f_number) ** 2 + 2e-5, d5


# ----------------------------------------------------------------------------- Hermite-Gaussian beamlets

def collins_quadrature_field(abcd, l0, lam, E1_of, r1m, r2, half, npts=1201):
    """collins_quadrature for an ARBITRARY input field E1_of(dx, dy) given on the offsets from r1m (Eq. 13)."""
    M = np.asarray(abcd, dtype=float).reshape(4, 4)
    A, B, D = M[:2, :2], M[:2, 2:], M[2:, 2:]
    Bi = np.linalg.inv(B)
    S, T = Bi @ A, D @ Bi
    k = 2 * math.pi / lam
    g = np.linspace(-half, half, npts)
    h = g[1] - g[0]
    dx, dy = np.meshgrid(g, g, indexing="xy")
    x1, y1 = dx + r1m[0], dy + r1m[1]
    E1 = E1_of(dx, dy)
    q11 = S[0, 0] * x1 * x1 + (S[0, 1] + S[1, 0]) * x1 * y1 + S[1, 1] * y1 * y1
    K = 1j / (lam * np.sqrt(np.linalg.det(B) + 0j)) * np.exp(-2j * math.pi * math.fmod(l0, lam) / lam)
    out = []
    for x2, y2 in zip(*r2):
        q22 = T[0, 0] * x2 * x2 + (T[0, 1] + T[1, 0]) * x2 * y2 + T[1, 1] * y2 * y2
        bx, by = Bi[0, 0] * x2 + Bi[0, 1] * y2, Bi[1, 0] * x2 + Bi[1, 1] * y2
        out.append(K * np.sum(E1 * np.exp(-0.5j * k * (q22 + q11 - 2 * (x1 * bx + y1 * by)))) * h * h)
    return np.array(out)


def twisted_system():
    """Two cylindrical lens pairs at DIFFERENT orientations with free space between them: A and B are products of
    non-commuting symmetric matrices, so A + B Q1^-1 and its inverse are NOT symmetric (rows != columns)."""
    def free(d):
        m = np.eye(4)
        m[0, 2] = m[1, 3] = d
        return m

    def lens(angle, f1, f2):
        c, s = math.cos(angle), math.sin(angle)
        R = np.array([[c, -s], [s, c]])
        m = np.eye(4)
        m[2:, :2] = -(R @ np.diag([1 / f1, 1 / f2]) @ R.T)
        return m
    return free(30.0) @ lens(1.1, 90.0, 170.0) @ free(20.0) @ lens(0.4, 100.0, 140.0) @ free(5.0), 55.0


def _mode_weights(wts, n=1):
    """(12, n) SoA of the six complex weights w00, w10, w01, w20, w11, w02 (missing ones zero)."""
    w = list(wts) + [0.0] * (6 - len(wts))
    return np.array([[complex(x).real, complex(x).imag] for x in w]).reshape(12, 1).repeat(n, axis=1)


@pytest.mark.parametrize("mode", ["10", "01", "mix", "mix-twisted", "20", "11", "02", "mix2-twisted"])
def test_hermite_gaussian_beamlet_against_collins_quadrature(mode):
    """Hermite-Gaussian beamlets of orders m+n <= 2 through the same phasor.  Brute-force trapezoid quadrature of
    P:82 Eq. 13 with the input field [sum w_mn H_m(sqrt2 x~/w0) H_n(sqrt2 y~/w0)] exp(-|r~|^2/w0^2) exp(-ik th.r~)
    through the astigmatic, non-orthogonal system of test_collins_quadrature_astigmatic_decentred_tilted, decentred
    and tilted: pins gbdo_hg_modes (M1^-1, the 2 sqrt2/w0 scaling, which column multiplies D_x and D_y, Gamma = 2 M1^-1 A
    - I and where its entries enter) and the mode factor of gbdo_field_rows_modes."""
    abcd, l0 = twisted_system() if mode.endswith("twisted") else rotated_cyl_system()
    if mode.endswith("twisted"):
        J = np.block([[np.zeros((2, 2)), np.eye(2)], [-np.eye(2), np.zeros((2, 2))]])
        assert np.max(np.abs(abcd.T @ J @ abcd - J)) < 1e-13 and abs(abcd[0, 1] - abcd[1, 0]) > 1e-3
    lam, w0 = 1.0e-3, 0.5
    r1m, th1 = (1.3, -0.7), (2e-3, -1e-3)
    wts = {"10": (0, 1, 0), "01": (0, 0, 1), "mix": (0.4 - 0.3j, 0.7 + 0.2j, -0.5 + 0.6j),
           "mix-twisted": (0.4 - 0.3j, 0.7 + 0.2j, -0.5 + 0.6j),
           "20": (0, 0, 0, 1, 0, 0), "11": (0, 0, 0, 0, 1, 0), "02": (0, 0, 0, 0, 0, 1),
           "mix2-twisted": (0.4 - 0.3j, 0.7 + 0.2j, -0.5 + 0.6j, 0.3 + 0.1j, -0.2 + 0.5j, 0.6 - 0.4j)}[mode]
    wts = tuple(wts) + (0,) * (6 - len(wts))
    k = 2 * math.pi / lam

    def E1(dx, dy):
        sx, sy = math.sqrt(2) * dx / w0, math.sqrt(2) * dy / w0
        h1x, h1y, h2x, h2y = 2 * sx, 2 * sy, 4 * sx * sx - 2, 4 * sy * sy - 2        # physicists' Hermite polynomials
        poly = wts[0] + wts[1] * h1x + wts[2] * h1y + wts[3] * h2x + wts[4] * h1x * h1y + wts[5] * h2y
        return poly * np.exp(-(dx ** 2 + dy ** 2) / w0 ** 2) * np.exp(-1j * k * (th1[0] * dx + th1[1] * dy))
    xy = np.array(r1m, dtype=float).reshape(2, 1)
    base = np.array([[th1[0]], [th1[1]], [0.0]])
    rec = oracle.propagate(xy, w0, lam, 1, abcd.reshape(16), l0, base)
    modes = oracle.hg_modes(1, w0, lam, 1, abcd.reshape(16), _mode_weights(wts))
    c = rec[0, :2]
    det = dict(n_u=3, n_v=2, du=0.07, dv=0.09, origin=[c[0] + 0.01, c[1] - 0.02, 0.0], e_u=X3, e_v=Y3)
    E = oracle.field_modes(oracle.to_detector(rec, det), modes, det, lam)
    uu, vv = np.meshgrid((np.arange(3) - 1.0) * 0.07 + det["origin"][0], (np.arange(2) - 0.5) * 0.09 + det["origin"][1],
                         indexing="xy")
    ref = collins_quadrature_field(abcd, l0, lam, E1, r1m, (uu.ravel(), vv.ravel()), half=6.4 * w0)
    assert np.max(np.abs(E.ravel() - ref)) < 1e-10 * np.max(np.abs(ref))
    assert np.min(np.abs(ref)) > 1e-3 * np.max(np.abs(ref))          # none of the points sits on a node


def test_hermite_gaussian_at_focus_is_the_textbook_mode():
    """Closed form: an HG10 beam through an ideal lens to its focus stays HG10 (textbook: Hermite-Gaussian modes are
    eigenmodes of the Fourier transform), with waist wf = lambda f/(pi w0) and an extra Gouy factor -i relative to
    the fundamental: E = E_fund(r) * H1(sqrt2 x/wf) * (-i)... the sign convention is fixed by quadrature above; here
    the MODULUS pattern |E| = |E_fund| 2 sqrt2 |x|/wf and the node line x = 0 are pinned."""
    lam, f, w0 = 0.6328e-3, 100.0, 1.7
    wf = lam * f / (math.pi * w0)
    xy = np.zeros((2, 1))
    abcd = gen.ideal_lens_abcd(f).reshape(16)
    rec = oracle.propagate(xy, w0, lam, 1, abcd, f)
    modes = oracle.hg_modes(1, w0, lam, 1, abcd, _mode_weights((0, 1, 0)))
    det = dict(n_u=9, n_v=5, du=0.4 * wf, dv=0.5 * wf, origin=[0.0, 0.0, 0.0], e_u=X3, e_v=Y3)
    E = oracle.field_modes(oracle.to_detector(rec, det), modes, det, lam)
    E0 = oracle.field(oracle.to_detector(rec, det), det, lam)
    x = (np.arange(9) - 4.0) * 0.4 * wf
    ratio = E / E0
    assert np.max(np.abs(np.abs(ratio) - 2 * math.sqrt(2) * np.abs(x)[None, :] / wf)) < 1e-12 * 10
    assert np.max(np.abs(E[:, 4])) < 1e-13 * np.max(np.abs(E))       # node line
    # antisymmetric in x, symmetric in y
    assert np.max(np.abs(E + E[:, ::-1])) < 1e-12 * np.max(np.abs(E))
    assert np.max(np.abs(E - E[::-1, :])) < 1e-12 * np.max(np.abs(E))


def test_first_order_laguerre_gaussian_is_covered_by_complex_mode_weights():
    """P:84 also names Laguerre-Gaussian beams [21]: the first-order modes LG(p=0, l=+-1) are HG10 +- i HG01 (textbook),
    i.e. mode weights (w00, w10, w01) = (0, 1, +-i).  At the focus of a lens the field is the donut
    |E| = |E_fund| 2 sqrt2 r/wf with the phase winding exp(+-i phi): the modulus is rotationally symmetric, vanishes
    on the axis, peaks at r = wf/sqrt2, and the phase of E/E_fund winds as +-phi."""
    lam, f, w0 = 0.6328e-3, 100.0, 1.7
    wf = lam * f / (math.pi * w0)
    abcd = gen.ideal_lens_abcd(f).reshape(16)
    rec = oracle.propagate(np.zeros((2, 1)), w0, lam, 1, abcd, f)
    n = 41
    det = dict(n_u=n, n_v=n, du=0.1 * wf, dv=0.1 * wf, origin=[0.0, 0.0, 0.0], e_u=X3, e_v=Y3)
    rd = oracle.to_detector(rec, det)
    E0 = oracle.field(rd, det, lam)
    u = (np.arange(n) - (n - 1) / 2) * 0.1 * wf
    uu, vv = np.meshgrid(u, u, indexing="xy")
    rr, phi = np.hypot(uu, vv), np.arctan2(vv, uu)
    wind = {}
    for sgn in (+1, -1):
        E = oracle.field_modes(rd, oracle.hg_modes(1, w0, lam, 1, abcd, _mode_weights((0, 1, 1j * sgn))), det, lam)
        ratio = E / E0
        assert np.max(np.abs(np.abs(ratio) - 2 * math.sqrt(2) * rr / wf)) < 1e-11 * 10      # donut modulus
        assert abs(E[n // 2, n // 2]) < 1e-13 * np.max(np.abs(E))                          # dark core
        ring = np.abs(rr - wf / math.sqrt(2)) < 0.06 * wf
        assert np.all(np.abs(E)[ring] > 0.99 * np.max(np.abs(E)))                           # peak radius wf/sqrt2
        m = rr > 0.3 * wf
        # an isotropic system multiplies D_x and D_y by the same complex number, so (w10, w01) = (1, +-i) gives
        # (x +- i y) = r exp(+-i phi): the phase of E/E_fund minus (+-phi) is one constant over the detector
        w = ratio[m] / np.abs(ratio[m]) * np.exp(-1j * sgn * phi[m])
        wind[sgn] = float(np.max(np.abs(w - w[0])))
    assert wind[+1] < 1e-9 and wind[-1] < 1e-9, wind


def test_trace_path_reduced_modulo_lambda_before_rounding():
    """R-24: with a wavelength the tracer returns fmod(OPL, lambda) taken BEFORE the result is rounded to double.
    Pins: (1) exactly representable numbers -- 2^14 of free space, lambda = 2^-11, pupil path 2^-45: the reduced path
    is 2^-45 exactly, whereas the unreduced double output is 2^14 (the 2^-45 is gone), so reducing after the rounding
    would give 0; negative paths keep their sign (fmod); (2) on the two-mirror telescope of Table 2 the reduced
    path agrees with fmod of the rounded full path to within the rounding of the latter (one ulp of 16 m), modulo
    lambda, and lies in [0, lambda)."""
    lam, L, tiny = 2.0 ** -11, 2.0 ** 14, 2.0 ** -45
    xy = np.array([[0.0, 0.25, -0.5], [0.0, -0.125, 0.75]])
    spec = dict(mirrors=[], z_pupil=0.0, dir_sign=1.0, origin=[0.0, 0.0, L], e_x=[1.0, 0.0, 0.0],
                e_y=[0.0, 1.0, 0.0], dq=1e-4, dp=1e-6, p_common=[0.0, 0.0])
    for Lz, opl0, want in ((L, tiny, tiny), (2.0 ** 4, -2.0 ** 5 - tiny, -tiny), (L, 3 * lam / 4, 3 * lam / 4),
                           (L, 0.0, 0.0)):
        spec["origin"] = [0.0, 0.0, Lz]
        o = np.full(3, opl0)
        assert float(o[0]) + 2.0 ** 5 in (2.0 ** 5 + tiny, -tiny, 2.0 ** 5 + 3 * lam / 4, 2.0 ** 5)   # inputs are exact
        _, red = oracle.trace_mirrors(xy, spec, None, o, wavelength=lam)
        _, full = oracle.trace_mirrors(xy, spec, None, o)
        assert np.array_equal(red[4], np.full(3, want)), (opl0, red[4])
        assert np.array_equal(full[4], np.full(3, float(np.float64(Lz) + np.float64(opl0))))
        assert np.array_equal(red[:4], full[:4]) and np.array_equal(red[0], xy[0]) and np.array_equal(red[1], xy[1])
    assert float(np.float64(L) + np.float64(tiny)) == L                  # what reducing after the rounding would see
    w = gen.workload(5)
    xy = oracle.lattice(21, w.pupil_diameter)
    spec = gen.trace_spec(w, xy)
    a_red, red = oracle.trace_mirrors(xy, spec, wavelength=w.wavelength)
    a_full, full = oracle.trace_mirrors(xy, spec)
    assert np.array_equal(a_red, a_full) and np.array_equal(red[:4], full[:4])
    assert np.all(red[4] >= 0.0) and np.all(red[4] < w.wavelength)
    d = np.abs(np.fmod(full[4], w.wavelength) - red[4])
    d = np.minimum(d, np.abs(d - w.wavelength))
    assert np.max(d) <= np.spacing(np.max(full[4])) and np.max(d) > 0.0  # ... and the rounding it avoids is real
