"""The numerical constants of the CUDA field-sum kernels (paper_2404_12454_b200/csrc/gbd_math.cuh), checked on the CPU:
the accuracy DESIGN.md section 6 states for every polynomial is re-derived here from the constants as they stand in
the source (parsed, not imported -- the header is CUDA), in numpy long double.  No GPU, no oracle."""
import math
import os
import re

import numpy as np

HDR = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2404_12454_b200", "csrc",
                   "gbd_math.cuh")
SRC = open(HDR).read() + open(os.path.join(os.path.dirname(HDR), "gbd_common.cuh")).read()
LD = np.longdouble


def _array(name):
    m = re.search(r"static __constant__ double %s\[\d+\] = \{(.*?)\};" % name, SRC, re.S)
    assert m, name
    body = re.sub(r"//[^\n]*", "", m.group(1))
    return [float.fromhex(t) if "0x" in t else float(t) for t in re.findall(r"-?0x[0-9a-fA-F.]+p[+-]?\d+|-?\d+\.\d+(?:e[+-]?\d+)?", body)]


def _define(name):
    m = re.search(r"#define %s\s+\(?([^/\n]*?)\)?\s*(/\*.*)?$" % name, SRC, re.M)
    assert m, name
    return m.group(1).strip()


def _horner(c, x):
    p = LD(c[-1]) * np.ones_like(x)
    for a in c[-2::-1]:
        p = p * x + LD(a)
    return p


def test_polynomial_kernel_constants():
    """accumulate_term: 2^f (degree 9) on |f| <= 1/2 to 1.9e-14 relative; sin(pi/2 h)/h (6 coeff.) and cos(pi/2 h)
    (7 coeff.) in h^2 on |h| <= 1/2 to 6.7e-15 and 2e-16 absolute."""
    f = np.linspace(LD(-0.5), LD(0.5), 20001)
    e = _horner(_array("c_exp2"), f)
    assert float(np.max(np.abs(e / np.exp2(f) - 1))) < 2.0e-14
    h = np.linspace(LD(0), LD(0.5), 10001)
    half_pi = LD(np.pi) / 2 if np.finfo(LD).eps > 1e-17 else LD("1.57079632679489661923132169163975144")
    s = h * _horner(_array("c_sin"), h * h)
    c = _horner(_array("c_cos"), h * h)
    assert float(np.max(np.abs(s - np.sin(half_pi * h)))) < 7e-15
    assert float(np.max(np.abs(c - np.cos(half_pi * h)))) < 3e-16


def test_table_kernel_constants():
    """term_tab: table sizes, magic constants and the three 2-term remainder polynomials.
    a0 b0 (1 + a1 r + a2 r^2) ~ 2^r cos-normalisation split: 2^r to 1.3e-11 on |r| <= 2^-10 (half an exponent-table
    step), b0 (1 + b1 h^2) ~ cos(pi/2 h) to 4.7e-13 and h (t0 + t1 h^2) ~ tan(pi/2 h) to 5e-15 on |h| <= 2^-9 (half a
    phase-table step in quarter turns)."""
    cis_n, exp_n = int(_define("GBD_CIS_N")), int(_define("GBD_EXP_N"))
    assert cis_n == 1024 and exp_n == 512
    assert int(_define("GBD_CIS_COPIES")) * 16 == 128 and int(_define("GBD_EXP_COPIES")) * 8 == 128   # one wavefront
    # magic constants: 1.5 * 2^(52 - b) leaves round(x * 2^b) in the low mantissa word
    assert float(_define("GBD_MAGIC_CIS")) == 1.5 * 2.0 ** (52 - 8) and cis_n == 4 * 2 ** 8          # quarter turns
    assert float(_define("GBD_MAGIC_EXP")) == 1.5 * 2.0 ** (52 - 9) and exp_n == 2 ** 9
    a0b0 = [float(t) for t in re.findall(r"\d+\.\d+", _define("GBD_TAB_A0"))]
    assert len(a0b0) == 2
    a0, b0 = a0b0
    a1, a2, b1, t0, t1 = _array("c_tab")
    r = np.linspace(LD(-2.0) ** -10, LD(2.0) ** -10, 20001)
    err_exp = np.max(np.abs(LD(a0) * (1 + r * (LD(a1) + LD(a2) * r)) / np.exp2(r) - 1))
    assert 1e-12 < float(err_exp) < 1.35e-11
    h = np.linspace(LD(0), LD(2.0) ** -9, 20001)
    half_pi = LD(np.pi) / 2
    err_cos = np.max(np.abs(LD(b0) * (1 + LD(b1) * h * h) - np.cos(half_pi * h)))
    err_tan = np.max(np.abs(h * (LD(t0) + LD(t1) * h * h) - np.tan(half_pi * h)))
    assert float(err_cos) < 4.7e-13 and float(err_tan) < 5e-15
    # the exponent table's own trick: entry k with k << 11 subtracted from its high word must stay a normal number
    # whose exponent field is not borrowed from: a0 b0 2^(k/512) - (k << 11) * 2^-20 * 2^0 ... checked bitwise
    for k in (0, 1, 255, 256, 511):
        v = a0 * b0 * 2.0 ** (k / exp_n)
        hi = np.array([v]).view(np.uint64)[0] >> np.uint64(32)
        assert int(hi) - (k << 11) > (1022 << 20)                  # still a positive high word with exponent >= 1022
        # adding lo << 11 with lo = 512 n + k restores exponent n on top of the entry's own
        for n in (-1000, -1, 0, 7, 100):
            lo = exp_n * n + k
            word = (int(hi) - (k << 11) + (lo << 11)) & 0xFFFFFFFF
            back = np.array([(word << 32) | (int(np.array([v]).view(np.uint64)[0]) & 0xFFFFFFFF)], dtype=np.uint64).view(np.float64)[0]
            assert back == v * 2.0 ** n, (k, n)


def test_folded_table_kernel_constants():
    """accumulate_term_fold (the fast direct kernel): the rounding constants that ride on the quadratics' constant terms,
    the re-expanded 2^r polynomial on the one-sided interval [0, 2^-9), the scaled tan / cos coefficients, and the
    bit-level bookkeeping of index, remainder and exponent bias -- replayed here in numpy on random arguments against
    2^g cis(pi/2 T4) in long double."""
    m = re.search(r"#define GBD_FOLD_MAGIC_T\s+\(([^)]*)\)", SRC)
    magic_t = eval(m.group(1))
    magic_g = float(_define("GBD_FOLD_MAGIC_G"))
    t_limit = float(_define("GBD_FOLD_T_LIMIT"))
    assert magic_t == 1.5 * 2.0 ** 12 + 2.0 ** -9 and magic_g == 1.5 * 2.0 ** 11
    assert 2048.0 - t_limit >= 8.0                       # |T4| <= limit keeps the sum inside [4096, 8192)
    a0f = float(_define("GBD_FOLD_A0"))
    body = re.search(r"static __constant__ double c_fold\[5\] = \{(.*?)\};", SRC, re.S).group(1)
    body = re.sub(r"//[^\n]*", "", body)
    A1, A2, b1, t0, t1 = [eval(t.strip().replace("0x1p", "2.0**")) for t in body.split(",")]
    _, b0 = [float(t) for t in re.findall(r"\d+\.\d+", _define("GBD_TAB_A0"))]
    # (1) the polynomial itself: A0 (1 + A1 r + A2 r^2) = b0 2^r on r in [0, 2^-9), r counted in units of 2^-41
    r = np.linspace(LD(0), LD(2.0) ** 32, 20001)           # the 32-bit remainder word
    p = LD(a0f) / LD(b0) * (1 + r * (LD(A1) + LD(A2) * r))
    err = np.max(np.abs(p / np.exp2(r * LD(2.0) ** -41) - 1))
    assert 1e-12 < float(err) < 1.35e-11
    # (2) replay of the whole evaluation on random (g, T4) in fp64, tables in long double
    rng = np.random.default_rng(5)
    n = 20000
    g = rng.uniform(-1000.0, 1000.0, n)
    t4 = rng.uniform(-t_limit, t_limit, n)
    mq = (t4 + magic_t).astype(np.float64)
    mg = (g + magic_g).astype(np.float64)
    assert np.all((mq >= 4096) & (mq < 8192) & (mg >= 2048) & (mg < 4096))
    bq, bg = mq.view(np.uint64), mg.view(np.uint64)
    hq, lq = (bq >> np.uint64(32)).astype(np.int64), (bq & np.uint64(0xFFFFFFFF)).astype(np.int64)
    hg, lg = (bg >> np.uint64(32)).astype(np.int64), (bg & np.uint64(0xFFFFFFFF)).astype(np.int64)
    m_idx = hq & 1023                                    # phase-table entry: cis(2 pi m / 1024)
    h = (lq ^ 0x80000000) - ((lq ^ 0x80000000) >> 31 << 32)   # (int)(lo ^ 0x80000000)
    k_idx = hg & 511
    # exponent: entry k = a0f 2^(k/512) with (k << 11) + (1024 << 20) taken off its high word, + (hg << 11)
    ent = a0f * np.exp2(k_idx / 512.0)
    eb = ent.view(np.uint64)
    hi = ((eb >> np.uint64(32)).astype(np.int64) - (k_idx << 11) - (1024 << 20) + (hg << 11)) & 0xFFFFFFFF
    T2 = ((hi.astype(np.uint64) << np.uint64(32)) | (eb & np.uint64(0xFFFFFFFF))).view(np.float64)
    rr = lg.astype(np.float64)
    hh = h.astype(np.float64)
    z = hh * hh
    ex = T2 * (1.0 + rr * (A1 + A2 * rr))
    td = hh * (t0 + t1 * z)
    e = ex * (z * b1) + ex
    ang = LD(np.pi) / 2 * m_idx.astype(LD) / 256
    Tx, Ty = np.cos(ang), np.sin(ang)
    re_, im_ = e * (Tx - Ty * td), e * (Ty + Tx * td)
    ref_mag = np.exp2(g.astype(LD))
    ref_ang = LD(np.pi) / 2 * t4.astype(LD)
    err_re = np.abs(re_ - ref_mag * np.cos(ref_ang)) / ref_mag
    err_im = np.abs(im_ - ref_mag * np.sin(ref_ang)) / ref_mag
    # 1.3e-11 (2^r) + 4.7e-13 (cos) + rounding of the sums at 2^-40 quarter turns / 2^-41 log2 units
    assert float(max(err_re.max(), err_im.max())) < 1.5e-11


def test_mixed_table_kernel_constants():
    """accumulate_term_mixed_tab: 2048 half-step entries x 8 copies of float2 = 128 KB; row address and remainder from
    the 32-bit fixed-point turn; first-order rotation.  Replayed in numpy against cis(2 pi T)."""
    n, copies = int(_define("GBD_MIXTAB_N")), int(_define("GBD_MIXTAB_COPIES"))
    assert n == 2048 and copies * 8 == 64                       # one row = 64 bytes, 8 lanes' copies
    assert n * copies * 8 + 2 * 128 * 12 * 8 + 1024 <= 232448    # table + record stages fit one CTA
    m = re.search(r"\(float\)rem \* ([0-9.e+-]+)f", SRC)
    k = float(m.group(1))
    assert abs(k / (2 * math.pi / n / 2.0 ** 32) - 1) < 1e-9
    assert float(_define("GBD_MAGIC_FX_FOLD")) == 1.5 * 2.0 ** 22
    rng = np.random.default_rng(6)
    t4 = rng.uniform(-2.0 ** 20, 2.0 ** 20, 100000)              # quarter turns
    mq = t4 + 1.5 * 2.0 ** 22
    fx = (mq.view(np.uint64) & np.uint64(0xFFFFFFFF)).astype(np.int64)      # turns * 2^32 (mod 1 turn)
    row = ((fx & 0xFFE00000) * 131072) >> 32                     # mad.hi: byte offset of the row, 64 bytes per row
    assert np.all(row % 64 == 0) and row.max() < n * 64
    rem = (fx * 2048 + 0x80000000) & 0xFFFFFFFF
    rem = rem - ((rem >> 31) << 32)                              # as signed 32-bit
    d = rem.astype(np.float32) * np.float32(k)
    ang_tab = (row // 64 + 0.5) * (2 * math.pi / n)
    c, s_ = np.cos(ang_tab).astype(np.float32), np.sin(ang_tab).astype(np.float32)
    re_, im_ = c - s_ * d, s_ + c * d
    true = 2 * math.pi * (np.round(t4 * 2.0 ** 30) / 2.0 ** 32)  # the phase the fixed-point word stands for
    err = np.maximum(np.abs(re_ - np.cos(true)), np.abs(im_ - np.sin(true)))
    assert float(err.max()) < 1.3e-6                             # d^2 / 2 <= (pi / 2048)^2 / 2 = 1.18e-6, + fp32 rounding


def test_table_shared_memory_fits_one_cta():
    """192 KB of tables + the record stages + barriers must fit the 227 KB a CTA can have (232,448 bytes)."""
    tab = 1024 * 8 * 16 + 512 * 16 * 8
    assert tab == 196608
    stages = 2 * 128 * 12 * 8            # field_tab_kernel: two stages of 128 records of 12 doubles
    stages_hg = 2 * 64 * 18 * 8
    assert tab + max(stages, stages_hg) + 1024 <= 232448
