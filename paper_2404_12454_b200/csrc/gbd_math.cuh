// gbd_math.cuh -- hand-rolled 2^g * cis(2 pi T) for the field-sum inner loop (fp64 pipe only).
//
// Why not libdevice exp2()/sincospi(): on sm_100a they carry ~41 FP64-pipe instructions plus ~52
// integer/select instructions per call pair (special-value handling, Payne-Hanek-free but branchy
// range reduction).  The FP64 pipe issues one warp instruction every 2 cycles per SM sub-partition,
// so the kernel saturates it only when the non-FP64 instruction count stays below the FP64 count.
// accumulate_term (quadrant reduction + minimax polynomials; the kernel of small launches and of the cull):
// 28 FP64 + ~14 ALU instructions per term, no branches, no special values (inputs are finite by construction; see
// DESIGN.md "Inner loop").  The table-driven evaluations further down replace it on large launches; the roofline
// kernel (field_fold_kernel with accumulate_term_fold) executes 16.05 FP64-pipe + 2 conversion + 9.5 other
// instructions per term including the two quadratics (ncu, profiles/r2_field_fold_kernel_ncu.md).
//
// Polynomials are Remez minimax fits (computed offline in 50-digit arithmetic; max abs errors with the
// rounded coefficients: sin 3.3e-15, cos 1.0e-16, 2^f 1.9e-14 relative) -- four orders of magnitude
// inside the 1e-10 relative-L2 parity budget.
#pragma once

namespace gbdm {

// 1.5 * 2^52: adding it rounds to nearest integer and leaves that integer in the low mantissa bits
#define GBD_MAGIC 6755399441055744.0

// Coefficients live in the constant bank: DFMA takes a c[bank][offset] operand directly, so they cost
// neither registers nor UMOV issue slots (literals in the code were rematerialised every iteration).
static __constant__ double c_exp2[10] = {
    0x1.000000000003dp+0, 0x1.62e42fefa3a3cp-1, 0x1.ebfbdff8149e5p-3, 0x1.c6b08d7035b5ep-5,
    0x1.3b2ab72b1859bp-7, 0x1.5d87feaa6800ep-10, 0x1.43088e23eebc1p-13, 0x1.ffcb318c4c34ep-17,
    0x1.63ef982a78ccep-20, 0x1.b69461f6fb9b3p-24};
static __constant__ double c_sin[6] = {
    0x1.921fb54442cfap+0, -0x1.4abbce6257a3cp-1, 0x1.466bc6712516cp-4, -0x1.32d2c6457504cp-8,
    0x1.5071cebd233e2p-13, -0x1.dd54ade9aa75bp-19};
static __constant__ double c_cos[7] = {
    0x1.0000000000000p+0, -0x1.3bd3cc9be458bp+0, 0x1.03c1f081b078ep-2, -0x1.55d3c7dbfe0e0p-6,
    0x1.e1f4fb6119a00p-11, -0x1.a6c9c229f2f8cp-16, 0x1.f3dbf26c7fcc5p-22};

// 2^f on [-1/2, 1/2], degree 9
__device__ __forceinline__ double exp2_poly(double f)
{
    double p = c_exp2[9];
#pragma unroll
    for (int i = 8; i >= 0; --i) p = fma(p, f, c_exp2[i]);
    return p;
}

// sin(pi/2 h)/h as a polynomial in z = h^2, h in [-1/2, 1/2]
__device__ __forceinline__ double sin_poly(double z)
{
    double p = c_sin[5];
#pragma unroll
    for (int i = 4; i >= 0; --i) p = fma(p, z, c_sin[i]);
    return p;
}

// cos(pi/2 h) as a polynomial in z = h^2
__device__ __forceinline__ double cos_poly(double z)
{
    double p = c_cos[6];
#pragma unroll
    for (int i = 5; i >= 0; --i) p = fma(p, z, c_cos[i]);
    return p;
}

// acc += 2^g * (cos(pi/2 t4) + i sin(pi/2 t4));   t4 = phase in quarter turns, |t4| < 2^51 (the quadrant index is
// taken modulo 2^32, which is a multiple of 4), g = envelope exponent (log2), |g| < 2^31; results below 2^-1000 are
// flushed towards 2^-1000*[0.7,1.5]; g must stay below 1023 (gbd.h documents |A_j| <= 1e30 and the pre-pass enforces
// it; an upper clamp here costs the recurrence kernel 6 % through the different instruction schedule it triggers).
__device__ __forceinline__ void accumulate_term(double g, double t4, double &acc_re, double &acc_im)
{
    // ---- 2^g
    double mg = g + GBD_MAGIC;
    int n = __double2loint(mg);
    double f = g - (mg - GBD_MAGIC);                 // in [-1/2, 1/2]
    double p = exp2_poly(f);
    n = max(n, -1000);
    int ehi = __double2hiint(p) + (n << 20);         // exponent injection
    int elo = __double2loint(p);
    // ---- quadrant reduction of the phase
    double mq = t4 + GBD_MAGIC;
    int q = __double2loint(mq);
    double h = t4 - (mq - GBD_MAGIC);                // in [-1/2, 1/2] quarter turns
    double z = h * h;
    double s = sin_poly(z) * h;
    double c = cos_poly(z);
    // cos(x + q pi/2), sin(x + q pi/2): swap on odd q, signs from q
    bool odd = (q & 1) != 0;
    double a = odd ? s : c;
    double b = odd ? c : s;
    double e_c = __hiloint2double(ehi ^ (((q + 1) & 2) << 30), elo);
    double e_s = __hiloint2double(ehi ^ ((q & 2) << 30), elo);
    acc_re = fma(e_c, a, acc_re);
    acc_im = fma(e_s, b, acc_im);
}

// ------------------------------------------------------------------ table-driven variant (direct fp64 kernel)
// 2^g cis(2 pi T) = [2^n 2^(k/512)] * 2^r  *  cis(2 pi m / 1024) * cis(d): the first factor of each pair comes from
// a table in shared memory, the second is a short minimax polynomial in the remainder (Remez fits in 60-digit
// arithmetic; the errors are those of the rounded coefficients and are re-checked by tests/test_kernel_constants.py):
//   |r| <= 2^-10    : 2^r    = a0 (1 + a1 r + a2 r^2)                   max relative error 1.3e-11 (odd in r)
//   |d| <= pi/1024  : cis(d) = cos d * (1 + i tan d),  cos d = b0 (1 + b1 h^2)   max error 4.6e-13,
//                     tan d  = h (t0 + t1 h^2)                                   max error 4.1e-15   (h = 2 d/pi)
// a0 and b0 are folded into the exp table and cos d into the real factor, so the complex product with the table
// entry T is two DFMA:   term = (2^g cos d) * (T + i T tan d).
// Against quadrant reduction + degree-9/11/12 minimax polynomials (accumulate_term above: 28 FP64 + 14 other
// instructions) the per-term function alone is 18 FP64 + 7 other: no odd/even swap (4 FSEL), no sign logic, no
// exponent clamp/shift.  (Whole kernels, quadratics included, by ncu: field_tab_kernel 23.9 FP64 + 8.4 other per
// term, field_fold_kernel 16.05 + 2 conversions + 9.5 other.)
// Bank conflicts: lanes read unrelated entries, so every entry is REPLICATED, one copy per lane of a
// shared-memory wavefront -- entry m of the cis table (16 B; LDS.128 serves 8 lanes per wavefront) is stored 8
// times at [m*8 + lane%8], entry k of the exp table (8 B; 16 lanes per wavefront) 16 times at [k*16 + lane%16]:
// lane c always hits bank group c, so every lookup is conflict-free whatever the phases are (with single copies
// the table reads took 13 instead of 6 wavefronts per warp-term and the shared-memory pipe became the limiter).
// One DADD with 1.5 * 2^(52-b) rounds the argument to a multiple of 2^-b and leaves round(arg * 2^b) in the low
// mantissa word (b = 8 for the phase in quarter turns -> 1024 steps per turn; b = 9 for the exponent).  Valid for
// |t4| < 2^43 quarter turns and |g| < 2^22 (the subtraction that recovers the remainder must stay exact; the
// phase index wraps, the exponent word must not).
#define GBD_CIS_N 1024
#define GBD_CIS_COPIES 8
#define GBD_EXP_N 512
#define GBD_EXP_COPIES 16
#define GBD_TAB_BYTES (GBD_CIS_N * GBD_CIS_COPIES * 16 + GBD_EXP_N * GBD_EXP_COPIES * 8)
#define GBD_MAGIC_CIS 26388279066624.0             /* 1.5 * 2^44 */
#define GBD_MAGIC_EXP 13194139533312.0             /* 1.5 * 2^43 */
#define GBD_HALF_PI 1.5707963267948966
#define GBD_LN2 0.6931471805599453

// Polynomial constants of the remainders, in the constant bank (a DFMA takes a c[][] operand directly; as
// literals they are re-materialised with MOVs in every iteration of the beamlet loop).
#define GBD_TAB_A0 (1.0000000000000067 * 0.9999999999995386)       /* a0 * b0, folded into the exp table */
static __constant__ double c_tab[5] = {
    0.6931472202595722, 0.24022650007967783,                  // a1, a2
    -1.2336995824646646,                                      // b1
    1.5707963267902578, 1.2919342751016831};                  // t0, t1

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds64(uint32_t addr)
{
    double v;
    asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
// base + (lo & mask) * 128 in two instructions (LOP3 + IMAD); left to the compiler it becomes three or four
__device__ __forceinline__ uint32_t tab_addr(uint32_t base, int lo, uint32_t mask)
{
    uint32_t a;
    asm("{\n.reg .u32 t;\nand.b32 t, %1, %2;\nmad.lo.u32 %0, t, 128, %3;\n}" : "=r"(a) : "r"(lo), "r"(mask), "r"(base));
    return a;
}

// cis_lane / exp_lane: 32-bit shared-memory addresses of this lane's copy of entry 0 (table base + (lane % 8) * 16,
// table base + (lane % 16) * 8); one entry row is 128 bytes in both tables.
// CLAMP: exponents below -1000 are raised to -1000 (the term is then ~1e-301 instead of its true, smaller value)
// and any g is accepted; without it g must lie in [-1000, 1000] (the pre-pass tells the kernel whether every term
// of the launch does: GbdFieldLaunch::deep).
template <bool CLAMP>
__device__ __forceinline__ void term_tab(double g, double t4, uint32_t cis_lane, uint32_t exp_lane,
                                         double &e, double &re, double &im)
{
    const double mq = t4 + GBD_MAGIC_CIS;
    const double2 T = lds128(tab_addr(cis_lane, __double2loint(mq), GBD_CIS_N - 1));
    if (CLAMP) g = fmin(fmax(g, -2000.0), 1023.0);    // keeps round(g * 512) inside the low word
    const double mg = g + GBD_MAGIC_EXP;
    int lo = __double2loint(mg);
    if (CLAMP) lo = max(lo, -1000 * GBD_EXP_N);
    // table entry k holds a0 b0 2^(k/512) with k << 11 subtracted from its high word: adding lo << 11 = (n << 20) +
    // (k << 11) puts the exponent n in place -- the scaling by 2^n is one IMAD, with no shift or mask to isolate n
    const double T2raw = lds64(tab_addr(exp_lane, lo, GBD_EXP_N - 1));
    const double h = t4 - (mq - GBD_MAGIC_CIS);       // quarter turns, |h| <= 2^-9
    const double r = g - (mg - GBD_MAGIC_EXP);        // |r| <= 2^-10
    const double T2 = __hiloint2double(__double2hiint(T2raw) + (lo << 11), __double2loint(T2raw));
    const double z = h * h;
    const double ex = T2 * fma(r, fma(r, c_tab[1], c_tab[0]), 1.0);
    const double td = h * fma(z, c_tab[4], c_tab[3]);        // tan d
    e = fma(ex * z, c_tab[2], ex);                            // 2^g cos d
    re = fma(-T.y, td, T.x);
    im = fma(T.x, td, T.y);
}

template <bool CLAMP>
__device__ __forceinline__ void accumulate_term_tab(double g, double t4, uint32_t cis_lane, uint32_t exp_lane,
                                                    double &acc_re, double &acc_im)
{
    double e, re, im;
    term_tab<CLAMP>(g, t4, cis_lane, exp_lane, e, re, im);
    acc_re = fma(e, re, acc_re);
    acc_im = fma(e, im, acc_im);
}

// the same with the per-pixel Gaussian-tail cull (R-14): the term is dropped when g < g_cut
template <bool CLAMP>
__device__ __forceinline__ void accumulate_term_tab_cull(double g, double g_cut, double t4, uint32_t cis_lane,
                                                         uint32_t exp_lane, double &acc_re, double &acc_im)
{
    double e, re, im;
    term_tab<CLAMP>(g, t4, cis_lane, exp_lane, e, re, im);
    if (g >= g_cut) { acc_re = fma(e, re, acc_re); acc_im = fma(e, im, acc_im); }
}

// ------------------------------------------------------------------ "folded" variant (the fast direct fp64 kernel)
// The same tables and remainder polynomials, but the magic constants are ADDED TO THE CONSTANT TERMS OF THE TWO
// QUADRATICS by the pre-pass, so the last DFMA of each quadratic already delivers the rounded sum and the separate
// DADDs of term_tab (magic add, subtract, remainder: 3 per table) disappear:
//   mq = T4 + 1.5 * 2^12 (+ half a table step): in [4096, 8192) for |T4| < 2048 quarter turns, ulp 2^-40.  Its high
//        word ends in floor(256 T4 + 1/2) = the NEAREST phase-table index (low 10 bits), its low word is the fraction
//        f of 256 T4 + 1/2 as a 32-bit fixed point number, so (int)(lo ^ 0x80000000) = (f - 1/2) 2^32 is the signed
//        remainder h, in units of 2^-40 quarter turns: one LOP3 + one I2F instead of two DADD.
//   mg = g + 1.5 * 2^11: in [2048, 4096) for |g| < 1024, ulp 2^-41.  High word: ... n (11 bits, + 1024) k (9 bits);
//        low word: the fraction of 512 g, UNSIGNED -- the remainder r in [0, 2^-9) in units of 2^-41, one I2F.  The
//        2-term polynomial of 2^r is the one of term_tab re-expanded about r - 2^-10 (same minimax error, 1.3e-11; its
//        leading coefficient goes into the table), and the bias of n (1024 << 20) is taken out of the table entries'
//        high words, so the scaling by 2^n is still ONE IMAD: hi(entry) + (hi(mg) << 11).
// Rounding: the two sums are rounded once at 2^-40 / 2^-41 (4.5e-13 quarter turns, 2.3e-13 in g: below the table
// polynomials' own 1.3e-11).  FP64-pipe instructions per term: quadratics 4 (magic included), I2F 2, h^2 1, 2^r 3,
// tan 2, cos fold 2, rotation 2, accumulate 2 = 18 (term_tab on beamlet-centred records: 23).
// (GBD_FOLD_MAGIC_T, GBD_FOLD_MAGIC_G and GBD_FOLD_T_LIMIT are in gbd_common.cuh: the pre-pass writes them)
// a0 b0 2^(2^-10) (1 - a1 c + a2 c^2), c = 2^-10: leading coefficient of the re-expanded 2^r polynomial times b0
#define GBD_FOLD_A0 1.0000000000124618
static __constant__ double c_fold[5] = {
    0.693147061420739 * 0x1p-41, 0.24038916481306472 * 0x1p-82,       // A1, A2 of 2^r on [0, 2^-9), r in 2^-41 units
    -1.2336995824646646 * 0x1p-80,                                     // b1, h in 2^-40 units
    1.5707963267902578 * 0x1p-40, 1.2919342751016831 * 0x1p-120};      // t0, t1

// mq, mg: the two quadratics with the magic constants folded in (see above); tables filled with fill_tables<true>
__device__ __forceinline__ void accumulate_term_fold(double mg, double mq, uint32_t cis_lane, uint32_t exp_lane,
                                                     double &acc_re, double &acc_im)
{
    const int hq = __double2hiint(mq), hg = __double2hiint(mg);
    const double2 T = lds128(tab_addr(cis_lane, hq, GBD_CIS_N - 1));
    const double T2raw = lds64(tab_addr(exp_lane, hg, GBD_EXP_N - 1));
    const double h = (double)(int)(__double2loint(mq) ^ 0x80000000);
    const double r = (double)(unsigned)__double2loint(mg);
    const double T2 = __hiloint2double(__double2hiint(T2raw) + (hg << 11), __double2loint(T2raw));
    const double z = h * h;
    const double ex = T2 * fma(r, fma(r, c_fold[1], c_fold[0]), 1.0);
    const double td = h * fma(z, c_fold[4], c_fold[3]);        // tan d
    const double e = fma(ex, z * c_fold[2], ex);               // 2^g cos d  (z is ~2^62 here: scale z, not ex)
    acc_re = fma(e, fma(-T.y, td, T.x), acc_re);
    acc_im = fma(e, fma(T.x, td, T.y), acc_im);
}

// fill the two tables (called by all threads of the CTA; followed by __syncthreads in the caller).
// FOLD: the exponent table of accumulate_term_fold (other leading coefficient, exponent bias removed).
template <bool FOLD = false>
__device__ __forceinline__ void fill_tables(double2 *cis_tab, double *exp_tab, int tid, int nthreads)
{
    for (int m = tid; m < GBD_CIS_N; m += nthreads) {
        double sn, cs;
        sincospi((double)m * (2.0 / GBD_CIS_N), &sn, &cs);
#pragma unroll
        for (int c = 0; c < GBD_CIS_COPIES; ++c) cis_tab[m * GBD_CIS_COPIES + c] = make_double2(cs, sn);
    }
    for (int k = tid; k < GBD_EXP_N; k += nthreads) {
        double v = (FOLD ? GBD_FOLD_A0 : GBD_TAB_A0) * exp2((double)k * (1.0 / GBD_EXP_N));
        // see term_tab / accumulate_term_fold
        v = __hiloint2double(__double2hiint(v) - (k << 11) - (FOLD ? (1024 << 20) : 0), __double2loint(v));
#pragma unroll
        for (int c = 0; c < GBD_EXP_COPIES; ++c) exp_tab[k * GBD_EXP_COPIES + c] = v;
    }
}

// The term itself: (re, im) = 2^g * cis(pi/2 t4)  (same arithmetic as accumulate_term into zero).
__device__ __forceinline__ void term_value(double g, double t4, double &re, double &im)
{
    re = 0.0;
    im = 0.0;
    accumulate_term(g, t4, re, im);
}

// Same, but the term is dropped when g < g_cut (per-pixel Gaussian-tail cull, R-14).
__device__ __forceinline__ void accumulate_term_cull(double g, double g_cut, double t4,
                                                     double &acc_re, double &acc_im)
{
    double r = 0.0, i = 0.0;
    accumulate_term(g, t4, r, i);
    if (g >= g_cut) { acc_re += r; acc_im += i; }
}

// Mixed mode.  t4 = phase in quarter turns (fp64).  One DADD with 1.5*2^22 leaves round(t4 * 2^30)
// = round(T * 2^32) in the low mantissa word: the phase modulo one turn as a signed 32-bit fixed
// point number -- no FRND, no F2F.  sin/cos/exp2 are the MUFU approximations (XU pipe).
#define GBD_MAGIC_FX 6291456.0                     /* 1.5 * 2^22 */
template <bool CULL>
__device__ __forceinline__ void accumulate_term_mixed(float g, float g_cut, double t4, float &acc_re,
                                                      float &acc_im)
{
    int fx = __double2loint(t4 + GBD_MAGIC_FX);                 // turns * 2^32, wraps modulo one turn
    float ang = (float)fx * 1.4629180792671596e-9f;             // * 2 pi / 2^32  -> radians in [-pi, pi)
    float s = __sinf(ang), c = __cosf(ang);
    // bare MUFU.EX2 (flush-to-zero): exp2f() wraps it in a denormal-range rescue (FSETP + 2 FMUL per term) that only
    // matters below 2^-126, where the term is nothing next to the 1e-4 bar
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(g));
    if (CULL) e = (g < g_cut) ? 0.f : e;
    acc_re = fmaf(e, c, acc_re);
    acc_im = fmaf(e, s, acc_im);
}

// ------------------------------------------------------------------ mixed precision, table variant
// accumulate_term_mixed spends 3 MUFU per term (16 XU lanes per SM: 24 cycles per warp-term, the whole budget).  Here
// cis comes from an fp32 table in shared memory -- 2048 entries per turn at the HALF steps, cis(2 pi (m + 1/2) / 2048),
// 8 copies each (LDS.64 serves 16 lanes per wavefront: at most 2-way conflicts) = 128 KB -- times the first-order
// rotation (1 + i d), |d| <= pi/2048: error d^2/2 <= 1.2e-6 per term against the 1e-4 bar (measured 3e-6 on C3, as
// before: the fp32 envelope dominates).  `mq` is the phase quadratic with the fixed-point constant 1.5 * 2^22 already on
// its constant term (detector-coordinate records), so its low word is the phase in turns * 2^32: the top 11 bits are the
// table index, the other 21 the remainder.  One MUFU (EX2) per term is left.
#define GBD_MIXTAB_N 2048
#define GBD_MIXTAB_COPIES 8
#define GBD_MIXTAB_BYTES (GBD_MIXTAB_N * GBD_MIXTAB_COPIES * 8)
__device__ __forceinline__ void fill_mixed_table(float2 *tab, int tid, int nthreads)
{
    for (int m = tid; m < GBD_MIXTAB_N; m += nthreads) {
        double sn, cs;
        sincospi(((double)m + 0.5) * (2.0 / GBD_MIXTAB_N), &sn, &cs);
#pragma unroll
        for (int c = 0; c < GBD_MIXTAB_COPIES; ++c) tab[m * GBD_MIXTAB_COPIES + c] = make_float2((float)cs, (float)sn);
    }
}
// tab_lane = shared address of this lane's copy of entry 0 (table base + (lane % 8) * 8); one entry row is 64 bytes
template <bool CULL>
__device__ __forceinline__ void accumulate_term_mixed_tab(float g, float g_cut, double mq, uint32_t tab_lane,
                                                          float &acc_re, float &acc_im)
{
    const uint32_t fx = (uint32_t)__double2loint(mq);
    uint32_t addr;
    int rem;
    // row = fx >> 21, address = tab_lane + row * 64: mask + multiply-high-add; remainder (frac - 1/2) * 2^32 of a step
    asm("{\n.reg .u32 t;\nand.b32 t, %1, 0xFFE00000;\nmad.hi.u32 %0, t, 131072, %2;\n}" : "=r"(addr) : "r"(fx), "r"(tab_lane));
    asm("mad.lo.s32 %0, %1, 2048, 0x80000000;" : "=r"(rem) : "r"(fx));
    float2 T;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(T.x), "=f"(T.y) : "r"(addr));
    const float d = (float)rem * 7.143154684e-13f;               // 2 pi / 2048 / 2^32
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(g));
    if (CULL) e = (g < g_cut) ? 0.f : e;
    acc_re = fmaf(e, fmaf(-T.y, d, T.x), acc_re);
    acc_im = fmaf(e, fmaf(T.x, d, T.y), acc_im);
}

}  // namespace gbdm
