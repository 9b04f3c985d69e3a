// gbd_math.cuh -- hand-rolled 2^g * cis(2 pi T) for the field-sum inner loop (fp64 pipe only).
//
// Why not libdevice exp2()/sincospi(): on sm_100a they carry ~41 FP64-pipe instructions plus ~52
// integer/select instructions per call pair (special-value handling, Payne-Hanek-free but branchy
// range reduction).  The FP64 pipe issues one warp instruction every 2 cycles per SM sub-partition,
// so the kernel saturates it only when the non-FP64 instruction count stays below the FP64 count.
// Here: 28 FP64 + ~14 ALU instructions per term, no branches, no special values (inputs are finite
// by construction).
//
// Polynomials are Remez minimax fits (computed offline in 50-digit arithmetic; max abs errors with the
// rounded coefficients: sin 6.7e-15, cos 1.0e-16, 2^f 1.4e-14 relative) -- four orders of magnitude
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

// acc += 2^g * (cos(pi/2 t4) + i sin(pi/2 t4));   t4 = phase in quarter turns, |t4| < 2^31,
// g = envelope exponent (log2), |g| < 2^31; results below 2^-1000 are flushed towards 2^-1000*[0.7,1.5].
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
    float e = exp2f(g);
    if (CULL) e = (g < g_cut) ? 0.f : e;
    acc_re = fmaf(e, c, acc_re);
    acc_im = fmaf(e, s, acc_im);
}

}  // namespace gbdm
