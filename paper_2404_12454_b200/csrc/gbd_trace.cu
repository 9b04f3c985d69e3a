// gbd_trace.cu -- a0: differential ray trace of the beamlets through reflecting conic surfaces and the
// ray-transfer (ABCD) matrix of each beamlet from its 5 parabasal rays ("5 parabasal rays for each
// beamlet", P:98 step 4 "differential ABCD matrix ... using differential ray tracing"; prescription form
// P:324-327 Table 2).
//
// Precision.  The optical path of a many-metre telescope is the largest number of the whole method and the field
// needs it modulo the wavelength: one fp64 ulp of a 16 m path is 4e-8 rad at 551 nm, and a chain of fp64 operations
// on such numbers loses several (round 2 measured 5e-8 in the C5 field, 500 x the bar of the field sum it feeds).
// A compensated sum of the segment lengths alone does not help: a hit point that sits eps * L off the mirror along
// its normal changes the path by twice that, to FIRST order.  So all five rays are traced in double-double
// arithmetic (an unevaluated sum hi + lo of two doubles, ~106 bits: Dekker / Knuth error-free transformations) and
// every output is rounded to double ONCE, at the end -- ray coordinates, direction cosines and path are then the
// correctly rounded values of the exact trace (R-20), and the finite differences (q_k - q_b) / h are taken before
// that rounding.  The trace is a set-up step of microseconds (one warp per ray kind, 32 beamlets per CTA), so the
// ~20 x cost per operation does not show in any timed path.
//
// This file is compiled with -fmad=false: the error-free transformations below rely on every + and * being rounded
// individually (the one fused operation they need is written as __fma_rn).
#include "gbd_common.cuh"

namespace {

struct TraceArgs {
    int n_mirrors;
    double curvature[GBD_MAX_MIRRORS], k1[GBD_MAX_MIRRORS], z_vertex[GBD_MAX_MIRRORS];
    double origin[3], ex[3], ey[3], ez[3];
    double p_common[2];
    double dir_sign, z_pupil, dq, dp;
};

// ---- double-double arithmetic: value = hi + lo, |lo| <= ulp(hi)/2
struct dd { double hi, lo; };

__device__ inline dd two_sum(double a, double b)          // a + b = s + e exactly (Knuth)
{
    const double s = a + b, bb = s - a;
    return { s, (a - (s - bb)) + (b - bb) };
}
__device__ inline dd fast_two_sum(double a, double b)     // the same for |a| >= |b| (Dekker)
{
    const double s = a + b;
    return { s, b - (s - a) };
}
__device__ inline dd two_prod(double a, double b)         // a * b = p + e exactly
{
    const double p = a * b;
    return { p, __fma_rn(a, b, -p) };
}
__device__ inline dd mk(double a) { return { a, 0.0 }; }
__device__ inline dd operator-(dd a) { return { -a.hi, -a.lo }; }
__device__ inline dd operator+(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    const dd t = two_sum(a.lo, b.lo);
    s = fast_two_sum(s.hi, s.lo + t.hi);
    return fast_two_sum(s.hi, s.lo + t.lo);
}
__device__ inline dd operator-(dd a, dd b) { return a + (-b); }
__device__ inline dd operator*(dd a, dd b)
{
    const dd p = two_prod(a.hi, b.hi);
    return fast_two_sum(p.hi, p.lo + (a.hi * b.lo + a.lo * b.hi));
}
__device__ inline dd operator*(dd a, double b)
{
    const dd p = two_prod(a.hi, b);
    return fast_two_sum(p.hi, p.lo + a.lo * b);
}
__device__ inline dd operator/(dd a, dd b)                // long division: three quotient digits
{
    const double q1 = a.hi / b.hi;
    dd r = a - b * q1;
    const double q2 = r.hi / b.hi;
    r = r - b * q2;
    const double q3 = r.hi / b.hi;
    return fast_two_sum(q1, q2) + mk(q3);
}
__device__ inline dd sqrt_dd(dd a)                        // one Newton step on the fp64 root (Karp / Markstein)
{
    if (a.hi <= 0.0) return mk(a.hi == 0.0 ? 0.0 : sqrt(a.hi));
    const double x = 1.0 / sqrt(a.hi), ax = a.hi * x;
    const dd err = a - two_prod(ax, ax);
    return two_sum(ax, err.hi * (x * 0.5));
}
// a modulo m > 0 as fmod defines it (truncated quotient: the sign of a, magnitude below m); |a / m| < 2^53
__device__ inline dd fmod_dd(dd a, double m)
{
    const double q = trunc(a.hi / m);                     // an integer, at most one off the exact quotient digit
    dd r = a - two_prod(q, m);                            // the product is exact; the difference good to ~2^-104 |a|
    const bool neg = a.hi < 0.0;
    if (neg) r = -r;                                      // fold onto [0, m), unfold at the end
    if (r.hi < 0.0) r = r + mk(m);
    else if (r.hi > m || (r.hi == m && r.lo >= 0.0)) r = r - mk(m);
    return neg ? -r : r;
}
__device__ inline dd dot3(const dd *a, const dd *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
__device__ inline dd dot3(const dd *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

struct RayOut { dd qx, qy, px, py, path; };

// Conic c(x^2 + y^2 + (1+k) z'^2) - 2 z' = 0, z' = z - z_vertex.  Two-step intersection: to the vertex
// tangent plane, then the root of A t^2 + 2 B t + C = 0 that vanishes with the sag.
__device__ RayOut trace_one(const TraceArgs &T, double x, double y, double px, double py)
{
    dd P[3] = { mk(x), mk(y), mk(T.z_pupil) };
    const dd pxd = mk(px), pyd = mk(py);
    dd d[3] = { pxd, pyd, sqrt_dd(mk(1.0) - (pxd * pxd + pyd * pyd)) * T.dir_sign };
    dd len = mk(0.0);
    for (int m = 0; m < T.n_mirrors; ++m) {
        const double c = T.curvature[m], k1 = T.k1[m];
        const dd t0 = (mk(T.z_vertex[m]) - P[2]) / d[2];
        const dd x0 = P[0] + t0 * d[0], y0 = P[1] + t0 * d[1];
        const dd A = (d[0] * d[0] + d[1] * d[1] + d[2] * d[2] * k1) * c;
        const dd B = (x0 * d[0] + y0 * d[1]) * c - d[2];
        const dd C = (x0 * x0 + y0 * y0) * c;
        const dd sq = sqrt_dd(B * B - A * C);
        const dd t1 = -C / (B + (B.hi >= 0.0 ? sq : -sq));
        P[0] = x0 + t1 * d[0];
        P[1] = y0 + t1 * d[1];
        const dd zp = t1 * d[2];
        P[2] = mk(T.z_vertex[m]) + zp;
        len = len + (t0 + t1);
        dd nrm[3] = { P[0] * c, P[1] * c, zp * (c * k1) - mk(1.0) };
        const dd nn = sqrt_dd(dot3(nrm, nrm));
        nrm[0] = nrm[0] / nn; nrm[1] = nrm[1] / nn; nrm[2] = nrm[2] / nn;
        const dd dn = dot3(d, nrm) * 2.0;
        d[0] = d[0] - dn * nrm[0]; d[1] = d[1] - dn * nrm[1]; d[2] = d[2] - dn * nrm[2];
    }
    const dd w[3] = { mk(T.origin[0]) - P[0], mk(T.origin[1]) - P[1], mk(T.origin[2]) - P[2] };
    const dd t = dot3(w, T.ez) / dot3(d, T.ez);
    const dd h[3] = { t * d[0] - w[0], t * d[1] - w[1], t * d[2] - w[2] };
    RayOut r;
    r.qx = dot3(h, T.ex); r.qy = dot3(h, T.ey);
    r.px = dot3(d, T.ex); r.py = dot3(d, T.ey);
    r.path = len + t;
    return r;
}

// One CTA = 32 beamlets x 5 rays: warp 0 traces the base rays, warp k = 1..4 the rays displaced in coordinate k - 1
// (warp-uniform control flow); the double-double results meet in shared memory, where warp k takes column k - 1 of
// the ray-transfer matrix and warp 0 writes the base ray.
constexpr int TRACE_BEAMLETS = 32;
__global__ void __launch_bounds__(5 * TRACE_BEAMLETS) trace_kernel(long n, const double *__restrict__ xy,
        long xy_stride, const double *__restrict__ p_in, const double *__restrict__ opl0, const TraceArgs T,
        double lambda, double *__restrict__ abcd, double *__restrict__ base)
{
    __shared__ RayOut sh[TRACE_BEAMLETS];                  // the base rays of this CTA
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long j = (long)blockIdx.x * TRACE_BEAMLETS + lane;
    const bool on = j < n;
    RayOut r = {};
    double h = 1.0;
    if (on) {
        double in[4] = { xy[j], xy[xy_stride + j], p_in ? p_in[j] : T.p_common[0],
                         p_in ? p_in[n + j] : T.p_common[1] };
        if (k > 0) {
            h = k <= 2 ? T.dq : T.dp;
            in[k - 1] += h;                                // the displaced start value is the fp64 sum (R-20)
        }
        r = trace_one(T, in[0], in[1], in[2], in[3]);
        if (k == 0) sh[lane] = r;
    }
    __syncthreads();
    if (!on) return;
    if (k == 0) {
        base[j] = r.qx.hi; base[n + j] = r.qy.hi; base[2 * n + j] = r.px.hi; base[3 * n + j] = r.py.hi;
        // the path leaves the trace already reduced modulo the wavelength (R-24): what a double can hold of a
        // 16 m path is 4e-8 rad coarse, what it holds of the remainder is exact to 1e-19
        base[4 * n + j] = fmod_dd(opl0 ? mk(opl0[j]) + r.path : r.path, lambda).hi;
    } else {
        const RayOut &b = sh[lane];
        const dd hd = mk(h);
        double *m = abcd + 16 * j + (k - 1);
        m[0] = ((r.qx - b.qx) / hd).hi;
        m[4] = ((r.qy - b.qy) / hd).hi;
        m[8] = ((r.px - b.px) / hd).hi;
        m[12] = ((r.py - b.py) / hd).hi;
    }
}

}  // namespace

cudaError_t gbd_launch_trace(long n, const double *d_xy, long xy_stride, const double *d_p_in,
                             const double *d_opl0, const gbd_trace_system &S, double lambda, double *d_abcd,
                             double *d_base, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    TraceArgs T;
    T.n_mirrors = S.n_mirrors;
    for (int m = 0; m < GBD_MAX_MIRRORS; ++m) {
        const bool on = m < S.n_mirrors;
        T.curvature[m] = on ? S.mirrors[m].curvature : 0.0;
        T.k1[m] = on ? 1.0 + S.mirrors[m].conic : 0.0;
        T.z_vertex[m] = on ? S.mirrors[m].z_vertex : 0.0;
    }
    for (int i = 0; i < 3; ++i) { T.origin[i] = S.origin[i]; T.ex[i] = S.e_x[i]; T.ey[i] = S.e_y[i]; }
    T.ez[0] = T.ex[1] * T.ey[2] - T.ex[2] * T.ey[1];
    T.ez[1] = T.ex[2] * T.ey[0] - T.ex[0] * T.ey[2];
    T.ez[2] = T.ex[0] * T.ey[1] - T.ex[1] * T.ey[0];
    T.p_common[0] = S.p_common[0]; T.p_common[1] = S.p_common[1];
    T.dir_sign = S.dir_sign; T.z_pupil = S.z_pupil; T.dq = S.dq; T.dp = S.dp;
    const unsigned blocks = (unsigned)((n + TRACE_BEAMLETS - 1) / TRACE_BEAMLETS);
    trace_kernel<<<blocks, 5 * TRACE_BEAMLETS, 0, st>>>(n, d_xy, xy_stride, d_p_in, d_opl0, T, lambda, d_abcd,
                                                              d_base);
    return cudaGetLastError();
}
