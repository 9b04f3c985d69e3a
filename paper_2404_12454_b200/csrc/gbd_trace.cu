// gbd_trace.cu -- a0: differential ray trace of the beamlets through reflecting conic surfaces and the
// ray-transfer (ABCD) matrix of each beamlet from its 5 parabasal rays ("5 parabasal rays for each
// beamlet", P:98 step 4 "differential ABCD matrix ... using differential ray tracing"; prescription form
// P:324-327 Table 2).  One thread per beamlet traces the base ray and four displaced rays.
//
// This file is compiled with -fmad=false: the ABCD entries are finite differences (q_k - q_b)/h with
// h down to 1e-6, so a last-bit difference in a ray coordinate is amplified a million-fold; with every
// operation individually rounded the result does not depend on the compiler's contraction choices.
#include "gbd_common.cuh"

namespace {

struct TraceArgs {
    int n_mirrors;
    double curvature[GBD_MAX_MIRRORS], k1[GBD_MAX_MIRRORS], z_vertex[GBD_MAX_MIRRORS];
    double origin[3], ex[3], ey[3], ez[3];
    double p_common[2];
    double dir_sign, z_pupil, dq, dp;
};

struct Ray2 { double qx, qy, px, py, path; };

__device__ inline double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// Conic c(x^2 + y^2 + (1+k) z'^2) - 2 z' = 0, z' = z - z_vertex.  Two-step intersection: to the vertex
// tangent plane, then the root of A t^2 + 2 B t + C = 0 that vanishes with the sag.
__device__ Ray2 trace_one(const TraceArgs &T, double x, double y, double px, double py)
{
    double P[3] = { x, y, T.z_pupil };
    double d[3] = { px, py, T.dir_sign * sqrt(1.0 - (px * px + py * py)) };
    double len = 0.0;
    for (int m = 0; m < T.n_mirrors; ++m) {
        const double c = T.curvature[m], k1 = T.k1[m];
        const double t0 = (T.z_vertex[m] - P[2]) / d[2];
        const double x0 = P[0] + t0 * d[0], y0 = P[1] + t0 * d[1];
        const double A = c * (d[0] * d[0] + d[1] * d[1] + k1 * d[2] * d[2]);
        const double B = c * (x0 * d[0] + y0 * d[1]) - d[2];
        const double C = c * (x0 * x0 + y0 * y0);
        const double sq = sqrt(B * B - A * C);
        const double t1 = -C / (B + (B >= 0.0 ? sq : -sq));
        P[0] = x0 + t1 * d[0];
        P[1] = y0 + t1 * d[1];
        const double zp = t1 * d[2];
        P[2] = T.z_vertex[m] + zp;
        len += t0 + t1;
        double n[3] = { c * P[0], c * P[1], c * k1 * zp - 1.0 };
        const double nn = sqrt(dot3(n, n));
        n[0] /= nn; n[1] /= nn; n[2] /= nn;
        const double dn = 2.0 * dot3(d, n);
        d[0] -= dn * n[0]; d[1] -= dn * n[1]; d[2] -= dn * n[2];
    }
    const double w[3] = { T.origin[0] - P[0], T.origin[1] - P[1], T.origin[2] - P[2] };
    const double t = dot3(w, T.ez) / dot3(d, T.ez);
    const double h[3] = { P[0] + t * d[0] - T.origin[0], P[1] + t * d[1] - T.origin[1],
                          P[2] + t * d[2] - T.origin[2] };
    Ray2 r;
    r.qx = dot3(h, T.ex); r.qy = dot3(h, T.ey);
    r.px = dot3(d, T.ex); r.py = dot3(d, T.ey);
    r.path = len + t;
    return r;
}

__global__ void __launch_bounds__(128) trace_kernel(long n, const double *__restrict__ xy, long xy_stride,
        const double *__restrict__ p_in, const double *__restrict__ opl0, const TraceArgs T,
        double *__restrict__ abcd, double *__restrict__ base)
{
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double in0[4] = { xy[j], xy[xy_stride + j], p_in ? p_in[j] : T.p_common[0],
                            p_in ? p_in[n + j] : T.p_common[1] };
    const Ray2 b = trace_one(T, in0[0], in0[1], in0[2], in0[3]);
    double *m = abcd + 16 * j;
#pragma unroll 1
    for (int k = 0; k < 4; ++k) {
        double in[4] = { in0[0], in0[1], in0[2], in0[3] };
        const double h = k < 2 ? T.dq : T.dp;
        in[k] += h;
        const Ray2 r = trace_one(T, in[0], in[1], in[2], in[3]);
        m[0 * 4 + k] = (r.qx - b.qx) / h;
        m[1 * 4 + k] = (r.qy - b.qy) / h;
        m[2 * 4 + k] = (r.px - b.px) / h;
        m[3 * 4 + k] = (r.py - b.py) / h;
    }
    base[j] = b.qx; base[n + j] = b.qy; base[2 * n + j] = b.px; base[3 * n + j] = b.py;
    base[4 * n + j] = (opl0 ? opl0[j] : 0.0) + b.path;
}

}  // namespace

cudaError_t gbd_launch_trace(long n, const double *d_xy, long xy_stride, const double *d_p_in,
                             const double *d_opl0, const gbd_trace_system &S, double *d_abcd, double *d_base,
                             cudaStream_t st)
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
    const unsigned blocks = (unsigned)((n + 127) / 128);
    trace_kernel<<<blocks, 128, 0, st>>>(n, d_xy, xy_stride, d_p_in, d_opl0, T, d_abcd, d_base);
    return cudaGetLastError();
}
