// gbd_pointeval.cu -- the POINT-evaluation algorithm (section 2.2, steps 1-6) as a comparison
// baseline: the algorithm the paper's plane evaluation replaces.  For every (pixel, beamlet) pair the 5 parabasal
// rays are carried to the transversal plane through the pixel (steps 2-3), the ray-transfer matrix is rebuilt
// there (step 4) and the Gaussian of Eq. 21/22 is evaluated with it (step 5): the complex 2x2 inverse, the two
// eigenvalues and three complex square roots are redone per pair -- "where its time goes".
// Deliberately a straightforward kernel (one thread per pixel, beamlet records broadcast from shared memory): it is
// here to restate the paper's plane / point ratio (Fig. 7) on one B200, not to be fast.
//
// DESIGN.md R-22 (the paper defers the mathematics to its ref. [14], which is not in the container): the parabasal
// rays are the base ray plus the columns of the ABCD, so steps 3-4 act on the differentials.  With the transversal
// frame (t1, t2, k^) of R-T, a ray displaced in-plane by dq and tilted by dp meets the plane normal to k^ at
// distance t with   dq~ = P0 dq + t Pd dp,  dp~ = Pd dp,
//   P0 = [[t1_x, t1_y],[t2_x, t2_y]],  Pd[i][j] = t_i[j] - t_i[z] p_j / p_z,
// hence  A' = P0 A + t Pd C,  B' = P0 B + t Pd D,  C' = Pd C,  D' = Pd D.  The products P0 A ... Pd D do not depend on
// the pixel and are formed once per beamlet (pe_setup_kernel); t, xi and everything after them are per pair.
#include "gbd_common.cuh"
#include "gbd_cplx.cuh"

namespace {

constexpr int PE_REC = 32;          // doubles per beamlet record (256 bytes)
constexpr int PE_KB = 32;           // beamlets per shared-memory stage
constexpr int PE_THREADS = 128;

// record: 0-1 c, 2-4 k^, 5-7 t1, 8-10 t2, 11 opl, 12-15 P0 A, 16-19 P0 B, 20-23 Pd C, 24-27 Pd D, 28-29 W
__global__ void __launch_bounds__(128) pe_setup_kernel(long n, const double *__restrict__ xy, long xy_stride,
        double lambda, int abcd_mode, const double *__restrict__ abcd, double l0_red,
        const double *__restrict__ base, const double *__restrict__ weight, double *__restrict__ rec)
{
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double *m = abcd_mode ? abcd : abcd + 16 * j;
    const double A[4] = { m[0], m[1], m[4], m[5] }, B[4] = { m[2], m[3], m[6], m[7] };
    const double C[4] = { m[8], m[9], m[12], m[13] }, D[4] = { m[10], m[11], m[14], m[15] };
    double cx, cy, px, py, opl;
    if (abcd_mode == 1) {
        const double rx = xy[j], ry = xy[xy_stride + j];
        double tx = 0.0, ty = 0.0, opd = 0.0;
        if (base) { tx = base[j]; ty = base[n + j]; opd = base[2 * n + j]; }
        cx = (A[0] * rx + A[1] * ry) + (B[0] * tx + B[1] * ty);
        cy = (A[2] * rx + A[3] * ry) + (B[2] * tx + B[3] * ty);
        px = (C[0] * rx + C[1] * ry) + (D[0] * tx + D[1] * ty);
        py = (C[2] * rx + C[3] * ry) + (D[2] * tx + D[3] * ty);
        opl = l0_red + (opd + 0.5 * ((px * cx + py * cy) - (tx * rx + ty * ry)));
    } else {
        cx = base[j]; cy = base[n + j]; px = base[2 * n + j]; py = base[3 * n + j];
        opl = fmod(base[4 * n + j], lambda);
    }
    const double pz = sqrt(1.0 - (px * px + py * py));
    // t1 = normalise(Y x k^) = (pz, 0, -px)/|.|,  t2 = k^ x t1
    const double inv_n = 1.0 / sqrt(pz * pz + px * px);
    const double t1[3] = { pz * inv_n, 0.0, -px * inv_n };
    const double t2[3] = { py * t1[2] - pz * t1[1], pz * t1[0] - px * t1[2], px * t1[1] - py * t1[0] };
    const double P0[4] = { t1[0], t1[1], t2[0], t2[1] };
    const double ipz = 1.0 / pz;
    const double Pd[4] = { t1[0] - t1[2] * px * ipz, t1[1] - t1[2] * py * ipz,
                           t2[0] - t2[2] * px * ipz, t2[1] - t2[2] * py * ipz };
    double *r = rec + (long)PE_REC * j;
    r[0] = cx; r[1] = cy; r[2] = px; r[3] = py; r[4] = pz;
    r[5] = t1[0]; r[6] = t1[1]; r[7] = t1[2]; r[8] = t2[0]; r[9] = t2[1]; r[10] = t2[2];
    r[11] = opl;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            r[12 + 2 * a + b] = P0[2 * a] * A[b] + P0[2 * a + 1] * A[2 + b];
            r[16 + 2 * a + b] = P0[2 * a] * B[b] + P0[2 * a + 1] * B[2 + b];
            r[20 + 2 * a + b] = Pd[2 * a] * C[b] + Pd[2 * a + 1] * C[2 + b];
            r[24 + 2 * a + b] = Pd[2 * a] * D[b] + Pd[2 * a + 1] * D[2 + b];
        }
    r[28] = weight ? weight[j] : 1.0;
    r[29] = weight ? weight[n + j] : 0.0;
    r[30] = 0.0; r[31] = 0.0;
}

struct PeArgs {
    long n_b;
    int n_u, n_v, n_split;
    double du, dv, origin[3], eu[3], ev[3];
    double q1_im;          // Q1^-1 = i q1_im I
    double inv_lambda;     // 1/lambda
    double env_scale;      // pi/lambda * log2(e): envelope exponent (log2) per unit Im(xi^T Q xi)
};

// One thread per pixel; blockIdx.y = beamlet split (deterministic partial sums, added by pe_reduce_kernel).
__global__ void __launch_bounds__(PE_THREADS) pe_field_kernel(const double *__restrict__ rec, const PeArgs a,
                                                              double2 *__restrict__ out)
{
    __shared__ __align__(16) double srec[PE_KB * PE_REC];
    const long n_px = (long)a.n_u * a.n_v;
    const long px = (long)blockIdx.x * PE_THREADS + threadIdx.x;
    const bool live = px < n_px;
    const long iv = live ? px / a.n_u : 0;
    const int iu = live ? (int)(px - iv * a.n_u) : 0;
    const double u = ((double)iu - 0.5 * (double)(a.n_u - 1)) * a.du;
    const double v = ((double)iv - 0.5 * (double)(a.n_v - 1)) * a.dv;
    const double R[3] = { a.origin[0] + u * a.eu[0] + v * a.ev[0], a.origin[1] + u * a.eu[1] + v * a.ev[1],
                          a.origin[2] + u * a.eu[2] + v * a.ev[2] };
    // this split's beamlet range
    const long per = (a.n_b + a.n_split - 1) / a.n_split;
    const long j_begin = (long)blockIdx.y * per, j_end = min(a.n_b, j_begin + per);
    double acc_re = 0.0, acc_im = 0.0;
    for (long jb = j_begin; jb < j_end; jb += PE_KB) {
        const int cnt = (int)min((long)PE_KB, j_end - jb);
        __syncthreads();
        for (int i = threadIdx.x; i < cnt * PE_REC; i += PE_THREADS) srec[i] = rec[jb * PE_REC + i];
        __syncthreads();
        if (!live) continue;
#pragma unroll 1
        for (int jj = 0; jj < cnt; ++jj) {
            const double *r = srec + jj * PE_REC;
            // step 2: distance along the ray to the transversal plane through R
            const double w0 = R[0] - r[0], w1 = R[1] - r[1], w2 = R[2];
            const double t = w0 * r[2] + w1 * r[3] + w2 * r[4];
            // step 3: local coordinates of R on that plane
            const double x1 = w0 * r[5] + w1 * r[6] + w2 * r[7];
            const double x2 = w0 * r[8] + w1 * r[9] + w2 * r[10];
            // step 4: ABCD from the pupil to the transversal plane;  step 5: M1 = A' + B' Q1^-1, N1 = C' + D' Q1^-1
            m2 M1, N1;
            M1.a = mk(fma(t, r[20], r[12]), fma(t, r[24], r[16]) * a.q1_im);
            M1.b = mk(fma(t, r[21], r[13]), fma(t, r[25], r[17]) * a.q1_im);
            M1.c = mk(fma(t, r[22], r[14]), fma(t, r[26], r[18]) * a.q1_im);
            M1.d = mk(fma(t, r[23], r[15]), fma(t, r[27], r[19]) * a.q1_im);
            N1.a = mk(r[20], r[24] * a.q1_im); N1.b = mk(r[21], r[25] * a.q1_im);
            N1.c = mk(r[22], r[26] * a.q1_im); N1.d = mk(r[23], r[27] * a.q1_im);
            const m2 Q = mul(N1, inv(M1));                               // P:176 Eq. 22
            const cd amp = mk(r[28], r[29]) / sqrt_det_by_eig(M1);        // P:171 Eq. 21 (branch R-5)
            const cd qs = Q.b + Q.c;
            const double qr = Q.a.re * (x1 * x1) + qs.re * (x1 * x2) + Q.d.re * (x2 * x2);
            const double qi = Q.a.im * (x1 * x1) + qs.im * (x1 * x2) + Q.d.im * (x2 * x2);
            // exp(-ik[opl + t + 1/2 (qr + i qi)]) = 2^(env_scale qi) cis(-2 pi T),  T = (opl + t + qr/2)/lambda
            double T = ((r[11] + t) + 0.5 * qr) * a.inv_lambda;
            T -= rint(T);
            double sn, cs;
            sincospi(-2.0 * T, &sn, &cs);
            const double e = exp2(a.env_scale * qi);
            acc_re = fma(e, amp.re * cs - amp.im * sn, acc_re);
            acc_im = fma(e, amp.re * sn + amp.im * cs, acc_im);
        }
    }
    if (live) out[(size_t)blockIdx.y * n_px + px] = make_double2(acc_re, acc_im);
}

__global__ void __launch_bounds__(256) pe_reduce_kernel(const double2 *__restrict__ part, long n_px, int n_split,
                                                        double2 *__restrict__ out)
{
    const long px = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (px >= n_px) return;
    double re = 0.0, im = 0.0;
    for (int s = 0; s < n_split; ++s) {          // fixed order: reproducible
        const double2 p = part[(size_t)s * n_px + px];
        re += p.x;
        im += p.y;
    }
    out[px] = make_double2(re, im);
}

}  // namespace

int gbd_pointeval_splits(long n_b, long n_px, int sms)
{
    const long tiles = (n_px + PE_THREADS - 1) / PE_THREADS;
    long want = (4L * sms + tiles - 1) / tiles;                 // ~4 CTAs of 128 threads per SM
    const long max_split = (n_b + 4 * PE_KB - 1) / (4 * PE_KB);  // at least 4 stages of beamlets per split
    if (want > max_split) want = max_split;
    if (want < 1) want = 1;
    if (want > 64) want = 64;
    return (int)want;
}

size_t gbd_pointeval_record_bytes(long n_b) { return (size_t)n_b * PE_REC * sizeof(double); }

cudaError_t gbd_launch_pointeval(long n, const double *d_xy, long xy_stride, double w0, double lambda, int abcd_mode,
                                 const double *d_abcd, double l0_red, const double *d_base, const double *d_weight,
                                 const gbd_detector &det, int n_split, double *d_rec, void *d_partial, void *d_field,
                                 int *n_launches, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1)
{
    *n_launches = 0;
    const long n_px = (long)det.n_u * det.n_v;
    pe_setup_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n, d_xy, xy_stride, lambda, abcd_mode, d_abcd,
                                                                 l0_red, d_base, d_weight, d_rec);
    PeArgs a;
    a.n_b = n; a.n_u = det.n_u; a.n_v = det.n_v; a.n_split = n_split; a.du = det.du; a.dv = det.dv;
    for (int i = 0; i < 3; ++i) { a.origin[i] = det.origin[i]; a.eu[i] = det.e_u[i]; a.ev[i] = det.e_v[i]; }
    const double PI = 3.14159265358979323846;
    a.q1_im = -lambda / (PI * w0 * w0);
    a.inv_lambda = 1.0 / lambda;
    a.env_scale = PI / lambda * 1.4426950408889634074;
    const dim3 grid((unsigned)((n_px + PE_THREADS - 1) / PE_THREADS), (unsigned)n_split);
    if (ev0 && ev1) cudaEventRecord(ev0, st);
    pe_field_kernel<<<grid, PE_THREADS, 0, st>>>(d_rec, a, reinterpret_cast<double2 *>(n_split > 1 ? d_partial : d_field));
    if (ev0 && ev1) cudaEventRecord(ev1, st);
    *n_launches = 2;
    if (n_split > 1) {
        pe_reduce_kernel<<<(unsigned)((n_px + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double2 *>(d_partial),
                                                                        n_px, n_split, reinterpret_cast<double2 *>(d_field));
        *n_launches = 3;
    }
    return cudaGetLastError();
}
