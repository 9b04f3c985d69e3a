// gbd_params.cu -- O(N_b) kernels: lattice (a1), per-beamlet parameters (a2), detector pre-pass (a3).
// "P:n" cites /root/reference/PAPER.md line n; "R-x" a reading in DESIGN.md.
#include "gbd_common.cuh"
#include "gbd_cplx.cuh"

namespace {

// ------------------------------------------------------------------ a1: lattice (R-10)
// Keep (ix, iy) iff x^2 + y^2 <= r2max with x = (ix - half) pitch, every operation individually rounded so that the
// decision does not depend on contraction (and is bit-identical to the oracle's and to the host's
// gbd_lattice_count).  Rounding is monotone, so along a row the predicate is monotone in |ix - half| and symmetric
// about the centre: a row keeps the contiguous columns [first, N-1-first], `first` found by bisection.
// Many CTAs: CTA c owns a contiguous block of rows; every CTA recomputes, cooperatively, the number of points kept
// by the rows before its block (one bisection per row and thread, block-reduced in integers) -- no inter-CTA
// communication, output order (iy slow, ix fast) as before.  N = 201: one launch of 26 CTAs, ~5 us instead of the
// 67 us of the single-CTA scan.
__device__ __forceinline__ bool lattice_keep(int ix, double half, double pitch, double yy, double r2max)
{
    const double x = __dmul_rn((double)ix - half, pitch);
    return __dadd_rn(__dmul_rn(x, x), yy) <= r2max;
}
// number of columns kept by row iy and the first of them
__device__ __forceinline__ int lattice_row(int iy, int n_across, double half, double pitch, double r2max, int *first)
{
    const double y = __dmul_rn((double)iy - half, pitch);
    const double yy = __dmul_rn(y, y);
    const int mid = (n_across + 1) / 2;
    int lo = 0, hi = mid;
    while (lo < hi) {
        const int m = (lo + hi) >> 1;
        if (lattice_keep(m, half, pitch, yy, r2max)) hi = m; else lo = m + 1;
    }
    *first = lo;
    return lo < mid ? n_across - 2 * lo : 0;
}

constexpr int LATTICE_THREADS = 256;
constexpr int LATTICE_ROWS = 8;          // rows per CTA

__device__ __forceinline__ void lattice_body(int n_across, double pitch, double r2max, double *__restrict__ xy,
                                             long capacity, long *count_out, int cta, int n_ctas)
{
    __shared__ long warp_sum[LATTICE_THREADS / 32];
    __shared__ long row_base[LATTICE_ROWS + 1];
    __shared__ int row_first[LATTICE_ROWS], row_count[LATTICE_ROWS];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const double half = 0.5 * (double)(n_across - 1);
    const int rows_per = (n_across + n_ctas - 1) / n_ctas;
    const int r0 = cta * rows_per, r1 = min(n_across, r0 + rows_per);
    const bool last = cta == n_ctas - 1;
    // points kept by the rows before this block (the last CTA also needs the grand total: it counts all rows)
    long mine = 0, all = 0;
    const int upto = last && count_out ? n_across : r0;
    for (int iy = tid; iy < upto; iy += LATTICE_THREADS) {
        int f;
        const int c = lattice_row(iy, n_across, half, pitch, r2max, &f);
        all += c;
        if (iy < r0) mine += c;
    }
    for (int o = 16; o > 0; o >>= 1) {
        mine += __shfl_down_sync(0xffffffffu, mine, o);
        all += __shfl_down_sync(0xffffffffu, all, o);
    }
    if (lane == 0) warp_sum[wid] = mine;
    __syncthreads();
    if (tid == 0) {
        long base = 0;
        for (int w = 0; w < LATTICE_THREADS / 32; ++w) base += warp_sum[w];
        row_base[0] = base;
    }
    __syncthreads();
    if (last && count_out) {                      // grand total, same fixed-order integer sum
        if (lane == 0) warp_sum[wid] = all;
        __syncthreads();
        if (tid == 0) {
            long tot = 0;
            for (int w = 0; w < LATTICE_THREADS / 32; ++w) tot += warp_sum[w];
            *count_out = tot;
        }
    }
    // own rows, LATTICE_ROWS at a time
    for (int rb = r0; rb < r1; rb += LATTICE_ROWS) {
        const int nr = min(LATTICE_ROWS, r1 - rb);
        __syncthreads();
        if (tid < nr) row_count[tid] = lattice_row(rb + tid, n_across, half, pitch, r2max, &row_first[tid]);
        __syncthreads();
        if (tid == 0)
            for (int r = 0; r < nr; ++r) row_base[r + 1] = row_base[r] + row_count[r];
        __syncthreads();
        for (int r = 0; r < nr; ++r) {
            const double y = __dmul_rn((double)(rb + r) - half, pitch);
            const long base = row_base[r];
            const int first = row_first[r];
            for (int k = tid; k < row_count[r]; k += LATTICE_THREADS) {
                const long pos = base + k;
                if (pos < capacity) {
                    xy[pos] = __dmul_rn((double)(first + k) - half, pitch);
                    xy[capacity + pos] = y;
                }
            }
        }
        __syncthreads();
        if (tid == 0) row_base[0] = row_base[nr];
    }
}

__global__ void __launch_bounds__(LATTICE_THREADS) lattice_kernel(int n_across, double pitch, double r2max,
                                                                double *__restrict__ xy, long capacity, long *count_out)
{
    lattice_body(n_across, pitch, r2max, xy, capacity, count_out, blockIdx.x, gridDim.x);
}
// batched sweep: blockIdx.y = run
__global__ void __launch_bounds__(LATTICE_THREADS) lattice_batch_kernel(const GbdRunJob *__restrict__ jobs)
{
    const GbdRunJob jb = jobs[blockIdx.y];
    lattice_body(jb.n_across, jb.pitch, jb.r2max, jb.xy, jb.n, jb.count, blockIdx.x, gridDim.x);
}

// ------------------------------------------------------------------ a2: parameters
__device__ __forceinline__ void propagate_body(long j, long n, const double *__restrict__ xy,
        long xy_stride, double q1_im /* = -lambda/(pi w0^2) */, double lambda, int abcd_mode,
        const double *__restrict__ abcd, double l0_red, const double *__restrict__ base,
        const double *__restrict__ weight, double *__restrict__ rec)
{
    const double *m = abcd_mode ? abcd : abcd + 16 * j;
    double A[4] = { m[0], m[1], m[4], m[5] };
    double B[4] = { m[2], m[3], m[6], m[7] };
    double C[4] = { m[8], m[9], m[12], m[13] };
    double D[4] = { m[10], m[11], m[14], m[15] };
    // Q1^-1 = i*q1_im * I  (R-1);  M1 = A + B Q1^-1,  N1 = C + D Q1^-1
    m2 M1, N1;
    M1.a = mk(A[0], B[0] * q1_im); M1.b = mk(A[1], B[1] * q1_im);
    M1.c = mk(A[2], B[2] * q1_im); M1.d = mk(A[3], B[3] * q1_im);
    N1.a = mk(C[0], D[0] * q1_im); N1.b = mk(C[1], D[1] * q1_im);
    N1.c = mk(C[2], D[2] * q1_im); N1.d = mk(C[3], D[3] * q1_im);
    m2 Q = mul(N1, inv(M1));                                  // P:176 Eq. 22
    cd W = weight ? mk(weight[j], weight[n + j]) : mk(1.0, 0.0);
    cd amp = W / sqrt_det_by_eig(M1);                         // P:171 Eq. 21

    double cx, cy, px, py, opl;
    if (abcd_mode == 1) {
        double rx = xy[j], ry = xy[xy_stride + j];
        double tx = 0.0, ty = 0.0, opd = 0.0;
        if (base) { tx = base[j]; ty = base[n + j]; opd = base[2 * n + j]; }
        cx = (A[0] * rx + A[1] * ry) + (B[0] * tx + B[1] * ty);     // P:318 Eq. 28
        cy = (A[2] * rx + A[3] * ry) + (B[2] * tx + B[3] * ty);
        px = (C[0] * rx + C[1] * ry) + (D[0] * tx + D[1] * ty);     // P:320 Eq. 29
        py = (C[2] * rx + C[3] * ry) + (D[2] * tx + D[3] * ty);
        // small terms are added to the ALREADY reduced axial path (R-9)
        opl = l0_red + (opd + 0.5 * ((px * cx + py * cy) - (tx * rx + ty * ry)));   // P:129 Eq. 17
    } else {
        cx = base[j]; cy = base[n + j]; px = base[2 * n + j]; py = base[3 * n + j];
        opl = fmod(base[4 * n + j], lambda);
    }
    double *r = rec + GBD_NREC * j;
    cd qs = Q.b + Q.c;                                        // R-15: no symmetrisation
    r[0] = cx; r[1] = cy; r[2] = px; r[3] = py; r[4] = opl;
    r[5] = Q.a.re; r[6] = Q.a.im; r[7] = qs.re; r[8] = qs.im; r[9] = Q.d.re; r[10] = Q.d.im;
    r[11] = amp.re; r[12] = amp.im;
}

__global__ void __launch_bounds__(128) propagate_kernel(long n, const double *__restrict__ xy,
        long xy_stride, double q1_im, double lambda, int abcd_mode, const double *__restrict__ abcd, double l0_red,
        const double *__restrict__ base, const double *__restrict__ weight, double *__restrict__ rec)
{
    long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    propagate_body(j, n, xy, xy_stride, q1_im, lambda, abcd_mode, abcd, l0_red, base, weight, rec);
}
// batched sweep: blockIdx.y = run (shared ABCD, unit weights, no per-beamlet tilts)
__global__ void __launch_bounds__(128) propagate_batch_kernel(const GbdRunJob *__restrict__ jobs,
                                                              const double *__restrict__ abcd)
{
    const GbdRunJob jb = jobs[blockIdx.y];
    long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= jb.n) return;
    propagate_body(j, jb.n, jb.xy, jb.n, jb.q1_im, jb.lambda, 1, abcd, jb.l0_red, nullptr, nullptr, jb.params);
}

// ------------------------------------------------------------------ a3: detector pre-pass (R-T)
struct DetArgs {
    double origin[3], eu[3], ev[3], nrm[3];
    int untilted;
    double half_u, half_v;     // half extent of the pixel centres along u and v
    int *deep;                 // see GbdFieldLaunch::deep (NULL: not wanted)
};
__device__ inline double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
__device__ inline void cross3(const double *a, const double *b, double *o)
{
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}

__device__ __forceinline__ void prepass_body(long j, const double *__restrict__ rec, const DetArgs &det,
        double lambda, int precision, int stride, double s2, double s2v, int *__restrict__ gate,
        double *__restrict__ ev, double *__restrict__ ev_abs = nullptr, int abs_stride = GBD_NEVAL)
{
    const double *a = rec + GBD_NREC * j;
    double cu, cv, pu, pv, opl;
    cd qxx, qs, qyy, amp;
    if (det.untilted) {
        cu = a[0] - det.origin[0]; cv = a[1] - det.origin[1];
        pu = a[2]; pv = a[3]; opl = a[4];
        qxx = mk(a[5], a[6]); qs = mk(a[7], a[8]); qyy = mk(a[9], a[10]); amp = mk(a[11], a[12]);
    } else {
        const double X[3] = { 1, 0, 0 }, Y[3] = { 0, 1, 0 };
        double px = a[2], py = a[3];
        double kh[3] = { px, py, sqrt(1.0 - (px * px + py * py)) };
        double t1[3], t2[3];
        cross3(Y, kh, t1);
        double inv_n = 1.0 / sqrt(dot3(t1, t1));
        t1[0] *= inv_n; t1[1] *= inv_n; t1[2] *= inv_n;
        cross3(kh, t1, t2);
        // in-plane curvature -> transverse curvature:  Mperp = P0^-T M P0^-1
        double P0[4] = { dot3(t1, X), dot3(t1, Y), dot3(t2, X), dot3(t2, Y) };
        double dP = 1.0 / (P0[0] * P0[3] - P0[1] * P0[2]);
        double Pi[4] = { P0[3] * dP, -P0[1] * dP, -P0[2] * dP, P0[0] * dP };
        cd hs = 0.5 * mk(a[7], a[8]);
        m2 M; M.a = mk(a[5], a[6]); M.b = hs; M.c = hs; M.d = mk(a[9], a[10]);
        m2 PiM, PiT;
        PiM.a = mk(Pi[0], 0); PiM.b = mk(Pi[1], 0); PiM.c = mk(Pi[2], 0); PiM.d = mk(Pi[3], 0);
        PiT.a = PiM.a; PiT.b = PiM.c; PiT.c = PiM.b; PiT.d = PiM.d;
        m2 Mp = mul(mul(PiT, M), PiM);
        // walk along the base ray to the detector plane
        double w3[3] = { det.origin[0] - a[0], det.origin[1] - a[1], det.origin[2] };
        double cosn = dot3(kh, det.nrm);
        double s = dot3(w3, det.nrm) / cosn;
        double hit[3] = { a[0] + s * kh[0] - det.origin[0], a[1] + s * kh[1] - det.origin[1],
                          s * kh[2] - det.origin[2] };
        m2 G;                                                   // I + s Mperp
        G.a = mk(1.0 + s * Mp.a.re, s * Mp.a.im); G.b = s * Mp.b;
        G.c = s * Mp.c; G.d = mk(1.0 + s * Mp.d.re, s * Mp.d.im);
        m2 Mps = mul(Mp, inv(G));
        amp = (sqrt(cosn / kh[2]) * mk(a[11], a[12])) / sqrt_det_by_eig(G);
        // transverse curvature -> detector in-plane curvature:  M' = P'^T Mperp' P'
        m2 Pd, PdT;
        Pd.a = mk(dot3(t1, det.eu), 0); Pd.b = mk(dot3(t1, det.ev), 0);
        Pd.c = mk(dot3(t2, det.eu), 0); Pd.d = mk(dot3(t2, det.ev), 0);
        PdT.a = Pd.a; PdT.b = Pd.c; PdT.c = Pd.b; PdT.d = Pd.d;
        m2 Md = mul(mul(PdT, Mps), Pd);
        cu = dot3(hit, det.eu); cv = dot3(hit, det.ev);
        pu = dot3(kh, det.eu); pv = dot3(kh, det.ev);
        opl = a[4] + s;
        qxx = Md.a; qs = Md.b + Md.c; qyy = Md.d;
    }
    // scale into phase (quarter turns) and envelope (log2) coefficients
    const double PI = 3.14159265358979323846, LOG2E = 1.4426950408889634074;
    double il = 1.0 / lambda;
    double mag = hypot(amp.re, amp.im);
    double t0, g0;
    if (mag == 0.0) {
        t0 = 0.0;
        g0 = -4096.0;                                                    // zero weight: a vanishing term
    } else if (mag <= 1.0e30) {
        double T = atan2(amp.im, amp.re) / (2.0 * PI) - opl * il;      // turns
        T -= rint(T);
        t0 = 4.0 * T;
        g0 = log2(mag);
    } else {
        // non-finite (or absurdly large: > 1e30, the documented limit that keeps every exponent the kernels inject
        // below 1023) amplitude -- a NaN / Inf weight, a singular A + B Q1^-1: the beamlet must not silently
        // disappear.  A NaN phase makes every pixel it is summed into NaN, as in the oracle.
        t0 = g0 = nan("");
    }
    double ge = PI * il * LOG2E;
    double e[GBD_NEVAL];
    e[0] = cu; e[1] = cv; e[2] = t0;
    e[3] = -4.0 * pu * il; e[4] = -4.0 * pv * il;
    e[5] = -2.0 * qxx.re * il; e[6] = -2.0 * qs.re * il; e[7] = -2.0 * qyy.re * il;
    double *o = ev + (long)stride * j;
    if (precision == 0) {
        e[8] = g0; e[9] = ge * qxx.im; e[10] = ge * qs.im; e[11] = ge * qyy.im;
        if (det.deep && mag == 0.0 && ev_abs) {
            // A zero-weight beamlet (obscured part of the pupil) must not push the whole launch off the fast path: its
            // detector-coordinate record is a constant 2^-1000 (1e-301 of a unit-weight term) with zero phase.  The
            // beamlet-centred record above keeps g0 = -4096, which the clamped twin flushes to the same magnitude.
            double *oa = ev_abs + (long)abs_stride * j;
#pragma unroll
            for (int i = 0; i < GBD_NEVAL; ++i) oa[i] = 0.0;
            oa[0] = GBD_FOLD_MAGIC_T;
            oa[6] = GBD_FOLD_MAGIC_G - 1000.0;
        } else if (det.deep) {
            // Is every envelope exponent of this beamlet on the detector inside [-1000, 1000]?  For a decaying
            // envelope (negative semi-definite quadratic form) the largest value is <= g0 and the smallest is at one
            // of the four corner pixels.  Anything else (growing envelope, NaN) takes the clamped path.
            bool safe = g0 <= 1000.0 && e[9] <= 0.0 && e[11] <= 0.0 && 4.0 * e[9] * e[11] >= e[10] * e[10];
#pragma unroll
            for (int k = 0; k < 4 && safe; ++k) {
                const double du = ((k & 1) ? det.half_u : -det.half_u) - cu;
                const double dv = ((k & 2) ? det.half_v : -det.half_v) - cv;
                const double g = g0 + (e[9] * du * du + e[10] * du * dv + e[11] * dv * dv);
                safe = g >= -1000.0;
            }
            if (ev_abs) {
                // The same two quadratics expanded about the detector centre (GbdFieldLaunch::rec_abs): the fast table
                // loop then needs no Du = u - cu per term.  The expansion (here) and its evaluation (in the kernel)
                // cancel terms as large as `big` against each other, so it is only used when every such term stays
                // below 2040 quarter turns / 4096 log2 units: <= 6 roundings x 2^-53 x 4096 = 2.7e-12, inside the budget of
                // the table evaluation (1.3e-11).  All the paper's focal-plane cases are far inside (C3: 35).
                const double tu = e[3], tv = e[4], tuu = e[5], tuv = e[6], tvv = e[7];
                const double guu = e[9], guv = e[10], gvv = e[11];
                const double U = det.half_u, V = det.half_v;
                double T0 = t0 - tu * cu - tv * cv + tuu * cu * cu + tuv * cu * cv + tvv * cv * cv;
                T0 -= 4.0 * rint(0.25 * T0);                          // whole turns do not matter
                const double Tu = tu - 2.0 * tuu * cu - tuv * cv, Tv = tv - 2.0 * tvv * cv - tuv * cu;
                const double G0 = g0 + guu * cu * cu + guv * cu * cv + gvv * cv * cv;
                const double Gu = -2.0 * guu * cu - guv * cv, Gv = -2.0 * gvv * cv - guv * cu;
                const double big_t = fmax(fabs(t0) + fabs(tu * cu) + fabs(tv * cv) + fabs(tuu) * cu * cu + fabs(tuv * cu * cv) + fabs(tvv) * cv * cv,
                                          4.0 + fabs(Tu) * U + fabs(Tv) * V + fabs(tuu) * U * U + fabs(tuv) * U * V + fabs(tvv) * V * V);
                const double big_g = fmax(fabs(g0) + fabs(guu) * cu * cu + fabs(guv * cu * cv) + fabs(gvv) * cv * cv,
                                          fabs(G0) + fabs(Gu) * U + fabs(Gv) * V + fabs(guu) * U * U + fabs(guv) * U * V + fabs(gvv) * V * V);
                // big_t also bounds |T4| itself, which the folded magic constant needs below 2048 quarter turns
                if (!(big_t <= GBD_FOLD_T_LIMIT && big_g <= 4096.0)) safe = false;        // also catches NaN
                double *oa = ev_abs + (long)abs_stride * j;
                // the rounding constants of accumulate_term_fold ride on the constant terms (gbd_math.cuh)
                oa[0] = T0 + GBD_FOLD_MAGIC_T; oa[1] = Tu; oa[2] = Tv; oa[3] = tuu; oa[4] = tuv; oa[5] = tvv;
                oa[6] = G0 + GBD_FOLD_MAGIC_G; oa[7] = Gu; oa[8] = Gv; oa[9] = guu; oa[10] = guv; oa[11] = gvv;
            }
            if (!safe) *det.deep = 1;
        }
#pragma unroll
        for (int i = 0; i < GBD_NEVAL; ++i) o[i] = e[i];
        if (stride == GBD_NEVAL + 2 || stride == GBD_NEVAL + 4) {
            // recurrence: S = exp of the constant second difference of the log-term along a row,
            // 2 s^2 (ln2 guu + i pi/2 tuu), s = spacing of a thread's pixels (s2 = s^2)
            double sn, cs;
            sincospi(s2 * e[5], &sn, &cs);
            double mag = exp2(2.0 * s2 * e[9]);
            o[12] = mag * cs;
            o[13] = mag * sn;
        }
        if (stride == GBD_NEVAL + 4) {
            // separable evaluation: the same factor along a column, and the gate: any cross term -> general path
            double sn, cs;
            sincospi(s2v * e[7], &sn, &cs);
            double mag = exp2(2.0 * s2v * e[11]);
            o[14] = mag * cs;
            o[15] = mag * sn;
            if (gate && (e[6] != 0.0 || e[10] != 0.0)) *gate = 1;
        }
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) o[i] = e[i];
        float *f = reinterpret_cast<float *>(o + 8);
        f[0] = (float)g0; f[1] = (float)(ge * qxx.im); f[2] = (float)(ge * qs.im);
        f[3] = (float)(ge * qyy.im); f[4] = (float)cu; f[5] = (float)cv; f[6] = 0.f; f[7] = 0.f;
        if (det.deep && ev_abs) {
            // Mixed-precision table kernel (field_mixed_tab_kernel): the PHASE quadratic expanded about the detector
            // centre with the fixed-point rounding constant on its constant term (the envelope stays beamlet-centred,
            // it is evaluated in fp32).  Allowed while every monomial stays below 2^20 quarter turns: the sum then
            // lies in [2^22, 2^23) with ulp 2^-30 (2^-32 of a turn) and the cancellation costs <= 6 x 2^-53 x 2^20
            // quarter turns, far below the fp32 arithmetic that follows.
            const double tu = e[3], tv = e[4], tuu = e[5], tuv = e[6], tvv = e[7];
            const double U = det.half_u, V = det.half_v;
            double T0 = t0 - tu * cu - tv * cv + tuu * cu * cu + tuv * cu * cv + tvv * cv * cv;
            T0 -= 4.0 * rint(0.25 * T0);
            const double Tu = tu - 2.0 * tuu * cu - tuv * cv, Tv = tv - 2.0 * tvv * cv - tuv * cu;
            const double big_t = fmax(fabs(t0) + fabs(tu * cu) + fabs(tv * cv) + fabs(tuu) * cu * cu + fabs(tuv * cu * cv) + fabs(tvv) * cv * cv,
                                      4.0 + fabs(Tu) * U + fabs(Tv) * V + fabs(tuu) * U * U + fabs(tuv) * U * V + fabs(tvv) * V * V);
            if (!(big_t <= 1048576.0)) *det.deep = 1;                       // also catches NaN
            double *oa = ev_abs + (long)abs_stride * j;
            oa[0] = T0 + GBD_MAGIC_FX_FOLD; oa[1] = Tu; oa[2] = Tv; oa[3] = tuu; oa[4] = tuv; oa[5] = tvv;
            oa[6] = 0.0; oa[7] = 0.0;
            float *fa = reinterpret_cast<float *>(oa + 8);
#pragma unroll
            for (int i = 0; i < 8; ++i) fa[i] = f[i];
        }
    }
}

__global__ void __launch_bounds__(128) prepass_kernel(long n, const double *__restrict__ rec,
        DetArgs det, double lambda, int precision, int stride, double s2, double s2v, int *__restrict__ gate,
        double *__restrict__ ev, double *__restrict__ ev_abs)
{
    long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    prepass_body(j, rec, det, lambda, precision, stride, s2, s2v, gate, ev, ev_abs);
}
// batched sweep: blockIdx.y = run; second = write the run's second record array (separable layout)
__global__ void __launch_bounds__(128) prepass_batch_kernel(const GbdRunJob *__restrict__ jobs, DetArgs det,
        int precision, int stride, double s2, double s2v, int *__restrict__ gate, int second)
{
    const GbdRunJob jb = jobs[blockIdx.y];
    long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= jb.n) return;
    // a direct-algorithm sweep (12-double records) also writes the detector-coordinate records into ev2 when given
    prepass_body(j, jb.params, det, jb.lambda, precision, stride, s2, s2v, gate, second ? jb.ev2 : jb.ev,
                 (!second && stride == GBD_NEVAL) ? jb.ev2 : nullptr);
}

// ------------------------------------------------------------------ Hermite-Gaussian beamlets, orders m+n <= 2 (R-23)
// Mode factor of beamlet j on the nominal plane (derived from P:82 Eq. 13 with the Hermite generating function,
// DESIGN.md R-23): with M1 = A + B Q1^-1, alpha_x = (2 sqrt2/w0) row 0 of M1^-1, alpha_y = row 1, Gamma = 2 M1^-1 A - I
// and X = alpha_x.D, Y = alpha_y.D:
//   factor = w00 + w10 X + w01 Y + w20 (X^2 - 2 Gamma_xx) + w11 (X Y - Gamma_xy - Gamma_yx) + w02 (Y^2 - 2 Gamma_yy)
// written out as the complex polynomial a0 + a_x D_x + a_y D_y + a_xx D_x^2 + a_xy D_x D_y + a_yy D_y^2.
__global__ void __launch_bounds__(128) hg_modes_kernel(long n, double c0, double q1_im, int abcd_mode,
        const double *__restrict__ abcd, const double *__restrict__ mw, double *__restrict__ modes)
{
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double *m = abcd_mode ? abcd : abcd + 16 * j;
    m2 M1, Ar;
    M1.a = mk(m[0], m[2] * q1_im); M1.b = mk(m[1], m[3] * q1_im);
    M1.c = mk(m[4], m[6] * q1_im); M1.d = mk(m[5], m[7] * q1_im);
    Ar.a = mk(m[0], 0.0); Ar.b = mk(m[1], 0.0); Ar.c = mk(m[4], 0.0); Ar.d = mk(m[5], 0.0);
    const m2 Mi = inv(M1);
    m2 G = mul(Mi, Ar);
    const cd one = mk(1.0, 0.0);
    G.a = 2.0 * G.a - one; G.b = 2.0 * G.b; G.c = 2.0 * G.c; G.d = 2.0 * G.d - one;
    cd w[6] = { one, mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0), mk(0.0, 0.0) };
    if (mw) {
#pragma unroll
        for (int q = 0; q < 6; ++q) w[q] = mk(mw[(2 * q) * n + j], mw[(2 * q + 1) * n + j]);
    }
    const cd ax0 = c0 * Mi.a, ax1 = c0 * Mi.b, ay0 = c0 * Mi.c, ay1 = c0 * Mi.d;
    cd a[6];
    a[0] = w[0] - 2.0 * (w[3] * G.a) - w[4] * (G.b + G.c) - 2.0 * (w[5] * G.d);
    a[1] = w[1] * ax0 + w[2] * ay0;
    a[2] = w[1] * ax1 + w[2] * ay1;
    a[3] = w[3] * (ax0 * ax0) + w[4] * (ax0 * ay0) + w[5] * (ay0 * ay0);
    a[4] = 2.0 * (w[3] * (ax0 * ax1)) + w[4] * (ax0 * ay1 + ax1 * ay0) + 2.0 * (w[5] * (ay0 * ay1));
    a[5] = w[3] * (ax1 * ax1) + w[4] * (ax1 * ay1) + w[5] * (ay1 * ay1);
    double *o = modes + GBD_NMODE * j;
#pragma unroll
    for (int q = 0; q < 6; ++q) { o[2 * q] = a[q].re; o[2 * q + 1] = a[q].im; }
}

// pre-pass of the mode field sum: the fp64 evaluation record of an UNTILTED detector + the mode factor appended
__global__ void __launch_bounds__(128) prepass_modes_kernel(long n, const double *__restrict__ rec,
        const double *__restrict__ modes, DetArgs det, double lambda, double *__restrict__ ev,
        double *__restrict__ ev_abs)
{
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    prepass_body(j, rec, det, lambda, 0, GBD_NEVAL_HG, 0.0, 0.0, nullptr, ev, ev_abs, GBD_NEVAL_HG);
    double *o = ev + (long)GBD_NEVAL_HG * j + GBD_NEVAL;
#pragma unroll
    for (int i = 0; i < GBD_NMODE; ++i) o[i] = modes[GBD_NMODE * j + i];
    if (ev_abs && det.deep) {
        // the mode factor expanded about the detector centre, for the fast kernel:
        //   a0 + a_u Du + a_v Dv + a_uu Du^2 + a_uv Du Dv + a_vv Dv^2,  Du = u - cu, Dv = v - cv
        //   = A0 + A_u u + A_v v + a_uu u^2 + a_uv u v + a_vv v^2
        // Its monomials cancel against each other, so it is only allowed while their sum stays within 2^10 of the
        // size the factor has in beamlet-centred form on the detector (relative error <= 6 x 2^-53 x 2^10 = 7e-13).
        const double cu = ev[(long)GBD_NEVAL_HG * j], cv = ev[(long)GBD_NEVAL_HG * j + 1];
        const double U = det.half_u, V = det.half_v;
        const double Ru = U + fabs(cu), Rv = V + fabs(cv);          // largest |Du|, |Dv| on the detector
        double *oa = ev_abs + (long)GBD_NEVAL_HG * j + GBD_NEVAL;
        double big_abs = 0.0, big_cen = 0.0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {                               // real and imaginary parts alike
            const double a0 = o[0 + c], au = o[2 + c], av = o[4 + c], auu = o[6 + c], auv = o[8 + c], avv = o[10 + c];
            const double A0 = a0 - au * cu - av * cv + auu * cu * cu + auv * cu * cv + avv * cv * cv;
            const double Au = au - 2.0 * auu * cu - auv * cv, Av = av - 2.0 * avv * cv - auv * cu;
            oa[0 + c] = A0; oa[2 + c] = Au; oa[4 + c] = Av; oa[6 + c] = auu; oa[8 + c] = auv; oa[10 + c] = avv;
            big_abs += fabs(a0) + fabs(au * cu) + fabs(av * cv) + fabs(auu) * cu * cu + fabs(auv * cu * cv) + fabs(avv) * cv * cv +
                       fabs(A0) + fabs(Au) * U + fabs(Av) * V + fabs(auu) * U * U + fabs(auv) * U * V + fabs(avv) * V * V;
            big_cen += fabs(a0) + fabs(au) * Ru + fabs(av) * Rv + fabs(auu) * Ru * Ru + fabs(auv) * Ru * Rv + fabs(avv) * Rv * Rv;
        }
        if (!(big_abs <= 1024.0 * big_cen)) *det.deep = 1;          // also catches NaN
    }
}

}  // namespace

cudaError_t gbd_launch_lattice(int n_across, double pitch, double r2max, double *d_xy, long capacity,
                               long *mapped_count, cudaStream_t st)
{
    // one CTA per LATTICE_ROWS rows, at most two waves of CTAs (every CTA recounts the rows before its block)
    int ctas = (n_across + LATTICE_ROWS - 1) / LATTICE_ROWS;
    if (ctas > 296) ctas = 296;
    lattice_kernel<<<ctas, LATTICE_THREADS, 0, st>>>(n_across, pitch, r2max, d_xy, capacity, mapped_count);
    return cudaGetLastError();
}

cudaError_t gbd_launch_propagate(long n, const double *d_xy, long xy_stride, double w0, double lambda,
                                 int abcd_mode, const double *d_abcd, double l0_red,
                                 const double *d_base, const double *d_weight, double *d_params,
                                 cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    double q1_im = -lambda / (3.14159265358979323846 * w0 * w0);
    unsigned blocks = (unsigned)((n + 127) / 128);
    propagate_kernel<<<blocks, 128, 0, st>>>(n, d_xy, xy_stride, q1_im, lambda, abcd_mode, d_abcd,
                                             l0_red, d_base, d_weight, d_params);
    return cudaGetLastError();
}

static DetArgs det_args(const gbd_detector &det)
{
    DetArgs a;
    for (int i = 0; i < 3; ++i) { a.origin[i] = det.origin[i]; a.eu[i] = det.e_u[i]; a.ev[i] = det.e_v[i]; }
    a.nrm[0] = a.eu[1] * a.ev[2] - a.eu[2] * a.ev[1];
    a.nrm[1] = a.eu[2] * a.ev[0] - a.eu[0] * a.ev[2];
    a.nrm[2] = a.eu[0] * a.ev[1] - a.eu[1] * a.ev[0];
    a.half_u = 0.5 * (det.n_u - 1) * det.du;
    a.half_v = 0.5 * (det.n_v - 1) * det.dv;
    a.deep = nullptr;
    a.untilted = det.e_u[0] == 1.0 && det.e_u[1] == 0.0 && det.e_u[2] == 0.0 && det.e_v[0] == 0.0 &&
                 det.e_v[1] == 1.0 && det.e_v[2] == 0.0 && det.origin[2] == 0.0;
    return a;
}

cudaError_t gbd_launch_prepass(long n, const double *d_params, const gbd_detector &det, double lambda,
                               int precision, int algo, double *d_eval, int *d_gate, cudaStream_t st, int *d_deep,
                               double *d_eval_abs)
{
    if (n == 0) return cudaSuccess;
    DetArgs a = det_args(det);
    a.deep = d_deep;
    unsigned blocks = (unsigned)((n + 127) / 128);
    const int stride = algo == GBD_ALGO_SEPARABLE ? GBD_NEVAL + 4 : algo == GBD_ALGO_RECURRENCE ? GBD_NEVAL + 2 : GBD_NEVAL;
    const double sp = det.du;            // recurrence step: one pixel pitch
    prepass_kernel<<<blocks, 128, 0, st>>>(n, d_params, a, lambda, precision, stride, sp * sp, det.dv * det.dv, d_gate,
                                           d_eval, stride == GBD_NEVAL ? d_eval_abs : nullptr);
    return cudaGetLastError();
}

cudaError_t gbd_launch_hg_modes(long n, double w0, double lambda, int abcd_mode, const double *d_abcd,
                                const double *d_mode_weight, double *d_modes, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const double q1_im = -lambda / (3.14159265358979323846 * w0 * w0);
    hg_modes_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n, 2.0 * sqrt(2.0) / w0, q1_im, abcd_mode, d_abcd,
                                                                 d_mode_weight, d_modes);
    return cudaGetLastError();
}

cudaError_t gbd_launch_prepass_modes(long n, const double *d_params, const double *d_modes, const gbd_detector &det,
                                     double lambda, double *d_eval, cudaStream_t st, int *d_deep, double *d_eval_abs)
{
    if (n == 0) return cudaSuccess;
    DetArgs a = det_args(det);
    a.deep = d_deep;
    prepass_modes_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n, d_params, d_modes, a, lambda, d_eval,
                                                                      d_deep ? d_eval_abs : nullptr);
    return cudaGetLastError();
}

// ---- batched sweep: every run's lattice / parameters / pre-pass in one launch each
cudaError_t gbd_launch_sweep_setup(const GbdRunJob *d_jobs, int n_runs, long max_n, const double *d_abcd,
                                   const gbd_detector &det, int precision, int algo, bool also_separable,
                                   int *d_gate, int *n_launches, cudaStream_t st, int *d_deep)
{
    *n_launches = 0;
    if (n_runs < 1) return cudaSuccess;
    lattice_batch_kernel<<<dim3(8, (unsigned)n_runs), LATTICE_THREADS, 0, st>>>(d_jobs);
    const dim3 grid((unsigned)((max_n + 127) / 128), (unsigned)n_runs);
    propagate_batch_kernel<<<grid, 128, 0, st>>>(d_jobs, d_abcd);
    DetArgs a = det_args(det);
    a.deep = d_deep;
    const int stride = algo == GBD_ALGO_RECURRENCE ? GBD_NEVAL + 2 : GBD_NEVAL;
    const double s2 = det.du * det.du, s2v = det.dv * det.dv;
    prepass_batch_kernel<<<grid, 128, 0, st>>>(d_jobs, a, algo == GBD_ALGO_RECURRENCE ? GBD_PRECISION_FP64 : precision,
                                               stride, s2, s2v, nullptr, 0);
    *n_launches = 3;
    if (also_separable) {
        prepass_batch_kernel<<<grid, 128, 0, st>>>(d_jobs, a, GBD_PRECISION_FP64, GBD_NEVAL + 4, s2, s2v, d_gate, 1);
        *n_launches = 4;
    }
    return cudaGetLastError();
}
