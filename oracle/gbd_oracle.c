/*
 * gbd_oracle.c -- CPU ORACLE for the plane-evaluation Gaussian Beamlet Decomposition hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with paper_2404_12454_b200/csrc (the CUDA path) and neither includes the other.
 *
 * Plain C99, fp64, `double complex`, libm cexp/csqrt/fmod; compiled -O2 -ffp-contract=off
 * (no fast-math).  Loops are written in the paper's order and notation; there is no blocking,
 * fusion or reordering beyond an OpenMP `parallel for` over independent detector pixels.
 *
 * Citations: "P:n" = /root/reference/PAPER.md line n.  "R-xx" = reading xx in DESIGN.md
 * (points where the paper is silent, garbled or inconsistent).
 *
 * What is computed:
 *   a1  gbdo_lattice      evenly spaced beamlets across the pupil          P:243-247, Eq. 24
 *   a2  gbdo_propagate    per beamlet Q2^-1 (Eq. 22), amplitude (Eq. 21),  P:171-177, P:318-320,
 *                         centre / tilt (Eq. 28-29), optical path
 *   a3  gbdo_to_detector  re-expansion onto the (possibly tilted) detector R-T (beyond the paper,
 *                                                                          which assumes an
 *                                                                          orthogonal plane)
 *   a4  gbdo_field_*      E(r) = sum_j A_j exp(-ik[opl_j + p_j.D + 1/2 D^T Q_j^-1 D])
 *                                                                          P:33 Eq. 3
 *                                                                          Eq. 19-20, Eq. 21
 *   a5  optional per-term Gaussian-tail cull (cull_tau)                    R-14
 *   a0  gbdo_trace_mirrors  5-ray differential trace through conic mirrors -> ABCD
 *   pe  gbdo_field_pointeval  the point-evaluation algorithm (comparison baseline)   P:88-100 steps 1-6
 *   hg  gbdo_hg_modes / gbdo_field_rows_modes  Hermite-Gaussian beamlets, orders m+n <= 2   P:84, P:271 (R-23)
 *   +   gbdo_psf_metrics  RMS difference to the Airy pattern, annular zones    P:249-269, R-13
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): closed-form focused Gaussian, brute-force
 * Collins quadrature of P:82 Eq. 13 (incl. the paper's own section 4.1 experiment), Airy
 * pattern, Dirichlet-kernel closed form of an unclipped lattice (at points, at pixel indices of a
 * non-square detector through gbdo_field_pixels, and on the full grid), D4 symmetry, per-beamlet
 * power on the nominal and on tilted planes (obliquity factor), value / gradient / Hessian of the 3-D
 * beam eikonal on tilted planes, direct ray trace onto the tilted plane, exact reduction of the path
 * modulo lambda, linearity / detector shift; ray trace: foci of conics, stigmatic paraboloid, sag of
 * the vertex sheet, an independent numpy trace, the paper's Table 2 -> Table 3 focal length.  The
 * paper prints no numeric field values and states no error bound, so there is no paper-printed
 * golden value; every function below is pinned by at least one of the above.
 *
 * Parameter record ("rec", 13 doubles per beamlet, array-of-structs [n][13]):
 *   0 c_x  1 c_y   centre: base-ray intercept on the plane (mm)
 *   2 p_x  3 p_y   in-plane direction cosines of the base ray there
 *   4 opl          optical path reduced modulo lambda BEFORE small terms are added (R-9)
 *   5,6   Re,Im Q_xx      7,8  Re,Im (Q_xy + Q_yx)      9,10 Re,Im Q_yy     (Q = Q2^-1, 1/mm)
 *   11,12 Re,Im amplitude
 */
#define _DEFAULT_SOURCE   /* j1() */
#include <complex.h>
#include <math.h>
#include <stddef.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

#define GBDO_NREC 13

typedef double complex cplx;

typedef struct {
    int n_u, n_v;
    double du, dv;
    double origin[3], e_u[3], e_v[3];
} gbdo_detector;

/* ------------------------------------------------------------------ 2x2 complex algebra */

static cplx det2(const cplx m[4]) { return m[0] * m[3] - m[1] * m[2]; }

static void inv2(const cplx m[4], cplx out[4])
{
    cplx d = det2(m);
    out[0] = m[3] / d;
    out[1] = -m[1] / d;
    out[2] = -m[2] / d;
    out[3] = m[0] / d;
}

static void mul2(const cplx a[4], const cplx b[4], cplx out[4])
{
    out[0] = a[0] * b[0] + a[1] * b[2];
    out[1] = a[0] * b[1] + a[1] * b[3];
    out[2] = a[2] * b[0] + a[3] * b[2];
    out[3] = a[2] * b[1] + a[3] * b[3];
}

/* eigenvalues of a 2x2: mean +- sqrt(((m00-m11)/2)^2 + m01 m10)  (textbook form) */
static void eig2(const cplx m[4], cplx *mu1, cplx *mu2)
{
    cplx mean = 0.5 * (m[0] + m[3]);
    cplx half = 0.5 * (m[0] - m[3]);
    cplx root = csqrt(half * half + m[1] * m[2]);
    *mu1 = mean + root;
    *mu2 = mean - root;
}

/* R-5: branch of 1/sqrt(det): product of principal square roots of the two eigenvalues, an
 * eigenvalue with Im == 0 exactly being taken as the limit from below (Im = -0). */
static cplx sqrt_lower(cplx mu)
{
    if (cimag(mu) == 0.0) mu = CMPLX(creal(mu), -0.0);
    return csqrt(mu);
}

static cplx sqrt_det_by_eig(const cplx m[4])
{
    cplx mu1, mu2;
    eig2(m, &mu1, &mu2);
    return sqrt_lower(mu1) * sqrt_lower(mu2);
}

/* ------------------------------------------------------------------ a1: lattice, R-10 */

/* Square lattice of n_across points across the diameter D, pitch D/n_across, cell-centred:
 * x_i = (i - (N-1)/2) * pitch; keep a point iff x^2 + y^2 <= (D/2)^2.  Order: iy slow, ix fast.
 * Returns the number kept (also when it exceeds capacity; then only `capacity` are written). */
long gbdo_lattice(int n_across, double diameter, double *x, double *y, long capacity)
{
    double pitch = diameter / (double)n_across;
    double r2max = (0.5 * diameter) * (0.5 * diameter);
    double half = 0.5 * (double)(n_across - 1);
    long n = 0;
    for (int iy = 0; iy < n_across; ++iy) {
        double yy = ((double)iy - half) * pitch;
        for (int ix = 0; ix < n_across; ++ix) {
            double xx = ((double)ix - half) * pitch;
            if (xx * xx + yy * yy <= r2max) {
                if (n < capacity) { x[n] = xx; y[n] = yy; }
                ++n;
            }
        }
    }
    return n;
}

/* P:245 Eq. 24: OF = N_g 2 w0 / W  ->  w0 = OF * pitch / 2 */
double gbdo_waist(double overlap_factor, double pitch) { return overlap_factor * pitch / 2.0; }

/* ------------------------------------------------------------------ a2: per-beamlet parameters */

/* abcd: row-major 4x4 [[A,B],[C,D]] acting on (q_x,q_y,p_x,p_y) (Eq. 23 layout).
 * abcd_mode 1: one shared matrix; base = SoA [3][n] (theta_x, theta_y, OPD) at the pupil or NULL
 *              (zeros); centre c = A r + B theta, tilt p = C r + D theta (Eq. 28-29);
 *              path = l0 + OPD + 1/2 (p.c - theta.r)  (Weber's phase P:129 Eq. 17; R-8).
 * abcd_mode 0: abcd = [n][16]; base = SoA [5][n] (c_x, c_y, p_x, p_y, OPL) of the traced base ray.
 * weight: SoA [2][n] (re, im) or NULL (1 + 0i).
 * Q1^-1 = -i lambda/(pi w0^2) I  (Eq. 4 with the sign that makes P:33 Eq. 3 decay; R-1).  */
int gbdo_propagate(long n, const double *x, const double *y, double w0, double lambda,
                   int abcd_mode, const double *abcd, double l0, const double *base,
                   const double *weight, double *rec)
{
    if (n < 0 || !(w0 > 0.0) || !(lambda > 0.0) || !abcd || !rec) return 1;
    if (abcd_mode != 0 && abcd_mode != 1) return 1;
    if (abcd_mode == 0 && !base) return 1;
    const cplx q1inv = -I * (lambda / (M_PI * w0 * w0));
    const double l0_red = fmod(l0, lambda);                     /* R-9 */
    for (long j = 0; j < n; ++j) {
        const double *m = abcd_mode ? abcd : abcd + 16 * j;
        const double A[4] = { m[0], m[1], m[4], m[5] };
        const double B[4] = { m[2], m[3], m[6], m[7] };
        const double C[4] = { m[8], m[9], m[12], m[13] };
        const double D[4] = { m[10], m[11], m[14], m[15] };
        cplx M1[4], N1[4], M1i[4], Q[4];
        for (int e = 0; e < 4; ++e) {
            M1[e] = A[e] + B[e] * q1inv;                        /* A + B Q1^-1  (Q1^-1 scalar) */
            N1[e] = C[e] + D[e] * q1inv;                        /* C + D Q1^-1 */
        }
        inv2(M1, M1i);
        mul2(N1, M1i, Q);                                       /* P:176 Eq. 22 */
        cplx W = weight ? CMPLX(weight[j], weight[n + j]) : 1.0;
        cplx amp = W / sqrt_det_by_eig(M1);                     /* P:171 Eq. 21, R-5, R-7 */

        double cx, cy, px, py, opl;
        if (abcd_mode == 1) {
            double rx = x[j], ry = y[j];
            double tx = base ? base[j] : 0.0;
            double ty = base ? base[n + j] : 0.0;
            double opd = base ? base[2 * n + j] : 0.0;
            cx = (A[0] * rx + A[1] * ry) + (B[0] * tx + B[1] * ty);       /* Eq. 28 */
            cy = (A[2] * rx + A[3] * ry) + (B[2] * tx + B[3] * ty);
            px = (C[0] * rx + C[1] * ry) + (D[0] * tx + D[1] * ty);       /* Eq. 29 */
            py = (C[2] * rx + C[3] * ry) + (D[2] * tx + D[3] * ty);
            opl = l0_red + (opd + 0.5 * ((px * cx + py * cy) - (tx * rx + ty * ry)));
        } else {
            cx = base[j]; cy = base[n + j]; px = base[2 * n + j]; py = base[3 * n + j];
            opl = fmod(base[4 * n + j], lambda);                /* R-9 */
        }
        double *r = rec + GBDO_NREC * j;
        r[0] = cx; r[1] = cy; r[2] = px; r[3] = py; r[4] = opl;
        r[5] = creal(Q[0]); r[6] = cimag(Q[0]);
        cplx qs = Q[1] + Q[2];                                  /* R-15: no symmetrisation */
        r[7] = creal(qs); r[8] = cimag(qs);
        r[9] = creal(Q[3]); r[10] = cimag(Q[3]);
        r[11] = creal(amp); r[12] = cimag(amp);
    }
    return 0;
}

/* ------------------------------------------------------------------ a3: onto the detector (R-T) */

static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static void cross3(const double a[3], const double b[3], double o[3])
{
    o[0] = a[1]*b[2] - a[2]*b[1];
    o[1] = a[2]*b[0] - a[0]*b[2];
    o[2] = a[0]*b[1] - a[1]*b[0];
}

int gbdo_detector_is_untilted(const gbdo_detector *d)
{
    return d->e_u[0] == 1.0 && d->e_u[1] == 0.0 && d->e_u[2] == 0.0 &&
           d->e_v[0] == 0.0 && d->e_v[1] == 1.0 && d->e_v[2] == 0.0 && d->origin[2] == 0.0;
}

/* Records on the nominal plane (frame X,Y in-plane, Z normal, z = 0) -> records in detector
 * coordinates (u,v): centre relative to `origin` along (e_u,e_v).
 * Untilted detector (e_u = X, e_v = Y, origin z = 0 exactly): only c' = c - origin.
 * Otherwise, per beamlet (DESIGN.md R-T):
 *   k^ = (p_x, p_y, +sqrt(1-|p|^2));  t1 = normalise(Y x k^), t2 = k^ x t1
 *   P0 = [[t1.X, t1.Y],[t2.X, t2.Y]],  Mperp = P0^-T M P0^-1,  M = [[Qxx, Qs/2],[Qs/2, Qyy]]
 *   s = ((origin - c3).n')/(k^.n'),  n' = e_u x e_v,  c3 = (c_x, c_y, 0)
 *   c' = in-plane coordinates of c3 + s k^;  opl' = opl + s
 *   Mperp' = Mperp (I + s Mperp)^-1;  nu = eig(I + s Mperp)
 *   amp' = amp / (sqrt(nu1) sqrt(nu2)) * sqrt((k^.n')/(k^.Z))
 *   P' = [[t1.e_u, t1.e_v],[t2.e_u, t2.e_v]];  M' = P'^T Mperp' P';  p' = (k^.e_u, k^.e_v)      */
int gbdo_to_detector(long n, const double *rec_in, const gbdo_detector *det, double *rec_out)
{
    if (n < 0 || !rec_in || !det || !rec_out) return 1;
    const int untilted = gbdo_detector_is_untilted(det);
    double nrm[3];
    cross3(det->e_u, det->e_v, nrm);
    const double X[3] = { 1, 0, 0 }, Y[3] = { 0, 1, 0 };
    for (long j = 0; j < n; ++j) {
        const double *a = rec_in + GBDO_NREC * j;
        double *o = rec_out + GBDO_NREC * j;
        if (untilted) {
            for (int e = 0; e < GBDO_NREC; ++e) o[e] = a[e];
            o[0] = a[0] - det->origin[0];
            o[1] = a[1] - det->origin[1];
            continue;
        }
        double px = a[2], py = a[3];
        double khat[3] = { px, py, sqrt(1.0 - (px * px + py * py)) };
        double t1[3], t2[3];
        cross3(Y, khat, t1);
        double t1n = sqrt(dot3(t1, t1));
        t1[0] /= t1n; t1[1] /= t1n; t1[2] /= t1n;
        cross3(khat, t1, t2);

        /* in-plane curvature -> transverse curvature */
        double P0[4] = { dot3(t1, X), dot3(t1, Y), dot3(t2, X), dot3(t2, Y) };
        double dP = P0[0] * P0[3] - P0[1] * P0[2];
        double Pi[4] = { P0[3] / dP, -P0[1] / dP, -P0[2] / dP, P0[0] / dP };      /* P0^-1 */
        cplx qxx = CMPLX(a[5], a[6]), qs = CMPLX(a[7], a[8]), qyy = CMPLX(a[9], a[10]);
        cplx M[4] = { qxx, 0.5 * qs, 0.5 * qs, qyy };
        cplx Pic[4] = { Pi[0], Pi[1], Pi[2], Pi[3] };
        cplx PiT[4] = { Pi[0], Pi[2], Pi[1], Pi[3] };
        cplx T[4], Mp[4];
        mul2(PiT, M, T);
        mul2(T, Pic, Mp);                                       /* Mperp */

        /* walk along the base ray to the detector plane */
        double c3[3] = { a[0], a[1], 0.0 };
        double w[3] = { det->origin[0] - c3[0], det->origin[1] - c3[1], det->origin[2] - c3[2] };
        double s = dot3(w, nrm) / dot3(khat, nrm);
        double hit[3] = { c3[0] + s * khat[0] - det->origin[0],
                          c3[1] + s * khat[1] - det->origin[1],
                          c3[2] + s * khat[2] - det->origin[2] };
        cplx G[4] = { 1.0 + s * Mp[0], s * Mp[1], s * Mp[2], 1.0 + s * Mp[3] };  /* I + s Mperp */
        cplx Gi[4], Mps[4];
        inv2(G, Gi);
        mul2(Mp, Gi, Mps);                                      /* Mperp' */
        /* obliquity: Eq. 21 normalises power per unit IN-PLANE area, so going from the plane with
         * normal Z to the plane with normal n' rescales by sqrt((k^.n')/(k^.Z)) (R-T) */
        cplx amp = CMPLX(a[11], a[12]) / sqrt_det_by_eig(G) * sqrt(dot3(khat, nrm) / khat[2]);

        /* transverse curvature -> detector in-plane curvature */
        cplx Pd[4] = { dot3(t1, det->e_u), dot3(t1, det->e_v), dot3(t2, det->e_u), dot3(t2, det->e_v) };
        cplx PdT[4] = { Pd[0], Pd[2], Pd[1], Pd[3] };
        cplx T2[4], Md[4];
        mul2(PdT, Mps, T2);
        mul2(T2, Pd, Md);                                       /* M' */
        cplx qsd = Md[1] + Md[2];

        o[0] = dot3(hit, det->e_u);
        o[1] = dot3(hit, det->e_v);
        o[2] = dot3(khat, det->e_u);
        o[3] = dot3(khat, det->e_v);
        o[4] = a[4] + s;
        o[5] = creal(Md[0]); o[6] = cimag(Md[0]);
        o[7] = creal(qsd);   o[8] = cimag(qsd);
        o[9] = creal(Md[3]); o[10] = cimag(Md[3]);
        o[11] = creal(amp);  o[12] = cimag(amp);
    }
    return 0;
}

/* ------------------------------------------------------------------ a4 (+a5): the field sum */

/* One pixel: direct sum over all beamlets of
 *   amp_j * cexp(-i k (opl_j + p_j.D + 1/2 (Qxx Du^2 + Qs Du Dv + Qyy Dv^2))),  D = (u,v) - c'_j.
 * cull_tau > 0: a term is dropped iff its envelope exp((k/2) Im(quad)) < cull_tau (R-14).   */
static cplx pixel_sum(long n, const double *rec, double k, double u, double v, double cull_tau)
{
    cplx E = 0.0;
    for (long j = 0; j < n; ++j) {
        const double *a = rec + GBDO_NREC * j;
        double du = u - a[0], dv = v - a[1];
        cplx quad = CMPLX(a[5], a[6]) * (du * du) + CMPLX(a[7], a[8]) * (du * dv)
                  + CMPLX(a[9], a[10]) * (dv * dv);
        if (cull_tau > 0.0 && exp(0.5 * k * cimag(quad)) < cull_tau) continue;
        cplx arg = a[4] + (a[2] * du + a[3] * dv) + 0.5 * quad;
        E += CMPLX(a[11], a[12]) * cexp(-I * k * arg);
    }
    return E;
}

static double pix_coord(int i, int n, double h) { return ((double)i - 0.5 * (double)(n - 1)) * h; }

/* Rows [v0, v1) with stride vstep of the detector; field is the FULL [n_v][n_u][2] array
 * (re,im interleaved, v slow); rows not visited are left untouched.  rec = detector records. */
int gbdo_field_rows(long n, const double *rec, const gbdo_detector *det, double lambda,
                    double cull_tau, int v0, int v1, int vstep, double *field)
{
    if (n < 0 || !rec || !det || !field || !(lambda > 0.0) || vstep < 1) return 1;
    if (v0 < 0 || v1 > det->n_v) return 1;
    const double k = 2.0 * M_PI / lambda;
    const int nu = det->n_u;
#pragma omp parallel for schedule(dynamic, 1)
    for (int iv = v0; iv < v1; iv += vstep) {
        double v = pix_coord(iv, det->n_v, det->dv);
        for (int iu = 0; iu < nu; ++iu) {
            double u = pix_coord(iu, nu, det->du);
            cplx E = pixel_sum(n, rec, k, u, v, cull_tau);
            field[2 * ((size_t)iv * nu + iu)] = creal(E);
            field[2 * ((size_t)iv * nu + iu) + 1] = cimag(E);
        }
    }
    return 0;
}

/* A list of pixels (iu[i], iv[i]); out = [npix][2]. */
int gbdo_field_pixels(long n, const double *rec, const gbdo_detector *det, double lambda,
                      double cull_tau, long npix, const int *iu, const int *iv, double *out)
{
    if (n < 0 || !rec || !det || !out || !(lambda > 0.0) || npix < 0) return 1;
    const double k = 2.0 * M_PI / lambda;
#pragma omp parallel for schedule(dynamic, 16)
    for (long i = 0; i < npix; ++i) {
        double u = pix_coord(iu[i], det->n_u, det->du);
        double v = pix_coord(iv[i], det->n_v, det->dv);
        cplx E = pixel_sum(n, rec, k, u, v, cull_tau);
        out[2 * i] = creal(E);
        out[2 * i + 1] = cimag(E);
    }
    return 0;
}

/* Arbitrary in-plane points (u[i], v[i]) in detector coordinates; out = [npts][2]. */
int gbdo_field_points(long n, const double *rec, double lambda, double cull_tau,
                      long npts, const double *u, const double *v, double *out)
{
    if (n < 0 || !rec || !out || !(lambda > 0.0) || npts < 0) return 1;
    const double k = 2.0 * M_PI / lambda;
    for (long i = 0; i < npts; ++i) {
        cplx E = pixel_sum(n, rec, k, u[i], v[i], cull_tau);
        out[2 * i] = creal(E);
        out[2 * i + 1] = cimag(E);
    }
    return 0;
}

/* ------------------------------------------------------------------ Hermite-Gaussian beamlets */

/* "Equation 13 has been solved ... to determine the propagation laws for Hermite [20] ... Gaussian beams.  All of
 * these solutions can be employed in beamlet decomposition".  Ref. [20] is not in the
 * container; the law for the orders used here follows from P:82 Eq. 13 directly (R-23).
 * Pupil field of a beamlet:  [sum_{m+n<=2} w_mn H_m(sqrt2 x~/w0) H_n(sqrt2 y~/w0)] exp(-|r~|^2/w0^2) exp(-ik th.r~),
 * r~ = r1 - r1M, physicists' Hermite polynomials (H0 = 1, H1 = 2 s, H2 = 4 s^2 - 2).
 * Generating function: sum_mn H_m(xi) H_n(zeta) s^m t^n/(m! n!) = exp(2 xi s - s^2 + 2 zeta t - t^2), so the input
 * exp(-|r~|^2/w0^2 + a.r~ - |sigma|^2), a = (2 sqrt2/w0) sigma, sigma = (s, t), generates all modes.  It is a Gaussian
 * with a linear term; completing the square in Eq. 13 (with B^-1 A and D B^-1 symmetric) gives
 *      E2[sigma] = E2,fundamental(D) * exp( 2 eta.sigma - sigma^T Gamma sigma ),
 *      eta = (sqrt2/w0) M1^-1 D,   Gamma = M1^-1 (A - B Q1^-1) = 2 M1^-1 A - I,   M1 = A + B Q1^-1,   D = r2 - c,
 * and the coefficient of s^m t^n/(m! n!) is mode (m, n):
 *      (1,0): 2 eta_x        (0,1): 2 eta_y
 *      (2,0): 4 eta_x^2 - 2 Gamma_xx      (0,2): 4 eta_y^2 - 2 Gamma_yy      (1,1): 4 eta_x eta_y - (Gamma_xy + Gamma_yx)
 * -- the same phasor times a complex polynomial of degree <= 2 in D (the complex scaling of the Hermite arguments
 * and the extra Gouy phase of each mode are inside M1^-1 and Gamma).  This function returns its coefficients:
 *   mode_weight: SoA [12][n] = Re, Im of w00, w10, w01, w20, w11, w02 (NULL -> w00 = 1, others 0)
 *   modes: [n][12] = Re, Im of a0, a_x, a_y, a_xx, a_xy, a_yy,
 *          factor(D) = a0 + a_x D_x + a_y D_y + a_xx D_x^2 + a_xy D_x D_y + a_yy D_y^2.
 * Evaluation planes orthogonal to the axis only (untilted detector; the paper's own restriction).  */
#define GBDO_NMODE 12
int gbdo_hg_modes(long n, double w0, double lambda, int abcd_mode, const double *abcd,
                  const double *mode_weight, double *modes)
{
    if (n < 0 || !(w0 > 0.0) || !(lambda > 0.0) || !abcd || !modes) return 1;
    if (abcd_mode != 0 && abcd_mode != 1) return 1;
    const cplx q1inv = -I * (lambda / (M_PI * w0 * w0));
    const double c0 = 2.0 * sqrt(2.0) / w0;
    for (long j = 0; j < n; ++j) {
        const double *m = abcd_mode ? abcd : abcd + 16 * j;
        const double A[4] = { m[0], m[1], m[4], m[5] }, B[4] = { m[2], m[3], m[6], m[7] };
        cplx M1[4], M1i[4], Ac[4], G[4];
        for (int e = 0; e < 4; ++e) { M1[e] = A[e] + B[e] * q1inv; Ac[e] = A[e]; }
        inv2(M1, M1i);
        mul2(M1i, Ac, G);                                        /* M1^-1 A */
        for (int e = 0; e < 4; ++e) G[e] *= 2.0;
        G[0] -= 1.0; G[3] -= 1.0;                                /* Gamma = 2 M1^-1 A - I */
        cplx w[6] = { 1.0, 0.0, 0.0, 0.0, 0.0, 0.0 };            /* w00 w10 w01 w20 w11 w02 */
        if (mode_weight)
            for (int q = 0; q < 6; ++q) w[q] = CMPLX(mode_weight[(2 * q) * n + j], mode_weight[(2 * q + 1) * n + j]);
        /* 2 eta_x = ax . D,  2 eta_y = ay . D */
        const cplx ax[2] = { c0 * M1i[0], c0 * M1i[1] }, ay[2] = { c0 * M1i[2], c0 * M1i[3] };
        cplx a[6];
        a[0] = w[0] - 2.0 * w[3] * G[0] - w[4] * (G[1] + G[2]) - 2.0 * w[5] * G[3];
        a[1] = w[1] * ax[0] + w[2] * ay[0];
        a[2] = w[1] * ax[1] + w[2] * ay[1];
        a[3] = w[3] * ax[0] * ax[0] + w[4] * ax[0] * ay[0] + w[5] * ay[0] * ay[0];
        a[4] = 2.0 * w[3] * ax[0] * ax[1] + w[4] * (ax[0] * ay[1] + ax[1] * ay[0]) + 2.0 * w[5] * ay[0] * ay[1];
        a[5] = w[3] * ax[1] * ax[1] + w[4] * ax[1] * ay[1] + w[5] * ay[1] * ay[1];
        double *o = modes + GBDO_NMODE * j;
        for (int q = 0; q < 6; ++q) { o[2 * q] = creal(a[q]); o[2 * q + 1] = cimag(a[q]); }
    }
    return 0;
}

/* The field sum with the mode factor: rows [v0, v1) step vstep of an UNTILTED detector (rec = detector
 * records from gbdo_to_detector, whose centres are relative to the detector origin; modes from gbdo_hg_modes). */
int gbdo_field_rows_modes(long n, const double *rec, const double *modes, const gbdo_detector *det, double lambda,
                          int v0, int v1, int vstep, double *field)
{
    if (n < 0 || !rec || !modes || !det || !field || !(lambda > 0.0) || vstep < 1) return 1;
    if (v0 < 0 || v1 > det->n_v || !gbdo_detector_is_untilted(det)) return 1;
    const double k = 2.0 * M_PI / lambda;
    const int nu = det->n_u;
#pragma omp parallel for schedule(dynamic, 1)
    for (int iv = v0; iv < v1; iv += vstep) {
        double v = pix_coord(iv, det->n_v, det->dv);
        for (int iu = 0; iu < nu; ++iu) {
            double u = pix_coord(iu, nu, det->du);
            cplx E = 0.0;
            for (long j = 0; j < n; ++j) {
                const double *a = rec + GBDO_NREC * j, *h = modes + GBDO_NMODE * j;
                double du = u - a[0], dv = v - a[1];
                cplx quad = CMPLX(a[5], a[6]) * (du * du) + CMPLX(a[7], a[8]) * (du * dv)
                          + CMPLX(a[9], a[10]) * (dv * dv);
                cplx arg = a[4] + (a[2] * du + a[3] * dv) + 0.5 * quad;
                cplx factor = CMPLX(h[0], h[1]) + CMPLX(h[2], h[3]) * du + CMPLX(h[4], h[5]) * dv
                            + CMPLX(h[6], h[7]) * (du * du) + CMPLX(h[8], h[9]) * (du * dv) + CMPLX(h[10], h[11]) * (dv * dv);
                E += CMPLX(a[11], a[12]) * factor * cexp(-I * k * arg);
            }
            field[2 * ((size_t)iv * nu + iu)] = creal(E);
            field[2 * ((size_t)iv * nu + iu) + 1] = cimag(E);
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ point evaluation (section 2.2) */

/* The "traditional" algorithm the paper accelerates, kept as the comparison baseline (Fig. 7): for every
 * evaluation point r_eval and every beamlet, steps 2-5 of P:92-99 (step 1, the trace to the evaluation plane, is the
 * input: base ray c, p, OPL and the differential ABCD of the 4 parabasal rays there; step 6 is the sum):
 *   2. distance from the base ray's intercept c3 = (c_x, c_y, 0) to the transversal plane P_trans -- the plane
 *      normal to the ray k^ = (p_x, p_y, sqrt(1-|p|^2)) through r_eval:          t = (r_eval - c3).k^
 *   3. propagate the 5 rays to P_trans and express them in its local frame (t1, t2) (t1 = normalise(Y x k^),
 *      t2 = k^ x t1, as in R-T).  The parabasal rays are the base ray plus the columns of the ABCD, so this is done on
 *      the differentials (R-22): a ray displaced in-plane by dq and tilted by dp (dp_z = -p.dp/p_z keeps it
 *      a unit vector) meets P_trans at  dq~ = P0 dq + t Pd dp  with direction  dp~ = Pd dp,  where
 *      P0 = [[t1_x, t1_y],[t2_x, t2_y]]  and  Pd[i][j] = t_i[j] - t_i[z] p_j / p_z   (first order, exact for rays).
 *   4. differential ABCD from the pupil to P_trans:  A' = P0 A + t Pd C,  B' = P0 B + t Pd D,  C' = Pd C,  D' = Pd D
 *   5. Gaussian field (Eq. 21, Eq. 22) with that ABCD at r_eval, whose local coordinates on P_trans are
 *      xi = ((r_eval - c3).t1, (r_eval - c3).t2) (the base ray pierces P_trans at xi = 0 with no tilt):
 *        Q' = (C' + D' Q1^-1)(A' + B' Q1^-1)^-1,   E = W / sqrt(det(A' + B' Q1^-1)) exp(-ik [opl + t + 1/2 xi^T Q' xi])
 *      (branch of the square root as in R-5; opl reduced modulo lambda as in R-9).
 * All of the 2x2 complex algebra (inverse, eigenvalues) is redone for every (point, beamlet) pair: this is where
 * the time of the point-evaluation code goes.  Note the normalisation: Eq. 21 applied on P_trans gives
 * power per unit area NORMAL TO THE RAY, the plane evaluation power per unit area of the evaluation plane; the two
 * differ by sqrt(k^.Z) per beamlet (1e-4 for the paper's f/24 telescope), beyond the parabasal residual.
 *
 * Arguments as gbdo_propagate (x, y, w0, lambda, abcd_mode, abcd, l0, base, weight) and gbdo_field_rows (detector in
 * the nominal-plane frame, rows [v0, v1) with stride vstep, field = full [n_v][n_u][2] array).                        */
int gbdo_field_pointeval(long n, const double *x, const double *y, double w0, double lambda,
                         int abcd_mode, const double *abcd, double l0, const double *base,
                         const double *weight, const gbdo_detector *det, int v0, int v1, int vstep,
                         double *field)
{
    if (n < 0 || !(w0 > 0.0) || !(lambda > 0.0) || !abcd || !det || !field || vstep < 1) return 1;
    if (abcd_mode != 0 && abcd_mode != 1) return 1;
    if (abcd_mode == 0 && !base) return 1;
    if (v0 < 0 || v1 > det->n_v) return 1;
    const cplx q1inv = -I * (lambda / (M_PI * w0 * w0));
    const double k = 2.0 * M_PI / lambda;
    const double l0_red = fmod(l0, lambda);
    const double Yax[3] = { 0, 1, 0 };
    const int nu = det->n_u;
#pragma omp parallel for schedule(dynamic, 1)
    for (int iv = v0; iv < v1; iv += vstep) {
        for (int iu = 0; iu < nu; ++iu) {
            const double u = pix_coord(iu, nu, det->du), v = pix_coord(iv, det->n_v, det->dv);
            double R[3];
            for (int i = 0; i < 3; ++i) R[i] = det->origin[i] + u * det->e_u[i] + v * det->e_v[i];
            cplx E = 0.0;
            for (long j = 0; j < n; ++j) {
                /* step 1 (input): rays on the evaluation plane */
                const double *m = abcd_mode ? abcd : abcd + 16 * j;
                const double A[4] = { m[0], m[1], m[4], m[5] }, B[4] = { m[2], m[3], m[6], m[7] };
                const double C[4] = { m[8], m[9], m[12], m[13] }, D[4] = { m[10], m[11], m[14], m[15] };
                double c[2], p[2], opl;
                if (abcd_mode == 1) {
                    const double rx = x[j], ry = y[j];
                    const double tx = base ? base[j] : 0.0, ty = base ? base[n + j] : 0.0;
                    const double opd = base ? base[2 * n + j] : 0.0;
                    c[0] = (A[0] * rx + A[1] * ry) + (B[0] * tx + B[1] * ty);
                    c[1] = (A[2] * rx + A[3] * ry) + (B[2] * tx + B[3] * ty);
                    p[0] = (C[0] * rx + C[1] * ry) + (D[0] * tx + D[1] * ty);
                    p[1] = (C[2] * rx + C[3] * ry) + (D[2] * tx + D[3] * ty);
                    opl = l0_red + (opd + 0.5 * ((p[0] * c[0] + p[1] * c[1]) - (tx * rx + ty * ry)));
                } else {
                    c[0] = base[j]; c[1] = base[n + j]; p[0] = base[2 * n + j]; p[1] = base[3 * n + j];
                    opl = fmod(base[4 * n + j], lambda);
                }
                const double pz = sqrt(1.0 - (p[0] * p[0] + p[1] * p[1]));
                const double khat[3] = { p[0], p[1], pz };
                double t1[3], t2[3];
                cross3(Yax, khat, t1);
                const double t1n = sqrt(dot3(t1, t1));
                for (int i = 0; i < 3; ++i) t1[i] /= t1n;
                cross3(khat, t1, t2);
                /* step 2: distance to the transversal plane through R */
                const double w3[3] = { R[0] - c[0], R[1] - c[1], R[2] };
                const double t = dot3(w3, khat);
                /* step 3: differentials onto P_trans, local frame */
                const double P0[4] = { t1[0], t1[1], t2[0], t2[1] };
                const double Pd[4] = { t1[0] - t1[2] * p[0] / pz, t1[1] - t1[2] * p[1] / pz,
                                       t2[0] - t2[2] * p[0] / pz, t2[1] - t2[2] * p[1] / pz };
                const double xi[2] = { dot3(w3, t1), dot3(w3, t2) };
                /* step 4: ABCD from the pupil to P_trans */
                double At[4], Bt[4], Ct[4], Dt[4];
                for (int r = 0; r < 2; ++r)
                    for (int q = 0; q < 2; ++q) {
                        Ct[2 * r + q] = Pd[2 * r] * C[q] + Pd[2 * r + 1] * C[2 + q];
                        Dt[2 * r + q] = Pd[2 * r] * D[q] + Pd[2 * r + 1] * D[2 + q];
                        At[2 * r + q] = (P0[2 * r] * A[q] + P0[2 * r + 1] * A[2 + q]) + t * Ct[2 * r + q];
                        Bt[2 * r + q] = (P0[2 * r] * B[q] + P0[2 * r + 1] * B[2 + q]) + t * Dt[2 * r + q];
                    }
                /* step 5: Eq. 22, Eq. 21 at xi */
                cplx M1[4], N1[4], M1i[4], Q[4];
                for (int e = 0; e < 4; ++e) { M1[e] = At[e] + Bt[e] * q1inv; N1[e] = Ct[e] + Dt[e] * q1inv; }
                inv2(M1, M1i);
                mul2(N1, M1i, Q);
                const cplx W = weight ? CMPLX(weight[j], weight[n + j]) : 1.0;
                const cplx amp = W / sqrt_det_by_eig(M1);
                const cplx quad = Q[0] * (xi[0] * xi[0]) + (Q[1] + Q[2]) * (xi[0] * xi[1]) + Q[3] * (xi[1] * xi[1]);
                E += amp * cexp(-I * k * ((opl + t) + 0.5 * quad));         /* step 6: coherent sum */
            }
            field[2 * ((size_t)iv * nu + iu)] = creal(E);
            field[2 * ((size_t)iv * nu + iu) + 1] = cimag(E);
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ differential ray trace */

/* "a set of beamlets whose propagation are described by 5 parabasal rays for each beamlet";
 * "Compute the differential ABCD matrix ... using differential ray tracing" (P:98 step 4).  The paper
 * names the operation and gives no formulas ([14] is not in the container): DESIGN.md R-20 is the
 * definition, written out here from analytic geometry in extended precision (x87 `long double`,
 * 64-bit significand), results rounded to double once at the end.  This is the definition's value
 * to ~1e-19 relative, NOT a copy of what the CUDA kernel does step by step: the kernel is compared
 * with it to a bound derived from fp64 rounding (tests/test_parity_gpu.py), not bit for bit.
 *
 * Surfaces: reflecting conics of revolution about the z axis (prescription form P:324-327 Table 2),
 *     F(x, y, z') = c (x^2 + y^2 + (1+k) z'^2) - 2 z' = 0,   z' = z - z_vertex,  c = 1/RoC signed along +z
 * (equivalent to the standard sag z' = c r^2 / (1 + sqrt(1 - (1+k) c^2 r^2))); refractive index 1.
 * A ray X(t) = X0 + t d put into F gives  a t^2 + 2 b t + g = 0  with
 *     a = c (dx^2 + dy^2 + (1+k) dz^2),  b = c (x0 dx + y0 dy + (1+k) z0' dz) - dz,  g = F(X0).
 * Of its intersections the mirror is the sheet through the vertex: since (1 - c(1+k)z')^2 =
 * 1 - (1+k) c^2 r^2 on the conic, that sheet is where dF/dz' = -2 (1 - c (1+k) z') < 0; when both
 * intersections lie on it (a paraboloid crossed twice) the one nearer the vertex plane, smaller |z'|.
 * Reflection about the surface gradient G = grad F / 2 = (c x, c y, c (1+k) z' - 1):
 *     d' = d - 2 (d.G)/(G.G) G.
 * Rays start on the pupil plane z = z_pupil at (x, y) with direction (p_x, p_y, dir_sign sqrt(1-|p|^2)) and end
 * on the evaluation plane through `origin` spanned by the orthonormal (e_x, e_y) (normal e_x x e_y).
 * Output coordinates are in-plane: q = ((hit-origin).e_x, (hit-origin).e_y), p = (d.e_x, d.e_y).
 * The ray-transfer matrix of beamlet j is the forward finite difference of the base ray and four rays whose
 * start values are the fp64 sums x+dq, y+dq, p_x+dp, p_y+dp (each divided by the nominal step; abcd[j]
 * row-major [[A,B],[C,D]] on (q_x,q_y,p_x,p_y)); base = SoA [5][n]: q_x, q_y, p_x, p_y, OPL = opl0 +
 * geometric path length.
 * wavelength > 0 (R-24, the extension of R-9 to the trace): the OPL row is fmod(OPL, wavelength), taken
 * in extended precision BEFORE the rounding to double -- the field uses the path only modulo the wavelength
 * (Eq. 3: exp(-ik OPL)), and a double holds the remainder exactly where it holds a 16 m path only to 2e-12 mm
 * = 2e-8 rad at 551 nm.  wavelength <= 0: the full path, rounded to double.  */
typedef struct { double curvature, conic, z_vertex; } gbdo_mirror;
typedef long double xreal;

typedef struct { xreal q[2], p[2], path; } gbdo_ray_out;

/* parameter t of the mirror intersection of the ray X0 + t d (X0 given relative to the vertex) */
static xreal conic_intersection(const gbdo_mirror *mr, const xreal X0[3], const xreal d[3])
{
    const xreal c = mr->curvature, e = 1.0L + (xreal)mr->conic;
    if (c == 0.0L) return -X0[2] / d[2];                                    /* flat mirror z' = 0 */
    const xreal a = c * (d[0] * d[0] + d[1] * d[1] + e * d[2] * d[2]);
    const xreal b = c * (X0[0] * d[0] + X0[1] * d[1] + e * X0[2] * d[2]) - d[2];
    const xreal g = c * (X0[0] * X0[0] + X0[1] * X0[1] + e * X0[2] * X0[2]) - 2.0L * X0[2];
    /* both roots without cancellation: w = -(b + sgn(b) sqrt(b^2 - a g)),  t = w/a  and  t = g/w */
    const xreal w = -(b + copysignl(sqrtl(b * b - a * g), b));
    xreal cand[2];
    int nc = 0;
    if (w != 0.0L) cand[nc++] = g / w;
    if (a != 0.0L) cand[nc++] = w / a;
    xreal best_t = NAN, best_z = INFINITY;
    for (int i = 0; i < nc; ++i) {
        const xreal z = X0[2] + cand[i] * d[2];
        if (1.0L - c * e * z > 0.0L && fabsl(z) < best_z) { best_z = fabsl(z); best_t = cand[i]; }
    }
    return best_t;                                                           /* NaN: the ray misses the mirror */
}

static gbdo_ray_out trace_ray(double x, double y, double px, double py, double dir_sign, double z_pupil,
                              int n_mirrors, const gbdo_mirror *mirrors, const double origin[3],
                              const double e_x[3], const double e_y[3])
{
    xreal X[3] = { x, y, z_pupil };
    xreal d[3] = { px, py, 0.0L };
    d[2] = (xreal)dir_sign * sqrtl(1.0L - (d[0] * d[0] + d[1] * d[1]));
    xreal path = 0.0L;
    for (int m = 0; m < n_mirrors; ++m) {
        const gbdo_mirror *mr = &mirrors[m];
        const xreal X0[3] = { X[0], X[1], X[2] - (xreal)mr->z_vertex };
        const xreal t = conic_intersection(mr, X0, d);
        xreal H[3];                                                          /* hit point, vertex frame */
        for (int i = 0; i < 3; ++i) H[i] = X0[i] + t * d[i];
        path += t;                                                           /* |d| = 1 */
        const xreal c = mr->curvature, e = 1.0L + (xreal)mr->conic;
        const xreal G[3] = { c * H[0], c * H[1], c * e * H[2] - 1.0L };
        const xreal f = 2.0L * (d[0] * G[0] + d[1] * G[1] + d[2] * G[2]) / (G[0] * G[0] + G[1] * G[1] + G[2] * G[2]);
        for (int i = 0; i < 3; ++i) d[i] -= f * G[i];
        X[0] = H[0]; X[1] = H[1]; X[2] = H[2] + (xreal)mr->z_vertex;
    }
    /* evaluation plane: (X + t d - origin) . n = 0,  n = e_x x e_y */
    const xreal n[3] = { (xreal)e_x[1] * e_y[2] - (xreal)e_x[2] * e_y[1],
                         (xreal)e_x[2] * e_y[0] - (xreal)e_x[0] * e_y[2],
                         (xreal)e_x[0] * e_y[1] - (xreal)e_x[1] * e_y[0] };
    xreal rel[3], num = 0.0L, den = 0.0L;
    for (int i = 0; i < 3; ++i) { rel[i] = X[i] - (xreal)origin[i]; num -= rel[i] * n[i]; den += d[i] * n[i]; }
    const xreal t = num / den;
    gbdo_ray_out r = { { 0.0L, 0.0L }, { 0.0L, 0.0L }, path + t };
    for (int i = 0; i < 3; ++i) {
        const xreal h = rel[i] + t * d[i];
        r.q[0] += h * e_x[i]; r.q[1] += h * e_y[i];
        r.p[0] += d[i] * e_x[i]; r.p[1] += d[i] * e_y[i];
    }
    return r;
}

int gbdo_trace_mirrors(long n, const double *x, const double *y, const double *px, const double *py,
                       const double p_common[2], double dir_sign, double z_pupil, const double *opl0,
                       int n_mirrors, const gbdo_mirror *mirrors, const double origin[3],
                       const double e_x[3], const double e_y[3], double dq, double dp, double wavelength,
                       double *abcd, double *base)
{
    if (n < 0 || !x || !y || n_mirrors < 0 || (n_mirrors && !mirrors) || !origin || !e_x || !e_y || !abcd || !base)
        return 1;
    if (!(dq > 0.0) || !(dp > 0.0) || (dir_sign != 1.0 && dir_sign != -1.0)) return 1;
    if ((!px || !py) && !p_common) return 1;
    for (long j = 0; j < n; ++j) {
        const double start[4] = { x[j], y[j], px ? px[j] : p_common[0], py ? py[j] : p_common[1] };
        const gbdo_ray_out b = trace_ray(start[0], start[1], start[2], start[3], dir_sign, z_pupil,
                                         n_mirrors, mirrors, origin, e_x, e_y);
        for (int col = 0; col < 4; ++col) {                                 /* the 4 parabasal rays */
            const double h = col < 2 ? dq : dp;
            double s[4] = { start[0], start[1], start[2], start[3] };
            s[col] = start[col] + h;                                         /* fp64 sum (see above) */
            const gbdo_ray_out r = trace_ray(s[0], s[1], s[2], s[3], dir_sign, z_pupil,
                                             n_mirrors, mirrors, origin, e_x, e_y);
            abcd[16 * j + 0 + col]  = (double)((r.q[0] - b.q[0]) / h);
            abcd[16 * j + 4 + col]  = (double)((r.q[1] - b.q[1]) / h);
            abcd[16 * j + 8 + col]  = (double)((r.p[0] - b.p[0]) / h);
            abcd[16 * j + 12 + col] = (double)((r.p[1] - b.p[1]) / h);
        }
        base[j] = (double)b.q[0]; base[n + j] = (double)b.q[1];
        base[2 * n + j] = (double)b.p[0]; base[3 * n + j] = (double)b.p[1];
        const xreal opl = (opl0 ? (xreal)opl0[j] : 0.0L) + b.path;
        base[4 * n + j] = (double)(wavelength > 0.0 ? fmodl(opl, (xreal)wavelength) : opl);
    }
    return 0;
}

/* ------------------------------------------------------------------ figure of merit */

/* RMS difference between the peak-normalised intensity |E|^2/|E0|^2 and the Airy pattern
 * (2 J1(x)/x)^2, x = pi r/(lambda F#)  (R-13), over all pixels and over the annular zones
 * 0-5, 5-10, 10-15 lambda/D (Fig. 9).  r is measured from the detector origin.
 * field: [n_v][n_u][2]; e0: the on-axis field (re, im).
 * out[0..3] = RMS {all, 0-5, 5-10, 10-15}; out[4..7] = pixel counts; out[8] = max |I - Airy|.   */
int gbdo_psf_metrics(const double *field, const gbdo_detector *det, double lambda_fnum,
                     const double *e0, double *out)
{
    if (!field || !det || !e0 || !out || !(lambda_fnum > 0.0)) return 1;
    double i0 = e0[0] * e0[0] + e0[1] * e0[1];
    double sum[4] = { 0, 0, 0, 0 }, cnt[4] = { 0, 0, 0, 0 }, dmax = 0.0;
    for (int iv = 0; iv < det->n_v; ++iv) {
        double v = pix_coord(iv, det->n_v, det->dv);
        for (int iu = 0; iu < det->n_u; ++iu) {
            double u = pix_coord(iu, det->n_u, det->du);
            double rl = sqrt(u * u + v * v) / lambda_fnum;
            double x = M_PI * rl;
            double airy = 1.0;
            if (x != 0.0) { double t = 2.0 * j1(x) / x; airy = t * t; }
            size_t k = 2 * ((size_t)iv * det->n_u + iu);
            double d = (field[k] * field[k] + field[k + 1] * field[k + 1]) / i0 - airy;
            sum[0] += d * d; cnt[0] += 1.0;
            int z = rl < 5.0 ? 1 : (rl < 10.0 ? 2 : (rl < 15.0 ? 3 : 0));
            if (z) { sum[z] += d * d; cnt[z] += 1.0; }
            if (fabs(d) > dmax) dmax = fabs(d);
        }
    }
    for (int z = 0; z < 4; ++z) {
        out[z] = cnt[z] > 0.0 ? sqrt(sum[z] / cnt[z]) : 0.0;
        out[4 + z] = cnt[z];
    }
    out[8] = dmax;
    return 0;
}

#ifdef _OPENMP
#include <omp.h>
int gbdo_num_threads(void) { return omp_get_max_threads(); }
void gbdo_set_num_threads(int t) { if (t > 0) omp_set_num_threads(t); }
#else
int gbdo_num_threads(void) { return 1; }
void gbdo_set_num_threads(int t) { (void)t; }
#endif
