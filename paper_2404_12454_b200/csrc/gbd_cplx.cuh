// gbd_cplx.cuh -- closed-form complex 2x2 algebra of the per-beamlet kernels (App. C: determinant, inverse
// and eigenvalues written out instead of a general linear-algebra routine).  Product code (gbd_params.cu,
// gbd_pointeval.cu); nothing here is shared with oracle/.
#pragma once

namespace {

struct cd { double re, im; };
__device__ inline cd mk(double a, double b) { cd r; r.re = a; r.im = b; return r; }
__device__ inline cd operator+(cd a, cd b) { return mk(a.re + b.re, a.im + b.im); }
__device__ inline cd operator-(cd a, cd b) { return mk(a.re - b.re, a.im - b.im); }
__device__ inline cd operator-(cd a) { return mk(-a.re, -a.im); }
__device__ inline cd operator*(cd a, cd b) { return mk(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
__device__ inline cd operator*(double s, cd a) { return mk(s * a.re, s * a.im); }
__device__ inline cd operator/(cd a, cd b)
{
    // scaled division (avoids overflow of |b|^2)
    double s = 1.0 / fmax(fabs(b.re), fabs(b.im));
    double br = b.re * s, bi = b.im * s;
    double d = 1.0 / (br * br + bi * bi);
    return mk((a.re * br + a.im * bi) * d * s, (a.im * br - a.re * bi) * d * s);
}
// principal square root; Im == 0 is taken as -0 (limit from below, R-5)
__device__ inline cd csqrt_lower(cd z)
{
    double a = z.re, b = z.im;
    if (b == 0.0) b = -0.0;
    double r = hypot(a, b);
    if (r == 0.0) return mk(0.0, -0.0);
    if (a >= 0.0) {
        double t = sqrt(0.5 * (r + a));
        return mk(t, b / (2.0 * t));
    }
    double t = sqrt(0.5 * (r - a));
    return mk(fabs(b) / (2.0 * t), copysign(t, b));
}
// plain principal square root (used for the eigenvalue discriminant)
__device__ inline cd csqrt_principal(cd z)
{
    double a = z.re, b = z.im;
    double r = hypot(a, b);
    if (r == 0.0) return mk(0.0, b);
    if (a >= 0.0) {
        double t = sqrt(0.5 * (r + a));
        return mk(t, b / (2.0 * t));
    }
    double t = sqrt(0.5 * (r - a));
    return mk(fabs(b) / (2.0 * t), copysign(t, b));
}
struct m2 { cd a, b, c, d; };   // [[a,b],[c,d]]
__device__ inline m2 mul(m2 x, m2 y)
{
    m2 r;
    r.a = x.a * y.a + x.b * y.c;
    r.b = x.a * y.b + x.b * y.d;
    r.c = x.c * y.a + x.d * y.c;
    r.d = x.c * y.b + x.d * y.d;
    return r;
}
__device__ inline m2 inv(m2 x)
{
    cd det = x.a * x.d - x.b * x.c;
    cd one = mk(1.0, 0.0);
    cd id = one / det;
    m2 r;
    r.a = x.d * id; r.b = -(x.b * id); r.c = -(x.c * id); r.d = x.a * id;
    return r;
}
// sqrt(det) as the product of the square roots of the eigenvalues (Gouy-continuous branch, R-5)
__device__ inline cd sqrt_det_by_eig(m2 x)
{
    cd mean = 0.5 * (x.a + x.d);
    cd half = 0.5 * (x.a - x.d);
    cd root = csqrt_principal(half * half + x.b * x.c);
    return csqrt_lower(mean + root) * csqrt_lower(mean - root);
}


}  // namespace
