// dd.cuh -- double-double (~106 bit) building blocks on the FP64 FMA pipe (D:R11).
// Error-free transformations (TwoSum, FastTwoSum, TwoProd with FMA) written with the explicit
// round-to-nearest intrinsics so that nvcc never contracts or re-associates them.
#pragma once
#include <cuda_runtime.h>

struct dd { double h, l; };
struct cdd { dd re, im; };

#define DD_HD __device__ __forceinline__

DD_HD dd two_sum(double a, double b) {
    double s = __dadd_rn(a, b);
    double bb = __dadd_rn(s, -a);
    double e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
    return {s, e};
}
// requires |a| >= |b| (or a == 0)
DD_HD dd fast_two_sum(double a, double b) {
    double s = __dadd_rn(a, b);
    double e = __dadd_rn(b, -__dadd_rn(s, -a));
    return {s, e};
}
DD_HD dd two_prod(double a, double b) {
    double p = __dmul_rn(a, b);
    double e = __fma_rn(a, b, -p);
    return {p, e};
}
DD_HD dd dd_neg(dd a) { return {-a.h, -a.l}; }
DD_HD dd dd_from(double a) { return {a, 0.0}; }

// accurate dd + dd (relative error ~ 3 * 2^-106)
DD_HD dd dd_add(dd x, dd y) {
    dd s = two_sum(x.h, y.h);
    dd t = two_sum(x.l, y.l);
    double c = __dadd_rn(s.l, t.h);
    dd v = fast_two_sum(s.h, c);
    double w = __dadd_rn(t.l, v.l);
    return fast_two_sum(v.h, w);
}
DD_HD dd dd_sub(dd x, dd y) { return dd_add(x, dd_neg(y)); }
DD_HD dd dd_add_d(dd x, double y) {
    dd s = two_sum(x.h, y);
    double w = __dadd_rn(s.l, x.l);
    return fast_two_sum(s.h, w);
}
// dd * dd (relative error ~ 5 * 2^-106)
DD_HD dd dd_mul(dd x, dd y) {
    dd p = two_prod(x.h, y.h);
    double t = __dmul_rn(x.h, y.l);
    t = __fma_rn(x.l, y.h, t);
    t = __fma_rn(x.l, y.l, t);
    double c = __dadd_rn(p.l, t);
    return fast_two_sum(p.h, c);
}
DD_HD dd dd_mul_d(dd x, double y) {
    dd p = two_prod(x.h, y);
    double c = __fma_rn(x.l, y, p.l);
    return fast_two_sum(p.h, c);
}
// x * 2^k, exact
DD_HD dd dd_scale2(dd x, double pow2) { return {__dmul_rn(x.h, pow2), __dmul_rn(x.l, pow2)}; }
// a*b + c*d with one renormalisation (sgn = +1 or -1 applied to the second product)
DD_HD dd dd_dot2(dd a, dd b, dd c, dd d, double sgn) {
    dd p = two_prod(a.h, b.h);
    dd q = two_prod(c.h, sgn * d.h);
    double t = __fma_rn(a.h, b.l, p.l);
    t = __fma_rn(a.l, b.h, t);
    t = __fma_rn(a.l, b.l, t);
    double u = __fma_rn(c.h, sgn * d.l, q.l);
    u = __fma_rn(c.l, sgn * d.h, u);
    u = __fma_rn(c.l, sgn * d.l, u);
    dd s = two_sum(p.h, q.h);
    double w = __dadd_rn(s.l, __dadd_rn(t, u));
    return fast_two_sum(s.h, w);
}
DD_HD cdd cdd_mul(cdd a, cdd b) {
    cdd r;
    r.re = dd_dot2(a.re, b.re, a.im, b.im, -1.0);
    r.im = dd_dot2(a.re, b.im, a.im, b.re, 1.0);
    return r;
}
DD_HD cdd cdd_conj(cdd a) { return {a.re, dd_neg(a.im)}; }
DD_HD dd dd_div_d(dd x, double y) {          // dd / double
    double q1 = __ddiv_rn(x.h, y);
    double r = __fma_rn(-q1, y, x.h);         // exact remainder
    double q2 = __ddiv_rn(__dadd_rn(r, x.l), y);
    return fast_two_sum(q1, q2);
}
DD_HD dd dd_sqrt(dd x) {                      // x >= 0
    if (x.h <= 0.0) return {0.0, 0.0};
    double s = __dsqrt_rn(x.h);
    dd p = two_prod(s, s);
    double r = __dadd_rn(__dadd_rn(__dadd_rn(x.h, -p.h), -p.l), x.l);
    double c = __ddiv_rn(r, __dmul_rn(2.0, s));
    return fast_two_sum(s, c);
}
DD_HD bool dd_less(dd a, dd b) { return a.h < b.h || (a.h == b.h && a.l < b.l); }
// dd / dd (relative error ~ 2^-103): three quotient digits with exact dd remainders
DD_HD dd dd_div(dd x, dd y) {
    double q1 = __ddiv_rn(x.h, y.h);
    dd r = dd_sub(x, dd_mul_d(y, q1));
    double q2 = __ddiv_rn(r.h, y.h);
    r = dd_sub(r, dd_mul_d(y, q2));
    double q3 = __ddiv_rn(r.h, y.h);
    dd q = fast_two_sum(q1, q2);
    return dd_add_d(q, q3);
}
