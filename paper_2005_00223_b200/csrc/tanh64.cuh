#pragma once
// fp64 tanh for the FP64 embedding kernels: branch-free (no divergence between the lanes of an MMA fragment), about 24
// fp64-pipe operations (the pipe DMMA shares), absolute error <= 3e-16 (measured against libdevice tanh).
//   tanh(x) = sign(x) (1 - 2 / (e^(2|x|) + 1)),  e^(2a) = 2^n e^r,  n = rint(2a / ln 2),  |r| <= ln 2 / 2,
//   e^r by its Taylor polynomial of degree 13 (remainder (ln2/2)^14 / 14! = 4e-18), 1 / d from a single-precision reciprocal
//   and two Newton steps.  |x| is clamped at 20 (tanh(20) rounds to 1).
__device__ __forceinline__ double dp_tanh64(double x) {
    const double a = fmin(fabs(x), 20.0);
    const double magic = 6755399441055744.0;                 // 1.5 * 2^52: the integer lands in the low mantissa bits
    const double t = fma(a, 2.8853900817779268, magic);      // 2 / ln 2
    const int n = __double2loint(t);
    const double nd = t - magic;
    double r = fma(nd, -6.93147180369123816490e-01, a + a);  // ln 2 = hi + lo, n * hi exact
    r = fma(nd, -1.90821492927058770002e-10, r);
    double p = 1.6059043836821613e-10;                       // 1 / 13!
    p = fma(p, r, 2.08767569878681e-09);                     // 1 / 12!
    p = fma(p, r, 2.505210838544172e-08);                    // 1 / 11!
    p = fma(p, r, 2.755731922398589e-07);                    // 1 / 10!
    p = fma(p, r, 2.7557319223985893e-06);                   // 1 / 9!
    p = fma(p, r, 2.48015873015873e-05);                     // 1 / 8!
    p = fma(p, r, 1.984126984126984e-04);                    // 1 / 7!
    p = fma(p, r, 1.388888888888889e-03);                    // 1 / 6!
    p = fma(p, r, 8.333333333333333e-03);                    // 1 / 5!
    p = fma(p, r, 4.1666666666666664e-02);                   // 1 / 4!
    p = fma(p, r, 1.6666666666666666e-01);                   // 1 / 3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);                                      // e^r in [0.707, 1.415]
    const double e = __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));     // 2^n e^r, n <= 58
    const double d = e + 1.0;
    double q = (double)__frcp_rn((float)d);
    q = fma(q, fma(-d, q, 1.0), q);
    q = fma(q, fma(-d, q, 1.0), q);
    return copysign(fma(-2.0, q, 1.0), x);
}
