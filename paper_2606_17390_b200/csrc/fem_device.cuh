// Small device helpers shared by the CUDA translation units of libfem_b200.so (fem_assemble.cu, fem_sens.cu).
#pragma once

// Branch-free reciprocal and reciprocal square root: the hardware approximation (20+ good bits) refined by ONE third-order
// step (error e -> e^3 < 2^-60, i.e. ~1 ulp after rounding): three / four dependent FP64 operations instead of the four / six
// of two Newton steps.  No special-case paths: callers guarantee normal, positive (rsqrt) arguments.
__device__ __forceinline__ double frcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);          // 1/x = r / (1 - e) = r (1 + e + e^2 + ...)
    const double t = fma(e, e, e);
    return fma(r, t, r);
}
__device__ __forceinline__ double frsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double xy = x * y;
    const double e = fma(-xy, y, 1.0);         // x^-1/2 = y (1 - e)^-1/2 = y (1 + e/2 + 3 e^2/8 + ...)
    const double p = fma(0.375, e, 0.5), ye = y * e;
    return fma(ye, p, y);
}

// sum_{k=0..10} x^k / (2k+1) by Estrin's scheme (dependency depth 4 instead of 10): atanh(w)/w with x = w^2.
// Remainder x^11/23: below 2^-56 for x <= 0.0295 (w <= 0.1716, i.e. arguments of ln within [1/sqrt2, sqrt2]).
__device__ __forceinline__ double atanh_poly(double x) {
    const double x2 = x * x, x4 = x2 * x2, x8 = x4 * x4;
    const double p01 = fma(1.0 / 3.0, x, 1.0), p23 = fma(1.0 / 7.0, x, 1.0 / 5.0), p45 = fma(1.0 / 11.0, x, 1.0 / 9.0),
                 p67 = fma(1.0 / 15.0, x, 1.0 / 13.0), p89 = fma(1.0 / 19.0, x, 1.0 / 17.0);
    const double q0 = fma(p23, x2, p01), q1 = fma(p67, x2, p45), q2 = fma(1.0 / 21.0, x2, p89);
    return fma(q2, x8, fma(q1, x4, q0));
}
// ln x for normal positive x: x = 2^k m, m in [1/sqrt2, sqrt2), ln m = 2 atanh((m-1)/(m+1)).  ~1 ulp; no special cases.
__device__ __forceinline__ double flog(double x) {
    int hi = __double2hiint(x);
    const int lo = __double2loint(x);
    int k = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;                  // m in [1, 2)
    const bool up = hi > 0x3ff6a09e;                      // m > sqrt2: use m/2
    hi = up ? hi - 0x00100000 : hi;
    k = up ? k + 1 : k;
    const double m = __hiloint2double(hi, lo);
    const double w = (m - 1.0) * frcp(m + 1.0);
    const double t = 2.0 * w * atanh_poly(w * w);
    const double kd = (double)k;
    return fma(kd, 6.93147180369123816490e-01, fma(kd, 1.90821492927058770002e-10, t));
}
// e^z for |z| < 700: z = n ln2 + r, |r| <= ln2/2, degree-13 Taylor polynomial by Estrin (remainder 4e-18), scaled by 2^n.
__device__ __forceinline__ double fexp(double z) {
    const double MAGIC = 6755399441055744.0;               // 1.5 * 2^52: the low word of z*log2e + MAGIC is rint(z*log2e)
    double t = fma(z, 1.4426950408889634074, MAGIC);
    const int n = __double2loint(t);
    t -= MAGIC;
    double r = fma(t, -6.93147180369123816490e-01, z);
    r = fma(t, -1.90821492927058770002e-10, r);
    const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
    const double p01 = 1.0 + r, p23 = fma(1.0 / 6.0, r, 0.5), p45 = fma(1.0 / 120.0, r, 1.0 / 24.0),
                 p67 = fma(1.0 / 5040.0, r, 1.0 / 720.0), p89 = fma(1.0 / 362880.0, r, 1.0 / 40320.0),
                 pab = fma(1.0 / 39916800.0, r, 1.0 / 3628800.0), pcd = fma(1.0 / 6227020800.0, r, 1.0 / 479001600.0);
    const double q0 = fma(p23, r2, p01), q1 = fma(p67, r2, p45), q2 = fma(pab, r2, p89);
    const double s = fma(fma(pcd, r4, q2), r8, fma(q1, r4, q0));
    return __hiloint2double(__double2hiint(s) + (n << 20), __double2loint(s));
}

// One cyclic-Jacobi rotation annihilating a_pq of a symmetric 3x3 (r = third index); V columns p,q updated.
__device__ __forceinline__ void jacobi_rot(double &app, double &aqq, double &apq, double &arp, double &arq, double &v0p,
                                           double &v0q, double &v1p, double &v1q, double &v2p, double &v2q) {
    // cos^2 = (1 + |d|/r)/2 with r = hypot(d, 2 a_pq); sin = sgn(d) a_pq / (r cos); tan = sin / cos.  Two rsqrt, no division.
    const double d = aqq - app;
    const double r2 = fma(d, d, 4.0 * apq * apq);
    const bool ok = r2 > 1e-280;                     // d = a_pq = 0 (e.g. C = I exactly): identity rotation
    const double ir = frsqrt(ok ? r2 : 1.0);         // branch-free: the rotations of a sweep stay in one basic block
    const double c2 = ok ? fma(0.5 * fabs(d), ir, 0.5) : 1.0;
    const double ic = frsqrt(c2);
    const double c = c2 * ic;
    const double s = ((d < 0.0) ? -apq : apq) * ir * ic;   // sgn(d) a_pq / (r c); d = 0 counts as positive
    const double t = s * ic;
    app = fma(-t, apq, app); aqq = fma(t, apq, aqq); apq = 0.0;
    double x = arp, y = arq;
    arp = c * x - s * y; arq = s * x + c * y;
    x = v0p; y = v0q; v0p = c * x - s * y; v0q = s * x + c * y;
    x = v1p; y = v1q; v1p = c * x - s * y; v1q = s * x + c * y;
    x = v2p; y = v2q; v2p = c * x - s * y; v2q = s * x + c * y;
}

