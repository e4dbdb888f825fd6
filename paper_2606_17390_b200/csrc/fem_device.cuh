// Small device helpers shared by the CUDA translation units of libfem_b200.so (fem_assemble.cu, fem_sens.cu).
#pragma once

// Branch-free reciprocal and reciprocal square root: the hardware approximation (relative error 2^-23) refined by two
// Newton steps (2^-46, 2^-92 -> ~1 ulp).  No special-case paths: callers guarantee normal, positive (rsqrt) arguments.
__device__ __forceinline__ double frcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}
__device__ __forceinline__ double frsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double h = 0.5 * x;
    double e = fma(-h * y, y, 0.5);
    y = fma(y, e, y);
    e = fma(-h * y, y, 0.5);
    return fma(y, e, y);
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

