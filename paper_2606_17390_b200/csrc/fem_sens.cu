// fem_assemble_vjp: vector-Jacobian products of one pass of the element path.
//
// The pass is the map (u, hist_in, theta) -> (R, hist_out) of Eq.(34)-(35) PAPER.md:253-257 with Alg. C1 :889-918 at every
// Gauss point.  Alg. 1 needs, for an adjoint vector lam (Eq.(51) :366) and a cotangent mu on hist_out,
//     g_u       = (dR/du)^T lam       + (dhist_out/du)^T mu
//     g_hist_in = (dR/dhist_in)^T lam + (dhist_out/dhist_in)^T mu
//     g_mat     = (dR/dtheta)^T lam   + (dhist_out/dtheta)^T mu            (Eq.(49) :355)
// The paper gets them from JAX reverse mode through the implicit layer of App. D (:1002-1019); here the reverse pass is
// written out by hand, one thread per Gauss point (8 lanes per element, 16 elements per CTA):
//   forward  : G = grad_0 N (Eq.(28) :220) rotated into the material frame (G' = G Theta, F' = F Theta, Eq.(A1) :774, so the
//              Hill tensor keeps its sparse local form Eq.(A2) :779), C' = F'^T F', cyclic Jacobi, eps = sum 1/2 ln(lam_a) n_a(x)n_a
//              (Eq.(4)-(5) :92-96), trial stress Eq.(16) :160, return map Eq.(19)-(24) :176-196 as one scalar equation
//              sigma_y(alpha)/phi(kappa) - 1 = 0 with T = (E^-1 + kappa H)^-1 : (eps - eps_p_n), kappa = dgam/sigma_y
//              (a 3x3 solve + 3 scalars per iterate), S = P_L : T in the eigenbasis of C
//   reverse  : Pbar = w lam^T G' (Eq.(35) :257), P = F S (Eq.(26) :208), dS = P_L:dT + (T:L_L):dC/2 (Eq.(25) :204) with first and
//              second divided differences of 1/2 ln, the transposed App. D solve J_y^T w = ybar on y = [T, alpha, dgam]
//              reduced by hand to Xi = (E^-1 + dgam dN/dT)^-1 (Sherman-Morrison on D - kappa N(x)N) and one scalar w_f,
//              then zbar = -(dG/dz)^T w for z = (eps, eps_p_n, alpha_n, theta), d eps = P_L:dC/2, C = F^T F, F = I + u^T G.
// theta = (E, nu, r11, r22, r33, r12, r23, r13, h0, h1, h2): positions 0-7 and 9-11 of the 16-double record; the law
// switch and the orientation quaternion are not differentiated (their entries of g_mat are 0).  Hill-48; standard element and
// F-bar (template FBAR = 1: Fbar = (Jbar/J)^(1/3) F, Eq.(31)-(32) :237-243, Jbar and the back-propagated sum by 8-lane butterflies).
// Sums are taken in a fixed order (per node: ascending element id; uniform material: fixed two-level tree), no atomics.
// Nothing here is shared with oracle/.
#include "fem_internal.h"
#include "fem_device.cuh"
#include <math.h>

#define SW23 0.81649658092772603273   // W = sqrt(2/3)
#define SEL 16                        // elements per CTA
#define STHREADS (8 * SEL)
#define NTHETA 11
// Phase barriers keep the warps of a CTA in the same code region so that they share instruction-cache lines (the pass is
// ~7,000 straight-line instructions per warp; instruction fetch was the top stall without them).
#ifndef SENS_PS_MASK
#define SENS_PS_MASK 0x0a   // re-swept after the round-2 rework: 0x0a 2.62, 0x1f 2.72, 0x0f 2.67, none 2.82 ms
#endif
#define SENS_SYNC(n) do { if ((SENS_PS_MASK >> (n)) & 1) __syncthreads(); } while (0)
#ifndef SENS_CTAS
#define SENS_CTAS 3                   // CTAs per SM the register allocation aims at
#endif

__device__ constexpr int S_THETA_IDX[NTHETA] = {0, 1, 2, 3, 4, 5, 6, 7, 9, 10, 11};
__device__ constexpr double S_XI[8][3] = {{-1, -1, -1}, {1, -1, -1}, {1, 1, -1}, {-1, 1, -1},
                                          {-1, -1, 1},  {1, -1, 1},  {1, 1, 1},  {-1, 1, 1}};

// symmetric tensors as 6 tensor components (11,22,33,12,23,13); full inner product A:B
__device__ __forceinline__ double dot6(const double a[6], const double b[6]) {
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2] + 2.0 * (a[3] * b[3] + a[4] * b[4] + a[5] * b[5]);
}
__device__ __forceinline__ void to33(const double a[6], double A[3][3]) {
    A[0][0] = a[0]; A[1][1] = a[1]; A[2][2] = a[2];
    A[0][1] = A[1][0] = a[3]; A[1][2] = A[2][1] = a[4]; A[0][2] = A[2][0] = a[5];
}
// B = Q^T A Q (TR = 0) or Q A Q^T (TR = 1) for symmetric A, both as 6 components
template <int TR>
__device__ __forceinline__ void rot6(const double Q[3][3], const double a[6], double b[6]) {
    double A[3][3], T[3][3];
    to33(a, A);
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const double q0 = TR ? Q[j][0] : Q[0][j], q1 = TR ? Q[j][1] : Q[1][j], q2 = TR ? Q[j][2] : Q[2][j];
            T[i][j] = A[i][0] * q0 + A[i][1] * q1 + A[i][2] * q2;
        }
    constexpr int PI[6] = {0, 1, 2, 0, 1, 0}, PJ[6] = {0, 1, 2, 1, 2, 2};
#pragma unroll
    for (int k = 0; k < 6; k++) {
        const int i = PI[k], j = PJ[k];
        const double q0 = TR ? Q[i][0] : Q[0][i], q1 = TR ? Q[i][1] : Q[1][i], q2 = TR ? Q[i][2] : Q[2][i];
        b[k] = q0 * T[0][j] + q1 * T[1][j] + q2 * T[2][j];
    }
}

struct SMat {
    double E, iE, nu, mu2, imu2, lam, law, h0, h1, h2;
    double p[9];        // Hill coefficients p1..p9 of Eq.(A3)-(A5) :784-801 in the local (material) frame
};

// H : a  (Eq.(A2) :779 in tensor components: H1212 = p7/2, so (H:a)_12 = p7 a_12)
__device__ __forceinline__ void applyH(const SMat &m, const double a[6], double b[6]) {
    b[0] = m.p[0] * a[0] + m.p[3] * a[1] + m.p[5] * a[2];
    b[1] = m.p[3] * a[0] + m.p[1] * a[1] + m.p[4] * a[2];
    b[2] = m.p[5] * a[0] + m.p[4] * a[1] + m.p[2] * a[2];
    b[3] = m.p[6] * a[3]; b[4] = m.p[7] * a[4]; b[5] = m.p[8] * a[5];
}
// E : a  (Eq.(8) :110, isotropic)
__device__ __forceinline__ void applyE(const SMat &m, const double a[6], double b[6]) {
    const double tr = m.lam * (a[0] + a[1] + a[2]);
#pragma unroll
    for (int i = 0; i < 3; i++) b[i] = m.mu2 * a[i] + tr;
#pragma unroll
    for (int i = 3; i < 6; i++) b[i] = m.mu2 * a[i];
}
__device__ __forceinline__ void applyEinv(const SMat &m, const double a[6], double b[6]) {
    const double s = m.nu * (a[0] + a[1] + a[2]);
#pragma unroll
    for (int i = 0; i < 3; i++) b[i] = ((1.0 + m.nu) * a[i] - s) * m.iE;
#pragma unroll
    for (int i = 3; i < 6; i++) b[i] = a[i] * m.imu2;
}
// D = E^-1 + kappa H : normal block 3x3 (symmetric, inverted once per kappa) + three shear scalars
struct SDinv { double n[6]; double s[3]; };   // inverse normal block as (11,22,33,12,23,13), inverse shear scalars
__device__ __forceinline__ void makeDinv(const SMat &m, double kap, SDinv &D) {
    const double ie = m.iE, o = -m.nu * ie;
    const double a = ie + kap * m.p[0], b = ie + kap * m.p[1], c = ie + kap * m.p[2];
    const double d = o + kap * m.p[3], e = o + kap * m.p[4], f = o + kap * m.p[5];   // 12, 23, 13
    const double c00 = b * c - e * e, c01 = f * e - d * c, c02 = d * e - f * b;
    const double idet = frcp(a * c00 + d * c01 + f * c02);
    D.n[0] = c00 * idet; D.n[3] = c01 * idet; D.n[5] = c02 * idet;
    D.n[1] = (a * c - f * f) * idet; D.n[4] = (d * f - a * e) * idet; D.n[2] = (a * b - d * d) * idet;
#pragma unroll
    for (int k = 0; k < 3; k++) D.s[k] = frcp(m.imu2 + kap * m.p[6 + k]);
}
__device__ __forceinline__ void applyDinv(const SDinv &D, const double a[6], double b[6]) {
    b[0] = D.n[0] * a[0] + D.n[3] * a[1] + D.n[5] * a[2];
    b[1] = D.n[3] * a[0] + D.n[1] * a[1] + D.n[4] * a[2];
    b[2] = D.n[5] * a[0] + D.n[4] * a[1] + D.n[2] * a[2];
    b[3] = D.s[0] * a[3]; b[4] = D.s[1] * a[4]; b[5] = D.s[2] * a[5];
}

// sigma_flow and d sigma_flow/d alpha: Voce Eq.(10) :121, Swift (BASELINE configs).  aux = (exp(-h2 alpha), -) for Voce,
// ((h1+alpha)^h2, ln(h1+alpha)) for Swift: what flow_dh needs at the same alpha.
__device__ __forceinline__ void flow2x(const SMat &m, double alpha, double &sf, double &dsf, double aux[2]) {
    if (m.law == 0.0) {
        const double e = fexp(-m.h2 * alpha);
        sf = m.h0 + m.h1 * (1.0 - e); dsf = m.h1 * m.h2 * e;
        aux[0] = e; aux[1] = 0.0;
    } else {
        const double b = m.h1 + alpha, lb = flog(b), pw = fexp(m.h2 * lb);
        sf = m.h0 * pw; dsf = m.h0 * m.h2 * pw * frcp(b);
        aux[0] = pw; aux[1] = lb;
    }
}
__device__ __forceinline__ void flow2(const SMat &m, double alpha, double &sf, double &dsf) {
    double aux[2];
    flow2x(m, alpha, sf, dsf, aux);
}
// d sigma_flow/d(h0,h1,h2) at the alpha of the flow2x call that produced (dsf, aux)
__device__ __forceinline__ void flow_dh(const SMat &m, double alpha, double dsf, const double aux[2], double dh[3]) {
    if (m.law == 0.0) {
        const double e = aux[0];
        dh[0] = 1.0; dh[1] = 1.0 - e; dh[2] = m.h1 * alpha * e;
    } else {
        dh[0] = aux[0]; dh[1] = dsf; dh[2] = m.h0 * aux[0] * aux[1];   // d/dh1 of h0 (h1+alpha)^h2 equals d/dalpha
    }
}

// d(x:H:t)/d s_k, s_k = 1/r_k^2 (Eq.(A3)-(A5): p1 = 2/3 s11, p4 = (p3-p1-p2)/2, p5 = (p1-p2-p3)/2, p6 = (p2-p1-p3)/2, p7 = s12, ...)
__device__ __forceinline__ void hill_bilinear_ds(const double x[6], const double t[6], double B[6]) {
    const double d12 = x[0] * t[1] + x[1] * t[0], d23 = x[1] * t[2] + x[2] * t[1], d13 = x[0] * t[2] + x[2] * t[0];
    B[0] = (2.0 / 3.0) * (x[0] * t[0] - 0.5 * d12 + 0.5 * d23 - 0.5 * d13);
    B[1] = (2.0 / 3.0) * (x[1] * t[1] - 0.5 * d12 - 0.5 * d23 + 0.5 * d13);
    B[2] = (2.0 / 3.0) * (x[2] * t[2] + 0.5 * d12 - 0.5 * d23 - 0.5 * d13);
    B[3] = 2.0 * x[3] * t[3]; B[4] = 2.0 * x[4] * t[4]; B[5] = 2.0 * x[5] * t[5];
}

// First divided difference of g = 1/2 ln between eigenvalues a, b with ga = g(a), gb = g(b):
// atanh(w)/w / (a+b), w = (a-b)/(a+b), by its series for |w| < 0.15 (remainder < 1e-19), else (ga - gb)/(a - b)
__device__ __forceinline__ double g_dd1(double a, double b, double ga, double gb) {
    const double is = frcp(a + b), w = (a - b) * is, w2 = w * w;
    const double s = atanh_poly(w2);
    const double big = (ga - gb) * frcp((w2 < 0.0225) ? 1.0 : a - b);
    return (w2 < 0.0225) ? s * is : big;
}
// Second divided difference of g = 1/2 ln over the nodes (x0, x1, x2) (coincident nodes allowed).  d02 = g[x0,x1], d12 =
// g[x1,x2] are the first divided differences on either side of the middle node x1, x0 and x2 the two nodes farthest apart.
// Nodes within 2e-3 (relative) of each other: series about the mean in the complete homogeneous polynomials h_k of the
// centred nodes, g[x0,x1,x2] = 1/(2 m^2) sum_{n>=2} (-1)^(n-1)/n h_{n-2}, h_k = -e2 h_{k-2} + e3 h_{k-3} (e1 = 0), through h_5
// (remainder < 1e-17); farther apart the recursion (g[x0,x1] - g[x1,x2])/(x0 - x2), whose cancellation costs 2 eps m/gap <= 1e-13.
__device__ __forceinline__ double g_dd2(double x0, double x1, double x2, double g01, double g12) {
    const double m = (x0 + x1 + x2) * (1.0 / 3.0), im = frcp(m);
    const double d0 = (x0 - m) * im, d1 = (x1 - m) * im, d2 = (x2 - m) * im;
    const double sp = fmax(fabs(d0), fmax(fabs(d1), fabs(d2)));
    const double e2 = d0 * d1 + d1 * d2 + d0 * d2, e3 = d0 * d1 * d2;
    // h0 = 1, h1 = 0, h2 = -e2, h3 = e3, h4 = e2^2, h5 = -2 e2 e3
    const double ser = -0.5 + e2 * 0.25 + e3 * 0.2 - e2 * e2 * (1.0 / 6.0) - 2.0 * e2 * e3 * (1.0 / 7.0);
    const bool close = sp < 2e-3;
    const double rec = (g01 - g12) * frcp(close ? 1.0 : x0 - x2);
    return close ? 0.5 * im * im * ser : rec;
}

template <int FBAR>
__global__ void __launch_bounds__(STHREADS, SENS_CTAS)
k_sens_point(long long n_elems, const double *__restrict__ coords, const int *__restrict__ conn, const int *__restrict__ eslot,
             const double *__restrict__ u, const double *__restrict__ hist_in, const double *__restrict__ mat, long long n_mat,
             const double *__restrict__ lamv, const double *__restrict__ muv,
             double *__restrict__ gu_scr /*[8 n_elems][3] incidence order, may be null*/,
             double *__restrict__ g_hist /*may be null*/, double *__restrict__ g_mat /*per element, may be null*/,
             double *__restrict__ part /*[gridDim.x][NTHETA] uniform material, may be null*/) {
    __shared__ double sX[SEL][8][3], sU[SEL][8][3], sL[SEL][8][3];
    __shared__ double sGu[SEL][8][25];      // per thread: G' (24 doubles, odd stride) during the pass, then its ubar contributions
    __shared__ double sTh[STHREADS][NTHETA];
    const int tid = threadIdx.x, el = tid >> 3, q = tid & 7;
    const long long e_raw = (long long)blockIdx.x * SEL + el;
    const bool live = e_raw < n_elems;
    const long long e = live ? e_raw : n_elems - 1;   // threads past the end redo the last element (no output): every thread
                                                      // reaches the phase barriers below
    // the material gradient of this point goes straight to its row of sTh (it is only read after the pass)
    double *const gth = &sTh[tid][0];
#pragma unroll
    for (int k = 0; k < NTHETA; k++) gth[k] = 0.0;
    {
        const int nd = conn[e * 8 + q];
#pragma unroll
        for (int i = 0; i < 3; i++) {
            sX[el][q][i] = coords[3LL * nd + i];
            sU[el][q][i] = u[3LL * nd + i];
            sL[el][q][i] = lamv ? lamv[3LL * nd + i] : 0.0;
        }
    }
    __syncthreads();
    {
        double *Gs = &sGu[el][q][0];
        // ---- material record
        const double *mp = mat + (n_mat == 1 ? 0 : e) * FEM_NPAR;
        SMat m;
        m.E = mp[0]; m.nu = mp[1]; m.iE = frcp(m.E); m.mu2 = m.E * frcp(1.0 + m.nu); m.imu2 = (1.0 + m.nu) * m.iE;
        m.lam = m.E * m.nu * frcp((1.0 + m.nu) * (1.0 - 2.0 * m.nu));
        m.law = mp[8]; m.h0 = mp[9]; m.h1 = mp[10]; m.h2 = mp[11];
        {
            const double s0 = frcp(mp[2] * mp[2]), s1 = frcp(mp[3] * mp[3]), s2 = frcp(mp[4] * mp[4]);
            m.p[0] = (2.0 / 3.0) * s0; m.p[1] = (2.0 / 3.0) * s1; m.p[2] = (2.0 / 3.0) * s2;
            m.p[6] = frcp(mp[5] * mp[5]); m.p[7] = frcp(mp[6] * mp[6]); m.p[8] = frcp(mp[7] * mp[7]);
            m.p[3] = 0.5 * (m.p[2] - m.p[0] - m.p[1]); m.p[4] = 0.5 * (m.p[0] - m.p[1] - m.p[2]); m.p[5] = 0.5 * (m.p[1] - m.p[0] - m.p[2]);
        }
        double Th[3][3];
        {
            const double qn = frsqrt(mp[12] * mp[12] + mp[13] * mp[13] + mp[14] * mp[14] + mp[15] * mp[15]);
            const double w = mp[12] * qn, x = mp[13] * qn, y = mp[14] * qn, z = mp[15] * qn;
            Th[0][0] = 1 - 2 * (y * y + z * z); Th[0][1] = 2 * (x * y - w * z);     Th[0][2] = 2 * (x * z + w * y);
            Th[1][0] = 2 * (x * y + w * z);     Th[1][1] = 1 - 2 * (x * x + z * z); Th[1][2] = 2 * (y * z - w * x);
            Th[2][0] = 2 * (x * z - w * y);     Th[2][1] = 2 * (y * z + w * x);     Th[2][2] = 1 - 2 * (x * x + y * y);
        }
        // ---- shape gradients at Gauss point q (Eq.(28) :220), rotated: G'_IJ = G_IK Theta_KJ, kept in shared memory
        const double gp = 0.57735026918962576451;
        const double xi0 = (q & 1) ? gp : -gp, xi1 = (q & 2) ? gp : -gp, xi2 = (q & 4) ? gp : -gp;
        double Jr[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
        for (int I = 0; I < 8; I++) {
            const double a = 1.0 + xi0 * S_XI[I][0], b = 1.0 + xi1 * S_XI[I][1], c = 1.0 + xi2 * S_XI[I][2];
            const double dn0 = 0.125 * S_XI[I][0] * b * c, dn1 = 0.125 * a * S_XI[I][1] * c, dn2 = 0.125 * a * b * S_XI[I][2];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                const double x = sX[el][I][i];
                Jr[i][0] = fma(x, dn0, Jr[i][0]); Jr[i][1] = fma(x, dn1, Jr[i][1]); Jr[i][2] = fma(x, dn2, Jr[i][2]);
            }
        }
        double wq;
        double F[3][3];
        {
            double Ji[3][3];
            Ji[0][0] = Jr[1][1] * Jr[2][2] - Jr[1][2] * Jr[2][1]; Ji[0][1] = Jr[0][2] * Jr[2][1] - Jr[0][1] * Jr[2][2]; Ji[0][2] = Jr[0][1] * Jr[1][2] - Jr[0][2] * Jr[1][1];
            Ji[1][0] = Jr[1][2] * Jr[2][0] - Jr[1][0] * Jr[2][2]; Ji[1][1] = Jr[0][0] * Jr[2][2] - Jr[0][2] * Jr[2][0]; Ji[1][2] = Jr[0][2] * Jr[1][0] - Jr[0][0] * Jr[1][2];
            Ji[2][0] = Jr[1][0] * Jr[2][1] - Jr[1][1] * Jr[2][0]; Ji[2][1] = Jr[0][1] * Jr[2][0] - Jr[0][0] * Jr[2][1]; Ji[2][2] = Jr[0][0] * Jr[1][1] - Jr[0][1] * Jr[1][0];
            wq = Jr[0][0] * Ji[0][0] + Jr[0][1] * Ji[1][0] + Jr[0][2] * Ji[2][0];   // det J_ref, weights 1
            const double iw = frcp(wq);
            double JT[3][3];   // J_ref^-1 Theta
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) JT[i][j] = (Ji[i][0] * Th[0][j] + Ji[i][1] * Th[1][j] + Ji[i][2] * Th[2][j]) * iw;
            // F' = F Theta = Theta + u^T G'  (Eq.(30) :228)
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) F[i][j] = Th[i][j];
#pragma unroll
            for (int I = 0; I < 8; I++) {
                const double a = 1.0 + xi0 * S_XI[I][0], b = 1.0 + xi1 * S_XI[I][1], c = 1.0 + xi2 * S_XI[I][2];
                const double dn0 = 0.125 * S_XI[I][0] * b * c, dn1 = 0.125 * a * S_XI[I][1] * c, dn2 = 0.125 * a * b * S_XI[I][2];
                double g[3];
#pragma unroll
                for (int j = 0; j < 3; j++) { g[j] = dn0 * JT[0][j] + dn1 * JT[1][j] + dn2 * JT[2][j]; Gs[3 * I + j] = g[j]; }
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    const double ui = sU[el][I][i];
                    F[i][0] = fma(ui, g[0], F[i][0]); F[i][1] = fma(ui, g[1], F[i][1]); F[i][2] = fma(ui, g[2], F[i][2]);
                }
            }
        }
        // ---- F-bar (Eq.(31)-(32) :237-243, reading G12): Fbar = (Jbar/J)^(1/3) F, Jbar = sum_q w_q J_q / V over the element's 8 lanes
        double fb_c = 1.0, fb_J = 1.0, fb_Jbar = 1.0, fb_wJV = 0.0;
        if (FBAR) {
            fb_J = F[0][0] * (F[1][1] * F[2][2] - F[1][2] * F[2][1]) - F[0][1] * (F[1][0] * F[2][2] - F[1][2] * F[2][0]) +
                   F[0][2] * (F[1][0] * F[2][1] - F[1][1] * F[2][0]);
            double V = wq, SJ = wq * fb_J;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) { V += __shfl_xor_sync(0xffffffffu, V, o); SJ += __shfl_xor_sync(0xffffffffu, SJ, o); }
            fb_Jbar = SJ / V;
            fb_wJV = wq * fb_J / V;
            fb_c = cbrt(fb_Jbar / fb_J);
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) F[i][j] *= fb_c;
        }
        SENS_SYNC(5);
        // ---- C' = F'^T F', cyclic Jacobi (4 sweeps, as in k_element), Hencky strain in the material frame (Eq.(4)-(5) :92-96, reading G1)
        double R[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}}, lm[3], gl[3];
        {
            double c00 = F[0][0] * F[0][0] + F[1][0] * F[1][0] + F[2][0] * F[2][0], c11 = F[0][1] * F[0][1] + F[1][1] * F[1][1] + F[2][1] * F[2][1];
            double c22 = F[0][2] * F[0][2] + F[1][2] * F[1][2] + F[2][2] * F[2][2], c01 = F[0][0] * F[0][1] + F[1][0] * F[1][1] + F[2][0] * F[2][1];
            double c12 = F[0][1] * F[0][2] + F[1][1] * F[1][2] + F[2][1] * F[2][2], c02 = F[0][0] * F[0][2] + F[1][0] * F[1][2] + F[2][0] * F[2][2];
#pragma unroll 1
            for (int sweep = 0; sweep < 4; sweep++) {
                jacobi_rot(c00, c11, c01, c02, c12, R[0][0], R[0][1], R[1][0], R[1][1], R[2][0], R[2][1]);
                jacobi_rot(c00, c22, c02, c01, c12, R[0][0], R[0][2], R[1][0], R[1][2], R[2][0], R[2][2]);
                jacobi_rot(c11, c22, c12, c01, c02, R[0][1], R[0][2], R[1][1], R[1][2], R[2][1], R[2][2]);
            }
            lm[0] = c00; lm[1] = c11; lm[2] = c22;
        }
#pragma unroll
        for (int a = 0; a < 3; a++) gl[a] = 0.5 * flog(lm[a]);
        double ee[6];
        {
            const double eh[6] = {gl[0], gl[1], gl[2], 0, 0, 0};
            rot6<1>(R, eh, ee);
        }
        // ---- history in, rotated into the material frame; elastic trial strain
        const double *hp = hist_in + (e * 8 + q) * 7;
        const double alpha_n = hp[6];
        {
            const double epn_g[6] = {hp[0], hp[1], hp[2], hp[3], hp[4], hp[5]};
            double epn[6];
            rot6<0>(Th, epn_g, epn);
#pragma unroll
            for (int k = 0; k < 6; k++) ee[k] -= epn[k];
        }
        SENS_SYNC(0);
        // ---- trial state (Eq.(16)-(17) :160-165)
        double T[6], HT[6], N[6];
        applyE(m, ee, T);
        applyH(m, T, HT);
        double phi; { const double p2 = fmax(dot6(T, HT), 0.0); phi = (p2 > 0.0) ? p2 * frsqrt(p2) : 0.0; }
        double sf, dsf, faux[2] = {0.0, 0.0};
        flow2(m, alpha_n, sf, dsf);
        double dgam = 0.0, alpha = alpha_n, kap = 0.0;
        const bool plastic = phi - SW23 * sf > 0.0;
        SDinv D;
        if (plastic) {
            // ---- return map: f(dgam) = sigma_y(alpha)/phi(kappa) - 1 = 0, monotone increasing, f(0) < 0
            double lo = 0.0, hi = -1.0;
#pragma unroll 1
            for (int it = 0; it < 60; it++) {
                alpha = alpha_n + SW23 * dgam;
                flow2(m, alpha, sf, dsf);
                const double sy = SW23 * sf, dsy = (2.0 / 3.0) * dsf, isy = frcp(sy);   // d sigma_y / d dgam = W^2 sigma_flow'
                kap = dgam * isy;
                makeDinv(m, kap, D);
                applyDinv(D, ee, T);
                applyH(m, T, HT);
                const double ph2 = dot6(T, HT), iphi = frsqrt(ph2);
                phi = ph2 * iphi;
                double mN[6];
                applyDinv(D, HT, mN);
                const double a_ = dot6(HT, mN) * iphi * iphi;   // N : D^-1 : N
                const double f = sy * iphi - 1.0;
                const double dk = (sy - dgam * dsy) * isy * isy;
                const double df = dsy * iphi + (sy * iphi) * a_ * dk;
                if (fabs(f) <= 1e-15) break;
                if (f < 0.0) lo = dgam; else hi = dgam;
                double nx = dgam - f * frcp(df);
                const bool inside = (nx > lo) && !(hi > 0.0 && !(nx < hi));
                if (!inside) nx = (hi > 0.0) ? 0.5 * (lo + hi) : 2.0 * dgam + 1e-6;
                // f is smooth and monotone: once |f| <= 1e-9 the Newton step just computed lands on the root to round-off
                // (error ~ f^2), so it is applied and the loop ends without a pass that only confirms it
                const bool done = (inside && fabs(f) <= 1e-9) || fabs(nx - dgam) <= 4e-16 * nx;
                dgam = nx;
                if (done) break;
            }
            // state at the solution
            alpha = alpha_n + SW23 * dgam;
            flow2x(m, alpha, sf, dsf, faux);
            kap = dgam * frcp(SW23 * sf);
            makeDinv(m, kap, D);
            applyDinv(D, ee, T);
            applyH(m, T, HT);
            const double ph2 = dot6(T, HT), iphi = frsqrt(ph2);
            phi = ph2 * iphi;
#pragma unroll
            for (int k = 0; k < 6; k++) N[k] = HT[k] * iphi;
            // kappa = dgam / phi with phi = sigma_y at the root: D above is already E^-1 + kappa H
        } else {
#pragma unroll
            for (int k = 0; k < 6; k++) N[k] = 0.0;
        }
        SENS_SYNC(1);
        // ---- divided differences of g = 1/2 ln at the eigenvalues of C
        double g1[3][3], g2[3][3][3];
        {
            const double il0 = frcp(lm[0]), il1 = frcp(lm[1]), il2 = frcp(lm[2]);
            g1[0][0] = 0.5 * il0; g1[1][1] = 0.5 * il1; g1[2][2] = 0.5 * il2;
            g1[0][1] = g1[1][0] = g_dd1(lm[0], lm[1], gl[0], gl[1]);
            g1[1][2] = g1[2][1] = g_dd1(lm[1], lm[2], gl[1], gl[2]);
            g1[0][2] = g1[2][0] = g_dd1(lm[0], lm[2], gl[0], gl[2]);
            g2[0][0][0] = -0.25 * il0 * il0; g2[1][1][1] = -0.25 * il1 * il1; g2[2][2][2] = -0.25 * il2 * il2;
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int b = 0; b < 3; b++)
                    if (a != b) {   // g[a,a,b]: nodes (a, a, b), middle node a
                        const double v = g_dd2(lm[a], lm[a], lm[b], g1[a][a], g1[a][b]);
                        g2[a][a][b] = g2[a][b][a] = g2[b][a][a] = v;
                    }
            // g[0,1,2]: the middle node is the one opposite the widest gap
            const double w01 = fabs(lm[0] - lm[1]), w12 = fabs(lm[1] - lm[2]), w02 = fabs(lm[0] - lm[2]);
            const int mid = (w02 >= w01 && w02 >= w12) ? 1 : ((w01 >= w12) ? 2 : 0);
            const int i0 = (mid == 0) ? 1 : 0, i2 = (mid == 2) ? 1 : 2;
            const double x0 = (i0 == 0) ? lm[0] : lm[1], x2 = (i2 == 2) ? lm[2] : lm[1], x1 = (mid == 0) ? lm[0] : ((mid == 1) ? lm[1] : lm[2]);
            const double ga = (mid == 0) ? g1[1][0] : ((mid == 1) ? g1[0][1] : g1[0][2]);   // g[x0, x1]
            const double gb = (mid == 0) ? g1[0][2] : ((mid == 1) ? g1[1][2] : g1[2][1]);   // g[x1, x2]
            const double v = g_dd2(x0, x1, x2, ga, gb);
            g2[0][1][2] = g2[0][2][1] = g2[1][0][2] = g2[1][2][0] = g2[2][0][1] = g2[2][1][0] = v;
        }
        SENS_SYNC(6);
        // ---- S^ = 2 g[a,b] T^_ab in the eigenbasis of C, S' = R S^ R^T
        double Tq[6], Tq33[3][3], S[3][3];
        rot6<0>(R, T, Tq);
        to33(Tq, Tq33);
        {
            const double Sq[6] = {2.0 * g1[0][0] * Tq[0], 2.0 * g1[1][1] * Tq[1], 2.0 * g1[2][2] * Tq[2],
                                  2.0 * g1[0][1] * Tq[3], 2.0 * g1[1][2] * Tq[4], 2.0 * g1[0][2] * Tq[5]};
            double S6[6];
            rot6<1>(R, Sq, S6);
            to33(S6, S);
        }
        SENS_SYNC(2);
        // ---- reverse: Pbar'_iK = w sum_I lam_Ii G'_IK (Eq.(35) :257);  P' = F' S'  (Eq.(26) :208)
        double Fb[3][3], Sbq33[3][3];
        {
            double Pb[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
            for (int I = 0; I < 8; I++) {
                const double g0 = Gs[3 * I], g1_ = Gs[3 * I + 1], g2_ = Gs[3 * I + 2];
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    const double l = sL[el][I][i];
                    Pb[i][0] = fma(l, g0, Pb[i][0]); Pb[i][1] = fma(l, g1_, Pb[i][1]); Pb[i][2] = fma(l, g2_, Pb[i][2]);
                }
            }
            double Sb[6], Sbq[6];
            constexpr int PI[6] = {0, 1, 2, 0, 1, 0}, PJ[6] = {0, 1, 2, 1, 2, 2};
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    Pb[i][j] *= wq;
                }
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) Fb[i][j] = Pb[i][0] * S[0][j] + Pb[i][1] * S[1][j] + Pb[i][2] * S[2][j];
#pragma unroll
            for (int k = 0; k < 6; k++) {   // sym(F^T Pbar)
                const int i = PI[k], j = PJ[k];
                Sb[k] = 0.5 * (F[0][i] * Pb[0][j] + F[1][i] * Pb[1][j] + F[2][i] * Pb[2][j] + F[0][j] * Pb[0][i] + F[1][j] * Pb[1][i] + F[2][j] * Pb[2][i]);
            }
            rot6<0>(R, Sb, Sbq);
            to33(Sbq, Sbq33);
        }
        // dS = P_L:dT + (T:L_L):dC/2  (Eq.(25) :204):  Tbar^_ab = 2 g[a,b] Sbar^_ab,
        // Cbar^_ac = 2 sum_b g[a,b,c] (T^_ab Sbar^_bc + Sbar^_ab T^_bc)
        double Cbq[6], Tb[6];
        {
            constexpr int PI[6] = {0, 1, 2, 0, 1, 0}, PJ[6] = {0, 1, 2, 1, 2, 2};
            double Tbq[6];
#pragma unroll
            for (int k = 0; k < 6; k++) {
                const int a = PI[k], c = PJ[k];
                Tbq[k] = 2.0 * g1[a][c] * Sbq33[a][c];
                double s = 0.0;
#pragma unroll
                for (int b = 0; b < 3; b++) s += g2[a][b][c] * (Tq33[a][b] * Sbq33[b][c] + Sbq33[a][b] * Tq33[b][c]);
                Cbq[k] = 2.0 * s;
            }
            rot6<1>(R, Tbq, Tb);
        }
        // ---- cotangent on hist_out: stored components -> tensor (shear / 2), rotated into the material frame
        double eb[6] = {0, 0, 0, 0, 0, 0}, ab = 0.0;
        if (muv) {
            const double *mq = muv + (e * 8 + q) * 7;
            const double t[6] = {mq[0], mq[1], mq[2], 0.5 * mq[3], 0.5 * mq[4], 0.5 * mq[5]};
            rot6<0>(Th, t, eb);
            ab = mq[6];
        }
        SENS_SYNC(3);
        // ---- transposed App. D solve (Eq.(D4)-(D7) :1002-1019)
        double v[6], wT[6], alb;
        if (plastic) {
            double Heb[6], yT[6], mN[6], b[6];
            applyH(m, eb, Heb);
            const double Neb = dot6(N, eb);
#pragma unroll
            for (int k = 0; k < 6; k++) yT[k] = Tb[k] + kap * (Heb[k] - N[k] * Neb);
            applyDinv(D, N, mN);
            applyDinv(D, yT, b);
            const double a_ = dot6(N, mN), iom = frcp(1.0 - kap * a_), myT = dot6(mN, yT);
            const double Hp = (2.0 / 3.0) * dsf;                       // W sigma_y' = 2/3 sigma_flow'
            const double wf = (myT * iom - SW23 * ab - Neb) * frcp(a_ * iom + Hp);
            const double cm = (kap * myT - wf) * iom;
#pragma unroll
            for (int k = 0; k < 6; k++) v[k] = b[k] + cm * mN[k];
            alb = ab + SW23 * dsf * wf;
            applyEinv(m, v, wT);
            // theta: r_k and hardening constants
            double x[6], B1[6], B2[6], dh[3];
#pragma unroll
            for (int k = 0; k < 6; k++) x[k] = dgam * (eb[k] - v[k]);
            hill_bilinear_ds(x, T, B1);
            hill_bilinear_ds(T, T, B2);
            const double iphi = frcp(phi), c2 = (0.5 * dot6(x, N) * iphi + 0.5 * wf) * iphi;
#pragma unroll
            for (int k = 0; k < 6; k++) {
                const double rk = mp[2 + k];
                gth[2 + k] = -2.0 * (B1[k] * iphi - c2 * B2[k]) * frcp(rk * rk * rk);
            }
            flow_dh(m, alpha, dsf, faux, dh);
#pragma unroll
            for (int k = 0; k < 3; k++) gth[8 + k] = SW23 * wf * dh[k];
        } else {
#pragma unroll
            for (int k = 0; k < 6; k++) wT[k] = Tb[k];
            applyE(m, Tb, v);
            alb = ab;
        }
        {
            // E and nu: dG_T/dE = -T/E, dG_T/dnu = -(dE/dnu):ee_el with ee_el = E^-1 T
            double eel[6], dEnu[6];
            applyEinv(m, T, eel);
            const double op = 1.0 + m.nu, om2 = 1.0 - 2.0 * m.nu;
            const double iop2 = frcp(op * op), dmu2 = -m.E * iop2, dlam = m.E * (1.0 + 2.0 * m.nu * m.nu) * iop2 * frcp(om2 * om2);
            const double tr = dlam * (eel[0] + eel[1] + eel[2]);
#pragma unroll
            for (int k = 0; k < 3; k++) dEnu[k] = dmu2 * eel[k] + tr;
#pragma unroll
            for (int k = 3; k < 6; k++) dEnu[k] = dmu2 * eel[k];
            gth[0] = dot6(wT, T) * m.iE;
            gth[1] = dot6(wT, dEnu);
        }
        SENS_SYNC(4);
        // ---- history-in cotangent back in the global frame, stored components (shear x 2)
        if (g_hist && live) {
            double epb[6], o6[6];
#pragma unroll
            for (int k = 0; k < 6; k++) epb[k] = eb[k] - v[k];
            rot6<1>(Th, epb, o6);
            double *go = g_hist + (e * 8 + q) * 7;
            go[0] = o6[0]; go[1] = o6[1]; go[2] = o6[2]; go[3] = 2.0 * o6[3]; go[4] = 2.0 * o6[4]; go[5] = 2.0 * o6[5];
            go[6] = alb;
        }
        SENS_SYNC(7);
        // ---- d eps = P_L : dC / 2:  Cbar^_ab += g[a,b] epsbar^_ab;  C = F^T F: Fbar += 2 F Cbar;  ubar_Ii = Fbar_iJ G_IJ
        if (gu_scr) {
            double vq[6], Cb[6], Cb33[3][3];
            rot6<0>(R, v, vq);
            Cbq[0] += g1[0][0] * vq[0]; Cbq[1] += g1[1][1] * vq[1]; Cbq[2] += g1[2][2] * vq[2];
            Cbq[3] += g1[0][1] * vq[3]; Cbq[4] += g1[1][2] * vq[4]; Cbq[5] += g1[0][2] * vq[5];
            rot6<1>(R, Cbq, Cb);
            to33(Cb, Cb33);
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) Fb[i][j] += 2.0 * (F[i][0] * Cb33[0][j] + F[i][1] * Cb33[1][j] + F[i][2] * Cb33[2][j]);
            if (FBAR) {
                // dFbar_q = c_q dF_q + F_q c_q/3 (dJbar/Jbar - dJ_q/J_q), dJ_p = J_p F_p^-T : dF_p  =>
                // Fb <- c_q Fb + F_q^-T ( (S/Jbar) w_q J_q / V - s_q ),  s_q = (Fb : Fbar_q)/3,  S = sum_q s_q,  F_q^-T = cof(Fbar_q)/(c_q^2 J_q)
                double sq = 0.0;
#pragma unroll
                for (int i = 0; i < 3; i++)
#pragma unroll
                    for (int j = 0; j < 3; j++) sq += Fb[i][j] * F[i][j];
                sq *= (1.0 / 3.0);
                double S = sq;
#pragma unroll
                for (int o = 1; o < 8; o <<= 1) S += __shfl_xor_sync(0xffffffffu, S, o);
                const double k = (S / fb_Jbar * fb_wJV - sq) / (fb_c * fb_c * fb_J);
                double cof[3][3];
                cof[0][0] = F[1][1] * F[2][2] - F[1][2] * F[2][1]; cof[0][1] = F[1][2] * F[2][0] - F[1][0] * F[2][2]; cof[0][2] = F[1][0] * F[2][1] - F[1][1] * F[2][0];
                cof[1][0] = F[0][2] * F[2][1] - F[0][1] * F[2][2]; cof[1][1] = F[0][0] * F[2][2] - F[0][2] * F[2][0]; cof[1][2] = F[0][1] * F[2][0] - F[0][0] * F[2][1];
                cof[2][0] = F[0][1] * F[1][2] - F[0][2] * F[1][1]; cof[2][1] = F[0][2] * F[1][0] - F[0][0] * F[1][2]; cof[2][2] = F[0][0] * F[1][1] - F[0][1] * F[1][0];
#pragma unroll
                for (int i = 0; i < 3; i++)
#pragma unroll
                    for (int j = 0; j < 3; j++) Fb[i][j] = fb_c * Fb[i][j] + k * cof[i][j];
            }
#pragma unroll
            for (int I = 0; I < 8; I++) {
                const double g0 = Gs[3 * I], g1_ = Gs[3 * I + 1], g2_ = Gs[3 * I + 2];
#pragma unroll
                for (int i = 0; i < 3; i++) Gs[3 * I + i] = Fb[i][0] * g0 + Fb[i][1] * g1_ + Fb[i][2] * g2_;
            }
        }
    }
    if (!live) {
#pragma unroll
        for (int k = 0; k < NTHETA; k++) gth[k] = 0.0;
    }
    __syncthreads();
    if (live) {
        // lane q sums local node q over the 8 Gauss points, ascending
        if (gu_scr) {
            const long long j = eslot[e * 8 + q];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                double s = 0.0;
#pragma unroll
                for (int p = 0; p < 8; p++) s += sGu[el][p][3 * q + i];
                gu_scr[3 * j + i] = s;
            }
        }
        if (g_mat) {   // per-element records: points summed ascending; the entries that are not differentiated are 0
            for (int k = q; k < FEM_NPAR; k += 8) {
                int t = -1;
#pragma unroll
                for (int j = 0; j < NTHETA; j++) t = (S_THETA_IDX[j] == k) ? j : t;
                double s = 0.0;
                if (t >= 0)
                    for (int p = 0; p < 8; p++) s += sTh[el * 8 + p][t];
                g_mat[e * FEM_NPAR + k] = s;
            }
        }
    }
    if (part && tid < NTHETA) {
        double s = 0.0;
        for (int t = 0; t < STHREADS; t++) s += sTh[t][tid];
        part[(long long)blockIdx.x * NTHETA + tid] = s;
    }
}

// g_u[n] = sum of the node's incidence entries, ascending element id
__global__ void k_sens_gather(long long n_nodes, const int *__restrict__ inc_ptr, const double *__restrict__ scr, double *__restrict__ g_u) {
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int j = inc_ptr[n]; j < inc_ptr[n + 1]; j++) { s0 += scr[3LL * j]; s1 += scr[3LL * j + 1]; s2 += scr[3LL * j + 2]; }
    g_u[3 * n] = s0; g_u[3 * n + 1] = s1; g_u[3 * n + 2] = s2;
}

// uniform material: g_mat[THETA_IDX[k]] = sum over CTAs of part[.][k]; block k, fixed strided partial sums + tree
__global__ void __launch_bounds__(256) k_sens_reduce(long long n_part, const double *__restrict__ part, double *__restrict__ g_mat) {
    __shared__ double sh[256];
    const int k = blockIdx.x, t = threadIdx.x;
    double s = 0.0;
    for (long long i = t; i < n_part; i += 256) s += part[i * NTHETA + k];
    sh[t] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (t < w) sh[t] += sh[t + w];
        __syncthreads();
    }
    if (t == 0) g_mat[S_THETA_IDX[k]] = sh[0];
    if (k == 0 && t < FEM_NPAR) {
        bool is_theta = false;
        for (int j = 0; j < NTHETA; j++) is_theta |= (S_THETA_IDX[j] == t);
        if (!is_theta) g_mat[t] = 0.0;
    }
}

extern "C" int fem_assemble_vjp(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                                const double *lam, const double *mu, double *g_u, double *g_hist_in, double *g_mat,
                                void *cuda_stream) {
    if (!c || !u || !hist_in || !mat) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (n_mat != 1 && n_mat != c->n_elems) return FEM_ERR_MAT;
    if (g_u && (!c->d_eslot || !c->d_Re)) return FEM_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long ne = c->n_elems;
    if (ne == 0) {
        if (g_u && c->n_rows) FEM_CUDA(cudaMemsetAsync(g_u, 0, sizeof(double) * c->n_rows, st));
        if (g_mat) FEM_CUDA(cudaMemsetAsync(g_mat, 0, sizeof(double) * FEM_NPAR * (n_mat == 1 ? 1 : 0), st));
        return FEM_OK;
    }
    const long long nblk = (ne + SEL - 1) / SEL;
    double *part = nullptr;
    if (g_mat && n_mat == 1) {
        if (c->n_sens_part < nblk) {
            if (c->d_sens_part) cudaFree(c->d_sens_part);
            c->d_sens_part = nullptr; c->n_sens_part = 0;
            FEM_CUDA(cudaMalloc(&c->d_sens_part, sizeof(double) * NTHETA * nblk));
            c->n_sens_part = nblk;
        }
        part = c->d_sens_part;
    }
    if (c->opt.fbar)
        k_sens_point<1><<<(unsigned)nblk, STHREADS, 0, st>>>(ne, c->d_coords, c->d_conn, c->d_eslot, u, hist_in, mat, n_mat, lam, mu,
                                                      g_u ? c->d_Re : nullptr, g_hist_in, (g_mat && n_mat != 1) ? g_mat : nullptr, part);
    else
        k_sens_point<0><<<(unsigned)nblk, STHREADS, 0, st>>>(ne, c->d_coords, c->d_conn, c->d_eslot, u, hist_in, mat, n_mat, lam, mu,
                                                      g_u ? c->d_Re : nullptr, g_hist_in, (g_mat && n_mat != 1) ? g_mat : nullptr, part);
    FEM_CUDA(cudaGetLastError());
    if (g_u) {
        k_sens_gather<<<(unsigned)((c->n_nodes + 255) / 256), 256, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_Re, g_u);
        FEM_CUDA(cudaGetLastError());
    }
    if (part) {
        k_sens_reduce<<<NTHETA, 256, 0, st>>>(nblk, part, g_mat);
        FEM_CUDA(cudaGetLastError());
    }
    return FEM_OK;
}
