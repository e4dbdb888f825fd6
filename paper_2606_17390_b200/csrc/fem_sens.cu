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
// switch and the orientation quaternion are not differentiated (their entries of g_mat are 0).  Hill-48, standard element.
// Sums are taken in a fixed order (per node: ascending element id; uniform material: fixed two-level tree), no atomics.
// Nothing here is shared with oracle/.
#include "fem_internal.h"
#include <math.h>

#define SW23 0.81649658092772603273   // W = sqrt(2/3)
#define SEL 16                        // elements per CTA
#define STHREADS (8 * SEL)
#define NTHETA 11

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
__device__ __forceinline__ void to6(const double A[3][3], double a[6]) {
    a[0] = A[0][0]; a[1] = A[1][1]; a[2] = A[2][2];
    a[3] = 0.5 * (A[0][1] + A[1][0]); a[4] = 0.5 * (A[1][2] + A[2][1]); a[5] = 0.5 * (A[0][2] + A[2][0]);
}
// B = Q^T A Q (tr = 0) or Q A Q^T (tr = 1) for symmetric A given as 6 components
__device__ __forceinline__ void rot6(const double Q[3][3], const double a[6], double b[6], int tr) {
    double A[3][3], T[3][3], B[3][3];
    to33(a, A);
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0.0;
            for (int k = 0; k < 3; k++) s += A[i][k] * (tr ? Q[j][k] : Q[k][j]);
            T[i][j] = s;
        }
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0.0;
            for (int k = 0; k < 3; k++) s += (tr ? Q[i][k] : Q[k][i]) * T[k][j];
            B[i][j] = s;
        }
    to6(B, b);
}

struct SMat {
    double E, nu, mu2, lam, law, h0, h1, h2;
    double p[9];        // Hill coefficients p1..p9 of Eq.(A3)-(A5) :784-801 in the local (material) frame
    double r[6];
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
    for (int i = 0; i < 3; i++) b[i] = m.mu2 * a[i] + tr;
    for (int i = 3; i < 6; i++) b[i] = m.mu2 * a[i];
}
__device__ __forceinline__ void applyEinv(const SMat &m, const double a[6], double b[6]) {
    const double s = m.nu * (a[0] + a[1] + a[2]);
    for (int i = 0; i < 3; i++) b[i] = ((1.0 + m.nu) * a[i] - s) / m.E;
    for (int i = 3; i < 6; i++) b[i] = a[i] / m.mu2;
}
// D = E^-1 + kappa H : normal block 3x3 (symmetric, inverted once per kappa) + three shear scalars
struct SDinv { double n[6]; double s[3]; };   // inverse normal block as (11,22,33,12,23,13), inverse shear scalars
__device__ __forceinline__ void makeDinv(const SMat &m, double kap, SDinv &D) {
    const double ie = 1.0 / m.E, o = -m.nu * ie;
    const double a = ie + kap * m.p[0], b = ie + kap * m.p[1], c = ie + kap * m.p[2];
    const double d = o + kap * m.p[3], e = o + kap * m.p[4], f = o + kap * m.p[5];   // 12, 23, 13
    const double c00 = b * c - e * e, c01 = f * e - d * c, c02 = d * e - f * b;
    const double idet = 1.0 / (a * c00 + d * c01 + f * c02);
    D.n[0] = c00 * idet; D.n[3] = c01 * idet; D.n[5] = c02 * idet;
    D.n[1] = (a * c - f * f) * idet; D.n[4] = (d * f - a * e) * idet; D.n[2] = (a * b - d * d) * idet;
    for (int k = 0; k < 3; k++) D.s[k] = 1.0 / (1.0 / m.mu2 + kap * m.p[6 + k]);
}
__device__ __forceinline__ void applyDinv(const SDinv &D, const double a[6], double b[6]) {
    b[0] = D.n[0] * a[0] + D.n[3] * a[1] + D.n[5] * a[2];
    b[1] = D.n[3] * a[0] + D.n[1] * a[1] + D.n[4] * a[2];
    b[2] = D.n[5] * a[0] + D.n[4] * a[1] + D.n[2] * a[2];
    b[3] = D.s[0] * a[3]; b[4] = D.s[1] * a[4]; b[5] = D.s[2] * a[5];
}

// sigma_flow, d sigma_flow/d alpha and d sigma_flow/d(h0,h1,h2): Voce Eq.(10) :121, Swift (BASELINE configs)
__device__ __forceinline__ void flow_all(const SMat &m, double alpha, double &sf, double &dsf, double dh[3]) {
    if (m.law == 0.0) {
        const double e = exp(-m.h2 * alpha);
        sf = m.h0 + m.h1 * (1.0 - e); dsf = m.h1 * m.h2 * e;
        dh[0] = 1.0; dh[1] = 1.0 - e; dh[2] = m.h1 * alpha * e;
    } else {
        const double b = m.h1 + alpha, lb = log(b), pw = exp(m.h2 * lb);
        sf = m.h0 * pw; dsf = m.h0 * m.h2 * pw / b;
        dh[0] = pw; dh[1] = m.h0 * m.h2 * pw / b; dh[2] = m.h0 * pw * lb;
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

// atanh(w)/w
__device__ __forceinline__ double s_atanhc(double w) {
    const double w2 = w * w;
    if (w2 < 0.01) {
        double s = 1.0 / 19.0;
        for (int k = 17; k >= 1; k -= 2) s = s * w2 + 1.0 / k;
        return s;
    }
    return 0.5 * log((1.0 + w) / (1.0 - w)) / w;
}
// first divided difference of ln:  ln[a,b] = 2 atanhc(w) / (a + b), w = (a-b)/(a+b)
__device__ __forceinline__ double ln_dd1(double a, double b) {
    const double s = a + b;
    return 2.0 * s_atanhc((a - b) / s) / s;
}
// second divided difference of ln over three (possibly coincident) nodes: series in the complete homogeneous polynomials of
// the centred nodes when they are close, else the recursion over the widest gap
__device__ double ln_dd2(double x0, double x1, double x2) {
    const double m = (x0 + x1 + x2) * (1.0 / 3.0);
    const double d0 = (x0 - m) / m, d1 = (x1 - m) / m, d2 = (x2 - m) / m;
    const double sp = fmax(fabs(d0), fmax(fabs(d1), fabs(d2)));
    if (sp < 0.08) {
        // ln[x0,x1,x2] = 1/m^2 sum_{n>=2} (-1)^(n-1)/n h_{n-2}(d);  h_k = -e2 h_{k-2} + e3 h_{k-3}  (e1 = 0)
        const double e2 = d0 * d1 + d1 * d2 + d0 * d2, e3 = d0 * d1 * d2;
        double hm2 = 0.0, hm1 = 0.0, h = 1.0, s = 0.0, sg = -1.0;
        for (int n = 2; n <= 22; n++) {
            s += sg * h / n;
            sg = -sg;
            const double hn = -e2 * hm1 + e3 * hm2;
            hm2 = hm1; hm1 = h; h = hn;
        }
        return s / (m * m);
    }
    // order so that lo <= mid <= hi
    double lo = fmin(x0, fmin(x1, x2)), hi = fmax(x0, fmax(x1, x2)), mid = x0 + x1 + x2 - lo - hi;
    const double f_hm = (hi == mid) ? 1.0 / hi : ln_dd1(hi, mid);
    const double f_ml = (mid == lo) ? 1.0 / lo : ln_dd1(mid, lo);
    return (f_hm - f_ml) / (hi - lo);
}

// cyclic Jacobi on a symmetric 3x3: A = V diag(lam) V^T, columns of V the eigenvectors
__device__ __forceinline__ void jacobi3(double A[3][3], double V[3][3], double lam[3]) {
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) V[i][j] = (i == j) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 6; sweep++) {
        for (int pq = 0; pq < 3; pq++) {
            const int p = (pq == 2) ? 1 : 0, q = (pq == 0) ? 1 : 2;
            const double apq = A[p][q];
            if (fabs(apq) < 1e-300) continue;
            const double th = (A[q][q] - A[p][p]) / (2.0 * apq);
            const double t = copysign(1.0, th) / (fabs(th) + sqrt(th * th + 1.0));
            const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            const int r = 3 - p - q;
            const double arp = A[r][p], arq = A[r][q];
            A[p][p] -= t * apq; A[q][q] += t * apq; A[p][q] = A[q][p] = 0.0;
            A[r][p] = A[p][r] = c * arp - s * arq;
            A[r][q] = A[q][r] = s * arp + c * arq;
            for (int k = 0; k < 3; k++) {
                const double vp = V[k][p], vq = V[k][q];
                V[k][p] = c * vp - s * vq; V[k][q] = s * vp + c * vq;
            }
        }
    }
    lam[0] = A[0][0]; lam[1] = A[1][1]; lam[2] = A[2][2];
}

__global__ void __launch_bounds__(STHREADS)
k_sens_point(long long n_elems, const double *__restrict__ coords, const int *__restrict__ conn, const int *__restrict__ eslot,
             const double *__restrict__ u, const double *__restrict__ hist_in, const double *__restrict__ mat, long long n_mat,
             const double *__restrict__ lamv, const double *__restrict__ muv,
             double *__restrict__ gu_scr /*[8 n_elems][3] incidence order, may be null*/,
             double *__restrict__ g_hist /*may be null*/, double *__restrict__ g_mat /*per element, may be null*/,
             double *__restrict__ part /*[gridDim.x][NTHETA] uniform material, may be null*/) {
    __shared__ double sX[SEL][8][3], sU[SEL][8][3], sL[SEL][8][3];
    __shared__ double sGu[SEL][8][25];      // [element][point][24 (+1 pad)]
    __shared__ double sTh[STHREADS][NTHETA];
    const int tid = threadIdx.x, el = tid >> 3, q = tid & 7;
    const long long e = (long long)blockIdx.x * SEL + el;
    const bool live = e < n_elems;
    double gth[NTHETA];
    for (int k = 0; k < NTHETA; k++) gth[k] = 0.0;
    if (live) {
        const int nd = conn[e * 8 + q];
        for (int i = 0; i < 3; i++) {
            sX[el][q][i] = coords[3LL * nd + i];
            sU[el][q][i] = u[3LL * nd + i];
            sL[el][q][i] = lamv ? lamv[3LL * nd + i] : 0.0;
        }
    }
    __syncthreads();
    if (live) {
        // ---- material record
        const double *mp = mat + (n_mat == 1 ? 0 : e) * FEM_NPAR;
        SMat m;
        m.E = mp[0]; m.nu = mp[1]; m.mu2 = m.E / (1.0 + m.nu); m.lam = m.E * m.nu / ((1.0 + m.nu) * (1.0 - 2.0 * m.nu));
        m.law = mp[8]; m.h0 = mp[9]; m.h1 = mp[10]; m.h2 = mp[11];
        for (int k = 0; k < 6; k++) m.r[k] = mp[2 + k];
        m.p[0] = 2.0 / (3.0 * m.r[0] * m.r[0]); m.p[1] = 2.0 / (3.0 * m.r[1] * m.r[1]); m.p[2] = 2.0 / (3.0 * m.r[2] * m.r[2]);
        m.p[6] = 1.0 / (m.r[3] * m.r[3]); m.p[7] = 1.0 / (m.r[4] * m.r[4]); m.p[8] = 1.0 / (m.r[5] * m.r[5]);
        m.p[3] = 0.5 * (m.p[2] - m.p[0] - m.p[1]); m.p[4] = 0.5 * (m.p[0] - m.p[1] - m.p[2]); m.p[5] = 0.5 * (m.p[1] - m.p[0] - m.p[2]);
        double Th[3][3];
        {
            const double qn = sqrt(mp[12] * mp[12] + mp[13] * mp[13] + mp[14] * mp[14] + mp[15] * mp[15]);
            const double w = mp[12] / qn, x = mp[13] / qn, y = mp[14] / qn, z = mp[15] / qn;
            Th[0][0] = 1 - 2 * (y * y + z * z); Th[0][1] = 2 * (x * y - w * z);     Th[0][2] = 2 * (x * z + w * y);
            Th[1][0] = 2 * (x * y + w * z);     Th[1][1] = 1 - 2 * (x * x + z * z); Th[1][2] = 2 * (y * z - w * x);
            Th[2][0] = 2 * (x * z - w * y);     Th[2][1] = 2 * (y * z + w * x);     Th[2][2] = 1 - 2 * (x * x + y * y);
        }
        // ---- shape gradients at Gauss point q (Eq.(28) :220), rotated: G'_IJ = G_IK Theta_KJ
        const double gp = 0.57735026918962576451;
        const double xi[3] = {(q & 1) ? gp : -gp, (q & 2) ? gp : -gp, (q & 4) ? gp : -gp};
        double dN[8][3], Jr[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (int I = 0; I < 8; I++) {
            const double a = 1.0 + xi[0] * S_XI[I][0], b = 1.0 + xi[1] * S_XI[I][1], c = 1.0 + xi[2] * S_XI[I][2];
            dN[I][0] = 0.125 * S_XI[I][0] * b * c; dN[I][1] = 0.125 * a * S_XI[I][1] * c; dN[I][2] = 0.125 * a * b * S_XI[I][2];
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) Jr[i][j] += sX[el][I][i] * dN[I][j];
        }
        double Ji[3][3];
        Ji[0][0] = Jr[1][1] * Jr[2][2] - Jr[1][2] * Jr[2][1]; Ji[0][1] = Jr[0][2] * Jr[2][1] - Jr[0][1] * Jr[2][2]; Ji[0][2] = Jr[0][1] * Jr[1][2] - Jr[0][2] * Jr[1][1];
        Ji[1][0] = Jr[1][2] * Jr[2][0] - Jr[1][0] * Jr[2][2]; Ji[1][1] = Jr[0][0] * Jr[2][2] - Jr[0][2] * Jr[2][0]; Ji[1][2] = Jr[0][2] * Jr[1][0] - Jr[0][0] * Jr[1][2];
        Ji[2][0] = Jr[1][0] * Jr[2][1] - Jr[1][1] * Jr[2][0]; Ji[2][1] = Jr[0][1] * Jr[2][0] - Jr[0][0] * Jr[2][1]; Ji[2][2] = Jr[0][0] * Jr[1][1] - Jr[0][1] * Jr[1][0];
        const double wq = Jr[0][0] * Ji[0][0] + Jr[0][1] * Ji[1][0] + Jr[0][2] * Ji[2][0];   // det J_ref, weights 1
        double JT[3][3];   // J_ref^-1 Theta
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) JT[i][j] = (Ji[i][0] * Th[0][j] + Ji[i][1] * Th[1][j] + Ji[i][2] * Th[2][j]) / wq;
        double G[8][3];
        for (int I = 0; I < 8; I++)
            for (int j = 0; j < 3; j++) G[I][j] = dN[I][0] * JT[0][j] + dN[I][1] * JT[1][j] + dN[I][2] * JT[2][j];
        // ---- F' = F Theta = Theta + u^T G'  (Eq.(30) :228), C' = F'^T F'
        double F[3][3];
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                double s = Th[i][j];
                for (int I = 0; I < 8; I++) s += sU[el][I][i] * G[I][j];
                F[i][j] = s;
            }
        double Cw[3][3], R[3][3], lm[3];
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) Cw[i][j] = F[0][i] * F[0][j] + F[1][i] * F[1][j] + F[2][i] * F[2][j];
        jacobi3(Cw, R, lm);
        // ---- Hencky strain in the material frame (Eq.(4)-(5) :92-96, reading G1: the factor 1/2)
        double eh[6] = {0.5 * log(lm[0]), 0.5 * log(lm[1]), 0.5 * log(lm[2]), 0, 0, 0}, eps[6];
        rot6(R, eh, eps, 1);
        // ---- history in, rotated into the material frame
        const double *hp = hist_in + (e * 8 + q) * 7;
        double epn_g[6] = {hp[0], hp[1], hp[2], hp[3], hp[4], hp[5]}, epn[6];
        rot6(Th, epn_g, epn, 0);
        const double alpha_n = hp[6];
        // ---- cotangent on hist_out: stored components -> tensor (shear / 2), rotated
        double eb[6] = {0, 0, 0, 0, 0, 0}, ab = 0.0;
        if (muv) {
            const double *mq = muv + (e * 8 + q) * 7;
            double t[6] = {mq[0], mq[1], mq[2], 0.5 * mq[3], 0.5 * mq[4], 0.5 * mq[5]};
            rot6(Th, t, eb, 0);
            ab = mq[6];
        }
        // ---- trial state (Eq.(16)-(17) :160-165)
        double ee[6], T[6], HT[6], N[6];
        for (int k = 0; k < 6; k++) ee[k] = eps[k] - epn[k];
        applyE(m, ee, T);
        applyH(m, T, HT);
        double phi = sqrt(fmax(dot6(T, HT), 0.0));
        double sf, dsf, dh[3];
        flow_all(m, alpha_n, sf, dsf, dh);
        double dgam = 0.0, alpha = alpha_n, kap = 0.0;
        const bool plastic = phi - SW23 * sf > 0.0;
        SDinv D;
        if (plastic) {
            // ---- return map: f(dgam) = sigma_y(alpha)/phi(kappa) - 1 = 0, monotone increasing, f(0) < 0
            double lo = 0.0, hi = -1.0;
            for (int it = 0; it < 60; it++) {
                alpha = alpha_n + SW23 * dgam;
                flow_all(m, alpha, sf, dsf, dh);
                const double sy = SW23 * sf, dsy = (2.0 / 3.0) * dsf;   // d sigma_y / d dgam = W * W sigma_flow'
                kap = dgam / sy;
                makeDinv(m, kap, D);
                applyDinv(D, ee, T);
                applyH(m, T, HT);
                phi = sqrt(dot6(T, HT));
                for (int k = 0; k < 6; k++) N[k] = HT[k] / phi;
                double mN[6];
                applyDinv(D, N, mN);
                const double a_ = dot6(N, mN);
                const double f = sy / phi - 1.0;
                const double dk = (sy - dgam * dsy) / (sy * sy);
                const double df = dsy / phi + (sy / phi) * a_ * dk;
                if (f < 0.0) lo = dgam; else hi = dgam;
                double nx = dgam - f / df;
                if (!(nx > lo) || (hi > 0.0 && !(nx < hi))) nx = (hi > 0.0) ? 0.5 * (lo + hi) : 2.0 * dgam + 1e-6;
                const double step = fabs(nx - dgam);
                const bool done = (fabs(f) <= 1e-15) || (step <= 4e-16 * nx);
                if (done) break;
                dgam = nx;
            }
        } else {
            makeDinv(m, 0.0, D);
        }
        // ---- state at the solution
        if (plastic) {
            alpha = alpha_n + SW23 * dgam;
            flow_all(m, alpha, sf, dsf, dh);
            makeDinv(m, dgam / (SW23 * sf), D);
            applyDinv(D, ee, T);
            applyH(m, T, HT);
            phi = sqrt(dot6(T, HT));
            for (int k = 0; k < 6; k++) N[k] = HT[k] / phi;
            kap = dgam / phi;
            makeDinv(m, kap, D);
        } else {
            for (int k = 0; k < 6; k++) N[k] = 0.0;
        }
        // ---- S^ = 2 g[a,b] T^_ab in the eigenbasis of C, S' = R S^ R^T
        double g1[3][3], g2[3][3][3];
        for (int a = 0; a < 3; a++)
            for (int b = a; b < 3; b++) g1[a][b] = g1[b][a] = (a == b) ? 0.5 / lm[a] : 0.5 * ln_dd1(lm[a], lm[b]);
        for (int a = 0; a < 3; a++)
            for (int b = a; b < 3; b++)
                for (int c = b; c < 3; c++) {
                    const double v = 0.5 * ln_dd2(lm[a], lm[b], lm[c]);
                    g2[a][b][c] = g2[a][c][b] = g2[b][a][c] = g2[b][c][a] = g2[c][a][b] = g2[c][b][a] = v;
                }
        double Tq[6], Tq33[3][3], Sq[6], S6[6], S[3][3];
        rot6(R, T, Tq, 0);
        to33(Tq, Tq33);
        {
            double Sq33[3][3];
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) Sq33[a][b] = 2.0 * g1[a][b] * Tq33[a][b];
            to6(Sq33, Sq);
        }
        rot6(R, Sq, S6, 1);
        to33(S6, S);
        // ---- reverse: Pbar'_iK = w sum_I lam_Ii G'_IK (Eq.(35) :257);  P' = F' S'  (Eq.(26) :208)
        double Pb[3][3], Fb[3][3], Sb33[3][3], Sb[6], Sbq[6], Sbq33[3][3];
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                double s = 0.0;
                for (int I = 0; I < 8; I++) s += sL[el][I][i] * G[I][j];
                Pb[i][j] = wq * s;
            }
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                Fb[i][j] = Pb[i][0] * S[0][j] + Pb[i][1] * S[1][j] + Pb[i][2] * S[2][j];
                Sb33[i][j] = F[0][i] * Pb[0][j] + F[1][i] * Pb[1][j] + F[2][i] * Pb[2][j];
            }
        to6(Sb33, Sb);
        rot6(R, Sb, Sbq, 0);
        to33(Sbq, Sbq33);
        // dS = P_L:dT + (T:L_L):dC/2  (Eq.(25) :204):  Tbar^_ab = 2 g[a,b] Sbar^_ab,
        // Cbar^_ac = 2 sum_b g[a,b,c] (T^_ab Sbar^_bc + Sbar^_ab T^_bc)
        double Tbq33[3][3], Cbq33[3][3], Tbq[6], Tb[6];
        for (int a = 0; a < 3; a++)
            for (int c = 0; c < 3; c++) {
                Tbq33[a][c] = 2.0 * g1[a][c] * Sbq33[a][c];
                double s = 0.0;
                for (int b = 0; b < 3; b++) s += g2[a][b][c] * (Tq33[a][b] * Sbq33[b][c] + Sbq33[a][b] * Tq33[b][c]);
                Cbq33[a][c] = 2.0 * s;
            }
        to6(Tbq33, Tbq);
        rot6(R, Tbq, Tb, 1);
        // ---- transposed App. D solve (Eq.(D4)-(D7) :1002-1019)
        double v[6], wT[6], epb[6], alb;
        if (plastic) {
            flow_all(m, alpha, sf, dsf, dh);
            double Heb[6], yT[6], mN[6], b[6];
            applyH(m, eb, Heb);
            const double Neb = dot6(N, eb);
            for (int k = 0; k < 6; k++) yT[k] = Tb[k] + kap * (Heb[k] - N[k] * Neb);
            applyDinv(D, N, mN);
            applyDinv(D, yT, b);
            const double a_ = dot6(N, mN), om = 1.0 - kap * a_, myT = dot6(mN, yT);
            const double Hp = (2.0 / 3.0) * dsf;                       // W sigma_y' = 2/3 sigma_flow'
            const double wf = (myT / om - SW23 * ab - Neb) / (a_ / om + Hp);
            for (int k = 0; k < 6; k++) v[k] = b[k] + ((kap * myT - wf) / om) * mN[k];
            alb = ab + SW23 * dsf * wf;
            applyEinv(m, v, wT);
            // theta: r_k and hardening constants
            double x[6], B1[6], B2[6];
            for (int k = 0; k < 6; k++) x[k] = dgam * (eb[k] - v[k]);
            hill_bilinear_ds(x, T, B1);
            hill_bilinear_ds(T, T, B2);
            const double xN = dot6(x, N);
            for (int k = 0; k < 6; k++)
                gth[2 + k] = (-2.0 / (m.r[k] * m.r[k] * m.r[k])) * (B1[k] / phi - (xN / (2.0 * phi * phi) + wf / (2.0 * phi)) * B2[k]);
            for (int k = 0; k < 3; k++) gth[8 + k] = SW23 * wf * dh[k];
        } else {
            for (int k = 0; k < 6; k++) wT[k] = Tb[k];
            applyE(m, Tb, v);
            alb = ab;
        }
        for (int k = 0; k < 6; k++) epb[k] = eb[k] - v[k];
        {
            // E and nu: dG_T/dE = -T/E, dG_T/dnu = -(dE/dnu):ee_el with ee_el = E^-1 T
            double eel[6], dEnu[6];
            applyEinv(m, T, eel);
            const double op = 1.0 + m.nu, om2 = 1.0 - 2.0 * m.nu;
            const double dmu2 = -m.E / (op * op), dlam = m.E * (1.0 + 2.0 * m.nu * m.nu) / (op * op * om2 * om2);
            const double tr = dlam * (eel[0] + eel[1] + eel[2]);
            for (int k = 0; k < 3; k++) dEnu[k] = dmu2 * eel[k] + tr;
            for (int k = 3; k < 6; k++) dEnu[k] = dmu2 * eel[k];
            gth[0] = dot6(wT, T) / m.E;
            gth[1] = dot6(wT, dEnu);
        }
        // ---- history-in cotangent back in the global frame, stored components (shear x 2)
        if (g_hist) {
            double o6[6];
            rot6(Th, epb, o6, 1);
            double *go = g_hist + (e * 8 + q) * 7;
            go[0] = o6[0]; go[1] = o6[1]; go[2] = o6[2]; go[3] = 2.0 * o6[3]; go[4] = 2.0 * o6[4]; go[5] = 2.0 * o6[5];
            go[6] = alb;
        }
        // ---- d eps = P_L : dC / 2:  Cbar^_ab += g[a,b] epsbar^_ab;  C = F^T F: Fbar += 2 F Cbar;  ubar_Ii = Fbar_iJ G_IJ
        double vq[6], vq33[3][3], Cb6[6], Cb[6], Cb33[3][3];
        rot6(R, v, vq, 0);
        to33(vq, vq33);
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) Cbq33[a][b] += g1[a][b] * vq33[a][b];
        to6(Cbq33, Cb6);
        rot6(R, Cb6, Cb, 1);
        to33(Cb, Cb33);
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) Fb[i][j] += 2.0 * (F[i][0] * Cb33[0][j] + F[i][1] * Cb33[1][j] + F[i][2] * Cb33[2][j]);
        for (int I = 0; I < 8; I++)
            for (int i = 0; i < 3; i++) sGu[el][q][3 * I + i] = Fb[i][0] * G[I][0] + Fb[i][1] * G[I][1] + Fb[i][2] * G[I][2];
    }
    for (int k = 0; k < NTHETA; k++) sTh[tid][k] = gth[k];
    __syncthreads();
    if (live) {
        // lane q sums local node q over the 8 Gauss points, ascending
        if (gu_scr) {
            const long long j = eslot[e * 8 + q];
            for (int i = 0; i < 3; i++) {
                double s = 0.0;
                for (int p = 0; p < 8; p++) s += sGu[el][p][3 * q + i];
                gu_scr[3 * j + i] = s;
            }
        }
        if (g_mat) {   // per-element records: points summed ascending
            for (int k = q; k < FEM_NPAR; k += 8) g_mat[e * FEM_NPAR + k] = 0.0;
        }
    }
    if (g_mat) {
        __syncthreads();
        if (live)
            for (int k = q; k < NTHETA; k += 8) {
                double s = 0.0;
                for (int p = 0; p < 8; p++) s += sTh[el * 8 + p][k];
                g_mat[e * FEM_NPAR + S_THETA_IDX[k]] = s;
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
    if (c->opt.fbar != 0) return FEM_ERR_ARG;
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
    k_sens_point<<<(unsigned)nblk, STHREADS, 0, st>>>(ne, c->d_coords, c->d_conn, c->d_eslot, u, hist_in, mat, n_mat, lam, mu,
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
