/* ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow fp64 CPU statement of what `fem_assemble` computes, written from
 * /root/reference/PAPER.md (arxiv 2606.17390) with the readings listed in
 * DESIGN.md ("Readings of the paper").  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may call it.  It shares
 * no code, header, table or helper with paper_2606_17390_b200/csrc.
 *
 * Conventions: units mm / MPa.  Symmetric 2-tensors are exchanged as 6 tensor
 * components in the order (11,22,33,12,23,13) (PAPER.md:779 Eq.(A2), :793-796
 * Eq.(A4): p7<->12, p8<->23, p9<->13).  4-tensors with minor symmetries are
 * exchanged as 6x6 Mandel matrices (shear rows/cols x sqrt2).  Internally
 * everything is full 3x3 / 3x3x3x3 loops.
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py
 * (-m "not gpu").  The fbar=1 reading (literal Eq.(35)) is pinned
 * by internal consistency only (finite differences, affine fields) — the paper
 * prints no value that would distinguish it: "parity unpinned (reading G12)".
 *
 * SURVEY.md 8(f) NEXT-2 (Barlat Yld2004-18p, Eq.(12), App. A.2 :808-830): section "Yld2004-18p" below.
 * Pins: tests/test_oracle_barlat.py (von Mises / Hill-48 reductions of :828, Hershey closed forms, the eigenvalue
 * definition against the power-sum form, finite differences, App. D against differences of the return map, and the
 * printed line-search example of App. B :871-877, zeta = 0.363 at the third iteration).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NPAR 16 /* mat record: E,nu,r11,r22,r33,r12,r23,r13,law,h0,h1,h2,q0..q3 */

/* ---------------------------------------------------------------- helpers */
static const int VI[6] = {0, 1, 2, 0, 1, 0}; /* (11,22,33,12,23,13) */
static const int VJ[6] = {0, 1, 2, 1, 2, 2};

static void sym6_to_mat(const double v[6], double A[3][3]) {
    for (int m = 0; m < 6; m++) { A[VI[m]][VJ[m]] = v[m]; A[VJ[m]][VI[m]] = v[m]; }
}
static void mat_to_sym6(const double A[3][3], double v[6]) {
    for (int m = 0; m < 6; m++) v[m] = 0.5 * (A[VI[m]][VJ[m]] + A[VJ[m]][VI[m]]);
}
static double mw(int m) { return m < 3 ? 1.0 : sqrt(2.0); } /* Mandel weight */

/* 4-tensor with minor symmetries -> 6x6 Mandel matrix and back */
static void t4_to_mandel(const double T[3][3][3][3], double M[6][6]) {
    for (int a = 0; a < 6; a++)
        for (int b = 0; b < 6; b++) M[a][b] = mw(a) * mw(b) * T[VI[a]][VJ[a]][VI[b]][VJ[b]];
}
static void mandel_to_t4(const double M[6][6], double T[3][3][3][3]) {
    for (int a = 0; a < 6; a++)
        for (int b = 0; b < 6; b++) {
            double v = M[a][b] / (mw(a) * mw(b));
            int i = VI[a], j = VJ[a], k = VI[b], l = VJ[b];
            T[i][j][k][l] = T[j][i][k][l] = T[i][j][l][k] = T[j][i][l][k] = v;
        }
}
static double det3(const double A[3][3]) {
    return A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0]) +
           A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
}
static void inv3(const double A[3][3], double B[3][3]) {
    double d = det3(A);
    B[0][0] = (A[1][1] * A[2][2] - A[1][2] * A[2][1]) / d;
    B[0][1] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) / d;
    B[0][2] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) / d;
    B[1][0] = (A[1][2] * A[2][0] - A[1][0] * A[2][2]) / d;
    B[1][1] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) / d;
    B[1][2] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) / d;
    B[2][0] = (A[1][0] * A[2][1] - A[1][1] * A[2][0]) / d;
    B[2][1] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) / d;
    B[2][2] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) / d;
}
/* dense solve A x = b (n<=8), Gaussian elimination with partial pivoting; nrhs columns */
static int solve_dense(int n, double *A, double *B, int nrhs) {
    for (int c = 0; c < n; c++) {
        int p = c;
        for (int r = c + 1; r < n; r++)
            if (fabs(A[r * n + c]) > fabs(A[p * n + c])) p = r;
        if (A[p * n + c] == 0.0) return -1;
        if (p != c) {
            for (int k = 0; k < n; k++) { double t = A[c * n + k]; A[c * n + k] = A[p * n + k]; A[p * n + k] = t; }
            for (int k = 0; k < nrhs; k++) { double t = B[c * nrhs + k]; B[c * nrhs + k] = B[p * nrhs + k]; B[p * nrhs + k] = t; }
        }
        for (int r = c + 1; r < n; r++) {
            double f = A[r * n + c] / A[c * n + c];
            for (int k = c; k < n; k++) A[r * n + k] -= f * A[c * n + k];
            for (int k = 0; k < nrhs; k++) B[r * nrhs + k] -= f * B[c * nrhs + k];
        }
    }
    for (int k = 0; k < nrhs; k++)
        for (int r = n - 1; r >= 0; r--) {
            double s = B[r * nrhs + k];
            for (int c = r + 1; c < n; c++) s -= A[r * n + c] * B[c * nrhs + k];
            B[r * nrhs + k] = s / A[r * n + r];
        }
    return 0;
}

/* ------------------------------------------------- O1: hex8 shape data
 * N_I(xi) = 1/8 (1+xi xi_I)(1+eta eta_I)(1+zeta zeta_I)  (trilinear HEX-8; Eq.(28) :220).
 * Node order and Gauss order are the boundary's: q = kx+2ky+4kz,
 * bit=0 <-> -1/sqrt3, weights 1.  Returns w_q = det Jr; G[I][J] = dN_I/dX_J. */
static const double XI[8][3] = {{-1, -1, -1}, {1, -1, -1}, {1, 1, -1}, {-1, 1, -1},
                                {-1, -1, 1},  {1, -1, 1},  {1, 1, 1},  {-1, 1, 1}};
double orc_shape_grad(const double *X /*[8][3]*/, int q, double *G /*[8][3]*/) {
    const double g = 1.0 / sqrt(3.0);
    double xi[3] = {(q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g};
    double dN[8][3], Jr[3][3] = {{0}}, Ji[3][3];
    for (int I = 0; I < 8; I++) {
        double a = 1 + xi[0] * XI[I][0], b = 1 + xi[1] * XI[I][1], c = 1 + xi[2] * XI[I][2];
        dN[I][0] = 0.125 * XI[I][0] * b * c;
        dN[I][1] = 0.125 * a * XI[I][1] * c;
        dN[I][2] = 0.125 * a * b * XI[I][2];
    }
    for (int I = 0; I < 8; I++)
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) Jr[i][j] += X[I * 3 + i] * dN[I][j]; /* Jr = sum X_I (x) dN_I/dxi */
    inv3(Jr, Ji);
    for (int I = 0; I < 8; I++)
        for (int J = 0; J < 3; J++) {
            double s = 0;
            for (int k = 0; k < 3; k++) s += dN[I][k] * Ji[k][J]; /* G = dN/dxi . Jr^-1 */
            G[I * 3 + J] = s;
        }
    return det3(Jr);
}

/* ------------------------------------------------- O3: spectral decomposition
 * cyclic Jacobi on a symmetric 3x3: A = V diag(lam) V^T, V columns = eigenvectors. */
static void jacobi3(const double Ain[3][3], double lam[3], double V[3][3]) {
    double A[3][3];
    memcpy(A, Ain, sizeof(A));
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) V[i][j] = (i == j);
    for (int sweep = 0; sweep < 30; sweep++) {
        double off = fabs(A[0][1]) + fabs(A[0][2]) + fabs(A[1][2]);
        if (off == 0.0) break;
        for (int p = 0; p < 2; p++)
            for (int q = p + 1; q < 3; q++) {
                if (A[p][q] == 0.0) continue;
                double tau = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
                double t = (tau >= 0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                for (int k = 0; k < 3; k++) { /* A <- A J */
                    double akp = A[k][p], akq = A[k][q];
                    A[k][p] = c * akp - s * akq;
                    A[k][q] = s * akp + c * akq;
                }
                for (int k = 0; k < 3; k++) { /* A <- J^T A */
                    double apk = A[p][k], aqk = A[q][k];
                    A[p][k] = c * apk - s * aqk;
                    A[q][k] = s * apk + c * aqk;
                }
                A[p][q] = A[q][p] = 0.0;
                for (int k = 0; k < 3; k++) {
                    double vkp = V[k][p], vkq = V[k][q];
                    V[k][p] = c * vkp - s * vkq;
                    V[k][q] = s * vkp + c * vkq;
                }
            }
    }
    for (int i = 0; i < 3; i++) lam[i] = A[i][i];
}

/* eps = sum_a 1/2 ln(lam_a) n_a (x) n_a, lam_a = eig(C), C = F^T F
 * (Eq.(4)-(5) with the 1/2 restored, reading G1; Alg. C1 step 1 :894). */
void orc_logstrain(const double *F /*[3][3] row-major F_iJ*/, double *eps6, double *lam, double *R /*[3][3] columns=n_a*/) {
    double C[3][3], V[3][3], l[3], E[3][3] = {{0}};
    for (int I = 0; I < 3; I++)
        for (int J = 0; J < 3; J++) {
            double s = 0;
            for (int k = 0; k < 3; k++) s += F[k * 3 + I] * F[k * 3 + J];
            C[I][J] = s;
        }
    jacobi3(C, l, V);
    for (int a = 0; a < 3; a++)
        for (int I = 0; I < 3; I++)
            for (int J = 0; J < 3; J++) E[I][J] += 0.5 * log(l[a]) * V[I][a] * V[J][a];
    mat_to_sym6(E, eps6);
    for (int a = 0; a < 3; a++) lam[a] = l[a];
    memcpy(R, V, sizeof(V));
}

/* ------------------------------------------------- O4/O5/O6: material
 * Isotropic E (Eq.(8); the nine orthotropic d_i of :113 are never given, reading G6). */
static void elast_mandel(const double *mat, double E6[6][6]) {
    double E = mat[0], nu = mat[1], mu = E / (2 * (1 + nu)), la = E * nu / ((1 + nu) * (1 - 2 * nu));
    double T[3][3][3][3];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            for (int k = 0; k < 3; k++)
                for (int l = 0; l < 3; l++)
                    T[i][j][k][l] = la * (i == j) * (k == l) + mu * ((i == k) * (j == l) + (i == l) * (j == k));
    t4_to_mandel(T, E6);
}
/* rotation matrix from unit quaternion (w,x,y,z); columns = material axes in the global frame (reading G4) */
static void quat_to_rot(const double *q, double Th[3][3]) {
    double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    double w = q[0] / n, x = q[1] / n, y = q[2] / n, z = q[3] / n;
    Th[0][0] = 1 - 2 * (y * y + z * z); Th[0][1] = 2 * (x * y - w * z);     Th[0][2] = 2 * (x * z + w * y);
    Th[1][0] = 2 * (x * y + w * z);     Th[1][1] = 1 - 2 * (x * x + z * z); Th[1][2] = 2 * (y * z - w * x);
    Th[2][0] = 2 * (x * z - w * y);     Th[2][1] = 2 * (y * z + w * x);     Th[2][2] = 1 - 2 * (x * x + y * y);
}
/* Hill-48 tensor, PAPER.md:774-801 Eq.(A1)-(A5); (A2) read as tensor components
 * H1212 = p7/2 etc. (reading G3) so that T:H:T contains 2 p7 T12^2. */
void orc_hill_mandel(const double *mat, double *H36) {
    double r11 = mat[2], r22 = mat[3], r33 = mat[4], r12 = mat[5], r23 = mat[6], r13 = mat[7];
    double p1 = 2 / (3 * r11 * r11), p2 = 2 / (3 * r22 * r22), p3 = 2 / (3 * r33 * r33);
    double p7 = 1 / (r12 * r12), p8 = 1 / (r23 * r23), p9 = 1 / (r13 * r13);
    double p4 = 0.5 * (p3 - p1 - p2), p5 = 0.5 * (p1 - p2 - p3), p6 = 0.5 * (p2 - p1 - p3);
    double L[3][3][3][3], G[3][3][3][3], Th[3][3];
    memset(L, 0, sizeof(L));
    L[0][0][0][0] = p1; L[1][1][1][1] = p2; L[2][2][2][2] = p3;
    L[0][0][1][1] = L[1][1][0][0] = p4;
    L[1][1][2][2] = L[2][2][1][1] = p5;
    L[0][0][2][2] = L[2][2][0][0] = p6;
    L[0][1][0][1] = L[0][1][1][0] = L[1][0][0][1] = L[1][0][1][0] = 0.5 * p7;
    L[1][2][1][2] = L[1][2][2][1] = L[2][1][1][2] = L[2][1][2][1] = 0.5 * p8;
    L[0][2][0][2] = L[0][2][2][0] = L[2][0][0][2] = L[2][0][2][0] = 0.5 * p9;
    quat_to_rot(mat + 12, Th);
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            for (int k = 0; k < 3; k++)
                for (int l = 0; l < 3; l++) {
                    double s = 0;
                    for (int a = 0; a < 3; a++)
                        for (int b = 0; b < 3; b++)
                            for (int c = 0; c < 3; c++)
                                for (int d = 0; d < 3; d++) s += Th[i][a] * Th[j][b] * Th[k][c] * Th[l][d] * L[a][b][c][d];
                    G[i][j][k][l] = s;
                }
    double M[6][6];
    t4_to_mandel(G, M);
    memcpy(H36, M, sizeof(M));
}
/* flow stress: Voce sigma0+Q(1-exp(-b a)) (Eq.(10)), Swift K(eps0+a)^n (BASELINE.json configs) */
void orc_flow(const double *mat, double alpha, double *sig, double *dsig) {
    double h0 = mat[9], h1 = mat[10], h2 = mat[11];
    if (mat[8] == 0.0) { *sig = h0 + h1 * (1 - exp(-h2 * alpha)); *dsig = h1 * h2 * exp(-h2 * alpha); }
    else               { *sig = h0 * pow(h1 + alpha, h2);        *dsig = h0 * h2 * pow(h1 + alpha, h2 - 1); }
}
#define WHILL 0.816496580927726032732428024902 /* W = sqrt(2/3) */
/* sigma_y(alpha) = sqrt(2/3) sigma_flow(alpha): reading G2 (Eq.(10) vs (A3)) */
static void yield_stress(const double *mat, double alpha, double *sy, double *dsy) {
    double s, d;
    orc_flow(mat, alpha, &s, &d);
    *sy = WHILL * s; *dsy = WHILL * d;
}
static void to_mandel6(const double v[6], double m[6]) { for (int a = 0; a < 6; a++) m[a] = mw(a) * v[a]; }
static void from_mandel6(const double m[6], double v[6]) { for (int a = 0; a < 6; a++) v[a] = m[a] / mw(a); }
static void mv6(const double M[6][6], const double x[6], double y[6]) {
    for (int a = 0; a < 6; a++) { double s = 0; for (int b = 0; b < 6; b++) s += M[a][b] * x[b]; y[a] = s; }
}
static double dot6(const double a[6], const double b[6]) { double s = 0; for (int i = 0; i < 6; i++) s += a[i] * b[i]; return s; }

/* h(dgam) of O7: T(dgam) = (I + kappa E:H)^-1 : Ttr with kappa = dgam/sigma_y(alpha_n + W dgam);
 * returns phi(T) - sigma_y and dh/ddgam (implicit differentiation of the same 6x6 system). */
static double rm_h(const double E6[6][6], const double H6[6][6], const double *mat, const double Ttr[6], double alphan,
                   double dg, double T[6], double *dh) {
    double sy, dsy, A[36], B[12], EH[6][6], HT[6], EHT[6];
    yield_stress(mat, alphan + WHILL * dg, &sy, &dsy);
    double kap = dg / sy;
    for (int a = 0; a < 6; a++)
        for (int b = 0; b < 6; b++) { double s = 0; for (int c = 0; c < 6; c++) s += E6[a][c] * H6[c][b]; EH[a][b] = s; }
    for (int a = 0; a < 6; a++)
        for (int b = 0; b < 6; b++) A[a * 6 + b] = (a == b) + kap * EH[a][b];
    for (int a = 0; a < 6; a++) B[a * 2] = Ttr[a];
    { /* first solve for T, then the derivative rhs needs T: do two solves */
        double A1[36], b1[6];
        memcpy(A1, A, sizeof(A));
        for (int a = 0; a < 6; a++) b1[a] = Ttr[a];
        solve_dense(6, A1, b1, 1);
        for (int a = 0; a < 6; a++) T[a] = b1[a];
    }
    mv6(H6, T, HT);
    double phi = sqrt(dot6(T, HT));
    mv6(EH, T, EHT);
    { double A2[36], b2[6]; memcpy(A2, A, sizeof(A)); for (int a = 0; a < 6; a++) b2[a] = -EHT[a]; solve_dense(6, A2, b2, 1);
      /* dT/dkappa = b2 */
      double dkap = 1.0 / sy - dg * dsy * WHILL / (sy * sy);
      double N[6]; for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
      *dh = dot6(N, b2) * dkap - dsy * WHILL; }
    (void)B;
    return phi - sy;
}

/* O7 primary solver + O8 tangent.  All tensors 6 tensor components; Cep as 6x6 Mandel.
 * Returns 1 if plastic.  iters = number of h evaluations. */
int orc_return_map(const double *mat, const double *eps6, const double *epn6, double alphan, double *T6, double *epnew6,
                   double *alphanew, double *dgam_out, double *Cep36, int *iters, int *nonconv) {
    double E6[6][6], H6[6][6], ee[6], Ttr[6], HT[6], sy, dsy;
    elast_mandel(mat, E6);
    orc_hill_mandel(mat, &H6[0][0]);
    for (int a = 0; a < 6; a++) ee[a] = mw(a) * (eps6[a] - epn6[a]);
    mv6(E6, ee, Ttr);                                   /* Eq.(16) */
    mv6(H6, Ttr, HT);
    double phitr = sqrt(fmax(dot6(Ttr, HT), 0.0));      /* Eq.(11) :127 */
    yield_stress(mat, alphan, &sy, &dsy);
    *iters = 0; *nonconv = 0;
    if (phitr - sy <= 0.0) {                            /* Eq.(17)-(18) :165-172; tie -> elastic (G10) */
        from_mandel6(Ttr, T6);
        for (int a = 0; a < 6; a++) epnew6[a] = epn6[a];
        *alphanew = alphan; *dgam_out = 0.0;
        memcpy(Cep36, E6, sizeof(E6));
        return 0;
    }
    /* bracket the unique root of the strictly decreasing h: h(0)=ftr>0 */
    double T[6], dh, lo = 0.0, hi = (phitr - sy) / (2.0 * mat[0]) + 1e-12, hv;
    for (int k = 0; k < 200; k++) { hv = rm_h(E6, H6, mat, Ttr, alphan, hi, T, &dh); (*iters)++; if (hv < 0) break; lo = hi; hi *= 2.0; }
    double x = 0.5 * (lo + hi), tolh, ttrn = sqrt(dot6(Ttr, Ttr)), ehn = 0.0;
    for (int a = 0; a < 6; a++)
        for (int b = 0; b < 6; b++) { double s = 0; for (int c = 0; c < 6; c++) s += E6[a][c] * H6[c][b]; ehn += s * s; }
    ehn = sqrt(ehn);
    int done = 0;
    for (int k = 0; k < 200 && !done; k++) {
        hv = rm_h(E6, H6, mat, Ttr, alphan, x, T, &dh); (*iters)++;
        double sycur, d2; yield_stress(mat, alphan + WHILL * x, &sycur, &d2);
        /* round-off floor of h: the 6x6 solve T = (I + kappa E:H)^-1 Ttr carries the full |Ttr| (pressure part
           included) times its condition number <= 1 + kappa |E:H|_F  (stop at the floor, then polish) */
        tolh = 4.0 * 2.220446049250313e-16 * fmax(sycur, ttrn * (1.0 + x / sycur * ehn));
        if (fabs(hv) <= tolh) done = 1;
        if (hv > 0) lo = x; else hi = x;
        double xn = x - hv / dh;                        /* Newton step */
        int inside = (xn >= lo && xn <= hi);
        if (done) { if (inside) x = xn; break; }        /* the Newton step taken after the test is the polish step */
        if (!inside) xn = 0.5 * (lo + hi);              /* bisect if Newton leaves the bracket */
        if (fabs(xn - x) <= 4.0 * 2.220446049250313e-16 * fabs(x)) done = 1;   /* stagnation at round-off */
        x = xn;
    }
    if (!done) *nonconv = 1;
    hv = rm_h(E6, H6, mat, Ttr, alphan, x, T, &dh); (*iters)++;
    /* update, Eq.(19)-(20) :176-178; Alg. C2 step 27 :979 */
    double N[6], epm[6], Tm[6];
    mv6(H6, T, HT);
    double phi = sqrt(dot6(T, HT));
    for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
    for (int a = 0; a < 6; a++) epm[a] = mw(a) * epn6[a] + x * N[a];
    for (int a = 0; a < 6; a++) ee[a] = mw(a) * eps6[a] - epm[a];
    mv6(E6, ee, Tm);
    from_mandel6(Tm, T6);
    from_mandel6(epm, epnew6);
    *alphanew = alphan + WHILL * x; *dgam_out = x;
    /* O8: Xi = (E^-1 + dgam dN/dT)^-1, dN/dT = (H - N(x)N)/phi; Cep = Xi - (Xi N)(Xi N)/(N Xi N + W sy') (App. D :1002-1019) */
    mv6(H6, Tm, HT); phi = sqrt(dot6(Tm, HT));
    for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
    double A[36], Xi[36];
    { double Ei[36], Ecp[36]; memcpy(Ecp, E6, sizeof(E6));
      for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) Ei[a * 6 + b] = (a == b);
      solve_dense(6, Ecp, Ei, 6);
      for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) A[a * 6 + b] = Ei[a * 6 + b] + x * (H6[a][b] - N[a] * N[b]) / phi; }
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) Xi[a * 6 + b] = (a == b);
    solve_dense(6, A, Xi, 6);
    double XN[6], sy1, dsy1;
    for (int a = 0; a < 6; a++) { double s = 0; for (int b = 0; b < 6; b++) s += Xi[a * 6 + b] * N[b]; XN[a] = s; }
    yield_stress(mat, *alphanew, &sy1, &dsy1);
    double den = dot6(N, XN) + WHILL * dsy1;
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) Cep36[a * 6 + b] = Xi[a * 6 + b] - XN[a] * XN[b] / den;
    return 1;
}

/* ------------------------------------------------- Alg. C2 literal (cross-check solver, pin P12)
 * y = [T(6, Mandel), alpha, dgam] (reading G8), G of Eq.(23) PAPER.md:189 with the T rows and the f row
 * divided by sigma_y(alpha_n) (reading G7); J^G by hand; Goldstein line search of App. B
 * Eq.(B1)-(B7) :838-867 taken as printed (reading G11), beta=1e-4, eta=0.1 (:871).
 * Returns iterations used, or -1 if not converged in kmax. */
static void c2_G(const double E6[6][6], const double H6[6][6], const double *mat, const double em[6], const double epn[6],
                 double alphan, double s0, const double y[8], double G[8]) {
    double HT[6], N[6], ee[6], ET[6], sy, dsy;
    mv6(H6, y, HT);
    double phi = sqrt(dot6(y, HT));
    for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
    for (int a = 0; a < 6; a++) ee[a] = em[a] - epn[a] - y[7] * N[a];
    mv6(E6, ee, ET);
    for (int a = 0; a < 6; a++) G[a] = (y[a] - ET[a]) / s0;
    G[6] = y[6] - alphan - WHILL * y[7];
    yield_stress(mat, y[6], &sy, &dsy);
    G[7] = (phi - sy) / s0;
}
int orc_return_map_c2(const double *mat, const double *eps6, const double *epn6, double alphan, double tol, int kmax,
                      int jmax, double beta, double eta, double *T6, double *alphanew, double *dgam, double *resnorms /*[kmax+1]*/,
                      int *n_linesearch) {
    double E6[6][6], H6[6][6], em[6], epn[6], ee[6], y[8], G[8], s0, d0;
    elast_mandel(mat, E6);
    orc_hill_mandel(mat, &H6[0][0]);
    to_mandel6(eps6, em); to_mandel6(epn6, epn);
    for (int a = 0; a < 6; a++) ee[a] = em[a] - epn[a];
    mv6(E6, ee, y); y[6] = alphan; y[7] = 0.0;
    yield_stress(mat, alphan, &s0, &d0);
    *n_linesearch = 0;
    int k, conv = -1;
    for (k = 0; k <= kmax; k++) {
        c2_G(E6, H6, mat, em, epn, alphan, s0, y, G);
        double nrm = 0; for (int a = 0; a < 8; a++) nrm += G[a] * G[a]; nrm = sqrt(nrm);
        if (resnorms) resnorms[k] = nrm;
        if (nrm <= tol) { conv = k; break; }
        if (k == kmax) break;
        /* Jacobian rows: [I + dgam E:dN/dT, 0, E:N] ; [0,1,-W] ; [N, -sy', 0] (scaled like G) */
        double HT[6], N[6], J[64], rhs[8], sy, dsy;
        mv6(H6, y, HT);
        double phi = sqrt(dot6(y, HT));
        for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
        yield_stress(mat, y[6], &sy, &dsy);
        memset(J, 0, sizeof(J));
        for (int a = 0; a < 6; a++) {
            double EN = 0;
            for (int b = 0; b < 6; b++) {
                double s = 0;
                for (int c = 0; c < 6; c++) s += E6[a][c] * (H6[c][b] - N[c] * N[b]) / phi;
                J[a * 8 + b] = ((a == b) + y[7] * s) / s0;
                EN += E6[a][b] * N[b];
            }
            J[a * 8 + 7] = EN / s0;
        }
        J[6 * 8 + 6] = 1.0; J[6 * 8 + 7] = -WHILL;
        for (int b = 0; b < 6; b++) J[7 * 8 + b] = N[b] / s0;
        J[7 * 8 + 6] = -dsy / s0;
        for (int a = 0; a < 8; a++) rhs[a] = -G[a];
        if (solve_dense(8, J, rhs, 1)) break;
        /* line search */
        double psi0 = 0.5 * nrm * nrm, yt[8], Gt[8], zeta = 1.0;
        for (int a = 0; a < 8; a++) yt[a] = y[a] + rhs[a];
        c2_G(E6, H6, mat, em, epn, alphan, s0, yt, Gt);
        double psi1 = 0; for (int a = 0; a < 8; a++) psi1 += Gt[a] * Gt[a]; psi1 *= 0.5;
        if (!(psi1 < (1 - 2 * beta) * psi0)) {                       /* Eq.(B3) */
            (*n_linesearch)++;
            double zj = psi0 / (psi0 + psi1);                        /* Eq.(B5) */
            zeta = zj;
            for (int j = 0; j <= jmax; j++) {
                for (int a = 0; a < 8; a++) yt[a] = y[a] + zj * rhs[a];
                c2_G(E6, H6, mat, em, epn, alphan, s0, yt, Gt);
                double psij = 0; for (int a = 0; a < 8; a++) psij += Gt[a] * Gt[a]; psij *= 0.5;
                double zn = psi0 / (psi0 + psij);                    /* Eq.(B6) */
                zn = fmax(eta * zj, zn);                             /* Eq.(B7) */
                for (int a = 0; a < 8; a++) yt[a] = y[a] + zn * rhs[a];
                c2_G(E6, H6, mat, em, epn, alphan, s0, yt, Gt);
                double psin = 0; for (int a = 0; a < 8; a++) psin += Gt[a] * Gt[a]; psin *= 0.5;
                zeta = zn;
                if (psin < (1 - 2 * beta * zn) * psi0) break;
                zj = zn;
            }
        }
        for (int a = 0; a < 8; a++) y[a] += zeta * rhs[a];
    }
    from_mandel6(y, T6);
    *alphanew = y[6]; *dgam = y[7];
    return conv;
}

/* 8x8 implicit differentiation of App. D (PAPER.md:1002-1019 Eq.(D4)-(D6)) at a converged state:
 * solves J_y ydot = -dG/deps edot for the six unit strain directions and returns the T rows (6x6 Mandel). Pin P7. */
void orc_cep_implicit(const double *mat, const double *T6, double alpha, double dgam, double *Cep36) {
    double E6[6][6], H6[6][6], y[6], HT[6], N[6], J[64], B[48], sy, dsy;
    elast_mandel(mat, E6);
    orc_hill_mandel(mat, &H6[0][0]);
    to_mandel6(T6, y);
    mv6(H6, y, HT);
    double phi = sqrt(dot6(y, HT));
    for (int a = 0; a < 6; a++) N[a] = HT[a] / phi;
    yield_stress(mat, alpha, &sy, &dsy);
    memset(J, 0, sizeof(J)); memset(B, 0, sizeof(B));
    for (int a = 0; a < 6; a++) {
        double EN = 0;
        for (int b = 0; b < 6; b++) {
            double s = 0;
            for (int c = 0; c < 6; c++) s += E6[a][c] * (H6[c][b] - N[c] * N[b]) / phi;
            J[a * 8 + b] = (a == b) + dgam * s;
            EN += E6[a][b] * N[b];
            B[a * 6 + b] = E6[a][b];          /* -dG_T/deps = +E */
        }
        J[a * 8 + 7] = EN;
    }
    J[6 * 8 + 6] = 1.0; J[6 * 8 + 7] = -WHILL;
    for (int b = 0; b < 6; b++) J[7 * 8 + b] = N[b];
    J[7 * 8 + 6] = -dsy;
    solve_dense(8, J, B, 6);
    memcpy(Cep36, B, 36 * sizeof(double));
}

/* ------------------------------------------------- Yld2004-18p
 * Barlat record bar[20]: c'12,c'13,c'21,c'23,c'31,c'32,c'44,c'55,c'66, the same nine for C'', m, 0.
 * Eq.(A7)-(A9) PAPER.md:812-824: s = P:T (deviator), s' = C':s, s'' = C'':s in the material frame;
 * reading B1: the shear rows follow the component order of App. A.1 (c44 <-> 12, c55 <-> 23, c66 <-> 13), and the
 * fourth row of [C''] that the print drops (:822) is c''44;
 * Eq.(12) :133 read as phi = [1/4 sum_{i,j=1..3} |s'_i - s''_j|^m]^(1/m) (reading B2: the print repeats |s'3-s''3|
 * and omits |s'3-s''1|); yield function f = phi - sigma_flow(alpha), W = 1 (:145) — with all c = 1 phi is the
 * uniaxial-equivalent stress, so no sqrt(2/3) appears here (the Hill reading G2 makes the two models agree, :828).
 * Material orientation as for Hill: T_mat = Theta^T T Theta (:826, Eq.(A1) :774).
 * Derivatives are taken for EVEN INTEGER m (2..16; the paper uses 8, and 2, 4 for its reductions), where
 * |x|^m = x^m and Phi = sum_ij (a_i - b_j)^m = sum_k binom(m,k) (-1)^k tr(A^(m-k)) tr(B^k) is a polynomial of the
 * two transformed tensors A = s', B = s'' (power sums of the eigenvalues are traces of powers): its first and
 * second derivatives are written out with plain index loops, no eigenvectors, no repeated-eigenvalue cases. */
#define NBAR 20
static void barlat_maps(const double *bar, double LA[6][6], double LB[6][6]) {
    /* L' = C'.P and L'' = C''.P as 6x6 Mandel matrices (the shear blocks are diagonal, so Voigt = Mandel there) */
    double Pd[6][6];
    memset(Pd, 0, sizeof(Pd));
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) Pd[i][j] = ((i == j) ? 2.0 : -1.0) / 3.0;   /* Eq.(A8) :816 */
    for (int i = 3; i < 6; i++) Pd[i][i] = 1.0;
    for (int t = 0; t < 2; t++) {
        const double *c = bar + 9 * t;
        double Cm[6][6];
        memset(Cm, 0, sizeof(Cm));
        Cm[0][1] = -c[0]; Cm[0][2] = -c[1]; Cm[1][0] = -c[2]; Cm[1][2] = -c[3]; Cm[2][0] = -c[4]; Cm[2][1] = -c[5];  /* Eq.(A9) */
        Cm[3][3] = c[6]; Cm[4][4] = c[7]; Cm[5][5] = c[8];
        double (*L)[6] = t ? LB : LA;
        for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) { double s = 0; for (int k = 0; k < 6; k++) s += Cm[a][k] * Pd[k][b]; L[a][b] = s; }
    }
}
static void mandel_to_mat(const double m[6], double A[3][3]) { double v[6]; from_mandel6(m, v); sym6_to_mat(v, A); }
static void matmul3(const double A[3][3], const double B[3][3], double C[3][3]) {
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { double s = 0; for (int k = 0; k < 3; k++) s += A[i][k] * B[k][j]; C[i][j] = s; }
}
static double trace3(const double A[3][3]) { return A[0][0] + A[1][1] + A[2][2]; }
static double binom(int n, int k) { double b = 1; for (int i = 1; i <= k; i++) b = b * (n - k + i) / i; return b; }

/* phi by the DEFINITION: eigenvalues of s', s'' (any real m >= 1).  Tm = stress in the material frame, Mandel. */
double orc_barlat_phi_eig(const double *bar, const double *Tm) {
    double LA[6][6], LB[6][6], a6[6], b6[6], A[3][3], B[3][3], a[3], b[3], V[3][3], m = bar[18], s = 0;
    barlat_maps(bar, LA, LB);
    mv6(LA, Tm, a6); mv6(LB, Tm, b6);
    mandel_to_mat(a6, A); mandel_to_mat(b6, B);
    jacobi3(A, a, V); jacobi3(B, b, V);
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) s += pow(fabs(a[i] - b[j]), m);
    return pow(0.25 * s, 1.0 / m);
}
/* phi, N = dphi/dT (Mandel), Hm = d2phi/dT2 (6x6 Mandel, may be NULL) in the material frame, even integer m. */
void orc_barlat_derivs(const double *bar, const double *Tm, double *phi_out, double *Nm, double *Hm) {
    int m = (int)bar[18];
    double LA[6][6], LB[6][6], a6[6], b6[6];
    double PA[17][3][3], PB[17][3][3], tA[17], tB[17];
    barlat_maps(bar, LA, LB);
    mv6(LA, Tm, a6); mv6(LB, Tm, b6);
    memset(PA, 0, sizeof(PA)); memset(PB, 0, sizeof(PB));
    for (int i = 0; i < 3; i++) PA[0][i][i] = PB[0][i][i] = 1.0;
    mandel_to_mat(a6, PA[1]); mandel_to_mat(b6, PB[1]);
    for (int n = 2; n <= m; n++) { matmul3(PA[n - 1], PA[1], PA[n]); matmul3(PB[n - 1], PB[1], PB[n]); }
    for (int n = 0; n <= m; n++) { tA[n] = trace3(PA[n]); tB[n] = trace3(PB[n]); }
    double Phi = 0, GA[3][3], GB[3][3];
    memset(GA, 0, sizeof(GA)); memset(GB, 0, sizeof(GB));
    for (int k = 0; k <= m; k++) {
        double c = binom(m, k) * ((k & 1) ? -1.0 : 1.0);
        Phi += c * tA[m - k] * tB[k];
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
            if (k < m) GA[i][j] += c * (m - k) * tB[k] * PA[m - k - 1][i][j];    /* d tr(A^n)/dA = n A^(n-1) */
            if (k > 0) GB[i][j] += c * k * tA[m - k] * PB[k - 1][i][j];
        }
    }
    double phi = pow(0.25 * Phi, 1.0 / m);
    double ga[6], gb[6], gam[6], gbm[6], dPhi[6];
    mat_to_sym6(GA, ga); mat_to_sym6(GB, gb); to_mandel6(ga, gam); to_mandel6(gb, gbm);
    for (int a = 0; a < 6; a++) { double s = 0; for (int b = 0; b < 6; b++) s += LA[b][a] * gam[b] + LB[b][a] * gbm[b]; dPhi[a] = s; }
    double cf = pow(phi, 1.0 - m) / (4.0 * m);      /* phi^m = Phi/4  =>  dphi = phi^(1-m)/(4m) dPhi */
    for (int a = 0; a < 6; a++) Nm[a] = cf * dPhi[a];
    *phi_out = phi;
    if (!Hm) return;
    /* second derivatives of Phi with respect to (A,A), (A,B), (B,B) as 4-tensors, then Mandel and the chain rule */
    double HAA[3][3][3][3], HBB[3][3][3][3], HAB[3][3][3][3];
    memset(HAA, 0, sizeof(HAA)); memset(HBB, 0, sizeof(HBB)); memset(HAB, 0, sizeof(HAB));
    for (int k = 0; k <= m; k++) {
        double c = binom(m, k) * ((k & 1) ? -1.0 : 1.0);
        int n = m - k - 1;                            /* GA term: c (m-k) tB[k] A^n ; d(A^n) = sum_r A^r dA A^(n-1-r) */
        for (int r = 0; n >= 1 && r < n; r++)
            for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int p = 0; p < 3; p++) for (int q = 0; q < 3; q++)
                HAA[i][j][p][q] += c * (m - k) * tB[k] * 0.5 * (PA[r][i][p] * PA[n - 1 - r][q][j] + PA[r][i][q] * PA[n - 1 - r][p][j]);
        int nb = k - 1;                               /* GB term: c k tA[m-k] B^nb */
        for (int r = 0; nb >= 1 && r < nb; r++)
            for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int p = 0; p < 3; p++) for (int q = 0; q < 3; q++)
                HBB[i][j][p][q] += c * k * tA[m - k] * 0.5 * (PB[r][i][p] * PB[nb - 1 - r][q][j] + PB[r][i][q] * PB[nb - 1 - r][p][j]);
        if (k >= 1 && k < m)                          /* d/dB of tB[k] = k B^(k-1) */
            for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int p = 0; p < 3; p++) for (int q = 0; q < 3; q++)
                HAB[i][j][p][q] += c * (m - k) * k * PA[m - k - 1][i][j] * PB[k - 1][p][q];
    }
    double MAA[6][6], MBB[6][6], MAB[6][6], d2Phi[6][6];
    t4_to_mandel(HAA, MAA); t4_to_mandel(HBB, MBB); t4_to_mandel(HAB, MAB);
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) {
        double s = 0;
        for (int c = 0; c < 6; c++) for (int d = 0; d < 6; d++)
            s += LA[c][a] * MAA[c][d] * LA[d][b] + LB[c][a] * MBB[c][d] * LB[d][b] + LA[c][a] * MAB[c][d] * LB[d][b] +
                 LB[c][a] * MAB[d][c] * LA[d][b];
        d2Phi[a][b] = s;
    }
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++)
        Hm[a * 6 + b] = cf * d2Phi[a][b] - (m - 1.0) / phi * Nm[a] * Nm[b];
}
/* 6x6 Mandel matrix Q of the frame change X_mat = Theta^T X Theta (X_mat = Q X_glob); Q is orthogonal */
static void mandel_rot(const double Th[3][3], double Q[6][6]) {
    double R4[3][3][3][3];
    for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++)
        R4[a][b][i][j] = 0.5 * (Th[i][a] * Th[j][b] + Th[j][a] * Th[i][b]);
    t4_to_mandel(R4, Q);
}
/* Yield function of either model in the GLOBAL frame: T6 tensor components -> phi, N (Mandel), H = dN/dT (6x6 Mandel
 * or NULL).  bar == NULL: Hill-48 (phi = sqrt(T:H:T), Eq.(11) :127). */
void orc_yield_eval(const double *mat, const double *bar, const double *T6, double *phi, double *N, double *H) {
    double Tg[6];
    to_mandel6(T6, Tg);
    if (!bar) {
        double H6[6][6], HT[6];
        orc_hill_mandel(mat, &H6[0][0]);
        mv6(H6, Tg, HT);
        *phi = sqrt(dot6(Tg, HT));
        for (int a = 0; a < 6; a++) N[a] = HT[a] / *phi;
        if (H) for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) H[a * 6 + b] = (H6[a][b] - N[a] * N[b]) / *phi;
        return;
    }
    double Th[3][3], Q[6][6], Tm[6], Nm[6], Hm[36];
    quat_to_rot(mat + 12, Th);
    mandel_rot(Th, Q);
    mv6(Q, Tg, Tm);
    orc_barlat_derivs(bar, Tm, phi, Nm, H ? Hm : NULL);
    for (int a = 0; a < 6; a++) { double s = 0; for (int b = 0; b < 6; b++) s += Q[b][a] * Nm[b]; N[a] = s; }
    if (H) for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) {
        double s = 0;
        for (int c = 0; c < 6; c++) for (int d = 0; d < 6; d++) s += Q[c][a] * Hm[c * 6 + d] * Q[d][b];
        H[a * 6 + b] = s;
    }
}
/* sigma_y(alpha) and W of Eq.(14)/(20): Hill sqrt(2/3) sigma_flow, W = sqrt(2/3); Barlat sigma_flow, W = 1 (:145) */
static double yld_W(const double *bar) { return bar ? 1.0 : WHILL; }
static void yld_sy(const double *mat, const double *bar, double alpha, double *sy, double *dsy) {
    double s, d;
    orc_flow(mat, alpha, &s, &d);
    *sy = yld_W(bar) * s; *dsy = yld_W(bar) * d;
}
/* G(y) of Eq.(23), y = [T (Mandel), alpha, dgam]; T rows and f row divided by s0 = sigma_y(alpha_n) (G7) */
static void gen_G(const double E6[6][6], const double *mat, const double *bar, const double em[6], const double epn[6],
                  double alphan, double s0, const double y[8], double G[8]) {
    double T6[6], N[6], ee[6], ET[6], phi, sy, dsy;
    from_mandel6(y, T6);
    orc_yield_eval(mat, bar, T6, &phi, N, NULL);
    for (int a = 0; a < 6; a++) ee[a] = em[a] - epn[a] - y[7] * N[a];
    mv6(E6, ee, ET);
    for (int a = 0; a < 6; a++) G[a] = (y[a] - ET[a]) / s0;
    G[6] = y[6] - alphan - yld_W(bar) * y[7];
    yld_sy(mat, bar, y[6], &sy, &dsy);
    G[7] = (phi - sy) / s0;
}
/* J^G = dG/dy (paper: by AD, :200; here from the hand-written second derivative), same row scaling as gen_G */
static void gen_J(const double E6[6][6], const double *mat, const double *bar, double s0, const double y[8], double J[64]) {
    double T6[6], N[6], H[36], phi, sy, dsy;
    from_mandel6(y, T6);
    orc_yield_eval(mat, bar, T6, &phi, N, H);
    yld_sy(mat, bar, y[6], &sy, &dsy);
    memset(J, 0, 64 * sizeof(double));
    for (int a = 0; a < 6; a++) {
        double EN = 0;
        for (int b = 0; b < 6; b++) {
            double s = 0;
            for (int c = 0; c < 6; c++) s += E6[a][c] * H[c * 6 + b];
            J[a * 8 + b] = ((a == b) + y[7] * s) / s0;
            EN += E6[a][b] * N[b];
        }
        J[a * 8 + 7] = EN / s0;
    }
    J[6 * 8 + 6] = 1.0; J[6 * 8 + 7] = -yld_W(bar);
    for (int b = 0; b < 6; b++) J[7 * 8 + b] = N[b] / s0;
    J[7 * 8 + 6] = -dsy / s0;
}
/* Alg. C1 steps 2-8 with Alg. C2 step by step for either yield function: elastic predictor, yield
 * test, Newton on the eight unknowns with the Goldstein line search of App. B Eq.(B1)-(B7) as printed (beta, eta of
 * :871), recovery (step 27), then C_ep by the implicit differentiation of App. D Eq.(D4)-(D6) :1002-1019.
 * Iterations run to the round-off floor: stop when |G| <= tol, or when |G| no longer halves after it fell below 1e-9.
 * trace (may be NULL) [kmax+1][3] = psi(0), psi(1), accepted zeta of every iteration (NaN-filled beyond the last).
 * Returns 1 if plastic. */
int orc_return_map_gen(const double *mat, const double *bar, const double *eps6, const double *epn6, double alphan,
                       double tol, int kmax, int jmax, double beta, double eta, double *T6, double *epnew6,
                       double *alphanew, double *dgam_out, double *Cep36, int *iters, int *nonconv, double *trace) {
    double E6[6][6], em[6], epn[6], ee[6], y[8], G[8], s0, d0, phitr, Ntr[6], Ttr6[6];
    elast_mandel(mat, E6);
    to_mandel6(eps6, em); to_mandel6(epn6, epn);
    for (int a = 0; a < 6; a++) ee[a] = em[a] - epn[a];
    mv6(E6, ee, y); y[6] = alphan; y[7] = 0.0;                       /* Eq.(16) :160; Alg. C2 steps 1-2 */
    from_mandel6(y, Ttr6);
    *iters = 0; *nonconv = 0;
    if (trace) for (int k = 0; k < 3 * (kmax + 1); k++) trace[k] = NAN;
    yld_sy(mat, bar, alphan, &s0, &d0);
    {
        double nrm2 = dot6(y, y);
        if (nrm2 == 0.0) phitr = 0.0; else orc_yield_eval(mat, bar, Ttr6, &phitr, Ntr, NULL);
    }
    if (phitr - s0 <= 0.0) {                                         /* Eq.(17)-(18) :165-172, tie -> elastic (G10) */
        memcpy(T6, Ttr6, sizeof(Ttr6));
        for (int a = 0; a < 6; a++) epnew6[a] = epn6[a];
        *alphanew = alphan; *dgam_out = 0.0;
        memcpy(Cep36, E6, sizeof(E6));
        return 0;
    }
    double prev = INFINITY;
    int conv = 0;
    for (int k = 0; k <= kmax; k++) {
        gen_G(E6, mat, bar, em, epn, alphan, s0, y, G);
        double nrm = 0; for (int a = 0; a < 8; a++) nrm += G[a] * G[a]; nrm = sqrt(nrm);
        *iters = k;
        if (nrm <= tol || (prev <= 1e-9 && nrm >= 0.5 * prev)) { conv = 1; break; }
        if (k == kmax) break;
        prev = nrm;
        double J[64], rhs[8];
        gen_J(E6, mat, bar, s0, y, J);
        for (int a = 0; a < 8; a++) rhs[a] = -G[a];
        if (solve_dense(8, J, rhs, 1)) break;                        /* Eq.(24) :196 */
        double psi0 = 0.5 * nrm * nrm, yt[8], Gt[8], zeta = 1.0;
        for (int a = 0; a < 8; a++) yt[a] = y[a] + rhs[a];
        gen_G(E6, mat, bar, em, epn, alphan, s0, yt, Gt);
        double psi1 = 0; for (int a = 0; a < 8; a++) psi1 += Gt[a] * Gt[a]; psi1 *= 0.5;
        if (!(psi1 < (1 - 2 * beta) * psi0)) {                       /* Eq.(B3) :852 */
            double zj = psi0 / (psi0 + psi1);                        /* Eq.(B5) :858 */
            zeta = zj;
            for (int j = 0; j <= jmax; j++) {
                for (int a = 0; a < 8; a++) yt[a] = y[a] + zj * rhs[a];
                gen_G(E6, mat, bar, em, epn, alphan, s0, yt, Gt);
                double psij = 0; for (int a = 0; a < 8; a++) psij += Gt[a] * Gt[a]; psij *= 0.5;
                if (j == 0 && psij < (1 - 2 * beta * zj) * psi0) break;   /* the first trial already passes Eq.(B3) */
                double zn = psi0 / (psi0 + psij);                    /* Eq.(B6) :862 */
                zn = fmax(eta * zj, zn);                             /* Eq.(B7) :866 */
                for (int a = 0; a < 8; a++) yt[a] = y[a] + zn * rhs[a];
                gen_G(E6, mat, bar, em, epn, alphan, s0, yt, Gt);
                double psin = 0; for (int a = 0; a < 8; a++) psin += Gt[a] * Gt[a]; psin *= 0.5;
                zeta = zn;
                if (psin < (1 - 2 * beta * zn) * psi0) break;
                zj = zn;
            }
        }
        if (trace) { trace[3 * k] = psi0; trace[3 * k + 1] = psi1; trace[3 * k + 2] = zeta; }
        for (int a = 0; a < 8; a++) y[a] += zeta * rhs[a];
    }
    if (!conv) *nonconv = 1;
    /* Alg. C2 step 27 :979: eps_p = eps_p_n + dgam N, T = E:(eps - eps_p) */
    double Tc6[6], N[6], phi, epm[6], Tm[6];
    from_mandel6(y, Tc6);
    orc_yield_eval(mat, bar, Tc6, &phi, N, NULL);
    for (int a = 0; a < 6; a++) epm[a] = epn[a] + y[7] * N[a];
    for (int a = 0; a < 6; a++) ee[a] = em[a] - epm[a];
    mv6(E6, ee, Tm);
    from_mandel6(Tm, T6);
    from_mandel6(epm, epnew6);
    *alphanew = y[6]; *dgam_out = y[7];
    /* App. D: J_y ydot = -dG/deps edot, unscaled rows; the T rows of the solution are C_ep (6x6 Mandel) */
    double yc[8], J[64], B[48];
    for (int a = 0; a < 6; a++) yc[a] = Tm[a];
    yc[6] = y[6]; yc[7] = y[7];
    gen_J(E6, mat, bar, 1.0, yc, J);
    memset(B, 0, sizeof(B));
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) B[a * 6 + b] = E6[a][b];
    solve_dense(8, J, B, 6);
    memcpy(Cep36, B, 36 * sizeof(double));
    return 1;
}

/* ------------------------------------------------- O9: divided differences of g(lam) = 1/2 ln(lam)
 * first:  g[a,b] = 1/2 log1p((lb-la)/la)/(lb-la),  g[a,a] = 1/(2 la)
 * second: recursive formula on the widest gap; series about the mean when the spread is small:
 *   g(m(1+x)) = c + 1/2 sum_{n>=1} (-1)^(n+1) x^n/n  =>  g[a,b,c] = 1/(2 m^2) sum_{n>=2} (-1)^(n+1)/n h_{n-2}(xa,xb,xc)
 *   (h_k = complete homogeneous symmetric polynomial = second divided difference of x^(k+2)). */
static double dd1(double la, double lb) {
    double d = lb - la;
    if (d == 0.0) return 0.5 / la;
    return 0.5 * log1p(d / la) / d;
}
static double hpoly3(int k, double x1, double x2, double x3) {
    /* sum over i+j+l=k of x1^i x2^j x3^l */
    double s = 0;
    for (int i = 0; i <= k; i++)
        for (int j = 0; i + j <= k; j++) s += pow(x1, i) * pow(x2, j) * pow(x3, k - i - j);
    return s;
}
static double dd2(double la, double lb, double lc) {
    double mx = fmax(la, fmax(lb, lc)), mn = fmin(la, fmin(lb, lc)), m = (la + lb + lc) / 3.0;
    if (mx - mn < 1e-2 * m) {
        double xa = (la - m) / m, xb = (lb - m) / m, xc = (lc - m) / m, s = 0;
        for (int n = 2; n <= 14; n++) s += ((n % 2) ? 1.0 : -1.0) / n * hpoly3(n - 2, xa, xb, xc);
        return 0.5 * s / (m * m);
    }
    /* order so that (p,r) is the widest gap, q the middle */
    double p = mn, r = mx, q = la + lb + lc - mn - mx;
    return (dd1(p, q) - dd1(q, r)) / (p - r);
}
void orc_divdiff(const double *lam, double *th /*[3][3]*/, double *ga /*[3][3][3]*/) {
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) {
            th[a * 3 + b] = dd1(lam[a], lam[b]);
            for (int c = 0; c < 3; c++) ga[(a * 3 + b) * 3 + c] = dd2(lam[a], lam[b], lam[c]);
        }
}
static void rot4(const double Q[3][3], const double A[3][3][3][3], double B[3][3][3][3]) {
    /* B_ijkl = Q_ia Q_jb Q_kc Q_ld A_abcd */
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int k = 0; k < 3; k++) for (int l = 0; l < 3; l++) {
        double s = 0;
        for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) for (int c = 0; c < 3; c++) for (int d = 0; d < 3; d++)
            s += Q[i][a] * Q[j][b] * Q[k][c] * Q[l][d] * A[a][b][c][d];
        B[i][j][k][l] = s;
    }
}
/* S = P_L : T and C_L = P_L^T : Cep : P_L + T : L_L  (Eq.(25) :204; analytic route of :288).
 * In the eigenbasis of C: S^_ab = 2 g[a,b] T^_ab ;
 * A^:(T:L_L):B^ = 4 sum_abc T^_ab g[a,b,c] (A^_ac B^_cb + B^_ac A^_cb). */
void orc_postprocess(const double *lam, const double *Rm /*[3][3]*/, const double *T6, const double *Cep36, double *S6,
                     double *CL36) {
    double R[3][3], Rt[3][3], T[3][3], Th[3][3] = {{0}}, Sh[3][3], S[3][3] = {{0}}, th[9], ga[27];
    memcpy(R, Rm, sizeof(R));
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) Rt[i][j] = R[j][i];
    sym6_to_mat(T6, T);
    orc_divdiff(lam, th, ga);
    for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++)
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) Th[a][b] += R[i][a] * T[i][j] * R[j][b];
    for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) Sh[a][b] = 2 * th[a * 3 + b] * Th[a][b];
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++)
        for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) S[i][j] += R[i][a] * Sh[a][b] * R[j][b];
    mat_to_sym6(S, S6);
    double Cm[6][6], C4[3][3][3][3], Ch[3][3][3][3], Gm[3][3][3][3], CLh[3][3][3][3], CL[3][3][3][3], out[6][6];
    memcpy(Cm, Cep36, sizeof(Cm));
    mandel_to_t4(Cm, C4);
    rot4(Rt, C4, Ch);                       /* hat components: C^_abcd = R_ia R_jb R_kc R_ld C_ijkl */
    memset(Gm, 0, sizeof(Gm));
    for (int p = 0; p < 3; p++) for (int q = 0; q < 3; q++) for (int r = 0; r < 3; r++) for (int s = 0; s < 3; s++) {
        /* unsymmetrised coefficient of A^_pq B^_rs, then averaged over p<->q and r<->s */
        double v = 0;
        int P[2] = {p, q}, Q[2] = {q, p}, Rr[2] = {r, s}, Ss[2] = {s, r};
        for (int x = 0; x < 2; x++) for (int y = 0; y < 2; y++) {
            int pp = P[x], qq = Q[x], rr = Rr[y], ss = Ss[y];
            v += 4.0 * ((qq == rr) * Th[pp][ss] * ga[(pp * 3 + ss) * 3 + qq] + (pp == ss) * Th[rr][qq] * ga[(rr * 3 + qq) * 3 + pp]);
        }
        Gm[p][q][r][s] = 0.25 * v;
    }
    for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) for (int c = 0; c < 3; c++) for (int d = 0; d < 3; d++)
        CLh[a][b][c][d] = 2 * th[a * 3 + b] * Ch[a][b][c][d] * 2 * th[c * 3 + d] + Gm[a][b][c][d];
    rot4(R, CLh, CL);
    t4_to_mandel(CL, out);
    memcpy(CL36, out, sizeof(out));
}

/* ------------------------------------------------- Alg. C1 at one point + O10
 * in: F (row-major F_iJ), hist_in (ep6, alpha), mat.  out: P[3][3], A[3][3][3][3] = dP_iJ/dF_kL, hist_out[7].
 * flags: bit0 plastic, bit1 local solve not converged, bit2 det F <= 0. */
static const double *g_dummy_bar = 0;
int orc_point_yld(const double *mat, const double *bar, const double *F, const double *hin, double *P, double *A, double *hout,
                  double *S6out, double *T6out, double *CL36out, int *iters);
int orc_point(const double *mat, const double *F, const double *hin, double *P, double *A, double *hout, double *S6out,
              double *T6out, double *CL36out, int *iters) {
    return orc_point_yld(mat, g_dummy_bar, F, hin, P, A, hout, S6out, T6out, CL36out, iters);
}
/* bar == NULL: Hill-48 (bracketed scalar solver); else Yld2004-18p through Alg. C2 (orc_return_map_gen) */
int orc_point_yld(const double *mat, const double *bar, const double *F, const double *hin, double *P, double *A, double *hout,
                  double *S6out, double *T6out, double *CL36out, int *iters) {
    double eps[6], lam[3], R[9], T6[6], Cep[36], S6[6], CL[36], dg, an;
    int nonconv, flags = 0;
    double Fm[3][3];
    memcpy(Fm, F, sizeof(Fm));
    if (det3(Fm) <= 0.0) flags |= 4;
    orc_logstrain(F, eps, lam, R);
    int pl = bar ? orc_return_map_gen(mat, bar, eps, hin, hin[6], 1e-14, 100, 20, 1e-4, 0.1, T6, hout, &an, &dg, Cep, iters,
                                      &nonconv, NULL)
                 : orc_return_map(mat, eps, hin, hin[6], T6, hout, &an, &dg, Cep, iters, &nonconv);
    hout[6] = an;
    if (pl) flags |= 1;
    if (nonconv) flags |= 2;
    orc_postprocess(lam, R, T6, Cep, S6, CL);
    double S[3][3], CLm[6][6], C4[3][3][3][3];
    sym6_to_mat(S6, S);
    memcpy(CLm, CL, sizeof(CLm));
    mandel_to_t4(CLm, C4);
    for (int i = 0; i < 3; i++) for (int J = 0; J < 3; J++) {
        double s = 0;
        for (int K = 0; K < 3; K++) s += F[i * 3 + K] * S[K][J];       /* P = F S, Eq.(26) :208 */
        P[i * 3 + J] = s;
    }
    for (int i = 0; i < 3; i++) for (int J = 0; J < 3; J++) for (int k = 0; k < 3; k++) for (int L = 0; L < 3; L++) {
        double s = (i == k) * S[J][L];
        for (int M = 0; M < 3; M++) for (int N = 0; N < 3; N++) s += F[i * 3 + M] * F[k * 3 + N] * C4[M][J][N][L];
        A[((i * 3 + J) * 3 + k) * 3 + L] = s;
    }
    if (S6out) memcpy(S6out, S6, sizeof(S6));
    if (T6out) memcpy(T6out, T6, sizeof(T6));
    if (CL36out) memcpy(CL36out, CL, sizeof(CL));
    return flags;
}

/* ------------------------------------------------- O11: element vectors (Eq.(35), :267 Eq.(37))
 * X[8][3], u[8][3], hin[8][7] -> Re[24], Ke[24][24] (a = 3*I+i), hout[8][7].
 * fbar=1: Eq.(31)-(32) :237-243, residual contracts P(Fbar) directly with grad N (reading G12).
 * stats[0..3] += plastic, nonconverged, detF<=0, (unused); returns max local iterations. */
int orc_element_yld(const double *X, const double *u, const double *hin, const double *mat, const double *bar, int fbar,
                    double *Re, double *Ke, double *hout, long long *stats);
int orc_element(const double *X, const double *u, const double *hin, const double *mat, int fbar, double *Re, double *Ke,
                double *hout, long long *stats) {
    return orc_element_yld(X, u, hin, mat, g_dummy_bar, fbar, Re, Ke, hout, stats);
}
int orc_element_yld(const double *X, const double *u, const double *hin, const double *mat, const double *bar, int fbar,
                    double *Re, double *Ke, double *hout, long long *stats) {
    double G[8][24], w[8], F[8][9], Jq[8], V = 0, Jbar = 0;
    int maxit = 0;
    memset(Re, 0, 24 * sizeof(double));
    memset(Ke, 0, 576 * sizeof(double));
    for (int q = 0; q < 8; q++) {
        w[q] = orc_shape_grad(X, q, G[q]);
        for (int i = 0; i < 3; i++) for (int J = 0; J < 3; J++) {
            double s = (i == J);
            for (int I = 0; I < 8; I++) s += u[I * 3 + i] * G[q][I * 3 + J];   /* Eq.(3) :88, Eq.(30) :228 */
            F[q][i * 3 + J] = s;
        }
        double Fm[3][3]; memcpy(Fm, F[q], sizeof(Fm));
        Jq[q] = det3(Fm);
        V += w[q]; Jbar += w[q] * Jq[q];
    }
    Jbar /= V;
    double gbar[24] = {0}, gq[8][24];
    if (fbar) {
        for (int q = 0; q < 8; q++) {
            double Fm[3][3], Fi[3][3]; memcpy(Fm, F[q], sizeof(Fm)); inv3(Fm, Fi);
            for (int K = 0; K < 8; K++) for (int k = 0; k < 3; k++) {
                double s = 0;
                for (int L = 0; L < 3; L++) s += G[q][K * 3 + L] * Fi[L][k];
                gq[q][K * 3 + k] = s;
                gbar[K * 3 + k] += w[q] * Jq[q] * s / (Jbar * V);
            }
        }
    }
    for (int q = 0; q < 8; q++) {
        double Fb[9], c = 1.0, P[9], A[81];
        int it;
        if (fbar) c = cbrt(Jbar / Jq[q]);
        for (int m = 0; m < 9; m++) Fb[m] = c * F[q][m];
        int fl = orc_point_yld(mat, bar, Fb, hin + q * 7, P, A, hout + q * 7, 0, 0, 0, &it);
        if (it > maxit) maxit = it;
        if (stats) { stats[0] += fl & 1; stats[1] += (fl >> 1) & 1; stats[2] += (Jq[q] <= 0.0); }
        for (int I = 0; I < 8; I++) for (int i = 0; i < 3; i++) {
            double s = 0;
            for (int J = 0; J < 3; J++) s += P[i * 3 + J] * G[q][I * 3 + J];
            Re[I * 3 + i] += w[q] * s;
        }
        for (int I = 0; I < 8; I++) for (int i = 0; i < 3; i++) for (int K = 0; K < 8; K++) for (int k = 0; k < 3; k++) {
            double s = 0;
            for (int J = 0; J < 3; J++) for (int L = 0; L < 3; L++)
                s += G[q][I * 3 + J] * A[((i * 3 + J) * 3 + k) * 3 + L] * G[q][K * 3 + L];
            Ke[(I * 3 + i) * 24 + K * 3 + k] += w[q] * c * s;
        }
        if (fbar) {
            double AF[9], r[24];
            for (int i = 0; i < 3; i++) for (int J = 0; J < 3; J++) {
                double s = 0;
                for (int k = 0; k < 3; k++) for (int L = 0; L < 3; L++) s += A[((i * 3 + J) * 3 + k) * 3 + L] * Fb[k * 3 + L];
                AF[i * 3 + J] = s;
            }
            for (int I = 0; I < 8; I++) for (int i = 0; i < 3; i++) {
                double s = 0;
                for (int J = 0; J < 3; J++) s += G[q][I * 3 + J] * AF[i * 3 + J];
                r[I * 3 + i] = s;
            }
            for (int a = 0; a < 24; a++) for (int b = 0; b < 24; b++)
                Ke[a * 24 + b] += w[q] * r[a] * (gbar[b] - gq[q][b]) / 3.0;
        }
    }
    return maxit;
}

/* ------------------------------------------------- O12: CSR pattern (triplets PAPER.md:296-298; Alg. E1 :1039-1049)
 * rows = 3 n_nodes; per row sorted unique columns; structural zeros kept.  Two-call protocol:
 * col_idx == NULL -> fills row_ptr and returns nnz; else fills col_idx and elem_slot. */
static int cmp_int(const void *a, const void *b) { int x = *(const int *)a, y = *(const int *)b; return (x > y) - (x < y); }
long long orc_pattern(long long n_nodes, long long n_elems, const int *conn, int *row_ptr, int *col_idx, int *elem_slot) {
    long long *cnt = calloc(n_nodes + 1, sizeof(long long));
    for (long long e = 0; e < n_elems; e++) for (int a = 0; a < 8; a++) cnt[conn[e * 8 + a] + 1] += 8;
    for (long long n = 0; n < n_nodes; n++) cnt[n + 1] += cnt[n];
    int *nb = malloc(cnt[n_nodes] * sizeof(int));
    long long *fill = malloc(n_nodes * sizeof(long long));
    for (long long n = 0; n < n_nodes; n++) fill[n] = cnt[n];
    for (long long e = 0; e < n_elems; e++) for (int a = 0; a < 8; a++) for (int b = 0; b < 8; b++)
        nb[fill[conn[e * 8 + a]]++] = conn[e * 8 + b];
    long long *nstart = malloc((n_nodes + 1) * sizeof(long long));
    nstart[0] = 0;
    for (long long n = 0; n < n_nodes; n++) {           /* sort + unique neighbour nodes in place */
        int *p = nb + cnt[n]; long long m = cnt[n + 1] - cnt[n], k = 0;
        qsort(p, m, sizeof(int), cmp_int);
        for (long long i = 0; i < m; i++) if (i == 0 || p[i] != p[i - 1]) p[k++] = p[i];
        fill[n] = k;
        nstart[n + 1] = nstart[n] + k;
    }
    long long nnz = 9 * nstart[n_nodes];
    row_ptr[0] = 0;
    for (long long n = 0; n < n_nodes; n++) for (int i = 0; i < 3; i++)
        row_ptr[3 * n + i + 1] = row_ptr[3 * n + i] + 3 * (int)fill[n];
    if (col_idx) {
        for (long long n = 0; n < n_nodes; n++) for (int i = 0; i < 3; i++) {
            int *c = col_idx + row_ptr[3 * n + i];
            for (long long j = 0; j < fill[n]; j++) for (int k = 0; k < 3; k++) c[3 * j + k] = 3 * nb[cnt[n] + j] + k;
        }
        if (elem_slot)
            for (long long e = 0; e < n_elems; e++) for (int a = 0; a < 24; a++) for (int b = 0; b < 24; b++) {
                int row = 3 * conn[e * 8 + a / 3] + a % 3, col = 3 * conn[e * 8 + b / 3] + b % 3;
                const int *c = col_idx + row_ptr[row];
                int len = row_ptr[row + 1] - row_ptr[row], s = -1;
                for (int j = 0; j < len; j++) if (c[j] == col) { s = row_ptr[row] + j; break; }   /* plain linear search */
                elem_slot[e * 576 + a * 24 + b] = s;
            }
    }
    free(cnt); free(nb); free(fill); free(nstart);
    return nnz;
}

/* ------------------------------------------------- O13: whole-mesh assemble (Eq.(34) :253, Eq.(38) :274)
 * Elements evaluated in parallel chunks; contributions added in ascending element id in long double,
 * rounded once; outputs overwritten.  mat: n_mat == 1 (uniform) or n_elems records.
 * stats[0..3] = plastic, nonconverged, detF<=0, max local iterations. */
int orc_assemble_yld(long long n_nodes, const double *coords, long long n_elems, const int *conn, int fbar, const double *u,
                     const double *hist_in, const double *mat, long long n_mat, const double *bar, const int *row_ptr,
                     const int *col_idx, double *residual, double *csr_vals, double *hist_out, long long *stats);
int orc_assemble(long long n_nodes, const double *coords, long long n_elems, const int *conn, int fbar, const double *u,
                 const double *hist_in, const double *mat, long long n_mat, const int *row_ptr, const int *col_idx,
                 double *residual, double *csr_vals, double *hist_out, long long *stats) {
    return orc_assemble_yld(n_nodes, coords, n_elems, conn, fbar, u, hist_in, mat, n_mat, g_dummy_bar, row_ptr, col_idx, residual,
                            csr_vals, hist_out, stats);
}
/* bar: NULL (Hill-48) or n_mat records of NBAR doubles (Yld2004-18p) */
int orc_assemble_yld(long long n_nodes, const double *coords, long long n_elems, const int *conn, int fbar, const double *u,
                     const double *hist_in, const double *mat, long long n_mat, const double *bar, const int *row_ptr,
                     const int *col_idx, double *residual, double *csr_vals, double *hist_out, long long *stats) {
    long long nnz = row_ptr[3 * n_nodes], CH = 8192;
    long double *acc = calloc(nnz, sizeof(long double)), *racc = calloc(3 * n_nodes, sizeof(long double));
    double *Kc = malloc(CH * 576 * sizeof(double)), *Rc = malloc(CH * 24 * sizeof(double));
    if (!acc || !racc || !Kc || !Rc) return -1;
    long long st[4] = {0, 0, 0, 0};
    for (long long e0 = 0; e0 < n_elems; e0 += CH) {
        long long e1 = e0 + CH < n_elems ? e0 + CH : n_elems;
        #pragma omp parallel
        {
            long long ls[4] = {0, 0, 0, 0};
            #pragma omp for schedule(dynamic, 16)
            for (long long e = e0; e < e1; e++) {
                double X[24], ue[24];
                for (int a = 0; a < 8; a++) for (int i = 0; i < 3; i++) {
                    X[a * 3 + i] = coords[3 * (long long)conn[e * 8 + a] + i];
                    ue[a * 3 + i] = u[3 * (long long)conn[e * 8 + a] + i];
                }
                int it = orc_element_yld(X, ue, hist_in + e * 56, mat + (n_mat == 1 ? 0 : e * NPAR),
                                         bar ? bar + (n_mat == 1 ? 0 : e * NBAR) : bar, fbar, Rc + (e - e0) * 24,
                                         Kc + (e - e0) * 576, hist_out + e * 56, ls);
                if (it > ls[3]) ls[3] = it;
            }
            #pragma omp critical
            { st[0] += ls[0]; st[1] += ls[1]; st[2] += ls[2]; if (ls[3] > st[3]) st[3] = ls[3]; }
        }
        for (long long e = e0; e < e1; e++)          /* serial, ascending element id */
            for (int a = 0; a < 24; a++) {
                int row = 3 * conn[e * 8 + a / 3] + a % 3;
                racc[row] += Rc[(e - e0) * 24 + a];
                const int *c = col_idx + row_ptr[row];
                int len = row_ptr[row + 1] - row_ptr[row];
                for (int b = 0; b < 24; b++) {
                    int col = 3 * conn[e * 8 + b / 3] + b % 3, lo = 0, hi = len - 1;
                    while (lo < hi) { int mid = (lo + hi) / 2; if (c[mid] < col) lo = mid + 1; else hi = mid; }
                    acc[row_ptr[row] + lo] += Kc[(e - e0) * 576 + a * 24 + b];
                }
            }
    }
    for (long long i = 0; i < nnz; i++) csr_vals[i] = (double)acc[i];
    for (long long i = 0; i < 3 * n_nodes; i++) residual[i] = (double)racc[i];
    if (stats) memcpy(stats, st, sizeof(st));
    free(acc); free(racc); free(Kc); free(Rc);
    return 0;
}
int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Lankford r0,r45,r90 -> paper yield ratios (r11,r22,r33,r12,r23,r13): textbook Hill-1948 plane-stress relations,
 * axis 1 = rolling direction, normalised so sigma11^y = sigma0 (reading D2). */
void orc_hill_from_lankford(double r0, double r45, double r90, double *r_out) {
    double G = 1 / (1 + r0), H = r0 / (1 + r0), F = H / r90, N = (r45 + 0.5) * (F + G), L = 1.5;
    r_out[0] = 1 / sqrt(G + H); r_out[1] = 1 / sqrt(F + H); r_out[2] = 1 / sqrt(F + G);
    r_out[3] = sqrt(3 / (2 * N)); r_out[4] = sqrt(3 / (2 * L)); r_out[5] = sqrt(3 / (2 * L));
}
