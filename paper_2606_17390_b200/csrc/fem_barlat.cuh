// Barlat Yld2004-18p in the constitutive step of k_element (Eq.(12), App. A.2
// :808-830, return map Eq.(19)-(24) :176-196 with the line search of App. B :836-869).  Included by fem_assemble.cu only.
//
// Formulation (nothing here is shared with oracle/):
//  * even integer exponent m (2..16): Phi = 4 phi^m = sum_ij (a_i - b_j)^m = sum_k binom(m,k)(-1)^k tr(A^(m-k)) tr(B^k) with
//    A = s' = C':P:T, B = s'' = C'':P:T.  Powers of the 3x3 tensors are reduced with Cayley-Hamilton,
//    A^n = alpha_n I + beta_n A + gamma_n A^2 (three-term scalar recurrence in the invariants), so Phi, its gradient and its
//    Hessian are polynomials in {I, A, A^2, B, B^2} with scalar coefficients: no eigenvectors, no repeated-eigenvalue cases,
//    no branches.
//  * return map: Newton on (T, dgam) (alpha = alpha_n + dgam eliminated: W = 1 and its equation is linear, so it holds
//    after every step of Alg. C2) with the merit function and Goldstein test of App. B.  With isotropic E and deviatoric N
//    the T-block of the Jacobian is the symmetric positive definite M = I + 2mu dgam d2phi/dT2 (Cholesky).
//  * C_ep = 2mu M^-1 + (K - 2mu/3) 1(x)1 - (2mu)^2 (M^-1 N)(x)(M^-1 N) / (2mu N.M^-1 N + sigma_flow')   (App. D in closed form)
// All 2-tensors are Mandel 6-vectors (11,22,33,sqrt2*12,sqrt2*23,sqrt2*13) in the material frame unless noted.
#pragma once

#define FEM_BARD 32   // derived Barlat record: [0..8] N' = C'n.Pn (row-major), [9..11] c'44,c'55,c'66, [12..23] the same for C'', [24] m
#define BAR_MMAX 16
#ifndef BAR_LOCKSTEP
#define BAR_LOCKSTEP 1
#endif
#ifndef BAR_TOLG
#define BAR_TOLG 1e-13
#endif
#ifndef BAR_START
#define BAR_START 1
#endif

// bad_m: counts records whose exponent is not an even integer in 2..BAR_MMAX; such an exponent is replaced by the nearest
// supported one so that the tables indexed by m (BAR_MMAX + 1 entries) are never overrun; fem_assemble_barlat reports
// FEM_ERR_ARG when the counter is non-zero and the caller asked for statistics.
__global__ void k_bar_prep(long long n_mat, const double *__restrict__ bar, double *__restrict__ bd, unsigned long long *bad_m) {
    long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (r >= n_mat) return;
    const double *p = bar + r * FEM_NBARLAT;
    double *o = bd + r * FEM_BARD;
    for (int t = 0; t < 2; t++) {
        const double *c = p + 9 * t;
        // Eq.(A9) :820-824 normal block times the deviatoric projector of Eq.(A8) :816
        const double Cn[3][3] = {{0.0, -c[0], -c[1]}, {-c[2], 0.0, -c[3]}, {-c[4], -c[5], 0.0}};
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                double s = 0.0;
                for (int k = 0; k < 3; k++) s += Cn[i][k] * ((k == j) ? 2.0 / 3.0 : -1.0 / 3.0);
                o[12 * t + 3 * i + j] = s;
            }
        o[12 * t + 9] = c[6]; o[12 * t + 10] = c[7]; o[12 * t + 11] = c[8];
    }
    {
        double m = p[18];
        const bool ok = (m >= 2.0) && (m <= (double)BAR_MMAX) && (m == 2.0 * floor(0.5 * m));
        if (!ok) {
            atomicAdd(bad_m, 1ull);
            m = 2.0 * rint(0.5 * (isfinite(m) ? m : 2.0));
            m = fmin(fmax(m, 2.0), (double)BAR_MMAX);
        }
        o[24] = m;
    }
    for (int i = 25; i < FEM_BARD; i++) o[i] = 0.0;
}

// pair tables of the component order (11,22,33,12,23,13)
__device__ constexpr int BI[6] = {0, 1, 2, 0, 1, 0};
__device__ constexpr int BJ[6] = {0, 1, 2, 1, 2, 2};
__device__ constexpr int BV[3][3] = {{0, 3, 5}, {3, 1, 4}, {5, 4, 2}};

// transformed tensor (tensor components) X = L T, L = (Nn, ds) from the derived record
__device__ __forceinline__ void bar_apply(const double *__restrict__ L, const double T[6], double x[6]) {
#pragma unroll
    for (int i = 0; i < 3; i++) x[i] = L[3 * i] * T[0] + L[3 * i + 1] * T[1] + L[3 * i + 2] * T[2];
#pragma unroll
    for (int i = 0; i < 3; i++) x[3 + i] = L[9 + i] * T[3 + i] * RSQRT2;
}
// y (Mandel) += L^T g, g given in tensor components
__device__ __forceinline__ void bar_apply_t(const double *__restrict__ L, const double g[6], double y[6]) {
#pragma unroll
    for (int j = 0; j < 3; j++) y[j] = fma(L[6 + j], g[2], fma(L[3 + j], g[1], fma(L[j], g[0], y[j])));
#pragma unroll
    for (int i = 0; i < 3; i++) y[3 + i] = fma(L[9 + i] * SQRT2, g[3 + i], y[3 + i]);
}
// c[n][p] of the Cayley-Hamilton table below is structurally zero for n < 3, p != n (X^n = unit vector n of {I, X, X^2})
__device__ __forceinline__ constexpr bool bar_cnz(int n, int p) { return n >= 3 || n == p; }
// X^2 of a symmetric 3x3 in tensor components, and the Cayley-Hamilton data: c[n] = (alpha,beta,gamma) of X^n, t[n] = tr X^n
template <int M>
__device__ __forceinline__ void bar_powers(const double a[6], int m, double a2[6], double (*c)[3], double *t) {
    a2[0] = a[0] * a[0] + a[3] * a[3] + a[5] * a[5];
    a2[1] = a[3] * a[3] + a[1] * a[1] + a[4] * a[4];
    a2[2] = a[5] * a[5] + a[4] * a[4] + a[2] * a[2];
    a2[3] = a[0] * a[3] + a[3] * a[1] + a[5] * a[4];
    a2[4] = a[3] * a[5] + a[1] * a[4] + a[4] * a[2];
    a2[5] = a[0] * a[5] + a[3] * a[4] + a[5] * a[2];
    const double I1 = a[0] + a[1] + a[2], tr2 = a2[0] + a2[1] + a2[2], I2 = 0.5 * (I1 * I1 - tr2);
    const double I3 = a[0] * (a[1] * a[2] - a[4] * a[4]) - a[3] * (a[3] * a[2] - a[4] * a[5]) + a[5] * (a[3] * a[4] - a[1] * a[5]);
    c[0][0] = 1.0; c[0][1] = 0.0; c[0][2] = 0.0;
    c[1][0] = 0.0; c[1][1] = 1.0; c[1][2] = 0.0;
    c[2][0] = 0.0; c[2][1] = 0.0; c[2][2] = 1.0;
#pragma unroll
    for (int n = 2; n < (M ? M : m); n++) {   // X^(n+1) = X X^n with X^3 = I1 X^2 - I2 X + I3 I
        const double al = c[n][0], be = c[n][1], ga = c[n][2];
        c[n + 1][0] = ga * I3; c[n + 1][1] = fma(-ga, I2, al); c[n + 1][2] = fma(ga, I1, be);
    }
#pragma unroll
    for (int n = 0; n <= (M ? M : m); n++) t[n] = 3.0 * c[n][0] + c[n][1] * I1 + c[n][2] * tr2;
}
// H (6x6 Mandel, full) += fully symmetrised "box" product 1/4 (X_ik Y_jl + X_il Y_jk + Y_ik X_jl + Y_il X_jk)
__device__ __forceinline__ void bar_box_acc(const double X[6], const double Y[6], double H[6][6]) {
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) {
            const int i = BI[A], j = BJ[A], k = BI[B], l = BJ[B];
            const double v = X[BV[i][k]] * Y[BV[j][l]] + X[BV[i][l]] * Y[BV[j][k]] + Y[BV[i][k]] * X[BV[j][l]] + Y[BV[i][l]] * X[BV[j][k]];
            const double w = ((A < 3) ? 1.0 : SQRT2) * ((B < 3) ? 1.0 : SQRT2) * 0.25;
            H[A][B] = fma(w, v, H[A][B]);
        }
}
// the same with X = I: 1/4 (d_ik Y_jl + d_il Y_jk + Y_ik d_jl + Y_il d_jk), the Kronecker deltas resolved at compile time
__device__ __forceinline__ void bar_box_id_acc(const double Y[6], double H[6][6]) {
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) {
            const int i = BI[A], j = BJ[A], k = BI[B], l = BJ[B];
            double v = 0.0;
            bool any = false;
            if (i == k) { v = Y[BV[j][l]]; any = true; }
            if (i == l) { v = any ? v + Y[BV[j][k]] : Y[BV[j][k]]; any = true; }
            if (j == l) { v = any ? v + Y[BV[i][k]] : Y[BV[i][k]]; any = true; }
            if (j == k) { v = any ? v + Y[BV[i][l]] : Y[BV[i][l]]; any = true; }
            const double w = ((A < 3) ? 1.0 : SQRT2) * ((B < 3) ? 1.0 : SQRT2) * 0.25;
            if (any) H[A][B] = fma(w, v, H[A][B]);
        }
}
// Out (upper triangle) += L^T H L for the block map L = (Nn 3x3, ds 3); H upper triangle (Mandel)
__device__ __forceinline__ void bar_congr_acc(const double *__restrict__ L, const double H[6][6], double Out[6][6]) {
    double T1[6][6];   // H L
#pragma unroll
    for (int a = 0; a < 6; a++) {
#pragma unroll
        for (int b = 0; b < 3; b++) {
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < 3; c++) s = fma((a <= c) ? H[a][c] : H[c][a], L[3 * c + b], s);
            T1[a][b] = s;
        }
#pragma unroll
        for (int b = 3; b < 6; b++) T1[a][b] = ((a <= b) ? H[a][b] : H[b][a]) * L[9 + b - 3];
    }
#pragma unroll
    for (int a = 0; a < 6; a++)
#pragma unroll
        for (int b = a; b < 6; b++) {
            if (a < 3) {
                double s = Out[a][b];
#pragma unroll
                for (int c = 0; c < 3; c++) s = fma(L[3 * c + a], T1[c][b], s);
                Out[a][b] = s;
            } else Out[a][b] = fma(L[9 + a - 3], T1[a][b], Out[a][b]);
        }
}

// phi (Eq.(12) :133), N = dphi/dT and (want_H) H = d2phi/dT2 (upper triangle) at the Mandel stress T, material frame.
// M > 0: exponent known at compile time (every loop unrolls, the Cayley-Hamilton tables live in registers and the
// binomial weights are immediates); M = 0: any even exponent up to BAR_MMAX with rolled loops and tables in local memory.
template <int M>
__device__ __forceinline__ void bar_eval_t(const double *__restrict__ bd, int m_rt, const double T[6], bool want_H, double &phi_out,
                                           double N[6], double H[6][6]) {
    const int m = M ? M : m_rt;
    const double *LA = bd, *LB = bd + 12;
    double a[6], b[6], a2[6], b2[6];
    double cA[BAR_MMAX + 1][3], cB[BAR_MMAX + 1][3], tA[BAR_MMAX + 1], tB[BAR_MMAX + 1];
    bar_apply(LA, T, a); bar_apply(LB, T, b);
    bar_powers<M>(a, m, a2, cA, tA); bar_powers<M>(b, m, b2, cB, tB);
    double Phi = 0.0, gA[3] = {0, 0, 0}, gB[3] = {0, 0, 0};
    {
        double sb = 1.0;   // (-1)^k binom(m,k)
#pragma unroll
        for (int k = 0; k <= m; k++) {
            Phi = fma(sb * tA[m - k], tB[k], Phi);
            if (k < m) { const double w = sb * (m - k) * tB[k];
#pragma unroll
                for (int p = 0; p < 3; p++) if (bar_cnz(m - k - 1, p)) gA[p] = fma(w, cA[m - k - 1][p], gA[p]); }
            if (k > 0) { const double w = sb * k * tA[m - k];
#pragma unroll
                for (int p = 0; p < 3; p++) if (bar_cnz(k - 1, p)) gB[p] = fma(w, cB[k - 1][p], gB[p]); }
            sb = -sb * (double)(m - k) / (double)(k + 1);
        }
    }
    // phi = (Phi/4)^(1/m): three nested square roots for m = 8 (the paper's exponent), exp(ln/m) otherwise
    double phi;
    if (M == 8) { double r = 0.25 * Phi; r = r * frsqrt(r); r = r * frsqrt(r); phi = r * frsqrt(r); }
    else phi = fexp(flog(0.25 * Phi) / m);
    phi_out = phi;
    const double cf = phi * frcp(m * Phi);   // dphi = phi^(1-m)/(4m) dPhi, 4 phi^m = Phi
    double GA[6], GB[6];
#pragma unroll
    for (int i = 0; i < 6; i++) {
        GA[i] = fma(gA[2], a2[i], fma(gA[1], a[i], (i < 3) ? gA[0] : 0.0));
        GB[i] = fma(gB[2], b2[i], fma(gB[1], b[i], (i < 3) ? gB[0] : 0.0));
    }
#pragma unroll
    for (int i = 0; i < 6; i++) N[i] = 0.0;
    bar_apply_t(LA, GA, N); bar_apply_t(LB, GB, N);
#pragma unroll
    for (int i = 0; i < 6; i++) N[i] *= cf;
    if (!want_H) return;
    // scalar coefficient matrices: HAA = sum_pq WA_pq box(A^p,A^q), HBB likewise, HAB = sum_pq V_pq A^p (x) B^q
    double WA[3][3], WB[3][3], V[3][3];
#pragma unroll
    for (int p = 0; p < 3; p++)
#pragma unroll
        for (int q = 0; q < 3; q++) { WA[p][q] = 0.0; WB[p][q] = 0.0; V[p][q] = 0.0; }
    {
        // d/dA of A^n is sum_{r=0}^{n-1} A^r (.) A^(n-1-r): with A^r = c[r][0] I + c[r][1] A + c[r][2] A^2 the coefficient
        // matrix of order j = n-1 is the convolution S_j[p][q] = sum_{r=0}^{j} c[r][p] c[j-r][q] (symmetric in p,q), formed
        // once per j for either side and weighted by the binomial term it belongs to
        double sbk[BAR_MMAX + 1];   // (-1)^k binom(m,k)
        {
            double sb = 1.0;
#pragma unroll
            for (int k = 0; k <= m; k++) { sbk[k] = sb; sb = -sb * (double)(m - k) / (double)(k + 1); }
        }
#pragma unroll
        for (int j = 0; j <= m - 2; j++) {
            double SA[3][3], SB[3][3];
#pragma unroll
            for (int p = 0; p < 3; p++)
#pragma unroll
                for (int q = p; q < 3; q++) { SA[p][q] = 0.0; SB[p][q] = 0.0; }
#pragma unroll
            for (int r = 0; r <= j; r++)
#pragma unroll
                for (int p = 0; p < 3; p++)
#pragma unroll
                    for (int q = p; q < 3; q++) {
                        if (!bar_cnz(r, p) || !bar_cnz(j - r, q)) continue;   // c[n] = unit vector n for n < 3
                        SA[p][q] = fma(cA[r][p], cA[j - r][q], SA[p][q]);
                        SB[p][q] = fma(cB[r][p], cB[j - r][q], SB[p][q]);
                    }
            const int kA = m - 2 - j, kB = j + 2;
            const double wA = sbk[kA] * (m - kA) * tB[kA];   // term k = kA of Phi: (m-k) tB[k] d(A^(m-k-1))
            const double wB = sbk[kB] * kB * tA[m - kB];     // term k = kB:        k tA[m-k] d(B^(k-1))
#pragma unroll
            for (int p = 0; p < 3; p++)
#pragma unroll
                for (int q = p; q < 3; q++) { WA[p][q] = fma(wA, SA[p][q], WA[p][q]); WB[p][q] = fma(wB, SB[p][q], WB[p][q]); }
        }
#pragma unroll
        for (int k = 1; k <= m - 1; k++) {
            const double w = sbk[k] * (m - k) * k;
#pragma unroll
            for (int p = 0; p < 3; p++)
#pragma unroll
                for (int q = 0; q < 3; q++) {
                    if (!bar_cnz(m - k - 1, p) || !bar_cnz(k - 1, q)) continue;
                    V[p][q] = fma(w * cA[m - k - 1][p], cB[k - 1][q], V[p][q]);
                }
        }
    }
    WA[1][0] = WA[0][1]; WA[2][0] = WA[0][2]; WA[2][1] = WA[1][2];   // sum_r c[r][p] c[j-r][q] is symmetric in (p,q)
    WB[1][0] = WB[0][1]; WB[2][0] = WB[0][2]; WB[2][1] = WB[1][2];
    const double id6[6] = {1.0, 1.0, 1.0, 0.0, 0.0, 0.0};
    double d2[6][6];
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = 0; B < 6; B++) d2[A][B] = 0.0;
    {
        double HX[6][6], Y[6];
#pragma unroll
        for (int side = 0; side < 2; side++) {
            const double (*W)[3] = side ? WB : WA;
            const double *x = side ? b : a, *x2 = side ? b2 : a2;
#pragma unroll
            for (int A = 0; A < 6; A++)
#pragma unroll
                for (int B = 0; B < 6; B++) HX[A][B] = 0.0;
#pragma unroll
            for (int i = 0; i < 6; i++) Y[i] = fma(W[0][2], x2[i], (i < 3) ? fma(W[0][1], x[i], W[0][0]) : W[0][1] * x[i]);
            bar_box_id_acc(Y, HX);
#pragma unroll
            for (int i = 0; i < 6; i++) Y[i] = fma(W[1][2], x2[i], (i < 3) ? fma(W[1][1], x[i], W[1][0]) : W[1][1] * x[i]);
            bar_box_acc(x, Y, HX);
#pragma unroll
            for (int i = 0; i < 6; i++) Y[i] = fma(W[2][2], x2[i], (i < 3) ? fma(W[2][1], x[i], W[2][0]) : W[2][1] * x[i]);
            bar_box_acc(x2, Y, HX);
            bar_congr_acc(side ? LB : LA, HX, d2);
        }
    }
    // mixed term: sum_q (L'^T u_q) (x) (L''^T B^q), u_q = sum_p V_pq A^p, and its transpose
#pragma unroll
    for (int q = 0; q < 3; q++) {
        double uq[6], bq[6], lu[6] = {0, 0, 0, 0, 0, 0}, lb[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < 6; i++) {
            uq[i] = fma(V[2][q], a2[i], (i < 3) ? fma(V[1][q], a[i], V[0][q]) : V[1][q] * a[i]);
            bq[i] = (q == 0) ? id6[i] : ((q == 1) ? b[i] : b2[i]);
        }
        bar_apply_t(LA, uq, lu); bar_apply_t(LB, bq, lb);
#pragma unroll
        for (int A = 0; A < 6; A++)
#pragma unroll
            for (int B = A; B < 6; B++) d2[A][B] = fma(lu[A], lb[B], fma(lb[A], lu[B], d2[A][B]));
    }
    const double cn = (m - 1.0) * frcp(phi);
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) H[A][B] = fma(cf, d2[A][B], -cn * N[A] * N[B]);
}

// The return map below has ONE evaluation site.  The paper's exponent (m = 8, Table 2) is inlined there, so that the
// stress, the gradient and the Hessian stay in registers across the iteration; every other exponent goes through an
// out-of-line copy whose arguments travel in a small block of local memory for the duration of the call only.
struct bar_io { double T[6], N[6], H[6][6], phi; };
__device__ __noinline__ void bar_eval_other(const double *__restrict__ bd, int m, bool want_H, bar_io &io) {
    if (m == 6) bar_eval_t<6>(bd, m, io.T, want_H, io.phi, io.N, io.H);   // steels
    else bar_eval_t<0>(bd, m, io.T, want_H, io.phi, io.N, io.H);
}
__device__ __forceinline__ void bar_eval(const double *__restrict__ bd, int m, const double T[6], bool want_H, double &phi_out,
                                         double N[6], double H[6][6]) {
    if (m == 8) bar_eval_t<8>(bd, m, T, want_H, phi_out, N, H);        // aluminium alloys, the paper's Table 2
    else {
        bar_io io;
#pragma unroll
        for (int i = 0; i < 6; i++) io.T[i] = T[i];
        bar_eval_other(bd, m, want_H, io);
        phi_out = io.phi;
#pragma unroll
        for (int i = 0; i < 6; i++) N[i] = io.N[i];
        if (want_H) {
#pragma unroll
            for (int A = 0; A < 6; A++)
#pragma unroll
                for (int B = A; B < 6; B++) H[A][B] = io.H[A][B];
        }
    }
}

// In-place Cholesky M = L L^T of a symmetric positive definite 6x6 (lower triangle of M on entry; on exit the strict lower
// triangle of L and, on the diagonal, the RECIPROCALS 1/L_jj, so that the solves multiply instead of dividing).
__device__ __forceinline__ void chol6(double M[6][6]) {
#pragma unroll
    for (int j = 0; j < 6; j++) {
        double d = M[j][j];
#pragma unroll
        for (int k = 0; k < j; k++) d = fma(-M[j][k], M[j][k], d);
        const double id = frsqrt(d);
        M[j][j] = id;
#pragma unroll
        for (int i = j + 1; i < 6; i++) {
            double s = M[i][j];
#pragma unroll
            for (int k = 0; k < j; k++) s = fma(-M[i][k], M[j][k], s);
            M[i][j] = s * id;
        }
    }
}
__device__ __forceinline__ void chol6_solve(const double L[6][6], const double rhs[6], double x[6]) {
    double y[6];
#pragma unroll
    for (int i = 0; i < 6; i++) {
        double s = rhs[i];
#pragma unroll
        for (int k = 0; k < i; k++) s = fma(-L[i][k], y[k], s);
        y[i] = s * L[i][i];
    }
#pragma unroll
    for (int i = 5; i >= 0; i--) {
        double s = y[i];
#pragma unroll
        for (int k = i + 1; k < 6; k++) s = fma(-L[k][i], x[k], s);
        x[i] = s * L[i][i];
    }
}

// Alg. C1 steps 2-8 / Alg. C2 for Yld2004-18p at one Gauss point, material frame.
//   ee   elastic trial strain eps - eps_p_n (tensor components)      out: T (Mandel stress), dep = dgam N (tensor components),
//   Cep  (6x6 Mandel, upper triangle), dg, iteration count, flags
#ifndef BAR_RM_INLINE
#define BAR_RM_INLINE 1
#endif
#if BAR_RM_INLINE
__device__ __forceinline__
#else
__device__ __noinline__
#endif
void bar_return_map(const double *__restrict__ bd, double mu2, double kb, double law, double hh0,
                                            double hh1, double hh2, const double ee[6], double alphan, int kmax, double T[6],
                                            double dep[6], double Cep[6][6], double &dg_out, int &iters, bool &plastic,
                                            bool &nonconv) {
    const int m_exp = (int)__ldg(bd + 24);
    const double tre = ee[0] + ee[1] + ee[2], pres = kb * tre, tm = tre * (1.0 / 3.0);
    double Ttr[6];   // Eq.(16) :160
#pragma unroll
    for (int i = 0; i < 3; i++) { Ttr[i] = fma(mu2, ee[i] - tm, pres); Ttr[3 + i] = SQRT2 * mu2 * ee[3 + i]; }
    double s0, ds0;
    flow_stress(law, hh0, hh1, hh2, alphan, s0, ds0);   // W = 1: sigma_y = sigma_flow (:145)
    double phi = 0.0, N[6], H[6][6];
    double tn2 = 0.0;
#pragma unroll
    for (int i = 0; i < 6; i++) { T[i] = Ttr[i]; dep[i] = 0.0; N[i] = 0.0; tn2 = fma(Ttr[i] - ((i < 3) ? pres : 0.0), Ttr[i] - ((i < 3) ? pres : 0.0), tn2); }
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = 0; B < 6; B++) H[A][B] = 0.0;
    iters = 0; nonconv = false; dg_out = 0.0;
    plastic = false;
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) Cep[A][B] = ((A < 3 && B < 3) ? kb - mu2 * (1.0 / 3.0) : 0.0) + ((A == B) ? mu2 : 0.0);
    const double is0 = frcp(s0);
    // the stop test below works on squared norms (no square root in the loop): tolG2 = tolG^2, tolG = BAR_TOLG max(1, |s^tr| / sigma_0)
    const double tolG2 = (BAR_TOLG * BAR_TOLG) * fmax(1.0, tn2 * is0 * is0);
    double dg = 0.0, sy = s0, dsy = ds0, prev = INFINITY;
    double GT[6], fv = 0.0, psi0 = 0.0;
    // merit of Eq.(B2) :846 with the rows of G scaled by sigma_y(alpha_n) (T rows and f row are stresses)
#define BAR_RESID(Tc, dgc, Nc, phic, syc, GTo, fo, psio)                                              \
    do {                                                                                               \
        psio = 0.0;                                                                                    \
        _Pragma("unroll") for (int i_ = 0; i_ < 6; i_++) {                                             \
            GTo[i_] = (Tc[i_] - Ttr[i_] + mu2 * dgc * Nc[i_]) * is0;                                   \
            psio = fma(GTo[i_], GTo[i_], psio);                                                        \
        }                                                                                              \
        fo = (phic - syc) * is0;                                                                       \
        psio = 0.5 * fma(fo, fo, psio);                                                                \
    } while (0)
    // ONE loop with ONE evaluation site of the (large, unrolled) yield function: every pass evaluates phi, N and H at the
    // point Te and then does what its mode says -- 0: the trial state (yield test Eq.(17)-(18) :165-172, starting point);
    // 1: a line-search point of the current Newton step (App. B Eq.(B1)-(B7) :838-867, beta = 1e-4, eta = 0.1, :871; the
    // full step j = 0 is accepted almost always, so the Hessian is taken along with every point instead of being
    // evaluated again at an accepted shortened step: H is then a pure output of the evaluation and nothing of it has to
    // survive one).  A pass that leaves (T, dgam) updated ends in the Newton head: convergence test, then the direction of
    // Eq.(24) :196.  The warps of the CTA walk the evaluation code together: every pass starts at a CTA-wide barrier and
    // the loop runs until no thread of the CTA is active (elastic points and converged points idle); ncu showed
    // instruction fetch as the top stall with every warp at its own place in ~60 KB of SASS.
    double Te[6], dT[6], ddg = 0.0, dgt = 0.0, zeta = 1.0, zj = 1.0;
#pragma unroll
    for (int i = 0; i < 6; i++) { Te[i] = Ttr[i]; dT[i] = 0.0; GT[i] = 0.0; }
    int mode = 0, j = 0, k = 0;
    bool conv = false, active = tn2 > 0.0;
    for (;;) {
#if BAR_LOCKSTEP
        if (!__syncthreads_or(active)) break;
#else
        if (!__any_sync(0xffffffffu, active)) break;
#endif
        if (!active) continue;
        double phie, Ne[6];
        bar_eval(bd, m_exp, Te, true, phie, Ne, H);
        if (mode == 0) {
            plastic = (phie - s0) > 0.0;                     // Eq.(17)-(18) :165-172, tie -> elastic
            if (!plastic) { active = false; continue; }
            phi = phie;
#pragma unroll
            for (int i = 0; i < 6; i++) N[i] = Ne[i];
#if BAR_START
            // Starting point (the root is unique, so any start reaches the state Alg. C2 reaches from T^tr): the trial deviator
            // scaled back onto the yield surface, T0 = p 1 + c s^tr, with dgam from the N-component of Eq.(19): phi^tr - 2mu dgam
            // N.N - sigma_y(alpha_n + dgam) = 0 (exact radial return for von Mises).  phi is homogeneous of degree one, so phi, N
            // and H at T0 follow from the trial evaluation without another one: phi0 = c phi^tr, N0 = N, H0 = H / c.
            {
                double nn = 0.0;
#pragma unroll
                for (int i = 0; i < 6; i++) nn = fma(N[i], N[i], nn);
                const double a = mu2 * nn;
                for (int it = 0; it < 6; it++) {   // convex, decreasing: Newton from dgam = 0 approaches the root from the left
                    const double g = phi - a * dg - sy, d = g * frcp(a + dsy);
                    dg += d;
                    flow_stress(law, hh0, hh1, hh2, alphan + dg, sy, dsy);
                    if (d <= 1e-3 * dg) break;
                }
                const double c = sy * frcp(phi), ic = phi * frcp(sy);
#pragma unroll
                for (int i = 0; i < 6; i++) T[i] = (i < 3) ? fma(c, Ttr[i] - pres, pres) : c * Ttr[i];
                phi = sy;
#pragma unroll
                for (int A = 0; A < 6; A++)
#pragma unroll
                    for (int B = A; B < 6; B++) H[A][B] *= ic;
            }
#endif
            BAR_RESID(T, dg, N, phi, sy, GT, fv, psi0);
        } else {
            double syt, dsyt, GTt[6], ft, psit;
            flow_stress(law, hh0, hh1, hh2, alphan + dgt, syt, dsyt);
            BAR_RESID(Te, dgt, Ne, phie, syt, GTt, ft, psit);
            if (!(psit < (1.0 - 2.0e-4 * zeta) * psi0 || j >= 12)) {             // Eq.(B3) fails: shorten the step
                const double zn = psi0 * frcp(psi0 + psit);                         // Eq.(B5)/(B6)
                zeta = (j == 0) ? zn : fmax(0.1 * zj, zn);                          // Eq.(B7)
                zj = zeta;
                j++;
                dgt = fma(zeta, ddg, dg);
#pragma unroll
                for (int i = 0; i < 6; i++) Te[i] = fma(zeta, dT[i], T[i]);
                continue;
            }
            dg = dgt; sy = syt; dsy = dsyt; phi = phie; fv = ft; psi0 = psit;
#pragma unroll
            for (int i = 0; i < 6; i++) { T[i] = Te[i]; N[i] = Ne[i]; GT[i] = GTt[i]; }
        }
        // ---- Newton head: (T, dgam, phi, N, H, sigma_y, G, psi) describe the current iterate k
        {
            const double nrm2 = 2.0 * psi0;   // |G|^2; `prev` holds the previous iterate's
            iters = k;
            if (nrm2 <= tolG2 || (prev <= 1e-18 && nrm2 >= 0.25 * prev)) { conv = true; active = false; continue; }
            if (k >= kmax) { active = false; continue; }
            prev = nrm2;
        }
        // Newton direction of Eq.(24) :196 on (T, dgam): M dT + 2mu N ddg = -G_T s0 ; N.dT - sigma' ddg = -f s0
        {
            double M[6][6], x1[6], x2[6], r1[6];
#pragma unroll
            for (int A = 0; A < 6; A++)
#pragma unroll
                for (int B = 0; B <= A; B++) M[A][B] = fma(mu2 * dg, H[B][A], (A == B) ? 1.0 : 0.0);
            chol6(M);
#pragma unroll
            for (int i = 0; i < 6; i++) r1[i] = GT[i] * s0;
            chol6_solve(M, r1, x1); chol6_solve(M, N, x2);
            double nx1 = 0.0, nx2 = 0.0;
#pragma unroll
            for (int i = 0; i < 6; i++) { nx1 = fma(N[i], x1[i], nx1); nx2 = fma(N[i], x2[i], nx2); }
            ddg = (fv * s0 - nx1) * frcp(fma(mu2, nx2, dsy));
#pragma unroll
            for (int i = 0; i < 6; i++) dT[i] = -fma(mu2 * ddg, x2[i], x1[i]);
        }
        zeta = 1.0; zj = 1.0; j = 0; k++;
        dgt = dg + ddg;
#pragma unroll
        for (int i = 0; i < 6; i++) Te[i] = T[i] + dT[i];
        mode = 1;
    }
#undef BAR_RESID
    if (!plastic) return;
    nonconv = !conv;
    dg_out = dg;
    // Alg. C2 step 27 :979: eps_p += dgam N, T = E:(eps - eps_p)
#pragma unroll
    for (int i = 0; i < 6; i++) {
        T[i] = fma(-mu2 * dg, N[i], Ttr[i]);
        dep[i] = dg * N[i] * ((i < 3) ? 1.0 : RSQRT2);
    }
    // C_ep (App. D :1002-1019 in closed form)
    double M[6][6], Li[6][6], x2[6];
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = 0; B <= A; B++) M[A][B] = fma(mu2 * dg, H[B][A], (A == B) ? 1.0 : 0.0);
    chol6(M);
    chol6_solve(M, N, x2);
    // Li = L^-1 (lower triangular), M^-1 = Li^T Li
#pragma unroll
    for (int j = 0; j < 6; j++) {
#pragma unroll
        for (int i = 0; i < 6; i++) {
            if (i < j) { Li[i][j] = 0.0; continue; }
            double s = (i == j) ? 1.0 : 0.0;
#pragma unroll
            for (int k = j; k < i; k++) s = fma(-M[i][k], Li[k][j], s);
            Li[i][j] = s * M[i][i];
        }
    }
    double nx2 = 0.0;
#pragma unroll
    for (int i = 0; i < 6; i++) nx2 = fma(N[i], x2[i], nx2);
    const double cden = mu2 * mu2 * frcp(fma(mu2, nx2, dsy));
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) {
            double s = 0.0;
#pragma unroll
            for (int k = B; k < 6; k++) s = fma(Li[k][A], Li[k][B], s);
            Cep[A][B] = fma(mu2, s, ((A < 3 && B < 3) ? kb - mu2 * (1.0 / 3.0) : 0.0)) - cden * x2[A] * x2[B];
        }
}
