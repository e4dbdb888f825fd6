// the steps on either side of fem_assemble in one global Newton iteration K dd = -R
// (Eq.(39)): Dirichlet rows (Alg. E1 steps 6-11 :1048-1053), y = K x on the library's
// own block-structured CSR, Jacobi-preconditioned BiCGSTAB (the paper's default Krylov method, :304) and the Newton loop
// of one load increment.  Every reduction has a fixed order (per-CTA partial sums, one final CTA): results are
// bit-identical run to run.  Nothing here is shared with oracle/.
#include "fem_internal.h"
#include <math.h>
#include <string.h>

#define RED_CTAS 1184      // grid-stride vector kernels: a FIXED number of CTAs on every device (the per-CTA partial sums
                           // are part of the reduction order, so results do not depend on the SM count)
#define RED_THREADS 256
#define SPMV_CTAS 4736     // likewise fixed: grid-stride over the nodes, 8 warps per CTA, so the dot partials stay few

static inline unsigned spmv_grid(const fem_ctx *c) {
    const long long need = (c->n_nodes + 7) / 8;
    return (unsigned)(need < SPMV_CTAS ? need : SPMV_CTAS);
}
static inline unsigned nblk3(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// ------------------------------------------------------------------------------------------------ small kernels
__global__ void k_diagpos(long long n_nodes, const int *__restrict__ nb_ptr, const int *__restrict__ nb, int *diagpos) {
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    const int o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    int lo = 0, hi = len - 1;
    while (lo < hi) { int mid = (lo + hi) >> 1; if (nb[o + mid] < (int)n) lo = mid + 1; else hi = mid; }
    diagpos[n] = (len > 0 && nb[o + lo] == (int)n) ? lo : -1;   // -1: node without elements (empty rows)
}

// Alg. E1 step 10: "Enforce identity rows with one CUDA thread per row".  rhs[d] = bc_rhs[i], or
// bc_vals[i] - u[d] inside the Newton loop (the update then lands on the prescribed value).
__global__ void k_dirichlet(long long n_bc, const int *__restrict__ bc_dofs, const double *__restrict__ bc_rhs,
                            const double *__restrict__ bc_vals, const double *__restrict__ u, const int *__restrict__ nb_ptr,
                            const int *__restrict__ diagpos, double *__restrict__ vals, double *__restrict__ rhs) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= n_bc) return;
    const int d = bc_dofs[t], n = d / 3, i = d - 3 * n;
    const int o = nb_ptr[n], len = nb_ptr[n + 1] - o, dp = diagpos[n];
    double *row = vals + 9LL * o + (long long)i * 3 * len;
    for (int j = 0; j < 3 * len; j++) row[j] = 0.0;
    if (dp >= 0) row[3 * dp + i] = 1.0;
    if (rhs) rhs[d] = bc_vals ? bc_vals[t] - u[d] : (bc_rhs ? bc_rhs[t] : 0.0);
}

__global__ void k_scatter_bc(long long n_bc, const int *__restrict__ bc_dofs, const double *__restrict__ rhs, double *__restrict__ x) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < n_bc) x[bc_dofs[t]] = rhs[bc_dofs[t]];
}
__global__ void k_check_dofs(long long n_bc, const int *__restrict__ bc_dofs, long long n_rows, int *flag) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < n_bc && (bc_dofs[t] < 0 || bc_dofs[t] >= n_rows)) atomicOr(flag, 1);
}

// inverse diagonal of K (Jacobi preconditioner); a zero or missing diagonal entry counts as 1
__global__ void k_dinv(long long n_nodes, const int *__restrict__ nb_ptr, const int *__restrict__ diagpos,
                       const double *__restrict__ vals, double *__restrict__ dinv) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= 3 * n_nodes) return;
    const long long n = t / 3;
    const int i = (int)(t - 3 * n), o = nb_ptr[n], len = nb_ptr[n + 1] - o, dp = diagpos[n];
    double dgl = (dp >= 0) ? vals[9LL * o + (long long)i * 3 * len + 3 * dp + i] : 1.0;
    dinv[t] = (dgl != 0.0 && isfinite(dgl)) ? 1.0 / dgl : 1.0;
}

// ------------------------------------------------------------------------------------------------ reductions
// CTA-wide sum of NV values per thread in a fixed order (warp xor-tree, then warps in ascending order); thread 0 returns it.
template <int NV>
__device__ __forceinline__ void cta_reduce(double (&v)[NV], double *smem /*[NV*32]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; k++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) smem[k * 32 + w] = v[k];
    __syncthreads();
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) {
            double s = 0.0;
            for (int j = 0; j < nw; j++) s += smem[k * 32 + j];
            v[k] = s;
        }
}
// final stage: one CTA sums `count` partial records of NV values each (record-major) into out[0..NV)
template <int NV>
__global__ void __launch_bounds__(1024) k_reduce_final(const double *__restrict__ part, long long count, double *out) {
    __shared__ double smem[NV * 32];
    double v[NV];
#pragma unroll
    for (int k = 0; k < NV; k++) v[k] = 0.0;
    for (long long j = threadIdx.x; j < count; j += blockDim.x)
#pragma unroll
        for (int k = 0; k < NV; k++) v[k] += part[j * NV + k];
    cta_reduce<NV>(v, smem);
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) out[k] = v[k];
}

// ------------------------------------------------------------------------------------------------ SpMV
// y = K x on the block structure of the pattern: one warp per node n, lane = neighbour position; row 3n+i holds the
// entries [pos][k] contiguously, so a lane reads 3 x 24 bytes of values, one block-column index (nb, 4 bytes per 3x3
// block instead of col_idx's 36) and 3 entries of x.  DOT = 1: partial sums of (w, y); DOT = 2: of (y, w) and (y, y).
template <int DOT, typename VT = double>   // VT = float: the fp32 copy of K used inside mixed-precision CG (vectors stay fp64)
__global__ void __launch_bounds__(256)
k_spmv(long long n_nodes, const int *__restrict__ nb_ptr, const int *__restrict__ nb, const VT *__restrict__ vals,
       const double *__restrict__ x, double *__restrict__ y, const double *__restrict__ w, double *__restrict__ part) {
    __shared__ double smem[2 * 32];
    const int lane = threadIdx.x & 31;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    double d[2] = {0.0, 0.0};   // lane 0: this warp's share of the dot products (fixed node order => fixed summation order)
    for (long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; n < n_nodes; n += warps) {
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        const int o = nb_ptr[n], len = nb_ptr[n + 1] - o;
        double w0 = 0.0, w1 = 0.0, w2 = 0.0;
        if (DOT) { w0 = w[3 * n]; w1 = w[3 * n + 1]; w2 = w[3 * n + 2]; }   // issued with the row loads, not after the reduction
        const VT *base = vals + 9LL * o;
        for (int pos = lane; pos < len; pos += 32) {
            const long long m = nb[o + pos];
            const double x0 = x[3 * m], x1 = x[3 * m + 1], x2 = x[3 * m + 2];
            const VT *r0 = base + 3 * pos, *r1 = r0 + 3 * len, *r2 = r1 + 3 * len;
            a0 = fma((double)r0[2], x2, fma((double)r0[1], x1, fma((double)r0[0], x0, a0)));
            a1 = fma((double)r1[2], x2, fma((double)r1[1], x1, fma((double)r1[0], x0, a1)));
            a2 = fma((double)r2[2], x2, fma((double)r2[1], x1, fma((double)r2[0], x0, a2)));
        }
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) {
            a0 += __shfl_xor_sync(0xffffffffu, a0, o2); a1 += __shfl_xor_sync(0xffffffffu, a1, o2); a2 += __shfl_xor_sync(0xffffffffu, a2, o2);
        }
        if (lane == 0) {
            y[3 * n] = a0; y[3 * n + 1] = a1; y[3 * n + 2] = a2;
            if (DOT) {
                d[0] += a0 * w0 + a1 * w1 + a2 * w2;
                d[1] += a0 * a0 + a1 * a1 + a2 * a2;
            }
        }
    }
    if (DOT) {   // lane 0 of each warp holds its share; warps summed in ascending order
        const int wi = threadIdx.x >> 5;
        if (lane == 0) { smem[wi] = d[0]; smem[32 + wi] = d[1]; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double s0 = 0.0, s1 = 0.0;
            for (int j = 0; j < (int)(blockDim.x >> 5); j++) { s0 += smem[j]; s1 += smem[32 + j]; }
            part[2LL * blockIdx.x] = s0; part[2LL * blockIdx.x + 1] = s1;
        }
    }
}

// ------------------------------------------------------------------------------------------------ BiCGSTAB vector kernels
// r = b - r (r holds K x on entry), rhat = r, p = v = 0 ; partials: (r, r), (b, b)
__global__ void __launch_bounds__(RED_THREADS)
k_bicg_init(long long n, const double *__restrict__ b, double *__restrict__ r, double *__restrict__ rhat, double *__restrict__ p,
            double *__restrict__ v, double *__restrict__ part) {
    __shared__ double smem[2 * 32];
    double s[2] = {0.0, 0.0};
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        const double bj = b[j], rj = bj - r[j];
        r[j] = rj; rhat[j] = rj; p[j] = 0.0; v[j] = 0.0;
        s[0] = fma(rj, rj, s[0]); s[1] = fma(bj, bj, s[1]);
    }
    cta_reduce<2>(s, smem);
    if (threadIdx.x == 0) { part[2LL * blockIdx.x] = s[0]; part[2LL * blockIdx.x + 1] = s[1]; }
}
// p = r + beta (p - omega v) ; y = M^-1 p
__global__ void __launch_bounds__(RED_THREADS)
k_bicg_p(long long n, const double *__restrict__ sc, const double *__restrict__ r, const double *__restrict__ v,
         const double *__restrict__ dinv, double *__restrict__ p, double *__restrict__ y) {
    const double beta = sc[4], omega = sc[3];   // omega of the previous iteration
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        const double pj = fma(beta, fma(-omega, v[j], p[j]), r[j]);
        p[j] = pj; y[j] = dinv[j] * pj;
    }
}
// s = r - alpha v ; z = M^-1 s ; partial (s, s)
__global__ void __launch_bounds__(RED_THREADS)
k_bicg_s(long long n, const double *__restrict__ sc, const double *__restrict__ r, const double *__restrict__ v,
         const double *__restrict__ dinv, double *__restrict__ s, double *__restrict__ z, double *__restrict__ part) {
    __shared__ double smem[32];
    double a[1] = {0.0};
    const double alpha = sc[2];
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        const double sj = fma(-alpha, v[j], r[j]);
        s[j] = sj; z[j] = dinv[j] * sj;
        a[0] = fma(sj, sj, a[0]);
    }
    cta_reduce<1>(a, smem);
    if (threadIdx.x == 0) part[blockIdx.x] = a[0];
}
// x += alpha y + omega z ; r = s - omega t ; partials (rhat, r), (r, r)
__global__ void __launch_bounds__(RED_THREADS)
k_bicg_xr(long long n, const double *__restrict__ sc, const double *__restrict__ y, const double *__restrict__ z,
          const double *__restrict__ s, const double *__restrict__ t, const double *__restrict__ rhat, double *__restrict__ x,
          double *__restrict__ r, double *__restrict__ part) {
    __shared__ double smem[2 * 32];
    double a[2] = {0.0, 0.0};
    const double alpha = sc[2], omega = sc[3];
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        x[j] = fma(omega, z[j], fma(alpha, y[j], x[j]));
        const double rj = fma(-omega, t[j], s[j]);
        r[j] = rj;
        a[0] = fma(rhat[j], rj, a[0]); a[1] = fma(rj, rj, a[1]);
    }
    cta_reduce<2>(a, smem);
    if (threadIdx.x == 0) { part[2LL * blockIdx.x] = a[0]; part[2LL * blockIdx.x + 1] = a[1]; }
}
// ---- BiCGSTAB scalars on the device: sc[0] rho, [1] rho_old, [2] alpha, [3] omega, [4] beta, [5] (r,r), [6] tol^2 (b,b),
//      [7] flag (0 running, 1 converged, 2 breakdown: the host restarts), [8] iterations, [9] |rhat|.  A solve whose flag is
//      set keeps alpha = omega = beta = 0, so the remaining iterations of a batch change neither x nor r.
template <int NV>
__device__ __forceinline__ void sum_partials(const double *__restrict__ part, long long count, double (&v)[NV], double *smem) {
#pragma unroll
    for (int k = 0; k < NV; k++) v[k] = 0.0;
    for (long long j = threadIdx.x; j < count; j += blockDim.x)
#pragma unroll
        for (int k = 0; k < NV; k++) v[k] += part[j * NV + k];
    cta_reduce<NV>(v, smem);
}
__device__ __forceinline__ void bi_next_beta(double *sc) {   // breakdown guard + beta of the next iteration
    const double rho = sc[0], omega = sc[3];
    if (!(fabs(rho) > 1e-12 * sqrt(sc[5]) * sc[9]) || !isfinite(rho) || omega == 0.0 || !isfinite(omega)) { sc[7] = 2.0; sc[4] = 0.0; }
    else sc[4] = (rho / sc[1]) * (sc[2] / omega);
}
__global__ void __launch_bounds__(1024) k_bi_alpha(const double *__restrict__ part, long long count, double *sc) {   // after v = K y
    __shared__ double smem[2 * 32];
    double v[2];
    sum_partials<2>(part, count, v, smem);
    if (threadIdx.x == 0) {
        if (sc[7] == 0.0) {
            sc[8] += 1.0;
            if (v[0] == 0.0 || !isfinite(v[0])) sc[7] = 2.0;
        }
        sc[2] = (sc[7] == 0.0) ? sc[0] / v[0] : 0.0;
    }
}
__global__ void __launch_bounds__(1024) k_bi_half(const double *__restrict__ part, long long count, double *sc) {    // after s = r - alpha v
    __shared__ double smem[32];
    double v[1];
    sum_partials<1>(part, count, v, smem);
    if (threadIdx.x == 0 && sc[7] == 0.0 && v[0] <= sc[6]) { sc[7] = 1.0; sc[5] = v[0]; }   // the half step suffices: omega = 0 below, x += alpha y, r = s
}
__global__ void __launch_bounds__(1024) k_bi_omega(const double *__restrict__ part, long long count, double *sc) {   // after t = K z
    __shared__ double smem[2 * 32];
    double v[2];
    sum_partials<2>(part, count, v, smem);
    if (threadIdx.x == 0) sc[3] = (sc[7] == 0.0 && v[1] > 0.0 && isfinite(v[1])) ? v[0] / v[1] : 0.0;
}
__global__ void __launch_bounds__(1024) k_bi_rho(const double *__restrict__ part, long long count, double *sc) {     // after the x, r update
    __shared__ double smem[2 * 32];
    double v[2];
    sum_partials<2>(part, count, v, smem);
    if (threadIdx.x == 0) {
        if (sc[7] == 0.0) {
            sc[1] = sc[0]; sc[0] = v[0]; sc[5] = v[1];
            if (v[1] <= sc[6]) sc[7] = 1.0;
            else bi_next_beta(sc);
        }
        if (sc[7] != 0.0) sc[4] = 0.0;
    }
}
// ---- CG scalars stay on the device (no host round trip per iteration).  sc[0] = (r,z), sc[1] = alpha, sc[2] = beta,
//      sc[3] = (r,r), sc[4] = tol^2 (b,b), sc[5] = done flag (1 converged, 2 breakdown), sc[6] = iterations performed.
// after q = K p: alpha = (r,z) / (p,q); a solve that is done keeps alpha = 0, so later iterations of the batch change nothing
__global__ void __launch_bounds__(1024) k_cg_alpha(const double *__restrict__ part, long long count, double *sc) {
    __shared__ double smem[2 * 32];
    double v[2] = {0.0, 0.0};
    for (long long j = threadIdx.x; j < count; j += blockDim.x) { v[0] += part[2 * j]; v[1] += part[2 * j + 1]; }
    cta_reduce<2>(v, smem);
    if (threadIdx.x == 0) {
        const double pq = v[0];
        if (sc[5] == 0.0 && (!(pq > 0.0) || !isfinite(pq))) sc[5] = 2.0;
        sc[1] = (sc[5] == 0.0) ? sc[0] / pq : 0.0;
        if (sc[5] == 0.0) sc[6] += 1.0;
    }
}
// after the update: beta = (r,z)_new / (r,z); convergence and breakdown tests
__global__ void __launch_bounds__(1024) k_cg_beta(const double *__restrict__ part, long long count, double *sc) {
    __shared__ double smem[2 * 32];
    double v[2] = {0.0, 0.0};
    for (long long j = threadIdx.x; j < count; j += blockDim.x) { v[0] += part[2 * j]; v[1] += part[2 * j + 1]; }
    cta_reduce<2>(v, smem);
    if (threadIdx.x == 0 && sc[5] == 0.0) {
        const double rz_new = v[0], rr = v[1];
        sc[3] = rr;
        if (rr <= sc[4]) sc[5] = 1.0;
        else if (!(rz_new > 0.0) || !isfinite(rz_new)) sc[5] = 2.0;
        sc[2] = rz_new / sc[0];
        sc[0] = rz_new;
    }
}
// ---- preconditioned CG vector kernels
// x += alpha p ; r -= alpha q ; z = M^-1 r ; partials (r, z), (r, r)
__global__ void __launch_bounds__(RED_THREADS)
k_cg_update(long long n, double alpha_h, const double *__restrict__ sc, const double *__restrict__ p, const double *__restrict__ q,
            const double *__restrict__ dinv, double *__restrict__ x, double *__restrict__ r, double *__restrict__ z,
            double *__restrict__ part) {
    __shared__ double smem[2 * 32];
    double a[2] = {0.0, 0.0};
    const double alpha = sc ? sc[1] : alpha_h;
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        x[j] = fma(alpha, p[j], x[j]);
        const double rj = fma(-alpha, q[j], r[j]), zj = dinv[j] * rj;
        r[j] = rj; z[j] = zj;
        a[0] = fma(rj, zj, a[0]); a[1] = fma(rj, rj, a[1]);
    }
    cta_reduce<2>(a, smem);
    if (threadIdx.x == 0) { part[2LL * blockIdx.x] = a[0]; part[2LL * blockIdx.x + 1] = a[1]; }
}
// p = z + beta p
__global__ void k_cg_p(long long n, double beta_h, const double *__restrict__ sc, const double *__restrict__ z, double *__restrict__ p) {
    const double beta = sc ? sc[2] : beta_h;
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x)
        p[j] = fma(beta, p[j], z[j]);
}
// x += alpha y (early exit after the first half step)
__global__ void k_axpy(long long n, double alpha, const double *__restrict__ y, double *__restrict__ x) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x)
        x[j] = fma(alpha, y[j], x[j]);
}
// rhs = -R ; partial (rhs, rhs) is taken later, after the Dirichlet rows
__global__ void k_neg(long long n, const double *__restrict__ a, double *__restrict__ out) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) out[j] = -a[j];
}
__global__ void __launch_bounds__(RED_THREADS) k_norm2(long long n, const double *__restrict__ a, double *__restrict__ part) {
    __shared__ double smem[32];
    double s[1] = {0.0};
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) s[0] = fma(a[j], a[j], s[0]);
    cta_reduce<1>(s, smem);
    if (threadIdx.x == 0) part[blockIdx.x] = s[0];
}

// ------------------------------------------------------------------------------------------------ host side
static int ensure_solver_ws(fem_ctx *c, bool newton) {
    const long long n = c->n_rows;
    if (!c->d_diagpos) {
        FEM_CUDA(cudaMalloc(&c->d_diagpos, sizeof(int) * c->n_nodes));
        k_diagpos<<<nblk3(c->n_nodes, 256), 256>>>(c->n_nodes, c->d_nb_ptr, c->d_nb, c->d_diagpos);
        FEM_CUDA(cudaGetLastError());
        FEM_CUDA(cudaDeviceSynchronize());
    }
    if (!c->d_sw) {
        const long long spmv_ctas = spmv_grid(c);
        c->n_part = 2 * (spmv_ctas > RED_CTAS ? spmv_ctas : RED_CTAS);
        // all or nothing: a failed allocation leaves no half-built workspace behind for the next call to trip over
        double *sw = nullptr, *part = nullptr, *scal = nullptr;
        cudaError_t e = cudaMalloc(&sw, sizeof(double) * 9 * n);
        if (e == cudaSuccess) e = cudaMalloc(&part, sizeof(double) * c->n_part);
        if (e == cudaSuccess) e = cudaMalloc(&scal, sizeof(double) * 64);   // [0..8) reduction results, [16..48) solver scalars
        if (e != cudaSuccess) {
            if (sw) cudaFree(sw);
            if (part) cudaFree(part);
            if (scal) cudaFree(scal);
            return fem_cuda_fail(e, "cudaMalloc(solver workspace)");
        }
        c->d_sw = sw; c->d_part = part; c->d_scal = scal;
    }
    if (newton && !c->d_nw) {
        double *nw = nullptr, *nv = nullptr;
        cudaError_t e = cudaMalloc(&nw, sizeof(double) * 4 * n);
        if (e == cudaSuccess) e = cudaMalloc(&nv, sizeof(double) * (size_t)c->nnz);
        if (e != cudaSuccess) {
            if (nw) cudaFree(nw);
            if (nv) cudaFree(nv);
            return fem_cuda_fail(e, "cudaMalloc(Newton workspace)");
        }
        c->d_nw = nw; c->d_nw_vals = nv;
    }
    return FEM_OK;
}

// reduces `count` partial records of NV values and brings them to the host (synchronises the stream)
template <int NV>
static int fetch_sums(fem_ctx *c, long long count, double *host, cudaStream_t st) {
    k_reduce_final<NV><<<1, 1024, 0, st>>>(c->d_part, count, c->d_scal);
    FEM_CUDA(cudaMemcpyAsync(host, c->d_scal, sizeof(double) * NV, cudaMemcpyDeviceToHost, st));
    FEM_CUDA(cudaStreamSynchronize(st));
    return FEM_OK;
}

template <int DOT>
static void launch_spmv(fem_ctx *c, const double *vals, const double *x, double *y, const double *w, cudaStream_t st) {
    k_spmv<DOT><<<spmv_grid(c), 256, 0, st>>>(c->n_nodes, c->d_nb_ptr, c->d_nb, vals, x, y, w, c->d_part);
}

static void launch_spmv32_dot(fem_ctx *c, const float *vals, const double *x, double *y, const double *w, cudaStream_t st) {
    k_spmv<1, float><<<spmv_grid(c), 256, 0, st>>>(c->n_nodes, c->d_nb_ptr, c->d_nb, vals, x, y, w, c->d_part);
}
__global__ void k_to_f32(long long n, const double *__restrict__ a, float *__restrict__ out) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) out[i] = (float)a[i];
}

extern "C" int fem_spmv(fem_ctx *c, const double *csr_vals, const double *x, double *y, void *cuda_stream) {
    if (!c || !csr_vals || !x || !y) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (x == y) return FEM_ERR_ALIAS;
    launch_spmv<0>(c, csr_vals, x, y, nullptr, (cudaStream_t)cuda_stream);
    FEM_CUDA(cudaGetLastError());
    return FEM_OK;
}

static int apply_dirichlet(fem_ctx *c, long long n_bc, const int *bc_dofs, const double *bc_rhs, const double *bc_vals,
                           const double *u, double *vals, double *rhs, cudaStream_t st) {
    if (n_bc == 0) return FEM_OK;
    k_dirichlet<<<nblk3(n_bc, 128), 128, 0, st>>>(n_bc, bc_dofs, bc_rhs, bc_vals, u, c->d_nb_ptr, c->d_diagpos, vals, rhs);
    FEM_CUDA(cudaGetLastError());
    return FEM_OK;
}

static int check_dofs(fem_ctx *c, long long n_bc, const int *bc_dofs, cudaStream_t st) {
    if (n_bc == 0) return FEM_OK;
    int h = 0;
    FEM_CUDA(cudaMemsetAsync(c->d_scal, 0, sizeof(int), st));
    k_check_dofs<<<nblk3(n_bc, 256), 256, 0, st>>>(n_bc, bc_dofs, c->n_rows, reinterpret_cast<int *>(c->d_scal));
    FEM_CUDA(cudaMemcpyAsync(&h, c->d_scal, sizeof(int), cudaMemcpyDeviceToHost, st));
    FEM_CUDA(cudaStreamSynchronize(st));
    return h ? FEM_ERR_ARG : FEM_OK;
}

extern "C" int fem_apply_dirichlet(fem_ctx *c, long long n_bc, const int *bc_dofs, const double *bc_rhs, double *csr_vals,
                                   double *rhs, void *cuda_stream) {
    if (!c || !csr_vals || (n_bc > 0 && !bc_dofs)) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (n_bc < 0) return FEM_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = ensure_solver_ws(c, false);
    if (rc != FEM_OK) return rc;
    rc = check_dofs(c, n_bc, bc_dofs, st);
    if (rc != FEM_OK) return rc;
    return apply_dirichlet(c, n_bc, bc_dofs, bc_rhs, nullptr, nullptr, csr_vals, rhs, st);
}

// Jacobi-preconditioned BiCGSTAB, right preconditioning (van der Vorst 1992; the paper's default Krylov method):
//   rho = (rhat, r); beta = (rho/rho_old)(alpha/omega); p = r + beta (p - omega v); y = M^-1 p; v = K y;
//   alpha = rho / (rhat, v); s = r - alpha v; z = M^-1 s; t = K z; omega = (t, s)/(t, t);
//   x += alpha y + omega z; r = s - omega t.
static int bicgstab(fem_ctx *c, const double *vals, const double *b, double *x, double rtol, int max_iter, int *iters,
                    double *relres, cudaStream_t st) {
    const long long n = c->n_rows;
    double *r = c->d_sw, *rhat = r + n, *p = rhat + n, *v = p + n, *s = v + n, *t = s + n, *y = t + n, *z = y + n, *dinv = z + n;
    const long long spmv_ctas = spmv_grid(c);
    double h[2];
    k_dinv<<<nblk3(n, 256), 256, 0, st>>>(c->n_nodes, c->d_nb_ptr, c->d_diagpos, vals, dinv);
    launch_spmv<0>(c, vals, x, r, nullptr, st);
    k_bicg_init<<<RED_CTAS, RED_THREADS, 0, st>>>(n, b, r, rhat, p, v, c->d_part);
    int rc = fetch_sums<2>(c, RED_CTAS, h, st);
    if (rc != FEM_OK) return rc;
    double rr = h[0];
    const double bb = h[1];
    int it = 0;
    bool conv = false;
    if (bb == 0.0) {   // b = 0: the solution is x = 0
        FEM_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
        if (iters) *iters = 0;
        if (relres) *relres = 0.0;
        return FEM_OK;
    }
    const double tol2 = rtol * rtol * bb;
    conv = rr <= tol2;
    // iterations run in batches without a host round trip (scalars in d_scal); the host looks at the flag after each batch
    // and restarts from the true residual of the current x (rhat = r = b - K x, p = v = 0) when the recurrence broke down
    double *sc = c->d_scal + 16;
    int restarts = 0;
    const int batch = 8;
    bool fresh = true;   // r, rhat, p, v and rr describe a fresh start
    while (!conv && it < max_iter) {
        if (!fresh) {
            if (++restarts > 50) break;
            launch_spmv<0>(c, vals, x, r, nullptr, st);
            k_bicg_init<<<RED_CTAS, RED_THREADS, 0, st>>>(n, b, r, rhat, p, v, c->d_part);
            if ((rc = fetch_sums<2>(c, RED_CTAS, h, st)) != FEM_OK) return rc;
            rr = h[0];
            if (rr <= tol2) { conv = true; break; }
            if (!isfinite(rr)) break;
        }
        // rho = (rhat, r) = rr, rho_old = alpha = omega = 1, beta irrelevant (p = v = 0)
        const double sc0[16] = {rr, 1.0, 1.0, 1.0, rr, rr, tol2, 0.0, (double)it, sqrt(rr), 0, 0, 0, 0, 0, 0};
        FEM_CUDA(cudaMemcpyAsync(sc, sc0, sizeof(sc0), cudaMemcpyHostToDevice, st));
        FEM_CUDA(cudaStreamSynchronize(st));   // sc0 is on the stack
        fresh = false;
        double hs[16];
        hs[7] = 0.0;
        while (it < max_iter && hs[7] == 0.0) {
            const int nb = (max_iter - it < batch) ? max_iter - it : batch;
            for (int j = 0; j < nb; j++) {
                k_bicg_p<<<RED_CTAS, RED_THREADS, 0, st>>>(n, sc, r, v, dinv, p, y);
                launch_spmv<1>(c, vals, y, v, rhat, st);
                k_bi_alpha<<<1, 1024, 0, st>>>(c->d_part, spmv_ctas, sc);
                k_bicg_s<<<RED_CTAS, RED_THREADS, 0, st>>>(n, sc, r, v, dinv, s, z, c->d_part);
                k_bi_half<<<1, 1024, 0, st>>>(c->d_part, RED_CTAS, sc);
                launch_spmv<2>(c, vals, z, t, s, st);
                k_bi_omega<<<1, 1024, 0, st>>>(c->d_part, spmv_ctas, sc);
                k_bicg_xr<<<RED_CTAS, RED_THREADS, 0, st>>>(n, sc, y, z, s, t, rhat, x, r, c->d_part);
                k_bi_rho<<<1, 1024, 0, st>>>(c->d_part, RED_CTAS, sc);
            }
            FEM_CUDA(cudaMemcpyAsync(hs, sc, sizeof(hs), cudaMemcpyDeviceToHost, st));
            FEM_CUDA(cudaStreamSynchronize(st));
            it = (int)hs[8];
        }
        if (hs[7] == 1.0) conv = true;
        // hs[7] == 2: breakdown -> the outer loop restarts; 0: iteration cap
    }
    // explicit residual of the returned x (the recurrence residual can drift)
    launch_spmv<0>(c, vals, x, r, nullptr, st);
    k_bicg_init<<<RED_CTAS, RED_THREADS, 0, st>>>(n, b, r, rhat, p, v, c->d_part);
    if ((rc = fetch_sums<2>(c, RED_CTAS, h, st)) != FEM_OK) return rc;
    const double rel = sqrt(h[0] / bb);
    if (iters) *iters = it;
    if (relres) *relres = rel;
    FEM_CUDA(cudaGetLastError());
    return (conv && rel <= 100.0 * rtol) ? FEM_OK : FEM_ERR_NOCONV;
}

// Jacobi-preconditioned conjugate gradients (Hestenes-Stiefel) for a symmetric positive definite K.  With identity rows for
// the constrained DOFs and an initial guess that already carries the prescribed values there, every Krylov vector is zero
// on the constrained DOFs and the iteration is CG on the symmetric reduced system K_ff (the row-eliminated K of Alg. E1 is
// not symmetric as a whole).  Returns FEM_ERR_NOCONV also when (p, K p) <= 0 (K not positive definite).
static int pcg(fem_ctx *c, const double *vals, const double *b, double *x, double rtol, int max_iter, int *iters, double *relres,
               cudaStream_t st) {
    const long long n = c->n_rows;
    double *r = c->d_sw, *z = r + n, *p = z + n, *q = p + n, *scratch = q + n, *dinv = c->d_sw + 8 * n;
    const long long spmv_ctas = spmv_grid(c);
    double h[2];
    int rc;
    // Mixed precision (fem_set_mixed_precision): the SpMV of the iteration reads an fp32 copy of K (half the bytes of an
    // HBM-bound kernel); every residual that decides convergence is b - K x with the fp64 matrix, and the iteration is
    // restarted from it (iterative refinement) until that residual meets rtol.  Vectors and scalars are fp64 throughout.
    const float *v32 = nullptr;
    if (c->mixed_precision) {
        if (!c->d_vals32) FEM_CUDA(cudaMalloc(&c->d_vals32, sizeof(float) * (size_t)c->nnz));
        k_to_f32<<<RED_CTAS * 8, RED_THREADS, 0, st>>>(c->nnz, vals, c->d_vals32);
        v32 = c->d_vals32;
    }
    k_dinv<<<nblk3(n, 256), 256, 0, st>>>(c->n_nodes, c->d_nb_ptr, c->d_diagpos, vals, dinv);
    launch_spmv<0>(c, vals, x, r, nullptr, st);
    k_bicg_init<<<RED_CTAS, RED_THREADS, 0, st>>>(n, b, r, scratch, p, q, c->d_part);   // r = b - K x, p = q = 0
    if ((rc = fetch_sums<2>(c, RED_CTAS, h, st)) != FEM_OK) return rc;
    const double bb = h[1];
    if (bb == 0.0) {
        FEM_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
        if (iters) *iters = 0;
        if (relres) *relres = 0.0;
        return FEM_OK;
    }
    const double tol2 = rtol * rtol * bb;
    bool conv = h[0] <= tol2, bad = false;
    int it = 0;
    for (int round = 0; !conv && !bad && it < max_iter && round < 10; round++) {
        const double rr = h[0];
        // a refinement round asks for at most five orders of magnitude: below that the fp32 matrix, not the iteration, sets the residual
        const double tol2_round = (v32 && 1e-10 * rr > tol2) ? 1e-10 * rr : tol2;
        // z = M^-1 r and (r, z): one k_cg_update with alpha = 0
        k_cg_update<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 0.0, nullptr, p, q, dinv, x, r, z, c->d_part);
        if ((rc = fetch_sums<2>(c, RED_CTAS, h, st)) != FEM_OK) return rc;
        // iterations run in batches without a host round trip; the scalars live in d_scal, a finished solve freezes itself
        double sc0[8] = {h[0], 0.0, 0.0, rr, tol2_round, 0.0, 0.0, 0.0};
        double *sc = c->d_scal + 16;
        FEM_CUDA(cudaMemcpyAsync(sc, sc0, sizeof(sc0), cudaMemcpyHostToDevice, st));
        FEM_CUDA(cudaStreamSynchronize(st));   // sc0 is on the stack
        const int batch = 16, it0 = it;
        bool round_conv = false;
        while (it < max_iter) {
            const int nb = (max_iter - it < batch) ? max_iter - it : batch;
            for (int j = 0; j < nb; j++) {
                k_cg_p<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 0.0, sc, z, p);              // p = z + beta p (beta = 0 at first)
                if (v32) launch_spmv32_dot(c, v32, p, q, p, st);                        // q = K p, partial (p, q)
                else launch_spmv<1>(c, vals, p, q, p, st);
                k_cg_alpha<<<1, 1024, 0, st>>>(c->d_part, spmv_ctas, sc);
                k_cg_update<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 0.0, sc, p, q, dinv, x, r, z, c->d_part);
                k_cg_beta<<<1, 1024, 0, st>>>(c->d_part, RED_CTAS, sc);
            }
            double hs[8];
            FEM_CUDA(cudaMemcpyAsync(hs, sc, sizeof(hs), cudaMemcpyDeviceToHost, st));
            FEM_CUDA(cudaStreamSynchronize(st));
            it = it0 + (int)hs[6];
            if (hs[5] == 1.0) { round_conv = true; break; }
            if (hs[5] == 2.0) { bad = true; break; }
        }
        // the residual that counts: b - K x with the fp64 matrix (also the start of the next refinement round)
        launch_spmv<0>(c, vals, x, r, nullptr, st);
        k_bicg_init<<<RED_CTAS, RED_THREADS, 0, st>>>(n, b, r, scratch, p, q, c->d_part);
        if ((rc = fetch_sums<2>(c, RED_CTAS, h, st)) != FEM_OK) return rc;
        conv = v32 ? (h[0] <= tol2) : round_conv;
        if (!v32 || !round_conv) break;
    }
    const double rel = sqrt(h[0] / bb);
    if (iters) *iters = it;
    if (relres) *relres = rel;
    FEM_CUDA(cudaGetLastError());
    return (conv && !bad && rel <= 100.0 * rtol) ? FEM_OK : FEM_ERR_NOCONV;
}

extern "C" int fem_set_mixed_precision(fem_ctx *c, int on) {
    if (!c) return FEM_ERR_NULL;
    c->mixed_precision = on ? 1 : 0;
    return FEM_OK;
}

extern "C" int fem_pcg(fem_ctx *c, const double *csr_vals, const double *b, double *x, double rtol, int max_iter, int *iters,
                       double *relres, void *cuda_stream) {
    if (!c || !csr_vals || !b || !x) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (!(rtol > 0.0) || max_iter < 0 || b == x) return FEM_ERR_ARG;
    int rc = ensure_solver_ws(c, false);
    if (rc != FEM_OK) return rc;
    return pcg(c, csr_vals, b, x, rtol, max_iter, iters, relres, (cudaStream_t)cuda_stream);
}

extern "C" int fem_bicgstab(fem_ctx *c, const double *csr_vals, const double *b, double *x, double rtol, int max_iter, int *iters,
                            double *relres, void *cuda_stream) {
    if (!c || !csr_vals || !b || !x) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (!(rtol > 0.0) || max_iter < 0 || b == x) return FEM_ERR_ARG;
    int rc = ensure_solver_ws(c, false);
    if (rc != FEM_OK) return rc;
    return bicgstab(c, csr_vals, b, x, rtol, max_iter, iters, relres, (cudaStream_t)cuda_stream);
}

__global__ void k_lincomb(long long n, double a, const double *__restrict__ x, double b, const double *__restrict__ y, double *out) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x)
        out[j] = fma(a, x[j], b * y[j]);
}
extern "C" int fem_lincomb(fem_ctx *c, double a, const double *x, double b, const double *y, double *out, void *cuda_stream) {
    if (!c || !x || !y || !out) return FEM_ERR_NULL;
    k_lincomb<<<RED_CTAS, RED_THREADS, 0, (cudaStream_t)cuda_stream>>>(c->n_rows, a, x, b, y, out);
    FEM_CUDA(cudaGetLastError());
    return FEM_OK;
}

extern "C" void fem_default_newton_options(fem_newton_options *o) {
    if (!o) return;
    o->rtol = 1e-9; o->atol = 1e-10; o->max_newton = 25; o->lin_rtol = 1e-10; o->lin_max_iter = 10000; o->linear_solver = 0;
}

// One load increment: K dd = -R, d <- d + dd (Eq.(39)) with identity rows for the constrained DOFs.
extern "C" int fem_newton_solve(fem_ctx *c, double *u, const double *hist_in, const double *mat, long long n_mat, long long n_bc,
                                const int *bc_dofs, const double *bc_vals, double *hist_out, const fem_newton_options *opt,
                                fem_newton_report *rep, void *cuda_stream) {
    if (!c || !u || !hist_in || !mat || !hist_out || (n_bc > 0 && (!bc_dofs || !bc_vals))) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (n_mat != 1 && n_mat != c->n_elems) return FEM_ERR_MAT;
    if (n_bc < 0) return FEM_ERR_ARG;
    fem_newton_options o;
    fem_default_newton_options(&o);
    if (opt) o = *opt;
    if (!(o.rtol >= 0.0) || !(o.atol >= 0.0) || o.max_newton < 1 || !(o.lin_rtol > 0.0) || o.lin_max_iter < 1 || o.linear_solver < 0 || o.linear_solver > 2) return FEM_ERR_ARG;
    if (fem_ranges_overlap(hist_in, hist_out, sizeof(double) * 56 * (size_t)c->n_elems)) return FEM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = ensure_solver_ws(c, true);
    if (rc != FEM_OK) return rc;
    if ((rc = check_dofs(c, n_bc, bc_dofs, st)) != FEM_OK) return rc;
    const long long n = c->n_rows;
    double *R = c->d_nw, *rhs = R + n, *dd = rhs + n, *u_entry = dd + n, *vals = c->d_nw_vals;
    FEM_CUDA(cudaMemcpyAsync(u_entry, u, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    fem_newton_report rp;
    memset(&rp, 0, sizeof(rp));
    int result = FEM_ERR_NOCONV;
    int err = FEM_OK;   // a hard error (CUDA, allocation) inside the loop: u is restored before it is returned
    for (int k = 0;; k++) {
        if ((err = fem_launch_assemble(c, u, hist_in, mat, n_mat, R, vals, hist_out, st)) != FEM_OK) break;
        if ((err = fem_read_stats(c, &rp.last_stats, st)) != FEM_OK) break;
        k_neg<<<RED_CTAS, RED_THREADS, 0, st>>>(n, R, rhs);
        if ((err = apply_dirichlet(c, n_bc, bc_dofs, nullptr, bc_vals, u, vals, rhs, st)) != FEM_OK) break;
        k_norm2<<<RED_CTAS, RED_THREADS, 0, st>>>(n, rhs, c->d_part);
        double h[1];
        if ((err = fetch_sums<1>(c, RED_CTAS, h, st)) != FEM_OK) break;
        rp.rhs_norm = sqrt(h[0]);
        if (k == 0) rp.rhs_norm0 = rp.rhs_norm;
        if (!isfinite(rp.rhs_norm)) break;
        if (rp.rhs_norm <= o.atol || rp.rhs_norm <= o.rtol * rp.rhs_norm0) {
            // a state that balances but holds inverted points, local solves that hit kmax or non-finite stresses is no root of
            // the discrete problem (hist_out is not the return-map solution there): the increment is rejected so that the
            // caller cuts the step back, as the paper's step control does
            const fem_stats &ls = rp.last_stats;
            rp.physics_trouble = (ls.n_nonconverged > 0 || ls.n_detF_nonpos > 0 || ls.n_nonfinite > 0) ? 1 : 0;
            if (!rp.physics_trouble) { rp.converged = 1; result = FEM_OK; }
            break;
        }
        if (k >= o.max_newton) break;
        int its = 0;
        rc = FEM_ERR_NOCONV;
        if (o.linear_solver != 1 && !c->opt.fbar) {
            // standard element: K_ff is symmetric -> CG from the guess dd = rhs on the constrained DOFs, 0 elsewhere
            if ((err = fem_cuda_rc(cudaMemsetAsync(dd, 0, sizeof(double) * n, st), "cudaMemsetAsync(dd)")) != FEM_OK) break;
            if (n_bc > 0) k_scatter_bc<<<nblk3(n_bc, 256), 256, 0, st>>>(n_bc, bc_dofs, rhs, dd);
            rc = pcg(c, vals, rhs, dd, o.lin_rtol, o.lin_max_iter, &its, nullptr, st);
            rp.lin_iters_total += its;
        }
        if (rc == FEM_ERR_NOCONV && (o.linear_solver != 2 || c->opt.fbar)) {   // unsymmetric (F-bar), or CG gave up: BiCGSTAB from zero
            if ((err = fem_cuda_rc(cudaMemsetAsync(dd, 0, sizeof(double) * n, st), "cudaMemsetAsync(dd)")) != FEM_OK) break;
            rc = bicgstab(c, vals, rhs, dd, o.lin_rtol, o.lin_max_iter, &its, nullptr, st);
            rp.lin_iters_total += its;
        }
        if (rc == FEM_ERR_NOCONV) rp.lin_failures++;
        else if (rc != FEM_OK) { err = rc; break; }
        k_axpy<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 1.0, dd, u);
        rp.newton_iters++;
    }
    if (result != FEM_OK || err != FEM_OK)   // failed increment or error: u goes back to its entry value, so the caller can cut the step back
        cudaMemcpyAsync(u, u_entry, sizeof(double) * n, cudaMemcpyDeviceToDevice, st);
    if (err != FEM_OK) { cudaStreamSynchronize(st); if (rep) *rep = rp; return err; }
    FEM_CUDA(cudaGetLastError());
    FEM_CUDA(cudaStreamSynchronize(st));
    if (rep) *rep = rp;
    return result;
}

// ---- load path: the paper's adaptive load stepping around the Newton increment (settings of the unit-cube
// benchmark :485).  Host control flow only: every number is produced by the kernels behind fem_newton_solve / fem_lincomb.
extern "C" void fem_default_path_options(fem_path_options *o) {
    if (!o) return;
    o->dt0 = 1e-3; o->dt_min = 1e-5; o->dt_max = 5e-2; o->grow = 1.5; o->cut = 0.5; o->grow_below = 5; o->max_steps = 10000;
    o->extrapolate = 1;
    fem_default_newton_options(&o->newton);
    o->newton.rtol = 1e-8; o->newton.max_newton = 12; o->newton.lin_rtol = 1e-6; o->newton.lin_max_iter = 20000;
}

__global__ void k_scale(long long n, double a, const double *__restrict__ x, double *__restrict__ out) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) out[j] = a * x[j];
}

extern "C" int fem_load_path(fem_ctx *c, double *u, double *hist, const double *mat, long long n_mat, long long n_bc,
                             const int *bc_dofs, const double *bc_full, const fem_path_options *opt, fem_path_report *rep,
                             double *t_accepted, int n_t_cap, void *cuda_stream) {
    if (!c || !u || !hist || !mat || (n_bc > 0 && (!bc_dofs || !bc_full))) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (n_mat != 1 && n_mat != c->n_elems) return FEM_ERR_MAT;
    fem_path_options o;
    fem_default_path_options(&o);
    if (opt) o = *opt;
    if (!(o.dt0 > 0.0) || !(o.dt_min > 0.0) || !(o.dt_max >= o.dt_min) || !(o.grow >= 1.0) || !(o.cut > 0.0 && o.cut < 1.0) ||
        o.max_steps < 1 || o.extrapolate < 0 || o.extrapolate > 2 || n_bc < 0 || (t_accepted && n_t_cap < 0))
        return FEM_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long n = c->n_rows;
    const size_t hb = sizeof(double) * 56 * (size_t)c->n_elems;
    if (!c->d_path) {   // u_try, u_prev, u_pp, bc values of the step (n_rows each) and the second history buffer: all or nothing
        double *pw = nullptr, *ph = nullptr;
        cudaError_t e = cudaMalloc(&pw, sizeof(double) * 4 * n);
        if (e == cudaSuccess) e = cudaMalloc(&ph, hb);
        if (e != cudaSuccess) { if (pw) cudaFree(pw); if (ph) cudaFree(ph); return fem_cuda_fail(e, "cudaMalloc(load path workspace)"); }
        c->d_path = pw; c->d_path_hist = ph;
    }
    double *u_try = c->d_path, *u_prev = u_try + n, *u_pp = u_prev + n, *bcv = u_pp + n;
    double *h_a = hist, *h_b = c->d_path_hist;          // history at the start of the step / written by the step
    FEM_CUDA(cudaMemcpyAsync(u_prev, u, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    FEM_CUDA(cudaMemcpyAsync(u_pp, u, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    fem_path_report rp;
    memset(&rp, 0, sizeof(rp));
    double t = 0.0, dt = o.dt0 < o.dt_max ? o.dt0 : o.dt_max, dt_prev = 0.0, dt_pp = 0.0;
    int rc = FEM_OK;
    while (t < 1.0 - 1e-12) {
        if (rp.steps + rp.rejected >= o.max_steps) { rc = FEM_ERR_NOCONV; break; }
        if (dt > 1.0 - t) dt = 1.0 - t;
        // initial guess: extrapolation of the converged states ("linear or quadratic extrapolation")
        if (o.extrapolate == 2 && dt_pp > 0.0) {   // Lagrange parabola through the last three converged states
            const double t0 = -(dt_prev + dt_pp), t1 = -dt_prev, t2 = 0.0, t3 = dt;
            const double l0 = (t3 - t1) * (t3 - t2) / ((t0 - t1) * (t0 - t2)), l1 = (t3 - t0) * (t3 - t2) / ((t1 - t0) * (t1 - t2)),
                         l2 = (t3 - t0) * (t3 - t1) / ((t2 - t0) * (t2 - t1));
            k_lincomb<<<RED_CTAS, RED_THREADS, 0, st>>>(n, l2, u, l1, u_prev, u_try);
            k_lincomb<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 1.0, u_try, l0, u_pp, u_try);
        } else {
            const double r = (o.extrapolate && dt_prev > 0.0) ? dt / dt_prev : 0.0;
            k_lincomb<<<RED_CTAS, RED_THREADS, 0, st>>>(n, 1.0 + r, u, -r, u_prev, u_try);   // u + (u - u_prev) dt / dt_prev
        }
        if (n_bc > 0) k_scale<<<nblk3(n_bc, 256), 256, 0, st>>>(n_bc, t + dt, bc_full, bcv);
        fem_newton_report nr;
        rc = fem_newton_solve(c, u_try, h_a, mat, n_mat, n_bc, bc_dofs, bcv, h_b, &o.newton, &nr, cuda_stream);
        rp.newton_iters_total += nr.newton_iters;
        rp.lin_iters_total += nr.lin_iters_total;
        if (rc != FEM_OK && rc != FEM_ERR_NOCONV) break;
        const bool ok = (rc == FEM_OK) && nr.converged && nr.lin_failures == 0;
        if (ok) {
            t += dt;
            if (t_accepted && rp.steps < n_t_cap) t_accepted[rp.steps] = t;
            rp.steps++;
            rp.last = nr;
            // rotate: u_pp <- u_prev <- u <- u_try (u is the caller's buffer: copies, three n_rows vectors per accepted step)
            FEM_CUDA(cudaMemcpyAsync(u_pp, u_prev, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
            FEM_CUDA(cudaMemcpyAsync(u_prev, u, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
            FEM_CUDA(cudaMemcpyAsync(u, u_try, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
            double *tmp = h_a; h_a = h_b; h_b = tmp;
            dt_pp = dt_prev; dt_prev = dt;
            if (nr.newton_iters <= o.grow_below) { dt *= o.grow; if (dt > o.dt_max) dt = o.dt_max; }
            rc = FEM_OK;
        } else {   // failed increment, a linear solve that gave up, or physics trouble at the converged state: cut back
            rp.rejected++;
            if (nr.physics_trouble) rp.rejected_physics++;
            dt *= o.cut;
            if (dt < o.dt_min) { rc = FEM_ERR_NOCONV; break; }
            rc = FEM_OK;
        }
    }
    rp.t_reached = t;
    if (h_a != hist) FEM_CUDA(cudaMemcpyAsync(hist, h_a, hb, cudaMemcpyDeviceToDevice, st));   // the history of the last accepted state
    FEM_CUDA(cudaStreamSynchronize(st));
    if (rep) *rep = rp;
    return rc;
}

// One step of the backward sweep of Alg. 1: right-hand side of Eq.(51) :366, adjoint solve on the tangent
// of the converged state (K_ff is symmetric for the standard element, so the row-eliminated K serves for K^T with lam = 0 on the
// constrained DOFs), then the products of Eq.(49) :355 and the history cotangent for the step before (reading G17).
// K^T on the same (structurally symmetric) pattern: one thread per 3x3 node-pair block (n, m); the position of n in the sorted
// neighbour list of m by binary search.  CSR row 3n+i starts at 9 nb_ptr[n] + 3 i len_n, block column pos at + 3 pos.
__global__ void k_transpose_vals(long long n_nodes, const int *__restrict__ nb_ptr, const int *__restrict__ nb,
                                 const double *__restrict__ vals, double *__restrict__ valsT) {
    const long long n = blockIdx.x * (long long)(blockDim.x >> 5) + (threadIdx.x >> 5);
    if (n >= n_nodes) return;
    const int lane = threadIdx.x & 31, o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    for (int pos = lane; pos < len; pos += 32) {
        const int m = nb[o + pos], om = nb_ptr[m], lm = nb_ptr[m + 1] - om;
        int lo = 0, hi = lm - 1;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (nb[om + mid] < (int)n) lo = mid + 1; else hi = mid; }
        const double *src = vals + 9LL * om + 3 * lo;     // block (m, n): entry (k, i) at src[k * 3 * lm + i]
        double *dst = valsT + 9LL * o + 3 * pos;          // block (n, m) of K^T: entry (i, k) = K[(m,k)][(n,i)]
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int k = 0; k < 3; k++) dst[(long long)i * 3 * len + k] = src[(long long)k * 3 * lm + i];
    }
}

__global__ void k_adj_rhs(long long n, const double *__restrict__ dJdu, const double *__restrict__ gu, double *__restrict__ rhs) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        rhs[i] = -((dJdu ? dJdu[i] : 0.0) + (gu ? gu[i] : 0.0));
}

extern "C" int fem_adjoint_step(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                                long long n_bc, const int *bc_dofs, const double *dJdu, const double *mu_in, double *lam,
                                double *mu_out, double *g_mat, double lin_rtol, int lin_max_iter, int *lin_iters,
                                void *cuda_stream) {
    if (!c || !u || !hist_in || !mat || !lam || !mu_out || !g_mat || (n_bc > 0 && !bc_dofs)) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (n_mat != 1 && n_mat != c->n_elems) return FEM_ERR_MAT;
    if (n_bc < 0 || !(lin_rtol > 0.0) || lin_max_iter < 1) return FEM_ERR_ARG;
    {
        const size_t hb = sizeof(double) * 56 * (size_t)c->n_elems;
        if (fem_ranges_overlap(mu_out, hist_in, hb) || (mu_in && fem_ranges_overlap(mu_out, mu_in, hb))) return FEM_ERR_ALIAS;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = ensure_solver_ws(c, true);
    if (rc != FEM_OK) return rc;
    if ((rc = check_dofs(c, n_bc, bc_dofs, st)) != FEM_OK) return rc;
    const long long n = c->n_rows;
    double *R = c->d_nw, *rhs = R + n, *gu = rhs + n, *vals = c->d_nw_vals;
    // tangent at the converged state; mu_out serves as the (unused) hist_out of this evaluation before it is overwritten below
    if ((rc = fem_launch_assemble(c, u, hist_in, mat, n_mat, R, vals, mu_out, st)) != FEM_OK) return rc;
    if (mu_in) {   // (dR^{n+1}/du^n)^T lam^{n+1} = (dhist_out/du)^T mu_in
        if ((rc = fem_assemble_vjp(c, u, hist_in, mat, n_mat, nullptr, mu_in, gu, nullptr, nullptr, cuda_stream)) != FEM_OK) return rc;
    }
    k_adj_rhs<<<RED_CTAS, RED_THREADS, 0, st>>>(n, dJdu, mu_in ? gu : nullptr, rhs);
    if (c->opt.fbar) {   // unsymmetric tangent: the adjoint system needs K^T explicitly
        if (!c->d_nw_valsT) FEM_CUDA(cudaMalloc(&c->d_nw_valsT, sizeof(double) * (size_t)c->nnz));
        k_transpose_vals<<<nblk3(c->n_nodes, 8), 256, 0, st>>>(c->n_nodes, c->d_nb_ptr, c->d_nb, vals, c->d_nw_valsT);
        FEM_CUDA(cudaGetLastError());
        vals = c->d_nw_valsT;
    }
    if ((rc = apply_dirichlet(c, n_bc, bc_dofs, nullptr, nullptr, nullptr, vals, rhs, st)) != FEM_OK) return rc;
    FEM_CUDA(cudaMemsetAsync(lam, 0, sizeof(double) * n, st));
    int its = 0, its2 = 0;
    rc = c->opt.fbar ? FEM_ERR_NOCONV : pcg(c, vals, rhs, lam, lin_rtol, lin_max_iter, &its, nullptr, st);
    if (rc == FEM_ERR_NOCONV) {   // F-bar, or K_ff not positive definite at this state: BiCGSTAB from zero
        FEM_CUDA(cudaMemsetAsync(lam, 0, sizeof(double) * n, st));
        rc = bicgstab(c, vals, rhs, lam, lin_rtol, lin_max_iter, &its2, nullptr, st);
    }
    if (lin_iters) *lin_iters = its + its2;
    if (rc != FEM_OK) return rc;
    return fem_assemble_vjp(c, u, hist_in, mat, n_mat, lam, mu_in, nullptr, mu_out, g_mat, cuda_stream);
}
