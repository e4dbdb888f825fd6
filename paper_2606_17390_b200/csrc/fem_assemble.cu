// fem_assemble: the hot path as three kernels on one stream
//   k_mat_prep  : per material record -> derived record (Lame constants, Hill eigen-system, orientation)
//   k_element   : 8 threads per element (one per Gauss point), 4 elements per warp, 16 per CTA.
//                 phase 1 (per point): shape gradients, F, C = F^T F, spectral decomposition, Hencky strain,
//                   Hill-48 return map as ONE scalar equation, algorithmic tangent as diagonal + rank-1,
//                   geometric post-processor in the eigenbasis of C, A^ = dP/dF in mixed axes -> shared memory;
//                   R^e by a shuffle butterfly over the element's 8 lanes
//                 phase 2 (whole warp per element): K^e = sum_q G^ A^ G^ on the FP64 tensor-core path
//                   (mma.sync.m8n8k4.f64, one 8x8 node matrix per component pair), F-bar rank-1 terms likewise
//                 phase 3: the accumulators go straight to the destination-major scratch (one 72-double record per
//                   (element, local node) in the node-sorted incidence order); only the coloured mode stages K^e
//   k_gather_fast / k_gather : one warp per node: copies the node's contiguous run of records to shared memory and sums the
//                 <= 8 contributions of each 3x3 node-pair block in ascending element id (fixed order, no atomics)
//                 into the CSR values and the residual.
// All formulas are derived by hand from PAPER.md (equation numbers at each step); nothing here is shared with oracle/.
#include "fem_internal.h"
#include "fem_device.cuh"
#include <math.h>
#include <stdio.h>
#include <mutex>

#define W23 0.81649658092772603273   // W = sqrt(2/3)
#define SQRT2 1.41421356237309504880
#define RSQRT2 0.70710678118654752440

// ------------------------------------------------------------------------------------------------ material pre-pass
// mat record (fem.h): E,nu,r11,r22,r33,r12,r23,r13,law,h0,h1,h2,q0..q3.
// Derived record (FEM_MATD doubles):
//   [0] 2mu  [1] lambda  [2] bulk modulus  [3] law  [4..6] h0,h1,h2
//   [7..11]  h_k : the five non-zero eigenvalues of the Hill tensor H (Mandel form), Eq.(A2)-(A5) PAPER.md:779-801
//   [12..14] v1, [15..17] v2 : eigenvectors of the normal 3x3 block of H in the deviatoric plane (unit, sum = 0);
//            eigenvectors 3..5 are the pure shears 12, 23, 13 with h = p7, p8, p9
//   [18..26] Theta row-major (columns = material axes in the global frame, Eq.(A1) :774) ; [27] 1 if Theta != I
// With isotropic elasticity (Eq.(8) :110) E:H = 2mu H, so in this eigenbasis the return map is diagonal.
__device__ __forceinline__ void mat_prep_record(const double *p, double *o) {
    double E = p[0], nu = p[1];
    double mu2 = E / (1.0 + nu), lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu));
    o[0] = mu2; o[1] = lam; o[2] = lam + mu2 / 3.0; o[3] = p[8]; o[4] = p[9]; o[5] = p[10]; o[6] = p[11];
    double p1 = 2.0 / (3.0 * p[2] * p[2]), p2 = 2.0 / (3.0 * p[3] * p[3]), p3 = 2.0 / (3.0 * p[4] * p[4]);
    double p7 = 1.0 / (p[5] * p[5]), p8 = 1.0 / (p[6] * p[6]), p9 = 1.0 / (p[7] * p[7]);
    double p4 = 0.5 * (p3 - p1 - p2), p5 = 0.5 * (p1 - p2 - p3), p6 = 0.5 * (p2 - p1 - p3);
    // normal block N3 = [[p1,p4,p6],[p4,p2,p5],[p6,p5,p3]] has null vector (1,1,1); project on d1=(1,-1,0)/sqrt2, d2=(1,1,-2)/sqrt6
    const double d1[3] = {RSQRT2, -RSQRT2, 0.0};
    const double d2[3] = {0.40824829046386301637, 0.40824829046386301637, -0.81649658092772603273};
    const double N3[3][3] = {{p1, p4, p6}, {p4, p2, p5}, {p6, p5, p3}};
    double m11 = 0, m22 = 0, m12 = 0;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            m11 += d1[i] * N3[i][j] * d1[j]; m22 += d2[i] * N3[i][j] * d2[j]; m12 += d1[i] * N3[i][j] * d2[j];
        }
    double c = 1.0, s = 0.0, e1 = m11, e2 = m22;
    if (m12 != 0.0) {
        double d = m22 - m11, r = sqrt(d * d + 4.0 * m12 * m12);
        double t = 2.0 * m12 / (d + copysign(r, d));
        c = 1.0 / sqrt(1.0 + t * t); s = t * c;
        e1 = m11 - t * m12; e2 = m22 + t * m12;
    }
    o[7] = e1; o[8] = e2; o[9] = p7; o[10] = p8; o[11] = p9;
    for (int i = 0; i < 3; i++) { o[12 + i] = c * d1[i] - s * d2[i]; o[15 + i] = s * d1[i] + c * d2[i]; }
    double qn = sqrt(p[12] * p[12] + p[13] * p[13] + p[14] * p[14] + p[15] * p[15]);
    double w = p[12] / qn, x = p[13] / qn, y = p[14] / qn, z = p[15] / qn;
    o[18] = 1 - 2 * (y * y + z * z); o[19] = 2 * (x * y - w * z);     o[20] = 2 * (x * z + w * y);
    o[21] = 2 * (x * y + w * z);     o[22] = 1 - 2 * (x * x + z * z); o[23] = 2 * (y * z - w * x);
    o[24] = 2 * (x * z - w * y);     o[25] = 2 * (y * z + w * x);     o[26] = 1 - 2 * (x * x + y * y);
    o[27] = (x == 0.0 && y == 0.0 && z == 0.0) ? 0.0 : 1.0;
    for (int i = 28; i < FEM_MATD; i++) o[i] = 0.0;
}

// One thread per record; the records of a CTA go through shared memory so that the global loads and stores are coalesced
// (per-element records, config 4: 700k x (128 B in, 256 B out); strided per-thread accesses took 0.20 ms).
#define MP_THREADS 64
__global__ void __launch_bounds__(MP_THREADS) k_mat_prep(long long n_mat, const double *__restrict__ mat, double *__restrict__ md) {
    __shared__ double sin_[MP_THREADS * (FEM_NPAR + 1)];     // +1: records start in different banks
    __shared__ double sout[MP_THREADS * (FEM_MATD + 1)];
    const long long m0 = (long long)blockIdx.x * MP_THREADS;
    const int cnt = (int)min((long long)MP_THREADS, n_mat - m0), t = threadIdx.x;
    for (int i = t; i < cnt * FEM_NPAR; i += MP_THREADS) sin_[(i / FEM_NPAR) * (FEM_NPAR + 1) + i % FEM_NPAR] = mat[m0 * FEM_NPAR + i];
    __syncthreads();
    if (t < cnt) mat_prep_record(sin_ + t * (FEM_NPAR + 1), sout + t * (FEM_MATD + 1));
    __syncthreads();
    for (int i = t; i < cnt * FEM_MATD; i += MP_THREADS) md[m0 * FEM_MATD + i] = sout[(i / FEM_MATD) * (FEM_MATD + 1) + i % FEM_MATD];
}

// ------------------------------------------------------------------------------------------------ small device helpers
// atanh(w)/w : first divided difference kernel of ln,  ln(b/a) = 2 atanh((b-a)/(b+a)).
__device__ __forceinline__ double atanhc(double w, double dlog /* = ln b - ln a */) {
    // branch-free (both forms are evaluated, one is selected) so that the calls of a thread interleave:
    // |w| < 0.15 : series 1 + w^2/3 + w^4/5 + ...  (11 terms, remainder < 1e-19), else ln(b/a) / (2 w)
    const double w2 = w * w;
    const double s = atanh_poly(w2);
    const double big = 0.5 * dlog * frcp(w);   // NaN for w = 0, never selected then
    return (w2 < 0.0225) ? s : big;
}

// Second divided difference g[a,b,c] of g = 1/2 ln for three eigenvalues within 1e-4 (relative) of each other:
// Taylor series about the mean m, g[a,b,c] = 1/(2 m^2) sum_{n>=2} (-1)^(n+1)/n h_{n-2}(x), x_i = (l_i - m)/m,
// h_k = complete homogeneous polynomial; |x| <= 1e-4 => the n = 5 term is already < 1e-13 of the leading one.
// Farther apart the recursion on the widest gap is used (error 4 eps l/gap <= 1e-11 of g2, which enters C_L with
// weight |T|/|C_ep| ~ 1e-2).
__device__ __forceinline__ double dd2_series(double la, double lb, double lc) {
    const double m = (la + lb + lc) * (1.0 / 3.0), im = frcp(m);
    const double xa = (la - m) * im, xb = (lb - m) * im, xc = (lc - m) * im;
    const double h1 = xa + xb + xc;                                   // = 0 up to rounding
    const double h2 = xa * xa + xb * xb + xc * xc + xa * xb + xb * xc + xa * xc;
    return 0.5 * im * im * (-0.5 + (1.0 / 3.0) * h1 - 0.25 * h2);
}

// ------------------------------------------------------------------------------------------------ element kernel
// Voigt pair index of tensor components (11,22,33,12,23,13)
__device__ constexpr int VG[3][3] = {{0, 3, 5}, {3, 1, 4}, {5, 4, 2}};
__host__ __device__ constexpr int sidx9(int r, int c) {  // packed upper triangle of a symmetric 9x9
    return (r <= c) ? (r * 9 - r * (r - 1) / 2 + (c - r)) : (c * 9 - c * (c - 1) / 2 + (r - c));
}

// shared-memory layout per element, in doubles (stride = 4 mod 16 so that broadcast reads of the 4 elements of a warp
// hit 4 disjoint bank groups; every per-point array is [entry][q] with the 8 Gauss points adjacent)
#define SM_GG 0     // G^_Ia = grad N_I in the eigenbasis of C at GGX(I,a) + q: node stride 25 (odd) so that both the per-point
                    // accesses (lanes = q) and the per-node reads of phase 2 (lanes = I) are bank-conflict free
#define GGX(I, a) (SM_GG + (I) * 25 + (a) * 8)
#define SM_AA 200   // 45 entries w * A^_(ia)(kb), packed symmetric: entry s < 44 at (s/2)*16 + 2 q + (s&1), entry 44 at 352 + q
#define SM_XE 200   // [24] element coordinates   (overlay: dead before AA is written)
#define SM_UE 224   // [24] element displacements (overlay)
#define SM_GQ 576   // [24][8]  (F-bar) g^q_Kk = G_KL F^-1_Lk
#define SM_YY 768   // [9][8]   (F-bar) w/3 (A^:F^)_ia
#define SM_GB 840   // [24]     (F-bar) gbar
#define SM_WQ 864   // [8]      (F-bar) w_q J_q / (Jbar V)
#define ES_STD 564   // >= 560, = 4 mod 16: the 4 elements of a warp start in 4 different bank groups
#define ES_FBAR 884  // >= 872, = 4 mod 16
#ifndef JAC_SWEEPS
#define JAC_SWEEPS 4
#endif
#ifndef EL_PER_CTA
#define EL_PER_CTA 16
#endif
#define CTA_THREADS (8 * EL_PER_CTA)
#ifndef THREADS_PER_SM
#define THREADS_PER_SM 384
#endif
#define CTAS_STD (THREADS_PER_SM / CTA_THREADS)   // 12 warps per SM: limited by 168 registers and ~4.5 KB shared memory per element
#define CTAS_FBAR (256 / CTA_THREADS)
#ifndef CTAS_YLD
#define CTAS_YLD CTAS_FBAR
#endif

__device__ __forceinline__ void flow_stress(double law, double h0, double h1, double h2, double alpha, double &sf,
                                            double &dsf) {
    if (law == 0.0) {  // Voce, Eq.(10) PAPER.md:121 (flow stress part; the sqrt(2/3) is applied by the caller, G2)
        double ex = fexp(-h2 * alpha);
        sf = fma(h1, 1.0 - ex, h0);
        dsf = h1 * h2 * ex;
    } else {           // Swift K (eps0 + alpha)^n (BASELINE.json configs)
        double b = h1 + alpha;
        sf = h0 * fexp(h2 * flog(b));
        dsf = h2 * sf * frcp(b);
    }
}

#ifndef BAR_PARK
#define BAR_PARK 1
#endif
#include "fem_barlat.cuh"

// ------------------------------------------------------------------------------------------------ node gather (S14), shared
// by the stand-alone gather kernels and by the gather CTAs of the fused mode.
// The scratch is destination-major: node n's contributions are the records inc_ptr[n] .. inc_ptr[n+1]-1 (72 doubles each:
// block row I of K^e of incident entry s = (e,I), ascending element id), one contiguous run.
__device__ __forceinline__ int ksoff(int K, int c) { return c * 8 + K; }
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
}
// L2 residency hints of the fused kernel: the scratch records are written once and read back once, ~one wave of CTAs
// later, so they are stored with an evict-last policy and read with evict-first; everything that streams (history, CSR
// values) is marked evict-first, so that it does not push the records out of the 126 MB L2 before they are consumed.
__device__ __forceinline__ unsigned long long l2_policy_last() {
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_first() {
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_hint(double *ptr, double a, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(ptr), "d"(a), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint2(double *ptr, double a, double b, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(ptr), "d"(a), "d"(b), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async16_hint(void *smem_dst, const void *gsrc, unsigned long long pol) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(sa), "l"(gsrc), "l"(pol) : "memory");
}
// K = A K^e, R = A R^e (Eq.(34) :253, Eq.(38) :274) for one node whose run of records sits in shared memory (buf).
// kvec[block] (built at setup) holds, for each incident entry s, the local node K of the block's column node (nibble s;
// 0xF = that element does not contain it), so lane = neighbour position adds <= 8 blocks in ascending s (fixed order, no
// atomics) with nine conflict-free shared loads per block.
__device__ __forceinline__ void gather_reduce_write(long long n, int b, int m, const double *buf, int lane,
                                                    const int *__restrict__ nb_ptr, const unsigned int *__restrict__ kvec,
                                                    const double *Re, double *__restrict__ csr_vals, double *__restrict__ residual) {
    const int o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    double rv = 0.0;
    if (lane < 3 * m) rv = __ldcg(Re + (long long)b * 3 + lane);
    for (int pos0 = 0; pos0 < len; pos0 += 32) {
        const int pos = pos0 + lane;
        const unsigned kv = (pos < len) ? kvec[o + pos] : 0xffffffffu;
        double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int s = 0; s < 8; s++) {
            if (s < m) {   // warp-uniform
                const unsigned K = (kv >> (4 * s)) & 15u;
                if (K != 15u) {
                    const double *rec = buf + s * 72 + K;   // [c][K]: the lanes of one incident entry read 8 adjacent doubles
#pragma unroll
                    for (int j = 0; j < 9; j++) acc[j] += rec[8 * j];
                }
            }
        }
        if (pos < len) {
            double *out = csr_vals + 9LL * o + 3 * pos;
#pragma unroll
            for (int i = 0; i < 3; i++) {
                out[(long long)i * 3 * len + 0] = acc[3 * i + 0];
                out[(long long)i * 3 * len + 1] = acc[3 * i + 1];
                out[(long long)i * 3 * len + 2] = acc[3 * i + 2];
            }
        }
    }
    {   // residual: lane 3 s + i holds R^e component i of incident entry s; lanes 0..2 add in ascending s
        double r = 0.0;
        for (int j = 0; j < m; j++) r += __shfl_sync(0xffffffffu, rv, (3 * j + lane) & 31);
        if (lane < 3) residual[3 * n + lane] = r;
    }
}
// One warp gathers up to NB nodes (lane j < cnt holds node id nd): asynchronous 16-byte copies of the runs into the
// warp's shared-memory buffer (NB x 576 doubles) are all in flight before the first reduction starts.
template <int NB>
__device__ __forceinline__ void gather_warp_nodes(int nd, int cnt, double *wbuf, int lane, const int *__restrict__ inc_ptr,
                                                  const int *__restrict__ nb_ptr, const unsigned int *__restrict__ kvec,
                                                  const double *Ke, const double *Re, double *__restrict__ csr_vals,
                                                  double *__restrict__ residual) {
    int b = 0, m = 0;
    if (lane < cnt) { b = inc_ptr[nd]; m = inc_ptr[nd + 1] - b; }
#pragma unroll
    for (int j = 0; j < NB; j++) {
        const int bj = __shfl_sync(0xffffffffu, b, j), lim = 36 * __shfl_sync(0xffffffffu, m, j);
        const double *src = Ke + (long long)bj * 72;
#pragma unroll
        for (int it = 0; it < 9; it++) {
            const int idx = it * 32 + lane;
            if (idx < lim) cp_async16(wbuf + j * 576 + 2 * idx, src + 2 * idx);
        }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
#pragma unroll 1
    for (int j = 0; j < cnt; j++)
        gather_reduce_write(__shfl_sync(0xffffffffu, nd, j), __shfl_sync(0xffffffffu, b, j), __shfl_sync(0xffffffffu, m, j),
                            wbuf + j * 576, lane, nb_ptr, kvec, Re, csr_vals, residual);
    __syncwarp();
}
// Keeping the warps of a CTA in the same code region lets them share instruction-cache lines (the kernel is ~94 KB of
// straight-line SASS); ncu showed instruction fetch as a top stall without it.
#ifndef PS_MASK
#define PS_MASK 0x010   // measured best subset of the ten phase boundaries (sweeps in DESIGN.md): one barrier, before the tangent
#endif
// barrier over the element warps of the CTA: the whole CTA, or (fused kernel) named barrier 1 over the element warpgroup
template <int FUSE> __device__ __forceinline__ void el_sync() {
    if (FUSE) asm volatile("bar.sync 1, 128;" ::: "memory");
    else __syncthreads();
}
#define PHASE_SYNC_N(n) do { if ((PS_MASK >> (n)) & 1) el_sync<FUSE>(); } while (0)
// Launch-time arguments of the assembly side of k_element.
// Fused, lagged gather (FUSE = 1): the scratch is consumed while it is still in L2, by warps that cost the element warps
// almost nothing.  The CTA has two warpgroups: warps 0-3 evaluate the chunk's 16 elements exactly as in the unfused
// kernel, warps 4-7 gather.  Measured: the element kernel loses only 9 % when it runs 2 CTAs per SM with 208 registers
// instead of 3 with 168, which frees a third of the shared memory; `setmaxnreg` moves the
// gather warps' registers to the element warps (2 CTAs x (128 x 208 + 128 x 48) = the whole register file).
// The nodes are cut into quads of four consecutive ids; at setup every quad is given to one gather warp of a chunk
// launched at least FUSE lag chunks (one wave of resident CTAs) after the last chunk that writes one of its records.
// CTAs are dispatched in index order, so those chunks are resident or retired: each chunk publishes a completion flag
// (threadfence + flag = epoch of this call); a gather warp polls the flags of its quad's chunks for a BOUNDED time (the
// chunks it waits for never wait for anything), and a quad that still is not ready (or is scheduled past the last
// chunk) goes to a short list that k_gather_list finishes after the element kernel.  Which warp sums a node never
// changes the order of the sum, so results are bit-identical to the unfused path.
#define FUSE_DEPW 16    // ints per quad dependency record: [0] = number of chunks (<= 15), [1..] chunk ids
#define FUSE_QPC 8      // quads a CTA can be given (two per gather warp)
#define FUSE_EREGS 208   // registers per thread of the element warpgroup / the gather warpgroup after setmaxnreg
#define FUSE_GREGS 48
#define FUSE_GNB 2       // nodes a gather warp holds in shared memory at a time (2 x 4608 B)
#ifndef FUSE_DISCARD
#define FUSE_DISCARD 1
#endif
#define FUSE_POLLS 96   // bounded wait of a gather warp for its quad's chunks: polls of ~0.25 us
struct scatter_args {
    const int *elist;   // element ids in processing order (the locality order built at setup for shuffled meshes); nullptr = identity
    const int *eslot;   // [e*8+I] -> scratch record of block row I (node-sorted incidence index)
    // fused gather
    const int *cta_quads;          // [n_chunks*FUSE_QPC] quad ids given to the warps of chunk c (warp w: entries 2w, 2w+1), -1 = none
    const int *quad_deps;          // [n_quads*FUSE_DEPW]
    unsigned int *chunk_flag;      // [n_chunks] epoch of the last call in which the chunk's records were complete
    unsigned int epoch;
    int *left_list;                // quads that were not ready when their warp looked
    unsigned int *left_count;
    long long n_nodes;
    const int *inc_ptr, *nb_ptr;
    const unsigned int *kvec;
    double *csr_vals, *residual;
};
#ifndef EL_PF_DIST
#define EL_PF_DIST 444   // L2 prefetch distance in chunks (one wave of CTAs): 3.135 -> 3.108 ms; 888 and 1776 gain nothing
#endif
// YLD 0: Hill-48 (scalar return map); YLD 1: Barlat Yld2004-18p (fem_barlat.cuh), bard = derived Barlat records
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

// The reduction of gather_reduce_write for a node with at most 8 incident elements (hence at most 27 <= 32 neighbours),
// with every table value already in registers: kv = kvec entry of this lane's neighbour position, rv = R^e value of
// lane 3 s + i.  Same sums in the same order.
__device__ __forceinline__ void gather_reduce_pre(long long n, int m, int o, int len, unsigned kv, double rv, const double *buf,
                                                  const double *zero, int lane, double *__restrict__ csr_vals,
                                                  double *__restrict__ residual) {
    // branch-free and select-free: a missing block (nibble 0xF, also every s >= m) is read from `zero`, 65 doubles of +0.0
    // in shared memory; adding +0.0 leaves a sum that started at +0.0 unchanged bit for bit.  One address select per
    // record instead of a branch or nine value selects: the gather warps share issue slots with the element warps.
    double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
    for (int s = 0; s < 8; s++) {
        const unsigned K = (kv >> (4 * s)) & 15u;
        const double *rec = (K != 15u) ? buf + s * 72 + K : zero;
#pragma unroll
        for (int j = 0; j < 9; j++) acc[j] += rec[8 * j];
    }
    if (lane < len) {
        double *out = csr_vals + 9LL * o + 3 * lane;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            __stcs(out + (long long)i * 3 * len + 0, acc[3 * i + 0]);   // streaming stores: written once, not read by this call
            __stcs(out + (long long)i * 3 * len + 1, acc[3 * i + 1]);
            __stcs(out + (long long)i * 3 * len + 2, acc[3 * i + 2]);
        }
    }
    double r = 0.0;
    for (int j = 0; j < m; j++) r += __shfl_sync(0xffffffffu, rv, (3 * j + lane) & 31);
    if (lane < 3) residual[3 * n + lane] = r;
}

// The gather warpgroup of the fused kernel (warps 4-7 of the CTA; gw = warp index in the group).  A warp is given up to
// two quads = eight nodes; lane j holds the tables of node j (loaded once, before anything is known to be ready: they are
// static).  The nodes of the quads whose chunks have all published their flag are then streamed through a two-slot
// buffer: the records (and table values) of node i+1 are on their way while node i is reduced.
__device__ __forceinline__ void fuse_gather_role(long long chunk, int gw, int lane, double *wbuf, double *zero, const double *Ke,
                                                 const double *Re, const scatter_args &sa) {
    zero[lane] = 0.0; zero[32 + lane] = 0.0; if (lane == 0) zero[64] = 0.0;   // the block of +0.0 read in place of a missing block
    __syncwarp();
    const int q0 = __ldg(sa.cta_quads + chunk * FUSE_QPC + 2 * gw), q1 = __ldg(sa.cta_quads + chunk * FUSE_QPC + 2 * gw + 1);
    if ((q0 & q1) < 0 && q0 < 0 && q1 < 0) return;
    // lane j < 8: node j of the two quads
    const int myq = (lane < 4) ? q0 : q1;
    long long node = -1;
    if (lane < 8 && myq >= 0) { node = 4LL * myq + (lane & 3); if (node >= sa.n_nodes) node = -1; }
    int b = 0, m = 0, o = 0, len = 0;
    if (node >= 0) {
        b = __ldg(sa.inc_ptr + node); m = __ldg(sa.inc_ptr + node + 1) - b;
        o = __ldg(sa.nb_ptr + node); len = __ldg(sa.nb_ptr + node + 1) - o;
    }
    // readiness of the two quads: bounded polling of their chunks' flags (lanes 0-15: quad 0, lanes 16-31: quad 1)
    unsigned live = 0;   // bit j: node j is to be gathered by this warp
    {
        const int qq = (lane < 16) ? q0 : q1, dl = lane & 15;
        int nd = 0;
        const volatile unsigned int *fl = sa.chunk_flag;
        if (qq >= 0) {
            const int *dep = sa.quad_deps + (long long)qq * FUSE_DEPW;
            nd = __ldg(dep);
            if (dl < nd) fl = sa.chunk_flag + __ldg(dep + 1 + dl);
        }
        unsigned okm = 0;
#pragma unroll 1
        for (int poll = 0; poll < FUSE_POLLS; poll++) {
            const bool ok = (dl < nd) ? (*fl == sa.epoch) : true;
            okm = __ballot_sync(0xffffffffu, ok);
            if (okm == 0xffffffffu) break;
            __nanosleep(250);
        }
        const bool r0 = (q0 >= 0) && ((okm & 0xffffu) == 0xffffu), r1 = (q1 >= 0) && ((okm >> 16) == 0xffffu);
        if (lane == 0 && q0 >= 0 && !r0) sa.left_list[atomicAdd(sa.left_count, 1u)] = q0;
        if (lane == 0 && q1 >= 0 && !r1) sa.left_list[atomicAdd(sa.left_count, 1u)] = q1;
        live = __ballot_sync(0xffffffffu, node >= 0 && ((lane < 4) ? r0 : r1)) & 0xffu;
    }
    if (!live) return;
    __threadfence();                         // the flags were read before any record is
    const unsigned long long pol_f = l2_policy_first();
    // stream the live nodes through the two slots
    int cur = __ffs(live) - 1;
    live &= live - 1;
    unsigned kv_c = 0xffffffffu, kv_n = 0xffffffffu;
    double rv_c = 0.0, rv_n = 0.0;
    int slot = 0;
    {   // prologue: node `cur` -> slot 0
        const int bj = __shfl_sync(0xffffffffu, b, cur), mj = __shfl_sync(0xffffffffu, m, cur), oj = __shfl_sync(0xffffffffu, o, cur),
                  lj = __shfl_sync(0xffffffffu, len, cur);
        const double *src = Ke + (long long)bj * 72;
#pragma unroll
        for (int it = 0; it < 9; it++) { const int idx = it * 32 + lane; if (idx < 36 * mj) cp_async16_hint(wbuf + 2 * idx, src + 2 * idx, pol_f); }
        asm volatile("cp.async.commit_group;" ::: "memory");
        kv_c = (lane < lj) ? __ldg(sa.kvec + oj + lane) : 0xffffffffu;
        rv_c = (lane < 3 * mj) ? __ldcg(Re + (long long)bj * 3 + lane) : 0.0;
    }
#pragma unroll 1
    while (cur >= 0) {
        const int nxt = live ? __ffs(live) - 1 : -1;
        live &= live - 1;
        if (nxt >= 0) {   // records and table values of the next node -> the other slot
            const int bj = __shfl_sync(0xffffffffu, b, nxt), mj = __shfl_sync(0xffffffffu, m, nxt), oj = __shfl_sync(0xffffffffu, o, nxt),
                      lj = __shfl_sync(0xffffffffu, len, nxt);
            const double *src = Ke + (long long)bj * 72;
            double *dst = wbuf + (slot ^ 1) * 576;
#pragma unroll
            for (int it = 0; it < 9; it++) { const int idx = it * 32 + lane; if (idx < 36 * mj) cp_async16_hint(dst + 2 * idx, src + 2 * idx, pol_f); }
            kv_n = (lane < lj) ? __ldg(sa.kvec + oj + lane) : 0xffffffffu;
            rv_n = (lane < 3 * mj) ? __ldcg(Re + (long long)bj * 3 + lane) : 0.0;
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 1;" ::: "memory");     // everything but the newest group: the current node is in
        __syncwarp();
        const long long n = __shfl_sync(0xffffffffu, node, cur);
        gather_reduce_pre(n, __shfl_sync(0xffffffffu, m, cur), __shfl_sync(0xffffffffu, o, cur), __shfl_sync(0xffffffffu, len, cur),
                          kv_c, rv_c, wbuf + slot * 576, zero, lane, sa.csr_vals, sa.residual);
        __syncwarp();                        // the slot is free for the node after next
#if FUSE_DISCARD
        {   // the records of this node have been consumed and are never read again in this call: drop their (dirty) L2 lines
            // instead of letting them be written back to HBM.  Only 128-byte lines that lie wholly inside the node's run.
            const unsigned long long a0 = (unsigned long long)(Ke + (long long)__shfl_sync(0xffffffffu, b, cur) * 72);
            const unsigned long long a1 = a0 + 576ull * (unsigned long long)__shfl_sync(0xffffffffu, m, cur);
            for (unsigned long long pl = ((a0 + 127ull) & ~127ull) + 128ull * lane; pl + 128ull <= a1; pl += 32ull * 128ull)
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(pl) : "memory");
        }
#endif
        cur = nxt; kv_c = kv_n; rv_c = rv_n; slot ^= 1;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

template <int FBAR, int FUSE, int YLD = 0>
__global__ void __launch_bounds__(FUSE ? 2 * CTA_THREADS : CTA_THREADS, FUSE ? 2 : (YLD ? CTAS_YLD : (FBAR ? CTAS_FBAR : CTAS_STD)))
k_element(long long n_elems, const double *__restrict__ coords, const int *__restrict__ conn,
          const double *__restrict__ u, const double *__restrict__ hist_in, const double *__restrict__ matd,
          int mat_stride, double tol, int kmax, double *__restrict__ Ke, double *__restrict__ Re,
          double *__restrict__ hist_out, unsigned long long *__restrict__ stats, const scatter_args sa,
          const double *__restrict__ bard = nullptr, int bar_stride = 0) {
    extern __shared__ __align__(16) double sm[];
    __shared__ unsigned int s_hist[64];
    __shared__ unsigned int s_done;
    constexpr int ES = FBAR ? ES_FBAR : ES_STD;
    const int tid = threadIdx.x, lane = tid & 31, q = lane & 7;
    const long long chunk = blockIdx.x;
    if (FUSE) {
        if (tid >= CTA_THREADS) {   // gather warpgroup: hands most of its registers to the element warpgroup
            reg_dec<FUSE_GREGS>();
            const int gw = (tid - CTA_THREADS) >> 5;
            fuse_gather_role(chunk, gw, lane, sm + EL_PER_CTA * ES + gw * FUSE_GNB * 576, sm + EL_PER_CTA * ES + 4 * FUSE_GNB * 576 + gw * 66,
                             Ke, Re, sa);
            return;
        }
        reg_inc<FUSE_EREGS>();
    }
    const unsigned long long pol_keep = FUSE ? l2_policy_last() : 0ull;
    const int el_cta = tid >> 3;
    double *se = sm + el_cta * ES;
    const long long e_raw = chunk * EL_PER_CTA + el_cta;
    const bool valid = e_raw < n_elems;
    const long long e_slot = valid ? e_raw : n_elems - 1;
    const long long e = sa.elist ? (long long)sa.elist[e_slot] : e_slot;
    // ---- S2 gather: thread q loads node q of its element and the history of its Gauss point
    const int my_node = conn[e * 8 + q];
    const int my_slot = __ldg(sa.eslot + e * 8 + q);
    double epn[6], xn[3], un[3];
    {
        const double *hin = hist_in + (e * 8 + q) * 7;
#pragma unroll
        for (int i = 0; i < 6; i++) epn[i] = __ldg(hin + i);
    }
    const double alphan = __ldg(hist_in + (e * 8 + q) * 7 + 6);
#pragma unroll
    for (int i = 0; i < 3; i++) { xn[i] = coords[3 * (long long)my_node + i]; un[i] = u[3 * (long long)my_node + i]; }
#if EL_PF_DIST > 0
    {   // streaming inputs of the chunk EL_PF_DIST launches ahead -> L2 (they are read exactly once)
        const long long ep = (chunk + EL_PF_DIST) * EL_PER_CTA + el_cta;
        if (ep < n_elems && !sa.elist) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(conn + ep * 8 + q));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(sa.eslot + ep * 8 + q));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(hist_in + (ep * 8 + q) * 7));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(hist_in + (ep * 8 + q) * 7 + 6));
        }
    }
#endif
    for (int j = tid; j < 64; j += CTA_THREADS) s_hist[j] = 0;
    if (tid == 0) s_done = 0;
    el_sync<FUSE>();
  {
#pragma unroll
    for (int i = 0; i < 3; i++) { se[SM_XE + 3 * q + i] = xn[i]; se[SM_UE + 3 * q + i] = un[i]; }
    __syncwarp();

    // ---- S1 shape gradients at this Gauss point (O1): Jr = sum X_I (x) dN_I/dxi, G_I = dN_I/dxi Jr^-1, w = det Jr
    const double gp = 0.57735026918962576451;
    const double xq = (q & 1) ? gp : -gp, yq = (q & 2) ? gp : -gp, zq = (q & 4) ? gp : -gp;
    const double fxp = 1.0 + xq, fxm = 1.0 - xq, fyp = 1.0 + yq, fym = 1.0 - yq, fzp = 1.0 + zq, fzm = 1.0 - zq;
    double Jr[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
    for (int I = 0; I < 8; I++) {
        const bool px = ((I ^ (I >> 1)) & 1), py = (I & 2), pz = (I & 4);
        const double fx = px ? fxp : fxm, fy = py ? fyp : fym, fz = pz ? fzp : fzm;
        const double d0 = (px ? 0.125 : -0.125) * fy * fz, d1 = (py ? 0.125 : -0.125) * fx * fz,
                     d2 = (pz ? 0.125 : -0.125) * fx * fy;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            double X = se[SM_XE + 3 * I + i];
            Jr[i][0] = fma(X, d0, Jr[i][0]); Jr[i][1] = fma(X, d1, Jr[i][1]); Jr[i][2] = fma(X, d2, Jr[i][2]);
        }
    }
    double Ji[3][3];
    double wq;
    {
        double c00 = Jr[1][1] * Jr[2][2] - Jr[1][2] * Jr[2][1], c01 = Jr[1][2] * Jr[2][0] - Jr[1][0] * Jr[2][2],
               c02 = Jr[1][0] * Jr[2][1] - Jr[1][1] * Jr[2][0];
        wq = Jr[0][0] * c00 + Jr[0][1] * c01 + Jr[0][2] * c02;
        double id = frcp(wq);
        Ji[0][0] = c00 * id; Ji[1][0] = c01 * id; Ji[2][0] = c02 * id;
        Ji[0][1] = (Jr[0][2] * Jr[2][1] - Jr[0][1] * Jr[2][2]) * id;
        Ji[1][1] = (Jr[0][0] * Jr[2][2] - Jr[0][2] * Jr[2][0]) * id;
        Ji[2][1] = (Jr[0][1] * Jr[2][0] - Jr[0][0] * Jr[2][1]) * id;
        Ji[0][2] = (Jr[0][1] * Jr[1][2] - Jr[0][2] * Jr[1][1]) * id;
        Ji[1][2] = (Jr[0][2] * Jr[1][0] - Jr[0][0] * Jr[1][2]) * id;
        Ji[2][2] = (Jr[0][0] * Jr[1][1] - Jr[0][1] * Jr[1][0]) * id;
    }
    // ---- S3 kinematics: F = I + sum u_I (x) G_I  (Eq.(3), Eq.(30) :228); G kept in shared memory
    double F[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
#pragma unroll
    for (int I = 0; I < 8; I++) {
        const bool px = ((I ^ (I >> 1)) & 1), py = (I & 2), pz = (I & 4);
        const double fx = px ? fxp : fxm, fy = py ? fyp : fym, fz = pz ? fzp : fzm;
        const double d0 = (px ? 0.125 : -0.125) * fy * fz, d1 = (py ? 0.125 : -0.125) * fx * fz,
                     d2 = (pz ? 0.125 : -0.125) * fx * fy;
        double G[3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            G[j] = d0 * Ji[0][j] + d1 * Ji[1][j] + d2 * Ji[2][j];
            se[GGX(I, j) + q] = G[j];
        }
#pragma unroll
        for (int i = 0; i < 3; i++) {
            double ui = se[SM_UE + 3 * I + i];
            F[i][0] = fma(ui, G[0], F[i][0]); F[i][1] = fma(ui, G[1], F[i][1]); F[i][2] = fma(ui, G[2], F[i][2]);
        }
    }
    __syncwarp();  // XE/UE (overlaying AA) are dead from here on
    double detF = F[0][0] * (F[1][1] * F[2][2] - F[1][2] * F[2][1]) - F[0][1] * (F[1][0] * F[2][2] - F[1][2] * F[2][0]) +
                  F[0][2] * (F[1][0] * F[2][1] - F[1][1] * F[2][0]);
    double wgt = wq;  // integration weight of the tangent (w_q, times c_q with F-bar)
    if (FBAR) {
        // ---- S4 F-bar (Eq.(31)-(32) PAPER.md:237-243): Jbar = sum w J / sum w ; Fbar = (Jbar/J)^(1/3) F
        double Fi[3][3];
        double idt = frcp(detF);
        Fi[0][0] = (F[1][1] * F[2][2] - F[1][2] * F[2][1]) * idt; Fi[0][1] = (F[0][2] * F[2][1] - F[0][1] * F[2][2]) * idt;
        Fi[0][2] = (F[0][1] * F[1][2] - F[0][2] * F[1][1]) * idt; Fi[1][0] = (F[1][2] * F[2][0] - F[1][0] * F[2][2]) * idt;
        Fi[1][1] = (F[0][0] * F[2][2] - F[0][2] * F[2][0]) * idt; Fi[1][2] = (F[0][2] * F[1][0] - F[0][0] * F[1][2]) * idt;
        Fi[2][0] = (F[1][0] * F[2][1] - F[1][1] * F[2][0]) * idt; Fi[2][1] = (F[0][1] * F[2][0] - F[0][0] * F[2][1]) * idt;
        Fi[2][2] = (F[0][0] * F[1][1] - F[0][1] * F[1][0]) * idt;
#pragma unroll
        for (int K = 0; K < 8; K++) {
            double g0 = se[GGX(K, 0) + q], g1 = se[GGX(K, 1) + q], g2 = se[GGX(K, 2) + q];
#pragma unroll
            for (int k = 0; k < 3; k++) se[SM_GQ + (3 * K + k) * 8 + q] = g0 * Fi[0][k] + g1 * Fi[1][k] + g2 * Fi[2][k];
        }
        double V = wq, WJ = wq * detF;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) { V += __shfl_xor_sync(0xffffffffu, V, o); WJ += __shfl_xor_sync(0xffffffffu, WJ, o); }
        double Jbar = WJ * frcp(V);
        double cq = cbrt(Jbar * idt);
        se[SM_WQ + q] = wq * detF * frcp(WJ);
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) F[i][j] *= cq;
        wgt = wq * cq;
    }

    PHASE_SYNC_N(0);
    // ---- S5 C = F^T F and its spectral decomposition by cyclic Jacobi (Eq.(4) :92; backward stable, fixed 4 sweeps)
    double c00 = F[0][0] * F[0][0] + F[1][0] * F[1][0] + F[2][0] * F[2][0];
    double c11 = F[0][1] * F[0][1] + F[1][1] * F[1][1] + F[2][1] * F[2][1];
    double c22 = F[0][2] * F[0][2] + F[1][2] * F[1][2] + F[2][2] * F[2][2];
    double c01 = F[0][0] * F[0][1] + F[1][0] * F[1][1] + F[2][0] * F[2][1];
    double c12 = F[0][1] * F[0][2] + F[1][1] * F[1][2] + F[2][1] * F[2][2];
    double c02 = F[0][0] * F[0][2] + F[1][0] * F[1][2] + F[2][0] * F[2][2];
    double R[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};  // columns = eigenvectors n_a
#pragma unroll 1
    for (int sweep = 0; sweep < JAC_SWEEPS; sweep++) {
        jacobi_rot(c00, c11, c01, c02, c12, R[0][0], R[0][1], R[1][0], R[1][1], R[2][0], R[2][1]);
        jacobi_rot(c00, c22, c02, c01, c12, R[0][0], R[0][2], R[1][0], R[1][2], R[2][0], R[2][2]);
        jacobi_rot(c11, c22, c12, c01, c02, R[0][1], R[0][2], R[1][1], R[1][2], R[2][1], R[2][2]);
    }
    double lam[3] = {c00, c11, c22};

    PHASE_SYNC_N(1);
    // ---- rotate F and G into the eigenbasis (Lagrangian principal axes): F^_ia = F_iJ R_Ja, G^_Ia = G_IJ R_Ja
    double Fh[3][3];
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int a = 0; a < 3; a++) Fh[i][a] = F[i][0] * R[0][a] + F[i][1] * R[1][a] + F[i][2] * R[2][a];
#pragma unroll
    for (int I = 0; I < 8; I++) {
        double g0 = se[GGX(I, 0) + q], g1 = se[GGX(I, 1) + q], g2 = se[GGX(I, 2) + q];
#pragma unroll
        for (int a = 0; a < 3; a++) se[GGX(I, a) + q] = g0 * R[0][a] + g1 * R[1][a] + g2 * R[2][a];
    }

    // ---- material (derived record), orientation
    const double *md = matd + (long long)mat_stride * e;
    const double mu2 = __ldg(md + 0), kb = __ldg(md + 2);
    const bool rot = __ldg(md + 27) != 0.0;
    double Rm[3][3];  // eigenvectors of C in the material frame: Rm = Theta^T R
    double Th[3][3];
    if (rot) {
#pragma unroll
        for (int i = 0; i < 9; i++) Th[i / 3][i % 3] = __ldg(md + 18 + i);
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int a = 0; a < 3; a++) Rm[i][a] = Th[0][i] * R[0][a] + Th[1][i] * R[1][a] + Th[2][i] * R[2][a];
    } else {
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int a = 0; a < 3; a++) { Rm[i][a] = R[i][a]; Th[i][a] = (i == a) ? 1.0 : 0.0; }
    }

    // ---- S5 Hencky strain eps = sum_a 1/2 ln(lam_a) n_a (x) n_a (Eq.(5) :96 with the 1/2 restored, G1), material frame
    double lg[3];   // ln(lam_a): for stretches within ~15 % of 1, ln l = 2 w atanh(w)/w with w = (l-1)/(l+1) (same series as atanhc)
    {
        double w[3];
#pragma unroll
        for (int a = 0; a < 3; a++) { w[a] = (lam[a] - 1.0) * frcp(lam[a] + 1.0); lg[a] = 2.0 * w[a] * atanhc(w[a], 0.0); }
#pragma unroll
        for (int a = 0; a < 3; a++) if (w[a] * w[a] >= 0.0225) lg[a] = flog(lam[a]);
    }
    double ee[6];  // elastic trial strain eps - eps_p_n, tensor components (11,22,33,12,23,13), material frame
    {
        const double e0 = 0.5 * lg[0], e1 = 0.5 * lg[1], e2 = 0.5 * lg[2];
        ee[0] = e0 * Rm[0][0] * Rm[0][0] + e1 * Rm[0][1] * Rm[0][1] + e2 * Rm[0][2] * Rm[0][2];
        ee[1] = e0 * Rm[1][0] * Rm[1][0] + e1 * Rm[1][1] * Rm[1][1] + e2 * Rm[1][2] * Rm[1][2];
        ee[2] = e0 * Rm[2][0] * Rm[2][0] + e1 * Rm[2][1] * Rm[2][1] + e2 * Rm[2][2] * Rm[2][2];
        ee[3] = e0 * Rm[0][0] * Rm[1][0] + e1 * Rm[0][1] * Rm[1][1] + e2 * Rm[0][2] * Rm[1][2];
        ee[4] = e0 * Rm[1][0] * Rm[2][0] + e1 * Rm[1][1] * Rm[2][1] + e2 * Rm[1][2] * Rm[2][2];
        ee[5] = e0 * Rm[0][0] * Rm[2][0] + e1 * Rm[0][1] * Rm[2][1] + e2 * Rm[0][2] * Rm[2][2];
    }
    // history in (global components) -> material frame
    double epm[6];  // eps_p_n in the material frame
    if (rot) {
        const double A[3][3] = {{epn[0], epn[3], epn[5]}, {epn[3], epn[1], epn[4]}, {epn[5], epn[4], epn[2]}};
        double B[3][3];  // B = A Theta
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) B[i][j] = A[i][0] * Th[0][j] + A[i][1] * Th[1][j] + A[i][2] * Th[2][j];
        epm[0] = Th[0][0] * B[0][0] + Th[1][0] * B[1][0] + Th[2][0] * B[2][0];
        epm[1] = Th[0][1] * B[0][1] + Th[1][1] * B[1][1] + Th[2][1] * B[2][1];
        epm[2] = Th[0][2] * B[0][2] + Th[1][2] * B[1][2] + Th[2][2] * B[2][2];
        epm[3] = Th[0][0] * B[0][1] + Th[1][0] * B[1][1] + Th[2][0] * B[2][1];
        epm[4] = Th[0][1] * B[0][2] + Th[1][1] * B[1][2] + Th[2][1] * B[2][2];
        epm[5] = Th[0][0] * B[0][2] + Th[1][0] * B[1][2] + Th[2][0] * B[2][2];
    } else {
#pragma unroll
        for (int i = 0; i < 6; i++) epm[i] = epn[i];
    }
#pragma unroll
    for (int i = 0; i < 6; i++) ee[i] -= epm[i];

    PHASE_SYNC_N(2);
    double Ch[6][6];   // C_ep in the eigenbasis of C, tensor components, upper triangle used
    double Tt[6];      // T in the eigenbasis of C
    int iters = 0;
    bool plastic = false, nonconv = false;
    if (YLD == 1) {
        // ---- S6-S8, S10 for Yld2004-18p: general return map in the material frame (fem_barlat.cuh), then C_ep and T are
        //      taken to the eigenbasis of C with the 6x6 matrix Q[A][I]: X^_A (tensor components) = sum_I Q[A][I] X_I (Mandel)
        const double law = __ldg(md + 3), hh0 = __ldg(md + 4), hh1 = __ldg(md + 5), hh2 = __ldg(md + 6);
        double Tm[6], dep[6], Cm[6][6], dg;
#if BAR_PARK
        // What the rest of the kernel needs after the return map waits in the (still unused) A^ region of shared memory:
        // the return map and the yield-function evaluation inside it want every register they can get.
#define PARK_ALL(OP)                                                                                          \
        _Pragma("unroll") for (int i_ = 0; i_ < 9; i_++) { OP(i_, Fh[i_ / 3][i_ % 3]); OP(9 + i_, Rm[i_ / 3][i_ % 3]); \
                                                           OP(30 + i_, Th[i_ / 3][i_ % 3]); }                  \
        _Pragma("unroll") for (int i_ = 0; i_ < 6; i_++) OP(18 + i_, epm[i_]);                                 \
        _Pragma("unroll") for (int i_ = 0; i_ < 3; i_++) { OP(24 + i_, lam[i_]); OP(27 + i_, lg[i_]); }        \
        OP(39, wq); OP(40, wgt); OP(41, detF);
#define PARK_ST(i, v) se[SM_AA + 8 * (i) + q] = (v)
#define PARK_LD(i, v) (v) = se[SM_AA + 8 * (i) + q]
        PARK_ALL(PARK_ST)
#endif
        bar_return_map(bard + (long long)bar_stride * e, mu2, kb, law, hh0, hh1, hh2, ee, alphan, kmax, Tm, dep, Cm, dg, iters,
                       plastic, nonconv);
#if BAR_PARK
        PARK_ALL(PARK_LD)
#undef PARK_ALL
#undef PARK_ST
#undef PARK_LD
#endif
        if (valid) {
            double *ho = hist_out + (e * 8 + q) * 7;
            double ep1[6];
#pragma unroll
            for (int i = 0; i < 6; i++) ep1[i] = epm[i] + dep[i];
            if (rot && plastic) {
                const double A[3][3] = {{ep1[0], ep1[3], ep1[5]}, {ep1[3], ep1[1], ep1[4]}, {ep1[5], ep1[4], ep1[2]}};
                double B[3][3];  // B = A Theta^T ; out = Theta B
#pragma unroll
                for (int i = 0; i < 3; i++)
#pragma unroll
                    for (int j = 0; j < 3; j++) B[i][j] = A[i][0] * Th[j][0] + A[i][1] * Th[j][1] + A[i][2] * Th[j][2];
                ep1[0] = Th[0][0] * B[0][0] + Th[0][1] * B[1][0] + Th[0][2] * B[2][0];
                ep1[1] = Th[1][0] * B[0][1] + Th[1][1] * B[1][1] + Th[1][2] * B[2][1];
                ep1[2] = Th[2][0] * B[0][2] + Th[2][1] * B[1][2] + Th[2][2] * B[2][2];
                ep1[3] = Th[0][0] * B[0][1] + Th[0][1] * B[1][1] + Th[0][2] * B[2][1];
                ep1[4] = Th[1][0] * B[0][2] + Th[1][1] * B[1][2] + Th[1][2] * B[2][2];
                ep1[5] = Th[0][0] * B[0][2] + Th[0][1] * B[1][2] + Th[0][2] * B[2][2];
            }
            if (!plastic) {   // elastic step: history copied unchanged (Eq.(18) :172), re-read rather than kept in registers
                const double *hin = hist_in + (e * 8 + q) * 7;
#pragma unroll
                for (int i = 0; i < 6; i++) ep1[i] = __ldg(hin + i);
            }
#pragma unroll
            for (int i = 0; i < 6; i++) ho[i] = ep1[i];
            ho[6] = alphan + dg;                              // Eq.(20) :178 with W = 1 (:145)
        }
        double Q[6][6];
#pragma unroll
        for (int A = 0; A < 6; A++) {
            const int a = (A < 3) ? A : (A == 3 ? 0 : (A == 4 ? 1 : 0)), b = (A < 3) ? A : (A == 3 ? 1 : 2);
#pragma unroll
            for (int I = 0; I < 6; I++) {
                const int i = (I < 3) ? I : (I == 3 ? 0 : (I == 4 ? 1 : 0)), j = (I < 3) ? I : (I == 3 ? 1 : 2);
                Q[A][I] = (I < 3) ? Rm[i][a] * Rm[i][b] : RSQRT2 * (Rm[i][a] * Rm[j][b] + Rm[j][a] * Rm[i][b]);
            }
        }
        double QC[6][6];
#pragma unroll
        for (int A = 0; A < 6; A++) {
            double t = 0.0;
#pragma unroll
            for (int I = 0; I < 6; I++) t = fma(Q[A][I], Tm[I], t);
            Tt[A] = t;
#pragma unroll
            for (int J = 0; J < 6; J++) {
                double s = 0.0;
#pragma unroll
                for (int I = 0; I < 6; I++) s = fma(Q[A][I], (I <= J) ? Cm[I][J] : Cm[J][I], s);
                QC[A][J] = s;
            }
        }
#pragma unroll
        for (int A = 0; A < 6; A++)
#pragma unroll
            for (int B = A; B < 6; B++) {
                double s = 0.0;
#pragma unroll
                for (int J = 0; J < 6; J++) s = fma(QC[A][J], Q[B][J], s);
                Ch[A][B] = s;
            }
    } else {
    // ---- S6 elastic predictor in the Hill eigenbasis: T_tr = p I + s, s = 2mu dev(ee) = sum_k c_k v_k (Eq.(16) :160)
    const double tre = ee[0] + ee[1] + ee[2];
    const double pres = kb * tre;
    double hk[5], ck[5], v1[3], v2[3];
#pragma unroll
    for (int k = 0; k < 5; k++) hk[k] = __ldg(md + 7 + k);
#pragma unroll
    for (int i = 0; i < 3; i++) { v1[i] = __ldg(md + 12 + i); v2[i] = __ldg(md + 15 + i); }
    {
        const double tm = tre * (1.0 / 3.0);
        const double s0 = mu2 * (ee[0] - tm), s1 = mu2 * (ee[1] - tm), s2 = mu2 * (ee[2] - tm);
        ck[0] = v1[0] * s0 + v1[1] * s1 + v1[2] * s2;
        ck[1] = v2[0] * s0 + v2[1] * s1 + v2[2] * s2;
        ck[2] = SQRT2 * mu2 * ee[3]; ck[3] = SQRT2 * mu2 * ee[4]; ck[4] = SQRT2 * mu2 * ee[5];
    }
    double hc2[5];
    double phitr2 = 0.0;
#pragma unroll
    for (int k = 0; k < 5; k++) { hc2[k] = hk[k] * ck[k] * ck[k]; phitr2 += hc2[k]; }
    const double phitr = (phitr2 > 0.0) ? phitr2 * frsqrt(phitr2) : 0.0;  // Eq.(11) :127
    const double law = __ldg(md + 3), hh0 = __ldg(md + 4), hh1 = __ldg(md + 5), hh2 = __ldg(md + 6);
    // ---- S6/S7 yield test and return map in ONE loop with a single evaluation site (code size): pass 0 evaluates the
    //      trial state (dgam = 0): f_tr = phi(T_tr) - sqrt(2/3) sigma_flow(alpha_n) (Eq.(17) :165, tie -> elastic); later
    //      passes are Newton on F(dgam) = sigma_y(alpha)/phi(x) - 1, x = 2mu dgam / sigma_y;
    //      the pass after convergence evaluates the state at the solution and leaves the loop.
    double dg = 0.0, sf = 0.0, dsf = 0.0;
    double rk[5] = {1.0, 1.0, 1.0, 1.0, 1.0};   // 1/(1 + x h_k)
    double phi2 = phitr2;
    {
        double lo = 0.0, hi = INFINITY;
        const double atol = 4.0e-16 * phitr * frcp(mu2);  // round-off floor of dgam (a strain): eps * |T| / 2mu
        bool conv = false;
        double prev_step = INFINITY, al_eval = alphan;
#pragma unroll 1
        for (int pass = 0;; pass++) {
            const double al = fma(W23, dg, alphan);
            if (conv && law != 0.0) {
                // state at the solution: the last Newton step moved alpha by delta with |delta| <= 1e-3 (eps0 + alpha), so the
                // Swift law is continued by its 4-term binomial series (remainder < 1e-16 relative) instead of a second pow
                const double bp = hh1 + al_eval, rho = (al - al_eval) * frcp(bp), n = hh2;
                const double c2 = 0.5 * n * (n - 1.0), c3 = c2 * (n - 2.0) * (1.0 / 3.0), c4 = c3 * (n - 3.0) * 0.25;
                sf *= fma(rho, fma(rho, fma(rho, fma(rho, c4, c3), c2), n), 1.0);
                dsf = n * sf * frcp(hh1 + al);
            } else flow_stress(law, hh0, hh1, hh2, al, sf, dsf);
            al_eval = al;
            const double sy = W23 * sf, dsy = W23 * dsf;
            const double isy = frcp(sy);
            const double x = mu2 * dg * isy;
            double S2 = 0.0, S3 = 0.0;
            {   // r_k = 1/(1 + x h_k) for the five k from ONE reciprocal of the product (prefix/suffix products)
                const double d0 = fma(x, hk[0], 1.0), d1_ = fma(x, hk[1], 1.0), d2 = fma(x, hk[2], 1.0), d3 = fma(x, hk[3], 1.0),
                             d4 = fma(x, hk[4], 1.0);
                const double p01 = d0 * d1_, p34 = d3 * d4, p012 = p01 * d2, p234 = d2 * p34;
                const double ip = frcp(p012 * p34);
                rk[0] = ip * (d1_ * p234); rk[1] = ip * (d0 * p234); rk[2] = ip * (p01 * p34);
                rk[3] = ip * (p012 * d4);  rk[4] = ip * (p012 * d3);
            }
#pragma unroll
            for (int k = 0; k < 5; k++) {
                const double t2 = hc2[k] * rk[k] * rk[k];
                S2 += t2; S3 = fma(t2 * rk[k], hk[k], S3);
            }
            phi2 = S2;
            if (pass == 0) {
                plastic = (phitr - sy) > 0.0;
                if (!plastic) break;
            }
            if (conv || pass > kmax) { nonconv = !conv; break; }
            iters = pass + 1;
            const double rphi = frsqrt(S2);
            const double Fv = fma(sy, rphi, -1.0);
            const double dxd = mu2 * isy * (1.0 - dg * dsy * W23 * isy);
            const double Fp = dsy * W23 * rphi + sy * S3 * rphi * rphi * rphi * dxd;
            if (Fv < 0.0) lo = dg; else hi = dg;
            double dgn = dg - Fv * frcp(Fp);
            if (!(dgn >= lo && dgn <= hi)) dgn = (hi < INFINITY) ? 0.5 * (lo + hi) : 2.0 * dg + 1e-12;
            // converged when the step is at the round-off floor, or when the residual is so small that the step just
            // computed (kept) lands on the root to round-off
            const double step = fabs(dgn - dg), lim = fma(tol, dgn, atol);
            // third exit: in the quadratic regime the error left after this step is ~ (step_k / step_{k-1}^2) step_k^2;
            // when that is 100x below the step tolerance the verification pass is skipped
            // (pred = step^3 / prev_step^2 <= 0.01 lim, written without the division; prev_step = inf on the first pass)
            conv = (step <= lim) || (fabs(Fv) <= 1e-12) ||
                   (step <= 1e-3 * dgn && step * step * step <= 0.01 * lim * (prev_step * prev_step));
            prev_step = step;
            dg = dgn;
        }
    }
    const double alpha1 = fma(W23, dg, alphan);
    double th[5], cn[5];   // theta_k = 2mu/(1+x h_k) ; c'_k = c_k/(1+x h_k)
#pragma unroll
    for (int k = 0; k < 5; k++) { th[k] = mu2 * rk[k]; cn[k] = ck[k] * rk[k]; }
    // flow direction N = H:T/phi (Eq.(13) :141) in the Hill eigenbasis, m = D^-1 N, beta of C_ep = D^-1 + beta m (x) m
    double mk[5], beta = 0.0;
    double nk[5];
    {
        const double iphi = plastic ? frsqrt(phi2) : 0.0;
        double a = 0.0;
#pragma unroll
        for (int k = 0; k < 5; k++) { nk[k] = hk[k] * cn[k] * iphi; mk[k] = th[k] * nk[k]; a = fma(mk[k], nk[k], a); }
        if (plastic) {
            const double kap = dg * iphi;                 // dgam / phi
            const double om = 1.0 - kap * a;
            const double Hp = (2.0 / 3.0) * dsf;          // W dsigma_y/dalpha = (2/3) sigma_flow'
            const double den = fma(om, Hp, a);
            beta = (kap * den - 1.0) * frcp(om * den);
        }
    }
    PHASE_SYNC_N(3);
    // ---- S10 history out: eps_p += dgam N, alpha += W dgam (Eq.(19)-(20) :176-178), back to global components
    if (valid) {
        double *ho = hist_out + (e * 8 + q) * 7;
        double ep1[6];
        ep1[0] = epm[0] + dg * (nk[0] * v1[0] + nk[1] * v2[0]);
        ep1[1] = epm[1] + dg * (nk[0] * v1[1] + nk[1] * v2[1]);
        ep1[2] = epm[2] + dg * (nk[0] * v1[2] + nk[1] * v2[2]);
        ep1[3] = epm[3] + dg * nk[2] * RSQRT2; ep1[4] = epm[4] + dg * nk[3] * RSQRT2; ep1[5] = epm[5] + dg * nk[4] * RSQRT2;
        if (rot && plastic) {
            const double A[3][3] = {{ep1[0], ep1[3], ep1[5]}, {ep1[3], ep1[1], ep1[4]}, {ep1[5], ep1[4], ep1[2]}};
            double B[3][3];  // B = A Theta^T ; out = Theta B
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) B[i][j] = A[i][0] * Th[j][0] + A[i][1] * Th[j][1] + A[i][2] * Th[j][2];
            ep1[0] = Th[0][0] * B[0][0] + Th[0][1] * B[1][0] + Th[0][2] * B[2][0];
            ep1[1] = Th[1][0] * B[0][1] + Th[1][1] * B[1][1] + Th[1][2] * B[2][1];
            ep1[2] = Th[2][0] * B[0][2] + Th[2][1] * B[1][2] + Th[2][2] * B[2][2];
            ep1[3] = Th[0][0] * B[0][1] + Th[0][1] * B[1][1] + Th[0][2] * B[2][1];
            ep1[4] = Th[1][0] * B[0][2] + Th[1][1] * B[1][2] + Th[1][2] * B[2][2];
            ep1[5] = Th[0][0] * B[0][2] + Th[0][1] * B[1][2] + Th[0][2] * B[2][2];
        }
        if (!plastic) {   // elastic step: history copied unchanged (Eq.(18) :172), re-read rather than kept in registers
            const double *hin = hist_in + (e * 8 + q) * 7;
#pragma unroll
            for (int i = 0; i < 6; i++) ep1[i] = __ldg(hin + i);
        }
#pragma unroll
        for (int i = 0; i < 6; i++) __stcs(ho + i, ep1[i]);   // streaming: written once, never read by this call
        __stcs(ho + 6, alpha1);
    }

    PHASE_SYNC_N(4);
    // ---- S8 algorithmic tangent in the eigenbasis of C (App. D :1002-1019 in closed form):
    //      C_ep = kb I(x)I + sum_k theta_k V^_k (x) V^_k + beta m^ (x) m^ ,  V^_k = Rm^T V_k Rm ; T^ = p I + sum c'_k V^_k
    double mh[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
    for (int A = 0; A < 6; A++) Tt[A] = (A < 3) ? pres : 0.0;
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) Ch[A][B] = (A < 3 && B < 3) ? kb : 0.0;
#pragma unroll
    for (int k = 0; k < 5; k++) {
        double Vh[6];
        if (k < 2) {
            const double *v = (k == 0) ? v1 : v2;
#pragma unroll
            for (int A = 0; A < 6; A++) {
                const int a = (A < 3) ? A : (A == 3 ? 0 : (A == 4 ? 1 : 0)), b = (A < 3) ? A : (A == 3 ? 1 : 2);
                Vh[A] = v[0] * Rm[0][a] * Rm[0][b] + v[1] * Rm[1][a] * Rm[1][b] + v[2] * Rm[2][a] * Rm[2][b];
            }
        } else {
            const int i = (k == 2) ? 0 : (k == 3 ? 1 : 0), j = (k == 2) ? 1 : 2;  // shear 12, 23, 13
#pragma unroll
            for (int A = 0; A < 6; A++) {
                const int a = (A < 3) ? A : (A == 3 ? 0 : (A == 4 ? 1 : 0)), b = (A < 3) ? A : (A == 3 ? 1 : 2);
                Vh[A] = RSQRT2 * (Rm[i][a] * Rm[j][b] + Rm[j][a] * Rm[i][b]);
            }
        }
#pragma unroll
        for (int A = 0; A < 6; A++) {
            Tt[A] = fma(cn[k], Vh[A], Tt[A]);
            mh[A] = fma(mk[k], Vh[A], mh[A]);
            const double tv = th[k] * Vh[A];
#pragma unroll
            for (int B = A; B < 6; B++) Ch[A][B] = fma(tv, Vh[B], Ch[A][B]);
        }
    }
#pragma unroll
    for (int A = 0; A < 6; A++) {
        const double bm = beta * mh[A];
#pragma unroll
        for (int B = A; B < 6; B++) Ch[A][B] = fma(bm, mh[B], Ch[A][B]);
    }
    }   // YLD == 0

    PHASE_SYNC_N(5);
    // ---- S9 geometric post-processor (Eq.(25) :204, analytic route of :288): with g = 1/2 ln,
    //      S^_ab = 2 g[a,b] T^_ab ;  C_L = P_L^T:C_ep:P_L + T:L_L  in the eigenbasis
    double d1[6];  // first divided differences g[a,b], Voigt-indexed: (00,11,22,01,12,02)
    d1[0] = 0.5 * frcp(lam[0]); d1[1] = 0.5 * frcp(lam[1]); d1[2] = 0.5 * frcp(lam[2]);
    {
        const double s01 = lam[0] + lam[1], s12 = lam[1] + lam[2], s02 = lam[0] + lam[2];
        const double i01 = frcp(s01), i12 = frcp(s12), i02 = frcp(s02);
        d1[3] = atanhc((lam[1] - lam[0]) * i01, lg[1] - lg[0]) * i01;
        d1[4] = atanhc((lam[2] - lam[1]) * i12, lg[2] - lg[1]) * i12;
        d1[5] = atanhc((lam[2] - lam[0]) * i02, lg[2] - lg[0]) * i02;
    }
    // second divided differences: g000,g111,g222 exact; gaab by recursion or series; g012
    const double lmean = (lam[0] + lam[1] + lam[2]) * (1.0 / 3.0);
    const double thr = 1.0e-4 * lmean;
    double g_aaa[3], g_aab[3][3], g012;
#pragma unroll
    for (int a = 0; a < 3; a++) g_aaa[a] = -d1[a] * d1[a];  // -1/(4 lam^2)
    {
        // recursion on the gaps with one reciprocal per eigenvalue pair (branch-free; a zero gap gives an unselected NaN),
        // series only where some point of the warp has a gap below the threshold (the nearly undeformed part of the mesh)
        const double gp01 = lam[0] - lam[1], gp12 = lam[1] - lam[2], gp02 = lam[0] - lam[2];
        const double i01 = frcp(gp01), i12 = frcp(gp12), i02 = frcp(gp02);
        g_aab[0][0] = g_aab[1][1] = g_aab[2][2] = 0.0;
        g_aab[0][1] = (d1[0] - d1[3]) * i01; g_aab[1][0] = (d1[3] - d1[1]) * i01;
        g_aab[1][2] = (d1[1] - d1[4]) * i12; g_aab[2][1] = (d1[4] - d1[2]) * i12;
        g_aab[0][2] = (d1[0] - d1[5]) * i02; g_aab[2][0] = (d1[5] - d1[2]) * i02;
        const double g01 = fabs(gp01), g12 = fabs(gp12), g02 = fabs(gp02);
        const double gmax = fmax(g01, fmax(g12, g02));
        // g[0,1,2] by recursion on the widest gap: (g[0,2]-g[2,1])/(l0-l1), (g[1,0]-g[0,2])/(l1-l2), (g[0,1]-g[1,2])/(l0-l2)
        g012 = (gmax == g01) ? (d1[5] - d1[4]) * i01 : ((gmax == g12) ? (d1[3] - d1[5]) * i12 : (d1[3] - d1[4]) * i02);
        const bool s01 = g01 < thr, s12 = g12 < thr, s02 = g02 < thr;
        if (__any_sync(0xffffffffu, s01 || s12 || s02)) {
            const double t01 = dd2_series(lam[0], lam[0], lam[1]), t10 = dd2_series(lam[1], lam[1], lam[0]);
            const double t12 = dd2_series(lam[1], lam[1], lam[2]), t21 = dd2_series(lam[2], lam[2], lam[1]);
            const double t02 = dd2_series(lam[0], lam[0], lam[2]), t20 = dd2_series(lam[2], lam[2], lam[0]);
            const double t012 = dd2_series(lam[0], lam[1], lam[2]);
            if (s01) { g_aab[0][1] = t01; g_aab[1][0] = t10; }
            if (s12) { g_aab[1][2] = t12; g_aab[2][1] = t21; }
            if (s02) { g_aab[0][2] = t02; g_aab[2][0] = t20; }
            if (gmax < thr) g012 = t012;
        }
    }
    // C_L^ = 4 g1_A g1_B C^_AB + Gamma_AB (T:L_L), weighted by the integration weight
    double CL[6][6];
#pragma unroll
    for (int A = 0; A < 6; A++)
#pragma unroll
        for (int B = A; B < 6; B++) CL[A][B] = 4.0 * d1[A] * d1[B] * Ch[A][B];
    // Gamma: [aa][aa] = 8 t_aa g_aaa ; [aa][ab] = 4 t_ab g_aab ; [ab][ab] = 2 (t_aa g_aab + t_bb g_abb) ;
    //        [ab][ac] = 2 t_bc g_abc ; all others 0
#pragma unroll
    for (int a = 0; a < 3; a++) CL[a][a] = fma(8.0 * Tt[a], g_aaa[a], CL[a][a]);
    // shear index 3 = (0,1), 4 = (1,2), 5 = (0,2)
    CL[0][3] = fma(4.0 * Tt[3], g_aab[0][1], CL[0][3]); CL[1][3] = fma(4.0 * Tt[3], g_aab[1][0], CL[1][3]);
    CL[1][4] = fma(4.0 * Tt[4], g_aab[1][2], CL[1][4]); CL[2][4] = fma(4.0 * Tt[4], g_aab[2][1], CL[2][4]);
    CL[0][5] = fma(4.0 * Tt[5], g_aab[0][2], CL[0][5]); CL[2][5] = fma(4.0 * Tt[5], g_aab[2][0], CL[2][5]);
    CL[3][3] += 2.0 * (Tt[0] * g_aab[0][1] + Tt[1] * g_aab[1][0]);
    CL[4][4] += 2.0 * (Tt[1] * g_aab[1][2] + Tt[2] * g_aab[2][1]);
    CL[5][5] += 2.0 * (Tt[0] * g_aab[0][2] + Tt[2] * g_aab[2][0]);
    CL[3][4] = fma(2.0 * Tt[5], g012, CL[3][4]);   // (01),(12) share 1 -> t_02
    CL[3][5] = fma(2.0 * Tt[4], g012, CL[3][5]);   // (01),(02) share 0 -> t_12
    CL[4][5] = fma(2.0 * Tt[3], g012, CL[4][5]);   // (12),(02) share 2 -> t_01
    double Sh[6];
#pragma unroll
    for (int A = 0; A < 6; A++) Sh[A] = 2.0 * d1[A] * Tt[A];

    // ---- stats flags
    bool nonfinite = false;
    {
        double chk = 0.0;
#pragma unroll
        for (int A = 0; A < 6; A++) chk += Sh[A];
        nonfinite = !isfinite(chk);
    }

    // ---- (F-bar) Y_ia = w/3 (A^:F^)_ia = w/3 [ P^_ia + F^_im C_L^[(ma)][(nn)] lam_n ]   (before weighting)
    if (FBAR) {
        double Z[6];
#pragma unroll
        for (int A = 0; A < 6; A++) {
            Z[A] = 0.0;
#pragma unroll
            for (int n = 0; n < 3; n++) Z[A] = fma((A <= n) ? CL[A][n] : CL[n][A], lam[n], Z[A]);
        }
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int a = 0; a < 3; a++) {
                double y = 0.0;
#pragma unroll
                for (int m = 0; m < 3; m++) y = fma(Fh[i][m], Sh[VG[m][a]] + Z[VG[m][a]], y);
                se[SM_YY + (3 * i + a) * 8 + q] = wq * (1.0 / 3.0) * y;
            }
    }

    // ---- S9/S10 P^ = F^ S^ (Eq.(26) :208) and A^_(ia)(kb) = delta_ik S^_ab + F^_im F^_kn C_L^[(ma)][(nb)] -> shared memory
    PHASE_SYNC_N(6);
    // ---- S11 element residual R^e_Ii = sum_q w P^_ia G^_Ia (Eq.(35) :257), P^ = F^ S^ (Eq.(26) :208): every thread forms
    //      its own point's 24 contributions, then a 3-step reduce-scatter butterfly over the 8 lanes of the element
    //      (fixed order => deterministic) leaves node I = q's three sums in this thread.
    double rI[3];
    {
        double Ph[3][3];
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int a = 0; a < 3; a++)
                Ph[i][a] = wq * (Fh[i][0] * Sh[VG[0][a]] + Fh[i][1] * Sh[VG[1][a]] + Fh[i][2] * Sh[VG[2][a]]);
        double r[24];
#pragma unroll
        for (int J = 0; J < 8; J++) {
            const double g0 = se[GGX(J, 0) + q], g1 = se[GGX(J, 1) + q], g2 = se[GGX(J, 2) + q];
#pragma unroll
            for (int i = 0; i < 3; i++) r[3 * J + i] = fma(Ph[i][2], g2, fma(Ph[i][1], g1, Ph[i][0] * g0));
        }
        const bool b4 = q & 4, b2 = q & 2, b1 = q & 1;
        double r12[12], r6[6];
#pragma unroll
        for (int j = 0; j < 12; j++) {   // keep nodes 0-3 (bit2 = 0) or 4-7, send the other half
            const double keep = b4 ? r[12 + j] : r[j], send = b4 ? r[j] : r[12 + j];
            r12[j] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
        }
#pragma unroll
        for (int j = 0; j < 6; j++) {
            const double keep = b2 ? r12[6 + j] : r12[j], send = b2 ? r12[j] : r12[6 + j];
            r6[j] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
        }
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const double keep = b1 ? r6[3 + j] : r6[j], send = b1 ? r6[j] : r6[3 + j];
            rI[j] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
        }
    }
    PHASE_SYNC_N(7);
    // ---- S9/S10 A^_(ia)(kb) = delta_ik S^_ab + F^_im F^_kn C_L^[(ma)][(nb)] (weighted) -> shared memory, packed symmetric,
    //      two entries per 16-byte slot so that phase 2 reads them with one broadcast LDS.128
#pragma unroll
    for (int A = 0; A < 6; A++) {
        Sh[A] *= wgt;
#pragma unroll
        for (int B = A; B < 6; B++) CL[A][B] *= wgt;
    }
    {
        double prev = 0.0;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            double X[3][6];  // X[a][B] = sum_m F^_im C_L^[(ma)][B]
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int B = 0; B < 6; B++) {
                    double x = 0.0;
#pragma unroll
                    for (int m = 0; m < 3; m++) {
                        const int A = VG[m][a];
                        x = fma(Fh[i][m], (A <= B) ? CL[A][B] : CL[B][A], x);
                    }
                    X[a][B] = x;
                }
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int k = i; k < 3; k++)
#pragma unroll
                    for (int b = 0; b < 3; b++) {
                        if (3 * k + b < 3 * i + a) continue;
                        double v = (k == i) ? Sh[VG[a][b]] : 0.0;
#pragma unroll
                        for (int n = 0; n < 3; n++) v = fma(X[a][VG[n][b]], Fh[k][n], v);
                        const int sI = sidx9(3 * i + a, 3 * k + b);   // 0..44, visited in increasing order
                        if (sI == 44) se[SM_AA + 352 + q] = v;
                        else if (sI & 1) *reinterpret_cast<double2 *>(se + SM_AA + (sI >> 1) * 16 + 2 * q) = make_double2(prev, v);
                        else prev = v;
                    }
        }
    }
    __syncwarp();

    PHASE_SYNC_N(8);
    // ---- S12 phase 2: K^e_(Ii)(Kk) = sum_q G^_Ia A^_(ia)(kb) G^_Kb (Eq.(37) :267) on the FP64 tensor-core path.
    //      For each component pair (i,k), i <= k, the 8x8 node matrix K^{ik}[I][K] = sum_{(q,a)} G^q_Ia H^{ik}_{(q,a),K} with
    //      H^{ik}_{(q,a),K} = sum_b A^q_(ia)(kb) G^q_Kb is an 8 x 24 x 8 product: six mma.m8n8k4.f64 steps over (a, q-half).
    //      The whole warp works on one element at a time; lane (gid = lane/4, tig = lane%4) holds G^q_{gid,a}, q = 4h + tig,
    //      which is both its A fragment (row I = gid) and the factor of its B fragment (column K = gid), and forms
    //      its B element H with three FMAs.  K^{ki} = (K^{ik})^T gives the remaining pairs.  DMMA runs at the DFMA rate on
    //      sm_100a, but one issue keeps the pipe busy for 16 cycles, so the contraction no longer stalls on
    //      dependent-issue latency, and the accumulators shrink from 45 to 12 doubles per thread.
    const int I = q;
    if (FBAR) {
        // gbar_Kk = sum_q (w_q J_q / (Jbar V)) g^q_Kk for node K = I
#pragma unroll
        for (int k = 0; k < 3; k++) {
            double sgb = 0.0;
#pragma unroll
            for (int qq = 0; qq < 8; qq++) sgb = fma(se[SM_WQ + qq], se[SM_GQ + (3 * I + k) * 8 + qq], sgb);
            se[SM_GB + 3 * I + k] = sgb;
        }
        __syncwarp();
    }
    {
        const int gid = lane >> 2, tig = lane & 3;
        double *const sw = sm + (tid >> 5) * 4 * ES;   // the warp's four elements
#pragma unroll 1
        for (int el = 0; el < 4; el++) {
            double *const sx = sw + el * ES;
            double g[2][3];
#pragma unroll
            for (int h = 0; h < 2; h++)
#pragma unroll
                for (int a_ = 0; a_ < 3; a_++) g[h][a_] = sx[GGX(gid, a_) + 4 * h + tig];
            double C[6][2];
#pragma unroll
            for (int p = 0; p < 6; p++) C[p][0] = C[p][1] = 0.0;
            const double *const sa_ = sx + SM_AA + 2 * tig;
#pragma unroll
            for (int a_ = 0; a_ < 3; a_++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    int p = 0;
#pragma unroll
                    for (int i = 0; i < 3; i++)
#pragma unroll
                        for (int k = i; k < 3; k++, p++) {
                            double hv = 0.0;
#pragma unroll
                            for (int b_ = 0; b_ < 3; b_++) {
                                const int sI = sidx9(3 * i + a_, 3 * k + b_);
                                const double av = (sI == 44) ? sx[SM_AA + 352 + 4 * h + tig] : sa_[(sI >> 1) * 16 + 8 * h + (sI & 1)];
                                hv = (b_ == 0) ? av * g[h][0] : fma(av, g[h][b_], hv);
                            }
                            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                         : "+d"(C[p][0]), "+d"(C[p][1]) : "d"(g[h][a_]), "d"(hv));
                        }
                }
            {
                // ---- phase 3: the accumulators go straight to the destination-major scratch.
                //      Lane holds K^{ik}[gid][2 tig + j] = component (i,k) of block (gid, 2 tig + j): one 16-byte store into block
                //      row gid.  Standard element: for i != k it is also component (k,i) of block (2 tig + j, gid): two 8-byte
                //      stores (the 8 lanes of equal tig fill 64 contiguous bytes).  Every 32-byte sector is written whole.
                const int w_el = (tid >> 5) * 4 + el;
                const bool el_ok = chunk * EL_PER_CTA + w_el < n_elems;
                const long long sd = __shfl_sync(0xffffffffu, my_slot, el * 8 + gid);
                if (!FBAR) {
                    const long long st0 = __shfl_sync(0xffffffffu, my_slot, el * 8 + 2 * tig);
                    const long long st1 = __shfl_sync(0xffffffffu, my_slot, el * 8 + 2 * tig + 1);
                    if (el_ok) {
                        int p = 0;
#pragma unroll
                        for (int i = 0; i < 3; i++)
#pragma unroll
                            for (int k = i; k < 3; k++, p++) {
                                if (FUSE) {
                                    st_hint2(Ke + sd * 72 + (3 * i + k) * 8 + 2 * tig, C[p][0], C[p][1], pol_keep);
                                    if (i != k) {
                                        st_hint(Ke + st0 * 72 + (3 * k + i) * 8 + gid, C[p][0], pol_keep);
                                        st_hint(Ke + st1 * 72 + (3 * k + i) * 8 + gid, C[p][1], pol_keep);
                                    }
                                } else {
                                    *reinterpret_cast<double2 *>(Ke + sd * 72 + (3 * i + k) * 8 + 2 * tig) = make_double2(C[p][0], C[p][1]);
                                    if (i != k) {
                                        Ke[st0 * 72 + (3 * k + i) * 8 + gid] = C[p][0];
                                        Ke[st1 * 72 + (3 * k + i) * 8 + gid] = C[p][1];
                                    }
                                }
                            }
                    }
                } else {
                    // F-bar: K^e_(Ii)(Kk) += sum_q r^q_Ii (gbar_Kk - g^q_Kk), r^q_Ii = sum_a Y^q_ia G^q_Ia
                    // (Y carries w_q/3): for each (i,k) an 8 x 8 x 8 product over q, two more DMMA steps per pair of the nine
                    // (the term is not symmetric).  A fragment: r^q_{gid,i}; B fragment: gbar_{gid,k} - g^q_{gid,k}; q = 4 h + tig.
                    double ra[2][3], hb[2][3];
#pragma unroll
                    for (int h = 0; h < 2; h++)
#pragma unroll
                        for (int i = 0; i < 3; i++) {
                            const double *yy = sx + SM_YY + 4 * h + tig;
                            ra[h][i] = fma(yy[(3 * i + 2) * 8], g[h][2], fma(yy[(3 * i + 1) * 8], g[h][1], yy[(3 * i) * 8] * g[h][0]));
                            hb[h][i] = sx[SM_GB + 3 * gid + i] - sx[SM_GQ + (3 * gid + i) * 8 + 4 * h + tig];
                        }
                    double D[3][3][2];
#pragma unroll
                    for (int i = 0; i < 3; i++)
#pragma unroll
                        for (int k = 0; k < 3; k++) {
                            D[i][k][0] = D[i][k][1] = 0.0;
#pragma unroll
                            for (int h = 0; h < 2; h++)
                                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                             : "+d"(D[i][k][0]), "+d"(D[i][k][1]) : "d"(ra[h][i]), "d"(hb[h][k]));
                        }
                    // symmetric part: pair (i,k), i <= k, is held as is; for i > k it is the transpose of pair (k,i), i.e. the
                    // accumulator of the lane that holds row 2 tig + j, column gid
                    {
                        int p = 0;
#pragma unroll
                        for (int i = 0; i < 3; i++)
#pragma unroll
                            for (int k = i; k < 3; k++, p++) {
                                D[i][k][0] += C[p][0]; D[i][k][1] += C[p][1];
                                if (i != k) {
#pragma unroll
                                    for (int j = 0; j < 2; j++) {
                                        const int src = (2 * tig + j) * 4 + (gid >> 1);
                                        const double c0 = __shfl_sync(0xffffffffu, C[p][0], src), c1 = __shfl_sync(0xffffffffu, C[p][1], src);
                                        D[k][i][j] += (gid & 1) ? c1 : c0;
                                    }
                                }
                            }
                    }
                    if (el_ok) {
#pragma unroll
                        for (int i = 0; i < 3; i++)
#pragma unroll
                            for (int k = 0; k < 3; k++)
                                *reinterpret_cast<double2 *>(Ke + sd * 72 + (3 * i + k) * 8 + 2 * tig) = make_double2(D[i][k][0], D[i][k][1]);
                    }
                }
            }
        }
        __syncwarp();
    }
    PHASE_SYNC_N(9);
    {
        // destination-major scratch: block row I of K^e and R^e_I go to the record of incidence entry (e,I) in the node-sorted
        // list, so that a gathering warp reads every node's contributions as one contiguous run
        if (valid) {
            double *ro = Re + (long long)my_slot * 3;
            if (FUSE) { st_hint(ro, rI[0], pol_keep); st_hint(ro + 1, rI[1], pol_keep); st_hint(ro + 2, rI[2], pol_keep); }
            else { ro[0] = rI[0]; ro[1] = rI[1]; ro[2] = rI[2]; }
        }
    }

    // ---- stats: warp-aggregated counters, per-CTA iteration histogram (a per-CTA shared-memory stage for the four counters and
    //      a ballot / match-based histogram were both measured slower: 3.04-3.05 vs 3.00 ms)
    {
        const unsigned mp = __ballot_sync(0xffffffffu, valid && plastic);
        const unsigned mn = __ballot_sync(0xffffffffu, valid && nonconv);
        const unsigned mj = __ballot_sync(0xffffffffu, valid && !(detF > 0.0));
        const unsigned mf = __ballot_sync(0xffffffffu, valid && nonfinite);
        if (lane == 0) {
            if (mp) atomicAdd(&stats[0], (unsigned long long)__popc(mp));
            if (mn) atomicAdd(&stats[1], (unsigned long long)__popc(mn));
            if (mj) atomicAdd(&stats[2], (unsigned long long)__popc(mj));
            if (mf) atomicAdd(&stats[3], (unsigned long long)__popc(mf));
        }
        if (valid && plastic) atomicAdd(&s_hist[iters < 63 ? iters : 63], 1u);
    }
  }
    if (FUSE) {
        // publish: every thread's records are visible device-wide (fence) before the chunk's flag takes this call's epoch
        __threadfence();
        el_sync<FUSE>();
        if (tid == 0) *reinterpret_cast<volatile unsigned int *>(sa.chunk_flag + chunk) = sa.epoch;
    }
    {
        __syncwarp();
        unsigned done = 0;
        if (lane == 0) { __threadfence_block(); done = atomicAdd(&s_done, 1u); }
        done = __shfl_sync(0xffffffffu, done, 0);
        if (done == (CTA_THREADS >> 5) - 1) {   // last element warp of the CTA: flush (no CTA-wide barrier at the tail)
            __threadfence_block();
            for (int b = lane; b < 64; b += 32) {
                const unsigned v = s_hist[b];
                if (v) atomicAdd(&stats[5 + b], (unsigned long long)v);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ gather kernels (S14)
// General node gather (a node with more than 8 incident elements, or collapsed elements): lane <-> neighbour position pos;
// the elem_pos bytes of each incident entry give the local nodes K whose column node sits at pos.  Reads the records from
// global memory directly.
__device__ __forceinline__ void gather_general_node(long long n, int b, int m, int lane, const int *__restrict__ inc,
                                                    const int *__restrict__ nb_ptr, const unsigned char *__restrict__ elem_pos,
                                                    const double *__restrict__ Ke, const double *__restrict__ Re,
                                                    double *__restrict__ csr_vals, double *__restrict__ residual) {
    const int o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    const uint2 *pos8 = reinterpret_cast<const uint2 *>(elem_pos);
    for (int pos = lane; pos < len; pos += 32) {
        double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        const unsigned pat = (unsigned)pos * 0x01010101u;
        for (int s = 0; s < m; s++) {
            const uint2 pk = pos8[inc[b + s]];
            unsigned long long hit = ((unsigned long long)(__vcmpeq4(pk.y, pat) & 0x01010101u) << 32) |
                                     (unsigned long long)(__vcmpeq4(pk.x, pat) & 0x01010101u);
            const double *rec = Ke + (long long)(b + s) * 72;
            while (hit) {
                const int K = (__ffsll((long long)hit) - 1) >> 3;
                hit &= hit - 1;
#pragma unroll
                for (int j = 0; j < 9; j++) acc[j] += rec[ksoff(K, j)];
            }
        }
        double *out = csr_vals + 9LL * o + 3 * pos;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            out[(long long)i * 3 * len + 0] = acc[3 * i + 0];
            out[(long long)i * 3 * len + 1] = acc[3 * i + 1];
            out[(long long)i * 3 * len + 2] = acc[3 * i + 2];
        }
    }
    if (lane < 3) {
        double r = 0.0;
        for (int s = 0; s < m; s++) r += Re[(long long)(b + s) * 3 + lane];
        residual[3 * n + lane] = r;
    }
}
// General kernel: every node through gather_general_node (meshes with collapsed elements).
__global__ void __launch_bounds__(256)
k_gather(long long n_nodes, const int *__restrict__ inc_ptr, const int *__restrict__ inc, const int *__restrict__ nb_ptr,
         const unsigned char *__restrict__ elem_pos, const double *__restrict__ Ke, const double *__restrict__ Re,
         double *__restrict__ csr_vals, double *__restrict__ residual) {
    const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (n >= n_nodes) return;
    const int b = inc_ptr[n], m = inc_ptr[n + 1] - b;
    gather_general_node(n, b, m, lane, inc, nb_ptr, elem_pos, Ke, Re, csr_vals, residual);
}

// Fast gather for meshes where no element lists a node twice: one warp per node copies the node's run of records
// (<= 4608 bytes) into shared memory with coalesced 16-byte loads and reduces it with gather_reduce_write; the few nodes
// of an unstructured hex mesh that belong to more than 8 elements take gather_general_node.
#define GW 8   // warps (nodes) per CTA
#ifndef GMINB
#define GMINB 5
#endif
template <int HV>   // HV = 1: the mesh has nodes with more than 8 elements (they take the general path)
__global__ void __launch_bounds__(GW * 32, GMINB)
k_gather_fast(long long n_nodes, const int *__restrict__ inc_ptr, const int *__restrict__ inc, const int *__restrict__ nb_ptr,
              const unsigned int *__restrict__ kvec, const unsigned char *__restrict__ elem_pos, const double *__restrict__ Ke,
              const double *__restrict__ Re, double *__restrict__ csr_vals, double *__restrict__ residual) {
    __shared__ __align__(16) double buf[GW][576];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long n = (long long)blockIdx.x * GW + w;
    if (n >= n_nodes) return;
    const int b = inc_ptr[n], m = inc_ptr[n + 1] - b;
    if (HV && m > 8) {   // warp-uniform
        gather_general_node(n, b, m, lane, inc, nb_ptr, elem_pos, Ke, Re, csr_vals, residual);
        return;
    }
    {
        const double2 *src = reinterpret_cast<const double2 *>(Ke + (long long)b * 72);
        double2 *dst = reinterpret_cast<double2 *>(buf[w]);
        const int lim = m * 36;
        double2 t[9];
#pragma unroll
        for (int it = 0; it < 9; it++) if (it * 32 + lane < lim) t[it] = src[it * 32 + lane];
#pragma unroll
        for (int it = 0; it < 9; it++) if (it * 32 + lane < lim) dst[it * 32 + lane] = t[it];
    }
    __syncwarp();
    gather_reduce_write(n, b, m, buf[w], lane, nb_ptr, kvec, Re, csr_vals, residual);
}

// After a fused element launch: the quads that no element warp gathered (scheduled past the last chunk: `tail`, fixed at
// setup; not ready when their warp looked: `left`, counted during the launch).  Every chunk has retired by now (stream
// order), so no flag is read.  4 warps x 4 nodes per CTA, grid-stride.
#define GL_WARPS 4
__global__ void __launch_bounds__(GL_WARPS * 32)
k_gather_list(long long n_nodes, const int *__restrict__ tail, int n_tail, const int *__restrict__ left,
              const unsigned int *__restrict__ left_count, const int *__restrict__ inc_ptr, const int *__restrict__ nb_ptr,
              const unsigned int *__restrict__ kvec, const double *__restrict__ Ke, const double *__restrict__ Re,
              double *__restrict__ csr_vals, double *__restrict__ residual) {
    extern __shared__ __align__(16) double dbuf[];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long total = (long long)n_tail + (long long)*left_count;
    for (long long it = (long long)blockIdx.x * GL_WARPS + w; it < total; it += (long long)gridDim.x * GL_WARPS) {
        const int quad = (it < n_tail) ? tail[it] : left[it - n_tail];
        const long long n0 = 4LL * quad;
        const int cnt = (int)min(4LL, n_nodes - n0);
        gather_warp_nodes<4>((int)n0 + lane, cnt, dbuf + w * 2304, lane, inc_ptr, nb_ptr, kvec, Ke, Re, csr_vals, residual);
    }
}

// ------------------------------------------------------------------------------------------------ launch
static inline unsigned nblk2(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

template <int FBAR, int FUSE, int YLD>
static int launch_element(fem_ctx *c, const double *u, const double *hist_in, int mstride, double *hist_out, const scatter_args &sa,
                          int bstride, cudaStream_t st) {
    constexpr int ES = FBAR ? ES_FBAR : ES_STD;
    const size_t smem = ((size_t)EL_PER_CTA * ES + (FUSE ? 4 * FUSE_GNB * 576 + 4 * 66 : 0)) * sizeof(double);   // + the zero blocks
    // the opt-in for > 48 KB of dynamic shared memory is per device and per kernel: remembered per context (= per device)
    const int slot = (FBAR ? 1 : 0) + 2 * (FUSE ? 1 : 0) + 4 * (YLD ? 1 : 0);
    if (!(c->attr_mask & (1u << slot))) {
        FEM_CUDA(cudaFuncSetAttribute(k_element<FBAR, FUSE, YLD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->attr_mask |= 1u << slot;
    }
    k_element<FBAR, FUSE, YLD><<<nblk2(c->n_elems, EL_PER_CTA), FUSE ? 2 * CTA_THREADS : CTA_THREADS, smem, st>>>(
        c->n_elems, c->d_coords, c->d_conn, u, hist_in, c->d_matd, mstride, c->opt.tol, c->opt.kmax, c->d_Ke, c->d_Re, hist_out,
        c->d_stats, sa, YLD ? c->d_bard : nullptr, bstride);
    return FEM_OK;
}

int fem_launch_assemble(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                        double *residual, double *csr_vals, double *hist_out, cudaStream_t st, const double *bar) {
    if (bar && n_mat > c->n_bard_cap) {
        if (c->d_bard) cudaFree(c->d_bard);
        c->d_bard = nullptr; c->n_bard_cap = 0;
        FEM_CUDA(cudaMalloc(&c->d_bard, sizeof(double) * FEM_BARD * n_mat));
        c->n_bard_cap = n_mat;
    }
    if (n_mat > c->n_matd_cap) {
        if (c->d_matd) cudaFree(c->d_matd);
        c->d_matd = nullptr; c->n_matd_cap = 0;
        FEM_CUDA(cudaMalloc(&c->d_matd, sizeof(double) * FEM_MATD * n_mat));
        c->n_matd_cap = n_mat;
    }
    // the fused kernel exists for the Hill-48 standard element (the F-bar and Yld2004-18p variants need all shared memory / registers)
    const bool fuse = c->fuse_ok && !c->opt.fbar && !bar;   // fuse_ok: the mesh qualifies and the mode asks for it (fem_build_csr_pattern)
    FEM_CUDA(cudaMemsetAsync(c->d_stats, 0, sizeof(unsigned long long) * 72, st));
    if (fuse) FEM_CUDA(cudaMemsetAsync(c->d_left_count, 0, sizeof(unsigned int), st));
    FEM_CUDA(cudaEventRecord(c->ev[0], st));
    k_mat_prep<<<nblk2(n_mat, MP_THREADS), MP_THREADS, 0, st>>>(n_mat, mat, c->d_matd);
    if (bar) {
        k_bar_prep<<<nblk2(n_mat, 128), 128, 0, st>>>(n_mat, bar, c->d_bard, c->d_stats + 69);
    }
    FEM_CUDA(cudaEventRecord(c->ev[1], st));
    const int mstride = (n_mat == 1) ? 0 : FEM_MATD, bstride = (n_mat == 1) ? 0 : FEM_BARD;
    c->epoch++;
    if (c->epoch == 0) c->epoch = 1;   // the flags start at 0
    scatter_args sa = {c->d_eorder, c->d_eslot, c->d_cta_quads, c->d_quad_deps, c->d_chunk_flag, c->epoch, c->d_left_list,
                       c->d_left_count, c->n_nodes, c->d_inc_ptr, c->d_nb_ptr, c->d_kvec, csr_vals, residual};
    int rc;
    if (bar)              rc = c->opt.fbar ? launch_element<1, 0, 1>(c, u, hist_in, mstride, hist_out, sa, bstride, st)
                                           : launch_element<0, 0, 1>(c, u, hist_in, mstride, hist_out, sa, bstride, st);
    else if (c->opt.fbar) rc = launch_element<1, 0, 0>(c, u, hist_in, mstride, hist_out, sa, 0, st);
    else if (fuse)        rc = launch_element<0, 1, 0>(c, u, hist_in, mstride, hist_out, sa, 0, st);
    else                  rc = launch_element<0, 0, 0>(c, u, hist_in, mstride, hist_out, sa, 0, st);
    if (rc != FEM_OK) return rc;
    FEM_CUDA(cudaEventRecord(c->ev[2], st));
    if (fuse) {
        if (!(c->attr_mask & (1u << 8))) {
            FEM_CUDA(cudaFuncSetAttribute(k_gather_list, cudaFuncAttributeMaxDynamicSharedMemorySize, GL_WARPS * 2304 * 8));
            c->attr_mask |= 1u << 8;
        }
        // the tail is known; what was left over is counted on the device: a fixed grid walks both lists
        k_gather_list<<<2 * c->n_sm, GL_WARPS * 32, GL_WARPS * 2304 * 8, st>>>(c->n_nodes, c->d_tail_quads, c->n_tail_quads, c->d_left_list,
                                                                          c->d_left_count, c->d_inc_ptr, c->d_nb_ptr, c->d_kvec, c->d_Ke,
                                                                          c->d_Re, csr_vals, residual);
    } else if (c->d_kvec) {   // no collapsed element: the table-driven gather (nodes with more than 8 elements take its general path)
        if (c->has_high_valence)
            k_gather_fast<1><<<nblk2(c->n_nodes, GW), GW * 32, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_kvec,
                                                                     c->d_elem_pos, c->d_Ke, c->d_Re, csr_vals, residual);
        else
            k_gather_fast<0><<<nblk2(c->n_nodes, GW), GW * 32, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_kvec,
                                                                     c->d_elem_pos, c->d_Ke, c->d_Re, csr_vals, residual);
    } else {
        k_gather<<<nblk2(c->n_nodes * 32, 256), 256, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_elem_pos, c->d_Ke,
                                                             c->d_Re, csr_vals, residual);
    }
    FEM_CUDA(cudaEventRecord(c->ev[3], st));
    FEM_CUDA(cudaGetLastError());
    c->ev_valid = true;
    return FEM_OK;
}

// ------------------------------------------------------------------------------------------------ no-allocation entry point
// fem_assemble_static (include/fem.h): the two-kernel schedule above (k_mat_prep, k_element<FBAR,0,0>, table-driven or
// general gather) with ALL of its scratch -- the K^e / R^e records, the derived material records and the counters -- in
// one file-scope device array instead of the context's cudaMalloc'd buffers.  For callers that may not allocate (CUDA
// graph capture, serving loops).  The array costs FEM_STATIC_SCRATCH_BYTES on every GPU that loads the library.
//   layout in doubles: [0, 576 M) K^e records | [576 M, 600 M) R^e records | [600 M, 600 M + FEM_MATD M) material
//   records | 72 x u64 counters, M = FEM_STATIC_MAX_ELEMS; every block starts on a 256-byte boundary.
#define ST_OFF_KE 0
#define ST_OFF_RE ((size_t)576 * FEM_STATIC_MAX_ELEMS)
#define ST_OFF_MATD ((size_t)600 * FEM_STATIC_MAX_ELEMS)
#define ST_OFF_STATS ((size_t)(600 + FEM_MATD) * FEM_STATIC_MAX_ELEMS)
#define ST_DOUBLES (ST_OFF_STATS + 96)
static_assert(ST_DOUBLES * sizeof(double) == FEM_STATIC_SCRATCH_BYTES, "include/fem.h states the size of the static scratch");
static_assert((ST_OFF_RE * 8) % 256 == 0 && (ST_OFF_MATD * 8) % 256 == 0 && (ST_OFF_STATS * 8) % 256 == 0, "block alignment");
static __device__ __align__(256) double g_static_scratch[ST_DOUBLES];

// In host code `g_static_scratch` is only a handle: the device address comes from cudaGetSymbolAddress, once per device.
#define ST_MAX_DEVICES 64
static double *g_static_ptr[ST_MAX_DEVICES];
static std::mutex g_static_mu;

// The device the context's buffers live on must be the current one: the symbol address and the launches below are per device.
static int static_device_of(const fem_ctx *c, int *dev) {
    FEM_CUDA(cudaGetDevice(dev));
    cudaPointerAttributes pa;
    FEM_CUDA(cudaPointerGetAttributes(&pa, c->d_coords));
    if (pa.type != cudaMemoryTypeDevice || pa.device != *dev || *dev < 0 || *dev >= ST_MAX_DEVICES) return FEM_ERR_ARG;
    return FEM_OK;
}

extern "C" int fem_assemble_static_prepare(fem_ctx *c) {
    if (!c) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (c->n_elems > FEM_STATIC_MAX_ELEMS) return FEM_ERR_TOO_LARGE;
    int dev = -1;
    int rc = static_device_of(c, &dev);
    if (rc != FEM_OK) return rc;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        double *p = nullptr;
        FEM_CUDA(cudaGetSymbolAddress((void **)&p, g_static_scratch));
        if (!p) return FEM_ERR_CUDA;
        g_static_ptr[dev] = p;
    }
    // dynamic shared-memory opt-in of the element kernel (same bookkeeping as launch_element)
    const int slot = c->opt.fbar ? 1 : 0;
    if (!(c->attr_mask & (1u << slot))) {
        const int smem = EL_PER_CTA * (c->opt.fbar ? ES_FBAR : ES_STD) * (int)sizeof(double);
        if (c->opt.fbar) FEM_CUDA(cudaFuncSetAttribute(k_element<1, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        else             FEM_CUDA(cudaFuncSetAttribute(k_element<0, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        c->attr_mask |= 1u << slot;
    }
    return FEM_OK;
}

extern "C" int fem_assemble_static(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                                   double *residual, double *csr_vals, double *hist_out, fem_stats *stats, void *cuda_stream) {
    if (!c || !u || !hist_in || !mat || !residual || !csr_vals || !hist_out) return FEM_ERR_NULL;
    if (!c->has_pattern) return FEM_ERR_NO_PATTERN;
    if (c->n_elems > FEM_STATIC_MAX_ELEMS) return FEM_ERR_TOO_LARGE;
    if (n_mat != 1 && n_mat != c->n_elems) return FEM_ERR_MAT;
    if (fem_ranges_overlap(hist_in, hist_out, sizeof(double) * 56 * (size_t)c->n_elems)) return FEM_ERR_ALIAS;
    int dev = -1;
    FEM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= ST_MAX_DEVICES) return FEM_ERR_ARG;
    double *base;
    { std::lock_guard<std::mutex> lk(g_static_mu); base = g_static_ptr[dev]; }
    if (!base || !(c->attr_mask & (1u << (c->opt.fbar ? 1 : 0)))) {   // first use on this device / context: the set-up step
        int rc = fem_assemble_static_prepare(c);
        if (rc != FEM_OK) return rc;
        std::lock_guard<std::mutex> lk(g_static_mu);
        base = g_static_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *Ke = base + ST_OFF_KE, *Re = base + ST_OFF_RE, *matd = base + ST_OFF_MATD;
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(base + ST_OFF_STATS);
    // the array keeps the last call's contents: the counters are the one block that must start at zero (every K^e, R^e and
    // material record the gather reads is rewritten by this call before it is read)
    FEM_CUDA(cudaMemsetAsync(cnt, 0, sizeof(unsigned long long) * 72, st));
    k_mat_prep<<<nblk2(n_mat, MP_THREADS), MP_THREADS, 0, st>>>(n_mat, mat, matd);
    const int mstride = (n_mat == 1) ? 0 : FEM_MATD;
    scatter_args sa = {c->d_eorder, c->d_eslot, nullptr, nullptr, nullptr, 0u, nullptr, nullptr, c->n_nodes, c->d_inc_ptr, c->d_nb_ptr,
                       c->d_kvec, csr_vals, residual};
    const unsigned grid = nblk2(c->n_elems, EL_PER_CTA);
    if (c->opt.fbar)
        k_element<1, 0, 0><<<grid, CTA_THREADS, (size_t)EL_PER_CTA * ES_FBAR * sizeof(double), st>>>(
            c->n_elems, c->d_coords, c->d_conn, u, hist_in, matd, mstride, c->opt.tol, c->opt.kmax, Ke, Re, hist_out, cnt, sa, nullptr, 0);
    else
        k_element<0, 0, 0><<<grid, CTA_THREADS, (size_t)EL_PER_CTA * ES_STD * sizeof(double), st>>>(
            c->n_elems, c->d_coords, c->d_conn, u, hist_in, matd, mstride, c->opt.tol, c->opt.kmax, Ke, Re, hist_out, cnt, sa, nullptr, 0);
    if (c->d_kvec) {
        if (c->has_high_valence)
            k_gather_fast<1><<<nblk2(c->n_nodes, GW), GW * 32, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_kvec,
                                                                     c->d_elem_pos, Ke, Re, csr_vals, residual);
        else
            k_gather_fast<0><<<nblk2(c->n_nodes, GW), GW * 32, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_kvec,
                                                                     c->d_elem_pos, Ke, Re, csr_vals, residual);
    } else {
        k_gather<<<nblk2(c->n_nodes * 32, 256), 256, 0, st>>>(c->n_nodes, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_elem_pos, Ke, Re,
                                                             csr_vals, residual);
    }
    FEM_CUDA(cudaGetLastError());
    if (stats) {   // copies the counters back and synchronises the stream (no allocation: the destination is on the stack)
        unsigned long long h[72];
        FEM_CUDA(cudaMemcpyAsync(h, cnt, sizeof(h), cudaMemcpyDeviceToHost, st));
        FEM_CUDA(cudaStreamSynchronize(st));
        stats->n_plastic = (long long)h[0];
        stats->n_nonconverged = (long long)h[1];
        stats->n_detF_nonpos = (long long)h[2];
        stats->n_nonfinite = (long long)h[3];
        stats->max_local_iters = 0;
        for (int k = 0; k < 64; k++) {
            stats->iter_hist[k] = (long long)h[5 + k];
            if (h[5 + k]) stats->max_local_iters = k;
        }
    }
    return FEM_OK;
}
