// fem_setup / fem_build_csr_pattern: mesh validation and the device-side CSR pattern build.
// Pattern = sorted union of all element DOF pairs (triplets of PAPER.md:296-298, Alg. E1 :1039-1049).  Because every
// node carries 3 DOFs the pattern is the node-adjacency graph blown up by 3x3: row 3n+i holds columns 3m+k for every
// neighbour node m (ascending) and k = 0..2.  The whole build runs on the device; integer atomics are used only for
// counting / unordered filling, and every list is sorted afterwards, so the result is deterministic.
#include "fem_internal.h"
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <math.h>
#include <new>
#include <stdio.h>
#include <string.h>

char g_fem_cuda_err[512] = "";
int fem_cuda_fail(cudaError_t e, const char *where) {
    snprintf(g_fem_cuda_err, sizeof(g_fem_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return FEM_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------ validation
// flags[0] |= 1 : connectivity out of range ; flags[0] |= 2 : det J_ref <= 0 at a Gauss point (O1, Eq.(28))
__global__ void k_validate(long long n_nodes, long long n_elems, const double *__restrict__ coords,
                           const int *__restrict__ conn, int *flags) {
    long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n_elems) return;
    int nd[8];
    bool ok = true;
    for (int a = 0; a < 8; a++) {
        nd[a] = conn[e * 8 + a];
        if (nd[a] < 0 || nd[a] >= n_nodes) ok = false;
    }
    if (!ok) { atomicOr(flags, 1); return; }
    for (int a = 0; a < 8; a++)
        for (int c = a + 1; c < 8; c++)
            if (nd[a] == nd[c]) atomicOr(flags, 8);   // collapsed element (a node listed twice)
    double X[8][3];
    for (int a = 0; a < 8; a++)
        for (int i = 0; i < 3; i++) X[a][i] = coords[3 * (long long)nd[a] + i];
    const double g = 0.57735026918962576451;
    bool inv = false;
    for (int q = 0; q < 8; q++) {
        double xi[3] = {(q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g};
        double J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (int a = 0; a < 8; a++) {
            double sx = ((a ^ (a >> 1)) & 1) ? 1.0 : -1.0, sy = (a & 2) ? 1.0 : -1.0, sz = (a & 4) ? 1.0 : -1.0;
            double fx = 1 + sx * xi[0], fy = 1 + sy * xi[1], fz = 1 + sz * xi[2];
            double d[3] = {0.125 * sx * fy * fz, 0.125 * fx * sy * fz, 0.125 * fx * fy * sz};
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) J[i][j] += X[a][i] * d[j];
        }
        double det = J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
                     J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
        if (!(det > 0.0)) inv = true;
    }
    if (inv) atomicOr(flags, 2);
}

// ------------------------------------------------------------------------------------------------ pattern kernels
__global__ void k_count_inc(long long n_elems, const int *__restrict__ conn, int *cnt) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < 8 * n_elems) atomicAdd(&cnt[conn[t]], 1);
}
__global__ void k_fill_inc(long long n_elems, const int *__restrict__ conn, const int *__restrict__ inc_ptr, int *cursor,
                           int *inc) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= 8 * n_elems) return;
    int n = conn[t];
    int p = atomicAdd(&cursor[n], 1);
    inc[inc_ptr[n] + p] = (int)t;  // t = e*8 + I
}
// sort each node's incident list ascending (=> ascending element id); flag nodes with too many elements
__global__ void k_sort_inc(long long n_nodes, const int *__restrict__ inc_ptr, int *inc, int *flags) {
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    int b = inc_ptr[n], m = inc_ptr[n + 1] - b;
    if (m > FEM_MAX_NODE_ELEMS) { atomicOr(flags, 4); return; }
    for (int i = 1; i < m; i++) {
        int v = inc[b + i], j = i - 1;
        while (j >= 0 && inc[b + j] > v) { inc[b + j + 1] = inc[b + j]; j--; }
        inc[b + j + 1] = v;
    }
}
// neighbour nodes of node n = union of the nodes of its incident elements, sorted ascending, unique.
// pass 0 (nb == nullptr): nnb[n] = count ; pass 1: write the list at nb_ptr[n].
__global__ void k_neighbours(long long n_nodes, const int *__restrict__ conn, const int *__restrict__ inc_ptr,
                             const int *__restrict__ inc, int *nnb, const int *__restrict__ nb_ptr, int *nb) {
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    int cand[8 * FEM_MAX_NODE_ELEMS];
    int b = inc_ptr[n], m = inc_ptr[n + 1] - b, k = 0;
    if (m > FEM_MAX_NODE_ELEMS) m = FEM_MAX_NODE_ELEMS;
    for (int s = 0; s < m; s++) {
        long long e = inc[b + s] >> 3;
        for (int a = 0; a < 8; a++) {
            int v = conn[e * 8 + a], j = k - 1;  // insertion keeping cand sorted & unique
            while (j >= 0 && cand[j] > v) j--;
            if (j >= 0 && cand[j] == v) continue;
            for (int t = k - 1; t > j; t--) cand[t + 1] = cand[t];
            cand[j + 1] = v;
            k++;
        }
    }
    if (nb == nullptr) { nnb[n] = k; return; }
    int o = nb_ptr[n];
    for (int j = 0; j < k; j++) nb[o + j] = cand[j];
}
__global__ void k_row_ptr(long long n_nodes, const int *__restrict__ nb_ptr, int *row_ptr) {
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n > n_nodes) return;
    if (n == n_nodes) { row_ptr[3 * n_nodes] = 9 * nb_ptr[n_nodes]; return; }
    int o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    for (int i = 0; i < 3; i++) row_ptr[3 * n + i] = 9 * o + i * 3 * len;
}
__global__ void k_col_idx(long long n_nodes, const int *__restrict__ nb_ptr, const int *__restrict__ nb, int *col_idx) {
    // one thread per neighbour-list entry j (global index); finds its node by binary search on nb_ptr
    long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long total = nb_ptr[n_nodes];
    if (j >= total) return;
    long long lo = 0, hi = n_nodes - 1;
    while (lo < hi) { long long mid = (lo + hi + 1) >> 1; if (nb_ptr[mid] <= j) lo = mid; else hi = mid - 1; }
    long long n = lo;
    int o = nb_ptr[n], len = nb_ptr[n + 1] - o, p = (int)(j - o), m = nb[j];
    for (int i = 0; i < 3; i++) {
        long long base = 9LL * o + (long long)i * 3 * len + 3 * p;
        col_idx[base] = 3 * m; col_idx[base + 1] = 3 * m + 1; col_idx[base + 2] = 3 * m + 2;
    }
}
__global__ void k_elem_pos(long long n_elems, const int *__restrict__ conn, const int *__restrict__ nb_ptr,
                           const int *__restrict__ nb, unsigned char *elem_pos) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;  // t = e*8 + I
    if (t >= 8 * n_elems) return;
    long long e = t >> 3;
    int n = conn[t], o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    for (int K = 0; K < 8; K++) {
        int m = conn[e * 8 + K], lo = 0, hi = len - 1;
        while (lo < hi) { int mid = (lo + hi) >> 1; if (nb[o + mid] < m) lo = mid + 1; else hi = mid; }
        elem_pos[t * 8 + K] = (unsigned char)lo;
    }
}
__global__ void k_elem_slot(long long n_elems, const int *__restrict__ conn, const int *__restrict__ row_ptr,
                            const unsigned char *__restrict__ elem_pos, int *elem_slot) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;  // t = e*24 + a
    if (t >= 24 * n_elems) return;
    long long e = t / 24;
    int a = (int)(t - e * 24), I = a / 3, i = a - 3 * I;
    int row = 3 * conn[e * 8 + I] + i, rp = row_ptr[row];
    for (int K = 0; K < 8; K++) {
        int p = elem_pos[(e * 8 + I) * 8 + K];
        for (int k = 0; k < 3; k++) elem_slot[e * 576 + a * 24 + 3 * K + k] = rp + 3 * p + k;
    }
}

// locality key of an element = its smallest node id; counts the descents of the key along the input order
__global__ void k_elem_key(long long n_elems, const int *__restrict__ conn, int *key, int *ids, unsigned long long *descents) {
    long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n_elems) return;
    int k = conn[e * 8];
    for (int a = 1; a < 8; a++) k = min(k, conn[e * 8 + a]);
    key[e] = k; ids[e] = (int)e;
    if (e > 0) {
        int kp = conn[(e - 1) * 8];
        for (int a = 1; a < 8; a++) kp = min(kp, conn[(e - 1) * 8 + a]);
        if (kp > k) atomicAdd(descents, 1ull);
    }
}

// inverse of the node-sorted incidence list: eslot[e*8+I] = j with inc[j] = e*8+I
__global__ void k_eslot(long long n_elems, const int *__restrict__ inc, int *eslot) {
    long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (j < 8 * n_elems) eslot[inc[j]] = (int)j;
}

// ---- fused, lagged gather (fem_assemble.cu): which chunks of the element launch write the records of a node quad
// epos[e] = position of element e in the processing order (only when a locality order exists)
__global__ void k_epos(long long n_elems, const int *__restrict__ eorder, int *epos) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n_elems) epos[eorder[i]] = (int)i;
}
// quad = nodes 4q .. 4q+3: deps[q*16] = number of distinct chunks (of el_per_cta consecutive elements of the processing
// order) that hold an element of one of these nodes (-1: more than 15), deps[q*16+1..] their ids; ready[q] = the largest.
__global__ void k_quad_deps(long long n_nodes, long long n_quads, int el_per_cta, const int *__restrict__ inc_ptr,
                            const int *__restrict__ inc, const int *__restrict__ epos, int *deps, int *ready) {
    long long qd = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (qd >= n_quads) return;
    int list[15], cnt = 0, mx = -1;
    bool over = false;
    for (long long n = 4 * qd; n < 4 * qd + 4 && n < n_nodes; n++)
        for (int s = inc_ptr[n]; s < inc_ptr[n + 1]; s++) {
            const int e = inc[s] >> 3, ch = (epos ? epos[e] : e) / el_per_cta;
            mx = max(mx, ch);
            bool found = false;
            for (int j = 0; j < cnt; j++) found |= (list[j] == ch);
            if (!found) { if (cnt < 15) list[cnt++] = ch; else over = true; }
        }
    deps[qd * 16] = over ? -1 : cnt;
    for (int j = 0; j < 15; j++) deps[qd * 16 + 1 + j] = (j < cnt) ? list[j] : 0;
    ready[qd] = over ? 0x7fffffff : mx;
}

// kvec for the fast gather; flags |= 16 if some node has more than 8 incident elements
__global__ void k_kvec(long long n_nodes, const int *__restrict__ inc_ptr, const int *__restrict__ inc,
                       const int *__restrict__ nb_ptr, const unsigned char *__restrict__ elem_pos, unsigned int *kvec, int *flags) {
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    const int b = inc_ptr[n], m = inc_ptr[n + 1] - b, o = nb_ptr[n], len = nb_ptr[n + 1] - o;
    if (m > 8) { atomicOr(flags, 16); return; }   // this node takes the general path of the gather kernel (kvec unused)
    // The in-kernel (fused) reduction keeps one neighbour position per lane: a node of a non-conforming mesh whose <= 8 elements do
    // not share faces can have up to 57 neighbours.  Such a mesh takes the two-kernel schedule (its gather loops over positions).
    if (len > 32) atomicOr(flags, 16);
    for (int p = 0; p < len; p++) kvec[o + p] = 0xffffffffu;
    for (int s = 0; s < m; s++) {
        const long long t = inc[b + s];
        for (int K = 0; K < 8; K++) {
            const int p = elem_pos[t * 8 + K];
            kvec[o + p] = (kvec[o + p] & ~(15u << (4 * s))) | ((unsigned)K << (4 * s));
        }
    }
}

static inline unsigned nblk(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// ------------------------------------------------------------------------------------------------ C ABI: host side
extern "C" void fem_default_options(fem_options *o) {
    if (!o) return;
    o->fbar = 0; o->quad_order = 2; o->tol = 1e-10; o->kmax = 60; o->jmax = 10; o->beta = 1e-4; o->eta = 0.1;
    o->assembly_mode = 0;
}

extern "C" const char *fem_strerror(int code) {
    switch (code) {
        case FEM_OK: return "ok";
        case FEM_ERR_NULL: return "null pointer argument";
        case FEM_ERR_ARG: return "invalid argument";
        case FEM_ERR_QUAD: return "unsupported quad_order (must be 2)";
        case FEM_ERR_CONN: return "connectivity index out of range";
        case FEM_ERR_INVERTED: return "det J_ref <= 0 (inverted element)";
        case FEM_ERR_CUDA: return "CUDA error";
        case FEM_ERR_NO_PATTERN: return "CSR pattern not built";
        case FEM_ERR_DEGREE: return "node belongs to too many elements";
        case FEM_ERR_ALIAS: return "hist_out aliases hist_in";
        case FEM_ERR_MAT: return "n_mat must be 1 or n_elems";
        case FEM_ERR_NOCONV: return "iterative solve did not converge";
        case FEM_ERR_TOO_LARGE: return "mesh exceeds FEM_STATIC_MAX_ELEMS (fem_assemble_static)";
        default: return "unknown error code";
    }
}
extern "C" const char *fem_last_cuda_error(void) { return g_fem_cuda_err; }

extern "C" int fem_hill_from_lankford(double r0, double r45, double r90, double r_out[6]) {
    if (!r_out) return FEM_ERR_NULL;
    if (!(r0 > 0) || !(r45 > 0) || !(r90 > 0)) return FEM_ERR_ARG;
    // Hill-1948 F,G,H,N from Lankford values with sigma11^y = sigma0 (G+H = 1); L = M = 3/2 (isotropic out-of-plane shear)
    double Gh = 1.0 / (1.0 + r0), Hh = r0 / (1.0 + r0), Fh = Hh / r90, Nh = (r45 + 0.5) * (Fh + Gh);
    r_out[0] = 1.0 / sqrt(Gh + Hh);
    r_out[1] = 1.0 / sqrt(Fh + Hh);
    r_out[2] = 1.0 / sqrt(Fh + Gh);
    r_out[3] = sqrt(1.5 / Nh);
    r_out[4] = 1.0;
    r_out[5] = 1.0;
    return FEM_OK;
}

static void ctx_free(fem_ctx *c) {
    if (!c) return;
    void *ptrs[] = {c->d_coords, c->d_conn, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_nb, c->d_row_ptr, c->d_col_idx,
                    c->d_eslot, c->d_eorder, c->d_diagpos, c->d_sw, c->d_part, c->d_scal, c->d_nw, c->d_nw_vals, c->d_cta_quads, c->d_quad_deps, c->d_tail_quads, c->d_chunk_flag, c->d_left_list, c->d_left_count, c->d_elem_pos, c->d_elem_slot, c->d_kvec, c->d_Ke, c->d_Re, c->d_matd, c->d_bard, c->d_stats, c->d_u, c->d_hin, c->d_hout,
                    c->d_mat, c->d_res, c->d_vals, c->d_sens_part, c->d_nw_valsT, c->d_vals32, c->d_path, c->d_path_hist};
    for (void *p : ptrs) if (p) cudaFree(p);
    for (int i = 0; i < 4; i++) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    delete c;
}
extern "C" void fem_destroy(fem_ctx *c) { ctx_free(c); }

extern "C" int fem_setup(fem_ctx **out, long long n_nodes, const double *coords, long long n_elems, const int *conn,
                         const fem_options *opt) {
    if (!out) return FEM_ERR_NULL;
    *out = nullptr;
    if (!coords || !conn) return FEM_ERR_NULL;
    if (n_nodes <= 0 || n_elems <= 0 || n_nodes > 700000000LL || n_elems > 200000000LL) return FEM_ERR_ARG;
    fem_options o;
    fem_default_options(&o);
    if (opt) o = *opt;
    if (o.quad_order != 2) return FEM_ERR_QUAD;
    if ((o.fbar != 0 && o.fbar != 1) || !(o.tol > 0) || o.kmax < 1 || (o.assembly_mode < 0 || o.assembly_mode > 2)) return FEM_ERR_ARG;
    int ndev = 0;
    FEM_CUDA(cudaGetDeviceCount(&ndev));
    if (ndev < 1) { snprintf(g_fem_cuda_err, sizeof(g_fem_cuda_err), "no CUDA device"); return FEM_ERR_CUDA; }
    fem_ctx *c = new (std::nothrow) fem_ctx;
    if (!c) return FEM_ERR_ARG;
    c->n_nodes = n_nodes; c->n_elems = n_elems; c->n_rows = 3 * n_nodes; c->opt = o;
    int rc = FEM_OK, hflags = 0, *dflags = nullptr;
    do {
#define TRY(call) { cudaError_t _e = (call); if (_e != cudaSuccess) { rc = fem_cuda_fail(_e, #call); break; } }
        TRY(cudaMalloc(&c->d_coords, sizeof(double) * 3 * n_nodes));
        TRY(cudaMalloc(&c->d_conn, sizeof(int) * 8 * n_elems));
        TRY(cudaMemcpy(c->d_coords, coords, sizeof(double) * 3 * n_nodes, cudaMemcpyDeviceToDevice));
        TRY(cudaMemcpy(c->d_conn, conn, sizeof(int) * 8 * n_elems, cudaMemcpyDeviceToDevice));
        TRY(cudaMalloc(&dflags, sizeof(int)));
        TRY(cudaMemset(dflags, 0, sizeof(int)));
        k_validate<<<nblk(n_elems, 128), 128>>>(n_nodes, n_elems, c->d_coords, c->d_conn, dflags);
        TRY(cudaGetLastError());
        TRY(cudaMemcpy(&hflags, dflags, sizeof(int), cudaMemcpyDeviceToHost));
        if (hflags & 1) { rc = FEM_ERR_CONN; break; }
        if (hflags & 2) { rc = FEM_ERR_INVERTED; break; }
        c->has_collapsed = (hflags & 8) != 0;
        {
            int dev = 0;
            TRY(cudaGetDevice(&dev));
            TRY(cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev));
        }
        TRY(cudaMalloc(&c->d_stats, sizeof(unsigned long long) * 72));
        for (int i = 0; i < 4; i++) TRY(cudaEventCreate(&c->ev[i]));
#undef TRY
    } while (0);
    if (dflags) cudaFree(dflags);
    if (rc != FEM_OK) { ctx_free(c); return rc; }
    *out = c;
    return FEM_OK;
}

extern "C" int fem_build_csr_pattern(fem_ctx *c, long long *n_rows, long long *nnz, const int **row_ptr,
                                     const int **col_idx, const int **elem_slot) {
    if (!c) return FEM_ERR_NULL;
    const long long nn = c->n_nodes, ne = c->n_elems;
    if (!c->has_pattern) {
        int *cnt = nullptr, *dflags = nullptr;
        void *tmp = nullptr;
        size_t tmp_bytes = 0;
        int rc = FEM_OK;
        do {
#define TRY(call) { cudaError_t _e = (call); if (_e != cudaSuccess) { rc = fem_cuda_fail(_e, #call); break; } }
            TRY(cudaMalloc(&cnt, sizeof(int) * (nn + 1)));
            TRY(cudaMalloc(&dflags, sizeof(int)));
            TRY(cudaMemset(dflags, 0, sizeof(int)));
            TRY(cudaMalloc(&c->d_inc_ptr, sizeof(int) * (nn + 1)));
            TRY(cudaMalloc(&c->d_inc, sizeof(int) * 8 * ne));
            TRY(cudaMalloc(&c->d_nb_ptr, sizeof(int) * (nn + 1)));
            TRY(cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, cnt, c->d_inc_ptr, (int)(nn + 1)));
            TRY(cudaMalloc(&tmp, tmp_bytes));
            // node -> incident elements
            TRY(cudaMemset(cnt, 0, sizeof(int) * (nn + 1)));
            k_count_inc<<<nblk(8 * ne, 256), 256>>>(ne, c->d_conn, cnt);
            TRY(cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, cnt, c->d_inc_ptr, (int)(nn + 1)));
            TRY(cudaMemset(cnt, 0, sizeof(int) * (nn + 1)));
            k_fill_inc<<<nblk(8 * ne, 256), 256>>>(ne, c->d_conn, c->d_inc_ptr, cnt, c->d_inc);
            k_sort_inc<<<nblk(nn, 128), 128>>>(nn, c->d_inc_ptr, c->d_inc, dflags);
            int hflags = 0;
            TRY(cudaMemcpy(&hflags, dflags, sizeof(int), cudaMemcpyDeviceToHost));
            if (hflags & 4) { rc = FEM_ERR_DEGREE; break; }
            // node -> neighbour nodes
            TRY(cudaMemset(cnt, 0, sizeof(int) * (nn + 1)));
            k_neighbours<<<nblk(nn, 64), 64>>>(nn, c->d_conn, c->d_inc_ptr, c->d_inc, cnt, nullptr, nullptr);
            TRY(cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, cnt, c->d_nb_ptr, (int)(nn + 1)));
            int nblocks = 0;
            TRY(cudaMemcpy(&nblocks, c->d_nb_ptr + nn, sizeof(int), cudaMemcpyDeviceToHost));
            if (9LL * nblocks > 2147483647LL) { rc = FEM_ERR_ARG; break; }  // int32 CSR offsets
            c->nnz = 9LL * nblocks;
            TRY(cudaMalloc(&c->d_nb, sizeof(int) * (size_t)nblocks));
            k_neighbours<<<nblk(nn, 64), 64>>>(nn, c->d_conn, c->d_inc_ptr, c->d_inc, cnt, c->d_nb_ptr, c->d_nb);
            TRY(cudaMalloc(&c->d_row_ptr, sizeof(int) * (c->n_rows + 1)));
            TRY(cudaMalloc(&c->d_col_idx, sizeof(int) * (size_t)c->nnz));
            k_row_ptr<<<nblk(nn + 1, 256), 256>>>(nn, c->d_nb_ptr, c->d_row_ptr);
            k_col_idx<<<nblk(nblocks, 256), 256>>>(nn, c->d_nb_ptr, c->d_nb, c->d_col_idx);
            TRY(cudaMalloc(&c->d_elem_pos, (size_t)64 * ne));
            k_elem_pos<<<nblk(8 * ne, 256), 256>>>(ne, c->d_conn, c->d_nb_ptr, c->d_nb, c->d_elem_pos);
            TRY(cudaGetLastError());
            if (!c->has_collapsed) {
                TRY(cudaMalloc(&c->d_kvec, sizeof(unsigned int) * (size_t)nblocks));
                TRY(cudaMemset(dflags, 0, sizeof(int)));
                k_kvec<<<nblk(nn, 128), 128>>>(nn, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_elem_pos, c->d_kvec, dflags);
                int kf = 0;
                TRY(cudaMemcpy(&kf, dflags, sizeof(int), cudaMemcpyDeviceToHost));
                c->has_high_valence = (kf & 16) != 0;   // some node has more than 8 elements: it is gathered by the general path
            }
            TRY(cudaDeviceSynchronize());
            {   // scratch (destination-major: one 72-double record per incidence entry)
                {   // processing order: when more than 5 % of the elements step back in node numbering (shuffled input), the element
                    // kernel walks the elements by ascending smallest node id (neighbouring CTAs then share nodes in L2 and
                    // write neighbouring scratch records); results do not depend on it
                    int *key = nullptr, *key2 = nullptr, *ids = nullptr;
                    unsigned long long *dsc = nullptr, hd = 0;
                    TRY(cudaMalloc(&key, sizeof(int) * ne)); TRY(cudaMalloc(&key2, sizeof(int) * ne)); TRY(cudaMalloc(&ids, sizeof(int) * ne));
                    TRY(cudaMalloc(&dsc, sizeof(unsigned long long)));
                    TRY(cudaMemset(dsc, 0, sizeof(unsigned long long)));
                    k_elem_key<<<nblk(ne, 256), 256>>>(ne, c->d_conn, key, ids, dsc);
                    TRY(cudaMemcpy(&hd, dsc, sizeof(hd), cudaMemcpyDeviceToHost));
                    if (hd * 20 > (unsigned long long)ne) {
                        void *t2 = nullptr; size_t t2b = 0;
                        TRY(cudaMalloc(&c->d_eorder, sizeof(int) * ne));
                        TRY(cub::DeviceRadixSort::SortPairs(nullptr, t2b, key, key2, ids, c->d_eorder, (int)ne));
                        TRY(cudaMalloc(&t2, t2b));
                        TRY(cub::DeviceRadixSort::SortPairs(t2, t2b, key, key2, ids, c->d_eorder, (int)ne));
                        TRY(cudaDeviceSynchronize());
                        cudaFree(t2);
                    }
                    cudaFree(key); cudaFree(key2); cudaFree(ids); cudaFree(dsc);
                }
                TRY(cudaMalloc(&c->d_eslot, sizeof(int) * 8 * ne));
                k_eslot<<<nblk(8 * ne, 256), 256>>>(ne, c->d_inc, c->d_eslot);
                TRY(cudaGetLastError());
                TRY(cudaMalloc(&c->d_Ke, sizeof(double) * 576 * ne));
                TRY(cudaMalloc(&c->d_Re, sizeof(double) * 24 * ne));
                TRY(cudaDeviceSynchronize());
            }
            // assembly_mode 0: fused gather where it pays (Hill-48 standard element, a mesh of at least FUSE_MIN_CHUNKS chunks of 16
            // elements - below that most quads are scheduled past the last chunk and the stand-alone gather is faster); 1: never;
            // 2: whenever the mesh qualifies (no collapsed element, no node with more than 8 elements)
            const long long FUSE_MIN_CHUNKS = 8LL * (2LL * c->n_sm + 32);
            const bool want_fuse = (c->opt.assembly_mode == 2) || (c->opt.assembly_mode == 0 && !c->opt.fbar && (ne + 15) / 16 >= FUSE_MIN_CHUNKS);
            if (want_fuse && c->d_kvec && !c->has_high_valence) {
                // fused, lagged gather: give every node quad to a gather warp of a chunk launched `lag` chunks after the last
                // chunk that writes one of its records (one wave of resident CTAs + a margin), at most two quads per warp
                const int EPC = 16, QPC = 8;                      // elements per CTA (fem_assemble.cu EL_PER_CTA), quads per chunk
                const long long n_chunks = (ne + EPC - 1) / EPC, n_quads = (nn + 3) / 4;
                const long long lag = 2LL * c->n_sm + 32;    // the fused kernel runs 2 CTAs per SM: one wave + a margin (328 ... 1000 measured alike)
                int *epos = nullptr, *d_ready = nullptr;
                if (c->d_eorder) {
                    TRY(cudaMalloc(&epos, sizeof(int) * ne));
                    k_epos<<<nblk(ne, 256), 256>>>(ne, c->d_eorder, epos);
                }
                TRY(cudaMalloc(&d_ready, sizeof(int) * n_quads));
                TRY(cudaMalloc(&c->d_quad_deps, sizeof(int) * 16 * n_quads));
                k_quad_deps<<<nblk(n_quads, 128), 128>>>(nn, n_quads, EPC, c->d_inc_ptr, c->d_inc, epos, c->d_quad_deps, d_ready);
                TRY(cudaGetLastError());
                int *ready = new (std::nothrow) int[n_quads], *cq = new (std::nothrow) int[n_chunks * QPC];
                int *nxt = new (std::nothrow) int[n_chunks + 1], *fill = new (std::nothrow) int[n_chunks], *tail = new (std::nothrow) int[n_quads];
                bool ok = ready && cq && nxt && fill && tail;
                cudaError_t ce = ok ? cudaMemcpy(ready, d_ready, sizeof(int) * n_quads, cudaMemcpyDeviceToHost) : cudaSuccess;
                int n_tail = 0;
                if (ok && ce == cudaSuccess) {
                    for (long long i = 0; i < n_chunks * QPC; i++) cq[i] = -1;
                    for (long long i = 0; i <= n_chunks; i++) nxt[i] = (int)i;       // next chunk >= i with a free slot (path-compressed)
                    for (long long i = 0; i < n_chunks; i++) fill[i] = 0;
                    static const int order[8] = {0, 2, 4, 6, 1, 3, 5, 7};             // one quad per warp first, then the second
                    const int cap = QPC;
                    for (long long qd = 0; qd < n_quads; qd++) {
                        long long want = (ready[qd] == 0x7fffffff) ? n_chunks : (long long)ready[qd] + lag;
                        if (want < 0) want = 0;
                        if (want >= n_chunks) { tail[n_tail++] = (int)qd; continue; }
                        long long r = want;
                        while (nxt[r] != r) r = nxt[r];
                        for (long long i = want; nxt[i] != r;) { const long long j = nxt[i]; nxt[i] = (int)r; i = j; }
                        if (r >= n_chunks) { tail[n_tail++] = (int)qd; continue; }
                        cq[r * QPC + order[fill[r]++]] = (int)qd;
                        if (fill[r] == cap) nxt[r] = (int)(r + 1);
                    }
                }
                if (ok && ce == cudaSuccess) ce = cudaMalloc(&c->d_cta_quads, sizeof(int) * n_chunks * QPC);
                if (ok && ce == cudaSuccess) ce = cudaMemcpy(c->d_cta_quads, cq, sizeof(int) * n_chunks * QPC, cudaMemcpyHostToDevice);
                if (ok && ce == cudaSuccess) ce = cudaMalloc(&c->d_tail_quads, sizeof(int) * (n_tail > 0 ? n_tail : 1));
                if (ok && ce == cudaSuccess && n_tail) ce = cudaMemcpy(c->d_tail_quads, tail, sizeof(int) * n_tail, cudaMemcpyHostToDevice);
                delete[] ready; delete[] cq; delete[] nxt; delete[] fill; delete[] tail;
                if (epos) cudaFree(epos);
                cudaFree(d_ready);
                if (!ok) { rc = FEM_ERR_ARG; break; }
                TRY(ce);
                c->n_tail_quads = n_tail;
                TRY(cudaMalloc(&c->d_chunk_flag, sizeof(unsigned int) * n_chunks));
                TRY(cudaMemset(c->d_chunk_flag, 0, sizeof(unsigned int) * n_chunks));
                TRY(cudaMalloc(&c->d_left_list, sizeof(int) * n_quads));
                TRY(cudaMalloc(&c->d_left_count, sizeof(unsigned int)));
                TRY(cudaMemset(c->d_left_count, 0, sizeof(unsigned int)));
                TRY(cudaDeviceSynchronize());
                c->fuse_ok = true;
            }
#undef TRY
        } while (0);
        if (cnt) cudaFree(cnt);
        if (dflags) cudaFree(dflags);
        if (tmp) cudaFree(tmp);
        if (rc != FEM_OK) return rc;
        c->has_pattern = true;
    }
    if (elem_slot && !c->d_elem_slot) {
        FEM_CUDA(cudaMalloc(&c->d_elem_slot, sizeof(int) * 576 * ne));
        k_elem_slot<<<nblk(24 * ne, 256), 256>>>(ne, c->d_conn, c->d_row_ptr, c->d_elem_pos, c->d_elem_slot);
        FEM_CUDA(cudaGetLastError());
        FEM_CUDA(cudaDeviceSynchronize());
    }
    if (n_rows) *n_rows = c->n_rows;
    if (nnz) *nnz = c->nnz;
    if (row_ptr) *row_ptr = c->d_row_ptr;
    if (col_idx) *col_idx = c->d_col_idx;
    if (elem_slot) *elem_slot = c->d_elem_slot;
    return FEM_OK;
}
