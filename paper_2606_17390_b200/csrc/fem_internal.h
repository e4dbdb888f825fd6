// Internal declarations shared by the translation units of libfem_b200.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/fem.h"

#define FEM_MATD 32  // doubles per derived material record (see k_mat_prep in fem_assemble.cu)

struct fem_ctx {
    long long n_nodes = 0, n_elems = 0, n_rows = 0, nnz = 0;
    fem_options opt;
    // mesh (library-owned copies)
    double *d_coords = nullptr;  // [n_nodes*3]
    int *d_conn = nullptr;       // [n_elems*8]
    // pattern
    bool has_pattern = false;
    int *d_inc_ptr = nullptr;    // [n_nodes+1]   node -> incident (element,local node) list
    int *d_inc = nullptr;        // [8*n_elems]   e*8+I, ascending within a node
    int *d_eorder = nullptr;     // [n_elems] processing order of the elements (ascending smallest node id) when the input order
                                 //   is not local (shuffled meshes); null = input order
    int *d_eslot = nullptr;      // [8*n_elems]   inverse of d_inc: index j of (e,I) in the node-sorted incidence list
    int *d_nb_ptr = nullptr;     // [n_nodes+1]   node -> sorted neighbour-node list
    int *d_nb = nullptr;         // [nnz/9]
    int *d_row_ptr = nullptr;    // [n_rows+1]
    int *d_col_idx = nullptr;    // [nnz]
    unsigned char *d_elem_pos = nullptr;  // [n_elems*64]  pos(conn[e][I], conn[e][K]) = rank of node K in nb list of node I
    int *d_elem_slot = nullptr;  // [n_elems*576], built on request
    unsigned int *d_kvec = nullptr;  // [nnz/9] per node-pair block: nibble s = local node K of the column node in incident entry s (0xF none); null if some node has > 8 elements
    // fused, lagged gather (fem_assemble.cu): node quads given to element warps at setup, chunk completion flags
    bool fuse_ok = false;                         // the mesh qualifies (no collapsed element, no node with more than 8 elements)
    int *d_cta_quads = nullptr;                   // [n_chunks*8] quad ids per chunk (two per warp), -1 = none
    int *d_quad_deps = nullptr;                   // [n_quads*16] [0] = number of chunks contributing to the quad's nodes, then their ids
    int *d_tail_quads = nullptr;                  // quads no element warp was given: gathered by k_gather_list after the element kernel
    int n_tail_quads = 0;
    unsigned int *d_chunk_flag = nullptr;         // [n_chunks] epoch of the last call in which the chunk finished
    int *d_left_list = nullptr;                   // [n_quads] quads whose chunks had not all finished when their warp looked
    unsigned int *d_left_count = nullptr;
    unsigned int epoch = 0;
    unsigned int attr_mask = 0;                   // kernels whose dynamic shared-memory opt-in has been set on this context's device
    int n_sm = 148;
    bool bad_barlat_m = false;                    // last fem_assemble_barlat saw an exponent outside the even integers 2..16
    bool has_high_valence = false;                // some node belongs to more than 8 elements
    bool has_collapsed = false;                   // some element lists a node twice
    // assemble workspace
    double *d_Ke = nullptr;      // [8*n_elems][72] destination-major scratch: record j = block row I of K^e of incidence entry j
                                 //   (node-sorted), component c of block (I,K) at (c>>1)*16 + 2K + (c&1) for c < 8, 64 + K for c = 8
    double *d_Re = nullptr;      // [8*n_elems][3]  R^e_I of incidence entry j
    double *d_matd = nullptr;    // [n_mat_cap*FEM_MATD]
    long long n_matd_cap = 0;
    double *d_bard = nullptr;    // [n_bard_cap*FEM_BARD] derived Yld2004-18p records (fem_barlat.cuh)
    long long n_bard_cap = 0;
    unsigned long long *d_stats = nullptr;  // [4 + 1 + 64] counters
    // NEXT-1 (fem_solve.cu): Dirichlet rows, SpMV, BiCGSTAB, Newton loop -- workspace allocated on first use
    int *d_diagpos = nullptr;      // [n_nodes] position of node n in its own neighbour list (diagonal block)
    double *d_sw = nullptr;        // [9*n_rows] Krylov vectors r, rhat, p, v, s, t, y, z and the inverse diagonal
    double *d_part = nullptr;      // partial sums of the deterministic reductions
    double *d_scal = nullptr;      // [8] reduced scalars
    double *d_nw = nullptr;        // [4*n_rows] Newton workspace: residual, rhs, dd, u at entry
    double *d_nw_vals = nullptr;   // [nnz] Newton workspace: stiffness values
    float *d_vals32 = nullptr;     // [nnz] fp32 copy of K for the SpMV inside mixed-precision CG (fem_set_mixed_precision)
    int mixed_precision = 0;
    double *d_nw_valsT = nullptr;  // [nnz] transposed stiffness values (adjoint step of the F-bar element), allocated on first use
    long long n_part = 0;
    double *d_path = nullptr;      // [4*n_rows] fem_load_path: trial state, two previous converged states, boundary values of the step
    double *d_path_hist = nullptr; // [n_elems*56] fem_load_path: second history buffer
    // NEXT-3 (fem_sens.cu): per-CTA partial sums of the material gradient (uniform material)
    double *d_sens_part = nullptr;
    long long n_sens_part = 0;
    // host-buffer path
    double *d_u = nullptr, *d_hin = nullptr, *d_hout = nullptr, *d_mat = nullptr, *d_res = nullptr, *d_vals = nullptr;
    long long n_mat_host_cap = 0;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
};

extern char g_fem_cuda_err[512];
int fem_cuda_fail(cudaError_t e, const char *where);
static inline int fem_cuda_rc(cudaError_t e, const char *where) { return e == cudaSuccess ? FEM_OK : fem_cuda_fail(e, where); }
// true when the byte ranges [a, a+bytes) and [b, b+bytes) intersect (hist_in / hist_out style aliasing checks)
static inline bool fem_ranges_overlap(const void *a, const void *b, size_t bytes) {
    const char *p = (const char *)a, *q = (const char *)b;
    return p < q + bytes && q < p + bytes;
}
#define FEM_CUDA(call)                                                   \
    do {                                                                 \
        cudaError_t _e = (call);                                         \
        if (_e != cudaSuccess) return fem_cuda_fail(_e, #call);          \
    } while (0)

// fem_api.cu
int fem_read_stats(fem_ctx *c, fem_stats *stats, cudaStream_t st);
// fem_assemble.cu
int fem_launch_assemble(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                        double *residual, double *csr_vals, double *hist_out, cudaStream_t st, const double *bar = nullptr);
