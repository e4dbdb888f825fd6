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
    // colouring (assembly_mode 1): elements grouped by colour, first-writer masks
    int *d_elist = nullptr;                       // [n_elems] element ids sorted by (colour, id)
    unsigned long long *d_first_mask = nullptr;   // [n_elems] bit I*8+K: this element stores block (I,K) instead of adding
    unsigned int *d_first_res = nullptr;          // [n_elems] bit I: this element stores the residual of its local node I
    int mode = 0;                                 // effective assembly mode (1 and 2 fall back to 0 where they do not apply)
    // fused mode (assembly_mode 2): per-node countdown of missing contributions + queue of completed nodes
    int *d_cnt_init = nullptr;                    // [n_nodes] number of incident elements
    int *d_cnt = nullptr;                         // [n_nodes] working copy, counted down by the element CTAs
    int *d_queue_init = nullptr;                  // [n_nodes] nodes without elements first, then -1
    int *d_queue = nullptr;                       // [n_nodes] working copy: node ids in order of completion
    unsigned int *d_qctl = nullptr;               // [0] tail (tickets handed out), [1] head (entries claimed), [2..3] initial values
    int n_isolated = 0;
    bool has_high_valence = false;                // some node belongs to more than 8 elements
    bool has_collapsed = false;                   // some element lists a node twice
    int n_colours = 0, colour_rounds = 0;
    long long colour_start[65] = {0};
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
#define FEM_CUDA(call)                                                   \
    do {                                                                 \
        cudaError_t _e = (call);                                         \
        if (_e != cudaSuccess) return fem_cuda_fail(_e, #call);          \
    } while (0)

// fem_api.cu
int fem_read_stats(fem_ctx *c, fem_stats *stats, cudaStream_t st);
// fem_colour.cu
int fem_build_colouring(fem_ctx *c);
// fem_assemble.cu
int fem_launch_assemble(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                        double *residual, double *csr_vals, double *hist_out, cudaStream_t st, const double *bar = nullptr);
