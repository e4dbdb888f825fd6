/* fem.h — C ABI of the B200-native finite-strain Hill-48 element evaluation + CSR assembly library.
 *
 * One call of fem_assemble is one pass of the hot path of the Newton–Raphson FEM loop of
 * arxiv 2606.17390 ("JAX-FEM-ANISO"): per-quadrature-point logarithmic-strain return mapping
 * (Alg. C1/C2 :889-982), hex8 element internal force and consistent tangent
 * (Eq.(35)-(37),(40) :255-296) and assembly into a fixed-pattern global CSR matrix
 * (Eq.(34),(38) :251-275; Alg. E1 :1037-1049).  Readings of the paper are listed in DESIGN.md.
 *
 * Conventions (all calls)
 *   - units mm / MPa; all floating point is IEEE double; all indices are int32.
 *   - "dev" = pointer to CUDA device memory of the current device, "host" = ordinary host memory.
 *   - DOF id = 3*node + component.  Symmetric 2-tensors are 6 tensor components in the order
 *     (11,22,33,12,23,13) (PAPER.md:779 Eq.(A2), :793-796 Eq.(A4)).
 *   - hex8 node order of conn[e][0..7]: xi-signs (-,-,-),(+,-,-),(+,+,-),(-,+,-),(-,-,+),(+,-,+),(+,+,+),(-,+,+)
 *     (trilinear HEX-8); Gauss point q = kx + 2 ky + 4 kz, bit 0 <-> -1/sqrt3, weights 1.
 *   - every array argument is caller-owned; outputs are caller-allocated and fully overwritten;
 *     pattern arrays returned by fem_build_csr_pattern are library-owned and live until fem_destroy.
 *   - every call returns FEM_OK (0) or a negative error code; nothing throws.  There is no CPU fallback:
 *     without a CUDA device fem_setup returns FEM_ERR_CUDA.
 */
#ifndef FEM_B200_H
#define FEM_B200_H
#ifdef __cplusplus
extern "C" {
#endif

#define FEM_NPAR 16 /* doubles per material record, see fem_assemble */
#define FEM_NBARLAT 20 /* doubles per Yld2004-18p record, see fem_assemble_barlat */

enum {
    FEM_OK = 0,
    FEM_ERR_NULL = -1,        /* a required pointer is NULL */
    FEM_ERR_ARG = -2,         /* invalid size / option value */
    FEM_ERR_QUAD = -3,        /* quad_order != 2 */
    FEM_ERR_CONN = -4,        /* connectivity index out of [0, n_nodes) */
    FEM_ERR_INVERTED = -5,    /* det J_ref <= 0 at a Gauss point of some element */
    FEM_ERR_CUDA = -6,        /* CUDA runtime error (message via fem_last_cuda_error) */
    FEM_ERR_NO_PATTERN = -7,  /* fem_assemble before fem_build_csr_pattern */
    FEM_ERR_DEGREE = -8,      /* a node belongs to more than FEM_MAX_NODE_ELEMS elements */
    FEM_ERR_ALIAS = -9,       /* hist_out aliases hist_in */
    FEM_ERR_MAT = -10,        /* n_mat is neither 1 nor n_elems */
    FEM_ERR_NOCONV = -11,     /* iterative solve (fem_bicgstab, fem_newton_solve) did not converge */
    FEM_ERR_TOO_LARGE = -12   /* fem_assemble_static: the mesh has more than FEM_STATIC_MAX_ELEMS elements */
};
#define FEM_MAX_NODE_ELEMS 32

typedef struct fem_ctx fem_ctx; /* opaque, owned by the library */

typedef struct {
    int fbar;          /* 0 = standard element (default); 1 = F-bar, Eq.(31)-(32) PAPER.md:233-245 */
    int quad_order;    /* must be 2 (2x2x2 Gauss) */
    double tol;        /* relative step tolerance of the local (return-map) Newton solve; default 1e-10,
                          the step that meets it is still applied, so the root is at round-off */
    int kmax;          /* local Newton iteration cap (default 60); a point that hits it is counted, not an error */
    int jmax;          /* kept for ABI parity with Alg. C2's line search; the scalar solve
                          uses a bracket instead, so it is unused */
    double beta, eta;  /* Alg. C2 / App. B constants; unused by the scalar solve */
    int assembly_mode; /* How S14 (K = A K^e, R = A R^e, Eq.(34) :253, Eq.(38) :274) is scheduled; the result is bit-identical in all modes.
                          The element kernel writes K^e, R^e to a destination-major scratch (one 72-double record per
                          (element, local node), node-sorted), and every CSR entry is the sum of its records in ascending element
                          id (deterministic, no atomics).
                          1 = two kernels: the element kernel, then a stand-alone node-row gather kernel over all nodes (nodes with
                          more than 8 elements / collapsed elements take a general path in it).
                          2 = fused, lagged gather: the element kernel's CTAs carry a second warpgroup that gathers.  At
                          pattern-build time the nodes are cut into quads of four and every quad is given to one gather warp of
                          an element CTA that is launched at least one wave of resident CTAs after the last CTA that writes one
                          of its records; that warp sums the quad's CSR rows while the CTA's element warps evaluate their own 16
                          elements, reading the records back from L2 (they are then discarded there and never reach HBM).
                          Completion is tracked by one flag per CTA; a gather warp polls for a bounded time only, and a quad
                          that is not ready (or is scheduled past the last CTA) is finished by a short gather kernel after the
                          element launch.  Hill-48 standard element only; F-bar, fem_assemble_barlat, meshes with collapsed
                          elements or a node with more than 8 elements use mode 1.
                          0 (default) = mode 2 where it is the faster one (standard element, at least 8 waves of element CTAs,
                          about 42k elements on a B200), mode 1 otherwise. */
} fem_options;

typedef struct {
    long long n_plastic;      /* quadrature points that took the plastic branch (f_trial > 0, Eq.(17) :165) */
    long long n_nonconverged; /* local solves that hit kmax */
    long long n_detF_nonpos;  /* points with det F <= 0 (computation continues, C stays SPD) */
    long long n_nonfinite;    /* points whose stress is not finite */
    int max_local_iters;      /* largest local Newton iteration count */
    long long iter_hist[64];  /* iter_hist[k] = plastic points that used k iterations (k >= 63 clipped) */
} fem_stats;

/* Fills *opt with the defaults named above. */
void fem_default_options(fem_options *opt /*host*/);

/* fem_setup — "fem_setup(coords, hex8 connectivity, quadrature)" of the problem statement.
 * Copies mesh to library-owned device memory, validates connectivity range and det J_ref > 0 at all 8 Gauss points
 * of every element (O1: J_ref = sum_I X_I (x) dN_I/dxi, Eq.(28)).
 *   coords  dev [n_nodes*3]  xyz interleaved          conn  dev [n_elems*8] int32
 *   opt     host, may be NULL (defaults)
 * Synchronises the device once.  On error *out is NULL. */
int fem_setup(fem_ctx **out, long long n_nodes, const double *coords, long long n_elems, const int *conn,
              const fem_options *opt);

/* fem_build_csr_pattern — sorted, duplicate-free CSR pattern of all element DOF pairs (triplets of PAPER.md:296-298,
 * Alg. E1 :1039-1049; structural zeros are kept) and the element-to-CSR slot map.
 *   n_rows = 3*n_nodes, row_ptr dev [n_rows+1], col_idx dev [nnz] ascending within a row,
 *   elem_slot dev [n_elems*576]: elem_slot[e*576 + a*24 + b] = index into the CSR values of (dof_a, dof_b),
 *   a,b = 3*local_node + component.  Any out-pointer may be NULL; the 576-wide map is only materialised when
 *   elem_slot != NULL (fem_assemble uses the compressed per-node-pair form internally).
 * Built entirely on the device; synchronises once.  Must precede fem_assemble.
 * Library-owned device memory after this call (bytes per element, hex meshes): pattern and gather tables ~1.5 kB
 * (col_idx 0.98 kB of it), assembly scratch 4.8 kB (8 block-row records of 576 B + R^e), i.e. ~6.3 GB at
 * 1M elements, plus 2.3 kB per element if elem_slot is requested.  A cudaMalloc failure returns FEM_ERR_CUDA. */
int fem_build_csr_pattern(fem_ctx *c, long long *n_rows, long long *nnz, const int **row_ptr, const int **col_idx,
                          const int **elem_slot);

/* fem_assemble — one evaluation of residual R = A R^e (internal force, Eq.(35) :257 without the traction term),
 * tangent K = A K^e (Eq.(37) :267 / Eq.(40) :294) and updated history (Alg. C1 :916).
 *   u         dev [n_rows]         nodal displacement
 *   hist_in   dev [n_elems*8*7]    per Gauss point (eps_p 11,22,33,12,23,13 ; alpha), Eq.(6) :98-102
 *   mat       dev [n_mat*16]       E, nu, r11, r22, r33, r12, r23, r13, law(0 Voce,1 Swift), h0, h1, h2, q0..q3
 *                                  Voce (sigma0,Q,b) Eq.(10) :121; Swift (K,eps0,n); r = yield-stress ratios of Eq.(A3) :784;
 *                                  q = unit quaternion (w,x,y,z) of the material orientation Theta, Eq.(A1) :774
 *   n_mat     1 (uniform) or n_elems
 *   residual  dev [n_rows]   csr_vals dev [nnz]   hist_out dev [n_elems*8*7] (must not alias hist_in)
 *   stats     host, may be NULL; when non-NULL the call synchronises `stream` and copies the counters back
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream); all work is ordered on it
 * Sums are taken in a fixed order (ascending element id per entry, in either assembly mode): two calls with equal
 * inputs give bit-identical output.  The call is ordered on `cuda_stream`; two fem_assemble calls on the SAME context must
 * not run concurrently on different streams (they share the scratch and the completion flags).
 * Physics trouble (local non-convergence, det F <= 0, non-finite) is counted in stats, never an error return. */
int fem_assemble(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                 double *residual, double *csr_vals, double *hist_out, fem_stats *stats, void *cuda_stream);

/* fem_assemble_barlat — SURVEY.md section 8(f) NEXT-2: the same pass with the Barlat Yld2004-18p yield function
 * (Eq.(12); App. A.2 :808-830 Eq.(A7)-(A9)) in place of Hill-48: phi = [1/4 sum_{i,j} |s'_i - s''_j|^m]^(1/m)
 * over the eigenvalues of s' = C':P:T and s'' = C'':P:T, f = phi - sigma_flow(alpha), W = 1 (:145), return map of
 * Eq.(19)-(24) :176-196 by Newton iterations with the Goldstein line search of App. B :836-869 (beta = 1e-4, eta = 0.1).
 *   barlat    dev [n_mat*20]  c'12,c'13,c'21,c'23,c'31,c'32,c'44,c'55,c'66, the same nine of C'', m, 0
 *                             (Table 2 :471-477 order; shear rows in the component order 12,23,13; m an even integer 2..16 —
 *                             the paper uses 8, and 2, 4 for its reductions.  Any other value is replaced by the nearest
 *                             supported exponent inside the call, and the call returns FEM_ERR_ARG when stats != NULL)
 *   mat       as in fem_assemble; r11..r13 are ignored, E, nu, the hardening law and the orientation quaternion apply
 * All other arguments, the outputs, determinism and error behaviour are those of fem_assemble; opt.kmax caps the Newton iterations, opt.tol is unused (the iteration stops at the round-off
 * floor of the residual).  Launches one more (tiny) kernel than fem_assemble. */
int fem_assemble_barlat(fem_ctx *c, const double *u, const double *hist_in, const double *mat, const double *barlat,
                        long long n_mat, double *residual, double *csr_vals, double *hist_out, fem_stats *stats,
                        void *cuda_stream);

/* fem_assemble_static — fem_assemble for callers that may not allocate device memory inside the call (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation, arguments, outputs, summation
 * order and error codes as fem_assemble (Hill-48 model, standard or F-bar element as the context was set up; S1-S14 of
 * SURVEY.md section 8(a)), in the two-kernel schedule, but the scratch of the pass — the K^e / R^e records, the derived
 * material records and the counters — lives in ONE file-scope device array of FEM_STATIC_SCRATCH_BYTES inside the library
 * instead of the context's buffers.  Every GPU that loads the library holds that array until the process exits.
 *   - The call itself calls no cudaMalloc / cudaFree / allocating library routine.  The context (fem_setup,
 *     fem_build_csr_pattern) is built beforehand as usual; those set-up calls do allocate.
 *   - Limit: n_elems <= FEM_STATIC_MAX_ELEMS, else FEM_ERR_TOO_LARGE (nothing is launched).
 *   - fem_assemble_static_prepare(c) is the set-up step: with the context's device current it resolves the array's device
 *     address (once per device) and opts the element kernel into its shared-memory size (once per context).  Call it
 *     before capturing a graph; otherwise the first fem_assemble_static on the context does it.  FEM_ERR_ARG when the
 *     current device is not the one the context was built on.
 *   - ALL calls on a device share the array, whatever the context or stream: calls that overlap on the GPU race on it.
 *     Order them on one stream (or with events).  The array keeps the last call's contents; the call clears the
 *     counters itself, and every record it reads was written earlier in the same call.
 *   - stats: host, may be NULL; non-NULL synchronises the stream (leave it NULL under capture).
 * Results are bit-identical to fem_assemble on a context in assembly_mode 1 (and equal to the default mode, which sums in
 * the same order). */
#define FEM_STATIC_MAX_ELEMS 4096
#define FEM_STATIC_SCRATCH_BYTES 20710144 /* (576 + 24 + 32) doubles per element x 4096 + 96 counters words */
int fem_assemble_static_prepare(fem_ctx *c);
int fem_assemble_static(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                        double *residual, double *csr_vals, double *hist_out, fem_stats *stats, void *cuda_stream);

/* Same call with HOST buffers for every array: copies in, assembles, copies out, synchronises (used for end-to-end timing). */
int fem_assemble_host(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                      double *residual, double *csr_vals, double *hist_out, fem_stats *stats);

/* Device time in milliseconds of the kernels of the last fem_assemble on this context, measured with CUDA events
 * on the call's stream: ms[0] = element kernel (S2-S12; in the fused mode it also gathers most node rows, S14),
 * ms[1] = the gather kernel that follows it (two-kernel mode: all nodes; fused mode: the quads left over), ms[2] = material pre-pass.
 * Synchronises on the recorded events. */
int fem_last_kernel_ms(fem_ctx *c, double ms[3] /*host*/);

/* Number of kernels launched by one fem_assemble on this context (for bench.py's gpu_launches). */
int fem_launches_per_assemble(const fem_ctx *c);

/* Dependent-chain-free DFMA throughput probe: runs a register-resident fused-multiply-add kernel for about `ms_target`
 * milliseconds and returns the achieved FP64 rate in TFLOP/s (FMA = 2 flops) in *tflops.  Roofline denominator only. */
int fem_probe_fp64_peak(double ms_target, double *tflops /*host*/, void *cuda_stream);

void fem_destroy(fem_ctx *c);
const char *fem_strerror(int code);
const char *fem_last_cuda_error(void);

/* Host helper: Lankford r0, r45, r90 -> the paper's yield-stress ratios (r11,r22,r33,r12,r23,r13) of Eq.(A3)-(A5)
 * (textbook Hill-1948 plane-stress relations, axis 1 = rolling direction, sigma11^y = sigma0; reading D2). */
int fem_hill_from_lankford(double r0, double r45, double r90, double r_out[6] /*host*/);

/* ------------------------------------------------------------------------------------------------------------------
 * the steps on either side of fem_assemble in one global Newton iteration
 * K dd = -R (Eq.(39)): Dirichlet rows (Alg. E1 steps 6-11 :1048-1053), a linear solve on
 * the library's own CSR (the paper's default Krylov method is BiCGSTAB, :304; AMGX / cuDSS themselves are out of scope)
 * and the Newton loop of one load increment.  All arrays are dev pointers on the pattern of fem_build_csr_pattern.
 * ------------------------------------------------------------------------------------------------------------------ */

/* y = K x with K = (pattern of this context, csr_vals).  x, y dev [n_rows], must not alias.  Deterministic
 * (fixed reduction order).  Uses the block structure of the pattern (one warp per node, three rows at a time). */
int fem_spmv(fem_ctx *c, const double *csr_vals /*dev [nnz]*/, const double *x, double *y, void *cuda_stream);

/* Dirichlet rows, Alg. E1 steps 6-11 ("zero off-diagonal entries and reset the diagonal to unity",
 * :298): for every listed DOF d the row d of K becomes the identity row and rhs[d] = bc_rhs[i] (0 when bc_rhs is NULL).
 * Columns are left alone, as in the paper (K becomes unsymmetric).  One thread per constrained row.
 *   bc_dofs dev [n_bc] int32, each in [0, n_rows), no duplicates required (duplicates write the same values)
 *   bc_rhs  dev [n_bc] or NULL        csr_vals dev [nnz] in/out        rhs dev [n_rows] in/out, may be NULL */
int fem_apply_dirichlet(fem_ctx *c, long long n_bc, const int *bc_dofs, const double *bc_rhs, double *csr_vals,
                        double *rhs, void *cuda_stream);

/* Jacobi-preconditioned BiCGSTAB (van der Vorst 1992; right preconditioning with M = diag K) for K x = b.
 *   x dev [n_rows]: initial guess on entry, solution on exit        b dev [n_rows]
 *   stops when ||b - K x||_2 <= rtol * ||b||_2 (recurrence residual, confirmed by one explicit residual at the end)
 *   or after max_iter iterations.  On breakdown ((rhat, r), (rhat, v) or omega collapses) the iteration restarts from the
 *   explicit residual of the current x (at most 50 times).
 *   *iters (host, may be NULL) = iterations used; *relres (host, may be NULL) = explicit ||b - K x|| / ||b|| at exit.
 * Returns FEM_OK when the recurrence residual met rtol AND the explicit residual of the returned x is within 100 rtol (the
 * two drift apart by round-off at tight tolerances; *relres reports the explicit one), FEM_ERR_NOCONV otherwise (x holds the
 * last iterate).  Dot products are reduced in a
 * fixed order: two calls with equal inputs give bit-identical results.  Synchronises the stream (the iteration scalars stay on the device; the host
 * checks the convergence flag after every batch of 8 iterations and restarts the recurrence on breakdown). */
int fem_bicgstab(fem_ctx *c, const double *csr_vals, const double *b, double *x, double rtol, int max_iter, int *iters,
                 double *relres, void *cuda_stream);

/* Jacobi-preconditioned conjugate gradients for symmetric positive definite K; same arguments, stopping rule, determinism
 * and return codes as fem_bicgstab.  After fem_apply_dirichlet K as a whole is not symmetric (rows only, as in the paper),
 * but if the initial guess x already holds b[d] on every constrained DOF d, all Krylov vectors vanish there and the
 * iteration is CG on the symmetric reduced system; fem_newton_solve calls it that way.  Also returns FEM_ERR_NOCONV when
 * (p, K p) <= 0 is met (K not positive definite). */
int fem_pcg(fem_ctx *c, const double *csr_vals, const double *b, double *x, double rtol, int max_iter, int *iters,
            double *relres, void *cuda_stream);

/* Mixed-precision CG (off by default).  on = 1: inside fem_pcg — and wherever the library calls it: fem_newton_solve,
 * fem_adjoint_step — the SpMV of the iteration reads an fp32 copy of K (half the bytes of an HBM-bound kernel; one more
 * nnz-sized float workspace, refreshed at every call), vectors and scalars stay fp64, and every residual that decides
 * convergence is b - K x with the fp64 matrix: the iteration is restarted from it (iterative refinement, at most five
 * orders of magnitude per round) until that residual meets rtol.  The returned x therefore satisfies the same test as with
 * on = 0; iteration counts differ slightly, repeats are still bit-identical.  fem_bicgstab is not affected. */
int fem_set_mixed_precision(fem_ctx *c, int on);

/* out = a x + b y on DOF vectors (dev [n_rows]; out may alias x or y).  For the caller's load-step control, e.g. the
 * extrapolated initial guess u + (u - u_prev) dt/dt_prev of the paper's time stepping. */
int fem_lincomb(fem_ctx *c, double a, const double *x, double b, const double *y, double *out, void *cuda_stream);

typedef struct {
    double rtol;      /* Newton stops when ||rhs||_2 <= rtol * ||rhs of iteration 0||_2 ... */
    double atol;      /* ... or <= atol (rhs = -R on free DOFs, prescribed - current on constrained DOFs); defaults 1e-9, 1e-10 */
    int max_newton;   /* default 25 */
    double lin_rtol;  /* BiCGSTAB tolerance per Newton iteration, default 1e-10 */
    int lin_max_iter; /* default 10000 */
    int linear_solver; /* 0 (default) = fem_pcg for the standard element (K_ff symmetric), falling back to fem_bicgstab when CG
                         gives up; F-bar (unsymmetric K) always uses fem_bicgstab.  1 = fem_bicgstab only, 2 = fem_pcg only */
} fem_newton_options;

typedef struct {
    int newton_iters;        /* assemble + solve + update cycles performed */
    int converged;           /* 1 when a residual test passed */
    int lin_iters_total;     /* BiCGSTAB iterations over all Newton iterations */
    int lin_failures;        /* linear solves that returned FEM_ERR_NOCONV (the update is applied anyway) */
    double rhs_norm0, rhs_norm; /* first and last ||rhs||_2 */
    fem_stats last_stats;    /* statistics of the last fem_assemble */
    int physics_trouble;     /* 1 when the residual test passed but last_stats shows local solves that hit kmax, points with
                                det F <= 0 or non-finite stresses: the increment is then NOT accepted (converged = 0, FEM_ERR_NOCONV) */
} fem_newton_report;

void fem_default_newton_options(fem_newton_options *o /*host*/);

/* One load increment: global Newton-Raphson K dd = -R, d <- d + dd (Eq.(39)) with Dirichlet data.
 *   u        dev [n_rows] in/out: initial guess (e.g. the last converged state) -> converged displacement; when the
 *            increment fails (FEM_ERR_NOCONV) u is restored to its entry value, so the caller can cut the step back
 *            (the paper's adaptive stepping, is host control flow and stays with the caller)
 *   hist_in  dev [n_elems*56] history at the start of the increment (unchanged)
 *   hist_out dev [n_elems*56] history at the returned u (from the last fem_assemble)
 *   bc_dofs  dev [n_bc] constrained DOFs, bc_vals dev [n_bc] their prescribed TOTAL displacement
 * Each iteration: fem_assemble(u) -> rhs = -R -> constrained rows: identity, rhs = bc_vals - u (so the update lands on
 * the prescribed value) -> test ||rhs|| (relative to the ||rhs|| of iteration 0 of THIS call, which includes the boundary
 * mismatch of the initial guess) -> linear solve (fem_newton_options.linear_solver) -> u += dd.  The stiffness matrix, residual and
 * Krylov vectors live in library-owned workspace (allocated on first use).  Returns FEM_OK when converged,
 * FEM_ERR_NOCONV when max_newton is reached or when the balanced state shows physics trouble (rep->physics_trouble);
 * FEM_ERR_ALIAS when hist_out overlaps hist_in.  On every non-OK return u holds its entry value.  *rep (host, may be NULL) is
 * always filled.  Synchronises the stream. */
int fem_newton_solve(fem_ctx *c, double *u, const double *hist_in, const double *mat, long long n_mat, long long n_bc,
                     const int *bc_dofs, const double *bc_vals, double *hist_out, const fem_newton_options *opt,
                     fem_newton_report *rep, void *cuda_stream);

typedef struct {
    double dt0;        /* first load increment, as a fraction of the full load (default 1e-3) */
    double dt_min;     /* the path is abandoned (FEM_ERR_NOCONV) when a cut-back goes below this (1e-5) */
    double dt_max;     /* largest increment (5e-2) */
    double grow;       /* factor applied to dt after an accepted step that needed <= grow_below Newton iterations (1.5) */
    double cut;        /* factor applied to dt after a rejected step (0.5) */
    int grow_below;    /* (5) */
    int max_steps;     /* cap on accepted + rejected steps (10000) */
    int extrapolate;   /* initial guess of a step: 0 = last converged state, 1 = linear, 2 = quadratic extrapolation of the
                          converged states ("extrapolated initial guess") */
    fem_newton_options newton; /* per-increment Newton options (defaults: rtol 1e-8, max_newton 12, lin_rtol 1e-6, lin_max_iter 20000) */
} fem_path_options;

typedef struct {
    int steps;               /* accepted load steps */
    int rejected;            /* rejected steps (each one cuts dt back) */
    int rejected_physics;    /* of those: balanced states rejected for fem_stats trouble (fem_newton_report.physics_trouble) */
    int newton_iters_total;  /* over accepted and rejected steps */
    int lin_iters_total;
    double t_reached;        /* load fraction of the last accepted state (1 when the path was completed) */
    fem_newton_report last;  /* report of the last accepted step */
} fem_path_report;

void fem_default_path_options(fem_path_options *o /*host*/);

/* fem_load_path — the adaptive load stepping of the paper around fem_newton_solve ("time step in
 * [dt_min, dt_max], cut back on failure or non-finite values, extrapolated initial guess"; benchmark settings :485):
 * the prescribed displacement bc_full is ramped from 0 to its full value, load fraction t in (0, 1].
 *   u        dev [n_rows] in/out   converged state at t = 0 on entry (e.g. zeros) -> state at t_reached
 *   hist     dev [n_elems*56] in/out   history at t = 0 -> history of the last accepted state
 *   bc_dofs  dev [n_bc], bc_full dev [n_bc]: constrained DOFs and their prescribed displacement at t = 1
 *   t_accepted host [n_t_cap] or NULL: load fractions of the accepted steps (the schedule an adjoint sweep repeats)
 * A step is: guess = extrapolation of the last converged states (fem_lincomb arithmetic) -> fem_newton_solve at t + dt ->
 * accepted when it converged with no failed linear solve and no physics trouble; then dt grows by `grow` if the step was
 * easy.  Otherwise the state is left at the last accepted one and dt is cut by `cut`.
 * Returns FEM_OK when t = 1 was reached, FEM_ERR_NOCONV when dt fell below dt_min or max_steps was used up (u, hist hold the
 * last accepted state, rep->t_reached says where), other codes as fem_newton_solve.  Allocates one history-sized and four
 * n_rows-sized workspace arrays on first use.  Synchronises the stream. */
int fem_load_path(fem_ctx *c, double *u, double *hist, const double *mat, long long n_mat, long long n_bc, const int *bc_dofs,
                  const double *bc_full, const fem_path_options *opt, fem_path_report *rep, double *t_accepted, int n_t_cap,
                  void *cuda_stream);

/* fem_assemble_vjp — SURVEY.md section 8(f) NEXT-3: vector-Jacobian products of one fem_assemble pass, i.e. of the map
 * (u, hist_in, mat) -> (residual, hist_out), for the discrete adjoint of Alg. 1 (Eq.(49)-(51) :355-366).
 * With lam an adjoint vector on the residual and mu a cotangent on hist_out (either may be NULL = zero):
 *   g_u       dev [n_rows]       = (dR/du)^T lam + (dhist_out/du)^T mu.  With lam = NULL this is the history leg of
 *                                  (dR^{n+1}/du^n)^T lam^{n+1} on the right-hand side of Eq.(51); with mu = NULL it is K^T lam
 *                                  (K = dR/du is symmetric for the standard element, so fem_pcg solves the adjoint system).
 *   g_hist_in dev [n_elems*8*7]  = (dR/dhist_in)^T lam + (dhist_out/dhist_in)^T mu, in the stored components of hist
 *                                  (it is the cotangent mu of the previous load step: the internal variables the paper
 *                                  calls "implicitly accounted for", carried backwards; reading G17)
 *   g_mat     dev [n_mat*16]     = (dR/dmat)^T lam + (dhist_out/dmat)^T mu (Eq.(49) :355) for E, nu, r11..r13, h0, h1, h2
 *                                  (record positions 0-7 and 9-11); the law switch and the quaternion get 0.  n_mat = 1: the
 *                                  sum over all elements; n_mat = n_elems: one record per element.
 * Any of the three outputs may be NULL (not computed).  u, hist_in, mat, n_mat as in fem_assemble; the state is
 * re-evaluated inside the call (nothing is kept from fem_assemble), the return map is differentiated implicitly at its
 * root (App. D Eq.(D4)-(D7) :1002-1019, transposed).  Hill-48 only; both element formulations: with fbar = 1 the
 * coupling of an element's 8 Gauss points through Jbar (Eq.(31)-(32) :237-243) is part of the product, and K^T differs
 * from K.  Sums run in a fixed order, no atomics: equal inputs give bit-identical outputs.  Uses the library's
 * R^e scratch: do not run concurrently with fem_assemble on another stream.  Asynchronous on `cuda_stream`. */
int fem_assemble_vjp(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat,
                     const double *lam, const double *mu, double *g_u, double *g_hist_in, double *g_mat, void *cuda_stream);

/* fem_adjoint_step — one step n of the backward sweep of Alg. 1, composed of the calls above:
 *   K = dR/du at (u^n, h^{n-1})                                   (fem_assemble; the tangent "assembled during the forward solve", :368)
 *   v = -[ dJdu + (dhist_out/du)^T mu_in ]                        (right-hand side of Eq.(51) :366; fem_assemble_vjp with lam = NULL)
 *   K^T lam = v on the free DOFs, lam = 0 on bc_dofs              (standard element: K_ff is symmetric, fem_pcg on the row-eliminated K,
 *                                                                  falling back to fem_bicgstab; F-bar: K^T is formed on the same
 *                                                                  pattern (one more nnz-sized workspace) and solved by fem_bicgstab)
 *   mu_out = g_hist_in(lam, mu_in),  g_mat = (dR/dmat)^T lam + (dhist_out/dmat)^T mu_in      (Eq.(49) :355; fem_assemble_vjp)
 *   u        dev [n_rows]       converged displacement u^n of the step
 *   hist_in  dev [n_elems*56]   history h^{n-1} at the start of the step
 *   dJdu     dev [n_rows]       (dJ^n/du^n)^T, may be NULL (no objective term at this step)
 *   mu_in    dev [n_elems*56]   cotangent on h^n handed back by step n+1; NULL at the last step (terminal condition lam^{N_T+1} = 0)
 *   lam      dev [n_rows] out   adjoint vector of the step
 *   mu_out   dev [n_elems*56] out  cotangent on h^{n-1} for step n-1 (must not alias hist_in or mu_in; also used as scratch)
 *   g_mat    dev [n_mat*16] out this step's term of dJ/dtheta (overwritten; the caller accumulates over the steps and adds dJ^n/dtheta)
 * Returns FEM_OK, or FEM_ERR_NOCONV when the adjoint solve did not reach lin_rtol (outputs undefined).
 * *lin_iters (host, may be NULL) = Krylov iterations used.  Synchronises the stream. */
int fem_adjoint_step(fem_ctx *c, const double *u, const double *hist_in, const double *mat, long long n_mat, long long n_bc,
                     const int *bc_dofs, const double *dJdu, const double *mu_in, double *lam, double *mu_out, double *g_mat,
                     double lin_rtol, int lin_max_iter, int *lin_iters, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
