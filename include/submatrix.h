/*
 * submatrix.h -- C-ABI of libsubmatrix_b200.so: the data-parallel hot path of the submatrix
 * method for density-matrix linear-scaling DFT (Lass, Schade, Kuehne, Plessl, arXiv:2004.10811)
 * on one NVIDIA B200 (sm_100a).
 *
 *     D~ = 1/2 ( I - sign( K~ - mu I ) )            (Eq.(16), inner factor)
 *
 * evaluated approximately by the submatrix method: for every generating group
 * of block columns a dense principal submatrix is cut out of the block-sparse symmetric K~
 * (step 1, L125/L196/L199), its matrix sign function is computed (step 2; here by Newton-Schulz
 * iterations, Eq.(11), in FP64 on the tensor-core DMMA path), and the generating columns are
 * copied back on the input sparsity pattern (step 3, L127).
 *
 * Conventions
 *  - "host" / "device" says where a pointer must live.  The library never takes ownership of a
 *    caller buffer; a plan owns only its own device index tables (freed by sm_plan_destroy).
 *  - Block-sparse layout (DBCSR-like, L107; ordering of L180): nb block rows/columns with sizes
 *    blk_size[nb]; pattern in block-CSC: colptr[nb+1] (int64), rowidx[nnzb] (int32, strictly
 *    ascending inside a column).  The pattern must be structurally symmetric and contain every
 *    diagonal block.  Values: blocks in pattern order, each block (r,c) dense COLUMN-major
 *    blk_size[r] x blk_size[c]; the element offset of block b is the exclusive prefix sum of
 *    blk_size[r]*blk_size[c].  K~ must be numerically symmetric.  The result D~ uses the same
 *    pattern and layout; block (r,c) of column c comes from the submatrix of c's group (it is NOT
 *    symmetrised, L127).
 *  - Groups: grp_ptr[ngroups+1], grp_cols[nb] must be a partition of 0..nb-1 (every block column
 *    in exactly one group), so every result block is written exactly once.
 *  - Errors: no exceptions cross the boundary (host allocation failures come back as
 *    SM_ERR_ALLOC), no abort.  Status < 0: hard error, outputs unspecified.  Status > 0: warning,
 *    outputs are written and sm_stats_t says what is suspect.  sm_strerror() names any status.
 *  - One plan may be used by one stream at a time.  Results are deterministic run to run for a
 *    fixed plan and options (fixed reduction orders, no floating-point atomics).
 */
#ifndef SUBMATRIX_B200_H
#define SUBMATRIX_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sm_plan sm_plan_t; /* opaque */
typedef int32_t sm_status_t;

enum {
    SM_OK = 0,
    SM_ERR_INVALID_ARG = -1,         /* NULL pointer, negative size, bad option value            */
    SM_ERR_STRUCTURE = -2,           /* unsorted/duplicate rows, asymmetric pattern, missing     */
                                     /* diagonal block, groups not a partition                   */
    SM_ERR_ALLOC = -3,               /* host or device allocation failed                         */
    SM_ERR_CUDA = -4,                /* a CUDA call or kernel failed (see sm_last_cuda_error)    */
    SM_ERR_WORKSPACE_TOO_SMALL = -5, /* workspace_bytes < sm_plan_info_t.workspace_bytes         */
    SM_WARN_SIGN_NOT_CONVERGED = 1,  /* >= 1 submatrix hit max_iter or stagnated                 */
    SM_WARN_MU_NOT_CONVERGED = 2     /* bisection ended on mu_tol / max_steps, not on tol_n      */
};

/* Options fixed at plan creation.  Pass NULL for the defaults written beside each field. */
typedef struct {
    int32_t max_iter;    /* Newton-Schulz iteration cap per sign evaluation            [100] */
    int32_t scaling;     /* spectral bound for X0 = (a - mu I)/s (reading A8):          [1]  */
                         /* 0 = Gershgorin row sums of the assembled submatrix;              */
                         /* 1 = min(that, interlacing bound): a_i is a principal submatrix   */
                         /*     of K~, so rho(a_i - mu I) <= max|lambda_minmax(K~) - mu|,    */
                         /*     extremes of K~ by a short Lanczos run per call, then / overshoot; */
                         /*     a run that breaks down is discarded (Gershgorin only), and the  */
                         /*     cap is never below the largest column 2-norm of a_i - mu I      */
    int32_t precision;   /* 0 = FP64 DMMA (the parity path);                           [0]   */
                         /* opt-in reduced precision on the tcgen05 tensor cores (FP32       */
                         /* accumulators in tensor memory; accuracy reported separately; no  */
                         /* steering early-out):                                             */
                         /* 2 = "3xTF32": operands stored as hi + lo TF32 pairs, products    */
                         /*     hi hi + hi lo + lo hi -- THE reduced-precision variant: it   */
                         /*     meets the <= 1e-3 elementwise bar (measured 1e-6 class);     */
                         /* 3 = "BF16x2": operands stored as hi + lo BF16 pairs (16 mantissa */
                         /*     bits, 4 bytes per element), products hi hi + hi lo + lo hi   */
                         /*     on kind::f16: the rung between the two others -- error 1e-5  */
                         /*     class at half the FP64 time or less (half the operand bytes)  */
                         /* 4 = "FP16x2": as 3 with hi + lo FP16 pairs (22 mantissa bits):    */
                         /*     the accuracy of 2 (1e-6 class) at the cost of 3 -- the rung   */
                         /*     to prefer on this part                                        */
                         /* 1 = FP32 storage, plain TF32 products: experimental, error 5e-4   */
                         /*     ... 2e-3, does NOT meet the 1e-3 bar in general and its      */
                         /*     n_elec is too coarse to steer the mu search on large systems */
    int32_t check_every; /* the stop decisions are taken on the device; the host enqueues  [16]  */
                         /* this many iterations ahead before it reads the control block     */
                         /* (>= 1; launches after the stop are empty)                        */
    int32_t max_mu_steps;/* bisection step cap of sm_density_matrix                    [64]  */
    int32_t bisect_iter; /* iteration cap of the NON-final bisection evaluations        [0]  */
                         /* (0 = max_iter). A capped evaluation is only used for the         */
                         /* direction of the step, never for acceptance (A11).     */
    double mu_tol;       /* bisection stops when the bracket is narrower than this     [1e-6]*/
    int32_t early_out;   /* 1: a bisection evaluation stops as soon as the bound           [1]  */
                         /* |n_elec(final) - n_elec(X_k)| <= 1/2 sum_gen min(S1, (S1 + S2)/2), */
                         /* S1 = 1 - (X_k^2)_kk, S2 = sum_j (delta_kj - (X_k^2)_kj)^2,         */
                         /* proves the sign of n_elec - n_target (reading A11c); such a step */
                         /* only steers, it is never accepted.  0: every evaluation converges*/
    int32_t order;       /* 2: Newton-Schulz X <- 1/2 X (3I - X^2), Eq.(11) L97          [2]  */
                         /* 3: the paper's GPU iteration X <- 1/8 X (15I - 10X^2 + 3X^4),     */
                         /*    Eq.(19) L348 (three products per iteration, one more          */
                         /*    workspace buffer, FP64 only, overshoot forced to 1)           */
    double overshoot;    /* scaling = 1 only: s = bound / overshoot, 1 <= overshoot <= 1.5 [1.45]*/
                         /* (eigenvalues of X0 in (1, 1.5] map back into [0.56, 1); 1.45 is   */
                         /* where the top and the bottom of the water-like spectra balance)  */
    int32_t predict;     /* 1: predicted exit (reading A9b): a submatrix whose next residual [2]  */
                         /* is bounded a factor 10 below eps by ||E'|| <= 3/4||E||^2+1/4||E||^3 */
                         /* stops after its update, without the confirming X^2 product;      */
                         /* 2: also the two-step exit (reading A9c): the residual of X_{k+1}  */
                         /* is certified from one product (I - Y_k)^2 without forming         */
                         /* X_{k+1}; if it passes the test above, only the generating rows    */
                         /* of X_{k+2} are formed (generating rows spanning <= max(16, n/16)); 0: off */
    int32_t mu_guess;    /* sm_density_matrix, scaling = 1 only: the first interior step of the   [1]  */
                         /* mu search goes to the estimate the Gauss quadrature of the Lanczos     */
                         /* run gives for the target filling (reading A11d) if that lies inside    */
                         /* the bracket; 0 = pure midpoint bisection (reading A11)                 */
    int32_t rescale;     /* scaling = 1, order = 2, precision = 0 only (reading A8b): every          [1]  */
                         /* iteration applies Eq.(11) to al_k X_k, al_k = sqrt(3/(1 + l_k + l_k^2)), */
                         /* l_k the tracked lower bound of the eigenvalue moduli (l_0 from the Ritz  */
                         /* values of the Lanczos run), al_k = 1 once l_k >= 0.9999; replaces overshoot */
    int32_t mu_start;    /* sm_density_matrix with mu_guess (reading A11e): 1 = step 0 evaluates the      [1]  */
                         /* quadrature estimate instead of *mu_inout when *mu_inout lies outside the    */
                         /* Ritz interval the estimate is the middle of (a caller's mu inside it, e.g.  */
                         /* the previous SCF step's, is evaluated first); 0 = step 0 always evaluates   */
                         /* *mu_inout (reading A11)                                                      */
    int32_t method;      /* how the function of a submatrix is evaluated:                        [0]  */
                         /* 0 = Newton-Schulz iteration (Eq.(11)), every mu step re-evaluates it;     */
                         /* 1 = eigendecomposition a_i = Q Lambda Q^T (Eq.(17)) once per     */
                         /*     call and Algorithm 1 as written (L272-276): the mu loop runs on       */
                         /*     (lambda, w) alone (L266), D~ = Q f(Lambda - mu) Q^T on the generating  */
                         /*     columns.  FP64; literal midpoint bisection of reading A11 in the       */
                         /*     Gershgorin bracket (no steering / quadrature options needed)           */
    int32_t reserved1;
    double kT;           /* method = 1 only: electronic temperature in the units of K~ (L255:    [0]  */
                         /* signum of Eq.(17) replaced by the Fermi function, f(x) = 1 / (1 +          */
                         /* exp(x / kT)) for the occupation 1/2 (1 - signum(x)), reading A18); 0 =      */
                         /* zero temperature (signum)                                                  */
    int32_t shard_rank;  /* this plan covers one contiguous chunk of the     [0]  */
    int32_t shard_world; /* generating groups, chunk shard_rank of shard_world chunks balanced   [1]  */
                         /* by sum n_i^3 with >= 1 group each (the greedy rule of PAPER.md L235,       */
                         /* sm_partition_groups; contiguous chunks share blocks, L188-190).  The       */
                         /* pattern and the values are replicated; the plan gathers, iterates and      */
                         /* scatters only its own groups (d_vals_out: only their block columns are     */
                         /* written), n_elec is the local partial unless sm_plan_set_allreduce has     */
                         /* given the plan a sum over the ranks; shard_world <= 1: no sharding.        */
                         /* The steering early-out (early_out) needs the global bound at every         */
                         /* iteration and is switched off when shard_world > 1.                        */
} sm_options_t;

/* Plan facts (all sizes in elements unless they say bytes). */
typedef struct {
    int32_t nb, ngroups;
    int64_t nnzb;             /* stored blocks                                               */
    int64_t nnz;              /* stored values = length of the value arrays                  */
    int64_t n_basis;          /* sum of blk_size                                             */
    int64_t sum_sub_blocks;   /* sum_i |S_i|                                                 */
    int32_t dim_min, dim_max; /* min / max submatrix dimension n_i                           */
    double dim_mean;
    int64_t sum_n2, sum_n3;   /* sum n_i^2, sum n_i^3 (Eq.(14) cost model L201)              */
    int64_t sum_ld2;          /* sum of padded ld_i^2 = doubles per workspace buffer         */
    int64_t n_tiles;          /* CTA tiles per GEMM launch                                   */
    int32_t n_buckets;        /* distinct padded sizes                                       */
    int32_t reserved0;
    size_t workspace_bytes;   /* what sm_sign_execute / sm_density_matrix need               */
    int64_t sum_n3_columns;   /* sum over single block columns c of n~_c^3, n~_c = rows of the */
                              /* submatrix generated by column c alone (numerator of Eq.(15))  */
    double est_speedup;       /* Eq.(15): S = sum_c n~_c^3 / sum_i n_i^3, the estimated    */
                              /* additional speed-up of this grouping over per-column          */
                              /* submatrices under the O(n^3) cost model of Eq.(14)       */
    int64_t index_alg_bytes;  /* algorithmic bytes of the index build: nnzb*4 read + nnzb*4 +  */
                              /* sum|S_i|*8 written                               */
    float ms_index_kernels;   /* CUDA-event time of the index-builder kernels (a2)              */
    float ms_plan_create;     /* host wall clock of the whole sm_plan_create call               */
    int32_t shard_group_begin, shard_group_end; /* groups of the caller's numbering this plan covers   */
    int64_t shard_val_begin, shard_val_end;     /* their result values, if those form ONE contiguous   */
                              /* range of the value array (groups of ascending consecutive block       */
                              /* columns), else -1, -1: the all-gather of D~ needs no index lists then */
    int32_t ngroups_total, reserved2; /* groups of the whole problem (ngroups = those of this plan)    */
} sm_plan_info_t;

/* Filled by sm_sign_execute / sm_density_matrix (may be NULL). Times are CUDA-event ms of the
 * LAST sign evaluation when timing was requested with sm_set_timing(plan, 1), else 0. */
typedef struct {
    int32_t iterations;       /* Newton-Schulz iterations launched in the last evaluation    */
    int32_t iter_min, iter_max; /* per-submatrix iteration counts at convergence             */
    int32_t not_converged;    /* submatrices that hit max_iter / stagnated                   */
    double max_residual;      /* max_i ||X^2 - I||_F / sqrt(n_i) at exit                     */
    double n_elec;            /* sum_i sum_{k in gen(i)} 1/2 (1 - X_kk) (Algorithm 1)   */
    double mu;                /* chemical potential of the returned result                   */
    int32_t mu_steps;         /* sign evaluations done by sm_density_matrix                  */
    int32_t gemm_launches;    /* GEMM kernel launches in the last evaluation                 */
    int64_t sum_iter_n3;      /* sum_i products_i * n_i^3 (=> dense-GEMM flop = 2x this); products_i */
                              /* = 2 iters_i + 1, or 2 iters_i when the predicted exit (opt.predict) */
                              /* skipped the confirming product; 3 per iteration for order = 3      */
    float ms_gather, ms_sign, ms_scatter, ms_total;
    double mu_trace[64];      /* bisection history: mu of step k                             */
    double ne_trace[64];      /* n_elec of step k (of the last iterate if the step ended early) */
    double ne_err_trace[64];  /* bound on |n_elec(converged) - ne_trace[k]| (0: converged)    */
    int32_t iter_trace[64];   /* Newton-Schulz iterations spent on step k                    */
    /* totals over ALL sign evaluations of the call (a bisection makes several) */
    int64_t tot_sum_iter_n3;  /* sum over evaluations of sum_iter_n3                         */
    int64_t tot_sym_flop;     /* sum over executed symmetric products of n_i^2 (n_i + 1)     */
    int32_t tot_gemm_launches;
    int32_t tot_evaluations;
    float tot_ms_gather, tot_ms_sign;
    double spec_lo, spec_hi;  /* scaling = 1: the widened Lanczos estimate of [lambda_min, lambda_max] */
                              /* of K~ the interlacing bound was taken from (else 0, 0)       */
    double bracket_lo, bracket_hi; /* sm_density_matrix: the initial bisection bracket        */
    double mu_guess;          /* sm_density_matrix: the quadrature estimate (NaN if not computed) */
    int32_t exits_predicted;  /* last evaluation: submatrices that left by the predicted exit (A9b) ... */
    int32_t exits_two_step;   /* ... and by the two-step exit (A9c); the rest met eps on a computed residual */
    float ms_gemm;            /* timing on: CUDA-event time of the Newton-Schulz PRODUCT launches of the last  */
                              /* evaluation alone (k_ns_gemm; event pairs around every launch), FP64 path      */
    float tot_ms_gemm;        /* ... summed over the evaluations of the call                                 */
} sm_stats_t;

/*
 * sm_plan_create -- device BSR container + submatrix index builder ("a principal
 * submatrix a_i is assembled by removing all rows and columns j where A_{j,i} = 0"; per block
 * column L196; per group of block columns L199; global sorted pattern L180).
 * For every group G_i it forms on the GPU S_i = ascending union of the row blocks of its columns,
 * n_i = sum of their sizes, the local offsets, and the position of every generating column in
 * S_i; then sizes the padded batched workspace and the GEMM tile lists.
 *   nb, blk_size[nb], colptr[nb+1], rowidx[nnzb]   host, copied
 *   ngroups, grp_ptr[ngroups+1], grp_cols[nb]       host, copied
 *   opt                                             host or NULL
 *   cuda_stream                                     cudaStream_t (NULL = default stream)
 * Returns SM_OK and *plan, or <0 and *plan == NULL.
 */
sm_status_t sm_plan_create(sm_plan_t** plan, int32_t nb, const int32_t* blk_size,
                           const int64_t* colptr, const int32_t* rowidx, int32_t ngroups,
                           const int32_t* grp_ptr, const int32_t* grp_cols, const sm_options_t* opt,
                           void* cuda_stream);

/*
 * sm_partition_groups -- the load balancer of PAPER.md IV-E (L235): "a greedy algorithm to assign submatrices
 * to ranks such that they have similar load ... one consecutive chunk of submatrices to each rank ... expected
 * number of floating-point operations assuming that processing a submatrix takes O(n^3) FLOP and assigns
 * submatrices to ranks as long as their load is expected to be lower than FLOP_total / #ranks.  Additionally,
 * we make sure that each rank obtains at least one submatrix."  Reading A19: rank r takes the next submatrix
 * while its load so far is below sum n^3 / world AND enough submatrices remain to give every later rank one;
 * the last rank takes what is left.  Host only (no GPU needed): sub_dim[ngroups] host, first[world + 1] host
 * out (rank r owns groups first[r] .. first[r+1] - 1).  world > ngroups is an error.
 */
sm_status_t sm_partition_groups(int32_t ngroups, const int32_t* sub_dim, int32_t world, int32_t* first);

/*
 * Sum over the ranks for a sharded plan (opt.shard_world > 1): fn(ctx, vals, n) must replace vals[0..n) by
 * their sums over all ranks (host doubles; called from the calling thread after a stream synchronisation,
 * the same number of times on every rank: once per sign evaluation / mu step).  The Python binding passes
 * a torch.distributed all_reduce.  NULL fn: counts stay local.
 */
typedef void (*sm_allreduce_fn)(void* ctx, double* vals, int32_t n);
sm_status_t sm_plan_set_allreduce(sm_plan_t* plan, sm_allreduce_fn fn, void* ctx);

/* Plan facts, including the workspace size. */
sm_status_t sm_plan_query(const sm_plan_t* plan, sm_plan_info_t* out);

/*
 * Host copies of the index the GPU built, for bit-exact parity checks (any pointer may be NULL):
 *   sub_ptr[ngroups+1] (int64)   exclusive prefix sum of |S_i|
 *   sub_blocks[sum|S_i|]         members of S_i, ascending
 *   sub_off[sum|S_i|]            element offset of each member inside a_i
 *   sub_dim[ngroups]             n_i
 *   gen_pos[nb]                  for grp_cols[g]: its position inside S_i
 */
sm_status_t sm_plan_export_index(const sm_plan_t* plan, int64_t* sub_ptr, int32_t* sub_blocks,
                                 int32_t* sub_off, int32_t* sub_dim, int32_t* gen_pos);

/*
 * sm_sign_execute -- the three steps of the method at a fixed mu (Eq.(16)):
 * gather a_i - mu I into the batched dense workspace, X0 = (a_i - mu I)/s_i with a Gershgorin
 * bound s_i, Newton-Schulz X <- 1/2 X (3I - X^2) (Eq.(11)) until ||X^2 - I||_F/sqrt(n_i) < eps
 * (involutority criterion, L354/Fig.13), then D~[r,c] = 1/2 (delta_rc I - X[loc r, loc c]) for
 * the generating columns.
 *   d_vals_in [nnz]  device, K~ values            d_vals_out [nnz] device, D~ values (may be NULL:
 *   mu, eps          scalars                                         only stats->n_elec is produced)
 *   d_workspace      device, >= workspace_bytes, 256-byte aligned; contents are scratch
 * Returns SM_OK, SM_WARN_SIGN_NOT_CONVERGED, or <0.
 */
sm_status_t sm_sign_execute(sm_plan_t* plan, const double* d_vals_in, double mu, double eps,
                            double* d_vals_out, void* d_workspace, size_t workspace_bytes,
                            sm_stats_t* stats, void* cuda_stream);

/* Same with HOST value arrays (pageable or pinned): copies h_vals_in to the device, runs
 * sm_sign_execute, copies D~ back.  The staging buffers are owned by the plan. */
sm_status_t sm_sign_execute_host(sm_plan_t* plan, const double* h_vals_in, double mu, double eps,
                                 double* h_vals_out, void* d_workspace, size_t workspace_bytes,
                                 sm_stats_t* stats, void* cuda_stream);

/*
 * sm_density_matrix -- canonical ensemble (PAPER.md IV-G, L259-266, Algorithm 1):
 * adjust mu until n_elec(mu) = sum_i sum_{k in gen(i)} 1/2 (1 - sign(a_i - mu I)_kk) matches
 * n_target, "using a simple bisection" (L266).  Newton-Schulz keeps no eigendecomposition, so
 * every step re-evaluates the sign function (the cost L266 warns about).
 * Rule (reading A11): step 0 evaluates *mu_inout; then midpoint bisection inside the
 * Gershgorin interval of K~ (n_elec = 0 below, = n_basis above; intersected with the interlacing
 * interval of K~'s extreme eigenvalues when scaling = 1; reported in stats->bracket_lo/hi), raising
 * mu if n_elec < n_target.  With opt.mu_guess (reading A11d) the step after step 0 goes to
 * stats->mu_guess instead of the midpoint when that lies strictly inside the bracket; with
 * opt.mu_start (reading A11e) step 0 itself goes there unless *mu_inout lies inside the Ritz
 * interval the estimate was taken from.
 * Stops when |n_elec - n_target| <= tol_n (SM_OK), or when the bracket is narrower than
 * opt.mu_tol or after opt.max_mu_steps evaluations (SM_WARN_MU_NOT_CONVERGED); returns in
 * *mu_inout the evaluated mu with the smallest |n_elec - n_target| and in d_vals_out D~ at that mu.
 */
sm_status_t sm_density_matrix(sm_plan_t* plan, const double* d_vals_in, double n_target,
                              double tol_n, double eps, double* mu_inout, double* d_vals_out,
                              void* d_workspace, size_t workspace_bytes, sm_stats_t* stats,
                              void* cuda_stream);

/* Host-buffer variant of sm_density_matrix (H2D of K~ and D2H of D~ inside the call). */
sm_status_t sm_density_matrix_host(sm_plan_t* plan, const double* h_vals_in, double n_target,
                                   double tol_n, double eps, double* mu_inout, double* h_vals_out,
                                   void* d_workspace, size_t workspace_bytes, sm_stats_t* stats,
                                   void* cuda_stream);

/*
 * Eigendecomposition path, SURVEY 8(f)1 (PAPER.md IV-F Eq.(17), IV-G Algorithm 1; any plan, whatever
 * opt.method says; sm_sign_execute / sm_density_matrix call these when opt.method = 1):
 *   sm_eig_decompose  gathers a_i (mu = 0) and computes a_i = Q Lambda Q^T for every submatrix by one-sided
 *                     Jacobi rotations on the GPU; Q stays in the workspace (second buffer), lambda_il and
 *                     the weights w_il = sum_{k in gen(i)} Q_kl^2 of Algorithm 1 (L270, L275) in the plan.
 *                     stats (may be NULL): iter_min / iter_max = Jacobi sweeps, not_converged.
 *                     Returns SM_OK or SM_WARN_SIGN_NOT_CONVERGED (a submatrix hit the sweep cap).
 *   sm_eig_export     host copies of what Algorithm 1 keeps: ptr[ngroups+1] (prefix of n_i), lam[sum n_i],
 *                     w[sum n_i] (order inside a submatrix unspecified); any pointer may be NULL.
 *   sm_eig_nelec      n_elec(mu) = sum_i sum_l w_il f(lambda_il - mu), f = 1/2 (1 - signum) for kT = 0 or the
 *                     Fermi function (L255): one step of Algorithm 1's loop, no decomposition.
 *   sm_eig_density    D~ = Q f(Lambda - mu) Q^T on the generating columns -> d_vals_out (same workspace as
 *                     the sm_eig_decompose call, untouched in between).
 */
sm_status_t sm_eig_decompose(sm_plan_t* plan, const double* d_vals_in, void* d_workspace,
                             size_t workspace_bytes, sm_stats_t* stats, void* cuda_stream);
sm_status_t sm_eig_export(const sm_plan_t* plan, int64_t* ptr, double* lam, double* w);
sm_status_t sm_eig_nelec(sm_plan_t* plan, double mu, double kT, double* n_elec, void* cuda_stream);
sm_status_t sm_eig_density(sm_plan_t* plan, double mu, double kT, double* d_vals_out, void* d_workspace,
                           size_t workspace_bytes, void* cuda_stream);

/*
 * sm_trace_dk -- tr(D) (Eq.(18)) and the band-structure energy tr(D K) (Eq.(10)) of two
 * value arrays on the plan's pattern: tr(DK) = sum over stored elements D o K (K symmetric).
 * d_D, d_K device [nnz]; tr_D, tr_DK host doubles.  Deterministic two-stage reduction.
 */
sm_status_t sm_trace_dk(sm_plan_t* plan, const double* d_D, const double* d_K, double* tr_D,
                        double* tr_DK, void* cuda_stream);

/*
 * sm_trace_dk_static -- the band-structure energy tr(D K) (Eq.(10)) = sum over stored elements D o K, for
 * callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  No plan; calls no cudaMalloc / cudaFree / allocating routine, and no synchronisation: everything is
 * enqueued on `cuda_stream`.
 *   nnz      number of stored values, 0 <= nnz <= SM_STATIC_MAX_NNZ; more is rejected with SM_ERR_INVALID_ARG
 *            (text in sm_last_cuda_error); use sm_trace_dk there.
 *   d_D, d_K DEVICE [nnz], read only (may be NULL if nnz == 0);  d_tr_DK DEVICE [1], written on the stream.
 * Scratch: a file-scope __device__ array of 512 KB + 256 B inside the library (one partial sum per 4096 values
 * and a ticket counter), held by every GPU that loads the library until the process exits.  ALL calls share it
 * and it keeps the last call's contents (the call clears what must start at zero): calls on one stream are
 * ordered and safe; calls whose kernels overlap on the GPU (other streams / threads) RACE -- serialise them.
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress, that device current);
 * make that first call outside a graph capture.  Deterministic (fixed summation order, independent of the grid).
 * Errors: SM_ERR_INVALID_ARG (negative / too large nnz, NULL pointer), SM_ERR_CUDA.
 */
#define SM_STATIC_MAX_NNZ 268435456LL
sm_status_t sm_trace_dk_static(int64_t nnz, const double* d_D, const double* d_K, double* d_tr_DK,
                               void* cuda_stream);

/*
 * Phase entry points used by the tests and the roofline benchmark (same kernels as above):
 *   sm_gather   : workspace X buffer <- a_i - mu I (rows / columns n_i .. ld_i - 1 zero: a fixed point of
 *                 the iteration); also the Gershgorin bounds (plain Gershgorin scaling, whatever the
 *                 previous call used)
 *   sm_scatter  : d_vals_out <- 1/2 (delta - xscale_i * X) from the workspace X buffer written by
 *                 the last sm_gather / sign evaluation; f = identity round trip when as_identity=1:
 *                 d_vals_out <- X (i.e. gather then scatter returns K~ - mu I on the pattern)
 *   sm_sign_iterate : run the Newton-Schulz loop on the gathered workspace
 */
sm_status_t sm_gather(sm_plan_t* plan, const double* d_vals_in, double mu, void* d_workspace,
                      size_t workspace_bytes, void* cuda_stream);
sm_status_t sm_sign_iterate(sm_plan_t* plan, double eps, void* d_workspace, size_t workspace_bytes,
                            sm_stats_t* stats, void* cuda_stream);
sm_status_t sm_scatter(sm_plan_t* plan, int32_t as_identity, double* d_vals_out, void* d_workspace,
                       size_t workspace_bytes, void* cuda_stream);

/*
 * sm_measure_peaks -- the roofline denominators of this library measured on the current device, for
 * bench.py (diagnostic; allocates and frees 2 GiB of device memory; ~50 ms):
 *   dmma_tflops  issue rate of mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the FP64 tensor-core instruction of
 *                the Newton-Schulz kernel) with register-resident operands, 16 warps per SM, 16
 *                independent accumulators per warp, best of 5
 *   hbm_copy_gbs read + write bytes per second of a 16-byte grid-stride copy of 1 GiB, best of 5
 */
typedef struct {
    double dmma_tflops, hbm_copy_gbs;
    double ms_dmma, ms_copy;
    int32_t num_sms, reserved;
} sm_peaks_t;
sm_status_t sm_measure_peaks(sm_peaks_t* out, void* cuda_stream);

/* Enable (1) / disable (0) per-phase CUDA-event timing into sm_stats_t (adds stream syncs). */
sm_status_t sm_set_timing(sm_plan_t* plan, int32_t enable);

/* Number of kernels this plan has launched since creation (for bench.py's gpu_launches). */
int64_t sm_launch_count(const sm_plan_t* plan);

void sm_plan_destroy(sm_plan_t* plan);
const char* sm_strerror(sm_status_t status);
/* Text of the last CUDA error seen by this library on the calling THREAD ("" if none). */
const char* sm_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SUBMATRIX_B200_H */
