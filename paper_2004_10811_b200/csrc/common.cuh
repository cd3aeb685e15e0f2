// Internal declarations of libsubmatrix_b200.so (sm_100a).  Not part of the C-ABI; the boundary
// is include/submatrix.h.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <vector>

#include "submatrix.h"

namespace smb {

constexpr int TILE = 64;        // CTA tile edge of the Newton-Schulz GEMMs
constexpr int LD_ALIGN = 8;     // padded leading dimension granularity (one DMMA k-step pair)

// One CTA tile of one submatrix: lower-triangular tile (ti >= tj) of a symmetric product, with
// the geometry of its submatrix inlined so that a CTA needs a single 32-byte load to start.
struct __align__(16) TileDesc {
    int64_t ws_off;      // offset (doubles) of the submatrix in each workspace buffer
    int32_t grp;         // submatrix (= generating group) index
    int32_t ld;          // padded leading dimension
    int32_t n;           // true dimension
    int32_t tij;         // ti | (tj << 16)
    int32_t tile_first;  // first tile of this submatrix in the tile list
    int32_t tile_count;  // number of tiles of this submatrix
};

// Workspace layout of one symmetric ld x ld matrix ("k8-panel" layout): rows are grouped in
// row-tiles of 64 (the last one holds rows_t = ld - 64 t rows); inside a row-tile the data is a
// sequence of panels, panel kp = the 8 consecutive columns 8 kp .. 8 kp + 7 of all rows_t rows,
// row-major (64 bytes per row).  The operand slice (64 rows x 16 k) that one pipeline stage of the
// Newton-Schulz GEMM needs is therefore ONE contiguous block of rows_t * 128 bytes -- a single
// cp.async.bulk -- and its dense 64-byte rows are bank-conflict-free for the 16-byte fragment loads.
// ld is a multiple of 8, the matrix occupies exactly ld * ld doubles.
__host__ __device__ __forceinline__ size_t panel_off(int r, int c, int ld) {
    const int t0 = r & ~63;
    const int rows_t = (ld - t0) < 64 ? (ld - t0) : 64;
    return (size_t)t0 * ld + (size_t)(c >> 3) * rows_t * 8 + (size_t)((r & 63) * 8 + (c & 7));
}

constexpr int THIN_MAX_ROWS = 16;  // generating-row span served by the thin last update (k_ns_thin, ns_sign.cu) ...
// ... or n / 16 if that is more: a thin product costs (span / 8) passes over n^2 values at HBM speed, a full one n^3
// multiply-adds at the FP64 rate, so the larger the submatrix, the more generating rows the thin form can carry
__host__ __device__ __forceinline__ bool thin_span_ok(int span, int n) {
    return span <= (THIN_MAX_ROWS > n / 16 ? THIN_MAX_ROWS : n / 16);
}

void set_cuda_error(cudaError_t e, const char* where);
void set_error_text(const char* msg);

// Frees a temporary device buffer on every return path.
struct DevTmp {
    void* p = nullptr;
    ~DevTmp() { if (p) cudaFree(p); }
};

#define SM_CUDA(call)                                        \
    do {                                                     \
        cudaError_t e__ = (call);                            \
        if (e__ != cudaSuccess) {                            \
            smb::set_cuda_error(e__, #call);                 \
            return SM_ERR_CUDA;                              \
        }                                                    \
    } while (0)

}  // namespace smb

// The plan: device BSR container (a1) + submatrix index (a2) + workspace/tile tables.
struct sm_plan {
    sm_options_t opt;
    sm_plan_info_t info;
    int32_t nb = 0, ngroups = 0;
    int64_t nnzb = 0, nnz = 0;
    int32_t max_sub_blocks = 0;  // max |S_i|
    // --- host copies
    std::vector<int32_t> h_blk_size, h_rowidx, h_grp_ptr, h_grp_cols, h_sub_dim, h_ld;
    std::vector<int64_t> h_colptr, h_sub_ptr, h_ws_off;
    std::vector<int32_t> h_tile_first, h_tile_count;
    // --- device: pattern
    int32_t *d_blk_size = nullptr, *d_blk_off = nullptr, *d_rowidx = nullptr;
    int64_t *d_colptr = nullptr, *d_val_off = nullptr;
    int32_t *d_grp_ptr = nullptr, *d_grp_cols = nullptr, *d_col_grp = nullptr;
    // --- device: submatrix index
    int64_t* d_sub_ptr = nullptr;
    int32_t *d_sub_blocks = nullptr, *d_sub_off = nullptr, *d_sub_dim = nullptr, *d_gen_pos = nullptr;
    int32_t *d_gen_off = nullptr;  // [nb]  element offset of column c inside its group's submatrix
    uint32_t *d_blk_pack = nullptr;// [nnzb] block (r,c): element row offset inside c's group's submatrix (low 20
                                   //        bits) | height blk_size[r] (high 12 bits)
    int32_t *d_gen_width = nullptr;// [ngroups] generating basis functions per group
    int2* d_gen_rng = nullptr;     // [ngroups] first / last generating row of a_i
    std::vector<int32_t> h_gen_rng;   // host copy (2 per group)
    std::vector<int64_t> h_final_flop;  // flop of a last update restricted to the generating rows' tiles
    // --- device: workspace geometry and tiles
    int64_t* d_ws_off = nullptr;   // [ngroups] offset (doubles) of submatrix i in each buffer
    int32_t* d_ld = nullptr;       // [ngroups] padded leading dimension
    smb::TileDesc* d_tiles = nullptr;
    int32_t *d_tile_first = nullptr, *d_tile_count = nullptr;
    int64_t n_tiles = 0, sum_ld2 = 0;
    // --- device: per-evaluation state
    int32_t* d_done_iter = nullptr;        // [ngroups] -1 = active, else iteration at which it stopped
    int32_t* d_flag = nullptr;             // [ngroups] 0 converged, 1 stagnated / max_iter
    double* d_res = nullptr;               // [2][ngroups] residual history (ping-pong)
    unsigned long long* d_gersh = nullptr; // [2][ngroups] bits of the Gershgorin bound | of the largest squared column norm (atomicMax)
    double* d_partials = nullptr;          // [n_tiles][4] per-tile, per-consumer-warp residual partials
    int32_t* d_counters = nullptr;         // [max_iter+2] still-active submatrices after iteration k
    int32_t* d_act = nullptr;              // [4][n_tiles] work lists of the GEMM launches (ns_sign.cu)
    int32_t* d_act_cnt = nullptr;          // [2 (max_iter + 3)] their lengths, then 4 x [max_iter + 3]: lengths of the thin, speculation, speculation-tile and thin3 lists
    int32_t* d_thin_list = nullptr;        // [4][ngroups]: 0, 1 submatrices whose last update is the thin product (k_ns_thin); 2 speculated, 3 certified (two-step exit)
    size_t thin_smem = 0;                  // 8 rows of the largest submatrix; 0: thin path off (too large)
    int thin_attr_set = 0;
    int32_t* d_spec_tiles = nullptr;       // [n_tiles] work list of the MODE 4 launch (two-step exit, ns_sign.cu)
    int32_t* d_spec_stat = nullptr;        // [2] certified / failed speculations since plan creation
    size_t thin3_smem = 0;                 // 2 x 8 rows of the largest submatrix; 0: two-step exit off
    int thin3_attr_set = 0;
    int32_t h_spec_prev[2] = {0, 0};       // totals of d_spec_stat at the previous evaluation's end
    int spec_pause = 0;                    // evaluations left during which the two-step exit is not tried (it kept failing)
    int32_t* d_sched = nullptr;            // [2*(max_iter+2)] work counters of the persistent GEMM launches
    double* d_ne_part = nullptr;           // [ngroups] per-group electron-count partials
    double* d_scalars = nullptr;           // [8] n_elec, tr D, tr DK, gersh lo/hi
    double* d_red = nullptr;               // [2*4096] reduction scratch
    int32_t* h_pinned = nullptr;           // pinned host mirror for counters
    double* h_pinned_d = nullptr;          // pinned host scalars
    double* d_gg = nullptr;                // [2 nb] per-column Gershgorin ends of k_gersh_global (allocated on first use)
    unsigned char* h_stats = nullptr;      // pinned mirror of done_iter / flag / res for collect_stats (first use)
    int last_eval_iters = 0;               // iterations the last converged evaluation took (sizes the enqueue-ahead batch)
    int cur_k = 0;                         // completed Newton-Schulz updates of the last evaluation
    int half_iter = 0;                     // 1: MODE 0 of iteration cur_k ran, its MODE 1 did not (steering stop)
    double* d_bound = nullptr;             // [max_iter+2][2] per iteration: n_elec(X_k), its error bound
    double* d_bound_part = nullptr;        // [2][nb] per-block-column partials of the two
    double* h_bound = nullptr;             // pinned mirror of d_bound
    // --- reduced-precision path (precision = 1, ns_tf32.cu)
    void* d_tiles32 = nullptr;
    int64_t* d_ws_off32 = nullptr;
    int32_t *d_tile_first32 = nullptr, *d_tile_count32 = nullptr;
    double* d_partials32 = nullptr;
    int64_t n_tiles32 = 0, sum_ldp2 = 0;
    int32_t* d_ctrl = nullptr;             // [8] + doubles: device-side stop decision of an evaluation (EvalCtrl)
    void* h_ctrl = nullptr;                // pinned mirror
    int64_t* d_gl_ptr = nullptr;           // gather list (built by the first gather): extents per member column
    uint32_t* d_gl = nullptr;              //   entries: member index << 16 | value offset inside the block column
    int gather_no_list = 0;
    uint32_t* d_src_map = nullptr;         // [nnz] scatter source map (built by the first scatter)
    int4* d_col_rec = nullptr;             // [nb] scatter column records (first value lo/hi, value count, group)
    int scatter_chunks = 1;
    double* d_lz = nullptr;                // Lanczos vectors / tridiagonal (spectral.cu), lazily allocated
    int64_t* d_col_val = nullptr;          // [nb + 1] offset of the first value of every block column
    uint32_t* d_lz_map = nullptr;          // [nnz] per stored value: index into x | dense column q << 28 (streaming mat-vec)
    int4* d_lz_rec = nullptr;              // [nnzb] per stored block: value offset (lo, hi), blk_off of its row, its height
    double lz_lo = 0.0, lz_hi = 0.0;       // estimated [lambda_min, lambda_max] of K~ (widened)
    double* d_alpha = nullptr;             // [2][ngroups] rescaling factor alpha_k of iteration k (slot k & 1), reading A8b
    int resc_eval = 0;                     // this evaluation runs the rescaled iteration (A8b)
    double* d_lmin = nullptr;              // [ngroups] tracked lower bound l_k of the schedule
    double* h_lz = nullptr;                // pinned [66]: lo, hi, Ritz values [32], cumulative quadrature weights [32]
    int lz_nodes = 0;
    int lz_grid = 0;                       // CTAs of the cooperative Lanczos launch
    int lz_valid = 0;                      // lz_lo / lz_hi belong to the current call's values
    int lz_ok = 0;                         // the run did not break down: cap, bracket and quadrature may be used
    int ns_attr_set = 0, tf32_attr_set = 0;  // dynamic shared-memory opt-in done on this plan's device
    // --- eigendecomposition path (eig.cu, option method = 1)
    int64_t* d_eig_ptr = nullptr;          // [ngroups + 1] prefix of n_i
    double *d_eig_lam = nullptr, *d_eig_w = nullptr;  // [sum n_i] eigenvalues, weights of Algorithm 1
    double* d_eig_sigma = nullptr;         // [ngroups] shift of B = a_i + sigma I
    int32_t* d_eig_order = nullptr;        // [ngroups] processing order, largest first
    int32_t* d_eig_state = nullptr;        // [2 ngroups + 2] sweeps, flags, work counter
    int64_t eig_total = 0;
    int eig_battr_set = 0, eig_valid = 0;
    // --- sharding: the plan holds only its own chunk of groups
    sm_allreduce_fn allreduce = nullptr;
    void* allreduce_ctx = nullptr;
    // --- staging for the *_host entry points
    double *d_stage_in = nullptr, *d_stage_out = nullptr;
    // --- misc
    int timing = 0;
    float ms_index_kernels = 0.f;          // CUDA-event time of the index-builder kernels (plan creation)
    int64_t launches = 0;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_iter[2] = {nullptr, nullptr};
    std::vector<cudaEvent_t> ev_gemm;      // timing: event pairs around the Newton-Schulz GEMM launches of an evaluation
    int ev_gemm_n = 0;
    int gather_warps = 8, gather_tile_ld = 0, gather_msb = 2, gather_split = 1;
    int gather_hash_size = 32, gather_hash_shift = 27, gather_mpad = 4, gather_mc = 2, gather_map16 = 0;
    int32_t max_col_blocks = 0;  // longest block column
    size_t gather_smem = 0;
    int num_sms = 148;
};

namespace smb {
// plan.cu
sm_status_t build_index_device(sm_plan* p, cudaStream_t st);
sm_status_t launch_excl_scan(const int32_t* in, int64_t n, int64_t* out, cudaStream_t st);  // out[n + 1], one CTA
// gather_scatter.cu
sm_status_t launch_gather(sm_plan* p, const double* vals, double mu, double* X, cudaStream_t st);
sm_status_t launch_scatter(sm_plan* p, int as_identity, const double* buf0, const double* buf1,
                           double* out, cudaStream_t st);
sm_status_t launch_nelec(sm_plan* p, const double* buf0, const double* buf1, cudaStream_t st);
sm_status_t launch_trace_dk(sm_plan* p, const double* D, const double* K, cudaStream_t st);
sm_status_t launch_gersh_global(sm_plan* p, const double* vals, cudaStream_t st);
sm_status_t launch_nelec_bound(sm_plan* p, int k, const double* buf0, const double* buf1, const double* bufY,
                               cudaStream_t st);
// ns_tf32.cu
sm_status_t build_tf32_tables(sm_plan* p, cudaStream_t st);
sm_status_t launch_to_f32(sm_plan* p, const double* buf0, double* buf1, cudaStream_t st);
sm_status_t launch_to_f64(sm_plan* p, double* buf0, const double* buf1, const double* bufY, cudaStream_t st);
sm_status_t launch_ns_pair_tf32(sm_plan* p, int k, double eps, int decide_only, double* buf0, double* buf1,
                                double* bufY, cudaStream_t st, int which);
// Device-side control block of one sign evaluation: set by k_eval_ctrl after the decision (and the
// steering bound) of iteration k; once stop != 0 every later launch of the evaluation is empty, so the
// host can enqueue iterations ahead without synchronising after each of them.
struct EvalCtrl {
    int32_t stop;      // 0 running, 1 all submatrices stopped, 2 steering decision (A11c)
    int32_t k_stop;    // iteration at which it was set
    int32_t decided;   // +1 / -1: n_elec proven above / below the target
    int32_t steer_off; // 1: |n_elec(X_k) - target| + bound < margin / 2 was seen: the final count is proven to lie
                       // inside the margin, no later iteration can prove a direction -- the bound is not evaluated again
    double ne, err;    // n_elec(X_k) and its bound at the decision
};
sm_status_t launch_eval_ctrl(sm_plan* p, int k, int steer, double n_target, double margin, cudaStream_t st);
// eig.cu
sm_status_t launch_eig_decompose(sm_plan* p, const double* vals, double* buf0, double* buf1, cudaStream_t st);
sm_status_t launch_eig_nelec(sm_plan* p, double mu, double kT, cudaStream_t st);
sm_status_t launch_eig_bjacobi(sm_plan* p, double* G, cudaStream_t st);  // eig_block.cu
sm_status_t launch_eig_density(sm_plan* p, double mu, double kT, double* buf0, const double* buf1, cudaStream_t st);
// spectral.cu
sm_status_t launch_lanczos_bounds(sm_plan* p, const double* vals, cudaStream_t st);
sm_status_t launch_apply_scale(sm_plan* p, double cap, double overshoot, double ell_abs, cudaStream_t st);
inline bool rescale_on(const sm_plan* p) { return p->resc_eval != 0; }  // set per evaluation by apply_scaling
// ns_sign.cu
sm_status_t launch_ns_pair(sm_plan* p, int k, double eps, int decide_only, double* buf0, double* buf1,
                           double* bufY, cudaStream_t st, int which = 3, double* bufW = nullptr);
}  // namespace smb
