// batched symmetric eigendecomposition of the submatrices + Algorithm 1 as written
// (PAPER.md IV-F Eq.(17), IV-G L259-278): a_i = Q Lambda Q^T once per call, then the mu loop
// runs on (lambda_il, w_il = sum_{k in gen(i)} Q_kl^2) alone -- "without recomputing the sign function
// or the eigendecomposition in each step" (L266) -- and the result is Q f(Lambda - mu) Q^T restricted
// to the generating columns, f = signum (Eq.(17)) or the Fermi function (L255, reading A18).
//
// Eigensolver: one-sided (Hestenes) Jacobi on B = a_i + sigma I, sigma = 1.5 x the Gershgorin bound, so
// that B is positive definite with condition number < 5.  Plane rotations from the right make the
// columns of G (G_0 = B) mutually orthogonal: G = B V with V orthogonal, and at convergence
// G^T G = V^T B^2 V is diagonal, i.e. the columns of V are eigenvectors of B^2, hence of B (all
// eigenvalues positive and B symmetric), and G = V Lambda_B.  So  lambda_l(a_i) = ||g_l|| - sigma  and
// q_l = g_l / ||g_l||: V is never accumulated, one n x n array per submatrix.
//
// Mapping: one persistent CTA per submatrix at a time, G column-major in the workspace (L2-resident: the
// working set is one matrix per SM).  Columns are processed in blocks of <= 16: a visit loads two
// blocks into shared memory, orthogonalises all cross pairs (16 rounds of 16 disjoint pairs, one warp
// per pair, columns cached in registers, dot products by warp shuffles) and stores them; block pairs follow
// a round-robin tournament, pairs inside a block are done once per sweep in a visit of their own.
// A sweep without a rotation ends the iteration (|g_p . g_q| <= tol ||g_p|| ||g_q|| for every pair).
#include "common.cuh"

namespace smb {

#ifndef EJ_MINB
#define EJ_MINB 2
#endif
constexpr int EJ_THREADS = 512;  // 16 warps
constexpr int EJ_MAXB = 16;      // columns per block (8 / 4 for very large submatrices: shared-memory budget)

struct EigArgs {
    const int32_t* sub_dim;
    const int32_t* ldv;
    const int64_t* ws_off;
    double* G;                 // column-major n_i x n_i, column stride ld_i, at ws_off[i]
    const double* sigma;       // [ngroups] shift
    const int32_t* order;      // processing order (largest first)
    int32_t* counter;          // work counter
    int32_t* sweeps;           // [ngroups] out
    int32_t* eflag;            // [ngroups] out: 1 = not converged in max_sweeps
    const int32_t* grp_ptr;
    const int32_t* grp_cols;
    const int32_t* gen_off;
    const int32_t* blk_size;
    const int64_t* eig_ptr;    // [ngroups + 1] prefix of n_i
    double* lam;               // [sum n_i]
    double* w;                 // [sum n_i]
    int ngroups, max_sweeps, bcols, smem_rows;
};

// Rotation of a column pair: tangent t of the angle that makes x' . y' vanish (root of t^2 + 2 zeta t - 1,
// zeta = (|y|^2 - |x|^2) / (2 x.y)), c = 1/sqrt(1 + t^2), s = c t.  t is formed in FP32 (relative error 1e-7:
// the pair is then orthogonal to 1e-7 of its former inner product instead of exactly, which the next sweep
// removes; the stop test is taken on FP64 inner products), c by an FP32 seed and two Newton steps in FP64,
// so that c^2 + s^2 = 1 to FP64 rounding: V stays orthogonal.  ~20 FP64 instructions instead of a FP64
// division, square root and reciprocal square root (~150), which bounded the first version of this kernel.
__device__ __forceinline__ void rotation(double a, double b, double g, double& c, double& s, double& t) {
    // fast FP32 intrinsics (2 ulp): the tangent only has to be good to ~1e-6
    const float zf = __fdividef((float)(b - a), 2.0f * (float)g);
    const float az = fabsf(zf);
    float tf = az < 1e15f ? __frcp_rn(az + __fsqrt_rn(fmaf(az, az, 1.0f))) : __fdividef(0.5f, az);
    tf = zf >= 0.0f ? tf : -tf;
    t = (double)tf;
    const double x = fma(t, t, 1.0);
    double y = (double)rsqrtf((float)x);
    y = y * fma(-0.5 * x, y * y, 1.5);
    y = y * fma(-0.5 * x, y * y, 1.5);
    c = y;
    s = y * t;
}

// One visit of the column pair (x, y) held in shared memory (stride-1 columns; x, y already point at this
// lane's first row; padding rows are zero and stay zero).  nx, ny: the squared norms of the two columns, kept
// in shared memory per column slot, refreshed when a block is loaded and updated here in closed form.
// NR > 0: the columns have exactly 32 NR rows and pass through registers; NR = 0: `rows` rows, two sweeps over
// shared memory.  Returns 1 if the pair was rotated.
template <int NR>
__device__ __forceinline__ int rotate_pair(double* __restrict__ x, double* __restrict__ y, double* nx, double* ny,
                                           int rows, int lane, double tol2) {
    constexpr int NRR = NR > 0 ? NR : 1;
    double xr[NRR], yr[NRR];
    double g = 0.0;
    if (NR > 0) {
#pragma unroll
        for (int j = 0; j < NRR; ++j) {
            xr[j] = x[32 * j];
            yr[j] = y[32 * j];
            g = fma(xr[j], yr[j], g);
        }
    } else {
        for (int r = lane; r < rows; r += 32) g = fma(x[r - lane], y[r - lane], g);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) g += __shfl_xor_sync(0xffffffffu, g, o);
    const double a = *nx, b = *ny;
    if (!(g * g > tol2 * a * b)) return 0;  // orthogonal to working precision (also a zero column, NaN)
    double c, s, t;
    rotation(a, b, g, c, s, t);
    if (NR > 0) {
#pragma unroll
        for (int j = 0; j < NRR; ++j) {
            x[32 * j] = c * xr[j] - s * yr[j];
            y[32 * j] = s * xr[j] + c * yr[j];
        }
    } else {
        for (int r = lane; r < rows; r += 32) {
            const double xv = x[r - lane], yv = y[r - lane];
            x[r - lane] = c * xv - s * yv;
            y[r - lane] = s * xv + c * yv;
        }
    }
    __syncwarp();
    if (lane == 0) {  // |x'|^2 = c^2 (a - 2 t g + t^2 b), |y'|^2 = c^2 (t^2 a + 2 t g + b): valid for any t
        const double c2 = c * c, tg = 2.0 * t * g, t2 = t * t;
        *nx = c2 * (a - tg + t2 * b);
        *ny = c2 * (fma(t2, a, tg) + b);
    }
    return 1;
}

// Squared norms of the columns in slots s0 .. s0 + w - 1 (one warp per column), from scratch.
__device__ __forceinline__ void block_norms(const double* __restrict__ sm, int rows, int s0, int w, double* __restrict__ nrm2) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int c = wid; c < w; c += nw) {
        const double* col = sm + (size_t)(s0 + c) * rows;
        double a = 0.0;
        for (int r = lane; r < rows; r += 32) a = fma(col[r], col[r], a);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (lane == 0) nrm2[s0 + c] = a;
    }
}

// Copy `w` columns (first column c0) of G between global memory and the shared slots s0 .. s0 + w - 1:
// one warp per column, 16 bytes per lane.
template <bool LOAD>
__device__ __forceinline__ void move_block(double* __restrict__ Gm, int ld, int nr2, double* __restrict__ sm, int rows,
                                           int c0, int w, int s0) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int per = nr2 >> 1;  // double2 per column
    for (int c = wid; c < w; c += nw) {
        double2* g = reinterpret_cast<double2*>(Gm + (size_t)(c0 + c) * ld);
        double2* sp = reinterpret_cast<double2*>(sm + (size_t)(s0 + c) * rows);
        for (int r2 = lane; r2 < per; r2 += 32) {
            if (LOAD) sp[r2] = g[r2]; else g[r2] = sp[r2];
        }
    }
}

// All sweeps of one submatrix.  NR > 0: columns of exactly 32 NR rows, blocks of 16 columns, everything about
// the shared-memory geometry is a compile-time constant; NR = 0: run-time rows and block width.
// Returns the number of sweeps done; *converged says whether the last one was free of rotations.
template <int NR>
__device__ __noinline__ int jacobi_matrix(double* __restrict__ Gm, int n, int ld, double* __restrict__ sm,
                                          double* __restrict__ s_n2, int* s_rot, int rows_rt, int B_rt, int max_sweeps,
                                          int* converged) {
    const int rows = NR > 0 ? NR * 32 : rows_rt;
    const int B = NR > 0 ? EJ_MAXB : B_rt;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nr2 = min((n + 1) & ~1, ld);  // rows moved per column (even; ld is a multiple of 8)
    const double tol = 2.2e-16 * sqrt((double)max(n, 1));
    const double tol2 = tol * tol;
    for (int e = threadIdx.x; e < 2 * B * rows; e += blockDim.x) sm[e] = 0.0;  // padding rows stay zero
    const int nblk = (n + B - 1) / B;
    const int bw = nblk ? (n + nblk - 1) / nblk : 0;  // balanced block width (<= B)
    const int N = nblk + (nblk & 1);
    double* const sml = sm + lane;
    int sweep = 0;
    *converged = 0;
    for (; sweep < max_sweeps; ++sweep) {
        if (threadIdx.x == 0) *s_rot = 0;
        __syncthreads();
        int my_rot = 0;
        // ---- pairs inside one block
        for (int k = 0; k < nblk; ++k) {
            const int c0 = k * bw, wk = min(bw, n - c0);
            if (wk < 2) continue;
            move_block<true>(Gm, ld, nr2, sm, rows, c0, wk, 0);
            __syncthreads();
            block_norms(sm, rows, 0, wk, s_n2);
            __syncthreads();
            const int M = wk + (wk & 1);
            for (int r = 0; r < M - 1; ++r) {
                for (int q = wid; q < M / 2; q += nw) {
                    int a = r + q, b = r - q + (M - 1);
                    a = a >= M - 1 ? a - (M - 1) : a;
                    b = b >= M - 1 ? b - (M - 1) : b;
                    if (q == 0) { a = M - 1; b = r; }
                    if (a < wk && b < wk)
                        my_rot += rotate_pair<NR>(sml + a * rows, sml + b * rows, s_n2 + a, s_n2 + b, rows, lane, tol2);
                }
                __syncthreads();
            }
            move_block<false>(Gm, ld, nr2, sm, rows, c0, wk, 0);
            __syncthreads();
        }
        // ---- pairs across two blocks: round-robin tournament of the blocks
        for (int r = 0; r < N - 1; ++r) {
            for (int q = 0; q < N / 2; ++q) {
                int I = (q == 0) ? N - 1 : (r + q) % (N - 1);
                int J = (q == 0) ? r : (r - q + (N - 1)) % (N - 1);
                if (I >= nblk || J >= nblk) continue;  // the dummy of an odd block count
                const int ci = I * bw, cj = J * bw;
                const int wi = min(bw, n - ci), wj = min(bw, n - cj);
                move_block<true>(Gm, ld, nr2, sm, rows, ci, wi, 0);
                move_block<true>(Gm, ld, nr2, sm, rows, cj, wj, B);
                __syncthreads();
                block_norms(sm, rows, 0, wi, s_n2);
                block_norms(sm, rows, B, wj, s_n2);
                __syncthreads();
                for (int rr = 0; rr < B; ++rr) {
                    for (int a = wid; a < B; a += nw) {
                        int b = a + rr;
                        b = b >= B ? b - B : b;
                        if (a < wi && b < wj)
                            my_rot += rotate_pair<NR>(sml + a * rows, sml + (B + b) * rows, s_n2 + a, s_n2 + B + b, rows,
                                                      lane, tol2);
                    }
                    __syncthreads();
                }
                move_block<false>(Gm, ld, nr2, sm, rows, ci, wi, 0);
                move_block<false>(Gm, ld, nr2, sm, rows, cj, wj, B);
                __syncthreads();
            }
        }
        if (lane == 0 && my_rot) atomicAdd(s_rot, my_rot);
        __syncthreads();
        const int rot = *s_rot;
        __syncthreads();
        if (rot == 0) { *converged = 1; ++sweep; break; }
    }
    return sweep;
}

__global__ void __launch_bounds__(EJ_THREADS, EJ_MINB) k_eig_jacobi(const EigArgs A) {
    extern __shared__ __align__(16) double sm[];
    __shared__ int s_next, s_rot;
    __shared__ double s_n2[2 * EJ_MAXB];  // squared column norms of the loaded blocks
    __shared__ int s_genrow[1024];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (;;) {
        if (threadIdx.x == 0) s_next = atomicAdd(A.counter, 1);
        __syncthreads();
        const int it = s_next;
        __syncthreads();
        if (it >= A.ngroups) return;
        const int i = A.order[it];
        const int n = A.sub_dim[i], ld = A.ldv[i];
        double* Gm = A.G + A.ws_off[i];
        const int rows = (n + 31) & ~31;  // padded column length in shared memory
        int sweeps = 0, converged = 1;
        if (n > 1) {
            const int nr = (A.bcols == EJ_MAXB) ? rows >> 5 : 0;
            switch (nr) {
                case 1: sweeps = jacobi_matrix<1>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 2: sweeps = jacobi_matrix<2>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 3: sweeps = jacobi_matrix<3>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 4: sweeps = jacobi_matrix<4>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 5: sweeps = jacobi_matrix<5>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 6: sweeps = jacobi_matrix<6>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 7: sweeps = jacobi_matrix<7>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                case 8: sweeps = jacobi_matrix<8>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
                default: sweeps = jacobi_matrix<0>(Gm, n, ld, sm, s_n2, &s_rot, rows, A.bcols, A.max_sweeps, &converged); break;
            }
        }
        if (threadIdx.x == 0) { A.sweeps[i] = sweeps; A.eflag[i] = converged ? 0 : 1; }
        // ---- eigenvalues, normalised eigenvectors (in place), weights of Algorithm 1
        int gw = 0;
        for (int gc = A.grp_ptr[i]; gc < A.grp_ptr[i + 1]; ++gc) {
            const int c = A.grp_cols[gc], o = A.gen_off[c], b = A.blk_size[c];
            for (int e = threadIdx.x; e < b; e += blockDim.x)
                if (gw + e < 1024) s_genrow[gw + e] = o + e;
            gw += b;
        }
        __syncthreads();
        const double sig = A.sigma[i];
        const int64_t ep = A.eig_ptr[i];
        for (int l = wid; l < n; l += nw) {
            double* col = Gm + (size_t)l * ld;
            double s2 = 0.0;
            for (int r = lane; r < n; r += 32) s2 = fma(col[r], col[r], s2);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            const double nrm = sqrt(s2), inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
            for (int r = lane; r < n; r += 32) col[r] *= inv;
            __syncwarp();
            double wl = 0.0;
            if (gw <= 1024) {
                for (int e = lane; e < gw; e += 32) { const double q = col[s_genrow[e]]; wl = fma(q, q, wl); }
            } else {  // very wide groups: walk the generating columns again
                for (int gc = A.grp_ptr[i]; gc < A.grp_ptr[i + 1]; ++gc) {
                    const int c = A.grp_cols[gc], o = A.gen_off[c], b = A.blk_size[c];
                    for (int e = lane; e < b; e += 32) { const double q = col[o + e]; wl = fma(q, q, wl); }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) wl += __shfl_xor_sync(0xffffffffu, wl, o);
            if (lane == 0) { A.lam[ep + l] = nrm - sig; A.w[ep + l] = wl; }
        }
        __syncthreads();
    }
}

// G <- a_i + sigma_i I as a plain column-major array (column stride ld) from the gathered k8-panel
// workspace (mu = 0); a_i is symmetric, so panel row r is column r.  sigma_i = 1.5 x the Gershgorin bound.
__global__ void __launch_bounds__(256)
k_eig_init(int ngroups, const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
           const int64_t* __restrict__ ws_off, const unsigned long long* __restrict__ gersh,
           const double* __restrict__ X, double* __restrict__ G, double* __restrict__ sigma) {
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g];
    const double* Xg = X + ws_off[g];
    double* Gg = G + ws_off[g];
    double sg = 1.5 * __longlong_as_double((long long)gersh[g]);
    if (!(sg > 0.0)) sg = 1.0;  // zero matrix
    if (blockIdx.y == 0 && threadIdx.x == 0) sigma[g] = sg;
    const int64_t total = (int64_t)ld * ld;
    for (int64_t pos = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; pos < total; pos += (int64_t)gridDim.y * blockDim.x) {
        const int t0 = (int)(pos / ((int64_t)64 * ld)) * 64;
        const int rows_t = min(64, ld - t0);
        const int rem = (int)(pos - (int64_t)t0 * ld);
        const int kp = rem / (rows_t * 8), rem2 = rem - kp * rows_t * 8;
        const int row = t0 + (rem2 >> 3), col = kp * 8 + (rem2 & 7);
        double v = Xg[pos];
        if (row == col && row < n) v += sg;
        Gg[(size_t)row * ld + col] = v;
    }
}

// Occupation of one eigenvalue: Fermi function (L255) for kT > 0, else 1/2 (1 - signum) (Eq.(16)/(17), Eq.(12)).
__device__ __forceinline__ double occupation(double lam, double mu, double kT) {
    if (kT > 0.0) return 1.0 / (1.0 + exp((lam - mu) / kT));
    const double x = lam - mu;
    return x > 0.0 ? 0.0 : (x < 0.0 ? 1.0 : 0.5);
}

// Algorithm 1 inner loops (L275) for one mu: partial sums of w_il f(lambda_il) over fixed slices.
__global__ void __launch_bounds__(256)
k_eig_nelec_part(int64_t total, const double* __restrict__ lam, const double* __restrict__ w, double mu, double kT,
                 double* __restrict__ part) {
    __shared__ double s[256];
    const int64_t per = (total + gridDim.x - 1) / gridDim.x;
    const int64_t b = (int64_t)blockIdx.x * per, e = min(b + per, total);
    double a = 0.0;
    for (int64_t i = b + threadIdx.x; i < e; i += 256) a = fma(w[i], occupation(lam[i], mu, kT), a);
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = s[0];
}

__global__ void k_eig_sum(const double* __restrict__ in, int n, double* __restrict__ out) {
    __shared__ double s[1024];
    double a = 0.0;
    for (int i = threadIdx.x; i < n; i += 1024) a += in[i];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = s[0];
}

// Rows of X = Q (1 - 2 f(Lambda)) Q^T for the generating functions of group g, written into the k8-panel
// workspace buffer that k_scatter reads (D = 1/2 (delta - X) = Q f Q^T on the generating columns, Eq.(17)).
constexpr int ED_QC = 8;  // generating rows per pass over Q
__global__ void __launch_bounds__(256)
k_eig_density(const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv, const int64_t* __restrict__ ws_off,
              const int32_t* __restrict__ grp_ptr, const int32_t* __restrict__ grp_cols,
              const int32_t* __restrict__ gen_off, const int32_t* __restrict__ blk_size,
              const int64_t* __restrict__ eig_ptr, const double* __restrict__ lam, const double* __restrict__ Q,
              double mu, double kT, double* __restrict__ X) {
    extern __shared__ double cs[];  // [ED_QC][n]
    __shared__ int s_row[ED_QC];
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g];
    const double* Qg = Q + ws_off[g];
    double* Xg = X + ws_off[g];
    const double* lg = lam + eig_ptr[g];
    int gc = grp_ptr[g], e_in = 0;  // cursor over the generating functions
    const int gc_end = grp_ptr[g + 1];
    for (;;) {
        // next chunk of up to ED_QC generating rows
        int cnt = 0;
        int gcc = gc, ee = e_in;
        while (cnt < ED_QC && gcc < gc_end) {
            const int c = grp_cols[gcc];
            if (ee < blk_size[c]) {
                if (threadIdx.x == 0) s_row[cnt] = gen_off[c] + ee;
                ++cnt; ++ee;
            } else { ++gcc; ee = 0; }
        }
        if (cnt == 0) break;
        gc = gcc; e_in = ee;
        __syncthreads();
        for (int e = threadIdx.x; e < cnt * n; e += blockDim.x) {
            const int q = e / n, l = e - q * n;
            cs[(size_t)q * n + l] = Qg[(size_t)l * ld + s_row[q]] * (1.0 - 2.0 * occupation(lg[l], mu, kT));
        }
        __syncthreads();
        for (int p = threadIdx.x; p < n; p += blockDim.x) {
            double acc[ED_QC];
#pragma unroll
            for (int q = 0; q < ED_QC; ++q) acc[q] = 0.0;
            for (int l = 0; l < n; ++l) {
                const double u = Qg[(size_t)l * ld + p];
#pragma unroll
                for (int q = 0; q < ED_QC; ++q)
                    if (q < cnt) acc[q] = fma(u, cs[(size_t)q * n + l], acc[q]);
            }
#pragma unroll
            for (int q = 0; q < ED_QC; ++q)
                if (q < cnt) Xg[panel_off(s_row[q], p, ld)] = acc[q];
        }
        __syncthreads();
    }
}

}  // namespace smb

// ------------------------------------------------------------------------------------- host side
namespace smb {

sm_status_t eig_ensure_tables(sm_plan* p, cudaStream_t st) {
    if (p->d_eig_ptr) return SM_OK;
    const int ng = p->ngroups;
    std::vector<int64_t> ptr(ng + 1, 0);
    for (int i = 0; i < ng; ++i) ptr[i + 1] = ptr[i] + p->h_sub_dim[i];
    p->eig_total = ptr[ng];
    std::vector<int32_t> order(ng);
    for (int i = 0; i < ng; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return p->h_sub_dim[a] > p->h_sub_dim[b]; });
    const size_t tot = (size_t)std::max<int64_t>(p->eig_total, 1);
    SM_CUDA(cudaMalloc((void**)&p->d_eig_ptr, (size_t)(ng + 1) * 8));
    SM_CUDA(cudaMalloc((void**)&p->d_eig_lam, tot * 8));
    SM_CUDA(cudaMalloc((void**)&p->d_eig_w, tot * 8));
    SM_CUDA(cudaMalloc((void**)&p->d_eig_sigma, (size_t)std::max(ng, 1) * 8));
    SM_CUDA(cudaMalloc((void**)&p->d_eig_order, (size_t)std::max(ng, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_eig_state, (size_t)(2 * std::max(ng, 1) + 2) * 4));
    SM_CUDA(cudaMemcpyAsync(p->d_eig_ptr, ptr.data(), (size_t)(ng + 1) * 8, cudaMemcpyHostToDevice, st));
    if (ng) SM_CUDA(cudaMemcpyAsync(p->d_eig_order, order.data(), (size_t)ng * 4, cudaMemcpyHostToDevice, st));
    SM_CUDA(cudaStreamSynchronize(st));  // the host vectors go out of scope
    // block width: as many columns per block as two blocks of the largest submatrix fit in shared memory
    const int rows = (std::max(p->info.dim_max, 1) + 31) & ~31;
    int B = EJ_MAXB;
    while (B > 1 && (size_t)2 * B * rows * 8 > (size_t)200 * 1024) B >>= 1;
    if ((size_t)2 * B * rows * 8 > (size_t)200 * 1024) return SM_ERR_INVALID_ARG;  // submatrix too large for this solver
    p->eig_bcols = B;
    p->eig_smem = (size_t)2 * B * rows * 8;
    return SM_OK;
}

// a_i = Q Lambda Q^T for every submatrix (Eq.(17) first line): gather at mu = 0 into buf0, G_0 = a_i +
// sigma I into buf1, Jacobi sweeps; afterwards buf1 holds Q (normalised columns), the plan lambda and w.
sm_status_t launch_eig_decompose(sm_plan* p, const double* vals, double* buf0, double* buf1, cudaStream_t st) {
    sm_status_t s = eig_ensure_tables(p, st);
    if (s) return s;
    if (p->ngroups == 0) { p->eig_valid = 1; return SM_OK; }
    p->resc_eval = 0;
    if ((s = launch_gather(p, vals, 0.0, buf0, st))) return s;
    const int ng = p->ngroups;
    int split = 1;
    while ((int64_t)ng * split < (int64_t)p->num_sms * 8 && split < 64) ++split;
    k_eig_init<<<dim3(ng, split), 256, 0, st>>>(ng, p->d_sub_dim, p->d_ld, p->d_ws_off, p->d_gersh, buf0, buf1,
                                                 p->d_eig_sigma);
    SM_CUDA(cudaMemsetAsync(p->d_eig_state, 0, (size_t)(2 * ng + 2) * 4, st));
#ifndef SM_EIG_BLOCK
#define SM_EIG_BLOCK 1
#endif
    if (SM_EIG_BLOCK) {  // block form on the DMMA path (eig_block.cu)
        p->launches += 1;
        if ((s = launch_eig_bjacobi(p, buf1, st))) return s;
        p->eig_valid = 1;
        return SM_OK;
    }
    if (!p->eig_attr_set) {  // static + dynamic shared memory may exceed the 48 KB default
        SM_CUDA(cudaFuncSetAttribute(k_eig_jacobi, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->eig_smem));
        p->eig_attr_set = 1;
    }
    EigArgs a;
    a.sub_dim = p->d_sub_dim; a.ldv = p->d_ld; a.ws_off = p->d_ws_off; a.G = buf1; a.sigma = p->d_eig_sigma;
    a.order = p->d_eig_order; a.counter = p->d_eig_state + 2 * ng; a.sweeps = p->d_eig_state; a.eflag = p->d_eig_state + ng;
    a.grp_ptr = p->d_grp_ptr; a.grp_cols = p->d_grp_cols; a.gen_off = p->d_gen_off; a.blk_size = p->d_blk_size;
    a.eig_ptr = p->d_eig_ptr; a.lam = p->d_eig_lam; a.w = p->d_eig_w;
    a.ngroups = ng; a.max_sweeps = 40; a.bcols = p->eig_bcols; a.smem_rows = 0;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(4, (size_t)(220 * 1024) / std::max<size_t>(p->eig_smem, 1)));
    const int grid = std::min(ng, p->num_sms * per_sm);
    k_eig_jacobi<<<grid, EJ_THREADS, p->eig_smem, st>>>(a);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    p->eig_valid = 1;
    return SM_OK;
}

// n_elec(mu) of Algorithm 1 from the stored (lambda, w): result in d_scalars[0] and (after the caller's
// synchronisation) h_pinned_d[0].
sm_status_t launch_eig_nelec(sm_plan* p, double mu, double kT, cudaStream_t st) {
    const int nblk = 592;
    k_eig_nelec_part<<<nblk, 256, 0, st>>>(p->eig_total, p->d_eig_lam, p->d_eig_w, mu, kT, p->d_red);
    k_eig_sum<<<1, 1024, 0, st>>>(p->d_red, nblk, p->d_scalars + 0);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    SM_CUDA(cudaMemcpyAsync(p->h_pinned_d, p->d_scalars, 8, cudaMemcpyDeviceToHost, st));
    return SM_OK;
}

// X rows of the generating functions into buf0 (k8-panel layout) from Q in buf1; prepares the state the
// scatter reads (no submatrix "stopped at iteration 0", result in buffer 0).
sm_status_t launch_eig_density(sm_plan* p, double mu, double kT, double* buf0, const double* buf1, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    const size_t smem = (size_t)ED_QC * std::max(p->info.dim_max, 1) * 8;
    if (smem > (size_t)200 * 1024) return SM_ERR_INVALID_ARG;  // submatrix too large for this path (n > 3200)
    if (smem > 40 * 1024) SM_CUDA(cudaFuncSetAttribute(k_eig_density, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_eig_density<<<p->ngroups, 256, smem, st>>>(p->d_sub_dim, p->d_ld, p->d_ws_off, p->d_grp_ptr, p->d_grp_cols,
                                                  p->d_gen_off, p->d_blk_size, p->d_eig_ptr, p->d_eig_lam, buf1, mu, kT, buf0);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    SM_CUDA(cudaMemsetAsync(p->d_done_iter, 0xff, (size_t)std::max(p->ngroups, 1) * 4, st));
    p->cur_k = 2;
    return SM_OK;
}

}  // namespace smb
