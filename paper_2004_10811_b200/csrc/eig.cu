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
// This file: the shifted start matrix, n_elec(mu) and the generating rows of Q f(Lambda - mu) Q^T; the
// Jacobi sweeps themselves are the block kernel of eig_block.cu.
#include "common.cuh"

namespace smb {

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
    p->launches += 1;
    if ((s = launch_eig_bjacobi(p, buf1, st))) return s;
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
