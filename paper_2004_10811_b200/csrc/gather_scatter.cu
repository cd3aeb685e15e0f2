// a3 gather/assemble, a4 Gershgorin bound, a6 extract/scatter, a7 trace reductions.
// All HBM-bandwidth-bound: coalesced 16-byte stores of whole dense columns, short L2-resident
// reads of the stored blocks, no floating-point atomics (fixed reduction orders).
#include "common.cuh"

namespace smb {

__device__ __forceinline__ int find_sorted64(const int32_t* __restrict__ a, int n, int key) {
    int lo = 0, hi = n - 1;
    while (lo <= hi) {
        int mid = (lo + hi) >> 1, v = __ldg(a + mid);
        if (v == key) return mid;
        if (v < key) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

// ---------------------------------------------------------------------------------------------
// Gather (PAPER.md L125 step 1; L187 "submatrix assembly becomes a purely local operation").
// grid = (ngroups, chunks of CB column blocks); one warp assembles one block column of a_i at a
// time: (1) lanes look up, for every member r of S_i, the stored block (r,c) of column c
// (binary search in the CSC column; -1 if absent -> zero fill, reading A4), (2) for each dense
// column the lanes sweep the ld rows two at a time and store 16 bytes each (coalesced), taking
// the values from the stored blocks, subtracting mu on the diagonal (Eq.(16)) and zero-padding
// rows/columns n..ld-1.  The column abs-sums give the Gershgorin bound s_i = max_q sum_p |a_pq|
// (symmetric: column sums = row sums), combined by atomicMax on the bits of a non-negative double.
// ---------------------------------------------------------------------------------------------
constexpr int GATHER_CB = 8;  // column blocks per CTA

__global__ void k_gather(const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                         const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
                         const double* __restrict__ vals, const int64_t* __restrict__ sub_ptr,
                         const int32_t* __restrict__ sub_blocks, const int32_t* __restrict__ sub_off,
                         const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
                         const int64_t* __restrict__ ws_off, double mu, double* __restrict__ X,
                         unsigned long long* __restrict__ gersh, int max_sub_blocks, int max_ld) {
    extern __shared__ unsigned char smem_raw[];
    const int g = blockIdx.x;
    const int m = (int)(sub_ptr[g + 1] - sub_ptr[g]);
    const int cb0 = blockIdx.y * GATHER_CB;
    const int n = sub_dim[g], ld = ldv[g];
    // column chunks past |S_i| only have padding columns to write (handled by the last chunk)
    const int nchunks = (m + GATHER_CB - 1) / GATHER_CB;
    if ((int)blockIdx.y >= nchunks) return;
    const int32_t* S = sub_blocks + sub_ptr[g];
    const int32_t* So = sub_off + sub_ptr[g];
    int32_t* row2blk = reinterpret_cast<int32_t*>(smem_raw);                       // [max_ld]
    int64_t* src_all = reinterpret_cast<int64_t*>(smem_raw + (((size_t)max_ld * 4 + 15) / 16) * 16);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int64_t* src = src_all + (size_t)wid * max_sub_blocks;                         // [m] per warp
    // row -> member map
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        int o = So[t], b = blk_size[S[t]];
        for (int e = 0; e < b; ++e) row2blk[o + e] = t;
    }
    __syncthreads();
    double* Xg = X + ws_off[g];
    double cmax = 0.0;
    const int cb1 = min(cb0 + GATHER_CB, m);
    for (int tc = cb0 + wid; tc < cb1; tc += nw) {
        const int c = S[tc];
        const int bc = blk_size[c];
        const int64_t p0 = colptr[c];
        const int clen = (int)(colptr[c + 1] - p0);
        for (int t = lane; t < m; t += 32) {
            int f = find_sorted64(rowidx + p0, clen, S[t]);
            src[t] = f >= 0 ? val_off[p0 + f] : (int64_t)-1;
        }
        __syncwarp();
        const int coff = So[tc];
        for (int q = 0; q < bc; ++q) {
            const int xrow = coff + q;  // symmetric: dense column q of a_i is stored as row q
            double asum = 0.0;
            for (int p = 2 * lane; p < ld; p += 64) {
                double v[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    int pp = p + u;
                    double x = 0.0;
                    if (pp < n) {
                        int t = row2blk[pp];
                        int64_t s0 = src[t];
                        if (s0 >= 0) {
                            int o = So[t];
                            int br = (t + 1 < m ? So[t + 1] : n) - o;
                            x = __ldg(vals + s0 + (int64_t)q * br + (pp - o));
                        }
                        if (pp == coff + q) x -= mu;
                    }
                    v[u] = x;
                    asum += fabs(x);
                }
                *reinterpret_cast<double2*>(Xg + panel_off(xrow, p, ld)) = make_double2(v[0], v[1]);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) asum += __shfl_xor_sync(0xffffffffu, asum, o);
            cmax = fmax(cmax, asum);
        }
        __syncwarp();
    }
    // zero padding columns n..ld-1 (last chunk only)
    if ((int)blockIdx.y == nchunks - 1) {
        for (int qq = n + wid; qq < ld; qq += nw) {
            for (int p = 2 * lane; p < ld; p += 64)
                *reinterpret_cast<double2*>(Xg + panel_off(qq, p, ld)) = make_double2(0.0, 0.0);
        }
    }
    if (lane == 0 && cmax > 0.0) atomicMax(gersh + g, (unsigned long long)__double_as_longlong(cmax));
}

sm_status_t launch_gather(sm_plan* p, const double* vals, double mu, double* X, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    SM_CUDA(cudaMemsetAsync(p->d_gersh, 0, (size_t)p->ngroups * 8, st));
    int chunks = (p->max_sub_blocks + GATHER_CB - 1) / GATHER_CB;
    dim3 grid(p->ngroups, chunks > 0 ? chunks : 1);
    if (p->gather_smem > 48 * 1024)
        SM_CUDA(cudaFuncSetAttribute(k_gather, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->gather_smem));
    k_gather<<<grid, p->gather_warps * 32, p->gather_smem, st>>>(
        p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_val_off, vals, p->d_sub_ptr, p->d_sub_blocks,
        p->d_sub_off, p->d_sub_dim, p->d_ld, p->d_ws_off, mu, X, p->d_gersh, p->max_sub_blocks,
        p->info.dim_max + LD_ALIGN);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// ---------------------------------------------------------------------------------------------
// Scatter (PAPER.md L127 step 3 + Eq.(16) inner factor): one CTA per block column c; threads
// sweep the column's contiguous value range (coalesced stores); element (e,q) of block (r,c)
// reads X_i[blk_loc(r) + e, gen_off(c) + q] of c's group i (X symmetric, so the read walks a
// contiguous column segment).  D = 1/2 (delta - xs * X), xs = 1/s_i if the submatrix converged at
// iteration 0 (the buffer then still holds the unscaled a_i - mu I), else 1.
// ---------------------------------------------------------------------------------------------
__global__ void k_scatter(const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                          const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
                          const int32_t* __restrict__ col_grp, const int32_t* __restrict__ gen_off,
                          const int32_t* __restrict__ blk_loc, const int32_t* __restrict__ ldv,
                          const int64_t* __restrict__ ws_off, const int32_t* __restrict__ done_iter,
                          const unsigned long long* __restrict__ gersh, int cur_k,
                          const double* __restrict__ buf0, const double* __restrict__ buf1,
                          double* __restrict__ out, int as_identity) {
    const int c = blockIdx.x;
    const int g = col_grp[c];
    const int bc = blk_size[c];
    const int64_t p0 = colptr[c], p1 = colptr[c + 1];
    const int64_t v0 = val_off[p0], v1 = val_off[p1];
    const int di = done_iter[g];
    const int kb = di >= 0 ? di : cur_k;
    const double* Xg = ((kb & 1) ? buf1 : buf0) + ws_off[g];
    const int ld = ldv[g];
    double xs = 1.0;
    if (kb == 0 && !as_identity) {
        double s = __longlong_as_double((long long)gersh[g]);
        xs = s > 0.0 ? 1.0 / s : 1.0;
    }
    const int go = gen_off[c];
    const int nblk = (int)(p1 - p0);
    for (int64_t e = v0 + threadIdx.x; e < v1; e += blockDim.x) {
        // block containing element e: largest b with val_off[b] <= e
        int lo = 0, hi = nblk - 1;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (__ldg(val_off + p0 + mid) <= e) lo = mid; else hi = mid - 1;
        }
        const int64_t b = p0 + lo;
        const int r = rowidx[b];
        const int br = blk_size[r];
        const int w = (int)(e - val_off[b]);
        const int q = w / br, el = w - q * br;
        double x = Xg[panel_off(go + q, blk_loc[b] + el, ld)];
        double d;
        if (as_identity) d = x;
        else d = 0.5 * (((r == c && q == el) ? 1.0 : 0.0) - xs * x);
        out[e] = d;
    }
    (void)bc;
}

sm_status_t launch_scatter(sm_plan* p, int as_identity, const double* buf0, const double* buf1,
                           double* out, cudaStream_t st) {
    if (p->nb == 0) return SM_OK;
    k_scatter<<<p->nb, 128, 0, st>>>(p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_val_off, p->d_col_grp,
                                     p->d_gen_off, p->d_blk_loc, p->d_ld, p->d_ws_off, p->d_done_iter,
                                     p->d_gersh, p->cur_k, buf0, buf1, out, as_identity);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// ---------------------------------------------------------------------------------------------
// Deterministic sum of n doubles by one CTA of 1024 threads (fixed strided + tree order).
// ---------------------------------------------------------------------------------------------
__global__ void k_sum_fixed(const double* __restrict__ in, int64_t n, double* __restrict__ out) {
    __shared__ double s[1024];
    double a = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 1024) a += in[i];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = s[0];
}

// a7 (Algorithm 1, Eq.(18)): n_elec partial of group g = sum over its generating functions k
// of 1/2 (1 - xs X_kk).  One warp per group, lanes strided over the diagonal entries, fixed order.
__global__ void k_nelec_part(int ngroups, const int32_t* __restrict__ grp_ptr, const int32_t* __restrict__ grp_cols,
                             const int32_t* __restrict__ blk_size, const int32_t* __restrict__ gen_off,
                             const int32_t* __restrict__ ldv, const int64_t* __restrict__ ws_off,
                             const int32_t* __restrict__ done_iter, const unsigned long long* __restrict__ gersh,
                             int cur_k, const double* __restrict__ buf0, const double* __restrict__ buf1,
                             double* __restrict__ part) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= ngroups) return;
    const int lane = threadIdx.x & 31;
    const int di = done_iter[g];
    const int kb = di >= 0 ? di : cur_k;
    const double* Xg = ((kb & 1) ? buf1 : buf0) + ws_off[g];
    const int ld = ldv[g];
    double xs = 1.0;
    if (kb == 0) {
        double s = __longlong_as_double((long long)gersh[g]);
        xs = s > 0.0 ? 1.0 / s : 1.0;
    }
    double a = 0.0;
    for (int gc = grp_ptr[g]; gc < grp_ptr[g + 1]; ++gc) {
        int c = grp_cols[gc];
        int o = gen_off[c], b = blk_size[c];
        for (int e = lane; e < b; e += 32) {
            const int d = o + e;
            a += 0.5 * (1.0 - xs * Xg[panel_off(d, d, ld)]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) part[g] = a;
}

sm_status_t launch_nelec(sm_plan* p, const double* buf0, const double* buf1, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    k_nelec_part<<<(p->ngroups + 7) / 8, 256, 0, st>>>(p->ngroups, p->d_grp_ptr, p->d_grp_cols, p->d_blk_size,
                                                       p->d_gen_off, p->d_ld, p->d_ws_off, p->d_done_iter,
                                                       p->d_gersh, p->cur_k, buf0, buf1, p->d_ne_part);
    k_sum_fixed<<<1, 1024, 0, st>>>(p->d_ne_part, p->ngroups, p->d_scalars + 0);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// tr(D) and tr(D K) (Eq.(18), Eq.(10)).  Stage 1: each CTA reduces a fixed contiguous
// slice of the value arrays (and the diagonal entries of the diagonal blocks it owns by block
// column); stage 2: k_sum_fixed.
__global__ void k_trace_dk_part(int64_t nnz, const double* __restrict__ D, const double* __restrict__ K,
                                double* __restrict__ part) {
    __shared__ double s[256];
    const int64_t per = (nnz + gridDim.x - 1) / gridDim.x;
    const int64_t b = (int64_t)blockIdx.x * per, e = min(b + per, nnz);
    double a = 0.0;
    for (int64_t i = b + threadIdx.x; i < e; i += 256) a += D[i] * K[i];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = s[0];
}

__global__ void k_trace_d_part(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                               const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
                               const double* __restrict__ D, double* __restrict__ part) {
    __shared__ double s[256];
    const int per = (nb + gridDim.x - 1) / gridDim.x;
    const int c0 = blockIdx.x * per, c1 = min(c0 + per, nb);
    double a = 0.0;
    for (int c = c0 + threadIdx.x; c < c1; c += 256) {
        const int64_t p0 = colptr[c];
        int f = find_sorted64(rowidx + p0, (int)(colptr[c + 1] - p0), c);
        if (f >= 0) {
            const int b = blk_size[c];
            const double* blk = D + val_off[p0 + f];
            for (int e = 0; e < b; ++e) a += blk[(size_t)e * b + e];
        }
    }
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = s[0];
}

sm_status_t launch_trace_dk(sm_plan* p, const double* D, const double* K, cudaStream_t st) {
    const int nblk = 1184;  // 8 x 148
    k_trace_dk_part<<<nblk, 256, 0, st>>>(p->nnz, D, K, p->d_red);
    k_sum_fixed<<<1, 1024, 0, st>>>(p->d_red, nblk, p->d_scalars + 2);
    k_trace_d_part<<<nblk, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_val_off, D,
                                         p->d_red + 2048);
    k_sum_fixed<<<1, 1024, 0, st>>>(p->d_red + 2048, nblk, p->d_scalars + 1);
    p->launches += 4;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// Gershgorin interval of the whole K~ (bracket of the mu bisection, reading A11): one warp per
// block column; per dense column q: centre = K_qq, radius = sum of |off-diagonal| of the column.
__global__ void k_gersh_global(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                               const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
                               const double* __restrict__ vals, double* __restrict__ lo_part,
                               double* __restrict__ hi_part) {
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= nb) return;
    const int lane = threadIdx.x & 31;
    const int bc = blk_size[c];
    double lo = 1e300, hi = -1e300;
    for (int q = 0; q < bc; ++q) {
        double rad = 0.0, dia = 0.0;
        for (int64_t b = colptr[c] + lane; b < colptr[c + 1]; b += 32) {
            const int r = rowidx[b];
            const int br = blk_size[r];
            const double* col = vals + val_off[b] + (size_t)q * br;
            for (int e = 0; e < br; ++e) {
                double v = col[e];
                if (r == c && e == q) dia = v; else rad += fabs(v);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            rad += __shfl_xor_sync(0xffffffffu, rad, o);
            dia += __shfl_xor_sync(0xffffffffu, dia, o);
        }
        lo = fmin(lo, dia - rad);
        hi = fmax(hi, dia + rad);
    }
    if (lane == 0) { lo_part[c] = lo; hi_part[c] = hi; }
}

__global__ void k_minmax_fixed(const double* __restrict__ lo, const double* __restrict__ hi, int n,
                               double* __restrict__ out) {
    __shared__ double s0[1024], s1[1024];
    double a = 1e300, b = -1e300;
    for (int i = threadIdx.x; i < n; i += 1024) { a = fmin(a, lo[i]); b = fmax(b, hi[i]); }
    s0[threadIdx.x] = a; s1[threadIdx.x] = b;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            s0[threadIdx.x] = fmin(s0[threadIdx.x], s0[threadIdx.x + o]);
            s1[threadIdx.x] = fmax(s1[threadIdx.x], s1[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = s0[0]; out[1] = s1[0]; }
}

sm_status_t launch_gersh_global(sm_plan* p, const double* vals, cudaStream_t st) {
    double *lo = nullptr, *hi = nullptr;
    SM_CUDA(cudaMalloc((void**)&lo, (size_t)p->nb * 8));
    SM_CUDA(cudaMalloc((void**)&hi, (size_t)p->nb * 8));
    k_gersh_global<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_val_off,
                                                    vals, lo, hi);
    k_minmax_fixed<<<1, 1024, 0, st>>>(lo, hi, p->nb, p->d_scalars + 4);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    SM_CUDA(cudaStreamSynchronize(st));
    cudaFree(lo);
    cudaFree(hi);
    return SM_OK;
}

}  // namespace smb
