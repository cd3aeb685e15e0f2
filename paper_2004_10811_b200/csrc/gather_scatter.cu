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
// grid = (ngroups, chunks of GATHER_CB column blocks).  Per CTA, once: S_i and its element
// offsets go to shared memory together with a hash table block-row -> member index and a
// per-dense-row record (member, row inside the member, member height).  Then one warp assembles
// one block column c = S_i[tc] of a_i at a time:
//  (1) the lanes walk the stored blocks (r,c) of column c (coalesced reads of rowidx / val_off),
//      look r up in the hash table and note the value offset of the block for member r;
//      members without a stored block stay -1 -> zero fill (reading A4);
//  (2) for up to four dense columns of the block column at once the lanes sweep the ld rows two
//      at a time and store 16 bytes each, taking the values from the stored blocks, subtracting
//      mu on the diagonal (Eq.(16)) and zero-padding rows/columns n..ld-1.
// The column abs-sums give the Gershgorin bound s_i = max_q sum_p |a_pq| (symmetric: column sums
// = row sums), combined by atomicMax on the bits of a non-negative double.
// ---------------------------------------------------------------------------------------------
constexpr int GATHER_CB = 16;  // column blocks per CTA

__device__ __forceinline__ unsigned gather_hash(int key, int shift) {
    return ((unsigned)key * 2654435761u) >> shift;
}

__global__ void __launch_bounds__(256)
k_gather(const int64_t* __restrict__ colptr, const int32_t* __restrict__ rowidx,
         const int64_t* __restrict__ val_off, const double* __restrict__ vals,
         const int64_t* __restrict__ sub_ptr, const int32_t* __restrict__ sub_blocks,
         const int32_t* __restrict__ sub_off, const int32_t* __restrict__ sub_dim,
         const int32_t* __restrict__ ldv, const int64_t* __restrict__ ws_off, double mu,
         double* __restrict__ X, unsigned long long* __restrict__ gersh, int max_sub_blocks, int max_ld,
         int hash_size, int hash_shift) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int g = blockIdx.x;
    const int m = (int)(sub_ptr[g + 1] - sub_ptr[g]);
    const int cb0 = blockIdx.y * GATHER_CB;
    // column chunks past |S_i| only have padding columns to write (handled by the last chunk)
    const int nchunks = (m + GATHER_CB - 1) / GATHER_CB;
    if ((int)blockIdx.y >= nchunks) return;
    const int n = sub_dim[g], ld = ldv[g];
    // shared-memory carve-up (all 8-byte aligned)
    int64_t* src_all = reinterpret_cast<int64_t*>(smem_raw);                  // [warps][max_sub_blocks]
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int2* rinfo = reinterpret_cast<int2*>(src_all + (size_t)nw * max_sub_blocks);  // [max_ld]
    int32_t* hk = reinterpret_cast<int32_t*>(rinfo + max_ld);                 // [hash_size] keys
    int32_t* hv = hk + hash_size;                                             // [hash_size] member index
    int32_t* S = hv + hash_size;                                              // [max_sub_blocks]
    int32_t* So = S + max_sub_blocks;                                         // [max_sub_blocks + 1]
    for (int h = threadIdx.x; h < hash_size; h += blockDim.x) hk[h] = -1;
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        S[t] = sub_blocks[sub_ptr[g] + t];
        So[t] = sub_off[sub_ptr[g] + t];
    }
    if (threadIdx.x == 0) So[m] = n;
    __syncthreads();
    const unsigned hmask = (unsigned)hash_size - 1u;
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        const int key = S[t];
        unsigned h = gather_hash(key, hash_shift);
        while (atomicCAS(&hk[h], -1, key) != -1) h = (h + 1) & hmask;
        hv[h] = t;
        const int o = So[t], b = So[t + 1] - o;
        for (int e = 0; e < b; ++e) rinfo[o + e] = make_int2(t, e | (b << 16));
    }
    for (int p = n + threadIdx.x; p < ld; p += blockDim.x) rinfo[p] = make_int2(-1, 0);
    __syncthreads();
    int64_t* src = src_all + (size_t)wid * max_sub_blocks;                    // [m] per warp
    double* Xg = X + ws_off[g];
    double cmax = 0.0;
    const int cb1 = min(cb0 + GATHER_CB, m);
    for (int tc = cb0 + wid; tc < cb1; tc += nw) {
        const int c = S[tc];
        const int coff = So[tc], bc = So[tc + 1] - coff;
        for (int t = lane; t < m; t += 32) src[t] = -1;
        __syncwarp();
        const int64_t p0 = colptr[c];
        const int clen = (int)(colptr[c + 1] - p0);
        for (int j = lane; j < clen; j += 32) {
            const int r = __ldg(rowidx + p0 + j);
            unsigned h = gather_hash(r, hash_shift);
            for (;;) {
                const int k = hk[h];
                if (k == r) { src[hv[h]] = __ldg(val_off + p0 + j); break; }
                if (k < 0) break;
                h = (h + 1) & hmask;
            }
        }
        __syncwarp();
        for (int q0 = 0; q0 < bc; q0 += 4) {
            const int nq = min(4, bc - q0);
            double asum[4] = {0.0, 0.0, 0.0, 0.0};
            // dense column q of a_i is stored as row coff+q of the symmetric X (k8-panel layout)
            size_t rbase[4];
            int rstride[4];
#pragma unroll
            for (int qq = 0; qq < 4; ++qq) {
                const int xrow = coff + q0 + (qq < nq ? qq : 0);
                const int t0 = xrow & ~63;
                const int rows_t = min(64, ld - t0);
                rbase[qq] = (size_t)t0 * ld + (size_t)(xrow & 63) * 8;
                rstride[qq] = rows_t * 8;
            }
            const int dq = coff + q0;  // diagonal position of dense column q0
            for (int p = 2 * lane; p < ld; p += 64) {
                double v[4][2];
#pragma unroll
                for (int qq = 0; qq < 4; ++qq) v[qq][0] = v[qq][1] = 0.0;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int2 ri = rinfo[p + u];
                    if (ri.x >= 0) {
                        const int64_t s0 = src[ri.x];
                        if (s0 >= 0) {
                            const int br = ri.y >> 16;
                            const double* vp = vals + s0 + (int64_t)q0 * br + (ri.y & 0xffff);
#pragma unroll
                            for (int qq = 0; qq < 4; ++qq)
                                if (qq < nq) v[qq][u] = __ldg(vp + qq * br);
                        }
                    }
                }
#pragma unroll
                for (int qq = 0; qq < 4; ++qq) {
                    if (qq < nq) {
                        if (dq + qq == p) v[qq][0] -= mu;
                        else if (dq + qq == p + 1) v[qq][1] -= mu;
                        asum[qq] += fabs(v[qq][0]) + fabs(v[qq][1]);
                        *reinterpret_cast<double2*>(Xg + rbase[qq] + (size_t)(p >> 3) * rstride[qq] + (p & 7)) =
                            make_double2(v[qq][0], v[qq][1]);
                    }
                }
            }
#pragma unroll
            for (int qq = 0; qq < 4; ++qq) {
                double a = asum[qq];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                cmax = fmax(cmax, a);
            }
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
        p->d_colptr, p->d_rowidx, p->d_val_off, vals, p->d_sub_ptr, p->d_sub_blocks, p->d_sub_off,
        p->d_sub_dim, p->d_ld, p->d_ws_off, mu, X, p->d_gersh, p->gather_msb, p->gather_max_ld,
        p->gather_hash_size, p->gather_hash_shift);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// ---------------------------------------------------------------------------------------------
// Scatter (PAPER.md L127 step 3 + Eq.(16) inner factor): one warp per block column c.  The values
// of a block column are one contiguous range of the result; the warp takes 32 of its blocks at a
// time (one packed record each: row offset inside the submatrix | block height), prefix-sums
// their sizes and then sweeps the contiguous output range with one element per lane (coalesced
// stores), finding the block of an element by a shuffle binary search over the prefix sums.
// Element (el,q) of block (r,c) reads X_i[gen_off(c) + q, blk_loc(r) + el] of c's group i
// (X symmetric, so the read walks a contiguous row segment).  D = 1/2 (delta - xs * X), xs = 1/s_i
// if the submatrix converged at iteration 0 (the buffer then still holds the unscaled
// a_i - mu I), else 1.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_scatter(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
          const int64_t* __restrict__ val_off, const int32_t* __restrict__ col_grp,
          const int32_t* __restrict__ gen_off, const uint32_t* __restrict__ blk_pack,
          const int32_t* __restrict__ ldv, const int64_t* __restrict__ ws_off,
          const int32_t* __restrict__ done_iter, const unsigned long long* __restrict__ gersh, int cur_k,
          const double* __restrict__ buf0, const double* __restrict__ buf1, double* __restrict__ out,
          int as_identity) {
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= nb) return;
    const int lane = threadIdx.x & 31;
    const int g = col_grp[c];
    const int bc = blk_size[c];
    const int64_t p0 = colptr[c];
    const int nblk = (int)(colptr[c + 1] - p0);
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
    double* o = out + val_off[p0];
    for (int base = 0; base < nblk; base += 32) {
        const int b = base + lane;
        const uint32_t pk = b < nblk ? __ldg(blk_pack + p0 + b) : 0u;
        const int sz = (int)(pk >> 20) * bc;
        int incl = sz;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        const int excl = incl - sz;
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        for (int e0 = 0; e0 < total; e0 += 32) {
            const int e = e0 + lane;
            int k = 0;  // number of blocks that end at or before element e
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                const int v = __shfl_sync(0xffffffffu, incl, k + d - 1);
                if (v <= e) k += d;
            }
            const uint32_t pkk = __shfl_sync(0xffffffffu, pk, k & 31);
            const int ex = __shfl_sync(0xffffffffu, excl, k & 31);
            if (e < total) {
                const int br = (int)(pkk >> 20), loc = (int)(pkk & 0xfffffu);
                const int w = e - ex;
                const int q = w / br, el = w - q * br;
                const double x = Xg[panel_off(go + q, loc + el, ld)];
                o[e] = as_identity ? x : 0.5 * (((loc + el == go + q) ? 1.0 : 0.0) - xs * x);
            }
        }
        o += total;
    }
}

sm_status_t launch_scatter(sm_plan* p, int as_identity, const double* buf0, const double* buf1,
                           double* out, cudaStream_t st) {
    if (p->nb == 0) return SM_OK;
    k_scatter<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_colptr, p->d_val_off, p->d_col_grp,
                                               p->d_gen_off, p->d_blk_pack, p->d_ld, p->d_ws_off,
                                               p->d_done_iter, p->d_gersh, p->cur_k, buf0, buf1, out,
                                               as_identity);
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
