// a4 spectral bound, option scaling = 1 ("interlacing"): every a_i is a PRINCIPAL submatrix of the
// symmetric K~, so by Cauchy interlacing  lambda_min(K~) <= lambda(a_i) <= lambda_max(K~)
// and  rho(a_i - mu I) <= max(|lambda_max(K~) - mu|, |lambda_min(K~) - mu|)  for EVERY submatrix and
// EVERY mu of the bisection.  The two extreme eigenvalues of the block-sparse K~ are estimated once
// per call by a short Lanczos run (block-CSC mat-vec, deterministic reductions) and widened by a
// safety margin.  The Ritz extremes approach the true ones from INSIDE, so the cap is an estimate, not
// a bound: Newton-Schulz tolerates rho/s < sqrt(3) (1.15 beyond the largest overshoot), and three
// guards keep the estimate from going below that (reading A8): (i) a run that breaks down
// (beta_j <= 1e-10 of the scale of T before the last step: the start vector lies in an invariant
// subspace) is discarded -- the call then uses the rigorous Gershgorin bounds only, no interlacing
// bracket, no quadrature guess; (ii) the cap of a submatrix is never taken below a rigorous LOWER bound
// of its spectral radius (largest column 2-norm of a_i - mu I, from the gather); (iii) s_i never exceeds
// the submatrix's own Gershgorin bound.  All arithmetic runs on the device; the host only sequences
// the launches and reads the resulting doubles.
#include <cooperative_groups.h>

#include "common.cuh"

namespace smb {

constexpr int LZ_STEPS = 24;  // extreme Ritz values within ~1 % of the spread (A8); margin 3 %

// y = K x for the symmetric block-CSC K~: y_c = sum_{(r,c) stored} K[r,c]^T x_r, one warp per block
// column (no atomics); lane b takes every 32nd block of the column.  part[c] = y_c . x_c.
// For the common block widths (1, 4, 5, 13: H and O in SZV / DZVP) the lane keeps the partial sums of
// all dense columns of the block column in registers, so index and values of a block are read once.
// rec[b] = (value offset lo, hi, first basis function of the block's row, its height): ONE 16-byte load per stored
// block instead of a chain of four dependent index loads.
// (Block columns of width 1, 4 and 5 take the streaming form lz_col_s below; this one serves the other widths.)
template <int BC>
__device__ __forceinline__ double lz_col(int lane, int oc, int64_t p0, int64_t p1, const int4* __restrict__ rec,
                                         const double* __restrict__ vals, const double* __restrict__ x,
                                         double* __restrict__ y) {
    double a[BC];
#pragma unroll
    for (int q = 0; q < BC; ++q) a[q] = 0.0;
    for (int64_t b = p0 + lane; b < p1; b += 32) {
        const int4 rc = __ldg(rec + b);
        const int br = rc.w;
        const double* blk = vals + (((int64_t)rc.y << 32) | (int64_t)(uint32_t)rc.x);
        const double* xr = x + rc.z;
        for (int e = 0; e < br; ++e) {
            const double xe = xr[e];
#pragma unroll
            for (int q = 0; q < BC; ++q) a[q] = fma(blk[q * br + e], xe, a[q]);
        }
    }
    double dot = 0.0;
#pragma unroll
    for (int q = 0; q < BC; ++q) {
        double v = a[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) y[oc + q] = v;
        dot = fma(v, x[oc + q], dot);
    }
    return dot;
}

// Streaming form of the same product: a per-value map (x index | q << 28, built once per plan by k_lz_map) lets the
// lanes of the warp walk the values of the block column in storage order -- coalesced 8-byte and 4-byte loads, four
// per lane in flight -- instead of one block per lane.
template <int BC>
__device__ __forceinline__ double lz_col_s(int lane, int oc, int64_t v0, int64_t v1, const uint32_t* __restrict__ map,
                                           const double* __restrict__ vals, const double* __restrict__ x,
                                           double* __restrict__ y) {
    double a[BC];
#pragma unroll
    for (int q = 0; q < BC; ++q) a[q] = 0.0;
    for (int64_t e0 = v0 + lane; e0 < v1; e0 += 128) {
        uint32_t m[4];
        double v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t e = e0 + 32 * u;
            m[u] = e < v1 ? __ldcs(map + e) : 0u;
            v[u] = e < v1 ? __ldcs(vals + e) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const double t = v[u] * x[m[u] & 0x0fffffffu];
            const int q = (int)(m[u] >> 28);
#pragma unroll
            for (int qq = 0; qq < BC; ++qq) a[qq] += (BC == 1 || q == qq) ? t : 0.0;
        }
    }
    double dot = 0.0;
#pragma unroll
    for (int q = 0; q < BC; ++q) {
        double s = a[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) y[oc + q] = s;
        dot = fma(s, x[oc + q], dot);
    }
    return dot;
}

// map[e] for every stored value e of block column c: one warp per block column, lanes over the elements of a block
__global__ void __launch_bounds__(256)
k_lz_map(int nb, const int32_t* __restrict__ blk_size, const int32_t* __restrict__ blk_off,
         const int64_t* __restrict__ colptr, const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
         uint32_t* __restrict__ map) {
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= nb) return;
    const int lane = threadIdx.x & 31, bc = blk_size[c];
    for (int64_t b = colptr[c]; b < colptr[c + 1]; ++b) {
        const int r = rowidx[b], br = blk_size[r], ro = blk_off[r];
        const int64_t v = val_off[b];
        for (int w = lane; w < br * bc; w += 32) {
            const int q = w / br, el = w - q * br;
            map[v + w] = (uint32_t)(ro + el) | ((uint32_t)q << 28);
        }
    }
}

// Gauss quadrature of the k x k Lanczos tridiagonal T (diag alpha, off-diagonal beta): thread j finds
// the j-th Ritz value by bisection on Sturm counts and its weight = squared first component of the
// eigenvector (1 / sum_i p_i(theta)^2 with the normalised Lanczos polynomials p_i).  out[0], out[1]:
// extreme Ritz values widened by margin * spread (interlacing bound, bisection bracket); out[2 + j]:
// Ritz values ascending; out[2 + 32 + j]: cumulative weights = the start vector's estimate of the
// fraction of eigenvalues of K~ below the node (used for the first interior step of the mu search,
// DESIGN.md reading A11d); out[66] = 1.0 if the recurrence broke down (some beta_i, i < k - 1, not above
// 1e-10 of the largest entry of T: everything after it is rounding noise), else 0.0.  One warp; k <= 32.
__device__ void lz_quadrature_body(int k, const double* __restrict__ alpha, const double* __restrict__ beta,
                                   double margin, double* __restrict__ out, double* th, double* wt) {
    const int j = threadIdx.x;
    double glo = 1e300, ghi = -1e300, tscale = 0.0;
    for (int i = 0; i < k; ++i) {
        const double r = (i > 0 ? fabs(beta[i - 1]) : 0.0) + (i + 1 < k ? fabs(beta[i]) : 0.0);
        glo = fmin(glo, alpha[i] - r);
        ghi = fmax(ghi, alpha[i] + r);
        tscale = fmax(tscale, fmax(fabs(alpha[i]), i + 1 < k ? fabs(beta[i]) : 0.0));
    }
    bool broken = false;
    for (int i = 0; i + 1 < k; ++i) broken = broken || !(fabs(beta[i]) > 1e-10 * tscale);
    auto count_below = [&](double x) {  // eigenvalues of T smaller than x
        int cnt = 0;
        double d = 1.0;
        for (int i = 0; i < k; ++i) {
            const double b2 = i > 0 ? beta[i - 1] * beta[i - 1] : 0.0;
            d = alpha[i] - x - (i > 0 ? b2 / d : 0.0);
            if (d == 0.0) d = -1e-300;
            if (d < 0.0) ++cnt;
        }
        return cnt;
    };
    if (j < k) {
        double lo = glo, hi = ghi;  // j-th smallest eigenvalue: first x with count_below(x) >= j + 1
        for (int it = 0; it < 64; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (count_below(mid) >= j + 1) hi = mid; else lo = mid;
        }
        const double t = 0.5 * (lo + hi);
        double pm = 0.0, pc = 1.0, sum = 1.0;  // p_{-1}, p_0
        for (int i = 0; i + 1 < k; ++i) {
            const double bi = beta[i];
            if (!(fabs(bi) > 1e-300)) break;   // breakdown: the rest of T is decoupled
            const double pn = ((t - alpha[i]) * pc - (i > 0 ? beta[i - 1] * pm : 0.0)) / bi;
            pm = pc; pc = pn;
            sum = fma(pn, pn, sum);
            if (!(sum < 1e280)) break;
        }
        th[j] = t;
        wt[j] = 1.0 / sum;
    }
    __syncwarp();
    if (j == 0) {
        const double emin = th[0], emax = th[k - 1], spread = emax - emin;
        out[0] = emin - margin * spread;
        out[1] = emax + margin * spread;
        double tot = 0.0;
        for (int i = 0; i < k; ++i) tot += wt[i];
        double cum = 0.0;
        for (int i = 0; i < 32; ++i) {
            if (i < k) cum += wt[i] / tot;
            out[2 + i] = i < k ? th[i] : th[k - 1];
            out[2 + 32 + i] = i < k ? cum : 1.0;
        }
        out[66] = broken ? 1.0 : 0.0;
    }
}

// The whole Lanczos run in ONE cooperative launch (grid-wide barriers instead of ~5 launches per step):
// start vector; per step  w = K v (block-CSC mat-vec, one warp per block column, columns dealt to the warps
// in a fixed order), alpha = w.v, w -= alpha v + beta_prev v_prev, beta = ||w||, v_next = w / beta;
// finally the Gauss quadrature of T.  Reductions: per-CTA partials in a fixed order, then the same fixed-order
// sum over the CTAs in every thread that needs it -- deterministic, no floating-point atomics.
__global__ void __launch_bounds__(256, 4)
k_lz_fused(int nb, int64_t n, int steps, const int32_t* __restrict__ blk_size, const int32_t* __restrict__ blk_off,
           const int64_t* __restrict__ colptr, const int4* __restrict__ rec,
           const uint32_t* __restrict__ vmap, const int64_t* __restrict__ val_off,
           const double* __restrict__ vals, double* __restrict__ vb0, double* __restrict__ vb1, double* __restrict__ vb2,
           double* __restrict__ alpha, double* __restrict__ beta, double* __restrict__ part, double margin,
           double* __restrict__ outp) {
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    __shared__ double s_red[8];
    __shared__ double s_th[32], s_wt[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int gw = blockIdx.x * 8 + wid, nwarps = gridDim.x * 8;
    const int64_t gtid = (int64_t)blockIdx.x * 256 + threadIdx.x, gthreads = (int64_t)gridDim.x * 256;
    double *vprev = vb0, *v = vb1, *w = vb2;
    {   // start vector: +-1/sqrt(n) by an integer hash of the index
        const double a = rsqrt((double)n);
        for (int64_t i = gtid; i < n; i += gthreads) {
            unsigned h = (unsigned)i * 2654435761u;
            h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
            v[i] = (h & 1u) ? a : -a;
            vprev[i] = 0.0;
        }
    }
    grid.sync();
    auto cta_sum = [&](double x) {  // fixed-order sum over the CTA's 8 warps; valid in thread 0
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if (lane == 0) s_red[wid] = x;
        __syncthreads();
        double t = 0.0;
        if (threadIdx.x == 0)
            for (int q = 0; q < 8; ++q) t += s_red[q];
        __syncthreads();
        return t;
    };
    auto grid_sum = [&](const double* p) {  // the same fixed-order sum over the per-CTA partials in every warp
        double t = 0.0;
        for (int q = lane; q < (int)gridDim.x; q += 32) t += p[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        return t;
    };
    double be_prev = 0.0;
    for (int j = 0; j < steps; ++j) {
        // w = K v, partial of w.v
        double dot = 0.0;
        for (int c = gw; c < nb; c += nwarps) {
            const int bc = blk_size[c], oc = blk_off[c];
            double d;
            if (vmap && (bc == 1 || bc == 4 || bc == 5)) {
                const int64_t v0 = val_off[c], v1 = val_off[c + 1];  // val_off: first value per block COLUMN here
                if (bc == 1) d = lz_col_s<1>(lane, oc, v0, v1, vmap, vals, v, w);
                else if (bc == 4) d = lz_col_s<4>(lane, oc, v0, v1, vmap, vals, v, w);
                else d = lz_col_s<5>(lane, oc, v0, v1, vmap, vals, v, w);
                dot += d;
                continue;
            }
            const int64_t p0 = colptr[c], p1 = colptr[c + 1];
            switch (bc) {
                case 1: d = lz_col<1>(lane, oc, p0, p1, rec, vals, v, w); break;
                case 4: d = lz_col<4>(lane, oc, p0, p1, rec, vals, v, w); break;
                case 5: d = lz_col<5>(lane, oc, p0, p1, rec, vals, v, w); break;
                case 13: d = lz_col<13>(lane, oc, p0, p1, rec, vals, v, w); break;
                default:
                    d = 0.0;
                    for (int q = 0; q < bc; ++q) {
                        double a = 0.0;
                        for (int64_t b = p0 + lane; b < p1; b += 32) {
                            const int4 rc = __ldg(rec + b);
                            const int br = rc.w;
                            const double* col = vals + (((int64_t)rc.y << 32) | (int64_t)(uint32_t)rc.x) + (size_t)q * br;
                            const double* xr = v + rc.z;
                            for (int e = 0; e < br; ++e) a = fma(col[e], xr[e], a);
                        }
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                        if (lane == 0) w[oc + q] = a;
                        d = fma(a, v[oc + q], d);
                    }
            }
            dot += d;  // identical in every lane
        }
        {
            const double t = cta_sum(lane == 0 ? dot : 0.0);
            if (threadIdx.x == 0) part[blockIdx.x] = t;
        }
        grid.sync();
        const double al = grid_sum(part);
        if (gtid == 0) alpha[j] = al;
        // w -= alpha v + beta_prev v_prev, partial of ||w||^2
        double nrm = 0.0;
        for (int64_t i = gtid; i < n; i += gthreads) {
            const double t = w[i] - al * v[i] - be_prev * vprev[i];
            w[i] = t;
            nrm = fma(t, t, nrm);
        }
        {
            const double t = cta_sum(nrm);
            if (threadIdx.x == 0) part[gridDim.x + blockIdx.x] = t;
        }
        grid.sync();
        const double be = sqrt(grid_sum(part + gridDim.x));
        if (gtid == 0) beta[j] = be;
        const double inv = be > 1e-300 ? 1.0 / be : 0.0;
        for (int64_t i = gtid; i < n; i += gthreads) vprev[i] = w[i] * inv;  // v_{j+1} over v_{j-1}
        grid.sync();
        double* t = vprev; vprev = v; v = t;
        be_prev = be;
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) lz_quadrature_body(steps, alpha, beta, margin, outp, s_th, s_wt);
}

// s_g <- min(Gershgorin_g, max(cap, rho_lo_g)) / overshoot  (in place, bits of a double as written by
// k_gather; rho_lo_g = largest column 2-norm of a_g - mu I, a rigorous lower bound of its spectral radius:
// the estimated cap is never taken below it).
// With alpha != null (reading A8b) the overshoot is not applied; instead iteration 0 works on al_0 X_0 with
// al_0 = min(sqrt(3 / (1 + l + l^2)), 1.5), l = ell_abs / s_g the estimated smallest eigenvalue modulus of X_0
// (1.5: the same safety against an underestimated bound as the overshoot limit of reading A8).
__global__ void k_apply_scale(int ng, unsigned long long* __restrict__ gersh,
                              const unsigned long long* __restrict__ col2, double cap, double inv_overshoot,
                              double ell_abs, double* __restrict__ alpha, double* __restrict__ lmin) {
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ng) return;
    double s = __longlong_as_double((long long)gersh[g]);
    const double c = fmax(cap, sqrt(__longlong_as_double((long long)col2[g])));
    if (cap > 0.0 && c < s) s = c;
    if (alpha) {
        double l = s > 0.0 ? ell_abs / s : 1.0;
        l = fmin(fmax(l, 1e-4), 1.0);
        alpha[g] = l < 0.9999 ? fmin(sqrt(3.0 / (1.0 + l + l * l)), 1.5) : 1.0;
        lmin[g] = l;
    } else {
        s *= inv_overshoot;
    }
    gersh[g] = (unsigned long long)__double_as_longlong(s);
}

sm_status_t launch_apply_scale(sm_plan* p, double cap, double overshoot, double ell_abs, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    const bool resc = rescale_on(p);
    k_apply_scale<<<(p->ngroups + 255) / 256, 256, 0, st>>>(p->ngroups, p->d_gersh, p->d_gersh + p->ngroups, cap,
                                                            1.0 / overshoot, ell_abs,
                                                            resc ? p->d_alpha : nullptr, resc ? p->d_lmin : nullptr);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// Lanczos estimate of [lambda_min, lambda_max] of K~ -> p->lz_lo / p->lz_hi (host), widened by 3 %
// of the spread, + the quadrature nodes.  One cooperative launch, LZ_STEPS steps.
sm_status_t launch_lanczos_bounds(sm_plan* p, const double* vals, cudaStream_t st) {
    int64_t n = p->info.n_basis;
    if (n == 0 || p->nb == 0) { p->lz_lo = p->lz_hi = 0.0; p->lz_ok = 0; return SM_OK; }
    if (!p->lz_grid) {  // as many CTAs as are co-resident (grid-wide barriers), at most 4 per SM
        int per_sm = 0;
        SM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_lz_fused, 256, 0));
        if (per_sm < 1) return SM_ERR_CUDA;
        p->lz_grid = p->num_sms * std::min(per_sm, 4);
    }
    if (!p->d_lz) SM_CUDA(cudaMalloc((void**)&p->d_lz, (size_t)(3 * n + 2 * LZ_STEPS + 72 + 2 * p->lz_grid) * 8));
    double *vb0 = p->d_lz, *vb1 = p->d_lz + n, *vb2 = p->d_lz + 2 * n;
    double* alpha = p->d_lz + 3 * n;
    double* beta = alpha + LZ_STEPS;
    double* outp = beta + LZ_STEPS;
    double* part = outp + 72;
    int steps = (int)std::min<int64_t>(LZ_STEPS, n), nb = p->nb;
    double margin = 0.03;
    if (!p->d_lz_map && n < (1 << 28)) {  // once per plan (pattern only): the map of the streaming mat-vec
        SM_CUDA(cudaMalloc((void**)&p->d_lz_map, (size_t)std::max<int64_t>(p->nnz, 1) * 4));
        k_lz_map<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_blk_off, p->d_colptr, p->d_rowidx, p->d_val_off,
                                                p->d_lz_map);
        p->launches++;
    }
    void* args[] = {&nb, &n, &steps, &p->d_blk_size, &p->d_blk_off, &p->d_colptr, &p->d_lz_rec, &p->d_lz_map, &p->d_col_val, &vals,
                    &vb0, &vb1, &vb2, &alpha, &beta, &part, &margin, &outp};
    SM_CUDA(cudaLaunchCooperativeKernel((const void*)k_lz_fused, dim3(p->lz_grid), dim3(256), args, 0, st));
    p->launches++;
    SM_CUDA(cudaMemcpyAsync(p->h_lz, outp, 67 * 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    p->lz_lo = p->h_lz[0];
    p->lz_hi = p->h_lz[1];
    p->lz_nodes = steps;
    // a broken-down or non-finite run is discarded: Gershgorin bounds only for this call (reading A8)
    p->lz_ok = (p->h_lz[66] == 0.0 && p->lz_lo == p->lz_lo && p->lz_hi == p->lz_hi && p->lz_lo <= p->lz_hi) ? 1 : 0;
    return SM_OK;
}

}  // namespace smb
