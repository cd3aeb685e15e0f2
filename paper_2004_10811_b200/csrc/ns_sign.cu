// a5 batched Newton-Schulz sign iteration (Eq.(11)):  X_{k+1} = 1/2 X_k (3 I - X_k^2),
// convergence monitor ||X_k^2 - I||_F / sqrt(n) (involutority, L354 / Fig.13).
//
// Two kernels per iteration over ALL submatrices at once (one CTA per 64x64 lower-triangular tile):
//   MODE 0:  Y  = alpha * X X          + per-tile partial of ||Y - I||_F^2
//   MODE 1:  X' = a X + b (X Y)        (a = 3/2, b = -1/2; iteration 0 folds the spectral scale
//                                        1/s_i into alpha, a, b so that no scaling pass is needed)
// X, Y and X' are symmetric polynomials of the same matrix, so only tiles on or below the diagonal
// are computed and every element is stored together with its mirror image: the stored matrices are
// bitwise symmetric, which also lets both GEMM operands be read as k-contiguous rows
// (B[k][n] = Y[n][k]).  FP64 math runs on the tensor-core DMMA path (mma.sync m8n8k4 f64 -- the
// only FP64 MMA sm_100a has; tcgen05 has no f64 kind), fed from shared memory by a 3-stage
// cp.async pipeline.  MODE 1 first reduces the per-tile partials of its submatrix in a fixed
// order (deterministic, no atomics on doubles) and decides convergence per submatrix.
#include "common.cuh"

namespace smb {

constexpr int BM = TILE, BN = TILE, BK = 16, STAGES = 3;
// Row stride of the staged operand tiles: 24 doubles = 192 B.  Fragments are read with 16-byte
// loads (two consecutive k per lane); consecutive rows then start 64 B apart modulo 128 B, so the
// eight lanes of a quarter-warp (2 rows x 4 lanes x 16 B) hit all 32 banks once: conflict-free.
constexpr int LDS_ROW = BK + 8;
constexpr int NTHREADS = 128;    // 4 warps as 2 x 2, warp tile 32 x 32 = 4 x 4 DMMA tiles
constexpr size_t NS_SMEM = (size_t)STAGES * (BM + BN) * LDS_ROW * sizeof(double);

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// One staged k-tile (BK = 16) of a warp's 32 x 32 tile: MT x NT DMMA sub-tiles (TRI: only nt <= mt).
// The contraction index may be visited in any order as long as A and B agree: lane (lr, lk) loads
// the two consecutive k = 8 j + 2 lk + {0,1} with one 16-byte load; the first DMMA of a pair
// contracts the even k of the 8-wide group, the second the odd k.
template <int MT, int NT, bool TRI>
__device__ __forceinline__ void ktile_mma(double (&acc)[4][4][2], const double* __restrict__ Aw,
                                          const double* __restrict__ Bw) {
#pragma unroll
    for (int j = 0; j < BK / 8; ++j) {
        double2 af[MT], bf[NT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) af[mt] = *reinterpret_cast<const double2*>(Aw + mt * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) bf[nt] = *reinterpret_cast<const double2*>(Bw + nt * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
                if (!TRI || nt <= mt) {
                    dmma(acc[mt][nt][0], acc[mt][nt][1], af[mt].x, bf[nt].x);
                    dmma(acc[mt][nt][0], acc[mt][nt][1], af[mt].y, bf[nt].y);
                }
    }
}

struct NsArgs {
    const TileDesc* tiles;
    const int64_t* ws_off;
    const int32_t* ld;
    const int32_t* dim;
    const int32_t* tile_first;
    const int32_t* tile_count;
    const unsigned long long* gersh;
    double* buf0;
    double* buf1;
    double* bufY;
    double* partials;
    int32_t* done_iter;
    int32_t* flag;
    double* res;  // [2][ngroups]
    int32_t* counters;
    int32_t ngroups;
    int32_t k;
    int32_t decide_only;  // k == max_iter: only record the decision, no update
    double eps;
};

template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 3) k_ns_gemm(NsArgs a) {
    extern __shared__ __align__(16) double smem[];
    __shared__ double s_red[4];
    __shared__ int s_stop;
    const TileDesc td = a.tiles[blockIdx.x];
    const int g = td.grp;
    if (a.done_iter[g] >= 0) return;
    const int ti = td.tij & 0xffff, tj = td.tij >> 16;
    const int ld = a.ld[g], n = a.dim[g];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int k = a.k;
    double s = __longlong_as_double((long long)a.gersh[g]);
    if (!(s > 0.0)) s = 1.0;

    if (MODE == 1) {
        // residual of X_k from the partials MODE 0 just wrote; fixed summation order
        if (wid == 0) {
            const int t0 = a.tile_first[g], tc = a.tile_count[g];
            double r2 = 0.0;
            for (int t = lane; t < tc; t += 32) r2 += a.partials[t0 + t];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
            if (lane == 0) {
                const double r = sqrt(r2 / (double)(n > 0 ? n : 1));
                const double prev = k > 0 ? a.res[(size_t)((k - 1) & 1) * a.ngroups + g] : 1e300;
                const bool conv = r < a.eps;
                const bool stag = (k > 0) && (r >= prev) && (r < 1e-6);
                const bool stop = conv || stag || a.decide_only || !(r == r);
                s_stop = stop ? 1 : 0;
                if (blockIdx.x == (unsigned)t0) {  // one CTA per submatrix records the decision
                    a.res[(size_t)(k & 1) * a.ngroups + g] = r;
                    if (stop) {
                        a.done_iter[g] = k;
                        a.flag[g] = conv ? 0 : 1;
                        if (!conv) a.res[(size_t)((k + 1) & 1) * a.ngroups + g] = r;
                    } else {
                        atomicAdd(a.counters + k, 1);
                    }
                }
            }
        }
        __syncthreads();
        if (s_stop) return;
    }

    const double* X = ((k & 1) ? a.buf1 : a.buf0) + a.ws_off[g];
    const double* Aop = X;
    const double* Bop = (MODE == 0) ? X : (a.bufY + a.ws_off[g]);
    const int row0 = ti * BM, col0 = tj * BN;
    const bool diag = (ti == tj);

    double* As = smem;
    double* Bs = smem + (size_t)STAGES * BM * LDS_ROW;
    const int KT = (ld + BK - 1) / BK;

    auto load_stage = [&](int stage, int kt) {
        const int k0 = kt * BK;
#pragma unroll
        for (int i = 0; i < (BM * BK / 2) / NTHREADS; ++i) {
            const int id = tid + i * NTHREADS;
            const int r = id >> 3, ch = id & 7;
            const int kk = k0 + ch * 2;
            {
                const int gr = row0 + r;
                const bool ok = (gr < ld) && (kk < ld);
                const double* src = ok ? (Aop + (size_t)gr * ld + kk) : Aop;
                cp_async16(As + ((size_t)stage * BM + r) * LDS_ROW + ch * 2, src, ok ? 16 : 0);
            }
            {
                const int gr = col0 + r;
                const bool ok = (gr < ld) && (kk < ld);
                const double* src = ok ? (Bop + (size_t)gr * ld + kk) : Bop;
                cp_async16(Bs + ((size_t)stage * BN + r) * LDS_ROW + ch * 2, src, ok ? 16 : 0);
            }
        }
    };

    const int wm = wid >> 1, wn = wid & 1;
    // Work of this warp: number of valid 8-row sub-tile rows (the padded matrix ends inside the last
    // tile) and, on diagonal tiles, only the sub-tiles that touch the lower triangle.  Off-diagonal
    // tiles always have all 64 columns (tj < ti <= last).  Warp-uniform: dispatched once per k-tile.
    const int rows_left = ld - (row0 + wm * 32), cols_left = ld - (col0 + wn * 32);
    int mt_cnt = rows_left <= 0 ? 0 : (rows_left >= 32 ? 4 : rows_left >> 3);
    int nt_cnt = cols_left <= 0 ? 0 : (cols_left >= 32 ? 4 : cols_left >> 3);
    bool tri = false;
    if (diag) {
        if (wm < wn) mt_cnt = 0;          // entirely above the diagonal
        else if (wm == wn) tri = true;    // mt_cnt == nt_cnt here
    }
    if (nt_cnt == 0) mt_cnt = 0;
    const int variant = mt_cnt == 0 ? 0 : (tri ? 4 + mt_cnt : mt_cnt);  // 1..4 FULL<MT,nt>, 5..8 TRI<S>

    double acc[4][4][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

#pragma unroll
    for (int st = 0; st < STAGES - 1; ++st) {
        if (st < KT) load_stage(st, st);
        cp_async_commit();
    }
    const int lr = lane >> 2, lk = lane & 3;
    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int nk = kt + STAGES - 1;
            if (nk < KT) load_stage(nk % STAGES, nk);
            cp_async_commit();
        }
        const int stage = kt % STAGES;
        const double* Aw = As + ((size_t)stage * BM + wm * 32 + lr) * LDS_ROW + 2 * lk;
        const double* Bw = Bs + ((size_t)stage * BN + wn * 32 + lr) * LDS_ROW + 2 * lk;
        if (nt_cnt == 4 || tri) {
            switch (variant) {
                case 4: ktile_mma<4, 4, false>(acc, Aw, Bw); break;
                case 3: ktile_mma<3, 4, false>(acc, Aw, Bw); break;
                case 2: ktile_mma<2, 4, false>(acc, Aw, Bw); break;
                case 1: ktile_mma<1, 4, false>(acc, Aw, Bw); break;
                case 8: ktile_mma<4, 4, true>(acc, Aw, Bw); break;
                case 7: ktile_mma<3, 3, true>(acc, Aw, Bw); break;
                case 6: ktile_mma<2, 2, true>(acc, Aw, Bw); break;
                case 5: ktile_mma<1, 1, true>(acc, Aw, Bw); break;
                default: break;
            }
        } else if (variant) {
            // cannot happen for lower-triangular tiles (see above); kept for safety: full 4 x 4 on
            // zero-filled operands is still correct
            ktile_mma<4, 4, false>(acc, Aw, Bw);
        }
    }
    cp_async_wait<0>();

    // ------------------------------------------------------------------ epilogue
    double alpha, ca, cb;
    if (k == 0) { alpha = 1.0 / (s * s); ca = 1.5 / s; cb = -0.5 / s; }
    else { alpha = 1.0; ca = 1.5; cb = -0.5; }
    double* Out = (MODE == 0) ? (a.bufY + a.ws_off[g]) : (((k & 1) ? a.buf0 : a.buf1) + a.ws_off[g]);
    double part = 0.0;
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            if (mt >= mt_cnt || nt >= nt_cnt || (tri && nt > mt)) continue;
            const int r = row0 + wm * 32 + mt * 8 + lr;
            const int c = col0 + wn * 32 + nt * 8 + 2 * lk;
            if (r >= ld || c >= ld) continue;  // ld is a multiple of 8: whole sub-tile in or out
            double v0 = acc[mt][nt][0], v1 = acc[mt][nt][1];
            if (MODE == 0) {
                v0 *= alpha; v1 *= alpha;
                if (r < n) {  // residual over the n x n part; strictly-lower elements count twice
                    if (c < n && c <= r) { double d = v0 - (c == r ? 1.0 : 0.0); part += (c == r ? 1.0 : 2.0) * d * d; }
                    if (c + 1 < n && c + 1 <= r) { double d = v1 - (c + 1 == r ? 1.0 : 0.0); part += (c + 1 == r ? 1.0 : 2.0) * d * d; }
                }
            } else {
                const double2 x = *reinterpret_cast<const double2*>(X + (size_t)r * ld + c);
                v0 = ca * x.x + cb * v0;
                v1 = ca * x.y + cb * v1;
            }
            if (!diag) {
                *reinterpret_cast<double2*>(Out + (size_t)r * ld + c) = make_double2(v0, v1);
                Out[(size_t)c * ld + r] = v0;
                Out[(size_t)(c + 1) * ld + r] = v1;
            } else {  // diagonal tile: keep the lower triangle, mirror it
                if (c <= r) { Out[(size_t)r * ld + c] = v0; if (c != r) Out[(size_t)c * ld + r] = v0; }
                if (c + 1 <= r) { Out[(size_t)r * ld + c + 1] = v1; if (c + 1 != r) Out[(size_t)(c + 1) * ld + r] = v1; }
            }
        }
    if (MODE == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if (lane == 0) s_red[wid] = part;
        __syncthreads();
        if (tid == 0) a.partials[blockIdx.x] = (s_red[0] + s_red[1]) + (s_red[2] + s_red[3]);
    }
}

sm_status_t launch_ns_pair(sm_plan* p, int k, double eps, int decide_only, double* buf0, double* buf1,
                           double* bufY, cudaStream_t st) {
    if (p->n_tiles == 0) return SM_OK;
    static bool attr_set = false;
    if (!attr_set) {
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        attr_set = true;
    }
    NsArgs a;
    a.tiles = p->d_tiles; a.ws_off = p->d_ws_off; a.ld = p->d_ld; a.dim = p->d_sub_dim;
    a.tile_first = p->d_tile_first; a.tile_count = p->d_tile_count; a.gersh = p->d_gersh;
    a.buf0 = buf0; a.buf1 = buf1; a.bufY = bufY; a.partials = p->d_partials;
    a.done_iter = p->d_done_iter; a.flag = p->d_flag; a.res = p->d_res; a.counters = p->d_counters;
    a.ngroups = p->ngroups; a.k = k; a.decide_only = decide_only; a.eps = eps;
    k_ns_gemm<0><<<(unsigned)p->n_tiles, NTHREADS, NS_SMEM, st>>>(a);
    k_ns_gemm<1><<<(unsigned)p->n_tiles, NTHREADS, NS_SMEM, st>>>(a);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

}  // namespace smb
