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
//
// Work split inside a CTA (4 warps).  The FP64 pipe is per SM sub-partition, so the four warps of
// a CTA must carry equal work whatever the tile looks like:
//   * rectangular tiles (off-diagonal, or the small last diagonal tile): warp w owns the two
//     8-column sub-tiles 2w, 2w+1 and ALL valid 8-row sub-tiles (M = 1..8, the padded matrix may
//     end inside the tile): M x 2 DMMA tiles per warp, identical for the four warps;
//   * full diagonal tiles: only the 36 sub-tiles on or below the diagonal are needed; warp w owns
//     the sub-tile rows w and 7-w, i.e. (w+1) + (8-w) = 9 sub-tiles for every warp.
#include "common.cuh"

namespace smb {

constexpr int BM = TILE, BN = TILE, BK = 16, STAGES = 3;
// Row stride of the staged operand tiles: 24 doubles = 192 B.  Fragments are read with 16-byte
// loads (two consecutive k per lane); consecutive rows then start 64 B apart modulo 128 B, so the
// eight lanes of a quarter-warp (2 rows x 4 lanes x 16 B) hit all 32 banks once: conflict-free.
constexpr int LDS_ROW = BK + 8;
constexpr int NTHREADS = 128;
constexpr size_t NS_SMEM = (size_t)STAGES * (BM + BN) * LDS_ROW * sizeof(double);

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// The contraction index may be visited in any order as long as A and B agree: lane (lr, lk) loads
// the two consecutive k = 8 j + 2 lk + {0,1} with one 16-byte load; the first DMMA of a pair
// contracts the even k of the 8-wide group, the second the odd k.
//
// Rectangular tile: M valid row sub-tiles x this warp's 2 column sub-tiles.  acc[2 mt + nt].
// Ap = stage A + lr * LDS_ROW + 2 lk;  Bp = stage B + (16 w + lr) * LDS_ROW + 2 lk.
template <int M>
__device__ __forceinline__ void ktile_rect(double (&acc)[16][2], const double* __restrict__ Ap,
                                           const double* __restrict__ Bp) {
#pragma unroll
    for (int j = 0; j < BK / 8; ++j) {
        double2 bf[2], af[M];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) bf[nt] = *reinterpret_cast<const double2*>(Bp + nt * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int mt = 0; mt < M; ++mt) af[mt] = *reinterpret_cast<const double2*>(Ap + mt * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int mt = 0; mt < M; ++mt)
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) dmma(acc[2 * mt + nt], af[mt].x, bf[nt].x);
#pragma unroll
        for (int mt = 0; mt < M; ++mt)
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) dmma(acc[2 * mt + nt], af[mt].y, bf[nt].y);
    }
}

// Full diagonal tile, warp W: sub-tile row W with columns 0..W  -> acc[0..W],
//                             sub-tile row 7-W with columns 0..7-W -> acc[W+1 .. 8].
// Ap = stage A + lr * LDS_ROW + 2 lk;  Bp = stage B + lr * LDS_ROW + 2 lk.
template <int W>
__device__ __forceinline__ void ktile_diag(double (&acc)[16][2], const double* __restrict__ Ap,
                                           const double* __restrict__ Bp) {
    constexpr int RA = W, RB = 7 - W, NB = 8 - W;
#pragma unroll
    for (int j = 0; j < BK / 8; ++j) {
        double2 bf[NB];
        const double2 aa = *reinterpret_cast<const double2*>(Ap + RA * 8 * LDS_ROW + j * 8);
        const double2 ab = *reinterpret_cast<const double2*>(Ap + RB * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int c = 0; c < NB; ++c) bf[c] = *reinterpret_cast<const double2*>(Bp + c * 8 * LDS_ROW + j * 8);
#pragma unroll
        for (int c = 0; c <= W; ++c) dmma(acc[c], aa.x, bf[c].x);
#pragma unroll
        for (int c = 0; c < NB; ++c) dmma(acc[W + 1 + c], ab.x, bf[c].x);
#pragma unroll
        for (int c = 0; c <= W; ++c) dmma(acc[c], aa.y, bf[c].y);
#pragma unroll
        for (int c = 0; c < NB; ++c) dmma(acc[W + 1 + c], ab.y, bf[c].y);
    }
}

struct NsArgs {
    const TileDesc* tiles;
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
    const int4* tdp = reinterpret_cast<const int4*>(a.tiles + blockIdx.x);
    const int4 t0 = __ldg(tdp), t1 = __ldg(tdp + 1);
    const int64_t ws_off = ((int64_t)(unsigned)t0.x) | ((int64_t)t0.y << 32);
    const int g = t0.z, ld = t0.w, n = t1.x, tij = t1.y, tile_first = t1.z, tile_count = t1.w;
    if (a.done_iter[g] >= 0) return;
    const int ti = tij & 0xffff, tj = tij >> 16;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int k = a.k;

    const double* X = ((k & 1) ? a.buf1 : a.buf0) + ws_off;
    const double* Aop = X;
    const double* Bop = (MODE == 0) ? X : (a.bufY + ws_off);
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

    // start filling the pipeline before anything else (MODE 1 decides convergence meanwhile)
#pragma unroll
    for (int st = 0; st < STAGES - 1; ++st) {
        if (st < KT) load_stage(st, st);
        cp_async_commit();
    }

    if (MODE == 1) {
        // residual of X_k from the partials MODE 0 just wrote; fixed summation order
        if (wid == 0) {
            double r2 = 0.0;
            for (int t = lane; t < tile_count; t += 32) r2 += a.partials[tile_first + t];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
            if (lane == 0) {
                const double r = sqrt(r2 / (double)(n > 0 ? n : 1));
                const double prev = k > 0 ? a.res[(size_t)((k - 1) & 1) * a.ngroups + g] : 1e300;
                const bool conv = r < a.eps;
                const bool stag = (k > 0) && (r >= prev) && (r < 1e-6);
                const bool stop = conv || stag || a.decide_only || !(r == r);
                s_stop = stop ? 1 : 0;
                if (blockIdx.x == (unsigned)tile_first) {  // one CTA per submatrix records the decision
                    a.res[(size_t)(k & 1) * a.ngroups + g] = r;
                    if (stop) {
                        a.done_iter[g] = k;
                        a.flag[g] = conv ? 0 : 1;
                    } else {
                        atomicAdd(a.counters + k, 1);
                    }
                }
            }
        }
        __syncthreads();
        if (s_stop) {
            cp_async_wait<0>();
            return;
        }
    }

    // Warp-uniform work selection (see the file header).
    const int s_rows = min(8, (ld - row0) >> 3);  // valid 8-row sub-tile rows of this tile, 1..8
    const bool full_diag = diag && s_rows == 8;
    int variant;  // 0 idle, 1..8 rect<M>, 9..12 diag<W>
    if (full_diag) variant = 9 + wid;
    else if (diag) variant = (2 * wid < s_rows) ? s_rows : 0;  // columns past the matrix: nothing to do
    else variant = s_rows;

    double acc[16][2];
#pragma unroll
    for (int e = 0; e < 16; ++e) acc[e][0] = acc[e][1] = 0.0;

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
        const double* Ap = As + ((size_t)stage * BM + lr) * LDS_ROW + 2 * lk;
        const double* Bp0 = Bs + ((size_t)stage * BN + lr) * LDS_ROW + 2 * lk;
        const double* Bp = Bp0 + (size_t)wid * 16 * LDS_ROW;
        switch (variant) {
            case 8: ktile_rect<8>(acc, Ap, Bp); break;
            case 7: ktile_rect<7>(acc, Ap, Bp); break;
            case 6: ktile_rect<6>(acc, Ap, Bp); break;
            case 5: ktile_rect<5>(acc, Ap, Bp); break;
            case 4: ktile_rect<4>(acc, Ap, Bp); break;
            case 3: ktile_rect<3>(acc, Ap, Bp); break;
            case 2: ktile_rect<2>(acc, Ap, Bp); break;
            case 1: ktile_rect<1>(acc, Ap, Bp); break;
            case 9: ktile_diag<0>(acc, Ap, Bp0); break;
            case 10: ktile_diag<1>(acc, Ap, Bp0); break;
            case 11: ktile_diag<2>(acc, Ap, Bp0); break;
            case 12: ktile_diag<3>(acc, Ap, Bp0); break;
            default: break;
        }
    }
    cp_async_wait<0>();

    // ------------------------------------------------------------------ epilogue
    double s = __longlong_as_double((long long)a.gersh[g]);
    if (!(s > 0.0)) s = 1.0;
    double alpha, ca, cb;
    if (k == 0) { alpha = 1.0 / (s * s); ca = 1.5 / s; cb = -0.5 / s; }
    else { alpha = 1.0; ca = 1.5; cb = -0.5; }
    double* Out = (MODE == 0) ? (a.bufY + ws_off) : (((k & 1) ? a.buf0 : a.buf1) + ws_off);
    double part = 0.0;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        int sr, sc;  // sub-tile row / column inside the CTA tile
        bool valid;
        if (full_diag) {
            valid = e < 9;
            if (e <= wid) { sr = wid; sc = e; } else { sr = 7 - wid; sc = e - wid - 1; }
        } else {
            sr = e >> 1; sc = 2 * wid + (e & 1);
            valid = variant != 0 && sr < s_rows;
        }
        if (!valid) continue;
        const int r = row0 + sr * 8 + lr;
        const int c = col0 + sc * 8 + 2 * lk;
        if (r >= ld || c >= ld) continue;  // ld is a multiple of 8: whole sub-tile in or out
        double v0 = acc[e][0], v1 = acc[e][1];
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
    a.tiles = p->d_tiles; a.gersh = p->d_gersh;
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
