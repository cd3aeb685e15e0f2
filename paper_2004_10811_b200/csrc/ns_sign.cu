// a5 batched Newton-Schulz sign iteration (Eq.(11)):  X_{k+1} = 1/2 X_k (3 I - X_k^2),
// convergence monitor ||X_k^2 - I||_F / sqrt(n) (involutority, L354 / Fig.13).
//
// Two persistent kernels per iteration over ALL submatrices at once; the unit of work is one 64x64
// lower-triangular tile of one submatrix, handed out by an atomic counter:
//   MODE 0:  Y  = alpha * X X          + ||Y - I||_F^2 per tile; the CTA that finishes the last
//                                        tile of a submatrix sums the partials in a fixed order and
//                                        records the convergence decision (deterministic)
//   MODE 1:  X' = a X + b (X Y)        (a = 3/2, b = -1/2; iteration 0 folds the spectral scale
//                                        1/s_i into alpha, a, b so that no scaling pass is needed)
// X, Y and X' are symmetric polynomials of the same matrix, so only tiles on or below the diagonal
// are computed and every element is stored together with its mirror image: the stored matrices are
// bitwise symmetric, which also lets both GEMM operands be read as k-contiguous rows
// (B[k][n] = Y[n][k]).
//
// Data movement (sm_100a): matrices live in the k8-panel layout of common.cuh, so the 64 x 16
// operand slice of one pipeline stage is ONE contiguous block; a producer warp streams it with
// cp.async.bulk (TMA, SASS UBLKCP) into a 4-stage shared-memory ring, completion counted on
// mbarriers (complete_tx).  Four consumer warps wait on the "full" barrier of a stage, issue the
// FP64 tensor-core MMAs (mma.sync m8n8k4 f64 -> SASS DMMA; tcgen05 has no f64 kind) and release the
// stage on its "empty" barrier.  There is no CTA-wide barrier in the main loop, and the producer
// runs ahead across tile boundaries, so the next tile's operands are already in flight while the
// consumers write the current tile's epilogue.
//
// Work split among the 4 consumer warps.  The FP64 pipe is per SM sub-partition, so the four warps
// must carry equal work whatever the tile looks like:
//   * rectangular tiles (off-diagonal, or the small last diagonal tile): warp w owns the two
//     8-column sub-tiles 2w, 2w+1 and ALL valid 8-row sub-tiles (M = 1..8, the padded matrix may
//     end inside the tile): M x 2 DMMA tiles per warp, identical for the four warps;
//   * full diagonal tiles: only the 36 sub-tiles on or below the diagonal are needed; warp w owns
//     the sub-tile rows w and 7-w, i.e. (w+1) + (8-w) = 9 sub-tiles for every warp.
// MODE 1 needs a X[r][c] at the accumulator's own position: that value passes through the A
// fragments when the k loop crosses the tile's own columns, where it is folded into the
// accumulator (acc += -3 x, result = b acc), so the epilogue reads nothing from global memory.
#include <algorithm>

#include "common.cuh"

namespace smb {

constexpr int BM = TILE, BN = TILE, BK = 16, STAGES = 4;
constexpr int NCONSUMER = 128, NTHREADS = NCONSUMER + 32;
constexpr int STAGE_DOUBLES = (BM + BN) * BK;  // A slice then B slice, dense
constexpr size_t NS_SMEM = (size_t)STAGES * STAGE_DOUBLES * sizeof(double);

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

// ---- mbarrier / bulk-copy primitives
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Per-stage metadata written by the producer before it arms the stage's "full" barrier.
struct __align__(16) StageInfo {
    int64_t ws_off;
    int32_t grp, ld, n, tij;
    int32_t tile, tile_first, tile_count;
    int32_t kt;     // k-tile index inside the tile (0 = first), -1 = no more work
    int32_t nj;     // valid 8-wide k panels in this stage (1 or 2)
    int32_t last;   // 1 = last k-tile of the tile
    int32_t rows_a, rows_b;  // valid rows of the A / B slice (B slice aliases A when b_is_a)
    int32_t b_is_a;
    int32_t pad;
};

// The contraction index may be visited in any order as long as A and B agree: lane (lr, lk) loads
// the two consecutive k = 8 j + 2 lk + {0,1} with one 16-byte load; the first DMMA of a pair
// contracts the even k of the 8-wide panel, the second the odd k.  Dense 64-byte panel rows make
// these loads conflict-free: a quarter-warp (2 rows x 4 lanes x 16 B) covers 128 contiguous bytes.
//
// Rectangular tile: M valid row sub-tiles x this warp's 2 column sub-tiles, acc[2 mt + nt].
// fold >= 0: this panel holds the tile's own column sub-tile `fold` (MODE 1: acc += -3 x).
template <int M>
__device__ __forceinline__ void panel_rect(double (&acc)[16][2], const double* __restrict__ Ap,
                                           const double* __restrict__ Bp) {
    double2 bf[2], af[M];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) bf[nt] = *reinterpret_cast<const double2*>(Bp + nt * 64);
#pragma unroll
    for (int mt = 0; mt < M; ++mt) af[mt] = *reinterpret_cast<const double2*>(Ap + mt * 64);
#pragma unroll
    for (int mt = 0; mt < M; ++mt)
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) dmma(acc[2 * mt + nt], af[mt].x, bf[nt].x);
#pragma unroll
    for (int mt = 0; mt < M; ++mt)
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) dmma(acc[2 * mt + nt], af[mt].y, bf[nt].y);
}

// Full diagonal tile, warp W: sub-tile row W with columns 0..W  -> acc[0..W],
//                             sub-tile row 7-W with columns 0..7-W -> acc[W+1 .. 8].
// fold_c >= 0: this panel holds the tile's own column sub-tile fold_c (MODE 1 only).
template <int W>
__device__ __forceinline__ void panel_diag(double (&acc)[16][2], const double* __restrict__ Ap,
                                           const double* __restrict__ Bp) {
    constexpr int RA = W, RB = 7 - W, NB = 8 - W;
    double2 bf[NB];
    const double2 aa = *reinterpret_cast<const double2*>(Ap + RA * 64);
    const double2 ab = *reinterpret_cast<const double2*>(Ap + RB * 64);
#pragma unroll
    for (int c = 0; c < NB; ++c) bf[c] = *reinterpret_cast<const double2*>(Bp + c * 64);
#pragma unroll
    for (int c = 0; c <= W; ++c) dmma(acc[c], aa.x, bf[c].x);
#pragma unroll
    for (int c = 0; c < NB; ++c) dmma(acc[W + 1 + c], ab.x, bf[c].x);
#pragma unroll
    for (int c = 0; c <= W; ++c) dmma(acc[c], aa.y, bf[c].y);
#pragma unroll
    for (int c = 0; c < NB; ++c) dmma(acc[W + 1 + c], ab.y, bf[c].y);
}

// MODE 1 only: the panel that carries the tile's own column sub-tile `sc` holds, in the A-fragment
// positions, exactly the X[r][c] of the accumulators of that column: acc += -3 x there
// (X' = b (X Y - 3 X)).  Compact, predicated code on purpose (runs on 8 of the ~27 panels of a tile).
__device__ __forceinline__ void fold_x(double (&acc)[16][2], const double* __restrict__ Ap, bool full_diag,
                                       int s_rows, int wid, int sc) {
    if (full_diag) {
        const int ea = (sc <= wid) ? sc : -1, eb = (sc <= 7 - wid) ? wid + 1 + sc : -1;
        const double2 xa = *reinterpret_cast<const double2*>(Ap + wid * 64);
        const double2 xb = *reinterpret_cast<const double2*>(Ap + (7 - wid) * 64);
#pragma unroll
        for (int e = 0; e < 9; ++e) {
            if (e == ea) { acc[e][0] = fma(-3.0, xa.x, acc[e][0]); acc[e][1] = fma(-3.0, xa.y, acc[e][1]); }
            if (e == eb) { acc[e][0] = fma(-3.0, xb.x, acc[e][0]); acc[e][1] = fma(-3.0, xb.y, acc[e][1]); }
        }
    } else if ((sc >> 1) == wid) {
        const int nt = sc & 1;
#pragma unroll
        for (int mt = 0; mt < 8; ++mt) {
            if (mt < s_rows) {
                const double2 x = *reinterpret_cast<const double2*>(Ap + mt * 64);
#pragma unroll
                for (int q = 0; q < 2; ++q)
                    if (q == nt) {
                        acc[2 * mt + q][0] = fma(-3.0, x.x, acc[2 * mt + q][0]);
                        acc[2 * mt + q][1] = fma(-3.0, x.y, acc[2 * mt + q][1]);
                    }
            }
        }
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
    int32_t* tile_done;  // [ngroups] tiles of the submatrix finished in this MODE 0 launch
    double* res;         // [2][ngroups]
    int32_t* counters;   // [max_iter+2] still-active submatrices after iteration k
    int32_t* sched;      // work counter of this launch
    int32_t n_tiles;
    int32_t ngroups;
    int32_t k;
    int32_t decide_only;  // k == max_iter: stop whatever the residual is
    double eps;
};

template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 3) k_ns_gemm(NsArgs a) {
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(16) StageInfo s_info[STAGES];
    __shared__ __align__(8) uint64_t s_full[STAGES], s_empty[STAGES];
    __shared__ double s_red[4];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int k = a.k;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const double* Xbase = (k & 1) ? a.buf1 : a.buf0;
    const double* Bbase = (MODE == 0) ? Xbase : a.bufY;

    if (wid == 4) {
        // =================================================================== producer warp
        int stage = 0;
        unsigned phase = 0;
        for (;;) {
            int tile = 0;
            if (lane == 0) tile = atomicAdd(a.sched, 1);
            tile = __shfl_sync(0xffffffffu, tile, 0);
            if (tile >= a.n_tiles) break;
            const int4* tdp = reinterpret_cast<const int4*>(a.tiles + tile);
            const int4 t0 = __ldg(tdp), t1 = __ldg(tdp + 1);
            const int g = t0.z;
            if (a.done_iter[g] >= 0) continue;
            const int64_t ws_off = ((int64_t)(unsigned)t0.x) | ((int64_t)t0.y << 32);
            const int ld = t0.w, tij = t1.y;
            const int ti = tij & 0xffff, tj = tij >> 16;
            const int row0 = ti * BM, col0 = tj * BN;
            const int rows_a = min(BM, ld - row0), rows_b = min(BN, ld - col0);
            const bool b_is_a = (MODE == 0) && (ti == tj);
            const int KP = ld >> 3;            // 8-wide k panels
            const int KT = (KP + 1) >> 1;      // stages of two panels
            const double* Asrc = Xbase + ws_off + (size_t)row0 * ld;
            const double* Bsrc = Bbase + ws_off + (size_t)col0 * ld;
            for (int kt = 0; kt < KT; ++kt) {
                mbar_wait(&s_empty[stage], phase ^ 1);
                if (lane == 0) {
                    const int nj = min(2, KP - 2 * kt);
                    StageInfo& si = s_info[stage];
                    si.ws_off = ws_off; si.grp = g; si.ld = ld; si.n = t1.x; si.tij = tij;
                    si.tile = tile; si.tile_first = t1.z; si.tile_count = t1.w;
                    si.kt = kt; si.nj = nj; si.last = (kt == KT - 1); si.rows_a = rows_a;
                    si.rows_b = b_is_a ? rows_a : rows_b; si.b_is_a = b_is_a ? 1 : 0;
                    const unsigned bytes_a = (unsigned)(rows_a * 8 * nj) * 8u;
                    const unsigned bytes_b = b_is_a ? 0u : (unsigned)(rows_b * 8 * nj) * 8u;
                    mbar_arrive_expect_tx(&s_full[stage], bytes_a + bytes_b);
                    double* sa = smem + (size_t)stage * STAGE_DOUBLES;
                    bulk_g2s(sa, Asrc + (size_t)(2 * kt) * rows_a * 8, bytes_a, &s_full[stage]);
                    if (!b_is_a)
                        bulk_g2s(sa + BM * BK, Bsrc + (size_t)(2 * kt) * rows_b * 8, bytes_b, &s_full[stage]);
                }
                __syncwarp();
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
        // end marker
        mbar_wait(&s_empty[stage], phase ^ 1);
        if (lane == 0) {
            s_info[stage].kt = -1;
            mbar_arrive(&s_full[stage]);
        }
        return;
    }

    // ======================================================================= consumer warps
    const int lr = lane >> 2, lk = lane & 3;
    int stage = 0;
    unsigned phase = 0;
    double acc[16][2];
    int variant = 0, s_rows = 0, row0 = 0, col0 = 0, kp_col0 = 0;
    bool diag = false, full_diag = false;
    for (;;) {
        mbar_wait(&s_full[stage], phase);
        const StageInfo si = s_info[stage];
        if (si.kt < 0) break;
        if (si.kt == 0) {
            const int ti = si.tij & 0xffff, tj = si.tij >> 16;
            row0 = ti * BM; col0 = tj * BN; kp_col0 = col0 >> 3;
            diag = (ti == tj);
            s_rows = min(8, (si.ld - row0) >> 3);  // valid 8-row sub-tile rows of this tile, 1..8
            full_diag = diag && s_rows == 8;
            // 0 idle, 1..8 rect<M>, 9..12 diag<W>
            if (full_diag) variant = 9 + wid;
            else if (diag) variant = (2 * wid < s_rows) ? s_rows : 0;  // columns past the matrix
            else variant = s_rows;
#pragma unroll
            for (int e = 0; e < 16; ++e) acc[e][0] = acc[e][1] = 0.0;
        }
        {
            const double* sa = smem + (size_t)stage * STAGE_DOUBLES;
            const double* sb = si.b_is_a ? sa : sa + BM * BK;
            const int ja = si.rows_a * 8, jb = si.rows_b * 8;  // panel strides (doubles)
#pragma unroll 1
            for (int j = 0; j < si.nj; ++j) {
                const double* Ap = sa + j * ja + lr * 8 + 2 * lk;
                const double* Bp0 = sb + j * jb + lr * 8 + 2 * lk;
                const double* Bp = Bp0 + wid * 128;
                switch (variant) {
                    case 8: panel_rect<8>(acc, Ap, Bp); break;
                    case 7: panel_rect<7>(acc, Ap, Bp); break;
                    case 6: panel_rect<6>(acc, Ap, Bp); break;
                    case 5: panel_rect<5>(acc, Ap, Bp); break;
                    case 4: panel_rect<4>(acc, Ap, Bp); break;
                    case 3: panel_rect<3>(acc, Ap, Bp); break;
                    case 2: panel_rect<2>(acc, Ap, Bp); break;
                    case 1: panel_rect<1>(acc, Ap, Bp); break;
                    case 9: panel_diag<0>(acc, Ap, Bp0); break;
                    case 10: panel_diag<1>(acc, Ap, Bp0); break;
                    case 11: panel_diag<2>(acc, Ap, Bp0); break;
                    case 12: panel_diag<3>(acc, Ap, Bp0); break;
                    default: break;
                }
                if (MODE == 1 && variant != 0) {
                    const int sc = 2 * si.kt + j - kp_col0;
                    if ((unsigned)sc < 8u) fold_x(acc, Ap, full_diag, s_rows, wid, sc);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_empty[stage]);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
        if (!si.last) continue;

        // ------------------------------------------------------------------ epilogue of the tile
        const int g = si.grp, ld = si.ld, n = si.n;
        double s = __longlong_as_double((long long)a.gersh[g]);
        if (!(s > 0.0)) s = 1.0;
        double alpha, cb;
        if (k == 0) { alpha = 1.0 / (s * s); cb = -0.5 / s; }
        else { alpha = 1.0; cb = -0.5; }
        double* Out = ((MODE == 0) ? a.bufY : ((k & 1) ? a.buf0 : a.buf1)) + si.ws_off;
        double part = 0.0;
        // k8-panel offsets of this thread's elements (common.cuh): all rows of the tile sit in one
        // row-tile, all its columns (as mirror rows) in another, so an element of sub-tile (sr, sc)
        // is at  base_d + sc * pd + sr * 64  and its mirror at  base_m + sr * pm + sc * 64 (+8 for c+1).
        const int pd = si.rows_a * 8, pm = min(BN, ld - col0) * 8;
        const int base_d = row0 * ld + kp_col0 * pd + lr * 8 + 2 * lk;
        const int base_m = col0 * ld + (row0 >> 3) * pm + 2 * lk * 8 + lr;
        const double scale = (MODE == 0) ? alpha : cb;  // MODE 1: acc = X Y - 3 X -> X' = b acc
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            int sr, sc;  // sub-tile row / column inside the CTA tile
            bool valid;
            if (full_diag) {
                valid = e < 9;
                if (e <= wid) { sr = wid; sc = e; } else { sr = 7 - wid; sc = e - wid - 1; }
            } else {
                sr = e >> 1; sc = 2 * wid + (e & 1);
                valid = variant != 0 && sr < s_rows && (col0 + sc * 8) < ld;
            }
            if (!valid) continue;
            const int r = row0 + sr * 8 + lr;
            const int c = col0 + sc * 8 + 2 * lk;
            double* pd_ = Out + (base_d + sc * pd + sr * 64);
            double* pm_ = Out + (base_m + sr * pm + sc * 64);
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int cc = c + q;
                if (cc > r) continue;  // upper triangle of a diagonal tile: its mirror image is stored
                const double v = acc[e][q] * scale;
                pd_[q] = v;
                if (cc != r) pm_[q * 8] = v;
                if (MODE == 0 && r < n) {  // residual over the n x n part; strictly-lower elements count twice
                    const double d = v - (cc == r ? 1.0 : 0.0);
                    part = fma((cc == r ? 1.0 : 2.0) * d, d, part);
                }
            }
        }
        if (MODE == 0) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (lane == 0) s_red[wid] = part;
            asm volatile("bar.sync 1, 128;" ::: "memory");  // consumer warps only
            int is_last = 0;
            if (tid == 0) {
                a.partials[si.tile] = (s_red[0] + s_red[1]) + (s_red[2] + s_red[3]);
                __threadfence();
                is_last = (atomicAdd(a.tile_done + g, 1) == si.tile_count - 1) ? 1 : 0;
            }
            if (wid == 0) {
                is_last = __shfl_sync(0xffffffffu, is_last, 0);
                if (is_last) {
                    // every tile of submatrix g has published its partial: fixed-order sum + decision
                    __threadfence();
                    double r2 = 0.0;
                    for (int t = lane; t < si.tile_count; t += 32) r2 += __ldcg(a.partials + si.tile_first + t);
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
                    if (lane == 0) {
                        const double r = sqrt(r2 / (double)(n > 0 ? n : 1));
                        const double prev = k > 0 ? a.res[(size_t)((k - 1) & 1) * a.ngroups + g] : 1e300;
                        const bool conv = r < a.eps;
                        const bool stag = (k > 0) && (r >= prev) && (r < 1e-6);
                        const bool stop = conv || stag || a.decide_only || !(r == r);
                        a.res[(size_t)(k & 1) * a.ngroups + g] = r;
                        a.tile_done[g] = 0;
                        if (stop) { a.flag[g] = conv ? 0 : 1; a.done_iter[g] = k; }
                        else atomicAdd(a.counters + k, 1);
                    }
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");  // s_red may be reused by the next tile
        }
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
    a.done_iter = p->d_done_iter; a.flag = p->d_flag; a.tile_done = p->d_tile_done; a.res = p->d_res;
    a.counters = p->d_counters; a.n_tiles = (int32_t)p->n_tiles;
    a.ngroups = p->ngroups; a.k = k; a.decide_only = decide_only; a.eps = eps;
    const int grid = (int)std::min<int64_t>(p->n_tiles, (int64_t)p->num_sms * 3);
    a.sched = p->d_sched + 2 * k;
    k_ns_gemm<0><<<grid, NTHREADS, NS_SMEM, st>>>(a);
    p->launches += 1;
    if (!decide_only) {
        a.sched = p->d_sched + 2 * k + 1;
        k_ns_gemm<1><<<grid, NTHREADS, NS_SMEM, st>>>(a);
        p->launches += 1;
    }
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

}  // namespace smb
