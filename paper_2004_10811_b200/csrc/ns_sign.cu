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

// Tile metadata, written by the producer into the slot of the tile's FIRST pipeline stage before it
// arms that stage's "full" barrier (the other stages of a tile carry operands only: the consumers
// derive the stage count and panel counts from ld).  valid == 0 is the end marker.
struct __align__(16) TileInfo {
    int64_t ws_off;
    int32_t grp, ld;
    int32_t n, tij;
    int32_t tile, tile_first;
    int32_t tile_count, valid;
};
__device__ __forceinline__ void mbar_wait_a(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive_a(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

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

// Rectangular tile with a run-time number M of valid row sub-tiles: ONE code body for every M
// (fall-through switches enter the unrolled row sequence at row M-1), so ragged tiles cost no
// extra instruction-cache footprint.  Three passes -- fragment loads, products with the even k of
// the panel, products with the odd k -- keep 2 M independent accumulators between dependent DMMAs.
#define SM_ROWS(STMT) \
    switch (M) {      \
        case 8: STMT(7) case 7: STMT(6) case 6: STMT(5) case 5: STMT(4) \
        case 4: STMT(3) case 3: STMT(2) case 2: STMT(1) case 1: STMT(0) \
        default: break; \
    }
__device__ __forceinline__ void panel_rect_dyn(double (&acc)[16][2], const double* __restrict__ Ap,
                                               const double* __restrict__ Bp, int M) {
    double2 af[8];
    const double2 b0 = *reinterpret_cast<const double2*>(Bp);
    const double2 b1 = *reinterpret_cast<const double2*>(Bp + 64);
#define SM_LD(mt) af[mt] = *reinterpret_cast<const double2*>(Ap + mt * 64);
#define SM_MX(mt) dmma(acc[2 * mt], af[mt].x, b0.x); dmma(acc[2 * mt + 1], af[mt].x, b1.x);
#define SM_MY(mt) dmma(acc[2 * mt], af[mt].y, b0.y); dmma(acc[2 * mt + 1], af[mt].y, b1.y);
    SM_ROWS(SM_LD)
    SM_ROWS(SM_MX)
    SM_ROWS(SM_MY)
#undef SM_LD
#undef SM_MX
#undef SM_MY
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
// (X' = b (X Y - 3 X)).  Runs on 8 of the K/8 panels of a tile; specialised per work shape so that
// each k loop carries only its own few instructions.
__device__ __forceinline__ void fold_rect(double (&acc)[16][2], const double* __restrict__ Ap, int s_rows, int wid,
                                          int sc) {
    if ((sc >> 1) != wid) return;
    const bool odd = sc & 1;
#pragma unroll
    for (int mt = 0; mt < 8; ++mt) {
        if (mt < s_rows) {
            const double2 x = *reinterpret_cast<const double2*>(Ap + mt * 64);
            if (odd) { acc[2 * mt + 1][0] = fma(-3.0, x.x, acc[2 * mt + 1][0]); acc[2 * mt + 1][1] = fma(-3.0, x.y, acc[2 * mt + 1][1]); }
            else { acc[2 * mt][0] = fma(-3.0, x.x, acc[2 * mt][0]); acc[2 * mt][1] = fma(-3.0, x.y, acc[2 * mt][1]); }
        }
    }
}
template <int W>
__device__ __forceinline__ void fold_diag(double (&acc)[16][2], const double* __restrict__ Ap, int sc) {
    // sub-tile row W holds columns 0..W in acc[0..W]; row 7-W holds columns 0..7-W in acc[W+1..8]
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if (c == sc) {
            if (c <= W) {
                const double2 x = *reinterpret_cast<const double2*>(Ap + W * 64);
                acc[c][0] = fma(-3.0, x.x, acc[c][0]); acc[c][1] = fma(-3.0, x.y, acc[c][1]);
            }
            if (c <= 7 - W) {
                const double2 x = *reinterpret_cast<const double2*>(Ap + (7 - W) * 64);
                acc[W + 1 + c][0] = fma(-3.0, x.x, acc[W + 1 + c][0]); acc[W + 1 + c][1] = fma(-3.0, x.y, acc[W + 1 + c][1]);
            }
        }
    }
}

// k loop of one tile for one consumer warp.  `variant` is the warp's work shape for this tile
// (0 idle, 1..8 rect<M>, 9..12 diag<W>); per stage: wait, its k panels (two, or one in the last
// stage of an odd panel count), release.  One panel body per shape, dispatched by a warp-uniform
// switch, keeps the kernel within the instruction cache.  The first stage of the tile has already
// been waited for by the caller (it carries the TileInfo).
template <int MODE>
__device__ __forceinline__ void k_loop(double (&acc)[16][2], const double* smem, unsigned full0, unsigned empty0,
                                       int& stage, unsigned& phase, int KP, int ja, int jb, bool b_is_a,
                                       int frag_off, int wid, int lane, int kp_col0, int s_rows, int variant) {
    const int KT = (KP + 1) >> 1;
    const int boff = frag_off + (variant <= 8 ? wid * 128 : 0);
#pragma unroll 1
    for (int kt = 0; kt < KT; ++kt) {
        if (kt > 0) mbar_wait_a(full0 + 8u * stage, phase);
        if (variant != 0) {
            const double* sa = smem + (size_t)stage * STAGE_DOUBLES;
            const double* Ap = sa + frag_off;
            const double* Bp = (b_is_a ? sa : sa + BM * BK) + boff;
            const int nj = min(2, KP - 2 * kt);
#pragma unroll 1
            for (int j = 0; j < nj; ++j, Ap += ja, Bp += jb) {
                switch (variant) {
                    case 8: panel_rect<8>(acc, Ap, Bp); break;
                    case 7: panel_rect<7>(acc, Ap, Bp); break;
                    case 6: panel_rect<6>(acc, Ap, Bp); break;
                    case 5: panel_rect<5>(acc, Ap, Bp); break;
                    case 4: panel_rect<4>(acc, Ap, Bp); break;
                    case 3: panel_rect<3>(acc, Ap, Bp); break;
                    case 2: panel_rect<2>(acc, Ap, Bp); break;
                    case 1: panel_rect<1>(acc, Ap, Bp); break;
                    case 9: panel_diag<0>(acc, Ap, Bp); break;
                    case 10: panel_diag<1>(acc, Ap, Bp); break;
                    case 11: panel_diag<2>(acc, Ap, Bp); break;
                    default: panel_diag<3>(acc, Ap, Bp); break;
                }
                if (MODE == 1) {
                    const int sc = 2 * kt + j - kp_col0;
                    if ((unsigned)sc < 8u) {
                        if (variant <= 8) fold_rect(acc, Ap, s_rows, wid, sc);
                        else if (variant == 9) fold_diag<0>(acc, Ap, sc);
                        else if (variant == 10) fold_diag<1>(acc, Ap, sc);
                        else if (variant == 11) fold_diag<2>(acc, Ap, sc);
                        else fold_diag<3>(acc, Ap, sc);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_a(empty0 + 8u * stage);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
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
    __shared__ __align__(16) TileInfo s_info[STAGES];
    __shared__ __align__(8) uint64_t s_full[STAGES], s_empty[STAGES];
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
        // ============================================================ producer (one thread)
        // Tile ids are drawn two tiles ahead and descriptors / "still active" flags one tile ahead,
        // so that the three dependent global reads of a tile hand-over are already done when the
        // current tile's last slice has been issued.
        if (lane != 0) return;
        int stage = 0;
        unsigned phase = 0;
        auto draw = [&]() { return atomicAdd(a.sched, 1); };
        auto load_desc = [&](int tile, int4& t0, int4& t1, int& done) {
            if (tile < a.n_tiles) {
                const int4* tdp = reinterpret_cast<const int4*>(a.tiles + tile);
                t0 = __ldg(tdp);
                t1 = __ldg(tdp + 1);
                done = a.done_iter[t0.z];
            }
        };
        int tile = draw();
        int tile_n = draw();
        int4 t0, t1, n0, n1;
        int done = 0, done_n = 0;
        t0 = t1 = n0 = n1 = make_int4(0, 0, 0, 0);
        load_desc(tile, t0, t1, done);
        while (tile < a.n_tiles) {
            load_desc(tile_n, n0, n1, done_n);  // in flight while this tile streams
            const int tile_nn = draw();
            if (done < 0) {
                const int g = t0.z;
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
                    const int nj = min(2, KP - 2 * kt);
                    if (kt == 0) {
                        TileInfo& ti_ = s_info[stage];
                        ti_.ws_off = ws_off; ti_.grp = g; ti_.ld = ld; ti_.n = t1.x; ti_.tij = tij;
                        ti_.tile = tile; ti_.tile_first = t1.z; ti_.tile_count = t1.w; ti_.valid = 1;
                    }
                    const unsigned bytes_a = (unsigned)(rows_a * 8 * nj) * 8u;
                    const unsigned bytes_b = b_is_a ? 0u : (unsigned)(rows_b * 8 * nj) * 8u;
                    mbar_arrive_expect_tx(&s_full[stage], bytes_a + bytes_b);
                    double* sa = smem + (size_t)stage * STAGE_DOUBLES;
                    bulk_g2s(sa, Asrc + (size_t)(2 * kt) * rows_a * 8, bytes_a, &s_full[stage]);
                    if (!b_is_a)
                        bulk_g2s(sa + BM * BK, Bsrc + (size_t)(2 * kt) * rows_b * 8, bytes_b, &s_full[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
            tile = tile_n; t0 = n0; t1 = n1; done = done_n;
            tile_n = tile_nn;
        }
        // end marker
        mbar_wait(&s_empty[stage], phase ^ 1);
        s_info[stage].valid = 0;
        mbar_arrive(&s_full[stage]);
        return;
    }

    // ======================================================================= consumer warps
    const int lr = lane >> 2, lk = lane & 3;
    const unsigned full0 = smem_u32(&s_full[0]), empty0 = smem_u32(&s_empty[0]);
    const int frag_off = lr * 8 + 2 * lk;
    int stage = 0;
    unsigned phase = 0;
    double acc[16][2];
    for (;;) {
        mbar_wait_a(full0 + 8u * stage, phase);  // first stage of the next tile (or the end marker)
        const TileInfo si = s_info[stage];
        if (!si.valid) break;
        const int ti = si.tij & 0xffff, tj = si.tij >> 16;
        const int row0 = ti * BM, col0 = tj * BN, kp_col0 = col0 >> 3;
        const bool diag = (ti == tj);
        const int s_rows = min(8, (si.ld - row0) >> 3);  // valid 8-row sub-tile rows of this tile, 1..8
        const bool full_diag = diag && s_rows == 8;
        const int rows_a = min(BM, si.ld - row0), rows_b = min(BN, si.ld - col0);
        const bool b_is_a = (MODE == 0) && diag;
        // 0 idle, 1..8 rect<M>, 9..12 diag<W>
        int variant;
        if (full_diag) variant = 9 + wid;
        else if (diag) variant = (2 * wid < s_rows) ? s_rows : 0;  // columns past the matrix
        else variant = s_rows;
#pragma unroll
        for (int e = 0; e < 16; ++e) acc[e][0] = acc[e][1] = 0.0;
        {
            const int KP = si.ld >> 3;
            const int ja = rows_a * 8, jb = (b_is_a ? rows_a : rows_b) * 8;  // panel strides (doubles)
            k_loop<MODE>(acc, smem, full0, empty0, stage, phase, KP, ja, jb, b_is_a, frag_off, wid, lane, kp_col0,
                         s_rows, variant);
        }

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
        const int pd = rows_a * 8, pm = min(BN, ld - col0) * 8;
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
            // Residual: every consumer warp publishes its partial of the tile; the warp that brings
            // the submatrix's count to 4 x tile_count sums all partials in a fixed order and records
            // the decision (deterministic; no CTA-wide barrier, no floating-point atomics).
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            int is_last = 0;
            if (lane == 0) {
                a.partials[(size_t)si.tile * 4 + wid] = part;
                __threadfence();
                is_last = (atomicAdd(a.tile_done + g, 1) == 4 * si.tile_count - 1) ? 1 : 0;
            }
            is_last = __shfl_sync(0xffffffffu, is_last, 0);
            if (is_last) {
                __threadfence();
                double r2 = 0.0;
                const double* pp = a.partials + (size_t)si.tile_first * 4;
                for (int t = lane; t < 4 * si.tile_count; t += 32) r2 += __ldcg(pp + t);
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
