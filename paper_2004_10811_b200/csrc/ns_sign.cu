// a5 batched Newton-Schulz sign iteration (Eq.(11)):  X_{k+1} = 1/2 X_k (3 I - X_k^2),
// convergence monitor ||X_k^2 - I||_F / sqrt(n) (involutority, L354 / Fig.13).
//
// Two persistent kernels per iteration over ALL submatrices at once; the unit of work is one 64x64
// lower-triangular tile of one submatrix, handed out by an atomic counter:
//   MODE 0:  Y  = alpha * X X          + per-warp partials of ||Y - I||_F^2 (plain stores);
//                                        k_ns_decide then sums them per submatrix in a fixed order
//                                        and records the convergence decision (deterministic)
//   MODE 1:  X' = -1/2 (X Y - 3 X)     (iteration 0 folds the spectral scale 1/s_i into the
//                                        coefficients, so that no scaling pass is needed)
//   MODE 2/3: the two products of the third-order iteration Eq.(19) L348 (option order = 3).
//   MODE 4:  P  = (I - Y)^2 + ||P||_F^2  the certificate of the two-step exit (reading A9c).
// The end of a submatrix's iteration is not made of full products: a predicted exit (A9b) forms only the
// generating rows of its last update (k_ns_thin), the two-step exit (A9c) certifies the residual of X_{k+1}
// from P and forms only the generating rows of X_{k+2} (k_ns_spec_decide, k_ns_thin3) -- thin products bound by
// HBM, further down in this file.
// A launch issued after the evaluation was stopped on the device (EvalCtrl, common.cuh) is empty.
// X, Y and X' are symmetric polynomials of the same matrix, so only tiles on or below the diagonal
// are computed and every element is stored together with its mirror image: the stored matrices are
// bitwise symmetric, which also lets both GEMM operands be read as k-contiguous rows
// (B[k][n] = Y[n][k]).
//
// Data movement (sm_100a): matrices live in the k8-panel layout of common.cuh, so the 64 x 32
// operand slice of one pipeline stage (four k8 panels) is ONE contiguous block; a producer warp streams it with
// cp.async.bulk (TMA, SASS UBLKCP) into a 2-stage shared-memory ring, completion counted on
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

// Pipeline shape: a stage holds BK = 32 contraction indices (four k8 panels: 32 KB for both operands), two
// stages.  Measured on config 4 (all-active launch): BK 16 x 4 stages 7.20 ms, 24 x 3 7.16, 32 x 2 6.99,
// 8 x 8 7.19 -- fewer hand-overs win slightly, the ring depth does not matter (three CTAs per SM overlap).
#ifndef SM_BK
#define SM_BK 32
#endif
#ifndef SM_STAGES
#define SM_STAGES 2
#endif
constexpr int BM = TILE, BN = TILE, BK = SM_BK, STAGES = SM_STAGES, PPS = BK / 8;  // PPS: k panels per stage

// Kernel modes.  Update modes compute  Out = cb (A B + fold A)  on symmetric operands:
//   MODE 0   Y  = alpha X X (+ residual partials)                          Eq.(11), Eq.(19)
//   MODE 1   X' = -1/2 (X Y - 3 X)          = 1/2 X (3 I - X^2)            Eq.(11)
//   MODE 2   W  = 3/8 (Y Y - 10/3 Y)        = 1/8 (3 X^4 - 10 X^2)         Eq.(19), first half
//   MODE 3   X' = X W + 15/8 X              = 1/8 X (15 I - 10 X^2 + 3 X^4) Eq.(19), second half
template <int MODE> struct ModeTraits;
template <> struct ModeTraits<0> { static constexpr double fold = 0.0, cb = 1.0; static constexpr bool scale_k0 = true; };
template <> struct ModeTraits<1> { static constexpr double fold = -3.0, cb = -0.5; static constexpr bool scale_k0 = true; };
template <> struct ModeTraits<2> { static constexpr double fold = -10.0 / 3.0, cb = 0.375; static constexpr bool scale_k0 = false; };
template <> struct ModeTraits<3> { static constexpr double fold = 1.875, cb = 1.0; static constexpr bool scale_k0 = true; };
//   MODE 4   P  = Y Y - 2 Y + I             = (I - Y)^2                    certificate of the two-step exit (A9c)
template <> struct ModeTraits<4> { static constexpr double fold = -2.0, cb = 1.0; static constexpr bool scale_k0 = false; };
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
// Producer-side wait: back off between polls so that the single producer thread does not take issue
// slots from the consumer warp that shares its SM sub-partition.
#ifndef SM_PROD_SLEEP
#define SM_PROD_SLEEP 0
#endif
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, unsigned parity) {
    const unsigned a = smem_u32(bar);
    for (;;) {
        unsigned ok;
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(a), "r"(parity) : "memory");
        if (ok) return;
        if (SM_PROD_SLEEP > 0) __nanosleep(SM_PROD_SLEEP);
    }
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
#ifndef SM_VLOAD
#define SM_VLOAD 0
#endif
__device__ __forceinline__ double2 lds2(const double* p) {
#if SM_VLOAD
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(smem_u32(p)));
    return v;
#else
    return *reinterpret_cast<const double2*>(p);
#endif
}
template <int M>
__device__ __forceinline__ void panel_rect(double (&acc)[16][2], const double* __restrict__ Ap,
                                           const double* __restrict__ Bp) {
    double2 bf[2], af[M];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) bf[nt] = lds2(Bp + nt * 64);
#pragma unroll
    for (int mt = 0; mt < M; ++mt) af[mt] = lds2(Ap + mt * 64);
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
                                          int sc, const double f) {
    if ((sc >> 1) != wid) return;
    const bool odd = sc & 1;
#pragma unroll
    for (int mt = 0; mt < 8; ++mt) {
        if (mt < s_rows) {
            const double2 x = *reinterpret_cast<const double2*>(Ap + mt * 64);
            if (odd) { acc[2 * mt + 1][0] = fma(f, x.x, acc[2 * mt + 1][0]); acc[2 * mt + 1][1] = fma(f, x.y, acc[2 * mt + 1][1]); }
            else { acc[2 * mt][0] = fma(f, x.x, acc[2 * mt][0]); acc[2 * mt][1] = fma(f, x.y, acc[2 * mt][1]); }
        }
    }
}
template <int W>
__device__ __forceinline__ void fold_diag(double (&acc)[16][2], const double* __restrict__ Ap, int sc, const double f) {
    // sub-tile row W holds columns 0..W in acc[0..W]; row 7-W holds columns 0..7-W in acc[W+1..8]
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if (c == sc) {
            if (c <= W) {
                const double2 x = *reinterpret_cast<const double2*>(Ap + W * 64);
                acc[c][0] = fma(f, x.x, acc[c][0]); acc[c][1] = fma(f, x.y, acc[c][1]);
            }
            if (c <= 7 - W) {
                const double2 x = *reinterpret_cast<const double2*>(Ap + (7 - W) * 64);
                acc[W + 1 + c][0] = fma(f, x.x, acc[W + 1 + c][0]); acc[W + 1 + c][1] = fma(f, x.y, acc[W + 1 + c][1]);
            }
        }
    }
}

// k loop of one tile for one consumer warp, specialised per work shape VAR (1..8 rect<M>, 9..12
// diag<W>, 0 idle): the shape is dispatched ONCE per tile, so the loop over the k panels carries
// only its own panel body, the stage hand-over every second panel and (MODE 1) the fold test.
// Per stage: wait "full", its k panels (two, or one in the last stage of an odd panel count),
// release "empty".  The first stage of the tile has already been waited for by the caller (it
// carries the TileInfo).
template <int MODE, int VAR>
__device__ __forceinline__ void k_loop_var(double (&acc)[16][2], const double* smem, unsigned full0, unsigned empty0,
                                           int& stage, unsigned& phase, int KP, int ja, int jb, bool b_is_a,
                                           int frag_off, int wid, int lane, int kp_col0, int s_rows) {
    const int KT = (KP + PPS - 1) / PPS;
    const int boff = frag_off + ((VAR <= 8 || VAR == 13) ? wid * 128 : 0);
#pragma unroll 1
    for (int kt = 0; kt < KT; ++kt) {
        if (kt > 0) mbar_wait_a(full0 + 8u * stage, phase);
        if (VAR != 0) {
            const double* sa = smem + (size_t)stage * STAGE_DOUBLES;
            const double* Ap = sa + frag_off;
            const double* Bp = (b_is_a ? sa : sa + BM * BK) + boff;
            const int nj = min(PPS, KP - PPS * kt);
            // one panel at a time (unrolling the panels of a stage was measured: the fragment registers of two
            // panels do not fit beside the accumulators, 7.57 / 8.32 ms per launch against 6.87)
#pragma unroll 1
            for (int j = 0; j < nj; ++j) {
                const double* Apj = Ap + j * ja;
                const double* Bpj = Bp + j * jb;
                if (VAR >= 1 && VAR <= 8) panel_rect<(VAR >= 1 && VAR <= 8) ? VAR : 1>(acc, Apj, Bpj);
                else if (VAR == 13) panel_rect_dyn(acc, Apj, Bpj, s_rows);
                else panel_diag<(VAR >= 9 && VAR <= 12) ? VAR - 9 : 0>(acc, Apj, Bpj);
                if (MODE >= 1) {
                    const int sc = PPS * kt + j - kp_col0;
                    if ((unsigned)sc < 8u) {
                        if (VAR <= 8 || VAR == 13) fold_rect(acc, Apj, VAR <= 8 ? VAR : s_rows, wid, sc, ModeTraits<MODE>::fold);
                        else fold_diag<(VAR >= 9 && VAR <= 12) ? VAR - 9 : 0>(acc, Apj, sc, ModeTraits<MODE>::fold);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_a(empty0 + 8u * stage);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
    }
}

// ---- epilogue of one tile.  k8-panel offsets of this thread's elements (common.cuh): all rows of
// the tile sit in one row-tile, all its columns (as mirror rows) in another, so an element of
// sub-tile (sr, sc) is at  base_d + sc * pd + sr * 64  and its mirror at  base_m + sr * pm + sc * 64
// (+8 for the next column).
struct EpiCtx {
    double* Out;
    double scale;  // MODE 0: alpha; MODE 1: b (acc = X Y - 3 X -> X' = b acc)
    double rinv;   // MODE 0 with rescaling (A8b): stored Y = al^2 X^2, the residual is taken of Y * rinv = X^2
    int base_d, base_m, pd, pm;
    int rlim;      // n - row0 - lr: rows sr*8 < rlim count for the residual (n x n part only)
};
// sub-tile strictly below the matrix diagonal: both elements stored, mirrored, counted twice
template <int MODE>
__device__ __forceinline__ void store_below(const EpiCtx& c, const double (&a)[2], int sr, int sc, double& part) {
    const double v0 = a[0] * c.scale, v1 = a[1] * c.scale;
    *reinterpret_cast<double2*>(c.Out + (c.base_d + sc * c.pd + sr * 64)) = make_double2(v0, v1);
    double* pm_ = c.Out + (c.base_m + sr * c.pm + sc * 64);
    pm_[0] = v0;
    pm_[8] = v1;
    if ((MODE == 0 || MODE == 4) && sr * 8 < c.rlim) {
        const double w0 = v0 * c.rinv, w1 = v1 * c.rinv;
        part = fma(2.0 * w0, w0, fma(2.0 * w1, w1, part));
    }
}
// sub-tile on the matrix diagonal (sr == sc of a diagonal tile): lower triangle only
template <int MODE>
__device__ __forceinline__ void store_ondiag(const EpiCtx& c, const double (&a)[2], int sr, int lr, int lk,
                                             double& part) {
    double* pd_ = c.Out + (c.base_d + sr * c.pd + sr * 64);
    double* pm_ = c.Out + (c.base_m + sr * c.pm + sr * 64);
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int cq = 2 * lk + q;
        if (cq > lr) continue;  // upper triangle: its mirror image is stored
        double v = a[q] * c.scale;
        if (MODE == 4 && cq == lr) v += 1.0;  // P = Y^2 - 2 Y + I
        pd_[q] = v;
        if (cq != lr) pm_[q * 8] = v;
        if (MODE == 0 && sr * 8 < c.rlim) {
            const double d = v * c.rinv - (cq == lr ? 1.0 : 0.0);
            part = fma((cq == lr ? 1.0 : 2.0) * d, d, part);
        }
        if (MODE == 4 && sr * 8 < c.rlim) part = fma((cq == lr ? 1.0 : 2.0) * v, v, part);  // ||P||_F^2
    }
}

struct TileGeo {
    int64_t ws_off;
    double* out;
    const unsigned long long* gersh;
    const double* alpha;  // null, or the rescaling factors of this iteration (one per submatrix)
    int ld, n, row0, col0, grp, k;
};

// One tile for one consumer warp: k loop + epilogue, specialised per work shape
//   VAR 1..8  rect<M> of an OFF-diagonal tile (no triangle tests in the epilogue)
//   VAR 9..12 diag<W> of a full diagonal tile
//   VAR 13    the small last diagonal tile (s_rows < 8 at run time; warps past the matrix idle)
//   VAR 0     idle warp of a small diagonal tile (takes part in the stage hand-over only)
template <int MODE, int VAR>
__device__ __forceinline__ void tile_var(double (&acc)[16][2], const double* smem, unsigned full0, unsigned empty0,
                                         int& stage, unsigned& phase, int KP, int ja, int jb, bool b_is_a,
                                         int frag_off, int wid, int lane, int kp_col0, int s_rows,
                                         const TileGeo& t, double& part) {
    k_loop_var<MODE, VAR>(acc, smem, full0, empty0, stage, phase, KP, ja, jb, b_is_a, frag_off, wid, lane, kp_col0,
                          s_rows);
    if (VAR == 0) return;
    const int lr = lane >> 2, lk = lane & 3;
    EpiCtx c;  // built after the k loop: only the tile geometry stays live across it
    c.scale = ModeTraits<MODE>::cb;
    if (t.k == 0 && ModeTraits<MODE>::scale_k0) {  // iteration 0 folds the spectral scale 1/s_i into the coefficients
        double sg = __longlong_as_double((long long)t.gersh[t.grp]);
        if (!(sg > 0.0)) sg = 1.0;
        c.scale = (MODE == 0) ? 1.0 / (sg * sg) : ModeTraits<MODE>::cb / sg;
    }
    c.rinv = 1.0;
    if ((MODE == 0 || MODE == 1) && t.alpha) {  // reading A8b: this iteration works on al X_k
        const double al = t.alpha[t.grp];
        if (MODE == 0) { c.scale *= al * al; c.rinv = 1.0 / (al * al); }
        else c.scale *= al;
    }
    c.Out = t.out + t.ws_off;
    c.pd = min(BM, t.ld - t.row0) * 8;
    c.pm = min(BN, t.ld - t.col0) * 8;
    c.base_d = t.row0 * t.ld + kp_col0 * c.pd + lr * 8 + 2 * lk;
    c.base_m = t.col0 * t.ld + (t.row0 >> 3) * c.pm + 2 * lk * 8 + lr;
    c.rlim = t.n - t.row0 - lr;
    if (VAR >= 1 && VAR <= 8) {
#pragma unroll
        for (int mt = 0; mt < (VAR <= 8 ? VAR : 0); ++mt)
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) store_below<MODE>(c, acc[2 * mt + nt], mt, 2 * wid + nt, part);
    } else if (VAR >= 9 && VAR <= 12) {
        constexpr int W = VAR >= 9 ? VAR - 9 : 0;
#pragma unroll
        for (int sc = 0; sc < W; ++sc) store_below<MODE>(c, acc[sc], W, sc, part);
        store_ondiag<MODE>(c, acc[W], W, lr, lk, part);
#pragma unroll
        for (int sc = 0; sc < 7 - W; ++sc) store_below<MODE>(c, acc[W + 1 + sc], 7 - W, sc, part);
        store_ondiag<MODE>(c, acc[8], 7 - W, lr, lk, part);
    } else if (VAR == 13) {
#pragma unroll
        for (int mt = 0; mt < 7; ++mt) {
            if (mt >= s_rows) break;
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                const int sc = 2 * wid + nt;
                if (sc < mt) store_below<MODE>(c, acc[2 * mt + nt], mt, sc, part);
                else if (sc == mt) store_ondiag<MODE>(c, acc[2 * mt + nt], mt, lr, lk, part);
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
    double* bufW;        // order 3 only (Eq.(19)): W = 1/8 (3 X^4 - 10 X^2)
    double* partials;
    int32_t* done_iter;
    int32_t* flag;
    double* res;         // [2][ngroups]
    int32_t* counters;   // [max_iter+2] still-active submatrices after iteration k
    int32_t* sched;      // work counter of this launch
    const int32_t* ctrl; // [0] != 0: the evaluation has been stopped on the device (k_eval_ctrl): do nothing
    double* alpha;       // null, or [2][ngroups] rescaling factors (slot k & 1 = iteration k), reading A8b
    double* lmin;        // [ngroups] lower bound l_k the schedule tracks
    const int2* gen_rng; // [ngroups] first / last generating row; non-null: restrict final updates (see producer)
    // Work lists written by k_ns_decide of iteration k (tiles of the submatrices that go on; bit 31 = "last update of a
    // predicted exit"): a launch draws from its list instead of scanning all tiles, so a launch with few active
    // submatrices costs what they cost.  act_list == null: every tile (MODE 0 of iteration 0).
    const int32_t* act_list;
    const int32_t* act_count;
    int32_t* next_upd_list;   // k_ns_decide: list of the update (MODE 1..3) of this iteration ...
    int32_t* next_upd_count;
    int32_t* next_sq_list;    // ... and of the squaring (MODE 0) of the next one
    int32_t* next_sq_count;
    int32_t* thin_list;       // k_ns_decide: submatrices whose LAST update is done by k_ns_thin (see there); null: none
    int32_t* thin_count;
    // two-step exit (reading A9c): k_ns_decide lists the submatrices it speculates on and their tiles (work list of the
    // MODE 4 launch); k_ns_spec_decide sorts them into the thin3 list (certified) or back into the update lists
    int32_t* spec_list;
    int32_t* spec_count;
    int32_t* spec_tiles;
    int32_t* spec_tile_count;
    int32_t* thin3_list;
    int32_t* thin3_count;
    int32_t n_tiles;
    int32_t ngroups;
    int32_t k;
    int32_t decide_only;  // k == max_iter: stop whatever the residual is
    int32_t predict;      // 1: predicted exit allowed (Eq.(11) path, eps well above the FP64 floor)
    int32_t max_iter;
    double eps;
};

template <int MODE>
#ifndef SM_MINB
#define SM_MINB 3
#endif
__global__ void __launch_bounds__(NTHREADS, SM_MINB) k_ns_gemm(NsArgs a) {
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

    const double* Xk = (k & 1) ? a.buf1 : a.buf0;
    const double* Xbase = (MODE == 2 || MODE == 4) ? a.bufY : Xk;                     // A operand
    const double* Bbase = (MODE == 0) ? Xk : (MODE == 3 ? a.bufW : a.bufY);           // B operand

    if (wid == 4) {
        // ============================================================ producer (one thread)
        // Tile ids are drawn two tiles ahead and descriptors / "still active" flags one tile ahead,
        // so that the three dependent global reads of a tile hand-over are already done when the
        // current tile's last slice has been issued.
        if (lane != 0) return;
        int stage = 0;
        unsigned phase = 0;
        const bool stopped = a.ctrl[0] != 0;  // decided / all converged earlier in the stream: empty launch
        const int n_work = stopped ? 0 : (a.act_list ? *a.act_count : a.n_tiles);
        auto draw = [&]() { return stopped ? 0x7fffffff : atomicAdd(a.sched, 1); };
        // MODE 1 with gen_rng: a submatrix that leaves by the predicted exit (done == k + 1: this update gives its
        // result, nothing reads it but the extraction of the generating columns, L127) only needs the tiles that
        // hold generating rows -- as rows (ti in range) or, mirrored, as columns (tj in range); skip = 1 otherwise
        auto load_desc = [&](int idx, int& tile, int4& t0, int4& t1, int& done) {
            if (idx < n_work) {
                tile = idx;
                bool listed_final = false;
                if (a.act_list) {
                    const int e = a.act_list[idx];
                    tile = e & 0x7fffffff;
                    listed_final = e < 0;
                }
                const int4* tdp = reinterpret_cast<const int4*>(a.tiles + tile);
                t0 = __ldg(tdp);
                t1 = __ldg(tdp + 1);
                done = a.act_list ? (listed_final ? k + 1 : -1) : a.done_iter[t0.z];
                if (MODE == 1 && a.gen_rng && done == k + 1) {
                    const int2 gr = __ldg(a.gen_rng + t0.z);
                    const int tl = gr.x / BM, th = gr.y / BM, ti = t1.y & 0xffff, tj = t1.y >> 16;
                    if (!((ti >= tl && ti <= th) || (tj >= tl && tj <= th))) done = k;  // not needed: treat as stopped
                }
            }
        };
        int idx = draw();
        int idx_n = draw();
        int4 t0, t1, n0, n1;
        int done = 0, done_n = 0, tile = 0, tile_n = 0;
        t0 = t1 = n0 = n1 = make_int4(0, 0, 0, 0);
        load_desc(idx, tile, t0, t1, done);
        while (idx < n_work) {
            load_desc(idx_n, tile_n, n0, n1, done_n);  // in flight while this tile streams
            const int idx_nn = draw();
            if (done < 0 || done > k) {  // active (done > k: stops after the update of iteration k, see k_ns_decide)
                const int g = t0.z;
                const int64_t ws_off = ((int64_t)(unsigned)t0.x) | ((int64_t)t0.y << 32);
                const int ld = t0.w, tij = t1.y;
                const int ti = tij & 0xffff, tj = tij >> 16;
                const int row0 = ti * BM, col0 = tj * BN;
                const int rows_a = min(BM, ld - row0), rows_b = min(BN, ld - col0);
                const bool b_is_a = (MODE == 0 || MODE == 2 || MODE == 4) && (ti == tj);
                const int KP = ld >> 3;            // 8-wide k panels
                const int KT = (KP + PPS - 1) / PPS;  // stages of PPS panels
                const double* Asrc = Xbase + ws_off + (size_t)row0 * ld;
                const double* Bsrc = Bbase + ws_off + (size_t)col0 * ld;
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait_backoff(&s_empty[stage], phase ^ 1);
                    const int nj = min(PPS, KP - PPS * kt);
                    if (kt == 0) {
                        TileInfo& ti_ = s_info[stage];
                        ti_.ws_off = ws_off; ti_.grp = g; ti_.ld = ld; ti_.n = t1.x; ti_.tij = tij;
                        ti_.tile = tile; ti_.tile_first = t1.z; ti_.tile_count = t1.w; ti_.valid = 1;
                    }
                    const unsigned bytes_a = (unsigned)(rows_a * 8 * nj) * 8u;
                    const unsigned bytes_b = b_is_a ? 0u : (unsigned)(rows_b * 8 * nj) * 8u;
                    mbar_arrive_expect_tx(&s_full[stage], bytes_a + bytes_b);
                    double* sa = smem + (size_t)stage * STAGE_DOUBLES;
                    bulk_g2s(sa, Asrc + (size_t)(PPS * kt) * rows_a * 8, bytes_a, &s_full[stage]);
                    if (!b_is_a)
                        bulk_g2s(sa + BM * BK, Bsrc + (size_t)(PPS * kt) * rows_b * 8, bytes_b, &s_full[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
            idx = idx_n; tile = tile_n; t0 = n0; t1 = n1; done = done_n;
            idx_n = idx_nn;
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
        const bool b_is_a = (MODE == 0 || MODE == 2 || MODE == 4) && diag;
        // work shape of this warp for this tile (see tile_var)
        int variant;
        if (full_diag) variant = 9 + wid;
        else if (diag) variant = (2 * wid < s_rows) ? 13 : 0;  // columns past the matrix: idle
        else variant = s_rows;
#pragma unroll
        for (int e = 0; e < 16; ++e) acc[e][0] = acc[e][1] = 0.0;
        const int ld = si.ld;
        TileGeo c;
        c.ws_off = si.ws_off; c.out = (MODE == 0) ? a.bufY : (MODE == 2 ? a.bufW : ((k & 1) ? a.buf0 : a.buf1)); c.gersh = a.gersh;
        c.alpha = a.alpha ? a.alpha + (size_t)(k & 1) * a.ngroups : nullptr;
        c.ld = ld; c.n = si.n; c.row0 = row0; c.col0 = col0; c.grp = si.grp; c.k = k;
        double part = 0.0;
        {
            const int KP = ld >> 3;
            const int ja = rows_a * 8, jb = (b_is_a ? rows_a : rows_b) * 8;  // panel strides (doubles)
#define SM_TV(V) case V: tile_var<MODE, V>(acc, smem, full0, empty0, stage, phase, KP, ja, jb, b_is_a, frag_off, wid, \
                                          lane, kp_col0, s_rows, c, part); break;
            switch (variant) {
                SM_TV(1) SM_TV(2) SM_TV(3) SM_TV(4) SM_TV(5) SM_TV(6) SM_TV(7) SM_TV(8)
                SM_TV(9) SM_TV(10) SM_TV(11) SM_TV(12) SM_TV(13)
                default: tile_var<MODE, 0>(acc, smem, full0, empty0, stage, phase, KP, ja, jb, b_is_a, frag_off, wid,
                                           lane, kp_col0, s_rows, c, part); break;
            }
#undef SM_TV
        }
        if (MODE == 0 || MODE == 4) {
            // Residual: every consumer warp publishes its partial of the tile (plain store, no fence,
            // no atomics); k_ns_decide sums them per submatrix in a fixed order after the launch.
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (lane == 0) a.partials[(size_t)si.tile * 4 + wid] = part;
        }
    }
}

// Convergence decision of iteration k (reading A9), one warp per still-active submatrix: residual
// r = sqrt(sum of its tile partials / n) in a fixed order (deterministic), then stop on r < eps,
// on stagnation (r not decreasing below 1e-6), at max_iter, or on NaN.
__global__ void __launch_bounds__(256) k_ns_decide(NsArgs a, const int32_t* __restrict__ tile_first,
                                                   const int32_t* __restrict__ tile_count,
                                                   const int32_t* __restrict__ sub_dim) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= a.ngroups || a.ctrl[0] != 0) return;
    if (a.done_iter[g] >= 0) return;
    const int lane = threadIdx.x & 31, k = a.k;
    const int cnt = 4 * tile_count[g], n = sub_dim[g];
    const double* pp = a.partials + (size_t)tile_first[g] * 4;
    int goes_on = 0;  // lane 0: 1 = takes part in the update and in the next squaring, 2 = in the update only (predicted exit)
    double r2 = 0.0;
    for (int t = lane; t < cnt; t += 32) r2 += pp[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
    if (lane == 0) {
        const double r = sqrt(r2 / (double)(n > 0 ? n : 1));
        const double prev = k > 0 ? a.res[(size_t)((k - 1) & 1) * a.ngroups + g] : 1e300;
        const bool conv = r < a.eps;
        const bool stag = (k > 0) && (r >= prev) && (r < 1e-6);
        const bool stop = conv || stag || a.decide_only || !(r == r);
        a.res[(size_t)(k & 1) * a.ngroups + g] = r;
        bool unscaled = true;
        if (a.alpha && !stop) {
            // Reading A8b: iteration k maps the eigenvalue moduli [l_k, 1] of X_k onto [l_{k+1}, 1] with
            // l_{k+1} = f(l_k) = f(1), f(x) = 1/2 al x (3 - al^2 x^2); al_{k+1} = sqrt(3 / (1 + l + l^2)) is the
            // factor that equalises both ends again; exactly 1 once l >= 0.9999 (plain Eq.(11) from there on,
            // which the predicted exit needs for the last two iterations).
            // l is an estimate: eigenvalues below it just converge later, the stop test is the residual.
            const double al = a.alpha[(size_t)(k & 1) * a.ngroups + g], l = a.lmin[g];
            unscaled = (al == 1.0);
            const double fl = 0.5 * al * l * (3.0 - al * al * l * l), f1 = 0.5 * al * (3.0 - al * al);
            const double ln = fmin(fmin(fl, f1), 1.0);  // f peaks (= 1) at x = 1/al inside [l, 1]: the ends bound it
            a.lmin[g] = ln;
            // al <= 1.7 keeps al |x| < sqrt(3) (no sign change) with |x| <= 1 + rounding
            a.alpha[(size_t)((k + 1) & 1) * a.ngroups + g] = ln < 0.9999 ? fmin(sqrt(3.0 / (1.0 + ln + ln * ln)), 1.7) : 1.0;
        }
        if (stop) { a.flag[g] = conv ? 0 : 1; a.done_iter[g] = k; }
        else {
            atomicAdd(a.counters + k, 1);
            goes_on = 1;
            // Predicted exit (reading A9): with E_k = X_k^2 - I symmetric, E_{k+1} = -3/4 E_k^2 + 1/4 E_k^3, so
            // ||E_{k+1}||_F <= 3/4 ||E_k||_F^2 + 1/4 ||E_k||_F^3.  If that bound is already a factor 10 below
            // eps, X_{k+1} is accepted without the product that would only confirm it: the submatrix takes part
            // in the update of this iteration (done_iter = k + 1 > k) and in nothing after it.
            if (a.predict && unscaled && k + 1 < a.max_iter) {
                const double sn = sqrt((double)(n > 0 ? n : 1)), f = r * sn;
                const double next = (0.75 * f * f + 0.25 * f * f * f) / sn;
                if (next < 0.1 * a.eps) {
                    a.done_iter[g] = k + 1;
                    a.flag[g] = 2;
                    a.res[(size_t)((k + 1) & 1) * a.ngroups + g] = next;
                    goes_on = 2;
                }
            }
        }
    }
    // Two-step exit (reading A9c): if X_{k+1} is likely to pass the predicted-exit test, its residual is certified
    // WITHOUT forming it: E_{k+1} = I - X_{k+1}^2 = 3/4 Et^2 + 1/4 Et^3 with Et = I - Y_k (Y_k = al^2 X_k^2 as stored),
    // so one product P = Et^2 (MODE 4) bounds ||E_{k+1}||_F; then only the generating rows of X_{k+2} are formed
    // (k_ns_thin3).  The estimate here only decides whether to try: r_{k+1} ~ rt^2 with rt = ||Et||_F / sqrt(n) ~ r / 2
    // for a rescaled step (the rescaling centres the spectrum of Et), r for a plain one.
    if (lane == 0 && goes_on == 1 && a.spec_list && k >= 1 && k + 2 <= a.max_iter &&
        thin_span_ok(a.gen_rng[g].y - a.gen_rng[g].x + 1, n)) {
        const double r = a.res[(size_t)(k & 1) * a.ngroups + g];
        const double al = a.alpha ? a.alpha[(size_t)(k & 1) * a.ngroups + g] : 1.0;
        const double rt = al != 1.0 ? 0.5 * r : r;
        const double sn = sqrt((double)(n > 0 ? n : 1)), f = rt * rt * sn;
        if ((0.75 * f * f + 0.25 * f * f * f) / sn < 0.1 * a.eps) goes_on = 3;
    }
    // work lists of the launches that follow (see NsArgs): every tile of a submatrix that goes on
    goes_on = __shfl_sync(0xffffffffu, goes_on, 0);
    if (goes_on == 3) {
        const int tf = tile_first[g], tc = tile_count[g];
        int base = 0;
        if (lane == 0) {
            a.spec_list[atomicAdd(a.spec_count, 1)] = g;
            base = atomicAdd(a.spec_tile_count, tc);
        }
        base = __shfl_sync(0xffffffffu, base, 0);
        for (int t = lane; t < tc; t += 32) a.spec_tiles[base + t] = tf + t;
        return;
    }
    if (goes_on == 2 && a.thin_list && a.gen_rng) {
        // predicted exit of a submatrix with few generating rows: its last update is the thin product of k_ns_thin
        const int2 gr = __ldg(a.gen_rng + g);
        if (thin_span_ok(gr.y - gr.x + 1, n)) {
            if (lane == 0) a.thin_list[atomicAdd(a.thin_count, 1)] = g;
            return;
        }
    }
    if (goes_on && a.next_upd_list) {
        const int tf = tile_first[g], tc = tile_count[g];
        int base = 0;
        if (lane == 0) base = atomicAdd(a.next_upd_count, tc);
        base = __shfl_sync(0xffffffffu, base, 0);
        const int fin = goes_on == 2 ? (int)0x80000000 : 0;
        for (int t = lane; t < tc; t += 32) a.next_upd_list[base + t] = (tf + t) | fin;
        if (goes_on == 1) {
            if (lane == 0) base = atomicAdd(a.next_sq_count, tc);
            base = __shfl_sync(0xffffffffu, base, 0);
            for (int t = lane; t < tc; t += 32) a.next_sq_list[base + t] = tf + t;
        }
    }
}

// Last update of the submatrices that leave by the predicted exit, for groups with few generating rows.
// Nothing reads X_{k+1} of such a submatrix but the extraction of the generating columns (PAPER.md L127 step 3) and
// the electron count (L275): rows r0..r1 of the symmetric X_{k+1} (scatter and k_nelec_part walk rows).  So the
// update is the THIN product  X'[r, :] = cb al (X[r, :] Y - 3 X[r, :]),  r = r0..r1 -- (r1 - r0 + 1) x n x n instead
// of the n x n x n of a full update (or the ~40 % of it that the tile-restricted final update of k_ns_gemm<1> costs
// at n ~ 200).  It reads all of Y once per 8 rows, i.e. it is bound by HBM, not by the FP64 pipe.
// One CTA per submatrix and chunk of 8 rows: the rows of X staged in shared memory (A fragments), each warp takes
// column sub-tiles j8 = w, w + 8, ..., four at a time; B fragments straight from global memory: lane (lr, lk) reads
// Y[8 j8 + lr][8 p + 2 lk .. + 1] (Y symmetric), 512 contiguous bytes per warp load in the k8-panel layout.
constexpr int THIN_WARPS = 8;
struct ThinArgs {
    const int32_t* list;
    const int32_t* count;
    const int32_t* sub_dim;
    const int32_t* ldv;
    const int64_t* ws_off;
    const int2* gen_rng;
    const unsigned long long* gersh;
    const double* alpha;   // rescaling factors of this iteration (slot k & 1), or null
    const double* X;       // X_k
    const double* Y;       // al^2 X_k^2
    double* Out;           // X_{k+1}
    const int32_t* ctrl;
    int k;
};
// One thin product for one warp: (8 rows in shared memory, sA[8][ld]) x (symmetric matrix Mg, k8-panel layout) for the
// column sub-tiles j8 = w, w + 8, ..., four at a time; emit(j8, acc) receives this lane's two results of sub-tile j8
// (row lr, columns 8 j8 + 2 lk, + 1).  (Reading only the blocks on or below the diagonal -- every 8 x 8 block is
// needed twice per pass, once transposed -- was measured: the second use does not come from the L2 often enough
// to pay for the extra loads, 76.4 against 75.6 ms per evaluation.)
template <class Emit>
__device__ __forceinline__ void thin_pass(const double* __restrict__ sA, const double* __restrict__ Mg, int ld, int w,
                                          int lane, Emit&& emit) {
    const int lr = lane >> 2, lk = lane & 3, nj8 = ld >> 3;
    for (int j0 = w; j0 < nj8; j0 += 4 * THIN_WARPS) {
        double acc[4][2];
        const double* yp[4];
        bool ok[4];
        int pst[4];  // k8 panel p of row r sits at (r's tile base) + p * rows_t * 8
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            acc[u][0] = acc[u][1] = 0.0;
            const int j8 = j0 + u * THIN_WARPS;
            ok[u] = j8 < nj8;
            const int r = 8 * (ok[u] ? j8 : 0) + lr;
            yp[u] = Mg + panel_off(r, 2 * lk, ld);
            pst[u] = min(64, ld - (r & ~63)) * 8;
        }
        const double* ap = sA + lr * ld + 2 * lk;
#pragma unroll 4
        for (int p = 0; p < nj8; ++p) {
            const double2 af = *reinterpret_cast<const double2*>(ap + 8 * p);
            double2 bf[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                bf[u] = ok[u] ? *reinterpret_cast<const double2*>(yp[u] + (size_t)p * pst[u]) : make_double2(0.0, 0.0);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                dmma(acc[u], af.x, bf[u].x);
                dmma(acc[u], af.y, bf[u].y);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (ok[u]) emit(j0 + u * THIN_WARPS, acc[u]);
    }
}

__global__ void __launch_bounds__(THIN_WARPS * 32, 4) k_ns_thin(ThinArgs a) {
    extern __shared__ __align__(16) double sA[];  // [8][ld] rows of X, row-major
    if (a.ctrl[0] != 0) return;
    const int cnt = *a.count;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, lr = lane >> 2, lk = lane & 3;
    for (int i = blockIdx.x; i < cnt; i += gridDim.x) {
        const int g = a.list[i];
        const int ld = a.ldv[g];
        const int2 gr = a.gen_rng[g];
        const int64_t ws = a.ws_off[g];
        const double* Xg = a.X + ws;
        const double* Yg = a.Y + ws;
        double* Og = a.Out + ws;
        double scale = -0.5;
        if (a.k == 0) {
            double sg = __longlong_as_double((long long)a.gersh[g]);
            if (!(sg > 0.0)) sg = 1.0;
            scale /= sg;
        }
        if (a.alpha) scale *= a.alpha[g];
        for (int c0 = gr.x; c0 <= gr.y; c0 += 8) {
            __syncthreads();  // the previous chunk's fragments have been read
            for (int e = threadIdx.x; e < 8 * ld; e += blockDim.x) {
                const int r = e / ld, c = e - r * ld;
                const int row = c0 + r;
                sA[e] = (row <= gr.y && row < ld) ? Xg[panel_off(row, c, ld)] : 0.0;
            }
            __syncthreads();
            const int row = c0 + lr;
            const bool row_ok = row <= gr.y && row < ld;
            thin_pass(sA, Yg, ld, w, lane, [&](int j8, const double (&acc)[2]) {
                if (!row_ok) return;
                const int col = 8 * j8 + 2 * lk;
                const double x0 = sA[lr * ld + col], x1 = sA[lr * ld + col + 1];
                *reinterpret_cast<double2*>(Og + panel_off(row, col, ld)) =
                    make_double2(scale * fma(-3.0, x0, acc[0]), scale * fma(-3.0, x1, acc[1]));
            });
        }
        __syncthreads();
    }
}

// ---- two-step exit (reading A9c), second half: the certificate and the generating rows of X_{k+2}
// k_ns_spec_decide, one warp per submatrix k_ns_decide speculated on: ||P||_F from the MODE 4 partials, then
//   ||E_{k+1}||_F <= (3/4 + 1/4 ||Et||_2) ||P||_F,   ||Et||_2 <= ||Et||_F <= (|1 - al^2| + al^2 r_k) sqrt(n)
// (Et = I - al^2 X_k^2 = (1 - al^2) I + al^2 E_k), and the test of the predicted exit (A9b) on that bound: if
// 3/4 f^2 + 1/4 f^3 (f = the bound) is a factor 10 below eps, X_{k+2} = 1/2 X_{k+1} (3 I - X_{k+1}^2) is accepted as the
// result (done_iter = k + 2, flag 3) and only its generating rows are formed; otherwise the submatrix goes on as if
// nothing had happened (its tiles join the update list of iteration k and the squaring list of k + 1): the
// speculation cost one product.
struct SpecArgs {
    const int32_t* list;
    const int32_t* count;
    const int32_t* tile_first;
    const int32_t* tile_count;
    const int32_t* sub_dim;
    const double* partials;
    double* res;
    const double* alpha;  // slot k & 1, or null
    int32_t* done_iter;
    int32_t* flag;
    int32_t* thin3_list;
    int32_t* thin3_count;
    int32_t* upd_list;
    int32_t* upd_count;
    int32_t* sq_list;
    int32_t* sq_count;
    int32_t* stat;        // [0] certified, [1] failed (per plan, running totals)
    const int32_t* ctrl;
    int ngroups, k;
    double eps;
};
__global__ void __launch_bounds__(256) k_ns_spec_decide(SpecArgs a) {
    if (a.ctrl[0] != 0) return;
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= *a.count) return;
    const int lane = threadIdx.x & 31, g = a.list[i], k = a.k;
    const int tf = a.tile_first[g], tc = a.tile_count[g], n = a.sub_dim[g];
    const double* pp = a.partials + (size_t)tf * 4;
    double p2 = 0.0;
    for (int t = lane; t < 4 * tc; t += 32) p2 += pp[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) p2 += __shfl_xor_sync(0xffffffffu, p2, o);
    int ok = 0;
    if (lane == 0) {
        const double sn = sqrt((double)(n > 0 ? n : 1));
        const double r = a.res[(size_t)(k & 1) * a.ngroups + g];
        const double al = a.alpha ? a.alpha[g] : 1.0;
        const double et = (fabs(1.0 - al * al) + al * al * r) * sn;
        const double f = (0.75 + 0.25 * et) * sqrt(p2);  // >= ||E_{k+1}||_F
        // + the term k_ns_thin3 leaves out: a perturbation of X_{k+2} of Frobenius norm <= al/16 ||P||_F^2 changes
        // ||X^2 - I||_F by at most twice that (||X||_2 <= 1)
        const double next = (0.75 * f * f + 0.25 * f * f * f + 0.125 * al * p2) / sn;
        ok = (next < 0.1 * a.eps) ? 1 : 0;  // false for NaN
        if (ok) {
            a.done_iter[g] = k + 2;
            a.flag[g] = 3;
            a.res[(size_t)(k & 1) * a.ngroups + g] = next;  // slot (k + 2) & 1: the residual bound of the result
            a.thin3_list[atomicAdd(a.thin3_count, 1)] = g;
            atomicAdd(a.stat, 1);
        } else {
            atomicAdd(a.stat + 1, 1);
        }
    }
    ok = __shfl_sync(0xffffffffu, ok, 0);
    if (ok) return;
    int base = 0;
    if (lane == 0) base = atomicAdd(a.upd_count, tc);
    base = __shfl_sync(0xffffffffu, base, 0);
    for (int t = lane; t < tc; t += 32) a.upd_list[base + t] = tf + t;
    if (lane == 0) base = atomicAdd(a.sq_count, tc);
    base = __shfl_sync(0xffffffffu, base, 0);
    for (int t = lane; t < tc; t += 32) a.sq_list[base + t] = tf + t;
}

// k_ns_thin3: generating rows r of X_{k+2} for the certified submatrices.  With Et = I - Y, P = Et^2 and
// X_{k+1} = 1/2 al X_k (2 I + Et),  X_{k+1}^2 = I - 3/4 P - 1/4 Et P  (everything commutes):
//   X_{k+2} = 1/2 X_{k+1} (3 I - X_{k+1}^2) = 1/2 al X_k (2 I + Et + 3/4 P + 5/8 Et P + 1/8 P^2).
// Row-wise, with A = X_k[r, :]:  U = A Et = A - A Y  (one thin pass over Y),  C = 3/4 A + 5/8 U,
//   X_{k+2}[r, :] = 1/2 al (2 A + U + C P)  (one thin pass over P)  + 1/16 al A P^2.
// The last term is NOT formed (it would be a third pass): ||1/16 al X_k P^2||_F <= al/16 ||P||_F^2 ~ 1e-13, and
// k_ns_spec_decide adds its effect on the residual, 2 x that / sqrt(n), to the bound it tests and reports.
// The rows go into the buffer of X_k (parity of k + 2), which nothing reads any more; P sits in the buffer X_{k+1}
// would have taken.
struct Thin3Args {
    const int32_t* list;
    const int32_t* count;
    const int32_t* ldv;
    const int64_t* ws_off;
    const int2* gen_rng;
    const double* alpha;  // slot k & 1, or null
    double* X;            // X_k in, rows of X_{k+2} out
    const double* Y;
    const double* P;
    const int32_t* ctrl;
};
__global__ void __launch_bounds__(THIN_WARPS * 32, 4) k_ns_thin3(Thin3Args a) {
    extern __shared__ __align__(16) double sm3[];  // two arrays [8][ld]
    if (a.ctrl[0] != 0) return;
    const int cnt = *a.count;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, lr = lane >> 2, lk = lane & 3;
    for (int i = blockIdx.x; i < cnt; i += gridDim.x) {
        const int g = a.list[i];
        const int ld = a.ldv[g];
        const int2 gr = a.gen_rng[g];
        const int64_t ws = a.ws_off[g];
        double* Xg = a.X + ws;
        const double* Yg = a.Y + ws;
        const double* Pg = a.P + ws;
        const double al = a.alpha ? a.alpha[g] : 1.0;
        double* s0 = sm3;            // A = X_k rows, then 2 A + U
        double* s1 = sm3 + 8 * ld;   // A Y, then C = 3/4 A + 5/8 U
        for (int c0 = gr.x; c0 <= gr.y; c0 += 8) {
            __syncthreads();
            for (int e = threadIdx.x; e < 8 * ld; e += blockDim.x) {
                const int r = e / ld, c = e - r * ld;
                const int row = c0 + r;
                s0[e] = (row <= gr.y && row < ld) ? Xg[panel_off(row, c, ld)] : 0.0;
            }
            __syncthreads();
            thin_pass(s0, Yg, ld, w, lane, [&](int j8, const double (&acc)[2]) {
                const int o = lr * ld + 8 * j8 + 2 * lk;
                s1[o] = acc[0];
                s1[o + 1] = acc[1];
            });
            __syncthreads();
            for (int e = threadIdx.x; e < 8 * ld; e += blockDim.x) {
                const double av = s0[e], u = av - s1[e];  // U = A - A Y
                s1[e] = fma(0.625, u, 0.75 * av);
                s0[e] = fma(2.0, av, u);
            }
            __syncthreads();
            const int row = c0 + lr;
            const bool row_ok = row <= gr.y && row < ld;
            thin_pass(s1, Pg, ld, w, lane, [&](int j8, const double (&acc)[2]) {
                if (!row_ok) return;
                const int col = 8 * j8 + 2 * lk, o = lr * ld + col;
                *reinterpret_cast<double2*>(Xg + panel_off(row, col, ld)) =
                    make_double2(0.5 * al * (s0[o] + acc[0]), 0.5 * al * (s0[o + 1] + acc[1]));
            });
        }
        __syncthreads();
    }
}

// which: bit 0 = MODE 0 + decision of iteration k, bit 1 = MODE 1 (update) of iteration k.
sm_status_t launch_ns_pair(sm_plan* p, int k, double eps, int decide_only, double* buf0, double* buf1,
                           double* bufY, cudaStream_t st, int which, double* bufW) {
    if (p->n_tiles == 0) return SM_OK;
    if (!p->ns_attr_set) {  // per plan: the attribute belongs to the device the plan was created on
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
        p->ns_attr_set = 1;
    }
    // timing: one event before and one after every product launch (sm_stats_t.ms_gemm)
    auto tick = [&]() -> sm_status_t {
        if (!p->timing) return SM_OK;
        if (p->ev_gemm_n == (int)p->ev_gemm.size()) {
            cudaEvent_t e = nullptr;
            SM_CUDA(cudaEventCreate(&e));
            p->ev_gemm.push_back(e);
        }
        SM_CUDA(cudaEventRecord(p->ev_gemm[p->ev_gemm_n++], st));
        return SM_OK;
    };
    sm_status_t ts;
    NsArgs a;
    a.tiles = p->d_tiles; a.gersh = p->d_gersh;
    a.buf0 = buf0; a.buf1 = buf1; a.bufY = bufY; a.bufW = bufW; a.partials = p->d_partials;
    a.done_iter = p->d_done_iter; a.flag = p->d_flag; a.res = p->d_res;
    a.counters = p->d_counters; a.n_tiles = (int32_t)p->n_tiles; a.ctrl = p->d_ctrl;
    a.ngroups = p->ngroups; a.k = k; a.decide_only = decide_only; a.eps = eps;
    const bool resc = rescale_on(p);
    a.alpha = resc ? p->d_alpha : nullptr; a.lmin = resc ? p->d_lmin : nullptr;
    a.gen_rng = (p->opt.order == 2) ? p->d_gen_rng : nullptr;
    // work lists: d_act = [upd 0][upd 1][sq 0][sq 1] x n_tiles entries, d_act_cnt[2 * iteration + {0: upd, 1: sq}]
    int32_t* const L = p->d_act;
    const size_t nt = (size_t)p->n_tiles;
    int32_t* const C = p->d_act_cnt;
    a.next_upd_list = L + (size_t)(k & 1) * nt;            a.next_upd_count = C + 2 * k;
    a.next_sq_list = L + (size_t)(2 + ((k + 1) & 1)) * nt; a.next_sq_count = C + 2 * (k + 1) + 1;
    const int32_t* sq_list = k > 0 ? L + (size_t)(2 + (k & 1)) * nt : nullptr;
    const int32_t* sq_count = C + 2 * k + 1;
    const int32_t* upd_list = L + (size_t)(k & 1) * nt;
    const int32_t* upd_count = C + 2 * k;
    a.predict = (p->opt.predict != 0 && p->opt.order == 2 && eps >= 1e-13) ? 1 : 0; a.max_iter = p->opt.max_iter;
    // thin last updates (k_ns_thin): list slot k & 1, count per iteration behind the tile-list counts
    const bool thin = a.predict && a.gen_rng && p->d_thin_list && p->thin_smem > 0;
    a.thin_list = thin ? p->d_thin_list + (size_t)(k & 1) * std::max(p->ngroups, 1) : nullptr;
    a.thin_count = thin ? C + 2 * (p->opt.max_iter + 3) + k : nullptr;
    // two-step exit (A9c): predict >= 2; lists: slot 2 = speculated submatrices, slot 3 = certified ones
    const int M = p->opt.max_iter + 3;
    const bool spec = thin && p->opt.predict >= 2 && p->thin3_smem > 0 && p->d_spec_tiles && p->spec_pause == 0;
    a.spec_list = spec ? p->d_thin_list + (size_t)2 * std::max(p->ngroups, 1) : nullptr;
    a.spec_count = spec ? C + 3 * M + k : nullptr;
    a.spec_tiles = spec ? p->d_spec_tiles : nullptr;
    a.spec_tile_count = spec ? C + 4 * M + k : nullptr;
    a.thin3_list = spec ? p->d_thin_list + (size_t)3 * std::max(p->ngroups, 1) : nullptr;
    a.thin3_count = spec ? C + 5 * M + k : nullptr;
    const int grid = (int)std::min<int64_t>(p->n_tiles, (int64_t)p->num_sms * SM_MINB);
    a.sched = p->d_sched + 4 * k;
    if (which & 1) {
        a.act_list = sq_list; a.act_count = sq_count;
        if ((ts = tick())) return ts;
        k_ns_gemm<0><<<grid, NTHREADS, NS_SMEM, st>>>(a);
        if ((ts = tick())) return ts;
        k_ns_decide<<<(p->ngroups + 7) / 8, 256, 0, st>>>(a, p->d_tile_first, p->d_tile_count, p->d_sub_dim);
        p->launches += 2;
    }
    if ((which & 2) && !decide_only) {
        a.act_list = upd_list; a.act_count = upd_count;
        if (p->opt.order == 3 && bufW) {  // Eq.(19): two products per update
            a.sched = p->d_sched + 4 * k + 1;
            if ((ts = tick())) return ts;
            k_ns_gemm<2><<<grid, NTHREADS, NS_SMEM, st>>>(a);
            a.sched = p->d_sched + 4 * k + 2;
            k_ns_gemm<3><<<grid, NTHREADS, NS_SMEM, st>>>(a);
            if ((ts = tick())) return ts;
            p->launches += 2;
        } else {
            if (spec) {
                if (!p->thin3_attr_set) {
                    SM_CUDA(cudaFuncSetAttribute(k_ns_gemm<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_SMEM));
                    SM_CUDA(cudaFuncSetAttribute(k_ns_thin3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->thin3_smem));
                    p->thin3_attr_set = 1;
                }
                NsArgs a4 = a;  // P = (I - Y)^2 of the speculated submatrices into the buffer of X_{k+1}
                a4.act_list = a.spec_tiles; a4.act_count = a.spec_tile_count; a4.sched = p->d_sched + 4 * k + 3;
                if ((ts = tick())) return ts;
                k_ns_gemm<4><<<grid, NTHREADS, NS_SMEM, st>>>(a4);
                if ((ts = tick())) return ts;
                SpecArgs sa;
                sa.list = a.spec_list; sa.count = a.spec_count; sa.tile_first = p->d_tile_first; sa.tile_count = p->d_tile_count;
                sa.sub_dim = p->d_sub_dim; sa.partials = p->d_partials; sa.res = p->d_res;
                sa.alpha = resc ? p->d_alpha + (size_t)(k & 1) * p->ngroups : nullptr;
                sa.done_iter = p->d_done_iter; sa.flag = p->d_flag; sa.thin3_list = a.thin3_list; sa.thin3_count = a.thin3_count;
                sa.upd_list = a.next_upd_list; sa.upd_count = a.next_upd_count;
                sa.sq_list = a.next_sq_list; sa.sq_count = a.next_sq_count;
                sa.stat = p->d_spec_stat; sa.ctrl = p->d_ctrl; sa.ngroups = p->ngroups; sa.k = k; sa.eps = eps;
                k_ns_spec_decide<<<(p->ngroups + 7) / 8, 256, 0, st>>>(sa);
                Thin3Args t3;
                t3.list = a.thin3_list; t3.count = a.thin3_count; t3.ldv = p->d_ld; t3.ws_off = p->d_ws_off;
                t3.gen_rng = p->d_gen_rng; t3.alpha = sa.alpha;
                t3.X = (k & 1) ? buf1 : buf0; t3.Y = bufY; t3.P = (k & 1) ? buf0 : buf1; t3.ctrl = p->d_ctrl;
                const int tgrid3 = (int)std::min<int64_t>(p->ngroups, (int64_t)p->num_sms * 8);
                k_ns_thin3<<<tgrid3, THIN_WARPS * 32, p->thin3_smem, st>>>(t3);
                p->launches += 3;
            }
            a.sched = p->d_sched + 4 * k + 1;
            if ((ts = tick())) return ts;
            k_ns_gemm<1><<<grid, NTHREADS, NS_SMEM, st>>>(a);
            if ((ts = tick())) return ts;
            p->launches += 1;
            if (thin) {
                if (!p->thin_attr_set) {
                    SM_CUDA(cudaFuncSetAttribute(k_ns_thin, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->thin_smem));
                    p->thin_attr_set = 1;
                }
                ThinArgs t;
                t.list = a.thin_list; t.count = a.thin_count; t.sub_dim = p->d_sub_dim; t.ldv = p->d_ld; t.ws_off = p->d_ws_off;
                t.gen_rng = p->d_gen_rng; t.gersh = p->d_gersh;
                t.alpha = resc ? p->d_alpha + (size_t)(k & 1) * p->ngroups : nullptr;
                t.X = (k & 1) ? buf1 : buf0; t.Y = bufY; t.Out = (k & 1) ? buf0 : buf1; t.ctrl = p->d_ctrl; t.k = k;
                const int tgrid = (int)std::min<int64_t>(p->ngroups, (int64_t)p->num_sms * 8);
                k_ns_thin<<<tgrid, THIN_WARPS * 32, p->thin_smem, st>>>(t);
                p->launches += 1;
            }
        }
    }
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

}  // namespace smb
