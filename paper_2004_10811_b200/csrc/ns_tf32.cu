// a5, opt-in reduced-precision variant (options.precision = 1): the same Newton-Schulz iteration
// (Eq.(11)) with FP32 storage and TF32 products on the 5th-generation tensor cores
// (tcgen05.mma kind::tf32, FP32 accumulators in tensor memory) -- the B200 counterpart of the
// paper's FP16 / FP32 cuBLAS experiment (L346-360, Table I).  Its accuracy is reported
// separately (north_star: <= 1e-3 elementwise); the FP64 DMMA path of ns_sign.cu stays the parity
// path.  NS never re-reads A, so the result carries the precision of the products.
//
// Data layout ("k4-panel/128", FP32): ldp = n rounded up to 16; rows in row-tiles of 128; inside a
// row-tile, chunk kc = the 4 consecutive columns 4 kc .. 4 kc + 3 of all its rows, row-major (16 B
// per row).  This IS the canonical K-major no-swizzle operand layout of tcgen05.mma (core matrix =
// 8 rows x 16 B contiguous, SBO = 128 B between row groups, LBO = rows_t * 16 B between chunks), so
// a pipeline stage (128 rows x 32 k) is one contiguous block in global memory: one cp.async.bulk,
// no tensor map, and the tensor core reads it as it landed.  It also makes the epilogue coalesced:
// thread r of a warp owns TMEM lane (row) r and writes 16 B per chunk next to its neighbours.
//
// Kernel: persistent, two CTAs per SM, warp-specialised:
//   warp 0 (one thread)  producer: cp.async.bulk of the A / B slices into a 2-stage ring (mbarrier tx)
//   warp 1 (one thread)  issues tcgen05.mma (M = 128, N = rows of the B half, K = 8 per instruction),
//                        tcgen05.commit releases the stage / hands the accumulator to the epilogue
//   warps 2..9           epilogue, two sets of four warps (one per TMEM lane quarter; the sets split the
//                        16-column chunks of a tile): tcgen05.ld of their 32 TMEM lanes, MODE 0: Y = X X and
//                        residual partials; MODE 1: X' = 3/2 X - 1/2 X Y.  Two CTAs per SM, one 256-column
//                        accumulator each: the epilogue of a tile overlaps the MMAs of the other CTA's tile.
//                        The launches are bound by epilogue latency, not by the tensor pipe or HBM (ncu: 15 %
//                        tensor, 33-51 % DRAM), which is why the second warp set pays.
// options.precision = 2 ("3xTF32") stores hi + lo TF32 planes (8 bytes per element) and issues three products per
// k step; options.precision = 3 ("BF16x2") stores hi + lo BF16 planes (4 bytes per element, 8 columns per 16-byte
// chunk) and issues the same three products with kind::f16 -- the launches are HBM-bound, so halving the bytes is
// what makes that rung faster than FP64 (Table I's ladder, L366-374, on this part's tensor pipes).
// Work unit: (submatrix, 128-row tile, 256-column tile on or below the diagonal), dealt to the CTAs in
// consecutive pairs (the units of one submatrix share operand rows).  Only the lower triangle is computed; every element is stored together with its
// mirror image, so X and Y are bitwise symmetric and B can be read as k-contiguous rows.
#include <algorithm>

#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "common.cuh"

namespace smb {

// R_CTAS = 1: one CTA per SM, 4-stage ring, two 256-column accumulators (epilogue of a tile overlaps the MMAs of
// the next).  R_CTAS = 2: two CTAs per SM, each with a 2-stage ring and ONE 256-column accumulator: the overlap
// comes from the other CTA, and every SM has two producers, two MMA issuers and eight epilogue warps.
#ifndef R_CTAS
#define R_CTAS 2
#endif
constexpr int R_BM = 128, R_BN = 256, R_BK = 32, R_STAGES = R_CTAS == 1 ? 4 : 2;
constexpr int R_TBUFS = R_CTAS == 1 ? 2 : 1, R_TCOLS = R_CTAS == 1 ? 512 : 256;
constexpr int R_STAGE_FLOATS = (R_BM + R_BN) * R_BK;  // 48 KB
constexpr size_t R_SMEM = (size_t)R_STAGES * R_STAGE_FLOATS * sizeof(float);
constexpr int R_EPI = 2;                 // epilogue warp sets (4 warps each: one per TMEM lane quarter)
constexpr int R_THREADS = 64 + 128 * R_EPI;

__host__ __device__ __forceinline__ size_t panel32_off(int r, int c, int ldp) {
    const int t0 = r & ~127;
    const int rows_t = (ldp - t0) < 128 ? (ldp - t0) : 128;
    return (size_t)t0 * ldp + (size_t)(c >> 2) * rows_t * 4 + (size_t)((r - t0) * 4 + (c & 3));
}

// BF16 planes (precision = 3): the same layout with 8 columns per 16-byte chunk ("k8-panel/128", 2-byte elements).
__host__ __device__ __forceinline__ size_t panel16_off(int r, int c, int ldp) {
    const int t0 = r & ~127;
    const int rows_t = (ldp - t0) < 128 ? (ldp - t0) : 128;
    return (size_t)t0 * ldp + (size_t)(c >> 3) * rows_t * 8 + (size_t)((r - t0) * 8 + (c & 7));
}

__device__ __forceinline__ unsigned r_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void r_mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(r_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void r_mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(r_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void r_mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(r_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void r_mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(r_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void r_bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     r_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(r_smem_u32(bar))
                 : "memory");
}
// Shared-memory matrix descriptor, K-major, no swizzle (bit layout as in the sm_100 UMMA descriptor:
// start address >> 4 in [0,14), leading byte offset >> 4 in [16,30), stride byte offset >> 4 in
// [32,46), version 1 in [46,48), layout type 0 in [61,64)).
__device__ __forceinline__ uint64_t r_desc(unsigned addr, unsigned lbo_bytes) {
    uint64_t d = (uint64_t)((addr & 0x3ffffu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
    d |= (uint64_t)(128u >> 4) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// Instruction descriptor: D = F32 ([4,6) = 1), A = B = TF32 ([7,10) = [10,13) = 2), both K-major,
// N >> 3 in [17,23), M >> 4 in [24,29).
__device__ __forceinline__ uint32_t r_idesc(int n_cols) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(n_cols >> 3) << 17) | ((unsigned)(R_BM >> 4) << 24);
}
__device__ __forceinline__ void r_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
// kind::f16: A and B formats in [7,10) and [10,13): 1 = BF16, 0 = FP16; K = 16 per instruction (32 bytes, as TF32's 8).
__device__ __forceinline__ uint32_t r_idesc_bf16(int n_cols, bool fp16 = false) {
    const unsigned fmt = fp16 ? 0u : 1u;
    return (1u << 4) | (fmt << 7) | (fmt << 10) | ((unsigned)(n_cols >> 3) << 17) | ((unsigned)(R_BM >> 4) << 24);
}
__device__ __forceinline__ void r_mma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void r_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(r_smem_u32(bar))
                 : "memory");
}

// Round to nearest TF32 (10-bit mantissa): kind::tf32 ignores the low 13 mantissa bits of its FP32
// operands, so values are rounded when they are stored instead of truncated when they are read.
__device__ __forceinline__ float r_tf32(float x) {
    uint32_t u;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
    return __uint_as_float(u);
}

// 4 x 4 transpose inside every quad of lanes: lane 4m + i holds row i (w[0..3]) and ends with column i.
__device__ __forceinline__ void quad_transpose(float (&w)[4], int lane) {
    const bool o1 = lane & 1, o2 = lane & 2;
    float s0 = o1 ? w[0] : w[1], s1 = o1 ? w[2] : w[3];
    float r0 = __shfl_xor_sync(0xffffffffu, s0, 1), r1 = __shfl_xor_sync(0xffffffffu, s1, 1);
    if (o1) { w[0] = r0; w[2] = r1; } else { w[1] = r0; w[3] = r1; }
    s0 = o2 ? w[0] : w[2]; s1 = o2 ? w[1] : w[3];
    r0 = __shfl_xor_sync(0xffffffffu, s0, 2); r1 = __shfl_xor_sync(0xffffffffu, s1, 2);
    if (o2) { w[0] = r0; w[1] = r1; } else { w[2] = r0; w[3] = r1; }
}

// x = hi + lo with hi = bf16(x), lo = bf16(x - hi): 16 mantissa bits in two BF16 numbers.
__device__ __forceinline__ void bf_split(float x, unsigned short& hi, unsigned short& lo) {
    const __nv_bfloat16 h = __float2bfloat16_rn(x);
    const __nv_bfloat16 l = __float2bfloat16_rn(x - __bfloat162float(h));
    hi = __bfloat16_as_ushort(h);
    lo = __bfloat16_as_ushort(l);
}
__device__ __forceinline__ float bf_val(unsigned short b) { return __uint_as_float((unsigned)b << 16); }
// The same pair of 16-bit planes in either format.  H16: hi = fp16(x), lo = fp16(x - hi): 22 mantissa bits for
// |x| >= 2^-3 (lo becomes subnormal below that: absolute resolution 2^-25), range 65504 -- enough here, the
// iterates have eigenvalues in [-1, 1] and Y = al^2 X^2 <= 2.25.
template <bool H16>
__device__ __forceinline__ void s16_split(float x, unsigned short& hi, unsigned short& lo) {
    if (H16) {
        const __half h = __float2half_rn(x);
        hi = __half_as_ushort(h);
        lo = __half_as_ushort(__float2half_rn(x - __half2float(h)));
    } else {
        bf_split(x, hi, lo);
    }
}
template <bool H16>
__device__ __forceinline__ float s16_val(unsigned short b) {
    return H16 ? __half2float(__ushort_as_half(b)) : bf_val(b);
}
template <bool H16>
__device__ __forceinline__ unsigned short s16_bits(float exact) {  // exact: a value that IS representable
    return H16 ? __half_as_ushort(__float2half_rn(exact)) : (unsigned short)(__float_as_uint(exact) >> 16);
}
__device__ __forceinline__ unsigned bf_pack2(unsigned short a, unsigned short b) { return (unsigned)a | ((unsigned)b << 16); }

// One work unit of the reduced-precision GEMMs.
struct __align__(16) Tile32 {
    int64_t off32;   // offset (floats) of the submatrix in each FP32 buffer
    int32_t grp, ldp, n;
    int32_t ti, tj;  // 128-row tile, 256-column tile
    int32_t tile;    // index in the list (slot of the residual partials)
};

// FP64 k8-panel a_i - mu I  ->  FP32 k4-panel/128 X0 = (a_i - mu I) / s_i (padding written as zeros).
__global__ void __launch_bounds__(256)
k_to_f32(int ngroups, const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
         const int64_t* __restrict__ ws_off, const int64_t* __restrict__ ws_off32,
         const unsigned long long* __restrict__ gersh, const double* __restrict__ X64, float* __restrict__ X32,
         int64_t lo_plane) {  // 0: single FP32 plane; else offset (floats) of the "lo" plane of the hi/lo split
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g], ldp = (n + 15) & ~15;
    double s = __longlong_as_double((long long)gersh[g]);
    const double inv = s > 0.0 ? 1.0 / s : 1.0;
    const double* src = X64 + ws_off[g];
    float* dst = X32 + ws_off32[g];
    const int chunks = ldp >> 2;
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < ldp * chunks; e += gridDim.y * blockDim.x) {
        // consecutive threads -> consecutive rows of one chunk: coalesced 16-byte stores
        const int t = e / (128 * chunks);                 // row tile (all full tiles hold 128 * chunks units)
        const int rows_t = min(128, ldp - 128 * t);
        const int w = e - t * 128 * chunks;
        const int kc = w / rows_t, r = 128 * t + (w - kc * rows_t);
        double x[4] = {0.0, 0.0, 0.0, 0.0};
        if (r < n) {
            const int c = 4 * kc;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (c + j < n) x[j] = src[panel_off(r, c + j, ld)] * inv;
        }
        float* d = dst + panel32_off(r, 4 * kc, ldp);
        if (lo_plane == 0) {
            *reinterpret_cast<float4*>(d) = make_float4((float)x[0], (float)x[1], (float)x[2], (float)x[3]);
        } else {
            float4 hi, lo;
            hi.x = r_tf32((float)x[0]); hi.y = r_tf32((float)x[1]); hi.z = r_tf32((float)x[2]); hi.w = r_tf32((float)x[3]);
            lo.x = (float)(x[0] - hi.x); lo.y = (float)(x[1] - hi.y); lo.z = (float)(x[2] - hi.z); lo.w = (float)(x[3] - hi.w);
            *reinterpret_cast<float4*>(d) = hi;
            *reinterpret_cast<float4*>(d + lo_plane) = lo;
        }
    }
}

// FP32 result -> FP64 k8-panel buffer (the layout scatter / trace kernels read).  A submatrix that
// stopped at iteration 0 is written back unscaled (x s_i), as the FP64 path leaves it.
__global__ void __launch_bounds__(256)
k_to_f64(int ngroups, const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
         const int64_t* __restrict__ ws_off, const int64_t* __restrict__ ws_off32,
         const unsigned long long* __restrict__ gersh, const int32_t* __restrict__ done_iter, int cur_k,
         const float* __restrict__ Xa, const float* __restrict__ Xb, double* __restrict__ X64, int64_t lo_plane) {
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g], ldp = (n + 15) & ~15;
    const int di = done_iter[g];
    const int kb = di >= 0 ? di : cur_k;
    const float* src = ((kb & 1) ? Xb : Xa) + ws_off32[g];
    double mul = 1.0;
    if (kb == 0) {
        const double s = __longlong_as_double((long long)gersh[g]);
        mul = s > 0.0 ? s : 1.0;
    }
    double* dst = X64 + ws_off[g];
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < ld * ld; e += gridDim.y * blockDim.x) {
        const int r = e / ld, c = e - r * ld;
        double v = 0.0;
        if (r < n && c < n) {
            const size_t o = panel32_off(r, c, ldp);
            v = (double)src[o];
            if (lo_plane) v += (double)src[o + lo_plane];
            v *= mul;
        }
        dst[panel_off(r, c, ld)] = v;
    }
}

// precision = 3: FP64 k8-panel a_i - mu I  ->  BF16 hi / lo planes (k8-panel/128, 2-byte elements) of X0.
template <bool H16>
__global__ void __launch_bounds__(256)
k_to_bf16(int ngroups, const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
          const int64_t* __restrict__ ws_off, const int64_t* __restrict__ ws_off32,
          const unsigned long long* __restrict__ gersh, const double* __restrict__ X64,
          unsigned short* __restrict__ X16, int64_t lo_plane) {
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g], ldp = (n + 15) & ~15;
    double s = __longlong_as_double((long long)gersh[g]);
    const double inv = s > 0.0 ? 1.0 / s : 1.0;
    const double* src = X64 + ws_off[g];
    unsigned short* dst = X16 + ws_off32[g];
    const int chunks = ldp >> 3;
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < ldp * chunks; e += gridDim.y * blockDim.x) {
        const int t = e / (128 * chunks);
        const int rows_t = min(128, ldp - 128 * t);
        const int w = e - t * 128 * chunks;
        const int kc = w / rows_t, r = 128 * t + (w - kc * rows_t);
        unsigned short hi[8], lo[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int c = 8 * kc + j;
            const double x = (r < n && c < n) ? src[panel_off(r, c, ld)] * inv : 0.0;
            unsigned short d0;
            s16_split<H16>((float)x, hi[j], d0);
            s16_split<H16>((float)(x - (double)s16_val<H16>(hi[j])), lo[j], d0);  // lo: the FP64 remainder, rounded
        }
        unsigned short* d = dst + panel16_off(r, 8 * kc, ldp);
        *reinterpret_cast<uint4*>(d) = make_uint4(bf_pack2(hi[0], hi[1]), bf_pack2(hi[2], hi[3]), bf_pack2(hi[4], hi[5]), bf_pack2(hi[6], hi[7]));
        *reinterpret_cast<uint4*>(d + lo_plane) = make_uint4(bf_pack2(lo[0], lo[1]), bf_pack2(lo[2], lo[3]), bf_pack2(lo[4], lo[5]), bf_pack2(lo[6], lo[7]));
    }
}

// precision = 3: BF16 hi + lo result -> FP64 k8-panel buffer (as k_to_f64).
template <bool H16>
__global__ void __launch_bounds__(256)
k_from_bf16(int ngroups, const int32_t* __restrict__ sub_dim, const int32_t* __restrict__ ldv,
            const int64_t* __restrict__ ws_off, const int64_t* __restrict__ ws_off32,
            const unsigned long long* __restrict__ gersh, const int32_t* __restrict__ done_iter, int cur_k,
            const unsigned short* __restrict__ Xa, const unsigned short* __restrict__ Xb, double* __restrict__ X64,
            int64_t lo_plane) {
    const int g = blockIdx.x;
    const int n = sub_dim[g], ld = ldv[g], ldp = (n + 15) & ~15;
    const int di = done_iter[g];
    const int kb = di >= 0 ? di : cur_k;
    const unsigned short* src = ((kb & 1) ? Xb : Xa) + ws_off32[g];
    double mul = 1.0;
    if (kb == 0) {
        const double s = __longlong_as_double((long long)gersh[g]);
        mul = s > 0.0 ? s : 1.0;
    }
    double* dst = X64 + ws_off[g];
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < ld * ld; e += gridDim.y * blockDim.x) {
        const int r = e / ld, c = e - r * ld;
        double v = 0.0;
        if (r < n && c < n) {
            const size_t o = panel16_off(r, c, ldp);
            v = ((double)s16_val<H16>(src[o]) + (double)s16_val<H16>(src[o + lo_plane])) * mul;
        }
        dst[panel_off(r, c, ld)] = v;
    }
}

struct Ns32Args {
    const Tile32* tiles;
    const float* A;        // X_k
    const float* B;        // MODE 0: X_k, MODE 1: Y_k
    float* Out;            // MODE 0: Y_k, MODE 1: X_{k+1}
    double* partials;      // [n_tiles][4]
    const int32_t* done_iter;
    int64_t lo_plane;      // SPLIT: offset (floats) of the lo plane inside A, B, Out
    const int32_t* ctrl;   // [0] != 0: evaluation stopped on the device: empty launch
    int32_t n_tiles;
};

// SPLIT = 0: plain TF32 (operands truncated to 10 mantissa bits by the tensor core).
// SPLIT = 1: "3xTF32": every operand is stored as hi + lo with hi = tf32(x), lo = x - hi, and a
//            product is hi hi + hi lo + lo hi accumulated in the same FP32 TMEM tile (FP32-class
//            accuracy, three MMAs per k step, 16-wide k slices so that a stage stays 48 KB).
// SPLIT = 2: "BF16x2": hi = bf16(x), lo = bf16(x - hi) in two BF16 planes, the same three products with
//            kind::f16 (K = 16 per instruction), 32-wide k slices (48 KB per stage).
template <int MODE, int SPLIT>
__global__ void __launch_bounds__(R_THREADS, R_CTAS) k_ns_tf32(Ns32Args a) {
    constexpr bool BF = SPLIT >= 2;                 // 16-bit hi / lo planes instead of FP32 ones (2: BF16, 3: FP16)
    constexpr bool H16 = SPLIT == 3;
    constexpr bool PIPE = SPLIT == 0;               // software-pipelined epilogue (the split variants lack the registers)
    constexpr int CW = BF ? 8 : 4;                  // columns per 16-byte chunk
    constexpr int ES = BF ? 2 : 4;                  // bytes per element
    constexpr int CH = SPLIT ? 4 : 8;               // chunks per stage and plane
    constexpr int BK = CH * CW;                     // k columns per stage
    constexpr int PL = SPLIT ? 2 : 1;               // operand planes
    constexpr int SA = R_BM * CH * 4;               // 4-byte units of one 128-row operand plane in a stage
    extern __shared__ __align__(128) float rsm[];
    __shared__ __align__(8) uint64_t s_full[R_STAGES], s_empty[R_STAGES], s_tfull[2], s_tempty[2];
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < R_STAGES; ++s) { r_mbar_init(&s_full[s], 1); r_mbar_init(&s_empty[s], 1); }
        for (int b = 0; b < 2; ++b) { r_mbar_init(&s_tfull[b], 1); r_mbar_init(&s_tempty[b], 4 * R_EPI); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (wid == 1) {  // tensor memory: all 512 columns (one CTA per SM), two 256-column accumulators
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(r_smem_u32(&s_tmem)), "n"(R_TCOLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = s_tmem;
    const int n_tiles = a.ctrl[0] != 0 ? 0 : a.n_tiles;
    // Tiles are dealt to the CTAs in consecutive PAIRS when there are enough of them: the 128-row units of one
    // submatrix share operand rows (unit 1 reads the rows of unit 0 as its first B half), and back to back on one
    // CTA the second read hits L2.
    const bool pair = a.n_tiles >= 4 * (int)gridDim.x;
#define R_TILES(t)                                                                     \
    for (int t = pair ? 2 * (int)blockIdx.x : (int)blockIdx.x; t < n_tiles;            \
         t += pair ? ((t & 1) ? 2 * (int)gridDim.x - 1 : 1) : (int)gridDim.x)

    if (wid == 0) {
        // ================================================================ producer (one thread)
        if (lane == 0) {
            int stage = 0;
            unsigned phase = 0;
            R_TILES(t) {
                const Tile32 T = a.tiles[t];
                if (a.done_iter[T.grp] >= 0) continue;
                const int ldp = T.ldp;
                const int row0 = T.ti * R_BM, rows_a = min(R_BM, ldp - row0);
                const int col0 = T.tj * R_BN, ncols = min(R_BN, min(ldp, row0 + R_BM) - col0);  // lower triangle only
                const int rows_b0 = min(128, ncols), rows_b1 = max(0, ncols - 128);
                // Y = X X: a B half that covers the rows of A IS the A slice (X is symmetric and B is read as rows):
                // it is loaded once and the issuer points both descriptors at it
                const bool b0_is_a = MODE == 0 && col0 == row0, b1_is_a = MODE == 0 && rows_b1 > 0 && col0 + 128 == row0;
                const char* Asrc = reinterpret_cast<const char*>(a.A) + ((size_t)T.off32 + (size_t)row0 * ldp) * ES;
                const char* B0 = reinterpret_cast<const char*>(a.B) + ((size_t)T.off32 + (size_t)col0 * ldp) * ES;
                const char* B1 = reinterpret_cast<const char*>(a.B) + ((size_t)T.off32 + (size_t)(col0 + 128) * ldp) * ES;
                for (int k0 = 0; k0 < ldp; k0 += BK) {
                    const int chunks = min(BK, ldp - k0) / CW;
                    r_mbar_wait(&s_empty[stage], phase ^ 1);
                    float* sa = rsm + (size_t)stage * R_STAGE_FLOATS;
                    const unsigned ba = (unsigned)(chunks * rows_a * 16), bb0 = (unsigned)(chunks * rows_b0 * 16),
                                   bb1 = (unsigned)(chunks * rows_b1 * 16);
                    r_mbar_expect_tx(&s_full[stage], PL * (ba + (b0_is_a ? 0u : bb0) + (b1_is_a ? 0u : bb1)));
#pragma unroll
                    for (int pl = 0; pl < PL; ++pl) {  // stage layout: [A planes][B0 planes][B1 planes]
                        const size_t po = (size_t)pl * a.lo_plane * ES, kc = (size_t)(k0 / CW) * 16;
                        r_bulk_g2s(sa + pl * SA, Asrc + po + kc * rows_a, ba, &s_full[stage]);
                        if (!b0_is_a) r_bulk_g2s(sa + (PL + pl) * SA, B0 + po + kc * rows_b0, bb0, &s_full[stage]);
                        if (rows_b1 > 0 && !b1_is_a)
                            r_bulk_g2s(sa + (2 * PL + pl) * SA, B1 + po + kc * rows_b1, bb1, &s_full[stage]);
                    }
                    if (++stage == R_STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (wid == 1) {
        // ================================================================ MMA issuer (one thread)
        if (lane == 0) {
            int stage = 0, buf = 0;
            unsigned phase = 0, tphase[2] = {0, 0};
            R_TILES(t) {
                const Tile32 T = a.tiles[t];
                if (a.done_iter[T.grp] >= 0) continue;
                const int ldp = T.ldp;
                const int row0 = T.ti * R_BM, rows_a = min(R_BM, ldp - row0);
                const int col0 = T.tj * R_BN, ncols = min(R_BN, min(ldp, row0 + R_BM) - col0);
                const int rows_b0 = min(128, ncols), rows_b1 = max(0, ncols - 128);
                const bool b0_is_a = MODE == 0 && col0 == row0, b1_is_a = MODE == 0 && rows_b1 > 0 && col0 + 128 == row0;
                r_mbar_wait(&s_tempty[buf], tphase[buf] ^ 1);  // epilogue has drained this accumulator
                asm volatile("tcgen05.fence::after_thread_sync;");
                const uint32_t d0 = tmem + (uint32_t)(buf * R_BN);
                const uint32_t id0 = BF ? r_idesc_bf16(rows_b0, H16) : r_idesc(rows_b0);
                const uint32_t id1 = BF ? r_idesc_bf16(rows_b1 > 0 ? rows_b1 : 16, H16) : r_idesc(rows_b1 > 0 ? rows_b1 : 16);
                auto mma = [&](uint32_t d, uint64_t da, uint64_t db, uint32_t id, uint32_t acc) {
                    if (BF) r_mma_bf16(d, da, db, id, acc); else r_mma(d, da, db, id, acc);
                };
                for (int k0 = 0; k0 < ldp; k0 += BK) {
                    const int ksteps = min(BK, ldp - k0) / (2 * CW);  // two 16-byte chunks per instruction
                    r_mbar_wait(&s_full[stage], phase);
                    asm volatile("tcgen05.fence::after_thread_sync;");
                    const unsigned sa = r_smem_u32(rsm + (size_t)stage * R_STAGE_FLOATS);
                    const unsigned sb0 = b0_is_a ? sa : sa + PL * SA * 4, sb1 = b1_is_a ? sa : sa + 2 * PL * SA * 4;
                    for (int ks = 0; ks < ksteps; ++ks) {
                        const uint32_t acc = (k0 > 0 || ks > 0) ? 1u : 0u;
                        const unsigned oa = (unsigned)(ks * 2 * rows_a * 16), ob0 = (unsigned)(ks * 2 * rows_b0 * 16),
                                       ob1 = (unsigned)(ks * 2 * rows_b1 * 16);
                        const unsigned la = (unsigned)(rows_a * 16), lb0 = (unsigned)(rows_b0 * 16), lb1 = (unsigned)(rows_b1 * 16);
                        const uint64_t da = r_desc(sa + oa, la);
                        mma(d0, da, r_desc(sb0 + ob0, lb0), id0, acc);                                  // hi hi
                        if (SPLIT) {
                            mma(d0, da, r_desc(sb0 + SA * 4 + ob0, lb0), id0, 1u);                      // hi lo
                            mma(d0, r_desc(sa + SA * 4 + oa, la), r_desc(sb0 + ob0, lb0), id0, 1u);      // lo hi
                        }
                        if (rows_b1 > 0) {
                            mma(d0 + 128, da, r_desc(sb1 + ob1, lb1), id1, acc);
                            if (SPLIT) {
                                mma(d0 + 128, da, r_desc(sb1 + SA * 4 + ob1, lb1), id1, 1u);
                                mma(d0 + 128, r_desc(sa + SA * 4 + oa, la), r_desc(sb1 + ob1, lb1), id1, 1u);
                            }
                        }
                    }
                    r_commit(&s_empty[stage]);  // the stage is free once these MMAs have read it
                    if (++stage == R_STAGES) { stage = 0; phase ^= 1; }
                }
                r_commit(&s_tfull[buf]);        // accumulator complete
                tphase[buf] ^= 1;
                if (R_TBUFS == 2) buf ^= 1;
            }
        }
    } else {
        // ================================================================ epilogue warps 2..9
        const int q = wid & 3;  // TMEM lane quarter this warp may access
        const int eset = (wid - 2) >> 2;  // warp set: the sets split the 16-column chunks of a tile between them
        int buf = 0;
        unsigned tphase[2] = {0, 0};
        R_TILES(t) {
            const Tile32 T = a.tiles[t];
            if (a.done_iter[T.grp] >= 0) continue;
            const int ldp = T.ldp, n = T.n;
            const int row0 = T.ti * R_BM, rows_a = min(R_BM, ldp - row0);
            const int col0 = T.tj * R_BN, ncols = min(R_BN, min(ldp, row0 + R_BM) - col0);
            const int rl = q * 32 + lane, r = row0 + rl;
            r_mbar_wait(&s_tfull[buf], tphase[buf]);
            tphase[buf] ^= 1;
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * R_BN);
            float* orow = a.Out + T.off32 + (size_t)row0 * ldp + (size_t)rl * 4;
            const float* xrow = a.A + T.off32 + (size_t)row0 * ldp + (size_t)rl * 4;
            double part = 0.0;
            const int nch = (ncols + 15) >> 4, csplit = ((nch + R_EPI - 1) / R_EPI) * 16;
            const int cbeg = min(ncols, eset * csplit), cend = min(ncols, cbeg + csplit);
            // Software pipeline over the 16-column chunks: the tensor-memory load of chunk c + 1 and (MODE 1) the
            // global loads of its X values are issued before chunk c is processed, so their latencies pass
            // behind the arithmetic and the stores of chunk c.
            uint32_t v[16], vn[16];
            auto tld = [&](uint32_t (&d)[16], int c0) {
                asm volatile(
                    "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                    : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]), "=r"(d[4]), "=r"(d[5]), "=r"(d[6]), "=r"(d[7]),
                      "=r"(d[8]), "=r"(d[9]), "=r"(d[10]), "=r"(d[11]), "=r"(d[12]), "=r"(d[13]), "=r"(d[14]), "=r"(d[15])
                    : "r"(taddr + (uint32_t)c0));
            };
            if constexpr (!BF) {
                float4 xc[4], xn[4], xlc[4], xln[4];
                auto xld = [&](float4 (&x)[4], float4 (&xl)[4], int c0) {  // MODE 1: X (and its lo plane) of this row
    #pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int c = col0 + c0 + 4 * j;
                        x[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                        xl[j] = x[j];
                        if (rl < rows_a && c <= r) {
                            const size_t o = (size_t)(c >> 2) * rows_a * 4;
                            x[j] = *reinterpret_cast<const float4*>(xrow + o);
                            if (SPLIT) xl[j] = *reinterpret_cast<const float4*>(xrow + o + a.lo_plane);
                        }
                    }
                };
                if (PIPE) { tld(v, cbeg); if (MODE == 1) xld(xc, xlc, cbeg); }
                for (int c0 = cbeg; c0 < cend; c0 += 16) {
                    if (!PIPE) { tld(v, c0); if (MODE == 1) xld(xc, xlc, c0); }
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    const bool more = PIPE && c0 + 16 < cend;
                    if (more) {
                        tld(vn, c0 + 16);
                        if (MODE == 1) xld(xn, xln, c0 + 16);
                    }
                    {
                        const bool row_ok = rl < rows_a;
                        const int rq = r & ~3;  // first row of this lane's quad (rows_a is a multiple of 16: quads are whole)
    #pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int c = col0 + c0 + 4 * j;
                            const bool act = row_ok && c <= r;  // upper triangle: the mirror image of (c, r) is stored instead
                            const size_t o = (size_t)(c >> 2) * rows_a * 4;
                            float w[4] = {__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                                          __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3])};
                            if (MODE == 0) {
                                if (act && r < n) {  // residual over the n x n part; strictly-lower elements count twice
                                    float p = 0.f;
    #pragma unroll
                                    for (int e = 0; e < 4; ++e) {
                                        const float d = w[e] - (c + e == r ? 1.f : 0.f);
                                        if (c + e < r) p += 2.f * d * d;
                                        else if (c + e == r) p += d * d;
                                    }
                                    part += (double)p;
                                }
                            } else {
                                float4 x = xc[j];
                                if (SPLIT) { x.x += xlc[j].x; x.y += xlc[j].y; x.z += xlc[j].z; x.w += xlc[j].w; }
                                w[0] = 1.5f * x.x - 0.5f * w[0]; w[1] = 1.5f * x.y - 0.5f * w[1];
                                w[2] = 1.5f * x.z - 0.5f * w[2]; w[3] = 1.5f * x.w - 0.5f * w[3];
                            }
                            float hi[4], lo[4];
    #pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                hi[e] = SPLIT ? r_tf32(w[e]) : w[e];
                                lo[e] = w[e] - hi[e];
                            }
                            // direct elements (r, c + e), c + e <= r: one 16-byte store when the whole group is
                            // on or below the diagonal.  Every stored element has exactly one writer, so X and Y stay
                            // bitwise symmetric, which is what lets B be read as rows (and keeps the iteration
                            // stable: the X X^T form amplifies any antisymmetric rounding noise).
                            if (act) {
                                if (c + 3 <= r) {
                                    *reinterpret_cast<float4*>(orow + o) = make_float4(hi[0], hi[1], hi[2], hi[3]);
                                    if (SPLIT) *reinterpret_cast<float4*>(orow + o + a.lo_plane) = make_float4(lo[0], lo[1], lo[2], lo[3]);
                                } else {
    #pragma unroll
                                    for (int e = 0; e < 4; ++e)
                                        if (c + e <= r) {
                                            orow[o + e] = hi[e];
                                            if (SPLIT) orow[o + e + a.lo_plane] = lo[e];
                                        }
                                }
                            }
                            // mirror elements (c + e, r), c + e < r.  A quad of lanes (rows rq .. rq + 3) holds a 4 x 4
                            // block; when it lies strictly below the diagonal it is transposed inside the quad (four
                            // shuffles per plane, executed by every lane) and lane e stores mirror row c + e as ONE
                            // 16-byte store; blocks touching the diagonal keep the 4-byte stores.
                            const bool blk = row_ok && c + 3 < rq;
                            float th[4] = {hi[0], hi[1], hi[2], hi[3]}, tl[4] = {lo[0], lo[1], lo[2], lo[3]};
                            quad_transpose(th, lane);
                            if (SPLIT) quad_transpose(tl, lane);
                            if (blk) {
                                float* mp = a.Out + T.off32 + panel32_off(c + (lane & 3), rq, ldp);
                                *reinterpret_cast<float4*>(mp) = make_float4(th[0], th[1], th[2], th[3]);
                                if (SPLIT) *reinterpret_cast<float4*>(mp + a.lo_plane) = make_float4(tl[0], tl[1], tl[2], tl[3]);
                            } else if (act) {
    #pragma unroll
                                for (int e = 0; e < 4; ++e)
                                    if (c + e < r) {
                                        float* mp = a.Out + T.off32 + panel32_off(c + e, r, ldp);
                                        *mp = hi[e];
                                        if (SPLIT) mp[a.lo_plane] = lo[e];
                                    }
                            }
                        }
                    }
                    if (more) {
    #pragma unroll
                        for (int e = 0; e < 16; ++e) v[e] = vn[e];
                        if (MODE == 1) {
    #pragma unroll
                            for (int j = 0; j < 4; ++j) { xc[j] = xn[j]; xlc[j] = xln[j]; }
                        }
                    }
                }
            } else {
                // BF16 hi / lo planes: 8 columns per 16-byte chunk.  Direct elements go out as 16-byte stores per
                // plane, mirror elements as 8-byte stores (4 x 4 blocks transposed inside the lane quads).
                unsigned short* o16 = reinterpret_cast<unsigned short*>(a.Out) + T.off32;
                unsigned short* orow16 = o16 + (size_t)row0 * ldp + (size_t)rl * 8;
                const unsigned short* xrow16 =
                    reinterpret_cast<const unsigned short*>(a.A) + T.off32 + (size_t)row0 * ldp + (size_t)rl * 8;
                uint4 xh[2], xl[2], xhn[2], xln[2];
                auto xld16 = [&](uint4 (&h)[2], uint4 (&l)[2], int c0) {
#pragma unroll
                    for (int jj = 0; jj < 2; ++jj) {
                        const int c = col0 + c0 + 8 * jj;
                        h[jj] = make_uint4(0u, 0u, 0u, 0u);
                        l[jj] = h[jj];
                        if (rl < rows_a && c <= r) {
                            const size_t o = (size_t)(c >> 3) * rows_a * 8;
                            h[jj] = *reinterpret_cast<const uint4*>(xrow16 + o);
                            l[jj] = *reinterpret_cast<const uint4*>(xrow16 + o + a.lo_plane);
                        }
                    }
                };
                if (PIPE) { tld(v, cbeg); if (MODE == 1) xld16(xh, xl, cbeg); }
                for (int c0 = cbeg; c0 < cend; c0 += 16) {
                    if (!PIPE) { tld(v, c0); if (MODE == 1) xld16(xh, xl, c0); }
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    const bool more = PIPE && c0 + 16 < cend;
                    if (more) {
                        tld(vn, c0 + 16);
                        if (MODE == 1) xld16(xhn, xln, c0 + 16);
                    }
                    const bool row_ok = rl < rows_a;
                    const int rq = r & ~3;
#pragma unroll
                    for (int jj = 0; jj < 2; ++jj) {
                        const int c = col0 + c0 + 8 * jj;
                        const bool act = row_ok && c <= r;
                        const size_t o = (size_t)(c >> 3) * rows_a * 8;
                        float w[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) w[e] = __uint_as_float(v[8 * jj + e]);
                        if (MODE == 0) {
                            if (act && r < n) {
                                float pr = 0.f;
#pragma unroll
                                for (int e = 0; e < 8; ++e) {
                                    const float d = w[e] - (c + e == r ? 1.f : 0.f);
                                    if (c + e < r) pr += 2.f * d * d;
                                    else if (c + e == r) pr += d * d;
                                }
                                part += (double)pr;
                            }
                        } else {
                            const unsigned hw[4] = {xh[jj].x, xh[jj].y, xh[jj].z, xh[jj].w};
                            const unsigned lw[4] = {xl[jj].x, xl[jj].y, xl[jj].z, xl[jj].w};
#pragma unroll
                            for (int e = 0; e < 8; ++e) {
                                const unsigned short hb = (unsigned short)(hw[e >> 1] >> (16 * (e & 1)));
                                const unsigned short lb = (unsigned short)(lw[e >> 1] >> (16 * (e & 1)));
                                const float x = s16_val<H16>(hb) + s16_val<H16>(lb);
                                w[e] = 1.5f * x - 0.5f * w[e];
                            }
                        }
                        unsigned short hi[8], lo[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) s16_split<H16>(w[e], hi[e], lo[e]);
                        if (act) {
                            if (c + 7 <= r) {
                                *reinterpret_cast<uint4*>(orow16 + o) = make_uint4(bf_pack2(hi[0], hi[1]), bf_pack2(hi[2], hi[3]),
                                                                                   bf_pack2(hi[4], hi[5]), bf_pack2(hi[6], hi[7]));
                                *reinterpret_cast<uint4*>(orow16 + o + a.lo_plane) =
                                    make_uint4(bf_pack2(lo[0], lo[1]), bf_pack2(lo[2], lo[3]), bf_pack2(lo[4], lo[5]), bf_pack2(lo[6], lo[7]));
                            } else {
#pragma unroll
                                for (int e = 0; e < 8; ++e)
                                    if (c + e <= r) { orow16[o + e] = hi[e]; orow16[o + e + a.lo_plane] = lo[e]; }
                            }
                        }
#pragma unroll
                        for (int q4 = 0; q4 < 2; ++q4) {
                            const int cc = c + 4 * q4;
                            const bool blk = row_ok && cc + 3 < rq;
                            float th[4], tl[4];
#pragma unroll
                            for (int e = 0; e < 4; ++e) { th[e] = s16_val<H16>(hi[4 * q4 + e]); tl[e] = s16_val<H16>(lo[4 * q4 + e]); }
                            quad_transpose(th, lane);
                            quad_transpose(tl, lane);
                            if (blk) {
                                unsigned short* mp = o16 + panel16_off(cc + (lane & 3), rq, ldp);
                                *reinterpret_cast<uint2*>(mp) =
                                    make_uint2(bf_pack2(s16_bits<H16>(th[0]), s16_bits<H16>(th[1])),
                                               bf_pack2(s16_bits<H16>(th[2]), s16_bits<H16>(th[3])));
                                *reinterpret_cast<uint2*>(mp + a.lo_plane) =
                                    make_uint2(bf_pack2(s16_bits<H16>(tl[0]), s16_bits<H16>(tl[1])),
                                               bf_pack2(s16_bits<H16>(tl[2]), s16_bits<H16>(tl[3])));
                            } else if (row_ok) {
#pragma unroll
                                for (int e = 0; e < 4; ++e)
                                    if (cc + e < r) {
                                        unsigned short* mp = o16 + panel16_off(cc + e, r, ldp);
                                        *mp = hi[4 * q4 + e];
                                        mp[a.lo_plane] = lo[4 * q4 + e];
                                    }
                            }
                        }
                    }
                    if (more) {
#pragma unroll
                        for (int e = 0; e < 16; ++e) v[e] = vn[e];
                        if (MODE == 1) {
#pragma unroll
                            for (int jj = 0; jj < 2; ++jj) { xh[jj] = xhn[jj]; xl[jj] = xln[jj]; }
                        }
                    }
                }
            }
            asm volatile("tcgen05.fence::before_thread_sync;");
            __syncwarp();
            if (lane == 0) r_mbar_arrive(&s_tempty[buf]);
            if (MODE == 0) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
                if (lane == 0) a.partials[(size_t)T.tile * (4 * R_EPI) + 4 * eset + q] = part;
            }
            if (R_TBUFS == 2) buf ^= 1;
        }
    }
#undef R_TILES
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (wid == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(R_TCOLS));
}

// Residual decision of the reduced-precision iteration: like k_ns_decide, but the residual has a
// precision floor.  r < 1/(2 sqrt(n)) means every eigenvalue satisfies |1 - x^2| < 1/2, i.e. the
// exact iteration at least halves r from there on; "two consecutive residuals inside that zone and
// no halving" is therefore the precision floor: the submatrix stops as converged-to-the-floor, and
// the floor is reported in sm_stats_t.max_residual.  Hard cap of 40 iterations (noise cannot be
// iterated away).
__global__ void __launch_bounds__(256)
k_ns_decide32(int ngroups, int k, int decide_only, double eps, double floor_zone,
              const int32_t* __restrict__ tile_first,
              const int32_t* __restrict__ tile_count, const int32_t* __restrict__ sub_dim,
              const double* __restrict__ partials, double* __restrict__ res, int32_t* __restrict__ done_iter,
              int32_t* __restrict__ flag, int32_t* __restrict__ counters, const int32_t* __restrict__ ctrl) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= ngroups || ctrl[0] != 0) return;
    if (done_iter[g] >= 0) return;
    const int lane = threadIdx.x & 31;
    const int cnt = 4 * R_EPI * tile_count[g], n = sub_dim[g];
    const double* pp = partials + (size_t)tile_first[g] * (4 * R_EPI);
    double r2 = 0.0;
    for (int t = lane; t < cnt; t += 32) r2 += pp[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
    if (lane == 0) {
        const double r = sqrt(r2 / (double)(n > 0 ? n : 1));
        const double prev = k > 0 ? res[(size_t)((k - 1) & 1) * ngroups + g] : 1e300;
        const bool conv = r < eps;
        const double zone = floor_zone / sqrt((double)(n > 0 ? n : 1));
        const bool floor_hit = (k > 0) && (prev < zone) && (r < zone) && (r >= 0.5 * prev);
        const bool stop = conv || floor_hit || decide_only || k >= 40 || !(r == r);
        res[(size_t)(k & 1) * ngroups + g] = r;
        if (stop) { flag[g] = (conv || floor_hit) ? 0 : 1; done_iter[g] = k; }
        else atomicAdd(counters + k, 1);
    }
}

// Tile list and FP32 offsets of the reduced-precision path (plan creation, precision = 1).
sm_status_t build_tf32_tables(sm_plan* p, cudaStream_t st) {
    const int ng = p->ngroups;
    std::vector<int64_t> off32(ng);
    std::vector<int32_t> first(ng), count(ng);
    std::vector<Tile32> tiles;
    int64_t off = 0;
    for (int g = 0; g < ng; ++g) {
        const int n = p->h_sub_dim[g], ldp = (n + 15) & ~15;
        off32[g] = off;
        off += (int64_t)ldp * ldp;
        first[g] = (int32_t)tiles.size();
        for (int ti = 0; ti * R_BM < ldp; ++ti)
            for (int tj = 0; tj * R_BN < std::min(ldp, (ti + 1) * R_BM); ++tj) {  // lower triangle only
                Tile32 t;
                t.off32 = off32[g]; t.grp = g; t.ldp = ldp; t.n = n; t.ti = ti; t.tj = tj; t.tile = (int32_t)tiles.size();
                tiles.push_back(t);
            }
        count[g] = (int32_t)tiles.size() - first[g];
    }
    p->sum_ldp2 = off;
    const int planes = p->opt.precision == 2 ? 2 : 1;
    p->n_tiles32 = (int64_t)tiles.size();
    auto up = [&](void** d, const void* h, size_t bytes) -> sm_status_t {
        SM_CUDA(cudaMalloc(d, std::max<size_t>(bytes, 16)));
        if (bytes) SM_CUDA(cudaMemcpyAsync(*d, h, bytes, cudaMemcpyHostToDevice, st));
        return SM_OK;
    };
    sm_status_t s;
    if ((s = up((void**)&p->d_ws_off32, off32.data(), (size_t)ng * 8))) return s;
    if ((s = up((void**)&p->d_tile_first32, first.data(), (size_t)ng * 4))) return s;
    if ((s = up((void**)&p->d_tile_count32, count.data(), (size_t)ng * 4))) return s;
    if ((s = up((void**)&p->d_tiles32, tiles.data(), tiles.size() * sizeof(Tile32)))) return s;
    SM_CUDA(cudaMalloc((void**)&p->d_partials32, std::max<size_t>((size_t)tiles.size() * 32 * R_EPI, 16)));
    SM_CUDA(cudaStreamSynchronize(st));
    // each of the three workspace buffers must hold the FP64 matrices and the FP32 ones
    const size_t need = std::max((size_t)p->sum_ld2 * 8, (size_t)p->sum_ldp2 * 4 * planes);
    const size_t buf = (need + 255) / 256 * 256;
    p->info.workspace_bytes = 3 * buf;
    return SM_OK;
}

// buf0: gathered FP64 a_i - mu I (in), afterwards Y (FP32) during the iteration and the FP64 result
// at the end; buf1 / bufY: X ping / pong (FP32).
sm_status_t launch_to_f32(sm_plan* p, const double* buf0, double* buf1, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    const int split = (int)std::min<int64_t>(8, std::max<int64_t>(1, (int64_t)p->num_sms * 8 / p->ngroups));
    if (p->opt.precision == 3)
        k_to_bf16<false><<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off,
                                                                   p->d_ws_off32, p->d_gersh, buf0,
                                                                   reinterpret_cast<unsigned short*>(buf1), p->sum_ldp2);
    else if (p->opt.precision == 4)
        k_to_bf16<true><<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off,
                                                                  p->d_ws_off32, p->d_gersh, buf0,
                                                                  reinterpret_cast<unsigned short*>(buf1), p->sum_ldp2);
    else
        k_to_f32<<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off, p->d_ws_off32,
                                                           p->d_gersh, buf0, reinterpret_cast<float*>(buf1),
                                                           p->opt.precision == 2 ? p->sum_ldp2 : 0);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

sm_status_t launch_to_f64(sm_plan* p, double* buf0, const double* buf1, const double* bufY, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    const int split = (int)std::min<int64_t>(8, std::max<int64_t>(1, (int64_t)p->num_sms * 8 / p->ngroups));
    if (p->opt.precision == 3)
        k_from_bf16<false><<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off,
                                                                     p->d_ws_off32, p->d_gersh, p->d_done_iter, p->cur_k,
                                                                     reinterpret_cast<const unsigned short*>(buf1),
                                                                     reinterpret_cast<const unsigned short*>(bufY), buf0,
                                                                     p->sum_ldp2);
    else if (p->opt.precision == 4)
        k_from_bf16<true><<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off,
                                                                    p->d_ws_off32, p->d_gersh, p->d_done_iter, p->cur_k,
                                                                    reinterpret_cast<const unsigned short*>(buf1),
                                                                    reinterpret_cast<const unsigned short*>(bufY), buf0,
                                                                    p->sum_ldp2);
    else
        k_to_f64<<<dim3(p->ngroups, split), 256, 0, st>>>(p->ngroups, p->d_sub_dim, p->d_ld, p->d_ws_off, p->d_ws_off32,
                                                           p->d_gersh, p->d_done_iter, p->cur_k,
                                                           reinterpret_cast<const float*>(buf1),
                                                           reinterpret_cast<const float*>(bufY), buf0,
                                                           p->opt.precision == 2 ? p->sum_ldp2 : 0);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

sm_status_t launch_ns_pair_tf32(sm_plan* p, int k, double eps, int decide_only, double* buf0, double* buf1,
                                double* bufY, cudaStream_t st, int which) {
    if (p->n_tiles32 == 0) return SM_OK;
    if (!p->tf32_attr_set) {  // per plan: the attribute belongs to the device the plan was created on
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<0, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<0, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        SM_CUDA(cudaFuncSetAttribute(k_ns_tf32<1, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)R_SMEM));
        p->tf32_attr_set = 1;
    }
    float* X[2] = {reinterpret_cast<float*>(buf1), reinterpret_cast<float*>(bufY)};
    float* Y = reinterpret_cast<float*>(buf0);
    Ns32Args a;
    a.tiles = reinterpret_cast<const Tile32*>(p->d_tiles32); a.partials = p->d_partials32; a.done_iter = p->d_done_iter;
    a.n_tiles = (int32_t)p->n_tiles32; a.ctrl = p->d_ctrl;
    const int split = p->opt.precision == 2 ? 1 : p->opt.precision == 3 ? 2 : p->opt.precision == 4 ? 3 : 0;
    a.lo_plane = split ? p->sum_ldp2 : 0;
    const int grid = (int)std::min<int64_t>(p->n_tiles32, (int64_t)p->num_sms * R_CTAS);
    if (which & 1) {
        a.A = X[k & 1]; a.B = X[k & 1]; a.Out = Y;
        if (split == 3) k_ns_tf32<0, 3><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else if (split == 2) k_ns_tf32<0, 2><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else if (split == 1) k_ns_tf32<0, 1><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else k_ns_tf32<0, 0><<<grid, R_THREADS, R_SMEM, st>>>(a);
        k_ns_decide32<<<(p->ngroups + 7) / 8, 256, 0, st>>>(p->ngroups, k, decide_only, eps, 0.5,
                                                            p->d_tile_first32,
                                                            p->d_tile_count32, p->d_sub_dim, p->d_partials32, p->d_res,
                                                            p->d_done_iter, p->d_flag, p->d_counters, p->d_ctrl);
        p->launches += 2;
    }
    if ((which & 2) && !decide_only) {
        a.A = X[k & 1]; a.B = Y; a.Out = X[(k + 1) & 1];
        if (split == 3) k_ns_tf32<1, 3><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else if (split == 2) k_ns_tf32<1, 2><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else if (split == 1) k_ns_tf32<1, 1><<<grid, R_THREADS, R_SMEM, st>>>(a);
        else k_ns_tf32<1, 0><<<grid, R_THREADS, R_SMEM, st>>>(a);
        p->launches += 1;
    }
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

}  // namespace smb
