// SURVEY 8(f)1, the eigensolver of method = 1 (Eq.(17) first line, L246-255): block one-sided Jacobi, the
// O(n^3) part on the FP64 tensor-core instruction (mma.sync m8n8k4 f64, SASS DMMA).
//
// Mathematics as stated in eig.cu (G = B V with B = a_i + sigma I positive definite; at convergence the columns of G
// are mutually orthogonal, lambda_l = ||g_l|| - sigma, q_l = g_l / ||g_l||).  The columns are visited in BLOCK pairs
// and a visit is three dense steps instead of 256 separate plane rotations of full-length columns:
//   1. Gram matrix M = [G_I G_J]^T [G_I G_J] (32 x 32) by DMMA straight from global memory (L2-resident matrix):
//      four column fragments per step of four rows feed the ten sub-tiles on or below the diagonal;
//   2. plane rotations on M in shared memory (one warp, 16 disjoint rotations per round, angles from M alone:
//      rotating columns p, q of G is the congruence J^T M J on its Gram matrix, so these ARE the plane rotations of
//      the one-sided method, applied to M instead of G), accumulated in W.  M: off-diagonal elements FP32, diagonal
//      FP64 (see bj_visit).  In the first tournament round of a sweep a visit runs all 496 pairs of its 32 columns
//      (31 rounds; every block is in exactly one pair of that round, so pairs inside a block are covered once per
//      sweep), afterwards only the 256 cross pairs (16 rounds);
//   3. [G_I G_J] <- [G_I G_J] W by DMMA, one 8-row strip at a time, in place, B fragments of W from shared memory.
// One warp owns a block pair; the pairs of a tournament round are disjoint, so the warps of a CTA work on different
// pairs of the same submatrix.  Rounds are not separated by CTA barriers: every block counts the rounds it has been
// through and a warp waits for its two blocks alone.  Two CTAs (two submatrices) per SM.
// A visit whose Gram matrix is already diagonal to the tolerance changes nothing; a sweep of such visits ends it.
#include "common.cuh"

namespace smb {

constexpr int BJ_B = 16;       // columns per block
constexpr int BJ_WARPS = 7;    // warps per CTA
constexpr int BJ_LDM = 33;     // leading dimension of the 32 x 32 matrices in shared memory (conflict-free both ways)
constexpr int BJ_LDW = 36;     // leading dimension of W (FP64): = 4 mod 16, so that the column rotations AND the reads
                               // of its B fragments in the update are free of bank conflicts
constexpr int BJ_PERW = 32 * BJ_LDW + 32 + 32 + 16 + 16 + 32 * BJ_LDM / 2 + 1;  // doubles of shared memory per warp
constexpr int BJ_MAXN = 1024;  // blocks per submatrix with barrier-free rounds (n <= 16384)
constexpr int BJ_INNER = 1;    // passes over a visit's pair schedule (the outer sweeps finish the job)

struct BjArgs {
    const int32_t* sub_dim;
    const int32_t* ldv;
    const int64_t* ws_off;
    double* G;
    const double* sigma;
    const int32_t* order;
    int32_t* counter;
    int32_t* sweeps;
    int32_t* eflag;
    const int32_t* grp_ptr;
    const int32_t* grp_cols;
    const int32_t* gen_off;
    const int32_t* blk_size;
    const int64_t* eig_ptr;
    double* lam;
    double* w;
    int ngroups, max_sweeps;
};

__device__ __forceinline__ void bj_dmma(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

// Two-sided rotation zeroing M_pq: t = tan(theta) root of t^2 + 2 zeta t - 1, zeta = (M_qq - M_pp) / (2 M_pq).
// The tangent is formed in FP32 (relative error 1e-7: the pair is then orthogonal to 1e-7 of its former
// inner product, which the next visit removes) and the cosine by an FP32 seed and two FP64 Newton steps, so that
// c^2 + s^2 = 1 to FP64 rounding and W stays orthogonal -- ~25 instructions instead of FP64 division, square root
// and reciprocal square root on the critical path of every round.
__device__ __forceinline__ void bj_rotation(double app, double aqq, double apq, double& c, double& s, double& t) {
    const float zf = __fdividef((float)(aqq - app), 2.0f * (float)apq);
    const float az = fabsf(zf);
    float tf = az < 1e15f ? __frcp_rn(az + __fsqrt_rn(fmaf(az, az, 1.0f))) : __fdividef(0.5f, az);
    tf = zf >= 0.0f ? tf : -tf;
    t = (double)tf;
    const double x = fma(t, t, 1.0);
    double y = (double)rsqrtf((float)x);
    y = y * fma(-0.5 * x, y * y, 1.5);
    y = y * fma(-0.5 * x, y * y, 1.5);
    c = y;
    s = y * t;
}

// One visit of the block pair (I, J) of the n x n matrix Gm (column-major, column stride ld) by one warp.
// W (FP64), M (FP32: off-diagonal elements of the Gram matrix), dg (FP64: its diagonal): this warp's 32 x 33 shared
// arrays; cs: 32 doubles, pq: 32 ints of shared scratch.  Returns 1 if it rotated.
// Only the ANGLES come from M, so its off-diagonal elements need relative accuracy only (FP32: the rotated pair is
// orthogonal to 1e-7 of its former inner product, removed by the next visit, whose Gram matrix is formed afresh in
// FP64); the diagonal stays FP64 because zeta = (M_qq - M_pp) / (2 M_pq) takes a difference of nearly equal numbers
// for close eigenvalues.  W and the columns of G never see FP32.
__device__ int bj_visit(double* __restrict__ Gm, int n, int ld, int I, int J, int nblk, float* __restrict__ M,
                        double* __restrict__ dg, double* __restrict__ W, double* __restrict__ cs,
                        int* __restrict__ pq, double tol2, int lane, bool full) {
    float* csf = reinterpret_cast<float*>(pq + 32);  // [32] (c, s) once more as floats, for the update of M
    const int lr = lane >> 2, lk = lane & 3;
    // global column of slot k of the pair (or -1): slots 0..15 block I, 16..31 block J
    auto colof = [&](int k) {
        const int blk = k < BJ_B ? I : J;
        const int c = blk * BJ_B + (k & (BJ_B - 1));
        return (blk < nblk && c < n) ? c : -1;
    };
    // ---- 1. Gram matrix: f[a] = G[4 s + lk][col(8 a + lr)] is the A fragment of sub-tile row a and the B fragment of
    //         sub-tile column a at once
    int colf[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) colf[a] = colof(8 * a + lr);
    double acc[10][2];
#pragma unroll
    for (int e = 0; e < 10; ++e) acc[e][0] = acc[e][1] = 0.0;
    const int ksteps = ld >> 2;  // rows n .. ld - 1 of G are zero
#pragma unroll 4
    for (int s = 0; s < ksteps; ++s) {
        double f[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) f[a] = colf[a] >= 0 ? Gm[(size_t)colf[a] * ld + 4 * s + lk] : 0.0;
        int e = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b <= a; ++b, ++e) bj_dmma(acc[e], f[a], f[b]);
    }
    {   // accumulator (row lr, columns 2 lk, 2 lk + 1 of sub-tile (a, b)) -> M and its mirror, diagonal -> dg
        int e = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b <= a; ++b, ++e) {
                const int r = 8 * a + lr, c0 = 8 * b + 2 * lk;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (r == c0 + h) dg[r] = acc[e][h];
                    else { M[r * BJ_LDM + c0 + h] = (float)acc[e][h]; M[(c0 + h) * BJ_LDM + r] = (float)acc[e][h]; }
                }
            }
    }
    __syncwarp();
    // largest |M_pq| / sqrt(M_pp M_qq) of the pair (squared): nothing to do if it is below the tolerance; one inner
    // sweep is enough when it is small already (the sweep squares it)
    double rmax2 = 0.0;
    {
        const double dl = dg[lane];
        const int kend = full ? lane : (lane >= 16 ? 16 : 0);  // cross-only visit: the elements (J slot, I slot) alone
        for (int k = 0; k < kend; ++k) {
            const double v = (double)M[lane * BJ_LDM + k], dk = dg[k];
            const double den = dl * dk;
            if (den > 0.0) rmax2 = fmax(rmax2, v * v / den);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rmax2 = fmax(rmax2, __shfl_xor_sync(0xffffffffu, rmax2, o));
    }
    if (!(rmax2 > tol2)) return 0;
    const int inner = rmax2 > 1e-12 ? BJ_INNER : 1;
    for (int k = 0; k < 32; ++k) W[lane * BJ_LDW + k] = (k == lane) ? 1.0 : 0.0;
    __syncwarp();
    // ---- 2. cyclic Jacobi on M (32 x 32), W accumulates the rotations
    int rotated_any = 0;
    for (int sw = 0; sw < inner; ++sw) {
        int rotated_sw = 0;
        for (int rd = 0; rd < (full ? 31 : 16); ++rd) {
            // pair of lane k < 16: round-robin tournament of 32 players
            int p = 0, q = 0;
            double c = 1.0, s = 0.0;
            if (lane < 16) {
                if (full) {
                    p = lane == 0 ? 31 : (rd + lane) % 31;
                    q = lane == 0 ? rd : (rd - lane + 31) % 31;
                } else {  // the 256 cross pairs (slot of I, slot of J) in 16 rounds
                    p = lane;
                    q = 16 + ((lane + rd) & 15);
                }
                const double app = dg[p], aqq = dg[q], apq = (double)M[p * BJ_LDM + q];
                if (apq * apq > tol2 * app * aqq) {
                    double t;
                    bj_rotation(app, aqq, apq, c, s, t);
                    dg[p] = app - t * apq;  // the rotated diagonal in closed form
                    dg[q] = aqq + t * apq;
                }
                cs[2 * lane] = c;
                cs[2 * lane + 1] = s;
                csf[2 * lane] = (float)c;
                csf[2 * lane + 1] = (float)s;
                pq[2 * lane] = p;
                pq[2 * lane + 1] = q;
            }
            const unsigned any = __ballot_sync(0xffffffffu, s != 0.0);
            __syncwarp();
            if (any) {
                rotated_sw = 1;
                // lane = (pair k, half h).  M <- J^T M J in one pass: the 2 x 2 block (rows of pair k, columns of
                // pair k') becomes R_k^T B R_k', and each block belongs to exactly one lane (k, k' in its half), so M
                // is read once and written once per round with no barrier in between -- shared-memory bandwidth is
                // what bounds this phase (8-byte accesses, 128 B/clk/SM).  W <- W J: columns of pair k, 16 rows.
                const int k = lane & 15, hh = lane >> 4, h16 = hh * 16;
                const double ck = cs[2 * k], sk = cs[2 * k + 1];
                const int pk = pq[2 * k], qk = pq[2 * k + 1];
                const float ckf = csf[2 * k], skf = csf[2 * k + 1];
                float b00[8], b01[8], b10[8], b11[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int p2 = pq[2 * (8 * hh + j)], q2 = pq[2 * (8 * hh + j) + 1];
                    b00[j] = M[pk * BJ_LDM + p2];
                    b01[j] = M[pk * BJ_LDM + q2];
                    b10[j] = M[qk * BJ_LDM + p2];
                    b11[j] = M[qk * BJ_LDM + q2];
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k2 = 8 * hh + j;
                    const float c2 = csf[2 * k2], s2 = csf[2 * k2 + 1];
                    if (skf == 0.f && s2 == 0.f) continue;
                    const int p2 = pq[2 * k2], q2 = pq[2 * k2 + 1];
                    if (k2 == k) {  // the pair's own block: diagonal done in closed form, its off-diagonal element vanishes
                        M[pk * BJ_LDM + qk] = 0.f;
                        M[qk * BJ_LDM + pk] = 0.f;
                        continue;
                    }
                    const float t00 = c2 * b00[j] - s2 * b01[j], t01 = s2 * b00[j] + c2 * b01[j];
                    const float t10 = c2 * b10[j] - s2 * b11[j], t11 = s2 * b10[j] + c2 * b11[j];
                    M[pk * BJ_LDM + p2] = ckf * t00 - skf * t10;
                    M[pk * BJ_LDM + q2] = ckf * t01 - skf * t11;
                    M[qk * BJ_LDM + p2] = skf * t00 + ckf * t10;
                    M[qk * BJ_LDM + q2] = skf * t01 + ckf * t11;
                }
                if (sk != 0.0) {  // columns p, q of W
                    double x[16], y[16];
#pragma unroll
                    for (int r = 0; r < 16; ++r) { x[r] = W[(h16 + r) * BJ_LDW + pk]; y[r] = W[(h16 + r) * BJ_LDW + qk]; }
#pragma unroll
                    for (int r = 0; r < 16; ++r) {
                        W[(h16 + r) * BJ_LDW + pk] = ck * x[r] - sk * y[r];
                        W[(h16 + r) * BJ_LDW + qk] = sk * x[r] + ck * y[r];
                    }
                }
            }
            __syncwarp();
        }
        rotated_any |= rotated_sw;
        if (!rotated_sw) break;
    }
    if (!rotated_any) return 0;
    // ---- 3. [G_I G_J] <- [G_I G_J] W by DMMA, 8-row strips in place.  The B fragments of W (k-step t = rows
    // 4 t .. 4 t + 3, sub-tile column d) are read from shared memory for every strip (conflict-free with BJ_LDW):
    // holding all 32 of them in registers costs 64 registers and the second CTA per SM.
    int cola[8], colc[4][2];
#pragma unroll
    for (int t = 0; t < 8; ++t) cola[t] = colof(4 * t + lk);
#pragma unroll
    for (int d = 0; d < 4; ++d) { colc[d][0] = colof(8 * d + 2 * lk); colc[d][1] = colof(8 * d + 2 * lk + 1); }
    const unsigned wbase = (unsigned)__cvta_generic_to_shared(W + lk * BJ_LDW + lr);
    const int strips = ld >> 3;
#pragma unroll 2
    for (int rs = 0; rs < strips; ++rs) {
        const int row = 8 * rs + lr;
        double af[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) af[t] = cola[t] >= 0 ? Gm[(size_t)cola[t] * ld + row] : 0.0;
        double c4[4][2];
#pragma unroll
        for (int d = 0; d < 4; ++d) c4[d][0] = c4[d][1] = 0.0;
#pragma unroll
        for (int t = 0; t < 8; ++t)
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                double wv;  // volatile: keeps the loads inside the strip loop
                asm volatile("ld.shared.f64 %0, [%1];" : "=d"(wv) : "r"(wbase + (unsigned)((4 * t * BJ_LDW + 8 * d) * 8)));
                bj_dmma(c4[d], af[t], wv);
            }
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            if (colc[d][0] >= 0) Gm[(size_t)colc[d][0] * ld + row] = c4[d][0];
            if (colc[d][1] >= 0) Gm[(size_t)colc[d][1] * ld + row] = c4[d][1];
        }
    }
    return 1;
}

__global__ void __launch_bounds__(BJ_WARPS * 32, 2) k_eig_bjacobi(const BjArgs A) {
    extern __shared__ __align__(16) double bsm[];  // per warp: W[32 x 33], dg[32], cs[32], pq[32 ints], M[32 x 33 floats]
    __shared__ int s_next, s_rot;
    __shared__ int s_ver[BJ_MAXN];
    __shared__ int s_genrow[1024];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double* W = bsm + (size_t)wid * BJ_PERW;          // [32 x 33] doubles
    double* dg = W + 32 * BJ_LDW;                       // [32] diagonal of the Gram matrix
    double* cs = dg + 32;                               // [32] (c, s) of the 16 pairs of a round
    int* pq = reinterpret_cast<int*>(cs + 32);          // [32] (p, q) of the 16 pairs
    float* M = reinterpret_cast<float*>(pq + 64);       // [32 x 33] floats (pq + 32: the float copies of (c, s))
    for (;;) {
        if (threadIdx.x == 0) s_next = atomicAdd(A.counter, 1);
        __syncthreads();
        const int it = s_next;
        __syncthreads();
        if (it >= A.ngroups) return;
        const int i = A.order[it];
        const int n = A.sub_dim[i], ld = A.ldv[i];
        double* Gm = A.G + A.ws_off[i];
        const double tol = 1e-15 * sqrt((double)max(n, 1));
        const double tol2 = tol * tol;
        const int nblk = (n + BJ_B - 1) / BJ_B;
        const int N = nblk + (nblk & 1);  // >= 2: a single block is paired with an empty one
        int sweep = 0, converged = n <= 1 ? 1 : 0;
        // Rounds are NOT separated by CTA barriers: a visit of (I, J) in round R only needs the round R - 1 visits
        // of I and of J, so every block carries the number of rounds it has been through (s_ver) and a warp waits
        // for its two blocks alone; warps whose visits end early (Gram matrix already diagonal) run ahead.  Every
        // block is visited exactly once per round, rounds are processed in order by every warp: no cycle of waits.
        const bool flow = N <= BJ_MAXN;
        for (int b = threadIdx.x; b < N && flow; b += blockDim.x) s_ver[b] = 0;
        __syncthreads();
        int R = 0;
        for (; sweep < A.max_sweeps && !converged; ++sweep) {
            if (threadIdx.x == 0) s_rot = 0;
            __syncthreads();
            int my_rot = 0;
            for (int r = 0; r < N - 1; ++r, ++R) {
                for (int q = wid; q < N / 2; q += BJ_WARPS) {
                    int I = (q == 0) ? N - 1 : (r + q) % (N - 1);
                    int J = (q == 0) ? r : (r - q + (N - 1)) % (N - 1);
                    if (I > J) { const int t = I; I = J; J = t; }
                    if (flow) {
                        if (lane == 0) {
                            volatile int* v = s_ver;
                            while (v[I] < R || v[J] < R) {}
                        }
                        __syncwarp();
                        __threadfence_block();
                    }
                    if (I < nblk) my_rot |= bj_visit(Gm, n, ld, I, J, nblk, M, dg, W, cs, pq, tol2, lane, r == 0);
                    if (flow) {
                        __threadfence_block();
                        __syncwarp();
                        if (lane == 0) {
                            volatile int* v = s_ver;
                            v[I] = R + 1;
                            v[J] = R + 1;
                        }
                    }
                }
                if (!flow) __syncthreads();  // the next round regroups the columns
            }
            if (lane == 0 && my_rot) atomicOr(&s_rot, 1);
            __syncthreads();
            if (s_rot == 0) converged = 1;
            __syncthreads();
        }
        if (threadIdx.x == 0) { A.sweeps[i] = sweep; A.eflag[i] = converged ? 0 : 1; }
        // ---- eigenvalues, normalised eigenvectors (in place), weights of Algorithm 1 (L270, L278)
        int gw = 0;
        for (int gc = A.grp_ptr[i]; gc < A.grp_ptr[i + 1]; ++gc) {
            const int c = A.grp_cols[gc], o = A.gen_off[c], b = A.blk_size[c];
            for (int e = threadIdx.x; e < b; e += blockDim.x)
                if (gw + e < 1024) s_genrow[gw + e] = o + e;
            gw += b;
        }
        __syncthreads();
        const double sig = A.sigma[i];
        const int64_t ep = A.eig_ptr[i];
        for (int l = wid; l < n; l += BJ_WARPS) {
            double* col = Gm + (size_t)l * ld;
            double s2 = 0.0;
            for (int r = lane; r < n; r += 32) s2 = fma(col[r], col[r], s2);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            const double nrm = sqrt(s2), inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
            for (int r = lane; r < n; r += 32) col[r] *= inv;
            __syncwarp();
            double wl = 0.0;
            if (gw <= 1024) {
                for (int e = lane; e < gw; e += 32) { const double qv = col[s_genrow[e]]; wl = fma(qv, qv, wl); }
            } else {
                for (int gc = A.grp_ptr[i]; gc < A.grp_ptr[i + 1]; ++gc) {
                    const int c = A.grp_cols[gc], o = A.gen_off[c], b = A.blk_size[c];
                    for (int e = lane; e < b; e += 32) { const double qv = col[o + e]; wl = fma(qv, qv, wl); }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) wl += __shfl_xor_sync(0xffffffffu, wl, o);
            if (lane == 0) { A.lam[ep + l] = nrm - sig; A.w[ep + l] = wl; }
        }
        __syncthreads();
    }
}

sm_status_t launch_eig_bjacobi(sm_plan* p, double* G, cudaStream_t st) {
    const int ng = p->ngroups;
    constexpr size_t smem = (size_t)BJ_WARPS * BJ_PERW * sizeof(double);
    if (!p->eig_battr_set) {
        SM_CUDA(cudaFuncSetAttribute(k_eig_bjacobi, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        p->eig_battr_set = 1;
    }
    BjArgs a;
    a.sub_dim = p->d_sub_dim; a.ldv = p->d_ld; a.ws_off = p->d_ws_off; a.G = G; a.sigma = p->d_eig_sigma;
    a.order = p->d_eig_order; a.counter = p->d_eig_state + 2 * ng; a.sweeps = p->d_eig_state; a.eflag = p->d_eig_state + ng;
    a.grp_ptr = p->d_grp_ptr; a.grp_cols = p->d_grp_cols; a.gen_off = p->d_gen_off; a.blk_size = p->d_blk_size;
    a.eig_ptr = p->d_eig_ptr; a.lam = p->d_eig_lam; a.w = p->d_eig_w;
    a.ngroups = ng; a.max_sweeps = 30;
    k_eig_bjacobi<<<std::min(ng, 2 * p->num_sms), BJ_WARPS * 32, smem, st>>>(a);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

}  // namespace smb
