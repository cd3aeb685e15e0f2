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
// grid = (ngroups, split); one CTA (or `split` CTAs sharing the dense rows) per submatrix, NO matrix
// data staged in shared memory.  Per CTA, in shared memory:
//   * posmap[p] for every dense row p of a_i: its member t, the row el inside the block, the block
//     height (p >= n: the "no member" column of the block map),
//   * the BLOCK MAP of a chunk of member columns:  bmap[tc][t] = offset of the stored block
//     (S_i[t], S_i[tc]) inside the values of block column S_i[tc] (16 bits when every block column
//     holds fewer than 65535 values), or all-ones if it is not stored (reading A4: zero fill).
//     LIST = true: filled from the plan's gather list -- the (t, offset) pairs of every submatrix
//     column, listed once per plan by k_glist (pattern only).  LIST = false (32-bit entries): built
//     in place by walking the stored block columns (coalesced reads of rowidx / val_off, one probe
//     of a hash table  block row -> member  per stored block; rows outside S_i are dropped).
// Sweep: dense column q of a_i is row q of the symmetric X; one warp per row, lanes two positions
// at a time in groups of four 64-wide steps (warp-uniform trip count): posmap (one 16-byte read),
// two block-map reads, predicated 8-byte loads of the stored values straight from global memory
// (L2-resident: every value is used by ~|S_i| submatrices), mu subtracted on the diagonal
// (Eq.(16)), one coalesced 16-byte store into the k8-panel workspace, abs-sums for the Gershgorin
// bound s_i = max_q sum_p |a_pq|, and squares for a rigorous LOWER bound of the spectral radius (the mean
// of ||a e_q||_2^2 over the columns a warp sweeps <= max_q ||a e_q||_2^2 <= rho^2; no per-column reduction
// needed): the estimated interlacing cap is never taken below it, reading A8; stored in gersh[ngroups + g].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned gather_hash(int key, int shift) {
    return ((unsigned)key * 2654435761u) >> shift;
}

struct GatherArgs {
    const int64_t* colptr;
    const int32_t* rowidx;
    const int64_t* val_off;
    const double* vals;
    const int64_t* sub_ptr;
    const int32_t* sub_blocks;
    const int32_t* sub_off;
    const int32_t* sub_dim;
    const int32_t* ldv;
    const int64_t* ws_off;
    double* X;
    unsigned long long* gersh;
    double mu;
    int tile_ld, msb, mpad, mc, hash_size, hash_shift;
    const int64_t* gl_ptr;   // LIST: per (submatrix, member column) extent in gl
    const uint32_t* gl;      // LIST: member index t << 16 | value offset of block (S_i[t], S_i[tc]) in its column
};

template <typename MapT, bool LIST>
__global__ void __launch_bounds__(256) k_gather(const GatherArgs A) {
    constexpr MapT NONE = (MapT)~(MapT)0;  // block (S_i[t], S_i[tc]) not stored
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int g = blockIdx.x;
    const int64_t sp = A.sub_ptr[g];
    const int m = (int)(A.sub_ptr[g + 1] - sp);
    const int n = A.sub_dim[g], ld = A.ldv[g];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int tile_ld = A.tile_ld, msb = A.msb, mpad = A.mpad, mc = A.mc;
    // shared-memory carve-up
    int64_t* mVb = reinterpret_cast<int64_t*>(smem_raw);                        // [msb] first value offset of the member's column
    uint2* posmap = reinterpret_cast<uint2*>(mVb + msb);                        // [tile_ld] member | (el | height << 16)
    MapT* bmap = reinterpret_cast<MapT*>(posmap + tile_ld);                     // [mc][mpad]
    int32_t* hk = reinterpret_cast<int32_t*>(bmap + (size_t)mc * mpad);                                    // [hash_size] keys
    int32_t* hv = hk + A.hash_size;                                             // [hash_size] member index
    int32_t* mSo = hv + A.hash_size;                                            // [msb + 1] element offsets
    int32_t* mKey = mSo + msb + 2;                                              // [msb] global block index of the member
    if (!LIST)
        for (int h = threadIdx.x; h < A.hash_size; h += blockDim.x) hk[h] = -1;
    for (int t = threadIdx.x; t < m; t += blockDim.x) mSo[t] = A.sub_off[sp + t];
    if (threadIdx.x == 0) mSo[m] = n;
    __syncthreads();
    const unsigned hmask = (unsigned)A.hash_size - 1u;
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        const int key = A.sub_blocks[sp + t];
        mKey[t] = key;
        mVb[t] = A.val_off[A.colptr[key]];
        if (!LIST) {
            unsigned h = gather_hash(key, A.hash_shift);
            while (atomicCAS(&hk[h], -1, key) != -1) h = (h + 1) & hmask;
            hv[h] = t;
        }
        const int so = mSo[t], br = mSo[t + 1] - so;
        for (int el = 0; el < br; ++el) posmap[so + el] = make_uint2((unsigned)t, (unsigned)el | ((unsigned)br << 16));
    }
    for (int p = n + threadIdx.x; p < tile_ld; p += blockDim.x) posmap[p] = make_uint2((unsigned)m, 1u << 16);
    double* Xg = A.X + A.ws_off[g];
    double cmax = 0.0, ssum = 0.0;
    int swept = 0;
    const int gw = blockIdx.y * nw + wid, gstride = nw * gridDim.y;

    for (int c0 = 0; c0 < m; c0 += mc) {
        const int c1 = min(m, c0 + mc);
        __syncthreads();  // tables ready / previous chunk swept
        for (int e = threadIdx.x; e < (c1 - c0) * mpad; e += blockDim.x) bmap[e] = NONE;
        __syncthreads();
        // block map of member columns c0..c1-1: one warp per column, lanes over its stored blocks
        for (int tc = c0 + wid; tc < c1; tc += nw) {
            MapT* row = bmap + (size_t)(tc - c0) * mpad;
            if (LIST) {  // the pairs (member, value offset) were listed when the plan first gathered
                const int64_t e1 = A.gl_ptr[sp + tc + 1];
                for (int64_t e = A.gl_ptr[sp + tc] + lane; e < e1; e += 32) {
                    const uint32_t v = __ldcs(A.gl + e);  // read once per gather: do not displace the values in L2
                    row[v >> 16] = (MapT)(v & 0xffffu);
                }
                continue;
            }
            const int key = mKey[tc];
            const int64_t p0 = A.colptr[key], p1 = A.colptr[key + 1], vb = mVb[tc];
            for (int64_t j = p0 + lane; j < p1; j += 32) {
                const int r = __ldg(A.rowidx + j);
                const int rel = (int)(__ldg(A.val_off + j) - vb);
                unsigned h = gather_hash(r, A.hash_shift);
                for (;;) {
                    const int k = hk[h];
                    if (k == r) { row[hv[h]] = (MapT)rel; break; }
                    if (k < 0) break;
                    h = (h + 1) & hmask;
                }
            }
        }
        __syncthreads();
        // sweep the dense rows of this chunk's members
        const int q_begin = mSo[c0], q_end = mSo[c1];
        for (int q = q_begin + gw; q < q_end; q += gstride) {
            const uint2 me = posmap[q];
            const int tc = (int)me.x, qq = (int)(me.y & 0xffffu);
            const MapT* row = bmap + (size_t)(tc - c0) * mpad;
            const double* vcol = A.vals + mVb[tc];
            const int t0 = q & ~63;
            const unsigned rows_t = (unsigned)min(64, ld - t0);
            unsigned xo = (unsigned)t0 * (unsigned)ld + (unsigned)(q & 63) * 8u + (unsigned)(lane >> 2) * rows_t * 8u +
                          2u * (lane & 3);
            const unsigned xstep = rows_t * 64u;
            double asum = 0.0;
            ++swept;
            // warp-uniform trip count (groups of four 64-wide steps, predicated inside): one loop body,
            // no divergent remainder loop; all look-ups and loads of a group are in flight together
            for (int base = 0, p0 = 2 * lane; base < ld; base += 256, p0 += 256, xo += 4 * xstep) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int p = p0 + 64 * u;
                    if (p < ld) {
                        const uint4 pm = *reinterpret_cast<const uint4*>(posmap + p);
                        const MapT r0 = row[pm.x], r1 = row[pm.z];
                        double2 v = make_double2(0.0, 0.0);
                        if (r0 != NONE) v.x = __ldg(vcol + (int)r0 + (int)(pm.y & 0xffffu) + qq * (int)(pm.y >> 16));
                        if (r1 != NONE) v.y = __ldg(vcol + (int)r1 + (int)(pm.w & 0xffffu) + qq * (int)(pm.w >> 16));
                        if (p == q) v.x -= A.mu;
                        if (p + 1 == q) v.y -= A.mu;
                        asum += fabs(v.x) + fabs(v.y);
                        ssum = fma(v.x, v.x, fma(v.y, v.y, ssum));
                        __stcs(reinterpret_cast<double2*>(Xg + xo + u * xstep), v);  // streaming: the workspace is far larger than L2
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) asum += __shfl_xor_sync(0xffffffffu, asum, o);
            cmax = fmax(cmax, asum);
        }
    }
    // zero padding columns n..ld-1 (first CTA of the submatrix)
    if (blockIdx.y == 0) {
        for (int qq = n + wid; qq < ld; qq += nw) {
            for (int p = 2 * lane; p < ld; p += 64)
                *reinterpret_cast<double2*>(Xg + panel_off(qq, p, ld)) = make_double2(0.0, 0.0);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ssum += __shfl_xor_sync(0xffffffffu, ssum, o);
    if (lane == 0 && cmax > 0.0) {
        atomicMax(A.gersh + g, (unsigned long long)__double_as_longlong(cmax));
        atomicMax(A.gersh + gridDim.x + g, (unsigned long long)__double_as_longlong(ssum / (double)max(swept, 1)));
    }
}

// Gather list (pattern only, built by the first gather of a plan when 16-bit entries suffice): for every
// submatrix i and member column tc the pairs (t, value offset) of the stored blocks (S_i[t], S_i[tc]).
// One CTA per submatrix, hash table of S_i in shared memory, one warp per member column; FILL = false
// counts, FILL = true writes (order inside a column: ascending stored position, by ballot ranks).
template <bool FILL>
__global__ void __launch_bounds__(256)
k_glist(const int64_t* __restrict__ colptr, const int32_t* __restrict__ rowidx, const int64_t* __restrict__ val_off,
        const int64_t* __restrict__ sub_ptr, const int32_t* __restrict__ sub_blocks, int hash_size, int hash_shift,
        int32_t* __restrict__ cnt, const int64_t* __restrict__ gl_ptr, uint32_t* __restrict__ gl) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int32_t* hk = reinterpret_cast<int32_t*>(smem_raw);
    int32_t* hv = hk + hash_size;
    const int g = blockIdx.x;
    const int64_t sp = sub_ptr[g];
    const int m = (int)(sub_ptr[g + 1] - sp);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int h = threadIdx.x; h < hash_size; h += blockDim.x) hk[h] = -1;
    __syncthreads();
    const unsigned hmask = (unsigned)hash_size - 1u;
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        const int key = sub_blocks[sp + t];
        unsigned h = gather_hash(key, hash_shift);
        while (atomicCAS(&hk[h], -1, key) != -1) h = (h + 1) & hmask;
        hv[h] = t;
    }
    __syncthreads();
    for (int tc = wid; tc < m; tc += nw) {
        const int key = sub_blocks[sp + tc];
        const int64_t p0 = colptr[key], p1 = colptr[key + 1], vb = val_off[p0];
        int64_t out = FILL ? gl_ptr[sp + tc] : 0;
        int total = 0;
        for (int64_t j0 = p0; j0 < p1; j0 += 32) {
            const int64_t j = j0 + lane;
            int t = -1;
            if (j < p1) {
                const int r = __ldg(rowidx + j);
                unsigned h = gather_hash(r, hash_shift);
                for (;;) {
                    const int k = hk[h];
                    if (k == r) { t = hv[h]; break; }
                    if (k < 0) break;
                    h = (h + 1) & hmask;
                }
            }
            const unsigned mask = __ballot_sync(0xffffffffu, t >= 0);
            if (FILL && t >= 0)
                gl[out + __popc(mask & ((1u << lane) - 1u))] = ((uint32_t)t << 16) | (uint32_t)(__ldg(val_off + j) - vb);
            out += __popc(mask);
            total += __popc(mask);
        }
        if (!FILL && lane == 0) cnt[sp + tc] = total;
    }
}

static sm_status_t build_gather_list(sm_plan* p, cudaStream_t st) {
    const int64_t tot = p->info.sum_sub_blocks;
    const size_t hbytes = (size_t)p->gather_hash_size * 8;
    if (hbytes > 48 * 1024) {
        SM_CUDA(cudaFuncSetAttribute(k_glist<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hbytes));
        SM_CUDA(cudaFuncSetAttribute(k_glist<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hbytes));
    }
    DevTmp cnt_tmp;
    SM_CUDA(cudaMalloc(&cnt_tmp.p, (size_t)std::max<int64_t>(tot, 1) * 4));
    int32_t* d_cnt = (int32_t*)cnt_tmp.p;
    k_glist<false><<<p->ngroups, 256, hbytes, st>>>(p->d_colptr, p->d_rowidx, p->d_val_off, p->d_sub_ptr, p->d_sub_blocks,
                                                    p->gather_hash_size, p->gather_hash_shift, d_cnt, nullptr, nullptr);
    // extents by a device prefix sum; the host only learns the total (8 bytes) to size the list
    SM_CUDA(cudaMalloc((void**)&p->d_gl_ptr, ((size_t)tot + 1) * 8));
    sm_status_t s = launch_excl_scan(d_cnt, tot, p->d_gl_ptr, st);
    if (s) return s;
    int64_t n_entries = 0;
    SM_CUDA(cudaMemcpyAsync(&n_entries, p->d_gl_ptr + tot, 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    SM_CUDA(cudaMalloc((void**)&p->d_gl, (size_t)std::max<int64_t>(n_entries, 1) * 4));
    k_glist<true><<<p->ngroups, 256, hbytes, st>>>(p->d_colptr, p->d_rowidx, p->d_val_off, p->d_sub_ptr, p->d_sub_blocks,
                                                   p->gather_hash_size, p->gather_hash_shift, nullptr, p->d_gl_ptr, p->d_gl);
    p->launches += 3;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

sm_status_t launch_gather(sm_plan* p, const double* vals, double mu, double* X, cudaStream_t st) {
    if (p->ngroups == 0) return SM_OK;
    const bool list = p->gather_map16 && p->gather_msb < 65536 && !p->gather_no_list;
    if (list && !p->d_gl) {
        sm_status_t s = build_gather_list(p, st);
        if (s) return s;
    }
    SM_CUDA(cudaMemsetAsync(p->d_gersh, 0, (size_t)p->ngroups * 16, st));  // Gershgorin bounds + squared column norms
    if (p->gather_smem > 48 * 1024) {
        SM_CUDA(cudaFuncSetAttribute(k_gather<uint16_t, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->gather_smem));
        SM_CUDA(cudaFuncSetAttribute(k_gather<uint16_t, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->gather_smem));
        SM_CUDA(cudaFuncSetAttribute(k_gather<uint32_t, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->gather_smem));
    }
    GatherArgs a;
    a.colptr = p->d_colptr; a.rowidx = p->d_rowidx; a.val_off = p->d_val_off; a.vals = vals;
    a.sub_ptr = p->d_sub_ptr; a.sub_blocks = p->d_sub_blocks; a.sub_off = p->d_sub_off; a.sub_dim = p->d_sub_dim;
    a.ldv = p->d_ld; a.ws_off = p->d_ws_off; a.X = X; a.gersh = p->d_gersh; a.mu = mu;
    a.tile_ld = p->gather_tile_ld; a.msb = p->gather_msb; a.mpad = p->gather_mpad; a.mc = p->gather_mc;
    a.hash_size = p->gather_hash_size; a.hash_shift = p->gather_hash_shift;
    a.gl_ptr = p->d_gl_ptr; a.gl = p->d_gl;
    const dim3 grid(p->ngroups, p->gather_split);
    if (list) k_gather<uint16_t, true><<<grid, p->gather_warps * 32, p->gather_smem, st>>>(a);
    else if (p->gather_map16) k_gather<uint16_t, false><<<grid, p->gather_warps * 32, p->gather_smem, st>>>(a);
    else k_gather<uint32_t, false><<<grid, p->gather_warps * 32, p->gather_smem, st>>>(a);
    p->launches++;
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// ---------------------------------------------------------------------------------------------
// Scatter (PAPER.md L127 step 3 + Eq.(16) inner factor).  Element (el,q) of result block (r,c) is
// X_i[gen_off(c) + q, blk_loc(r) + el] of c's group i (X symmetric, so the read walks a row).
// Where each stored value comes from depends on the pattern only, so the first scatter of a plan
// builds a SOURCE MAP: one 32-bit entry per stored value = its offset inside the submatrix's
// workspace matrix (k8-panel layout) | "diagonal element" in bit 31.  k_scatter_map_build walks
// the block columns once (one warp per block column: 32 packed block records at a time, prefix
// sums of their sizes, shuffle binary search of an element's block); k_scatter is then a plain
// parallel sweep (one warp per block column and chunk of 1024 values), any block size:
//     D = 1/2 (delta - xs * X),  xs = 1/s_i if the submatrix stopped at iteration 0 (the buffer
// then still holds the unscaled a_i - mu I), else 1.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_scatter_map_build(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                    const int64_t* __restrict__ val_off, const int32_t* __restrict__ col_grp,
                    const int32_t* __restrict__ gen_off, const uint32_t* __restrict__ blk_pack,
                    const int32_t* __restrict__ ldv, uint32_t* __restrict__ src_map, int4* __restrict__ col_rec) {
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= nb) return;
    const int lane = threadIdx.x & 31;
    const int g = col_grp[c];
    if (g < 0) {  // block column of another shard: an empty record, k_scatter skips it
        if (lane == 0) col_rec[c] = make_int4(0, 0, 0, -1);
        return;
    }
    const int bc = blk_size[c];
    const int64_t p0 = colptr[c];
    if (lane == 0) {  // column record of k_scatter: first value, value count, group -- one 16-byte load
        const int64_t v0 = val_off[p0];
        col_rec[c] = make_int4((int)(v0 & 0xffffffffll), (int)(v0 >> 32), (int)(val_off[colptr[c + 1]] - v0), g);
    }
    const int nblk = (int)(colptr[c + 1] - p0);
    const int ld = ldv[g];
    const int go = gen_off[c];
    uint32_t* o = src_map + val_off[p0];
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
                o[e] = (uint32_t)panel_off(go + q, loc + el, ld) | ((loc + el == go + q) ? 0x80000000u : 0u);
            }
        }
        o += total;
    }
}

constexpr int SCATTER_THREADS = 256, SCATTER_CHUNK = 1024;  // one warp per (block column, chunk of values)
constexpr int SCATTER_U = 12;  // values per lane in flight (384 per warp: a typical SZV block column in one pass)

__global__ void __launch_bounds__(SCATTER_THREADS)
k_scatter(int nb, const int4* __restrict__ col_rec, const int64_t* __restrict__ ws_off,
          const int32_t* __restrict__ done_iter, const unsigned long long* __restrict__ gersh, int cur_k,
          const uint32_t* __restrict__ src_map, const double* __restrict__ buf0, const double* __restrict__ buf1,
          double* __restrict__ out, int as_identity) {
    const int c = blockIdx.x * (SCATTER_THREADS >> 5) + (threadIdx.x >> 5);
    if (c >= nb) return;
    const int lane = threadIdx.x & 31;
    const int4 rec = __ldg(col_rec + c);
    const int nv = rec.z - (int)blockIdx.y * SCATTER_CHUNK;  // values of this chunk
    if (nv <= 0) return;
    const int cnt = min(nv, SCATTER_CHUNK);
    const int64_t b = (((int64_t)rec.y << 32) | (int64_t)(uint32_t)rec.x) + (int64_t)blockIdx.y * SCATTER_CHUNK;
    const uint32_t* sm = src_map + b;
    double* o = out + b;
    const int g = rec.w;
    // the source-map entries of the first pass do not depend on the group: in flight with its scalars
    uint32_t m[SCATTER_U];
#pragma unroll
    for (int u = 0; u < SCATTER_U; ++u) m[u] = (lane + 32 * u < cnt) ? __ldcs(sm + lane + 32 * u) : 0u;
    const int di = done_iter[g];
    const int kb = di >= 0 ? di : cur_k;
    const double* Xg = ((kb & 1) ? buf1 : buf0) + ws_off[g];
    double xs = 1.0;
    if (kb == 0 && !as_identity) {
        const double s = __longlong_as_double((long long)gersh[g]);
        xs = s > 0.0 ? 1.0 / s : 1.0;
    }
    for (int e0 = 0;;) {
        double x[SCATTER_U];
#pragma unroll
        for (int u = 0; u < SCATTER_U; ++u) x[u] = (e0 + lane + 32 * u < cnt) ? __ldcs(Xg + (m[u] & 0x7fffffffu)) : 0.0;
#pragma unroll
        for (int u = 0; u < SCATTER_U; ++u)
            if (e0 + lane + 32 * u < cnt)
                __stcs(o + e0 + lane + 32 * u, as_identity ? x[u] : 0.5 * ((double)(m[u] >> 31) - xs * x[u]));
        e0 += 32 * SCATTER_U;
        if (e0 >= cnt) break;
#pragma unroll
        for (int u = 0; u < SCATTER_U; ++u) m[u] = (e0 + lane + 32 * u < cnt) ? __ldcs(sm + e0 + lane + 32 * u) : 0u;
    }
}

sm_status_t launch_scatter(sm_plan* p, int as_identity, const double* buf0, const double* buf1,
                           double* out, cudaStream_t st) {
    if (p->nb == 0 || p->nnz == 0) return SM_OK;
    if (!p->d_src_map) {  // once per plan (pattern only)
        SM_CUDA(cudaMalloc((void**)&p->d_src_map, (size_t)p->nnz * 4));
        SM_CUDA(cudaMalloc((void**)&p->d_col_rec, (size_t)p->nb * 16));
        k_scatter_map_build<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_colptr, p->d_val_off,
                                                             p->d_col_grp, p->d_gen_off, p->d_blk_pack, p->d_ld,
                                                             p->d_src_map, p->d_col_rec);
        p->launches++;
        int64_t mx = 0;
        for (int c = 0; c < p->nb; ++c) {
            int64_t rows = 0;
            for (int64_t q = p->h_colptr[c]; q < p->h_colptr[c + 1]; ++q) rows += p->h_blk_size[p->h_rowidx[q]];
            mx = std::max(mx, rows * p->h_blk_size[c]);
        }
        p->scatter_chunks = (int)std::max<int64_t>(1, (mx + SCATTER_CHUNK - 1) / SCATTER_CHUNK);
    }
    k_scatter<<<dim3((p->nb + 7) / 8, p->scatter_chunks), SCATTER_THREADS, 0, st>>>(
        p->nb, p->d_col_rec, p->d_ws_off, p->d_done_iter, p->d_gersh, p->cur_k, p->d_src_map, buf0, buf1, out, as_identity);
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

// Steering bound of the mu bisection (reading A11c).  After MODE 0 of iteration k >= 1 the
// workspace holds X_k and Y_k = X_k^2, all eigenvalues x_l of X_k lie in [-1,1] and move monotonically
// towards +-1, so with w_l = sum_{k in gen} Q_kl^2 (Algorithm 1)
//   |n_elec(final) - n_elec(X_k)| <= 1/2 sum_l w_l (1 - |x_l|).
// With u_l = 1 - x_l^2 in [0,1]:  1 - |x_l| = 1 - sqrt(1 - u_l) <= min(u_l, u_l/2 + u_l^2/2)  (the second
// is tangent at u = 0 and exact at u = 1), and per generating row k (weights Q_kl^2, summing to 1)
//   sum_l Q_kl^2 u_l = 1 - (Y_k)_kk =: S1,   sum_l Q_kl^2 u_l^2 = ((I - Y_k)^2)_kk = sum_j (delta_kj - Y_kj)^2 =: S2,
// so row k contributes at most 1/2 min(S1, (S1 + S2)/2): half of the first-order bound once the
// iteration is close to convergence.  The rows of Y_k for the generating functions are read in full.
// part[c] = n_elec partial of X_k, part[nb + c] = bound partial of block column c.
__global__ void k_nelec_bound(int nb, const int32_t* __restrict__ col_grp, const int32_t* __restrict__ blk_size,
                              const int32_t* __restrict__ gen_off, const int32_t* __restrict__ ldv,
                              const int64_t* __restrict__ ws_off, const int32_t* __restrict__ done_iter,
                              const unsigned long long* __restrict__ gersh, int k, const double* __restrict__ buf0,
                              const double* __restrict__ buf1, const double* __restrict__ bufY,
                              double* __restrict__ part, const int32_t* __restrict__ ctrl,
                              const double* __restrict__ alpha, int ngroups, const int32_t* __restrict__ flag) {
    // one warp per generating block column c (partials per block column: more warps in flight than one per group)
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= nb || ctrl[0] != 0 || ctrl[3] != 0) return;  // evaluation stopped, or steering proven idle (EvalCtrl::steer_off): empty launch
    const int lane = threadIdx.x & 31;
    const int g = col_grp[c];
    if (g < 0) {  // block column of another shard
        if (lane == 0) { part[c] = 0.0; part[nb + c] = 0.0; }
        return;
    }
    const int di = done_iter[g];
    if (di >= 0 && flag[g] == 3) {
        // finished by the two-step exit (reading A9c): the generating rows of the result are in the buffer of parity
        // di, X_{di-1} was never formed; the count is final, nothing is left to bound
        const double* Xf = ((di & 1) ? buf1 : buf0) + ws_off[g];
        const int ldf = ldv[g];
        double af = 0.0;
        const int of = gen_off[c], bf = blk_size[c];
        for (int e = lane; e < bf; e += 32) af += 0.5 * (1.0 - Xf[panel_off(of + e, of + e, ldf)]);
#pragma unroll
        for (int w = 16; w > 0; w >>= 1) af += __shfl_xor_sync(0xffffffffu, af, w);
        if (lane == 0) { part[c] = af; part[nb + c] = 0.0; }
        return;
    }
    const int kb = (di >= 0 && di <= k) ? di : k;  // di = k + 1: predicted exit, its last update has not run yet
    const double* Xg = ((kb & 1) ? buf1 : buf0) + ws_off[g];
    const double* Yg = bufY + ws_off[g];
    const int ld = ldv[g];
    double xs = 1.0;
    if (kb == 0) {  // stopped at iteration 0: the buffer still holds the unscaled a_i - mu I
        const double s = __longlong_as_double((long long)gersh[g]);
        xs = s > 0.0 ? 1.0 / s : 1.0;
    }
    double rinv = 1.0;  // reading A8b: the stored Y is al^2 X^2
    if (alpha) { const double al = alpha[(size_t)(kb & 1) * ngroups + g]; rinv = 1.0 / (al * al); }
    double a = 0.0, d = 0.0;
    const int o = gen_off[c], b = blk_size[c];
    for (int e = 0; e < b; ++e) {      // generating function (row) o + e: the lanes sweep its row of Y
        const int row = o + e;
        const int t0 = row & ~63;
        const double* yr = Yg + (size_t)t0 * ld + (size_t)(row & 63) * 8;
        const size_t pstride = (size_t)min(64, ld - t0) * 8;
        double s2 = 0.0, ykk = 0.0;
        for (int j = lane; j < ld; j += 32) {
            const double y = yr[(size_t)(j >> 3) * pstride + (j & 7)] * rinv;
            const double t = (j == row ? 1.0 : 0.0) - y;
            s2 = fma(t, t, s2);
            if (j == row) ykk = y;
        }
#pragma unroll
        for (int w = 16; w > 0; w >>= 1) {
            s2 += __shfl_xor_sync(0xffffffffu, s2, w);
            ykk += __shfl_xor_sync(0xffffffffu, ykk, w);
        }
        if (lane == 0) {
            const double s1 = fmax(1.0 - ykk, 0.0);
            a += 0.5 * (1.0 - xs * Xg[panel_off(row, row, ld)]);
            d += 0.5 * fmin(s1, 0.5 * (s1 + s2));
        }
    }
    if (lane == 0) { part[c] = a; part[nb + c] = d; }
}

// Called after MODE 0 + decision of iteration k >= 1 (the update touches neither X_k nor Y_k).
sm_status_t launch_nelec_bound(sm_plan* p, int k, const double* buf0, const double* buf1, const double* bufY,
                               cudaStream_t st) {
    if (p->ngroups == 0 || p->nb == 0) return SM_OK;
    k_nelec_bound<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_col_grp, p->d_blk_size, p->d_gen_off, p->d_ld, p->d_ws_off,
                                                   p->d_done_iter, p->d_gersh, k, buf0, buf1, bufY, p->d_bound_part,
                                                   p->d_ctrl, rescale_on(p) ? p->d_alpha : nullptr, p->ngroups, p->d_flag);
    p->launches += 1;  // the two sums are taken by k_eval_ctrl
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

// Device-side end of an evaluation (one CTA, after k_ns_decide and k_nelec_bound of iteration k): the fixed-order
// sums of the steering partials (count of X_k and its bound; same order as k_sum_fixed), then the decision.
__global__ void __launch_bounds__(1024)
k_eval_ctrl(EvalCtrl* __restrict__ c, int k, const int32_t* __restrict__ counters, double* __restrict__ bound,
            const double* __restrict__ bound_part, int nb, int steer, double n_target, double margin) {
    __shared__ double s0[1024], s1[1024];
    if (c->stop != 0) return;  // uniform: set by an earlier launch
    if (c->steer_off != 0) steer = 0;  // uniform
    if (steer && k >= 1) {
        double a = 0.0, b = 0.0;
        for (int i = threadIdx.x; i < nb; i += 1024) { a += bound_part[i]; b += bound_part[nb + i]; }
        s0[threadIdx.x] = a; s1[threadIdx.x] = b;
        __syncthreads();
        for (int o = 512; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) { s0[threadIdx.x] += s0[threadIdx.x + o]; s1[threadIdx.x] += s1[threadIdx.x + o]; }
            __syncthreads();
        }
    }
    if (threadIdx.x != 0) return;
    if (steer && k >= 1) { bound[2 * k] = s0[0]; bound[2 * k + 1] = s1[0]; }
    if (counters[k] == 0) { c->stop = 1; c->k_stop = k; return; }
    if (steer && k >= 1) {
        const double ne = s0[0], err = s1[0];
        if (ne == ne && err == err && err >= 0.0) {
            const double g = ne - n_target, m = err + margin;
            if (g > m || g < -m) { c->stop = 2; c->k_stop = k; c->decided = g > 0 ? 1 : -1; c->ne = ne; c->err = err; }
            // the count of the converged X lies in [ne - err, ne + err]: once that interval is inside (-m/2, m/2)
            // around the target, no later iteration can satisfy the test above -- stop paying for the bound
            else if (fabs(g) + err < 0.5 * m) c->steer_off = 1;
        }
    }
}

sm_status_t launch_eval_ctrl(sm_plan* p, int k, int steer, double n_target, double margin, cudaStream_t st) {
    k_eval_ctrl<<<1, 1024, 0, st>>>(reinterpret_cast<EvalCtrl*>(p->d_ctrl), k, p->d_counters, p->d_bound, p->d_bound_part,
                                    p->nb, steer, n_target, margin);
    p->launches++;
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

// Enqueues the Gershgorin interval of the whole K~ into d_scalars[4..5] and its copy into h_pinned_d[4..5];
// the caller synchronises the stream before reading them (no allocation, no synchronisation here).
sm_status_t launch_gersh_global(sm_plan* p, const double* vals, cudaStream_t st) {
    if (!p->d_gg) SM_CUDA(cudaMalloc((void**)&p->d_gg, (size_t)std::max(p->nb, 1) * 16));
    double *lo = p->d_gg, *hi = p->d_gg + p->nb;
    k_gersh_global<<<(p->nb + 7) / 8, 256, 0, st>>>(p->nb, p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_val_off,
                                                    vals, lo, hi);
    k_minmax_fixed<<<1, 1024, 0, st>>>(lo, hi, p->nb, p->d_scalars + 4);
    p->launches += 2;
    SM_CUDA(cudaGetLastError());
    SM_CUDA(cudaMemcpyAsync(p->h_pinned_d + 4, p->d_scalars + 4, 16, cudaMemcpyDeviceToHost, st));
    return SM_OK;
}

}  // namespace smb
