// a1 device BSR container + a2 submatrix index builder.
//
// Index builder: one CTA per generating group G_i.  A bitmap of nb bits in shared memory marks
// every block row that has a stored block in one of the group's columns (atomicOr); an ordered
// compaction of the set bits (popc prefix sums over the bitmap words) yields S_i in ascending
// order together with the running element offset.  Two passes: count (|S_i|, n_i), then fill.
// Integer only; the output is canonical, so it is compared bit-exactly with the oracle's
// (which sorts and deduplicates concatenated row lists instead).
#include <algorithm>
#include <cstring>
#include <numeric>

#include "common.cuh"

namespace smb {

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// In-place bitonic sort of P (a power of two) keys in shared memory by the whole CTA.
__device__ void bitonic_sort_smem(int32_t* key, int P) {
    for (int k = 2; k <= P; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < P; i += blockDim.x) {
                const int l = i ^ j;
                if (l > i) {
                    const int a = key[i], b = key[l];
                    if ((a > b) == ((i & k) == 0)) { key[i] = b; key[l] = a; }
                }
            }
            __syncthreads();
        }
}

// CTA-wide exclusive scan of one value per thread (chunk of blockDim values); returns the exclusive
// prefix and adds the chunk total to `carry` (uniform).  s_w: 32 ints of shared scratch.
__device__ int block_excl_scan(int v, int& carry, int* s_w) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int inc = warp_incl_scan(v, lane);
    if (lane == 31) s_w[wid] = inc;
    __syncthreads();
    int before = 0, total = 0;
    for (int w = 0; w < nw; ++w) {
        if (w < wid) before += s_w[w];
        total += s_w[w];
    }
    const int ex = carry + before + inc - v;
    carry += total;
    __syncthreads();
    return ex;
}

// Sort key[0..fill) and drop duplicates in place; returns the number of distinct keys (uniform).
// Compaction runs chunk by chunk in ascending order: an element only ever moves to a position at or
// below its own, and every chunk has its keys in registers before it writes.
__device__ int sort_unique_smem(int32_t* key, int fill, int* s_w) {
    int P = 2;
    while (P < fill) P <<= 1;
    for (int i = fill + threadIdx.x; i < P; i += blockDim.x) key[i] = INT32_MAX;
    __syncthreads();
    bitonic_sort_smem(key, P);
    int u = 0;
    for (int base = 0; base < fill; base += blockDim.x) {
        const int i = base + threadIdx.x;
        int cur = INT32_MAX, keep = 0;
        if (i < fill) {
            cur = key[i];
            keep = (i == 0 || key[i - 1] != cur) ? 1 : 0;
        }
        __syncthreads();
        const int pos = block_excl_scan(keep, u, s_w);
        if (keep) key[pos] = cur;
        __syncthreads();
    }
    return u;
}

// a2, pass 1: S_i = ascending union of the row lists of the group's block columns (L125, L199), by
// SORTING -- work proportional to the group's own stored blocks, independent of nb: the lists are
// appended to a shared buffer of `cap` keys behind the union found so far; when the next list does not
// fit, and at the end, the buffer is sorted and deduplicated.  Output: scratch[eptr[g] ..] (eptr =
// exclusive prefix of the groups' stored-block counts, so the scratch holds nnzb keys) and sub_cnt[g].
__global__ void __launch_bounds__(256)
k_index_union(const int64_t* __restrict__ colptr, const int32_t* __restrict__ rowidx,
              const int32_t* __restrict__ grp_ptr, const int32_t* __restrict__ grp_cols,
              const int64_t* __restrict__ eptr, int cap, int32_t* __restrict__ scratch,
              int32_t* __restrict__ sub_cnt, int32_t* __restrict__ err) {
    extern __shared__ int32_t key[];
    __shared__ int s_w[32];
    const int g = blockIdx.x;
    int u = 0, fill = 0;
    for (int gc = grp_ptr[g]; gc < grp_ptr[g + 1]; ++gc) {
        const int c = grp_cols[gc];
        const int64_t p0 = colptr[c];
        const int len = (int)(colptr[c + 1] - p0);
        if (fill + len > cap) {
            if (fill > u) { u = sort_unique_smem(key, fill, s_w); fill = u; }
            if (fill + len > cap) {  // more member blocks than one pass holds: unsupported size
                if (threadIdx.x == 0) { atomicExch(err, 2); sub_cnt[g] = 0; }
                return;
            }
        }
        for (int t = threadIdx.x; t < len; t += blockDim.x) key[fill + t] = rowidx[p0 + t];
        fill += len;
        __syncthreads();
    }
    if (fill > u) u = sort_unique_smem(key, fill, s_w);
    int32_t* out = scratch + eptr[g];
    for (int t = threadIdx.x; t < u; t += blockDim.x) out[t] = key[t];
    if (threadIdx.x == 0) sub_cnt[g] = u;
}

// Exclusive prefix sum of n int32 counts into n + 1 int64 offsets by one CTA (fixed order; plan time).
__global__ void __launch_bounds__(1024) k_excl_scan_i32_i64(const int32_t* __restrict__ in, int64_t n,
                                                            int64_t* __restrict__ out) {
    __shared__ int s_w[32];
    int64_t carry = 0;
    for (int64_t base = 0; base < n; base += blockDim.x) {
        const int64_t i = base + threadIdx.x;
        const int v = i < n ? in[i] : 0;
        int c32 = 0;
        const int ex = block_excl_scan(v, c32, s_w);
        if (i < n) out[i] = carry + ex;
        carry += c32;
    }
    if (threadIdx.x == 0) out[n] = carry;
}

__device__ __forceinline__ int find_sorted(const int32_t* a, int n, int key) {
    int lo = 0, hi = n - 1;
    while (lo <= hi) {
        int mid = (lo + hi) >> 1, v = a[mid];
        if (v == key) return mid;
        if (v < key) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

// a2, pass 2: members, element offsets (running sum of the block sizes), n_i, and for every generating
// column its position / offset in S_i and the local row offset of each of its stored blocks.
__global__ void __launch_bounds__(256)
k_index_fill(const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
             const int32_t* __restrict__ rowidx, const int32_t* __restrict__ grp_ptr,
             const int32_t* __restrict__ grp_cols, const int64_t* __restrict__ eptr,
             const int32_t* __restrict__ scratch, const int64_t* __restrict__ sub_ptr,
             int32_t* __restrict__ sub_blocks, int32_t* __restrict__ sub_off, int32_t* __restrict__ sub_dim,
             int32_t* __restrict__ gen_pos, int32_t* __restrict__ gen_off, uint32_t* __restrict__ blk_pack,
             int32_t* __restrict__ col_grp, int32_t* __restrict__ gen_width, int2* __restrict__ gen_rng,
             int32_t* __restrict__ err) {
    __shared__ int s_w[32];
    const int g = blockIdx.x;
    int32_t* S = sub_blocks + sub_ptr[g];
    int32_t* So = sub_off + sub_ptr[g];
    const int m = (int)(sub_ptr[g + 1] - sub_ptr[g]);
    const int32_t* in = scratch + eptr[g];
    int carry = 0;
    for (int base = 0; base < m; base += blockDim.x) {
        const int t = base + threadIdx.x;
        int r = 0, sz = 0;
        if (t < m) { r = in[t]; sz = blk_size[r]; }
        const int ex = block_excl_scan(sz, carry, s_w);
        if (t < m) { S[t] = r; So[t] = ex; }
    }
    if (threadIdx.x == 0) sub_dim[g] = carry;
    __syncthreads();  // S, So of this group are complete and visible to the CTA
    int gw = 0, glo = INT32_MAX, ghi = -1;  // first / last generating row of a_i
    for (int gc = grp_ptr[g]; gc < grp_ptr[g + 1]; ++gc) {
        const int c = grp_cols[gc];
        gw += blk_size[c];
        const int pos = find_sorted(S, m, c);
        if (pos >= 0) { glo = min(glo, So[pos]); ghi = max(ghi, So[pos] + blk_size[c] - 1); }
        if (threadIdx.x == 0) {
            gen_pos[gc] = pos;
            col_grp[c] = g;
            if (pos < 0) atomicExch(err, 1); else gen_off[c] = So[pos];
        }
        for (int64_t p = colptr[c] + threadIdx.x; p < colptr[c + 1]; p += blockDim.x) {
            const int r = rowidx[p];
            const int t = find_sorted(S, m, r);  // always found: S_i contains the rows of its own columns
            blk_pack[p] = (t >= 0 ? (uint32_t)So[t] : 0xfffffu) | ((uint32_t)blk_size[r] << 20);
        }
    }
    if (threadIdx.x == 0) { gen_width[g] = gw; gen_rng[g] = make_int2(glo, ghi); }
}

sm_status_t launch_excl_scan(const int32_t* in, int64_t n, int64_t* out, cudaStream_t st) {
    k_excl_scan_i32_i64<<<1, 1024, 0, st>>>(in, n, out);
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}

template <typename T>
static sm_status_t upload(T** d, const T* h, size_t n, cudaStream_t st) {
    SM_CUDA(cudaMalloc((void**)d, std::max<size_t>(n, 1) * sizeof(T)));
    if (n) SM_CUDA(cudaMemcpyAsync(*d, h, n * sizeof(T), cudaMemcpyHostToDevice, st));
    return SM_OK;
}

sm_status_t build_index_device(sm_plan* p, cudaStream_t st) {
    const int nb = p->nb, ng = p->ngroups;
    sm_status_t s;
    // a1: device BSR container
    std::vector<int32_t> blk_off(nb + 1, 0);
    for (int i = 0; i < nb; ++i) blk_off[i + 1] = blk_off[i] + p->h_blk_size[i];
    std::vector<int64_t> val_off(p->nnzb + 1, 0);
    for (int c = 0; c < nb; ++c)
        for (int64_t q = p->h_colptr[c]; q < p->h_colptr[c + 1]; ++q)
            val_off[q + 1] = val_off[q] + (int64_t)p->h_blk_size[p->h_rowidx[q]] * p->h_blk_size[c];
    p->nnz = val_off[p->nnzb];
    p->max_col_blocks = 0;
    for (int c = 0; c < nb; ++c)
        p->max_col_blocks = std::max<int32_t>(p->max_col_blocks, (int32_t)(p->h_colptr[c + 1] - p->h_colptr[c]));
    if ((s = upload(&p->d_blk_size, p->h_blk_size.data(), nb, st))) return s;
    if ((s = upload(&p->d_blk_off, blk_off.data(), nb + 1, st))) return s;
    if ((s = upload(&p->d_colptr, p->h_colptr.data(), nb + 1, st))) return s;
    if ((s = upload(&p->d_rowidx, p->h_rowidx.data(), p->nnzb, st))) return s;
    if ((s = upload(&p->d_val_off, val_off.data(), p->nnzb + 1, st))) return s;
    if (p->opt.scaling == 1) {  // packed block records of the Lanczos mat-vec (spectral.cu)
        std::vector<int64_t> colval((size_t)nb + 1);  // first value of every block column: one load instead of two dependent ones
        for (int c = 0; c <= nb; ++c) colval[c] = val_off[p->h_colptr[c]];
        if ((s = upload(&p->d_col_val, colval.data(), (size_t)nb + 1, st))) return s;
        std::vector<int4> rec((size_t)p->nnzb);
        for (int64_t q = 0; q < p->nnzb; ++q) {
            const int r = p->h_rowidx[q];
            rec[q] = make_int4((int)(val_off[q] & 0xffffffffll), (int)(val_off[q] >> 32), blk_off[r], p->h_blk_size[r]);
        }
        if ((s = upload(&p->d_lz_rec, rec.data(), (size_t)p->nnzb, st))) return s;
        SM_CUDA(cudaStreamSynchronize(st));  // rec goes out of scope
    }
    if ((s = upload(&p->d_grp_ptr, p->h_grp_ptr.data(), ng + 1, st))) return s;
    if ((s = upload(&p->d_grp_cols, p->h_grp_cols.data(), p->h_grp_cols.size(), st))) return s;

    // a2: index builder.  eptr = exclusive prefix of the groups' stored-block counts (every block column is
    // in exactly one group, so the scratch of pass 1 holds nnzb keys); O(nb) integers on the host.
    std::vector<int64_t> eptr(ng + 1, 0);
    int64_t max_e = 1;
    for (int i = 0; i < ng; ++i) {
        int64_t e = 0;
        for (int q = p->h_grp_ptr[i]; q < p->h_grp_ptr[i + 1]; ++q)
            e += p->h_colptr[p->h_grp_cols[q] + 1] - p->h_colptr[p->h_grp_cols[q]];
        eptr[i + 1] = eptr[i] + e;
        max_e = std::max(max_e, e);
    }
    int cap = 256;  // keys of one sort pass in shared memory: enough for the largest group, at most 32768 (128 KB)
    while (cap < max_e && cap < 32768) cap <<= 1;
    const size_t key_bytes = (size_t)cap * 4;
    if (key_bytes > 48 * 1024)
        SM_CUDA(cudaFuncSetAttribute(k_index_union, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)key_bytes));
    DevTmp cnt_tmp, err_tmp, eptr_tmp, scratch_tmp;
    SM_CUDA(cudaMalloc(&cnt_tmp.p, (size_t)std::max(ng, 1) * 4));
    SM_CUDA(cudaMalloc(&err_tmp.p, 4));
    SM_CUDA(cudaMalloc(&eptr_tmp.p, (size_t)(ng + 1) * 8));
    SM_CUDA(cudaMalloc(&scratch_tmp.p, (size_t)std::max<int64_t>(p->nnzb, 1) * 4));
    int32_t* d_cnt = (int32_t*)cnt_tmp.p;
    int32_t* d_err = (int32_t*)err_tmp.p;
    int64_t* d_eptr = (int64_t*)eptr_tmp.p;
    int32_t* d_scratch = (int32_t*)scratch_tmp.p;
    SM_CUDA(cudaMemcpyAsync(d_eptr, eptr.data(), (size_t)(ng + 1) * 8, cudaMemcpyHostToDevice, st));
    SM_CUDA(cudaMemsetAsync(d_err, 0, 4, st));
    SM_CUDA(cudaMalloc((void**)&p->d_sub_ptr, (size_t)(ng + 1) * 8));
    SM_CUDA(cudaMalloc((void**)&p->d_sub_dim, (size_t)std::max(ng, 1) * 4));
    cudaEvent_t ev[4];
    for (auto& e : ev) SM_CUDA(cudaEventCreate(&e));
    struct EvFree { cudaEvent_t* e; ~EvFree() { for (int i = 0; i < 4; ++i) cudaEventDestroy(e[i]); } } ev_free{ev};
    // pass 1: sorted unions + their sizes, device prefix sum
    SM_CUDA(cudaEventRecord(ev[0], st));
    if (ng > 0) k_index_union<<<ng, 256, key_bytes, st>>>(p->d_colptr, p->d_rowidx, p->d_grp_ptr, p->d_grp_cols, d_eptr,
                                                          cap, d_scratch, d_cnt, d_err);
    k_excl_scan_i32_i64<<<1, 1024, 0, st>>>(d_cnt, ng, p->d_sub_ptr);
    SM_CUDA(cudaEventRecord(ev[1], st));
    p->launches += 2;
    int64_t tot = 0;
    int32_t herr = 0;
    SM_CUDA(cudaMemcpyAsync(&tot, p->d_sub_ptr + ng, 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaMemcpyAsync(&herr, d_err, 4, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));  // the only host round trip of the build: 12 bytes, to size the index
    SM_CUDA(cudaGetLastError());
    if (herr == 2) return SM_ERR_INVALID_ARG;  // a submatrix with more member blocks than one sort pass holds
    SM_CUDA(cudaMalloc((void**)&p->d_sub_blocks, std::max<int64_t>(tot, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_sub_off, std::max<int64_t>(tot, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_pos, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_off, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_col_grp, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMemsetAsync(p->d_col_grp, 0xff, (size_t)std::max(nb, 1) * 4, st));  // -1: column of another shard
    SM_CUDA(cudaMalloc((void**)&p->d_blk_pack, std::max<int64_t>(p->nnzb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_width, (size_t)std::max(ng, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_rng, (size_t)std::max(ng, 1) * 8));
    // pass 2
    SM_CUDA(cudaEventRecord(ev[2], st));
    if (ng > 0) k_index_fill<<<ng, 256, 0, st>>>(p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_grp_ptr, p->d_grp_cols,
                                                 d_eptr, d_scratch, p->d_sub_ptr, p->d_sub_blocks, p->d_sub_off,
                                                 p->d_sub_dim, p->d_gen_pos, p->d_gen_off, p->d_blk_pack, p->d_col_grp,
                                                 p->d_gen_width, p->d_gen_rng, d_err);
    SM_CUDA(cudaEventRecord(ev[3], st));
    p->launches++;
    p->h_sub_dim.resize(ng);
    p->h_sub_ptr.assign(ng + 1, 0);
    SM_CUDA(cudaMemcpyAsync(&herr, d_err, 4, cudaMemcpyDeviceToHost, st));
    if (ng) SM_CUDA(cudaMemcpyAsync(p->h_sub_dim.data(), p->d_sub_dim, (size_t)ng * 4, cudaMemcpyDeviceToHost, st));
    p->h_gen_rng.resize((size_t)2 * ng);
    if (ng) SM_CUDA(cudaMemcpyAsync(p->h_gen_rng.data(), p->d_gen_rng, (size_t)ng * 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaMemcpyAsync(p->h_sub_ptr.data(), p->d_sub_ptr, (size_t)(ng + 1) * 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));  // sizes for the workspace geometry and tile list below
    SM_CUDA(cudaGetLastError());
    if (herr) return SM_ERR_STRUCTURE;
    float ms1 = 0.f, ms2 = 0.f;
    cudaEventElapsedTime(&ms1, ev[0], ev[1]);
    cudaEventElapsedTime(&ms2, ev[2], ev[3]);
    p->ms_index_kernels = ms1 + ms2;
    p->max_sub_blocks = 0;
    for (int i = 0; i < ng; ++i)
        p->max_sub_blocks = std::max<int32_t>(p->max_sub_blocks, (int32_t)(p->h_sub_ptr[i + 1] - p->h_sub_ptr[i]));

    // workspace geometry (group order, keeps the locality of consecutive submatrices, L188) and
    // the GEMM tile list, largest padded size first (size buckets = equal ld).
    p->h_ld.resize(ng);
    p->h_ws_off.resize(ng);
    int64_t off = 0, n2 = 0, n3 = 0;
    int dmin = INT32_MAX, dmax = 0;
    for (int i = 0; i < ng; ++i) {
        int n = p->h_sub_dim[i];
        int ld = (n + LD_ALIGN - 1) / LD_ALIGN * LD_ALIGN;
        p->h_ld[i] = ld;
        p->h_ws_off[i] = off;
        off += (int64_t)ld * ld;
        n2 += (int64_t)n * n;
        n3 += (int64_t)n * n * n;
        dmin = std::min(dmin, n);
        dmax = std::max(dmax, n);
    }
    p->sum_ld2 = off;
    if (dmax >= (1 << 20) - LD_ALIGN) return SM_ERR_INVALID_ARG;  // packed block records hold 20-bit offsets
    if ((int64_t)(dmax + LD_ALIGN) * (dmax + LD_ALIGN) >= (1LL << 31)) return SM_ERR_INVALID_ARG;  // 31-bit scatter map / tile offsets
    std::vector<int32_t> order(ng);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return p->h_ld[a] > p->h_ld[b]; });
    std::vector<TileDesc> tiles;
    p->h_tile_first.assign(ng, 0);
    p->h_tile_count.assign(ng, 0);
    int nbuckets = 0, last_ld = -1;
    for (int oi = 0; oi < ng; ++oi) {
        int i = order[oi];
        if (p->h_ld[i] != last_ld) { ++nbuckets; last_ld = p->h_ld[i]; }
        int nt = (p->h_ld[i] + TILE - 1) / TILE;
        p->h_tile_first[i] = (int32_t)tiles.size();
        const int32_t first = (int32_t)tiles.size(), count = nt * (nt + 1) / 2;
        auto push = [&](int ti, int tj) {
            TileDesc t;
            t.ws_off = p->h_ws_off[i]; t.grp = i; t.ld = p->h_ld[i]; t.n = p->h_sub_dim[i];
            t.tij = ti | (tj << 16); t.tile_first = first; t.tile_count = count;
            tiles.push_back(t);
        };
        // off-diagonal (full) tiles first, diagonal (half-empty) tiles last
        for (int ti = 0; ti < nt; ++ti)
            for (int tj = 0; tj < ti; ++tj) push(ti, tj);
        for (int ti = 0; ti < nt; ++ti) push(ti, ti);
        p->h_tile_count[i] = (int32_t)tiles.size() - p->h_tile_first[i];
    }
    p->n_tiles = (int64_t)tiles.size();
    // algorithmic flop of the last update of a submatrix that leaves by the predicted exit: only the tiles that
    // hold generating rows (as rows, or mirrored as columns) are computed (ns_sign.cu)
    // ... or, for groups whose generating rows span at most THIN_MAX_ROWS rows (or n / 16), the thin product of k_ns_thin: span x n x n
    int max_ld = 8;
    for (int i = 0; i < ng; ++i) max_ld = std::max(max_ld, p->h_ld[i]);
    p->thin_smem = (size_t)8 * max_ld * 8 <= (size_t)200 * 1024 ? (size_t)8 * max_ld * 8 : 0;  // 8 rows of X in shared memory
    p->thin3_smem = (size_t)16 * max_ld * 8 <= (size_t)200 * 1024 ? (size_t)16 * max_ld * 8 : 0;  // two such arrays (k_ns_thin3)
    p->h_final_flop.assign(ng, 0);
    for (int i = 0; i < ng; ++i) {
        const int ld = p->h_ld[i], n = p->h_sub_dim[i], nt = (ld + TILE - 1) / TILE;
        const int tl = p->h_gen_rng[2 * i] / TILE, th = p->h_gen_rng[2 * i + 1] / TILE;
        const int span = p->h_gen_rng[2 * i + 1] - p->h_gen_rng[2 * i] + 1;
        if (p->thin_smem > 0 && thin_span_ok(span, n)) {
            p->h_final_flop[i] = 2 * (int64_t)span * n * n;
            continue;
        }
        int64_t f = 0;
        for (int ti = 0; ti < nt; ++ti)
            for (int tj = 0; tj <= ti; ++tj) {
                if (!((ti >= tl && ti <= th) || (tj >= tl && tj <= th))) continue;
                const int64_t ri = std::max(0, std::min(TILE, n - ti * TILE)), rj = std::max(0, std::min(TILE, n - tj * TILE));
                f += (ti == tj ? ri * (ri + 1) : 2 * ri * rj) * (int64_t)n;
            }
        p->h_final_flop[i] = f;
    }
    if ((s = upload(&p->d_ld, p->h_ld.data(), ng, st))) return s;
    if ((s = upload(&p->d_ws_off, p->h_ws_off.data(), ng, st))) return s;
    if ((s = upload(&p->d_tiles, tiles.data(), tiles.size(), st))) return s;
    if ((s = upload(&p->d_tile_first, p->h_tile_first.data(), ng, st))) return s;
    if ((s = upload(&p->d_tile_count, p->h_tile_count.data(), ng, st))) return s;
    SM_CUDA(cudaStreamSynchronize(st));

    sm_plan_info_t& I = p->info;
    memset(&I, 0, sizeof(I));
    I.nb = nb; I.ngroups = ng; I.nnzb = p->nnzb; I.nnz = p->nnz; I.n_basis = blk_off[nb];
    I.sum_sub_blocks = tot; I.dim_min = ng ? dmin : 0; I.dim_max = dmax;
    I.dim_mean = ng ? (double)std::accumulate(p->h_sub_dim.begin(), p->h_sub_dim.end(), (int64_t)0) / ng : 0.0;
    I.sum_n2 = n2; I.sum_n3 = n3; I.sum_ld2 = p->sum_ld2; I.n_tiles = p->n_tiles; I.n_buckets = nbuckets;
    const size_t buf = ((size_t)p->sum_ld2 * 8 + 255) / 256 * 256;
    I.workspace_bytes = 3 * buf;
    // cost model of the grouping (Eq.(14), Eq.(15)): integer sums on the host
    int64_t n3c = 0;
    for (int c : p->h_grp_cols) {  // the block columns of this plan's groups (all of them unless sharded)
        int64_t nc = 0;
        for (int64_t q = p->h_colptr[c]; q < p->h_colptr[c + 1]; ++q) nc += p->h_blk_size[p->h_rowidx[q]];
        n3c += nc * nc * nc;
    }
    I.sum_n3_columns = n3c;
    I.est_speedup = n3 > 0 ? (double)n3c / (double)n3 : 0.0;
    I.ms_index_kernels = p->ms_index_kernels;
    // the pattern is read once (nnzb x 4), members and offsets (sum |S_i| x 8) and the packed
    // block records (nnzb x 4) are written
    I.index_alg_bytes = p->nnzb * 8 + tot * 8;
    return SM_OK;
}

}  // namespace smb
