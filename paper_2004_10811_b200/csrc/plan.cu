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

// Marks the row blocks of group g in the shared bitmap.
__device__ void mark_rows(uint32_t* bitmap, int words, const int64_t* colptr, const int32_t* rowidx,
                          const int32_t* grp_ptr, const int32_t* grp_cols, int g) {
    for (int w = threadIdx.x; w < words; w += blockDim.x) bitmap[w] = 0u;
    __syncthreads();
    for (int gc = grp_ptr[g]; gc < grp_ptr[g + 1]; ++gc) {
        int c = grp_cols[gc];
        for (int64_t p = colptr[c] + threadIdx.x; p < colptr[c + 1]; p += blockDim.x) {
            int r = rowidx[p];
            atomicOr(&bitmap[r >> 5], 1u << (r & 31));
        }
    }
    __syncthreads();
}

// Block-wide exclusive scan of (cnt, size) pairs over one chunk of blockDim words; returns the
// exclusive prefix for this thread and adds the chunk totals to the running carries.
__device__ void block_scan2(int cnt, int sz, int& ex_cnt, int& ex_sz, int& carry_cnt, int& carry_sz,
                            int* s_w /*[2*32]*/) {
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int ic = warp_incl_scan(cnt, lane), is = warp_incl_scan(sz, lane);
    if (lane == 31) { s_w[wid] = ic; s_w[32 + wid] = is; }
    __syncthreads();
    int bc = 0, bsz = 0, tc = 0, tsz = 0;
    for (int w = 0; w < nw; ++w) {
        if (w < wid) { bc += s_w[w]; bsz += s_w[32 + w]; }
        tc += s_w[w]; tsz += s_w[32 + w];
    }
    ex_cnt = carry_cnt + bc + ic - cnt;
    ex_sz = carry_sz + bsz + is - sz;
    carry_cnt += tc;
    carry_sz += tsz;
    __syncthreads();
}

__global__ void k_index_count(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                              const int32_t* __restrict__ rowidx, const int32_t* __restrict__ grp_ptr,
                              const int32_t* __restrict__ grp_cols, int32_t* __restrict__ sub_cnt,
                              int32_t* __restrict__ sub_dim) {
    extern __shared__ uint32_t bitmap[];
    __shared__ int s_w[64];
    const int g = blockIdx.x, words = (nb + 31) >> 5;
    mark_rows(bitmap, words, colptr, rowidx, grp_ptr, grp_cols, g);
    int carry_c = 0, carry_s = 0;
    for (int base = 0; base < words; base += blockDim.x) {
        int w = base + threadIdx.x, cnt = 0, sz = 0;
        if (w < words) {
            uint32_t bits = bitmap[w];
            cnt = __popc(bits);
            while (bits) {
                int b = __ffs(bits) - 1;
                bits &= bits - 1;
                sz += blk_size[(w << 5) + b];
            }
        }
        int ec, es;
        block_scan2(cnt, sz, ec, es, carry_c, carry_s, s_w);
    }
    if (threadIdx.x == 0) { sub_cnt[g] = carry_c; sub_dim[g] = carry_s; }
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

__global__ void k_index_fill(int nb, const int32_t* __restrict__ blk_size, const int64_t* __restrict__ colptr,
                             const int32_t* __restrict__ rowidx, const int32_t* __restrict__ grp_ptr,
                             const int32_t* __restrict__ grp_cols, const int64_t* __restrict__ sub_ptr,
                             int32_t* __restrict__ sub_blocks, int32_t* __restrict__ sub_off,
                             int32_t* __restrict__ gen_pos, int32_t* __restrict__ gen_off,
                             uint32_t* __restrict__ blk_pack, int32_t* __restrict__ col_grp,
                             int32_t* __restrict__ gen_width, int32_t* __restrict__ err) {
    extern __shared__ uint32_t bitmap[];
    __shared__ int s_w[64];
    const int g = blockIdx.x, words = (nb + 31) >> 5;
    mark_rows(bitmap, words, colptr, rowidx, grp_ptr, grp_cols, g);
    int32_t* S = sub_blocks + sub_ptr[g];
    int32_t* So = sub_off + sub_ptr[g];
    const int m = (int)(sub_ptr[g + 1] - sub_ptr[g]);
    int carry_c = 0, carry_s = 0;
    for (int base = 0; base < words; base += blockDim.x) {
        int w = base + threadIdx.x, cnt = 0, sz = 0;
        uint32_t bits = 0;
        if (w < words) {
            bits = bitmap[w];
            cnt = __popc(bits);
            uint32_t t = bits;
            while (t) {
                int b = __ffs(t) - 1;
                t &= t - 1;
                sz += blk_size[(w << 5) + b];
            }
        }
        int ec, es;
        block_scan2(cnt, sz, ec, es, carry_c, carry_s, s_w);
        while (bits) {  // ordered compaction: ascending bit order inside the word
            int b = __ffs(bits) - 1;
            bits &= bits - 1;
            int r = (w << 5) + b;
            S[ec] = r;
            So[ec] = es;
            ++ec;
            es += blk_size[r];
        }
    }
    __syncthreads();  // S, So of this group are complete and visible to the CTA
    // position / offset of every generating column, local row offset of each of its blocks
    int gw = 0;
    for (int gc = grp_ptr[g]; gc < grp_ptr[g + 1]; ++gc) {
        int c = grp_cols[gc];
        gw += blk_size[c];
        int pos = find_sorted(S, m, c);
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
    if (threadIdx.x == 0) gen_width[g] = gw;
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
    if ((s = upload(&p->d_grp_ptr, p->h_grp_ptr.data(), ng + 1, st))) return s;
    if ((s = upload(&p->d_grp_cols, p->h_grp_cols.data(), nb, st))) return s;

    // a2: index builder, pass 1
    const size_t bm_bytes = (size_t)((nb + 31) / 32) * 4;
    if (bm_bytes > 200 * 1024) return SM_ERR_INVALID_ARG;  // nb > 1.6 M block rows: bitmap does not fit
    if (bm_bytes > 48 * 1024) {
        SM_CUDA(cudaFuncSetAttribute(k_index_count, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bm_bytes));
        SM_CUDA(cudaFuncSetAttribute(k_index_fill, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bm_bytes));
    }
    int32_t* d_cnt = nullptr;
    SM_CUDA(cudaMalloc((void**)&d_cnt, (size_t)std::max(ng, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_sub_dim, (size_t)std::max(ng, 1) * 4));
    if (ng > 0) k_index_count<<<ng, 256, bm_bytes, st>>>(nb, p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_grp_ptr,
                                            p->d_grp_cols, d_cnt, p->d_sub_dim);
    p->launches++;
    std::vector<int32_t> cnt(ng);
    p->h_sub_dim.resize(ng);
    SM_CUDA(cudaMemcpyAsync(cnt.data(), d_cnt, (size_t)ng * 4, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaMemcpyAsync(p->h_sub_dim.data(), p->d_sub_dim, (size_t)ng * 4, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    cudaFree(d_cnt);
    p->h_sub_ptr.assign(ng + 1, 0);
    p->max_sub_blocks = 0;
    for (int i = 0; i < ng; ++i) {
        p->h_sub_ptr[i + 1] = p->h_sub_ptr[i] + cnt[i];
        p->max_sub_blocks = std::max(p->max_sub_blocks, cnt[i]);
    }
    const int64_t tot = p->h_sub_ptr[ng];
    if ((s = upload(&p->d_sub_ptr, p->h_sub_ptr.data(), ng + 1, st))) return s;
    SM_CUDA(cudaMalloc((void**)&p->d_sub_blocks, std::max<int64_t>(tot, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_sub_off, std::max<int64_t>(tot, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_pos, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_off, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_col_grp, (size_t)std::max(nb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_blk_pack, std::max<int64_t>(p->nnzb, 1) * 4));
    SM_CUDA(cudaMalloc((void**)&p->d_gen_width, (size_t)std::max(ng, 1) * 4));
    int32_t* d_err = nullptr;
    SM_CUDA(cudaMalloc((void**)&d_err, 4));
    SM_CUDA(cudaMemsetAsync(d_err, 0, 4, st));
    // pass 2
    if (ng > 0) k_index_fill<<<ng, 256, bm_bytes, st>>>(nb, p->d_blk_size, p->d_colptr, p->d_rowidx, p->d_grp_ptr,
                                           p->d_grp_cols, p->d_sub_ptr, p->d_sub_blocks, p->d_sub_off,
                                           p->d_gen_pos, p->d_gen_off, p->d_blk_pack, p->d_col_grp,
                                           p->d_gen_width, d_err);
    p->launches++;
    int32_t herr = 0;
    SM_CUDA(cudaMemcpyAsync(&herr, d_err, 4, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    cudaFree(d_err);
    SM_CUDA(cudaGetLastError());
    if (herr) return SM_ERR_STRUCTURE;

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
    for (int c = 0; c < nb; ++c) {
        int64_t nc = 0;
        for (int64_t q = p->h_colptr[c]; q < p->h_colptr[c + 1]; ++q) nc += p->h_blk_size[p->h_rowidx[q]];
        n3c += nc * nc * nc;
    }
    I.sum_n3_columns = n3c;
    I.est_speedup = n3 > 0 ? (double)n3c / (double)n3 : 0.0;
    return SM_OK;
}

}  // namespace smb
