// C-ABI entry points (include/submatrix.h): argument checks, plan lifetime, the Newton-Schulz
// host loop, the mu bisection (a8).  Every floating-point step of the path runs in the kernels of
// plan.cu / gather_scatter.cu / ns_sign.cu; the host only sequences launches and compares scalars.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstdio>
#include <cstring>
#include <new>

#include "common.cuh"

namespace smb {
static thread_local char g_cuda_err[512] = "";
void set_cuda_error(cudaError_t e, const char* where) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
}
// A message of the library's own (argument errors that deserve more than a status code): read back through
// sm_last_cuda_error like the CUDA ones.
void set_error_text(const char* msg) { snprintf(g_cuda_err, sizeof(g_cuda_err), "%s", msg); }
}  // namespace smb

using namespace smb;

static void default_options(sm_options_t* o) {
    memset(o, 0, sizeof(*o));
    o->max_iter = 100;
    o->scaling = 1;
    o->early_out = 1;
    o->overshoot = 1.45;
    o->order = 2;
    o->predict = 2;
    o->mu_guess = 1;
    o->mu_start = 1;
    o->rescale = 1;
    o->precision = 0;
    o->check_every = 16;
    o->max_mu_steps = 64;
    o->bisect_iter = 0;
    o->mu_tol = 1e-6;
    o->method = 0;
    o->kT = 0.0;
    o->shard_rank = 0;
    o->shard_world = 1;
}

static sm_status_t validate(int32_t nb, const int32_t* bs, const int64_t* colptr, const int32_t* rowidx,
                            int32_t ng, const int32_t* gp, const int32_t* gc) {
    if (nb < 0 || ng < 0 || (nb > 0 && (!bs || !colptr || !rowidx || !gp || !gc))) return SM_ERR_INVALID_ARG;
    if (nb == 0) return ng == 0 ? SM_OK : SM_ERR_STRUCTURE;
    if (colptr[0] != 0) return SM_ERR_STRUCTURE;
    for (int c = 0; c < nb; ++c) {
        if (bs[c] <= 0 || bs[c] > 4095) return SM_ERR_INVALID_ARG;  // 12-bit block heights (scatter records)
        if (colptr[c + 1] < colptr[c]) return SM_ERR_STRUCTURE;
        bool diag = false;
        for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
            int r = rowidx[p];
            if (r < 0 || r >= nb) return SM_ERR_STRUCTURE;
            if (p > colptr[c] && rowidx[p - 1] >= r) return SM_ERR_STRUCTURE;  // unsorted / duplicate
            if (r == c) diag = true;
        }
        if (!diag) return SM_ERR_STRUCTURE;  // reading A3
    }
    // structural symmetry: (r,c) stored => (c,r) stored
    for (int c = 0; c < nb; ++c)
        for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
            int r = rowidx[p];
            if (r == c) continue;
            const int32_t* b = rowidx + colptr[r];
            const int32_t* e = rowidx + colptr[r + 1];
            if (!std::binary_search(b, e, c)) return SM_ERR_STRUCTURE;
        }
    // groups: a partition of 0..nb-1 (reading A6)
    if (gp[0] != 0 || gp[ng] != nb) return SM_ERR_STRUCTURE;
    std::vector<char> seen(nb, 0);
    for (int g = 0; g < ng; ++g) {
        if (gp[g + 1] <= gp[g]) return SM_ERR_STRUCTURE;  // empty group
        for (int q = gp[g]; q < gp[g + 1]; ++q) {
            int c = gc[q];
            if (c < 0 || c >= nb || seen[c]) return SM_ERR_STRUCTURE;
            seen[c] = 1;
        }
    }
    return SM_OK;
}

extern "C" void sm_plan_destroy(sm_plan_t* p) {
    if (!p) return;
    void* ptrs[] = {p->d_blk_size, p->d_blk_off, p->d_rowidx, p->d_colptr, p->d_val_off, p->d_grp_ptr,
                    p->d_grp_cols, p->d_col_grp, p->d_sub_ptr, p->d_sub_blocks, p->d_sub_off, p->d_sub_dim,
                    p->d_gen_pos, p->d_gen_off, p->d_blk_pack, p->d_gen_width, p->d_gen_rng, p->d_ws_off, p->d_ld, p->d_tiles,
                    p->d_tile_first, p->d_tile_count, p->d_done_iter, p->d_flag, p->d_res, p->d_gersh,
                    p->d_partials, p->d_counters, p->d_sched, p->d_act, p->d_act_cnt, p->d_thin_list, p->d_spec_tiles, p->d_spec_stat, p->d_ne_part, p->d_scalars, p->d_red, p->d_stage_in,
                    p->d_stage_out, p->d_bound, p->d_bound_part, p->d_lz, p->d_tiles32, p->d_ws_off32,
                    p->d_tile_first32, p->d_tile_count32, p->d_partials32, p->d_src_map, p->d_col_rec, p->d_gg, p->d_ctrl, p->d_gl_ptr, p->d_gl,
                    p->d_alpha, p->d_lmin, p->d_lz_rec, p->d_lz_map, p->d_col_val, p->d_eig_ptr, p->d_eig_lam, p->d_eig_w, p->d_eig_sigma, p->d_eig_order,
                    p->d_eig_state};
    for (void* q : ptrs)
        if (q) cudaFree(q);
    if (p->h_pinned) cudaFreeHost(p->h_pinned);
    if (p->h_pinned_d) cudaFreeHost(p->h_pinned_d);
    if (p->h_stats) cudaFreeHost(p->h_stats);
    if (p->h_bound) cudaFreeHost(p->h_bound);
    if (p->h_ctrl) cudaFreeHost(p->h_ctrl);
    if (p->h_lz) cudaFreeHost(p->h_lz);
    for (auto& e : p->ev)
        if (e) cudaEventDestroy(e);
    for (auto& e : p->ev_iter)
        if (e) cudaEventDestroy(e);
    for (auto& e : p->ev_gemm)
        if (e) cudaEventDestroy(e);
    delete p;
}

namespace {
struct PlanGuard {  // destroys a half-built plan on every error path, exceptions included
    sm_plan* p = nullptr;
    ~PlanGuard() { if (p) sm_plan_destroy(p); }
};
sm_status_t plan_create_impl(sm_plan_t** plan, int32_t nb, const int32_t* blk_size, const int64_t* colptr,
                             const int32_t* rowidx, int32_t ngroups, const int32_t* grp_ptr,
                             const int32_t* grp_cols, const sm_options_t* opt, void* cuda_stream);
}  // namespace

extern "C" sm_status_t sm_plan_create(sm_plan_t** plan, int32_t nb, const int32_t* blk_size,
                                      const int64_t* colptr, const int32_t* rowidx, int32_t ngroups,
                                      const int32_t* grp_ptr, const int32_t* grp_cols,
                                      const sm_options_t* opt, void* cuda_stream) {
    if (!plan) return SM_ERR_INVALID_ARG;
    *plan = nullptr;
    try {  // host containers may throw: nothing crosses the C boundary
        return plan_create_impl(plan, nb, blk_size, colptr, rowidx, ngroups, grp_ptr, grp_cols, opt, cuda_stream);
    } catch (const std::bad_alloc&) {
        *plan = nullptr;
        return SM_ERR_ALLOC;
    } catch (...) {
        *plan = nullptr;
        return SM_ERR_INVALID_ARG;
    }
}

namespace {
sm_status_t plan_create_impl(sm_plan_t** plan, int32_t nb, const int32_t* blk_size, const int64_t* colptr,
                             const int32_t* rowidx, int32_t ngroups, const int32_t* grp_ptr,
                             const int32_t* grp_cols, const sm_options_t* opt, void* cuda_stream) {
    const auto t_begin = std::chrono::steady_clock::now();
    sm_status_t s = validate(nb, blk_size, colptr, rowidx, ngroups, grp_ptr, grp_cols);
    if (s) return s;
    sm_plan* p = new (std::nothrow) sm_plan();
    if (!p) return SM_ERR_ALLOC;
    PlanGuard guard;
    guard.p = p;
    if (opt) p->opt = *opt; else default_options(&p->opt);
    if (p->opt.max_iter <= 0) p->opt.max_iter = 100;
    if (p->opt.check_every <= 0) p->opt.check_every = 1;
    if (p->opt.max_mu_steps <= 0) p->opt.max_mu_steps = 64;
    if (p->opt.max_mu_steps > 64) p->opt.max_mu_steps = 64;
    if (!(p->opt.mu_tol > 0)) p->opt.mu_tol = 1e-6;
    if (!(p->opt.overshoot >= 1.0)) p->opt.overshoot = 1.0;     // zero-initialised struct: no overshoot
    if (p->opt.overshoot > 1.5) p->opt.overshoot = 1.5;         // f(x) = x(3 - x^2)/2 keeps [1, 1.5] inside [0.56, 1]
    if (p->opt.order == 0) p->opt.order = 2;                    // zero-initialised struct: Eq.(11)
    if (p->opt.order != 2 && p->opt.order != 3) return SM_ERR_INVALID_ARG;
    if (p->opt.order == 3) {
        if (p->opt.precision != 0) return SM_ERR_INVALID_ARG;
        p->opt.overshoot = 1.0;  // Eq.(19)'s map is increasing beyond 1: eigenvalues of X0 must not exceed 1
    }
    if (p->opt.precision < 0 || p->opt.precision > 4 || p->opt.scaling < 0 || p->opt.scaling > 1) return SM_ERR_INVALID_ARG;
    if (p->opt.method < 0 || p->opt.method > 1 || !(p->opt.kT >= 0.0)) return SM_ERR_INVALID_ARG;
    if (p->opt.method == 1 && (p->opt.precision != 0 || p->opt.order != 2)) return SM_ERR_INVALID_ARG;
    p->nb = nb; p->ngroups = ngroups; p->nnzb = nb ? colptr[nb] : 0;
    p->h_blk_size.assign(blk_size, blk_size + nb);
    p->h_colptr.assign(colptr, colptr + nb + 1);
    p->h_rowidx.assign(rowidx, rowidx + p->nnzb);
    p->h_grp_ptr.assign(grp_ptr, grp_ptr + ngroups + 1);
    p->h_grp_cols.assign(grp_cols, grp_cols + nb);
    // keep only this rank's contiguous chunk of groups (the pattern stays whole)
    const int world = std::max(p->opt.shard_world, 1), rank = p->opt.shard_rank;
    const int32_t ngroups_total = ngroups;
    if (rank < 0 || rank >= world) return SM_ERR_INVALID_ARG;
    int shard_gb = 0, shard_ge = ngroups;
    int64_t shard_vb = -1, shard_ve = -1;
    if (world > 1) {
        if (world > ngroups) return SM_ERR_INVALID_ARG;
        std::vector<int32_t> dims(ngroups), rows;
        for (int g = 0; g < ngroups; ++g) {  // n_i of every group: sorted union of its columns' row lists (host, plan time)
            rows.clear();
            for (int q = grp_ptr[g]; q < grp_ptr[g + 1]; ++q)
                rows.insert(rows.end(), rowidx + colptr[grp_cols[q]], rowidx + colptr[grp_cols[q] + 1]);
            std::sort(rows.begin(), rows.end());
            rows.erase(std::unique(rows.begin(), rows.end()), rows.end());
            int32_t n = 0;
            for (int32_t r : rows) n += blk_size[r];
            dims[g] = n;
        }
        std::vector<int32_t> first(world + 1);
        if ((s = sm_partition_groups(ngroups, dims.data(), world, first.data()))) return s;
        shard_gb = first[rank]; shard_ge = first[rank + 1];
        std::vector<int32_t> gp(shard_ge - shard_gb + 1), gc(grp_cols + grp_ptr[shard_gb], grp_cols + grp_ptr[shard_ge]);
        for (int g = shard_gb; g <= shard_ge; ++g) gp[g - shard_gb] = grp_ptr[g] - grp_ptr[shard_gb];
        p->h_grp_ptr.swap(gp);
        p->h_grp_cols.swap(gc);
        p->ngroups = ngroups = shard_ge - shard_gb;
        bool contiguous = !p->h_grp_cols.empty();
        for (size_t k = 1; k < p->h_grp_cols.size(); ++k) contiguous = contiguous && p->h_grp_cols[k] == p->h_grp_cols[k - 1] + 1;
        if (contiguous) {  // value offsets of the first owned column and of the one after the last
            std::vector<int64_t> cv(nb + 1, 0);
            for (int c = 0; c < nb; ++c) {
                int64_t e = 0;
                for (int64_t q = colptr[c]; q < colptr[c + 1]; ++q) e += blk_size[rowidx[q]];
                cv[c + 1] = cv[c] + e * blk_size[c];
            }
            shard_vb = cv[p->h_grp_cols.front()];
            shard_ve = cv[p->h_grp_cols.back() + 1];
        }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        set_cuda_error(cudaGetLastError(), "cudaGetDevice");
        return SM_ERR_CUDA;
    }
    s = build_index_device(p, st);
    if (s) return s;
    if (p->opt.precision != 0 && (s = build_tf32_tables(p, st))) return s;
    if (p->opt.order == 3) p->info.workspace_bytes = p->info.workspace_bytes / 3 * 4;  // + W of Eq.(19)
    // per-evaluation state
    const int ng = std::max(ngroups, 1);
    auto A = [&](void** d, size_t bytes) { return cudaMalloc(d, std::max<size_t>(bytes, 8)); };
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = A((void**)&p->d_done_iter, (size_t)ng * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_flag, (size_t)ng * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_res, (size_t)ng * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_gersh, (size_t)ng * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_alpha, (size_t)ng * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_lmin, (size_t)ng * 8);
    if (e == cudaSuccess) e = A((void**)&p->d_partials, (size_t)p->n_tiles * 4 * 8);
    if (e == cudaSuccess) e = A((void**)&p->d_counters, (size_t)(p->opt.max_iter + 2) * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_sched, (size_t)(p->opt.max_iter + 2) * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_act, (size_t)std::max<int64_t>(p->n_tiles, 1) * 4 * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_act_cnt, (size_t)(p->opt.max_iter + 3) * 24);
    if (e == cudaSuccess) e = A((void**)&p->d_thin_list, (size_t)std::max(ng, 1) * 4 * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_spec_tiles, (size_t)std::max<int64_t>(p->n_tiles, 1) * 4);
    if (e == cudaSuccess) e = A((void**)&p->d_spec_stat, 8);
    if (e == cudaSuccess) e = cudaMemset(p->d_spec_stat, 0, 8);
    if (e == cudaSuccess) e = A((void**)&p->d_ne_part, (size_t)ng * 8);
    if (e == cudaSuccess) e = A((void**)&p->d_scalars, 8 * 8);
    if (e == cudaSuccess) e = A((void**)&p->d_red, 4096 * 8);
    if (e == cudaSuccess) e = A((void**)&p->d_bound, (size_t)(p->opt.max_iter + 2) * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_bound_part, (size_t)std::max(nb, 1) * 16);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&p->h_bound, (size_t)(p->opt.max_iter + 2) * 16);
    if (e == cudaSuccess) e = A((void**)&p->d_ctrl, 64);
    if (e == cudaSuccess) e = cudaMemset(p->d_ctrl, 0, 64);
    if (e == cudaSuccess) e = cudaMallocHost(&p->h_ctrl, 64);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&p->h_lz, 68 * 8);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&p->h_pinned, (size_t)(p->opt.max_iter + 2) * 4);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&p->h_pinned_d, 8 * 8);
    for (auto& ev : p->ev)
        if (e == cudaSuccess) e = cudaEventCreate(&ev);
    for (auto& ev : p->ev_iter)
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        set_cuda_error(e, "plan state allocation");
        return e == cudaErrorMemoryAllocation ? SM_ERR_ALLOC : SM_ERR_CUDA;
    }
    // gather launch shape: member tables + hash table of S_i + position map + block map of a chunk
    // of mc member columns (as many as fit ~24 KB: measured best, occupancy beats fewer chunks)
    {
        const int msb = (std::max(p->max_sub_blocks, 1) + 1) & ~1;
        const int tile_ld = (p->info.dim_max + LD_ALIGN + 3) & ~3;
        const int mpad = (msb + 2 + 15) & ~15;  // + the "no member" column of padding positions; 32-byte rows
        int hs = 32, shift = 27;
        while (hs < 2 * msb) { hs <<= 1; --shift; }
        const size_t fixed = (size_t)msb * 8 + (size_t)tile_ld * 8 + (size_t)hs * 8 + (size_t)(msb + 2) * 4 +
                             (size_t)msb * 4;
        // a block-map entry is the value offset of a block inside its block column: 16 bits when
        // every block column holds fewer than 65535 values (halves the table), else 32 bits
        int64_t max_col_elems = 0;
        for (int c = 0; c < nb; ++c) {
            int64_t elems = 0;
            for (int64_t q = colptr[c]; q < colptr[c + 1]; ++q) elems += blk_size[rowidx[q]];
            max_col_elems = std::max(max_col_elems, elems * blk_size[c]);
        }
        if (max_col_elems >= (int64_t)UINT32_MAX) return SM_ERR_INVALID_ARG;
        const int esz = max_col_elems < 65535 ? 2 : 4;
        p->gather_map16 = esz == 2;
        auto bytes = [&](int mc) { return fixed + (((size_t)mc * mpad * esz + 15) & ~(size_t)15); };
        int mc = msb;
        const size_t want = 24 * 1024, budget = 200 * 1024;
        if (bytes(mc) > want) mc = (int)std::max<int64_t>(((int64_t)want - (int64_t)fixed) / (mpad * esz), 16);
        mc = std::min(mc, msb);
        while (mc > 1 && bytes(mc) > budget) mc >>= 1;
        if (bytes(mc) > budget) return SM_ERR_INVALID_ARG;
        p->gather_warps = 8; p->gather_tile_ld = tile_ld; p->gather_mpad = mpad; p->gather_mc = mc;
        p->gather_msb = msb; p->gather_hash_size = hs; p->gather_hash_shift = shift;
        p->gather_smem = bytes(mc);
        // CTAs per submatrix: enough CTAs to fill the GPU a few times over
        int split = 1;
        const int64_t want_ctas = (int64_t)p->num_sms * 12;
        while ((int64_t)ngroups * split < want_ctas && split * 8 * 4 < p->info.dim_max) ++split;
        p->gather_split = std::max(split, 1);
    }
    p->info.shard_group_begin = shard_gb; p->info.shard_group_end = shard_ge;
    p->info.shard_val_begin = world > 1 ? shard_vb : 0; p->info.shard_val_end = world > 1 ? shard_ve : p->nnz;
    p->info.ngroups_total = ngroups_total;
    p->info.ms_plan_create =
        std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    guard.p = nullptr;
    *plan = p;
    return SM_OK;
}
}  // namespace

// PAPER.md L235 (reading A19): consecutive chunks, a rank takes the next submatrix while its load so far is
// below sum n^3 / world and every later rank can still get one; the last rank takes the rest.
extern "C" sm_status_t sm_partition_groups(int32_t ngroups, const int32_t* sub_dim, int32_t world, int32_t* first) {
    if (ngroups < 0 || world < 1 || !first || (ngroups > 0 && !sub_dim) || world > std::max(ngroups, 1)) return SM_ERR_INVALID_ARG;
    typedef unsigned __int128 u128;  // exact: n^3 sums of any realistic size, compared as load * world < total
    u128 total = 0;
    for (int i = 0; i < ngroups; ++i) total += (u128)sub_dim[i] * (u128)sub_dim[i] * (u128)sub_dim[i];
    int i = 0;
    for (int r = 0; r < world; ++r) {
        first[r] = i;
        if (r == world - 1) { i = ngroups; break; }
        u128 load = 0;
        const int last_allowed = ngroups - (world - 1 - r);  // leave one submatrix for every later rank
        bool took = false;
        while (i < last_allowed && (!took || load * (u128)world < total)) {
            load += (u128)sub_dim[i] * (u128)sub_dim[i] * (u128)sub_dim[i];
            ++i;
            took = true;
        }
    }
    first[world] = ngroups;
    return SM_OK;
}

extern "C" sm_status_t sm_plan_set_allreduce(sm_plan_t* p, sm_allreduce_fn fn, void* ctx) {
    if (!p) return SM_ERR_INVALID_ARG;
    p->allreduce = fn;
    p->allreduce_ctx = ctx;
    return SM_OK;
}

extern "C" sm_status_t sm_plan_query(const sm_plan_t* p, sm_plan_info_t* out) {
    if (!p || !out) return SM_ERR_INVALID_ARG;
    *out = p->info;
    return SM_OK;
}

extern "C" sm_status_t sm_plan_export_index(const sm_plan_t* p, int64_t* sub_ptr, int32_t* sub_blocks,
                                            int32_t* sub_off, int32_t* sub_dim, int32_t* gen_pos) {
    if (!p) return SM_ERR_INVALID_ARG;
    const int ng = p->ngroups;
    const int64_t tot = p->info.sum_sub_blocks;
    if (sub_ptr) memcpy(sub_ptr, p->h_sub_ptr.data(), (size_t)(ng + 1) * 8);
    if (sub_blocks && tot) SM_CUDA(cudaMemcpy(sub_blocks, p->d_sub_blocks, (size_t)tot * 4, cudaMemcpyDeviceToHost));
    if (sub_off && tot) SM_CUDA(cudaMemcpy(sub_off, p->d_sub_off, (size_t)tot * 4, cudaMemcpyDeviceToHost));
    if (sub_dim && ng) SM_CUDA(cudaMemcpy(sub_dim, p->d_sub_dim, (size_t)ng * 4, cudaMemcpyDeviceToHost));
    if (gen_pos && p->nb) SM_CUDA(cudaMemcpy(gen_pos, p->d_gen_pos, (size_t)p->nb * 4, cudaMemcpyDeviceToHost));
    return SM_OK;
}

extern "C" sm_status_t sm_set_timing(sm_plan_t* p, int32_t enable) {
    if (!p) return SM_ERR_INVALID_ARG;
    p->timing = enable ? 1 : 0;
    return SM_OK;
}

extern "C" int64_t sm_launch_count(const sm_plan_t* p) { return p ? p->launches : 0; }

namespace {
struct Bufs {
    double *b0, *b1, *y, *w;
};
sm_status_t carve(const sm_plan* p, void* ws, size_t bytes, Bufs* b) {
    if (bytes < p->info.workspace_bytes) return SM_ERR_WORKSPACE_TOO_SMALL;
    if (!ws && p->info.workspace_bytes) return SM_ERR_INVALID_ARG;
    if (((uintptr_t)ws & 255) != 0) return SM_ERR_INVALID_ARG;
    const size_t buf = p->info.workspace_bytes / (p->opt.order == 3 ? 4 : 3);
    b->b0 = (double*)ws;
    b->b1 = (double*)((char*)ws + buf);
    b->y = (double*)((char*)ws + 2 * buf);
    b->w = p->opt.order == 3 ? (double*)((char*)ws + 3 * buf) : nullptr;
    return SM_OK;
}

sm_status_t reset_state(sm_plan* p, cudaStream_t st) {
    const int ng = std::max(p->ngroups, 1);
    SM_CUDA(cudaMemsetAsync(p->d_done_iter, 0xff, (size_t)ng * 4, st));
    SM_CUDA(cudaMemsetAsync(p->d_flag, 0, (size_t)ng * 4, st));
    SM_CUDA(cudaMemsetAsync(p->d_counters, 0, (size_t)(p->opt.max_iter + 2) * 4, st));
    SM_CUDA(cudaMemsetAsync(p->d_sched, 0, (size_t)(p->opt.max_iter + 2) * 16, st));
    SM_CUDA(cudaMemsetAsync(p->d_act_cnt, 0, (size_t)(p->opt.max_iter + 3) * 24, st));
    SM_CUDA(cudaMemsetAsync(p->d_ctrl, 0, sizeof(EvalCtrl), st));
    p->cur_k = 0;
    p->ev_gemm_n = 0;
    return SM_OK;
}

// Steering of one bisection evaluation (reading A11c): the evaluation may stop as soon as the bound
// of k_nelec_bound proves on which side of n_target the converged n_elec lies.
struct Steer {
    double n_target = 0.0, tol_n = 0.0, slack = 0.0;
    int decided = 0;        // out: +1 n_elec > n_target + tol_n proven, -1 the opposite, 0 not decided
    int k = -1;             // out: iterate the decision was taken on
    double ne = 0.0, err = 0.0;  // out: n_elec(X_k) and its bound
};

// One iteration's launches on the path the plan was created for (FP64 DMMA, or TF32 tcgen05).
sm_status_t launch_pair(sm_plan* p, int k, double eps, int last, const Bufs& b, cudaStream_t st, int which) {
    if (p->opt.precision != 0) return launch_ns_pair_tf32(p, k, eps, last, b.b0, b.b1, b.y, st, which);
    return launch_ns_pair(p, k, eps, last, b.b0, b.b1, b.y, st, which, b.w);
}

// Newton-Schulz host loop: iterations k = cur_k .. k_end-1.  Iteration k = MODE 0 (Y = X_k^2, residual)
// + decision [+ steering bound] + k_eval_ctrl + update (X_{k+1}); at k == max_iter only the decision
// is recorded.  Every stop decision -- all submatrices converged, or a proven steering direction --
// is taken ON THE DEVICE (EvalCtrl): once it is set, the remaining launches of the evaluation are
// empty.  The host therefore enqueues `check_every` iterations ahead and only then reads the
// control block: the GPU never waits for the host, and a stalled host thread costs nothing while
// work is queued.  Returns with *all_done = 1 if every submatrix has stopped.
sm_status_t ns_loop(sm_plan* p, const Bufs& b, double eps, int k_end, int* all_done, int* launched,
                    cudaStream_t st, Steer* steer = nullptr) {
    *all_done = 0;
    if (p->ngroups == 0) { *all_done = 1; return SM_OK; }
    const int max_iter = p->opt.max_iter, upd = p->opt.order == 3 ? 2 : 1;
    const EvalCtrl* hc = reinterpret_cast<const EvalCtrl*>(p->h_ctrl);
    const int k_begin = p->cur_k;
    const double margin = steer ? steer->slack + steer->tol_n : 0.0;
    p->half_iter = 0;
    int k = k_begin, since = 0;
    bool stopped = false;
    sm_status_t s;
    // how far to enqueue before the first look at the control block: what the previous evaluation of this plan
    // needed, plus one (launches behind the device-side stop are empty but not free), at most check_every
    int batch = p->opt.check_every;
    if (p->last_eval_iters > 0) batch = std::min(batch, p->last_eval_iters + 1);
    for (; k < k_end && k <= max_iter && !stopped; ++k) {
        const int last = k == max_iter ? 1 : 0;
        if ((s = launch_pair(p, k, eps, last, b, st, 1))) return s;
        const int steer_k = (steer && k >= 1) ? 1 : 0;
        if (steer_k && (s = launch_nelec_bound(p, k, b.b0, b.b1, b.y, st))) return s;
        if ((s = launch_eval_ctrl(p, k, steer_k, steer ? steer->n_target : 0.0, margin, st))) return s;
        if (!last && (s = launch_pair(p, k, eps, 0, b, st, 2))) return s;
        if (++since >= batch || last || k == k_end - 1) {
            SM_CUDA(cudaMemcpyAsync(p->h_ctrl, p->d_ctrl, sizeof(EvalCtrl), cudaMemcpyDeviceToHost, st));
            SM_CUDA(cudaStreamSynchronize(st));
            since = 0;
            batch = std::min(p->opt.check_every, 4);  // the estimate was short: continue in small batches
            stopped = hc->stop != 0;
        }
    }
    if (stopped) {
        const int ks = hc->k_stop;
        if (hc->stop == 1) p->last_eval_iters = ks - k_begin + 1;  // a converged evaluation: the next one will be alike
        p->cur_k = ks;
        (*launched) += (ks - k_begin + 1) + (ks - k_begin) * upd;  // launches that did work; later ones were empty
        if (hc->stop == 1) {
            *all_done = 1;
        } else {
            p->half_iter = 1;  // MODE 0 of iteration ks ran, its update did not: X_ks in buf[ks & 1], not converged
            if (steer) { steer->decided = hc->decided; steer->k = ks; steer->ne = hc->ne; steer->err = hc->err; }
        }
        return SM_OK;
    }
    // iteration cap reached with active submatrices: they have received k updates, X lives in buf[k & 1]
    (*launched) += (k - k_begin) * (1 + upd);
    p->cur_k = std::min(k, max_iter);
    return SM_OK;
}

sm_status_t collect_stats(sm_plan* p, sm_stats_t* stats, int* not_conv, cudaStream_t st) {
    const int ng = p->ngroups;
    if (!p->h_stats) SM_CUDA(cudaMallocHost((void**)&p->h_stats, (size_t)std::max(ng, 1) * 24));
    const double* res = reinterpret_cast<const double*>(p->h_stats);                       // [2 ng]
    const int32_t* di = reinterpret_cast<const int32_t*>(p->h_stats + (size_t)ng * 16);   // [ng]
    const int32_t* fl = di + ng;                                                           // [ng]
    if (ng) {
        SM_CUDA(cudaMemcpyAsync((void*)di, p->d_done_iter, (size_t)ng * 4, cudaMemcpyDeviceToHost, st));
        SM_CUDA(cudaMemcpyAsync((void*)fl, p->d_flag, (size_t)ng * 4, cudaMemcpyDeviceToHost, st));
        SM_CUDA(cudaMemcpyAsync((void*)res, p->d_res, (size_t)ng * 16, cudaMemcpyDeviceToHost, st));
    }
    SM_CUDA(cudaMemcpyAsync(p->h_pinned_d, p->d_scalars, 8, cudaMemcpyDeviceToHost, st));
    int32_t* h_spec = reinterpret_cast<int32_t*>(p->h_pinned_d + 6);  // two ints behind the scalars that are read back
    if (p->d_spec_stat) SM_CUDA(cudaMemcpyAsync(h_spec, p->d_spec_stat, 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    if (p->d_spec_stat) {
        // two-step exit (A9c): a failed certificate costs one product.  If the last evaluation's speculations mostly
        // failed, the estimate of k_ns_decide does not fit this input: do not try for the next 8 evaluations.
        const int ok = h_spec[0] - p->h_spec_prev[0], fail = h_spec[1] - p->h_spec_prev[1];
        p->h_spec_prev[0] = h_spec[0]; p->h_spec_prev[1] = h_spec[1];
        if (p->spec_pause > 0) --p->spec_pause;
        else if (fail > ok && fail >= 16) p->spec_pause = 8;
    }
    int imin = INT32_MAX, imax = 0, nc = 0, n_pred = 0, n_two = 0;
    double rmax = 0.0;
    int64_t sin3 = 0, symf = 0;
    for (int i = 0; i < ng; ++i) {
        int it = di[i] >= 0 ? di[i] : p->cur_k;
        if (di[i] < 0 || fl[i] == 1) ++nc;  // flag 2 = converged by the predicted exit
        imin = std::min(imin, it);
        imax = std::max(imax, it);
        int slot = di[i] >= 0 ? (di[i] & 1) : ((std::max(p->cur_k, 1) - 1) & 1);
        double r = res[(size_t)slot * ng + i];
        if (r == r) rmax = std::max(rmax, r); else rmax = INFINITY;
        int64_t n = p->h_sub_dim[i];
        // executed symmetric products: stopped at iteration it: one X^2 per tested iterate (it + 1)
        // and one update per iteration (it); still active after cur_k launch pairs: 2 cur_k (+1 if a steering decision came between the two modes)
        const int64_t ppi = p->opt.order == 3 ? 3 : 2;  // products per iteration (Eq.(11): 2, Eq.(19): 3)
        // flag 3 (two-step exit, reading A9c, it = k + 2): k + 1 squarings, k updates, the certificate product, and three
        // thin products instead of the two last updates and the last squaring
        const int64_t prods = di[i] >= 0 ? (fl[i] == 3 ? ppi * it - 2 : ppi * it + (fl[i] == 2 ? 0 : 1))
                                         : ppi * (int64_t)p->cur_k + p->half_iter;
        sin3 += prods * n * n * n;
        symf += prods * n * n * (n + 1);
        // predicted exit (flag 2): its last update only computed the tiles of the generating rows
        if (fl[i] == 2 && p->opt.order == 2 && p->opt.precision == 0) symf += p->h_final_flop[i] - n * n * (n + 1);
        if (fl[i] == 3) symf += 3 * p->h_final_flop[i];
        if (fl[i] == 2) ++n_pred;
        if (fl[i] == 3) ++n_two;
    }
    *not_conv = nc;
    if (stats) {
        stats->iter_min = ng ? imin : 0;
        stats->iter_max = imax;
        stats->not_converged = nc;
        stats->max_residual = rmax;
        stats->n_elec = p->h_pinned_d[0];
        stats->sum_iter_n3 = sin3;
        stats->tot_sym_flop = symf;  // per evaluation here; callers accumulate
        stats->exits_predicted = n_pred;
        stats->exits_two_step = n_two;
    }
    return SM_OK;
}

// Spectral scale of the evaluation at mu (option scaling = 1): s_i = min(Gershgorin_i, cap(mu)) / overshoot.
sm_status_t ensure_bounds(sm_plan* p, const double* d_in, cudaStream_t st) {
    if (p->opt.scaling != 1 || p->lz_valid) return SM_OK;
    sm_status_t s = launch_lanczos_bounds(p, d_in, st);
    if (s) return s;
    p->lz_valid = 1;
    return SM_OK;
}
sm_status_t apply_scaling(sm_plan* p, double mu, cudaStream_t st) {
    p->resc_eval = 0;
    if (p->opt.scaling != 1) return SM_OK;
    // a Lanczos run that broke down is not used (cap = 0: the rigorous Gershgorin bounds alone, reading A8)
    const double cap = p->lz_ok ? std::max(std::fabs(p->lz_hi - mu), std::fabs(p->lz_lo - mu)) : 0.0;
    // reading A8b: distance from mu to the nearest Ritz value of the Lanczos run = estimate of the smallest
    // eigenvalue modulus of K~ - mu I (Ritz values sit inside the bands, so it errs on the large side)
    // Only where mu sits in a hole of the Ritz spectrum (l_0 >= 0.05): inside a band the evaluation is most
    // likely a steering one, and there the rescaling, which folds the top of the spectrum down onto l_k,
    // loosens the bound of reading A11c (measured: 4 instead of 2 iterations until the side is proven).
    double ell = 0.0;
    if (p->opt.rescale != 0 && p->opt.order == 2 && p->opt.precision == 0 && p->lz_nodes > 0 && cap > 0.0) {
        ell = INFINITY;
        for (int j = 0; j < p->lz_nodes; ++j) ell = std::min(ell, std::fabs(p->h_lz[2 + j] - mu));
        p->resc_eval = (ell >= 0.05 * cap) ? 1 : 0;
    }
    return launch_apply_scale(p, cap, p->opt.overshoot, ell, st);
}

// One sign evaluation at fixed mu: gather -> NS loop (up to iter_cap iterations) -> n_elec.
// With `steer` the loop may end early on a proven direction (steer->decided != 0): the workspace
// is then NOT converged and stats->n_elec is the last iterate's count.
sm_status_t evaluate(sm_plan* p, const double* d_in, double mu, double eps, const Bufs& b, int iter_cap,
                     sm_stats_t* stats, int* not_conv, cudaStream_t st, Steer* steer = nullptr) {
    sm_status_t s;
    int launched = 0, all_done = 0;
    if ((s = ensure_bounds(p, d_in, st))) return s;  // once per call, outside the gather timing
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[0], st));
    if ((s = reset_state(p, st))) return s;
    if ((s = launch_gather(p, d_in, mu, b.b0, st))) return s;
    if ((s = apply_scaling(p, mu, st))) return s;
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[1], st));
    const bool reduced = p->opt.precision != 0;
    if (reduced && (s = launch_to_f32(p, b.b0, b.b1, st))) return s;  // X0 = (a_i - mu I)/s_i in FP32
    if ((s = ns_loop(p, b, eps, iter_cap, &all_done, &launched, st, reduced ? nullptr : steer))) return s;
    if (reduced && (s = launch_to_f64(p, b.b0, b.b1, b.y, st))) return s;  // result back in buf0, FP64 layout
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[2], st));
    if ((s = launch_nelec(p, b.b0, reduced ? b.b0 : b.b1, st))) return s;
    if ((s = collect_stats(p, stats, not_conv, st))) return s;
    if (p->allreduce) {  // sharded plan: global electron count and non-convergence count (same on every rank)
        double v[2] = {p->h_pinned_d[0], (double)*not_conv};
        p->allreduce(p->allreduce_ctx, v, 2);
        p->h_pinned_d[0] = v[0];
        *not_conv = (int)(v[1] + 0.5);
        if (stats) { stats->n_elec = v[0]; stats->not_converged = *not_conv; }
    }
    if (stats) {
        if (steer && steer->decided) stats->n_elec = steer->ne;
        stats->iterations = launched / (p->opt.order == 3 ? 3 : 2);
        stats->gemm_launches = launched;
        stats->mu = mu;
        if (p->timing) {
            cudaEventElapsedTime(&stats->ms_gather, p->ev[0], p->ev[1]);
            cudaEventElapsedTime(&stats->ms_sign, p->ev[1], p->ev[2]);
            float g = 0.f;  // the product launches alone (event pairs recorded by launch_ns_pair)
            for (int i = 0; i + 1 < p->ev_gemm_n; i += 2) {
                float t = 0.f;
                if (cudaEventElapsedTime(&t, p->ev_gemm[i], p->ev_gemm[i + 1]) == cudaSuccess) g += t;
            }
            stats->ms_gemm = g;
        }
        stats->tot_ms_gemm = stats->ms_gemm;
        stats->tot_sum_iter_n3 = stats->sum_iter_n3;
        stats->tot_gemm_launches = launched;
        stats->tot_evaluations = 1;
        stats->tot_ms_gather = stats->ms_gather;
        stats->tot_ms_sign = stats->ms_sign;
        if (p->opt.scaling == 1 && p->lz_ok) { stats->spec_lo = p->lz_lo; stats->spec_hi = p->lz_hi; }
    }
    return SM_OK;
}

sm_status_t do_scatter(sm_plan* p, const Bufs& b, double* d_out, sm_stats_t* stats, cudaStream_t st) {
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[3], st));
    sm_status_t s = launch_scatter(p, 0, b.b0, p->opt.precision != 0 ? b.b0 : b.b1, d_out, st);
    if (s) return s;
    if (p->timing) {
        SM_CUDA(cudaEventRecord(p->ev[4], st));
        SM_CUDA(cudaEventSynchronize(p->ev[4]));
        if (stats) {
            cudaEventElapsedTime(&stats->ms_scatter, p->ev[3], p->ev[4]);
            cudaEventElapsedTime(&stats->ms_total, p->ev[0], p->ev[4]);
        }
    }
    return SM_OK;
}

// Eigendecomposition path (option method = 1, eig.cu): decomposition + its statistics.
sm_status_t eig_decompose(sm_plan* p, const double* d_in, const Bufs& b, sm_stats_t* stats, int* not_conv,
                          cudaStream_t st) {
    sm_status_t s;
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[0], st));
    if ((s = reset_state(p, st))) return s;
    if ((s = launch_eig_decompose(p, d_in, b.b0, b.b1, st))) return s;
    if (p->timing) SM_CUDA(cudaEventRecord(p->ev[2], st));
    const int ng = p->ngroups;
    std::vector<int32_t> state((size_t)2 * ng + 2, 0);
    if (ng) SM_CUDA(cudaMemcpyAsync(state.data(), p->d_eig_state, (size_t)2 * ng * 4, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    int smin = INT32_MAX, smax = 0, nc = 0;
    for (int i = 0; i < ng; ++i) {
        smin = std::min(smin, state[i]);
        smax = std::max(smax, state[i]);
        nc += state[ng + i] != 0;
    }
    if (p->allreduce) {
        double v[1] = {(double)nc};
        p->allreduce(p->allreduce_ctx, v, 1);
        nc = (int)(v[0] + 0.5);
    }
    *not_conv = nc;
    if (stats) {
        stats->iter_min = ng ? smin : 0;
        stats->iter_max = smax;
        stats->iterations = smax;
        stats->not_converged = nc;
        stats->tot_evaluations = 1;
        if (p->timing) {
            cudaEventElapsedTime(&stats->ms_sign, p->ev[0], p->ev[2]);
            stats->tot_ms_sign = stats->ms_sign;
        }
    }
    return SM_OK;
}

sm_status_t eig_count(sm_plan* p, double mu, double kT, double* ne, cudaStream_t st) {
    if (p->eig_total == 0) {  // a shard without basis functions still takes part in the sum
        double v = 0.0;
        if (p->allreduce) p->allreduce(p->allreduce_ctx, &v, 1);
        if (ne) *ne = v;
        return SM_OK;
    }
    sm_status_t s = launch_eig_nelec(p, mu, kT, st);
    if (s) return s;
    SM_CUDA(cudaStreamSynchronize(st));
    if (p->allreduce) p->allreduce(p->allreduce_ctx, p->h_pinned_d, 1);
    if (ne) *ne = p->h_pinned_d[0];
    return SM_OK;
}

// Algorithm 1 as written (L272-276) on the stored decompositions: the mu loop costs one reduction over
// (lambda, w) per step and no sign evaluation (L266).  Update rule = reading A11: step 0 at the caller's mu,
// midpoint bisection inside the Gershgorin interval of K~, same stopping rules as the Newton-Schulz path.
sm_status_t density_matrix_eig(sm_plan* p, const double* d_in, double n_target, double tol_n, double* mu_inout,
                               double* d_out, const Bufs& b, sm_stats_t* S, cudaStream_t st) {
    sm_status_t s;
    int nc = 0;
    if ((s = launch_gersh_global(p, d_in, st))) return s;  // bracket; read after the next synchronisation
    if ((s = eig_decompose(p, d_in, b, S, &nc, st))) return s;
    double lo = p->h_pinned_d[4], hi = p->h_pinned_d[5];
    S->bracket_lo = lo; S->bracket_hi = hi;
    S->mu_guess = NAN;
    const double kT = p->opt.kT;
    double mu = *mu_inout, best_mu = mu, best_g = INFINITY, best_ne = 0.0;
    int steps = 0;
    bool accepted = false;
    for (; steps < p->opt.max_mu_steps;) {
        double ne = 0.0;
        if ((s = eig_count(p, mu, kT, &ne, st))) return s;
        const double g = ne - n_target;
        S->mu_trace[steps] = mu;
        S->ne_trace[steps] = ne;
        S->ne_err_trace[steps] = 0.0;
        S->iter_trace[steps] = 0;
        if (std::fabs(g) < std::fabs(best_g)) { best_g = g; best_mu = mu; best_ne = ne; }
        ++steps;
        if (std::fabs(g) <= tol_n) { accepted = true; break; }
        if (g < 0) lo = std::max(lo, mu); else hi = std::min(hi, mu);
        if (hi - lo <= p->opt.mu_tol) break;
        mu = 0.5 * (lo + hi);
    }
    S->mu = best_mu;
    S->mu_steps = steps;
    S->n_elec = best_ne;
    *mu_inout = best_mu;
    if (d_out) {
        if ((s = launch_eig_density(p, best_mu, kT, b.b0, b.b1, st))) return s;
        if ((s = do_scatter(p, b, d_out, S, st))) return s;
    }
    SM_CUDA(cudaStreamSynchronize(st));
    if (!accepted) return SM_WARN_MU_NOT_CONVERGED;
    return nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
}

sm_status_t ensure_stage(sm_plan* p) {
    const size_t bytes = std::max<size_t>((size_t)p->nnz * 8, 8);
    if (!p->d_stage_in) SM_CUDA(cudaMalloc((void**)&p->d_stage_in, bytes));
    if (!p->d_stage_out) SM_CUDA(cudaMalloc((void**)&p->d_stage_out, bytes));
    return SM_OK;
}
}  // namespace

extern "C" sm_status_t sm_sign_execute(sm_plan_t* p, const double* d_vals_in, double mu, double eps,
                                       double* d_vals_out, void* d_workspace, size_t workspace_bytes,
                                       sm_stats_t* stats, void* cuda_stream) {
    if (!p || (!d_vals_in && p->nnz) || !(eps > 0.0) || !(mu == mu)) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    if (stats) memset(stats, 0, sizeof(*stats));
    int nc = 0;
    if (p->opt.method == 1) {  // Eq.(17): decomposition, then f(Lambda - mu)
        if ((s = eig_decompose(p, d_vals_in, b, stats, &nc, st))) return s;
        if ((s = eig_count(p, mu, p->opt.kT, stats ? &stats->n_elec : nullptr, st))) return s;
        if (d_vals_out) {
            if ((s = launch_eig_density(p, mu, p->opt.kT, b.b0, b.b1, st))) return s;
            if ((s = do_scatter(p, b, d_vals_out, stats, st))) return s;
        }
        if (stats) { stats->mu = mu; stats->mu_steps = 1; }
        return nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
    }
    p->lz_valid = 0;  // the values may have changed since the last call
    if ((s = evaluate(p, d_vals_in, mu, eps, b, p->opt.max_iter + 1, stats, &nc, st))) return s;
    if (d_vals_out && (s = do_scatter(p, b, d_vals_out, stats, st))) return s;
    if (stats) stats->mu_steps = 1;
    return nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
}

extern "C" sm_status_t sm_gather(sm_plan_t* p, const double* d_vals_in, double mu, void* d_workspace,
                                 size_t workspace_bytes, void* cuda_stream) {
    if (!p || (!d_vals_in && p->nnz)) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    if ((s = reset_state(p, st))) return s;
    p->resc_eval = 0;  // phase entry: plain Gershgorin scaling, whatever the previous call used
    return launch_gather(p, d_vals_in, mu, b.b0, st);
}

extern "C" sm_status_t sm_sign_iterate(sm_plan_t* p, double eps, void* d_workspace, size_t workspace_bytes,
                                       sm_stats_t* stats, void* cuda_stream) {
    if (!p || !(eps > 0.0) || p->opt.precision != 0) return SM_ERR_INVALID_ARG;  // phase entry: FP64 path only
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    if (stats) memset(stats, 0, sizeof(*stats));
    int launched = 0, all_done = 0, nc = 0;
    if ((s = ns_loop(p, b, eps, p->opt.max_iter + 1, &all_done, &launched, st))) return s;
    if ((s = launch_nelec(p, b.b0, b.b1, st))) return s;
    if ((s = collect_stats(p, stats, &nc, st))) return s;
    if (stats) { stats->iterations = launched / (p->opt.order == 3 ? 3 : 2); stats->gemm_launches = launched; }
    return nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
}

extern "C" sm_status_t sm_scatter(sm_plan_t* p, int32_t as_identity, double* d_vals_out, void* d_workspace,
                                  size_t workspace_bytes, void* cuda_stream) {
    if (!p || (!d_vals_out && p->nnz)) return SM_ERR_INVALID_ARG;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    return launch_scatter(p, as_identity ? 1 : 0, b.b0, b.b1, d_vals_out, (cudaStream_t)cuda_stream);
}

extern "C" sm_status_t sm_sign_execute_host(sm_plan_t* p, const double* h_vals_in, double mu, double eps,
                                            double* h_vals_out, void* d_workspace, size_t workspace_bytes,
                                            sm_stats_t* stats, void* cuda_stream) {
    if (!p || (!h_vals_in && p->nnz)) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    sm_status_t s = ensure_stage(p);
    if (s) return s;
    if (p->nnz) SM_CUDA(cudaMemcpyAsync(p->d_stage_in, h_vals_in, (size_t)p->nnz * 8, cudaMemcpyHostToDevice, st));
    s = sm_sign_execute(p, p->d_stage_in, mu, eps, h_vals_out ? p->d_stage_out : nullptr, d_workspace,
                        workspace_bytes, stats, cuda_stream);
    if (s < 0) return s;
    if (h_vals_out && p->nnz)
        SM_CUDA(cudaMemcpyAsync(h_vals_out, p->d_stage_out, (size_t)p->nnz * 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    return s;
}

extern "C" sm_status_t sm_density_matrix(sm_plan_t* p, const double* d_vals_in, double n_target, double tol_n,
                                         double eps, double* mu_inout, double* d_vals_out, void* d_workspace,
                                         size_t workspace_bytes, sm_stats_t* stats, void* cuda_stream) {
    if (!p || (!d_vals_in && p->nnz) || !mu_inout || !(eps > 0.0) || !(tol_n >= 0.0) || !(*mu_inout == *mu_inout))
        return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    sm_stats_t local;
    sm_stats_t* S = stats ? stats : &local;
    memset(S, 0, sizeof(*S));
    if (p->opt.method == 1) return density_matrix_eig(p, d_vals_in, n_target, tol_n, mu_inout, d_vals_out, b, S, st);
    // bracket (n_elec = 0 below, n_basis above): the Gershgorin interval of the whole K~, intersected with
    // the interlacing interval [lambda_min, lambda_max](K~) of the Lanczos run when scaling = 1 has it
    // (every submatrix eigenvalue lies inside both, reading A11)
    if ((s = launch_gersh_global(p, d_vals_in, st))) return s;  // result read after the next synchronisation
    p->lz_valid = 0;  // one Lanczos run serves every mu of this call
    if (p->opt.scaling == 1 && (s = ensure_bounds(p, d_vals_in, st))) return s;  // ends with a synchronisation
    SM_CUDA(cudaStreamSynchronize(st));  // no-op after the Lanczos run
    double lo = p->h_pinned_d[4], hi = p->h_pinned_d[5];
    if (p->opt.scaling == 1 && p->lz_ok) {
        lo = std::max(lo, p->lz_lo);
        hi = std::min(hi, p->lz_hi);
    }
    S->bracket_lo = lo; S->bracket_hi = hi;
    // reading A11d: the Gauss quadrature of the same Lanczos run estimates the fraction of eigenvalues of
    // K~ below each Ritz value; the first interior step goes to the middle of the widest Ritz interval
    // near the target filling instead of the bracket midpoint (a guess only: the bracket logic is unchanged)
    double guess = NAN, guess_a = NAN, guess_b = NAN;  // the estimate and the Ritz interval it is the middle of
    if (p->opt.mu_guess && p->opt.scaling == 1 && p->lz_ok && p->lz_nodes >= 2 && p->info.n_basis > 0) {
        const int k = p->lz_nodes;
        const double* th = p->h_lz + 2;
        const double* cum = p->h_lz + 34;
        const double frac = n_target / (double)p->info.n_basis;
        int m = 0;
        for (int i = 1; i + 1 < k; ++i)
            if (std::fabs(cum[i] - frac) < std::fabs(cum[m] - frac)) m = i;
        int gi = std::max(0, m - 2);
        for (int i = gi + 1; i <= std::min(k - 2, m + 2); ++i)
            if (th[i + 1] - th[i] > th[gi + 1] - th[gi]) gi = i;
        guess = 0.5 * (th[gi] + th[gi + 1]);
        guess_a = th[gi]; guess_b = th[gi + 1];
    }
    S->mu_guess = guess;
    double mu = *mu_inout;
    // reading A11e: a caller's mu outside the Ritz interval the quadrature takes for the gap is not worth an
    // evaluation of its own -- step 0 goes to the estimate (the bracket alone keeps the search correct: every
    // accepted mu is verified by a converged evaluation); a caller's mu inside that interval (e.g. the mu of
    // the previous SCF step) is as good as the estimate and is evaluated first, as in reading A11
    if (p->opt.mu_start && guess > lo && guess < hi && !(mu > guess_a && mu < guess_b)) mu = guess;
    const int cap = (p->opt.precision == 0 && p->opt.bisect_iter > 0 && p->opt.bisect_iter < p->opt.max_iter)
                        ? p->opt.bisect_iter : p->opt.max_iter + 1;
    double best_mu = mu, best_g = INFINITY;
    int best_step = -1, steps = 0, nc = 0, last_nc = 0;
    bool accepted = false, last_partial = false;
    sm_stats_t ev;
    int64_t acc_n3 = 0, acc_sym = 0;
    int acc_launch = 0, acc_eval = 0;
    float acc_g = 0.f, acc_s = 0.f, acc_gemm = 0.f;
    auto accumulate = [&](const sm_stats_t& e) {
        acc_n3 += e.tot_sum_iter_n3; acc_sym += e.tot_sym_flop; acc_launch += e.tot_gemm_launches;
        acc_eval += 1; acc_g += e.tot_ms_gather; acc_s += e.tot_ms_sign; acc_gemm += e.tot_ms_gemm;
    };
    const bool early = p->opt.early_out != 0 && p->opt.precision == 0 && p->opt.shard_world <= 1;
    for (; steps < p->opt.max_mu_steps;) {
        memset(&ev, 0, sizeof(ev));
        Steer steer;
        steer.n_target = n_target; steer.tol_n = tol_n;
        steer.slack = 1e-10 * (double)std::max<int64_t>(p->info.n_basis, 1);
        if ((s = evaluate(p, d_vals_in, mu, eps, b, cap, &ev, &nc, st, early ? &steer : nullptr))) return s;
        double g = ev.n_elec - n_target;
        const bool partial = steer.decided != 0;  // direction proven, sign function not converged
        if (!partial && nc > 0 && cap <= p->opt.max_iter && std::fabs(g) <= std::max(tol_n, 0.0) + 1e-300) {
            // a capped evaluation may not accept: finish this one to convergence first
            int launched = 0, all_done = 0;
            if ((s = ns_loop(p, b, eps, p->opt.max_iter + 1, &all_done, &launched, st))) return s;
            if ((s = launch_nelec(p, b.b0, b.b1, st))) return s;
            if ((s = collect_stats(p, &ev, &nc, st))) return s;
            ev.iterations += launched / (p->opt.order == 3 ? 3 : 2);
            ev.tot_gemm_launches += launched;
            ev.tot_sum_iter_n3 = ev.sum_iter_n3;
            g = ev.n_elec - n_target;
        }
        accumulate(ev);
        S->mu_trace[steps] = mu;
        S->ne_trace[steps] = ev.n_elec;
        S->ne_err_trace[steps] = partial ? steer.err : 0.0;
        S->iter_trace[steps] = ev.iterations;
        last_nc = nc;
        last_partial = partial;
        // |g| of a partial step is only known up to its bound: rank it by the pessimistic end
        const double g_rank = std::fabs(g) + (partial ? steer.err : 0.0);
        if (g_rank < std::fabs(best_g)) { best_g = g_rank; best_mu = mu; best_step = steps; }
        ++steps;
        if (!partial && std::fabs(g) <= tol_n) { accepted = true; break; }
        if (g < 0) lo = std::max(lo, mu); else hi = std::min(hi, mu);
        if (hi - lo <= p->opt.mu_tol) break;
        mu = (steps == 1 && guess > lo && guess < hi) ? guess : 0.5 * (lo + hi);
    }
    // the workspace holds the last evaluated mu; re-evaluate if the best one was an earlier step
    // or if the last evaluation ended before convergence (capped or steering-only)
    if (best_step != steps - 1 || last_partial || (last_nc > 0 && cap <= p->opt.max_iter)) {
        memset(&ev, 0, sizeof(ev));
        if ((s = evaluate(p, d_vals_in, best_mu, eps, b, p->opt.max_iter + 1, &ev, &nc, st))) return s;
        last_nc = nc;
        accumulate(ev);
    }
    double tr_mu[64], tr_ne[64], tr_err[64];
    int32_t tr_it[64];
    memcpy(tr_mu, S->mu_trace, sizeof(tr_mu));
    memcpy(tr_ne, S->ne_trace, sizeof(tr_ne));
    memcpy(tr_err, S->ne_err_trace, sizeof(tr_err));
    memcpy(tr_it, S->iter_trace, sizeof(tr_it));
    const double br_lo = S->bracket_lo, br_hi = S->bracket_hi, br_guess = S->mu_guess;
    *S = ev;
    S->bracket_lo = br_lo; S->bracket_hi = br_hi; S->mu_guess = br_guess;
    memcpy(S->mu_trace, tr_mu, sizeof(tr_mu));
    memcpy(S->ne_trace, tr_ne, sizeof(tr_ne));
    memcpy(S->ne_err_trace, tr_err, sizeof(tr_err));
    memcpy(S->iter_trace, tr_it, sizeof(tr_it));
    S->mu = best_mu;
    S->mu_steps = steps;
    S->tot_sum_iter_n3 = acc_n3; S->tot_sym_flop = acc_sym; S->tot_gemm_launches = acc_launch;
    S->tot_evaluations = acc_eval; S->tot_ms_gather = acc_g; S->tot_ms_sign = acc_s; S->tot_ms_gemm = acc_gemm;
    *mu_inout = best_mu;
    if (d_vals_out && (s = do_scatter(p, b, d_vals_out, S, st))) return s;
    SM_CUDA(cudaStreamSynchronize(st));
    if (!accepted) return SM_WARN_MU_NOT_CONVERGED;
    return last_nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
}

extern "C" sm_status_t sm_density_matrix_host(sm_plan_t* p, const double* h_vals_in, double n_target,
                                              double tol_n, double eps, double* mu_inout, double* h_vals_out,
                                              void* d_workspace, size_t workspace_bytes, sm_stats_t* stats,
                                              void* cuda_stream) {
    if (!p || (!h_vals_in && p->nnz)) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    sm_status_t s = ensure_stage(p);
    if (s) return s;
    if (p->nnz) SM_CUDA(cudaMemcpyAsync(p->d_stage_in, h_vals_in, (size_t)p->nnz * 8, cudaMemcpyHostToDevice, st));
    s = sm_density_matrix(p, p->d_stage_in, n_target, tol_n, eps, mu_inout, h_vals_out ? p->d_stage_out : nullptr,
                          d_workspace, workspace_bytes, stats, cuda_stream);
    if (s < 0) return s;
    if (h_vals_out && p->nnz)
        SM_CUDA(cudaMemcpyAsync(h_vals_out, p->d_stage_out, (size_t)p->nnz * 8, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    return s;
}

extern "C" sm_status_t sm_eig_decompose(sm_plan_t* p, const double* d_vals_in, void* d_workspace,
                                        size_t workspace_bytes, sm_stats_t* stats, void* cuda_stream) {
    if (!p || (!d_vals_in && p->nnz) || p->opt.precision != 0 || p->opt.order != 2) return SM_ERR_INVALID_ARG;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    if (stats) memset(stats, 0, sizeof(*stats));
    int nc = 0;
    if ((s = eig_decompose(p, d_vals_in, b, stats, &nc, (cudaStream_t)cuda_stream))) return s;
    return nc ? SM_WARN_SIGN_NOT_CONVERGED : SM_OK;
}

extern "C" sm_status_t sm_eig_export(const sm_plan_t* p, int64_t* ptr, double* lam, double* w) {
    if (!p || !p->eig_valid) return SM_ERR_INVALID_ARG;
    const int ng = p->ngroups;
    if (ptr) {
        ptr[0] = 0;
        for (int i = 0; i < ng; ++i) ptr[i + 1] = ptr[i] + p->h_sub_dim[i];
    }
    if (lam && p->eig_total) SM_CUDA(cudaMemcpy(lam, p->d_eig_lam, (size_t)p->eig_total * 8, cudaMemcpyDeviceToHost));
    if (w && p->eig_total) SM_CUDA(cudaMemcpy(w, p->d_eig_w, (size_t)p->eig_total * 8, cudaMemcpyDeviceToHost));
    return SM_OK;
}

extern "C" sm_status_t sm_eig_nelec(sm_plan_t* p, double mu, double kT, double* n_elec, void* cuda_stream) {
    if (!p || !p->eig_valid || !n_elec || !(mu == mu) || !(kT >= 0.0)) return SM_ERR_INVALID_ARG;
    return eig_count(p, mu, kT, n_elec, (cudaStream_t)cuda_stream);
}

extern "C" sm_status_t sm_eig_density(sm_plan_t* p, double mu, double kT, double* d_vals_out, void* d_workspace,
                                      size_t workspace_bytes, void* cuda_stream) {
    if (!p || !p->eig_valid || (!d_vals_out && p->nnz) || !(mu == mu) || !(kT >= 0.0)) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Bufs b;
    sm_status_t s = carve(p, d_workspace, workspace_bytes, &b);
    if (s) return s;
    if ((s = launch_eig_density(p, mu, kT, b.b0, b.b1, st))) return s;
    return launch_scatter(p, 0, b.b0, b.b1, d_vals_out, st);
}

extern "C" sm_status_t sm_trace_dk(sm_plan_t* p, const double* d_D, const double* d_K, double* tr_D,
                                   double* tr_DK, void* cuda_stream) {
    if (!p || (p->nnz && (!d_D || !d_K))) return SM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    sm_status_t s = launch_trace_dk(p, d_D, d_K, st);
    if (s) return s;
    SM_CUDA(cudaMemcpyAsync(p->h_pinned_d + 1, p->d_scalars + 1, 16, cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    if (tr_D) *tr_D = p->h_pinned_d[1];
    if (tr_DK) *tr_DK = p->h_pinned_d[2];
    return SM_OK;
}

extern "C" const char* sm_strerror(sm_status_t s) {
    switch (s) {
        case SM_OK: return "ok";
        case SM_ERR_INVALID_ARG: return "invalid argument";
        case SM_ERR_STRUCTURE: return "invalid block-sparse structure or grouping";
        case SM_ERR_ALLOC: return "allocation failed";
        case SM_ERR_CUDA: return "CUDA error";
        case SM_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case SM_WARN_SIGN_NOT_CONVERGED: return "warning: sign iteration not converged for at least one submatrix";
        case SM_WARN_MU_NOT_CONVERGED: return "warning: mu bisection ended without meeting tol_n";
        default: return "unknown status";
    }
}

extern "C" const char* sm_last_cuda_error(void) { return smb::g_cuda_err; }
