"""SURVEY 8(f)4 on one GPU: sharded plans (contiguous chunks of groups balanced by sum n^3)
run one after the other; their block columns put together must be the unsharded result, bit for bit, and
the partial electron counts must add up.  The cross-rank sum itself is torch.distributed plumbing
(tests/test_bench_dist.py, gloo); here it is a callback that adds what the other shards hold."""
import ctypes as C

import numpy as np
import pytest

from paper_2004_10811_b200 import workloads as W

pytestmark = pytest.mark.gpu
EPS = 1e-12


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2004_10811_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("world,method", [(2, 0), (3, 0), (2, 1)])
def test_sharded_fixed_mu_equals_unsharded(B, oracle, cfg0, world, method):
    import torch
    m = cfg0
    vin = torch.from_numpy(m.values).cuda()
    plan = B.plan_from_matrix(m, B.default_options(method=method))
    ws = B.alloc_workspace(plan)
    ref = torch.full_like(vin, float("nan"))
    st_ref = B.sm_stats_t()
    assert B.sm_sign_execute(plan, vin, 0.05, EPS, ref, ws, st_ref) == B.SM_OK
    idx = oracle.Index(m)
    first = oracle.partition_groups(idx.sub_dim, world)
    B.sm_plan_destroy(plan)
    out = torch.full_like(vin, float("nan"))
    ne = 0.0
    vo = m.val_off()
    for r in range(world):
        p = B.plan_from_matrix(m, B.default_options(method=method, shard_rank=r, shard_world=world))
        info = B.sm_plan_query(p)
        assert (info.shard_group_begin, info.shard_group_end) == (first[r], first[r + 1])  # the oracle's chunks
        assert info.ngroups == first[r + 1] - first[r] and info.ngroups_total == m.ngroups
        c0, c1 = int(m.grp_cols[m.grp_ptr[first[r]]]), int(m.grp_cols[m.grp_ptr[first[r + 1]] - 1])
        assert (info.shard_val_begin, info.shard_val_end) == (vo[m.colptr[c0]], vo[m.colptr[c1 + 1]])
        w = B.alloc_workspace(p)
        st = B.sm_stats_t()
        assert B.sm_sign_execute(p, vin, 0.05, EPS, out, w, st) == B.SM_OK  # writes only its own block columns
        ne += st.n_elec
        B.sm_plan_destroy(p)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)  # every value written exactly once, bitwise the unsharded result
    assert abs(ne - st_ref.n_elec) <= 1e-9
    d_or = oracle.density(idx, m.values, 0.05)
    assert np.abs(out.cpu().numpy() - d_or).max() <= 1e-9


@pytest.mark.parametrize("method", [0, 1])
def test_sharded_density_matrix_with_allreduce_callback(B, oracle, cfg0, method):
    """The canonical loop on shard 0 of 2 with the library's all-reduce hook: the callback adds shard 1's
    count at the same mu (taken from an unsharded twin restricted to shard 1's groups through a second sharded
    plan), so every decision of the search is taken on the global count, as it would be over NCCL."""
    import torch
    m = cfg0
    vin = torch.from_numpy(m.values).cuda()
    opts = dict(method=method, mu_guess=0, mu_start=0)
    full = B.plan_from_matrix(m, B.default_options(**opts))
    wsf = B.alloc_workspace(full)
    ref = torch.full_like(vin, float("nan"))
    st_ref = B.sm_stats_t()
    rc_ref, mu_ref = B.sm_density_matrix(full, vin, float(m.n_occ), 0.5, EPS, -1.0, ref, wsf, st_ref)
    assert rc_ref == B.SM_OK
    p0 = B.plan_from_matrix(m, B.default_options(shard_rank=0, shard_world=2, **opts))
    p1 = B.plan_from_matrix(m, B.default_options(shard_rank=1, shard_world=2, **opts))
    w0, w1 = B.alloc_workspace(p0), B.alloc_workspace(p1)
    calls = []
    state = {"mu": None}
    st1 = B.sm_stats_t()

    def other_rank(ctx, vals, n):  # what rank 1 would contribute at the mu rank 0 has just evaluated
        k = len(calls)
        mu_k = trace_mu[k] if k < len(trace_mu) else state["mu"]
        assert B.sm_sign_execute(p1, vin, mu_k, EPS, None, w1, st1) in (B.SM_OK, B.SM_WARN_SIGN_NOT_CONVERGED)
        if n >= 1:
            vals[0] += st1.n_elec
        if n >= 2:
            vals[1] += st1.not_converged
        calls.append(mu_k)

    # the steering early-out is off for sharded plans, so the mu trace is the midpoint rule's: known in advance
    # from the unsharded run with early_out = 0
    twin = B.plan_from_matrix(m, B.default_options(early_out=0, **opts))
    st_t = B.sm_stats_t()
    tmp = torch.empty_like(vin)
    B.sm_density_matrix(twin, vin, float(m.n_occ), 0.5, EPS, -1.0, tmp, wsf, st_t)
    trace_mu = [st_t.mu_trace[k] for k in range(st_t.mu_steps)]
    B.sm_plan_destroy(twin)
    cb = B.ALLREDUCE_FN(other_rank)
    if method == 1:
        # one reduction for the decomposition's status, then one per mu step
        def other_rank_eig(ctx, vals, n):
            k = len(calls)
            if k == 0:
                calls.append(None)
                return
            mu_k = trace_mu[k - 1]
            B.sm_sign_execute(p1, vin, mu_k, EPS, None, w1, st1)
            vals[0] += st1.n_elec
            calls.append(mu_k)
        cb = B.ALLREDUCE_FN(other_rank_eig)
    B.sm_plan_set_allreduce(p0, cb)
    out = torch.full_like(vin, float("nan"))
    st0 = B.sm_stats_t()
    rc, mu = B.sm_density_matrix(p0, vin, float(m.n_occ), 0.5, EPS, -1.0, out, w0, st0)
    torch.cuda.synchronize()
    assert rc == B.SM_OK and mu == mu_ref
    assert st0.mu_steps == len(trace_mu) and [st0.mu_trace[k] for k in range(st0.mu_steps)] == trace_mu
    assert abs(st0.n_elec - st_ref.n_elec) <= 1e-9  # the GLOBAL count
    info = B.sm_plan_query(p0)
    b, e = info.shard_val_begin, info.shard_val_end
    assert torch.equal(out[b:e], ref[b:e]) and bool(torch.isnan(out[e:]).all())
    for p in (full, p0, p1):
        B.sm_plan_destroy(p)
