"""SURVEY 8(f)1 on the GPU: batched eigendecomposition of the submatrices + Algorithm 1 as written
(Eq.(17), Algorithm 1, Fermi function L255), through the C-ABI, against the
CPU oracle (cyclic Jacobi in C) on the same seeded inputs.  Bars: eigenvalues <= 1e-10, electron counts
<= 1e-9, D~ <= 1e-9 elementwise, band energy <= 1e-10 relative, bisection traces identical."""
import numpy as np
import pytest

from paper_2004_10811_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_D = 1e-9
TOL_E = 1e-10
TOL_LAM = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2004_10811_b200 import binding
    binding.lib()
    return binding


def _torch():
    import torch
    return torch


def _decompose(B, m, **opt):
    torch = _torch()
    plan = B.plan_from_matrix(m, B.default_options(**opt))
    ws = B.alloc_workspace(plan)
    vin = torch.from_numpy(m.values).cuda()
    stats = B.sm_stats_t()
    st = B.sm_eig_decompose(plan, vin, ws, stats)
    torch.cuda.synchronize()
    return plan, ws, vin, st, stats


def _compare_spectra(B, oracle, m, plan, groups=None):
    """lambda per submatrix (sorted) <= 1e-10; the weights of Algorithm 1 through what is unique about them:
    their cumulative sums at well separated eigenvalues (inside a cluster of nearly equal eigenvalues the
    eigenvectors, hence the individual w, are not unique) and their total = generating width."""
    idx = oracle.Index(m)
    lam_o, w_o, ptr_o, g = oracle.eig_groups(idx, m.values, groups)
    ptr, lam, w = B.sm_eig_export(plan)
    assert np.array_equal(ptr, np.concatenate([[0], np.cumsum(idx.sub_dim)]))
    worst_l = worst_w = 0.0
    for j, i in enumerate(g):
        lo = np.sort(lam_o[ptr_o[j]:ptr_o[j + 1]])
        order_o = np.argsort(lam_o[ptr_o[j]:ptr_o[j + 1]], kind="stable")
        lg = lam[ptr[i]:ptr[i + 1]]
        order_g = np.argsort(lg, kind="stable")
        worst_l = max(worst_l, np.abs(lg[order_g] - lo).max())
        cw_o = np.cumsum(w_o[ptr_o[j]:ptr_o[j + 1]][order_o])
        cw_g = np.cumsum(w[ptr[i]:ptr[i + 1]][order_g])
        sep = np.concatenate([np.diff(lo) > 1e-5, [True]])  # cumulative weight up to a well separated eigenvalue
        worst_w = max(worst_w, np.abs(cw_g - cw_o)[sep].max())
        assert abs(cw_g[-1] - idx.gen_width[i]) <= 1e-11 * max(1, idx.gen_width[i])
    assert worst_l <= TOL_LAM, worst_l
    assert worst_w <= 1e-9, worst_w
    return idx, lam_o, w_o, g


def test_eig_config0_spectra_counts_density(B, oracle, cfg0):
    m = cfg0
    plan, ws, vin, st, stats = _decompose(B, m)
    assert st == B.SM_OK and stats.not_converged == 0 and 2 <= stats.iter_max <= 20
    idx, lam_o, w_o, g = _compare_spectra(B, oracle, m, plan)
    for mu in (-2.5, -0.464, 0.0, 0.11, 0.7, 2.5):  # Algorithm 1's count, no new decomposition (L266)
        assert abs(B.sm_eig_nelec(plan, mu) - oracle.nelec(idx, lam_o, w_o, g, mu)) <= 1e-9
    torch = _torch()
    vout = torch.full_like(vin, float("nan"))
    for mu in (0.0, -0.464):
        B.sm_eig_density(plan, mu, 0.0, vout, ws)
        torch.cuda.synchronize()
        d_or = oracle.density(idx, m.values, mu)
        assert np.abs(vout.cpu().numpy() - d_or).max() <= TOL_D
        _, tdk_o = oracle.traces(idx, d_or, m.values)
        td_g, tdk_g = B.sm_trace_dk(plan, vout, vin)
        assert abs(tdk_g - tdk_o) <= TOL_E * abs(tdk_o)
        assert abs(td_g - B.sm_eig_nelec(plan, mu)) <= 1e-9  # Algorithm 1's count == tr D~
    B.sm_plan_destroy(plan)


def test_eig_ragged_blocks_scattered_groups_and_tiny(B, oracle):
    cases = [W.random_block_pattern(nb=30 + s, density=0.2, max_bs=7, seed=10 + s) for s in range(3)]
    cases.append(W.dense_batch_as_blocks(np.array([[[3.0, 4.0], [4.0, -3.0]]])))          # Eq.(8): eigenvalues +-5
    cases.append(W.dense_batch_as_blocks(np.array([[[-0.7]]])))                            # 1 x 1
    cases.append(W.dense_batch_as_blocks(np.diag([-2.0, 0.5, 3.0, -1e-3, 0.25, -0.5, 1.0, 2.0, -4.0])[None]))
    cases.append(W.dense_batch_as_blocks(np.eye(5)[None]))                                 # fully degenerate
    for m in cases:
        plan, ws, vin, st, stats = _decompose(B, m)
        assert st == B.SM_OK
        idx, lam_o, w_o, g = _compare_spectra(B, oracle, m, plan)
        srt = np.sort(lam_o)
        k = int(np.argmax(np.diff(srt))) if len(srt) > 1 else 0
        mu = 0.5 * (srt[k] + srt[k + 1]) if len(srt) > 1 else srt[0] + 1.0
        torch = _torch()
        vout = torch.full_like(vin, float("nan"))
        B.sm_eig_density(plan, mu, 0.0, vout, ws)
        torch.cuda.synchronize()
        assert np.abs(vout.cpu().numpy() - oracle.density(idx, m.values, mu)).max() <= TOL_D
        B.sm_plan_destroy(plan)


def test_eig_dzvp_and_large_rows(B, oracle):
    """DZVP blocks (23 generating functions per group: three passes of the density kernel) and n > 384
    (columns no longer cached in registers)."""
    for m, k in ((W.water_like(16, "DZVP", 6.0, seed=3), None), (W.water_like(96, "SZV", 9.0, seed=5), 3)):
        plan, ws, vin, st, stats = _decompose(B, m)
        assert st == B.SM_OK
        idx0 = oracle.Index(m)
        groups = None if k is None else np.array([0, idx0.ngroups // 2, idx0.ngroups - 1], dtype=np.int32)
        idx, lam_o, w_o, g = _compare_spectra(B, oracle, m, plan, groups)
        torch = _torch()
        vout = torch.full_like(vin, float("nan"))
        B.sm_eig_density(plan, 0.0, 0.0, vout, ws)
        torch.cuda.synchronize()
        d_or = oracle.density(idx, m.values, 0.0, groups)
        cols = oracle.column_ids_of_groups(idx, g)
        mask = np.repeat(np.isin(m.block_cols(), cols), np.diff(idx.val_off))
        assert np.abs(vout.cpu().numpy() - d_or)[mask].max() <= TOL_D
        B.sm_plan_destroy(plan)


@pytest.mark.parametrize("mu0,tol_n", [(-1.0, 0.5), (1.2, 0.5), (0.0, 1e-8), (-1.0, 1e-8)])
def test_algorithm1_trace_identical_to_oracle(B, oracle, cfg0, mu0, tol_n):
    """method = 1: Algorithm 1 as written.  The mu trace, the counts and the stopping reason are those of
    oracle.bisect_mu run in the oracle's own Gershgorin bracket -- including the literal tol_n = 1e-8 of
    BASELINE config 4, which ends on the guards (reading A11: the plateau is offset from the integer)."""
    torch = _torch()
    m = cfg0
    idx = oracle.Index(m)
    lam, w, ptr, g = oracle.eig_groups(idx, m.values)
    lo, hi = oracle.gershgorin_interval(m)
    mu_o, ne_o, trace_o = oracle.bisect_mu(idx, lam, w, g, m.n_occ, mu0, lo, hi, tol_n)
    plan = B.plan_from_matrix(m, B.default_options(method=1))
    ws = B.alloc_workspace(plan)
    vin = torch.from_numpy(m.values).cuda()
    vout = torch.full_like(vin, float("nan"))
    stats = B.sm_stats_t()
    st, mu = B.sm_density_matrix(plan, vin, float(m.n_occ), tol_n, 1e-12, mu0, vout, ws, stats)
    torch.cuda.synchronize()
    accepted = abs(ne_o - m.n_occ) <= tol_n
    assert st == (B.SM_OK if accepted else B.SM_WARN_MU_NOT_CONVERGED)
    assert (tol_n == 0.5) == accepted
    assert abs(stats.bracket_lo - lo) <= 1e-12 * abs(lo) and abs(stats.bracket_hi - hi) <= 1e-12 * abs(hi)
    assert stats.mu_steps == len(trace_o) and stats.tot_evaluations == 1  # one decomposition, however many steps
    for k, (mo, no) in enumerate(trace_o):
        assert abs(stats.mu_trace[k] - mo) <= 1e-12 * max(1.0, abs(mo))
        assert abs(stats.ne_trace[k] - no) <= 1e-9
    assert abs(mu - mu_o) <= 1e-12 * max(1.0, abs(mu_o)) and abs(stats.n_elec - ne_o) <= 1e-9
    assert np.abs(vout.cpu().numpy() - oracle.density(idx, m.values, mu)).max() <= TOL_D
    B.sm_plan_destroy(plan)


def test_method1_sign_execute_config2_all_submatrices(B, oracle):
    """sm_sign_execute with method = 1 (Eq.(17)) on BASELINE config 2: every one of the 1024 submatrices
    against the oracle, plus agreement with the Newton-Schulz path of the same library."""
    torch = _torch()
    m = W.make_config(2)
    idx = oracle.Index(m)
    d_or = oracle.density(idx, m.values, 0.0)
    out = {}
    for method in (1, 0):
        plan = B.plan_from_matrix(m, B.default_options(method=method))
        ws = B.alloc_workspace(plan)
        vin = torch.from_numpy(m.values).cuda()
        vout = torch.full_like(vin, float("nan"))
        stats = B.sm_stats_t()
        st = B.sm_sign_execute(plan, vin, 0.0, 1e-12, vout, ws, stats)
        torch.cuda.synchronize()
        assert st == B.SM_OK
        out[method] = vout.cpu().numpy()
        assert np.abs(out[method] - d_or).max() <= TOL_D
        td, tdk = B.sm_trace_dk(plan, vout, vin)
        _, tdk_o = oracle.traces(idx, d_or, m.values)
        assert abs(tdk - tdk_o) <= TOL_E * abs(tdk_o) and abs(stats.n_elec - td) <= 1e-9
        B.sm_plan_destroy(plan)
        del ws
    assert np.abs(out[0] - out[1]).max() <= 1e-11


def test_finite_temperature_fermi(B, oracle, cfg0):
    """L255: signum of Eq.(17) replaced by the Fermi function.  D~ against the oracle at fixed mu, and the
    canonical loop: at kT > 0 the count is continuous, so the LITERAL tolerance 1e-8 is met (SM_OK), with
    the oracle's trace."""
    torch = _torch()
    m, kT = cfg0, 0.02
    idx = oracle.Index(m)
    lam, w, ptr, g = oracle.eig_groups(idx, m.values)
    lo, hi = oracle.gershgorin_interval(m)
    plan = B.plan_from_matrix(m, B.default_options(method=1, kT=kT, mu_tol=1e-14))
    ws = B.alloc_workspace(plan)
    vin = torch.from_numpy(m.values).cuda()
    vout = torch.full_like(vin, float("nan"))
    stats = B.sm_stats_t()
    assert B.sm_sign_execute(plan, vin, 0.1, 1e-12, vout, ws, stats) == B.SM_OK
    torch.cuda.synchronize()
    d_or = oracle.density_fermi(idx, m.values, 0.1, kT)
    assert np.abs(vout.cpu().numpy() - d_or).max() <= TOL_D
    assert abs(stats.n_elec - oracle.nelec_fermi(idx, lam, w, g, 0.1, kT)) <= 1e-9
    mu_o, ne_o, trace_o = oracle.bisect_mu_fermi(idx, lam, w, g, m.n_occ, -1.0, lo, hi, 1e-8, kT, mu_tol=1e-14)
    st, mu = B.sm_density_matrix(plan, vin, float(m.n_occ), 1e-8, 1e-12, -1.0, vout, ws, stats)
    torch.cuda.synchronize()
    assert st == B.SM_OK and abs(stats.n_elec - m.n_occ) <= 1e-8
    assert abs(stats.mu_steps - len(trace_o)) <= 1  # the last halvings work at the 1e-9 level of the two counts
    for k in range(min(stats.mu_steps, len(trace_o)) - 1):
        assert abs(stats.mu_trace[k] - trace_o[k][0]) <= 1e-12 and abs(stats.ne_trace[k] - trace_o[k][1]) <= 1e-9
    assert np.abs(vout.cpu().numpy() - oracle.density_fermi(idx, m.values, mu, kT)).max() <= TOL_D
    td, _ = B.sm_trace_dk(plan, vout, vin)
    assert abs(td - stats.n_elec) <= 1e-9
    B.sm_plan_destroy(plan)


def test_eig_config4_full_size_sampled(B, oracle):
    """BASELINE config 4 at full size through Algorithm 1 (method = 1): spectra of 64 sampled groups against
    the oracle, the canonical loop (plateau acceptance) and D~ on the sampled columns."""
    torch = _torch()
    m = W.make_config(4)
    idx = oracle.Index(m)
    order = np.argsort(idx.sub_dim, kind="stable")
    rng = np.random.default_rng(3)
    groups = np.array(sorted({int(order[0]), int(order[len(order) // 2]), int(order[-1])} |
                             set(int(x) for x in rng.permutation(idx.ngroups)[:61])), dtype=np.int32)
    plan = B.plan_from_matrix(m, B.default_options(method=1))
    ws = B.alloc_workspace(plan)
    vin = torch.from_numpy(m.values).cuda()
    vout = torch.full_like(vin, float("nan"))
    stats = B.sm_stats_t()
    st, mu = B.sm_density_matrix(plan, vin, float(m.n_occ), 0.5, 1e-12, -1.0, vout, ws, stats)
    torch.cuda.synchronize()
    assert st == B.SM_OK and stats.not_converged == 0 and abs(stats.n_elec - m.n_occ) <= 0.5
    _compare_spectra(B, oracle, m, plan, groups)
    d_gpu = vout.cpu().numpy()
    d_or = oracle.density(idx, m.values, mu, groups)
    cols = oracle.column_ids_of_groups(idx, groups)
    mask = np.repeat(np.isin(m.block_cols(), cols), np.diff(idx.val_off))
    assert np.abs(d_gpu - d_or)[mask].max() <= TOL_D
    _, tdk_o = oracle.traces(idx, d_or, m.values, cols)
    _, tdk_g = oracle.traces(idx, d_gpu, m.values, cols)
    assert abs(tdk_g - tdk_o) <= TOL_E * abs(tdk_o)
    td_all, _ = B.sm_trace_dk(plan, vout, vin)
    assert abs(td_all - stats.n_elec) <= 1e-9 * td_all and np.all(np.isfinite(d_gpu))
    print(f"config 4 method=1: mu={mu:.6f} steps={stats.mu_steps} sweeps {stats.iter_min}-{stats.iter_max}")
    B.sm_plan_destroy(plan)
