"""Pins of the CPU oracle against what the paper and the mathematics fix (not against itself).

Each test names the passage (PAPER.md line) or the textbook fact it rests on."""
import os

import numpy as np
import pytest

from paper_2004_10811_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    return np.loadtxt(os.path.join(GOLD, name), comments="#")


def _blocks_from_dense(a, bs, mask=None, groups=None):
    """Pack a dense symmetric matrix into the block layout (data movement only)."""
    bs = np.asarray(bs, dtype=np.int32)
    nb = len(bs)
    off = np.concatenate([[0], np.cumsum(bs)])
    rows, cols, vals = [], [], []
    for c in range(nb):
        for r in range(nb):
            blk = a[off[r]:off[r + 1], off[c]:off[c + 1]]
            keep = (mask[r, c] if mask is not None else (np.any(blk != 0) or r == c))
            if keep:
                rows.append(r); cols.append(c); vals.append(blk.T.reshape(-1))
    colptr = np.zeros(nb + 1, dtype=np.int64)
    np.cumsum(np.bincount(cols, minlength=nb), out=colptr[1:])
    if groups is None:
        groups = [[c] for c in range(nb)]
    grp_ptr = np.concatenate([[0], np.cumsum([len(g) for g in groups])]).astype(np.int32)
    grp_cols = np.concatenate(groups).astype(np.int32)
    return W.BlockSparseSym(nb, bs, colptr, np.array(rows, dtype=np.int32), np.concatenate(vals),
                            grp_ptr, grp_cols)


# ---------------------------------------------------------------- golden closed forms
def test_golden_sign_2x2(oracle):
    g = _load("sign_2x2.txt")
    assert np.allclose(oracle.dense_sign(g[:2]), g[2:], atol=1e-15)


def test_golden_zero_eigenvalue(oracle):
    """Eq.(12): an eigenvalue exactly 0 maps to 0."""
    g = _load("sign_zero_eig.txt")
    assert np.allclose(oracle.dense_sign(g[:2]), g[2:], atol=1e-15)
    # mu shifts the spectrum (Eq.16): A - 2I has eigenvalues -2, 0 -> sign = -v0 v0^T
    assert np.allclose(oracle.dense_sign(g[:2], mu=2.0), [[-0.5, 0.5], [0.5, -0.5]], atol=1e-15)


def test_golden_submatrix_3x3(oracle):
    """Steps 1-3 (L125-127) worked by hand on a 3x3 tridiagonal matrix with 1x1 blocks."""
    a = np.array([[3.0, 4, 0], [4, -3, 4], [0, 4, 3]])
    m = _blocks_from_dense(a, [1, 1, 1])
    idx = oracle.Index(m)
    assert list(idx.sub_dim) == [2, 3, 2]
    assert list(idx.sub_blocks) == [0, 1, 0, 1, 2, 1, 2]
    assert list(idx.gen_pos) == [0, 1, 1]
    d = m.to_dense(oracle.density(idx, m.values, 0.0))
    sign_tilde = np.where(a != 0, np.eye(3) - 2 * d, 0.0)
    assert np.allclose(sign_tilde, _load("submatrix_3x3.txt"), atol=1e-14)
    assert d[0, 2] == 0 and d[2, 0] == 0  # pattern retained (L127)


def test_ns_scalar_fixture_is_consistent_with_sign():
    """Eq.(11): the scalar recursion converges to signum(x0); fixture values are exact rationals."""
    g = _load("ns_scalar.txt")
    x = 0.5
    for k in range(3):
        assert x == g[k]
        x = 0.5 * x * (3 - x * x)


# ---------------------------------------------------------------- Jacobi vs library / closed form
@pytest.mark.parametrize("n", [1, 2, 7, 64])
def test_jacobi_vs_lapack(oracle, n):
    """Library pin: eigenvalues equal numpy.linalg.eigvalsh (LAPACK), a = Q L Q^T, Q orthogonal."""
    rng = np.random.default_rng(n)
    a = rng.standard_normal((n, n)); a = 0.5 * (a + a.T)
    lam, q = oracle.jacobi_eig(a)
    assert np.allclose(np.sort(lam), np.linalg.eigvalsh(a), atol=1e-13 * max(1, n))
    assert np.allclose(q @ np.diag(lam) @ q.T, a, atol=1e-13 * max(1, n))
    assert np.allclose(q.T @ q, np.eye(n), atol=1e-13)


def test_sign_closed_form_haar(oracle):
    """P1 (BASELINE config 1 recipe): A = Q diag(lam) Q^T  =>  sign(A) = Q diag(sgn lam) Q^T."""
    a, q, lam = W.haar_spectrum_batch(3, 96, seed=5)
    for b in range(3):
        expect = (q[b] * np.sign(lam[b])) @ q[b].T
        assert np.abs(oracle.dense_sign(a[b]) - expect).max() < 5e-13


def test_sign_invariants(oracle, cfg0):
    """P2: sign(a)^2 = I (Fig.13 involutority), commutes with a (Eq.8), symmetric; D_i idempotent,
    tr D_i = number of eigenvalues below mu (Eq.6/7; count from LAPACK)."""
    idx = oracle.Index(cfg0)
    for i, mu in ((0, 0.0), (7, 0.1), (31, -0.9)):
        a = oracle.assemble(idx, cfg0.values, i)
        n = a.shape[0]
        assert np.array_equal(a, a.T)
        s = oracle.dense_sign(a, mu)
        am = a - mu * np.eye(n)
        assert np.abs(s @ s - np.eye(n)).max() < 1e-12
        assert np.abs(s @ am - am @ s).max() < 1e-12
        assert np.abs(s - s.T).max() < 1e-13
        d = 0.5 * (np.eye(n) - s)
        assert np.abs(d @ d - d).max() < 1e-12
        assert abs(np.trace(d) - np.sum(np.linalg.eigvalsh(a) < mu)) < 1e-10


def test_diagonal_and_2x2_family(oracle):
    """P3: diagonal matrix -> elementwise signum; [[a,b],[b,-a]] -> A / sqrt(a^2+b^2)."""
    dvals = np.array([-2.0, 0.5, 0.0, 3.0, -1e-3])
    assert np.array_equal(oracle.dense_sign(np.diag(dvals)), np.diag(np.sign(dvals)))
    rng = np.random.default_rng(3)
    for _ in range(5):
        a, b = rng.standard_normal(2)
        m = np.array([[a, b], [b, -a]])
        assert np.allclose(oracle.dense_sign(m), m / np.hypot(a, b), atol=1e-14)


# ---------------------------------------------------------------- index: brute force
@pytest.mark.parametrize("seed", range(6))
def test_index_bruteforce(oracle, seed):
    """P6: S_i = {r : any stored block (r,c), c in G_i}, from a dense boolean mask."""
    m = W.random_block_pattern(nb=13 + seed, density=0.25, max_bs=4, seed=seed)
    idx = oracle.Index(m)
    mask = np.zeros((m.nb, m.nb), dtype=bool)
    mask[m.rowidx, m.block_cols()] = True
    for i in range(m.ngroups):
        gc = m.grp_cols[m.grp_ptr[i]:m.grp_ptr[i + 1]]
        S = np.nonzero(mask[:, gc].any(axis=1))[0]
        got = idx.sub_blocks[idx.sub_ptr[i]:idx.sub_ptr[i + 1]]
        assert np.array_equal(got, S)
        assert idx.sub_dim[i] == m.blk_size[S].sum()
        off = np.concatenate([[0], np.cumsum(m.blk_size[S])[:-1]])
        assert np.array_equal(idx.sub_off[idx.sub_ptr[i]:idx.sub_ptr[i + 1]], off)
        for g, c in zip(range(m.grp_ptr[i], m.grp_ptr[i + 1]), gc):
            assert S[idx.gen_pos[g]] == c


def test_assemble_is_principal_submatrix(oracle):
    """L125: a_i equals the dense matrix restricted to the rows/columns of S_i."""
    m = W.random_block_pattern(nb=11, density=0.3, max_bs=5, seed=42)
    idx = oracle.Index(m)
    k = m.to_dense()
    off = m.blk_off()
    for i in range(m.ngroups):
        S = idx.sub_blocks[idx.sub_ptr[i]:idx.sub_ptr[i + 1]]
        el = np.concatenate([np.arange(off[r], off[r + 1]) for r in S])
        assert np.array_equal(oracle.assemble(idx, m.values, i), k[np.ix_(el, el)])


# ---------------------------------------------------------------- whole pipeline: exactness cases
def test_full_cutoff_equals_dense_sign(oracle):
    """P5 (L125): if every column is full, every a_i is the whole matrix and the method is exact:
    D~ = 1/2 (I - sign(K~)) computed with LAPACK eigh on the whole matrix; tr = N_occ exactly."""
    m = W.water_like(8, "SZV", cutoff=1e9, seed=3)
    assert m.nnzb == m.nb * m.nb
    idx = oracle.Index(m)
    assert np.all(idx.sub_dim == m.n_basis)
    d = m.to_dense(oracle.density(idx, m.values, 0.0, nthreads=4))
    k = m.to_dense()
    ev, v = np.linalg.eigh(k)
    dex = v[:, ev < 0] @ v[:, ev < 0].T
    assert np.abs(d - dex).max() < 1e-12
    td, tdk = oracle.traces(idx, oracle.density(idx, m.values, 0.0, nthreads=4), m.values)
    assert abs(td - np.sum(ev < 0)) < 1e-11
    assert abs(tdk - ev[ev < 0].sum()) < 1e-11  # Eq.(10): Tr(DK) = sum of occupied eigenvalues


def test_block_diagonal_is_exact(oracle):
    """P3: cutoff below the nearest neighbour -> K~ is its on-site diagonal -> D~ = diag(1 on the
    N(-1,.) functions, 0 on the N(+1,.) ones)."""
    m = W.water_like(8, "SZV", cutoff=0.1, seed=2)
    assert m.nnzb == m.nb
    idx = oracle.Index(m)
    d = m.to_dense(oracle.density(idx, m.values, 0.0))
    k = m.to_dense()
    assert np.array_equal(d, np.diag((np.diag(k) < 0).astype(float)))
    assert oracle.traces(idx, oracle.density(idx, m.values, 0.0), m.values)[0] == m.n_occ


def test_symmetries(oracle, cfg0):
    """P7: D~(-K,-mu) = I - D~(K,mu) on the pattern; D~(K,mu) = D~(K - mu I, 0); D~(cK, c mu) = D~(K, mu)."""
    m = cfg0
    idx = oracle.Index(m)
    groups = [0, 5, 17]
    mu = 0.07
    d = oracle.density(idx, m.values, mu, groups)
    cols = oracle.column_ids_of_groups(idx, groups)
    sel = np.zeros(m.nnzb, dtype=bool)
    bc = m.block_cols()
    sel[np.isin(bc, cols)] = True
    emask = np.repeat(sel, np.diff(idx.val_off))
    # identity on the pattern
    eye = np.zeros_like(m.values)
    vo = idx.val_off
    for b in np.nonzero(m.rowidx == bc)[0]:
        n = m.blk_size[bc[b]]
        eye[vo[b]:vo[b + 1]] = np.eye(n).reshape(-1)
    d_neg = oracle.density(idx, -m.values, -mu, groups)
    assert np.abs((eye - d)[emask] - d_neg[emask]).max() < 1e-12
    d_shift = oracle.density(idx, m.values - mu * eye, 0.0, groups)
    assert np.abs(d_shift - d)[emask].max() < 1e-12
    d_scale = oracle.density(idx, 3.5 * m.values, 3.5 * mu, groups)
    assert np.abs(d_scale - d)[emask].max() < 1e-12
    assert np.all(d[~emask] == 0)  # nothing outside the listed groups' columns


def test_atom_relabelling_permutes_result(oracle):
    """P7: relabelling block columns permutes D~ (index maps carry no hidden order dependence)."""
    m = W.random_block_pattern(nb=9, density=0.35, max_bs=3, seed=7, ngroups=9, contiguous_groups=True)
    k = m.to_dense()
    off = m.blk_off()
    perm = np.random.default_rng(1).permutation(m.nb)
    el = np.concatenate([np.arange(off[p], off[p + 1]) for p in perm])
    kp = k[np.ix_(el, el)]
    mask = np.zeros((m.nb, m.nb), dtype=bool); mask[m.rowidx, m.block_cols()] = True
    mp = _blocks_from_dense(kp, m.blk_size[perm], mask=mask[np.ix_(perm, perm)])
    m1 = _blocks_from_dense(k, m.blk_size, mask=mask)
    d1 = m1.to_dense(oracle.density(oracle.Index(m1), m1.values, 0.1))
    dp = mp.to_dense(oracle.density(oracle.Index(mp), mp.values, 0.1))
    assert np.abs(dp - d1[np.ix_(el, el)]).max() < 1e-12


def test_grouping_one_group_is_exact(oracle):
    """L199: with all block columns in ONE group the single submatrix contains every row that has
    any stored block, i.e. the whole matrix: result = dense sign restricted to the pattern."""
    m = W.random_block_pattern(nb=10, density=0.3, max_bs=4, seed=11, ngroups=1)
    idx = oracle.Index(m)
    assert idx.sub_dim[0] == m.n_basis
    d = m.to_dense(oracle.density(idx, m.values, 0.0))
    k = m.to_dense()
    ev, v = np.linalg.eigh(k)
    dex = v[:, ev < 0] @ v[:, ev < 0].T
    mask = np.zeros_like(k, dtype=bool)
    off = m.blk_off()
    for r, c in zip(m.rowidx, m.block_cols()):
        mask[off[r]:off[r + 1], off[c]:off[c + 1]] = True
    assert np.abs(d - dex)[mask].max() < 1e-12
    assert np.all(d[~mask] == 0)


# ---------------------------------------------------------------- Algorithm 1
def test_nelec_matches_trace_and_is_monotone(oracle, cfg0):
    """Algorithm 1 (L275) vs Eq.(18): n_elec(mu) from (lam, w) equals tr(D~(mu)) of the extracted
    result; monotone non-decreasing, 0 below and n above the Gershgorin interval (P9)."""
    m = cfg0
    idx = oracle.Index(m)
    groups = np.arange(m.ngroups)
    lam, w, ptr, g = oracle.eig_groups(idx, m.values, groups, nthreads=8)
    # weights of each submatrix sum to the generating width (rows of an orthogonal Q)
    for j in range(len(g)):
        assert abs(w[ptr[j]:ptr[j + 1]].sum() - idx.gen_width[g[j]]) < 1e-12
    for mu in (0.0, -0.8):
        d = oracle.density(idx, m.values, mu, nthreads=8)
        assert abs(oracle.nelec(idx, lam, w, g, mu) - oracle.traces(idx, d, m.values)[0]) < 1e-10
    lo, hi = oracle.gershgorin_interval(m)
    kd = m.to_dense()
    ev = np.linalg.eigvalsh(kd)
    assert lo <= ev.min() and hi >= ev.max()
    assert abs(oracle.nelec(idx, lam, w, g, lo - 1e-9)) < 1e-10
    assert abs(oracle.nelec(idx, lam, w, g, hi + 1e-9) - m.n_basis) < 1e-10
    mus = np.linspace(lo, hi, 200)
    ne = np.array([oracle.nelec(idx, lam, w, g, x) for x in mus])
    assert np.all(np.diff(ne) >= -1e-12)
    # inside the gap the count is the occupied count up to the method's own error (A11)
    assert abs(oracle.nelec(idx, lam, w, g, 0.0) - m.n_occ) < 1e-2


def test_bisection_finds_gap_plateau(oracle, cfg0):
    """A11: starting outside the gap, midpoint bisection ends on the plateau whose rounded count is
    the target; with an unreachable tolerance it stops on the mu_tol / max_steps guards."""
    m = cfg0
    idx = oracle.Index(m)
    groups = np.arange(m.ngroups)
    lam, w, ptr, g = oracle.eig_groups(idx, m.values, groups, nthreads=8)
    lo, hi = oracle.gershgorin_interval(m)
    mu, ne, tr = oracle.bisect_mu(idx, lam, w, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5)
    kd = m.to_dense()
    ev = np.linalg.eigvalsh(kd)
    homo, lumo = ev[ev < 0].max(), ev[ev > 0].min()
    assert abs(ne - m.n_occ) <= 0.5 and len(tr) > 1
    assert homo - 0.2 < mu < lumo + 0.2
    mu2, ne2, tr2 = oracle.bisect_mu(idx, lam, w, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=1e-8,
                                     mu_tol=1e-6, max_steps=64)
    assert abs(ne2 - m.n_occ) > 1e-8 and len(tr2) <= 64  # unreachable by construction
    assert abs(ne2 - m.n_occ) < 1e-2


def test_flop_model_eq14_eq15(oracle):
    """Eq.(14)/(15): with one group per block column the estimated speed-up is exactly 1; merging all
    columns into one group gives S = sum_c n~_c^3 / n_basis^3; a hand-worked 3-column case."""
    from paper_2004_10811_b200 import workloads as W
    import dataclasses
    m = W.random_block_pattern(nb=12, density=0.3, max_bs=4, seed=2)
    per_col = dataclasses.replace(m, grp_ptr=np.arange(m.nb + 1, dtype=np.int32), grp_cols=np.arange(m.nb, dtype=np.int32))
    ops, ops_cols, S = oracle.flop_model(per_col, oracle.Index(per_col))
    assert ops == ops_cols and S == 1.0
    one = dataclasses.replace(m, grp_ptr=np.array([0, m.nb], np.int32), grp_cols=np.arange(m.nb, dtype=np.int32))
    idx1 = oracle.Index(one)
    ops1, ops_cols1, S1 = oracle.flop_model(one, idx1)
    assert ops_cols1 == ops_cols and ops1 == int(idx1.sub_dim[0]) ** 3
    # tridiagonal block pattern, sizes 2,3,1: columns generate n~ = 5, 6, 4; groups {0,1},{2}: n = 6, 4
    tri = W.BlockSparseSym(3, np.array([2, 3, 1], np.int32), np.array([0, 2, 5, 7], np.int64),
                           np.array([0, 1, 0, 1, 2, 1, 2], np.int32), np.zeros(4 + 6 + 6 + 9 + 3 + 3 + 1),
                           np.array([0, 2, 3], np.int32), np.array([0, 1, 2], np.int32))
    ops, ops_cols, S = oracle.flop_model(tri, oracle.Index(tri))
    assert (ops, ops_cols) == (6 ** 3 + 4 ** 3, 5 ** 3 + 6 ** 3 + 4 ** 3) and abs(S - 405 / 280) < 1e-15


def test_steering_bound_inequality(oracle, cfg0):
    """DESIGN.md reading A11c, checked with the oracle's eigendecompositions (no CUDA): for the
    Newton-Schulz iterate x_k of every eigenvalue (scalar map of Eq.(11)) and Algorithm 1's weights
    w_l = sum_{k in gen} Q_kl^2, the distance of the running count to the final count is bounded by
    1/2 sum_k min(S1_k, (S1_k + S2_k)/2), S1 = 1 - (X^2)_kk, S2 = sum_j (delta_kj - (X^2)_kj)^2 over the
    generating rows k -- and the bound tightens monotonically."""
    m = cfg0
    idx = oracle.Index(m)
    for g in (0, 7, 19):
        a = oracle.assemble(idx, m.values, g) - (-0.9) * np.eye(idx.sub_dim[g])  # mu inside the occupied band
        lam, q = np.linalg.eigh(a)
        gen = []
        for c in idx.grp_cols[idx.grp_ptr[g]:idx.grp_ptr[g + 1]]:
            t = int(np.searchsorted(idx.sub_blocks[idx.sub_ptr[g]:idx.sub_ptr[g + 1]], c))
            o = int(idx.sub_off[idx.sub_ptr[g] + t])
            gen.extend(range(o, o + int(m.blk_size[c])))
        w = (q[gen, :] ** 2).sum(0)
        n_final = (w * 0.5 * (1.0 - np.sign(lam))).sum()
        x = lam / (np.abs(lam).max() * 1.02)
        prev = np.inf
        for k in range(1, 25):
            x = 0.5 * x * (3.0 - x * x)
            xm = (q * x) @ q.T
            y = xm @ xm
            n_k = (0.5 * (1.0 - np.diag(xm)[gen])).sum()
            s1 = np.maximum(1.0 - np.diag(y)[gen], 0.0)
            s2 = ((np.eye(len(lam))[gen] - y[gen]) ** 2).sum(1)
            bound = (0.5 * np.minimum(s1, 0.5 * (s1 + s2))).sum()
            assert abs(n_final - n_k) <= bound + 1e-10
            assert bound <= prev + 1e-10
            prev = bound
        assert prev < 1e-2


def test_predicted_residual_bound(oracle, cfg0):
    """DESIGN.md reading A9b: for a symmetric iterate, E_{k+1} = X_{k+1}^2 - I = -3/4 E_k^2 + 1/4 E_k^3 with
    E_k = X_k^2 - I (Eq.(11) L97 squared), hence ||E_{k+1}||_F <= 3/4 ||E_k||_F^2 + 1/4 ||E_k||_F^3."""
    m = cfg0
    idx = oracle.Index(m)
    a = oracle.assemble(idx, m.values, 3)
    x = a / (np.abs(np.linalg.eigvalsh(a)).max() * 1.01)
    eye = np.eye(len(a))
    for k in range(12):
        e = x @ x - eye
        xn = 0.5 * x @ (3.0 * eye - x @ x)
        en = xn @ xn - eye
        assert np.abs(en - (-0.75 * e @ e + 0.25 * e @ e @ e)).max() <= 1e-12
        f = np.linalg.norm(e)
        assert np.linalg.norm(en) <= 0.75 * f * f + 0.25 * f ** 3 + 1e-13
        x = xn


def test_lanczos_quadrature_is_gauss_quadrature(oracle):
    """A11d pins: (1) the sparse assembly equals the dense one; (2) with as many steps as rows the Ritz
    values are the eigenvalues and the weights the squared projections of the start vector (textbook);
    (3) with k < n steps the rule integrates the moments v^T K^j v exactly for j <= 2k - 1, the weights
    sum to 1 and the Ritz values lie inside the spectrum."""
    m = W.random_block_pattern(nb=10, density=0.4, max_bs=3, seed=5)
    kd = m.to_dense()
    A = oracle.sparse_matrix(m)
    assert np.array_equal(A.toarray(), kd)
    n = kd.shape[0]
    lam, Q = np.linalg.eigh(kd)
    v = oracle.v_start_of(n)
    assert abs(v @ v - 1.0) < 1e-14 and set(np.round(np.abs(v) * np.sqrt(n), 12)) == {1.0}
    k = 6
    th, w = oracle.lanczos_quadrature(m, steps=k)
    assert len(th) == k and abs(w.sum() - 1.0) < 1e-13
    assert lam[0] - 1e-12 <= th[0] and th[-1] <= lam[-1] + 1e-12
    scale = max(abs(lam[0]), abs(lam[-1]))
    for j in range(2 * k):
        exact = v @ np.linalg.matrix_power(kd / scale, j) @ v
        assert abs(np.sum(w * (th / scale) ** j) - exact) < 1e-11, j
    j = 2 * k  # the first moment the k-point rule does NOT reproduce
    assert abs(np.sum(w * (th / scale) ** j) - v @ np.linalg.matrix_power(kd / scale, j) @ v) > 1e-9
    small = W.random_block_pattern(nb=3, density=1.0, max_bs=3, seed=2)
    ks = small.to_dense()
    ns = ks.shape[0]
    th, w = oracle.lanczos_quadrature(small, steps=ns)
    lam, Q = np.linalg.eigh(ks)
    assert np.allclose(th, lam, atol=1e-10)
    assert np.allclose(w, (Q.T @ oracle.v_start_of(ns)) ** 2, atol=1e-9)
    lo, hi = oracle.lanczos_interval(th)
    assert lo < lam[0] and hi > lam[-1]


def test_mu_start_rule(oracle, cfg0):
    """A11e: hand-worked cases of the step-0 rule (the caller's mu is kept only inside the Ritz interval taken for
    the gap, the estimate must lie strictly inside the bracket); on the water-like workload a start from mu0 = -1
    goes straight to the estimate and the search ends after ONE evaluation on the plateau of the target, the same
    plateau the search of reading A11 (which spends an evaluation on mu0) ends on."""
    th = np.array([0.0, 1.0, 2.0, 10.0, 11.0])
    w = np.full(5, 0.2)
    assert oracle.mu_guess_interval(th, w, 0.6) == (2.0, 10.0)
    assert oracle.mu_start(th, w, 0.6, mu0=-1.0, lo=-3.0, hi=12.0) == 6.0   # mu0 outside (2, 10): the estimate
    assert oracle.mu_start(th, w, 0.6, mu0=10.5, lo=-3.0, hi=12.0) == 6.0
    assert oracle.mu_start(th, w, 0.6, mu0=2.0, lo=-3.0, hi=12.0) == 6.0    # the interval is open
    assert oracle.mu_start(th, w, 0.6, mu0=3.0, lo=-3.0, hi=12.0) == 3.0    # inside: the caller knows better
    assert oracle.mu_start(th, w, 0.6, mu0=9.9, lo=-3.0, hi=12.0) == 9.9
    assert oracle.mu_start(th, w, 0.6, mu0=-1.0, lo=-3.0, hi=6.0) == -1.0   # estimate not strictly inside the bracket
    assert oracle.mu_start(th, w, 0.6, mu0=-1.0, lo=6.0, hi=12.0) == -1.0
    m = cfg0
    th, w = oracle.lanczos_quadrature(m, steps=24)
    frac = m.n_occ / m.n_basis
    idx = oracle.Index(m)
    lam, wq, ptr, g = oracle.eig_groups(idx, m.values, np.arange(m.ngroups), nthreads=8)
    lo, hi = oracle.gershgorin_interval(m)
    llo, lhi = oracle.lanczos_interval(th)
    lo, hi = max(lo, llo), min(hi, lhi)
    guess = oracle.mu_guess(th, w, frac)
    start = oracle.mu_start(th, w, frac, -1.0, lo, hi)
    assert start == guess
    mu_e, ne_e, tr_e = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=start, lo=lo, hi=hi, tol_n=0.5, mu_first=guess)
    mu_d, ne_d, tr_d = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5, mu_first=guess)
    assert len(tr_e) == 1 and len(tr_d) == 2 and mu_e == mu_d and ne_e == ne_d
    a, b = oracle.mu_guess_interval(th, w, frac)
    inside = 0.25 * a + 0.75 * b
    assert oracle.mu_start(th, w, frac, inside, lo, hi) == inside


def test_mu_guess_rule(oracle, cfg0):
    """A11d: a hand-worked case of the widest-interval rule; on the water-like workload the guess lands
    inside the HOMO-LUMO gap, and the search with that first step ends on the same plateau in fewer
    evaluations than the midpoint search; a guess outside the bracket is ignored."""
    th = np.array([0.0, 1.0, 2.0, 10.0, 11.0])
    w = np.full(5, 0.2)
    assert oracle.mu_guess(th, w, 0.6) == 6.0      # cum = .2 .4 .6 .8: m = 2, window 0..3, widest (2, 10)
    assert oracle.mu_guess(th, w, 0.05) == 6.0     # m = 0, window 0..2 still holds (2, 10)
    th2 = np.array([0.0, 1.0, 2.0, 2.5, 3.0, 3.5, 12.0])
    assert oracle.mu_guess(th2, np.full(7, 1 / 7), 0.1) == 0.5  # m = 0, window 0..2: first of the widest
    m = cfg0
    kd = m.to_dense()
    ev = np.linalg.eigvalsh(kd)
    homo, lumo = ev[m.n_occ - 1], ev[m.n_occ]
    th, w = oracle.lanczos_quadrature(m, steps=24)
    guess = oracle.mu_guess(th, w, m.n_occ / kd.shape[0])
    assert homo < guess < lumo
    idx = oracle.Index(m)
    lam, wq, ptr, g = oracle.eig_groups(idx, m.values, np.arange(m.ngroups), nthreads=8)
    lo, hi = oracle.gershgorin_interval(m)
    llo, lhi = oracle.lanczos_interval(th)
    lo, hi = max(lo, llo), min(hi, lhi)
    mu_a, ne_a, tr_a = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5)
    mu_b, ne_b, tr_b = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5,
                                        mu_first=guess)
    assert len(tr_b) == 2 and tr_b[1][0] == guess and len(tr_a) >= len(tr_b)
    assert abs(ne_a - m.n_occ) <= 0.5 and abs(ne_b - m.n_occ) <= 0.5
    _, _, tr_c = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5, mu_first=hi + 1.0)
    assert tr_c == tr_a
    _, _, tr_d = oracle.bisect_mu(idx, lam, wq, g, m.n_occ, mu0=-1.0, lo=lo, hi=hi, tol_n=0.5, mu_first=-2.0)
    assert tr_d == tr_a  # below the evaluated mu0: outside the bracket after step 0


def test_rescaled_newton_schulz_scalar_properties():
    """Reading A8b, the properties the schedule relies on, checked numerically on the scalar map
    f(x) = 1/2 al x (3 - al^2 x^2): with al = sqrt(3 / (1 + l + l^2)) both ends of [l, 1] map to the same
    value, the image of [l, 1] is [f(l), 1], signs are kept for al <= 1.7 and |x| <= 1, and the iteration
    count to |1 - x| < 1e-13 over [l0, 1] is smaller than that of the plain map."""
    xs = np.linspace(0.0, 1.0, 20001)
    for l in (1e-4, 0.01, 0.08, 0.3, 0.7, 0.89):
        al = np.sqrt(3.0 / (1.0 + l + l * l))
        f = lambda x: 0.5 * al * x * (3.0 - al * al * x * x)
        assert abs(f(l) - f(1.0)) < 1e-14
        img = f(xs[xs >= l])
        assert img.min() >= f(l) - 1e-14 and img.max() <= 1.0 + 1e-14 and img.max() > 1.0 - 1e-6
        assert f(l) > 0.5 * l * (3.0 - l * l)  # the lower end moves faster than under the plain map
    for al in (1.5, 1.7):
        assert np.all(0.5 * al * xs[1:] * (3.0 - al * al * xs[1:] ** 2) > 0.0)
    def count(l0, rescale):
        x = np.linspace(l0, 1.0, 4001)
        l = l0
        for k in range(200):
            if np.abs(1.0 - x).max() < 1e-13:
                return k
            al = min(np.sqrt(3.0 / (1.0 + l + l * l)), 1.5 if k == 0 else 1.7) if (rescale and l < 0.9999) else 1.0
            g = lambda t: 0.5 * al * t * (3.0 - al * al * t * t)
            x, l = g(x), min(g(l), g(1.0), 1.0)
        return 200
    for l0 in (0.01, 0.08, 0.2):
        assert count(l0, True) < count(l0, False)


# ---------------------------------------------------------------- finite temperature (L255)
def test_golden_fermi_2x2(oracle):
    """L255: signum of Eq.(17) replaced by the Fermi function; closed form on A^2 = 25 I (hand-derived)."""
    g = _load("fermi_2x2.txt")
    m = _blocks_from_dense(g[:2], [2])
    idx = oracle.Index(m)
    d = oracle.density_fermi(idx, m.values, 0.0, 2.0)
    assert np.allclose(m.to_dense(d), g[2:], atol=1e-15)


def test_fermi_diagonal_and_limits(oracle, cfg0):
    """Diagonal matrix: elementwise Fermi function (scipy's logistic as the independent witness);
    kT -> 0: the zero-temperature D~ (gap 0.3 >> kT); f(-x) = 1 - f(x): D~(-K, -mu, kT) = I - D~(K, mu, kT);
    kT -> infinity: every occupation 1/2."""
    from scipy.special import expit
    dv = np.array([-2.0, 0.5, 3.0, -1e-3, 0.25, -0.5, 1.0, 2.0, -4.0])
    m = W.dense_batch_as_blocks(np.diag(dv)[None])
    idx = oracle.Index(m)
    for mu, kT in ((0.0, 0.3), (0.4, 0.05), (-1.0, 2.0)):
        d = m.to_dense(oracle.density_fermi(idx, m.values, mu, kT))
        assert np.abs(d - np.diag(expit(-(dv - mu) / kT))).max() < 1e-15
        assert np.abs(oracle.occupation(dv, mu, kT) - expit(-(dv - mu) / kT)).max() < 1e-15
    assert np.array_equal(oracle.occupation([-1.0, 0.0, 2.0], 0.0, 0.0), [1.0, 0.5, 0.0])  # Eq.(12) at kT = 0
    m = cfg0
    idx = oracle.Index(m)
    groups = np.array([0, 7, 19], dtype=np.int32)
    d0 = oracle.density(idx, m.values, 0.0, groups)
    dT = oracle.density_fermi(idx, m.values, 0.0, 1e-3, groups)
    assert np.abs(dT - d0).max() < 1e-13
    dp = oracle.density_fermi(idx, m.values, 0.2, 0.1, groups)
    dm = oracle.density_fermi(idx, -m.values, -0.2, 0.1, groups)
    eye = np.zeros_like(m.values)
    vo, bc = m.val_off(), m.block_cols()
    for b in np.nonzero(m.rowidx == bc)[0]:
        n = int(m.blk_size[bc[b]])
        eye[vo[b]:vo[b + 1]] = np.eye(n).reshape(-1)
    cols = oracle.column_ids_of_groups(idx, groups)
    mask = np.repeat(np.isin(bc, cols), np.diff(vo))
    assert np.abs((dp + dm - eye)[mask]).max() < 1e-12
    dh = oracle.density_fermi(idx, m.values, 0.0, 1e9, groups)
    assert np.abs((dh - 0.5 * eye)[mask]).max() < 1e-8


def test_fermi_full_cutoff_equals_lapack(oracle):
    """P5 at finite temperature: with every a_i the whole matrix, D~ = U f(Lambda) U^T of LAPACK's eigh,
    tr D~ = sum f(lambda), and Algorithm 1's count from (lambda, w) equals tr D~ (L275 with f for signum)."""
    m = W.water_like(8, "SZV", cutoff=1e9, seed=3)
    idx = oracle.Index(m)
    mu, kT = 0.1, 0.05
    dd = oracle.density_fermi(idx, m.values, mu, kT, nthreads=4)
    ev, v = np.linalg.eigh(m.to_dense())
    f = 1.0 / (1.0 + np.exp((ev - mu) / kT))
    assert np.abs(m.to_dense(dd) - (v * f) @ v.T).max() < 1e-12
    td, tdk = oracle.traces(idx, dd, m.values)
    assert abs(td - f.sum()) < 1e-11 and abs(tdk - (f * ev).sum()) < 1e-11
    lam, w, ptr, g = oracle.eig_groups(idx, m.values, nthreads=4)
    assert abs(oracle.nelec_fermi(idx, lam, w, g, mu, kT) - td) < 1e-11


def test_fermi_count_is_continuous_and_bisection_meets_1e8(oracle, cfg0):
    """At kT > 0 the electron count is continuous and strictly increasing in mu (no plateau offset problem
    of reading A11): the literal tolerance 1e-8 of BASELINE config 4 is reachable; nelec_fermi = tr D~."""
    m = cfg0
    idx = oracle.Index(m)
    lam, w, ptr, g = oracle.eig_groups(idx, m.values, nthreads=4)
    kT = 0.02
    mus = np.linspace(-2.5, 2.5, 41)
    ne = np.array([oracle.nelec_fermi(idx, lam, w, g, x, kT) for x in mus])
    assert np.all(np.diff(ne) > 0) and ne[0] < 1e-6 and abs(ne[-1] - m.n_basis) < 1e-6
    lo, hi = oracle.gershgorin_interval(m)
    mu, ne_f, trace = oracle.bisect_mu_fermi(idx, lam, w, g, m.n_occ, -1.0, lo, hi, 1e-8, kT, mu_tol=1e-14)
    assert abs(ne_f - m.n_occ) <= 1e-8 and len(trace) < 64
    td, _ = oracle.traces(idx, oracle.density_fermi(idx, m.values, mu, kT, nthreads=4), m.values)
    assert abs(td - ne_f) < 1e-9


# ---------------------------------------------------------------- load balancing (IV-E L235)
def test_partition_rule_hand_worked_and_properties(oracle):
    """L235: greedy consecutive chunks by n^3.  Hand-worked: dims (2,2,2,2,2,2,2,2), 4 ranks: total 64,
    target 16 -> two per rank.  dims (10,1,1,1,1,1), 3 ranks: total 1005, target 335: rank 0 stops after the
    first (1000 >= 335), rank 1 takes while below target but must leave one: (1,1,1,1), rank 2 the last.
    dims (1,1,1,1,1,10), 3 ranks: rank 0 would go on (load 4 < 335) but must leave two: takes four.
    Properties on random sizes: a contiguous cover, >= 1 each, every rank but the last below
    target + max n^3; the last at most the target when nobody was cut short by the leave-one rule."""
    assert oracle.partition_groups([2] * 8, 4) == [0, 2, 4, 6, 8]
    assert oracle.partition_groups([10, 1, 1, 1, 1, 1], 3) == [0, 1, 5, 6]
    assert oracle.partition_groups([1, 1, 1, 1, 1, 10], 3) == [0, 4, 5, 6]
    assert oracle.partition_groups([5, 7], 1) == [0, 2]
    rng = np.random.default_rng(0)
    for trial in range(50):
        ng = int(rng.integers(1, 200))
        world = int(rng.integers(1, min(ng, 16) + 1))
        dims = rng.integers(1, 300, ng)
        f = oracle.partition_groups(dims, world)
        assert f[0] == 0 and f[-1] == ng and all(f[r + 1] > f[r] for r in range(world))
        n3 = dims.astype(object) ** 3
        total, mx = int(n3.sum()), int(n3.max())
        loads = [int(n3[f[r]:f[r + 1]].sum()) for r in range(world)]
        cut = [f[r + 1] == ng - (world - 1 - r) for r in range(world - 1)]
        for r in range(world - 1):
            assert loads[r] * world < total + mx * world
        if not any(cut):
            assert loads[-1] * world <= total


def test_library_partition_equals_oracle(oracle):
    """sm_partition_groups (host function of the C-ABI, no GPU) against the oracle's restatement."""
    from paper_2004_10811_b200 import binding as B
    rng = np.random.default_rng(1)
    for trial in range(100):
        ng = int(rng.integers(1, 300))
        world = int(rng.integers(1, min(ng, 12) + 1))
        dims = rng.integers(1, 2500, ng).astype(np.int32)
        assert list(B.sm_partition_groups(dims, world)) == oracle.partition_groups(dims, world)
    m = W.make_config(2)
    idx = oracle.Index(m)
    for world in (2, 3, 8):
        assert list(B.sm_partition_groups(idx.sub_dim, world)) == oracle.partition_groups(idx.sub_dim, world)
