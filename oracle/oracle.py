"""ctypes front-end of the C oracle + the mu loop of Algorithm 1.

TEST INFRASTRUCTURE, NOT PRODUCT CODE: importable only from tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs.  Shares nothing with the CUDA path; the
only common module is the seeded input generator (paper_2004_10811_b200.workloads), which
contains none of the method's arithmetic.

All arithmetic of the method lives in submatrix_oracle.c; this file marshals arrays and runs
the scalar mu loop:
    n_elec(mu) = sum_i sum_{k in gen(i)} ( 1/2 - 1/2 sum_l Q_{k,l}^2 signum(lambda_l - mu) )
               = sum_i ( |gen(i)|/2 - 1/2 sum_l w_{i,l} signum(lambda_{i,l} - mu) )   (Algorithm 1)
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_index_count.restype = C.c_int64
        _lib.orc_jacobi_eig.restype = C.c_int
        _lib.orc_dense_sign.restype = C.c_int
        _lib.orc_occupation.restype = C.c_double
        _lib.orc_occupation.argtypes = [C.c_double, C.c_double, C.c_double]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Index:
    """Submatrix index of a pattern + grouping (step "index", L125/L199)."""

    def __init__(self, m):
        L = lib()
        self.m = m
        self.blk_size, self.colptr, self.rowidx = _i32(m.blk_size), _i64(m.colptr), _i32(m.rowidx)
        self.grp_ptr, self.grp_cols = _i32(m.grp_ptr), _i32(m.grp_cols)
        ng = len(self.grp_ptr) - 1
        self.sub_ptr = np.zeros(ng + 1, dtype=np.int64)
        tot = L.orc_index_count(C.c_int32(m.nb), _p(self.colptr, C.c_int64), _p(self.rowidx, C.c_int32),
                                C.c_int32(ng), _p(self.grp_ptr, C.c_int32), _p(self.grp_cols, C.c_int32),
                                _p(self.sub_ptr, C.c_int64))
        self.sub_blocks = np.zeros(max(tot, 1), dtype=np.int32)[:tot]
        self.sub_off = np.zeros(max(tot, 1), dtype=np.int32)[:tot]
        self.sub_dim = np.zeros(ng, dtype=np.int32)
        self.gen_pos = np.zeros(len(self.grp_cols), dtype=np.int32)
        L.orc_index_fill(C.c_int32(m.nb), _p(self.blk_size, C.c_int32), _p(self.colptr, C.c_int64),
                         _p(self.rowidx, C.c_int32), C.c_int32(ng), _p(self.grp_ptr, C.c_int32),
                         _p(self.grp_cols, C.c_int32), _p(self.sub_ptr, C.c_int64),
                         _p(self.sub_blocks, C.c_int32), _p(self.sub_off, C.c_int32),
                         _p(self.sub_dim, C.c_int32), _p(self.gen_pos, C.c_int32))
        self.val_off = _i64(m.val_off())
        self.ngroups = ng
        # number of generating basis functions per group (|gen(i)| in Algorithm 1)
        self.gen_width = np.array([int(self.blk_size[self.grp_cols[self.grp_ptr[i]:self.grp_ptr[i + 1]]].sum())
                                   for i in range(ng)], dtype=np.int64)


def assemble(idx: Index, values, i: int) -> np.ndarray:
    """Dense a_i (step "assemble", L125).  Returns an (n_i, n_i) array (symmetric)."""
    n = int(idx.sub_dim[i])
    a = np.zeros((n, n))
    s, e = int(idx.sub_ptr[i]), int(idx.sub_ptr[i + 1])
    S, So = _i32(idx.sub_blocks[s:e]), _i32(idx.sub_off[s:e])
    v = _f64(values)
    lib().orc_assemble(_p(idx.blk_size, C.c_int32), _p(idx.colptr, C.c_int64), _p(idx.rowidx, C.c_int32),
                       _p(idx.val_off, C.c_int64), _p(v, C.c_double), C.c_int64(e - s),
                       _p(S, C.c_int32), _p(So, C.c_int32), C.c_int32(n), _p(a, C.c_double))
    return a.T  # column-major -> numpy view


def jacobi_eig(a: np.ndarray):
    """Cyclic Jacobi: returns (lam[n], Q[n,n]) with a = Q diag(lam) Q^T (Eq.(17))."""
    n = a.shape[0]
    w = _f64(a).copy()
    qt = np.zeros((n, n))
    lam = np.zeros(n)
    lib().orc_jacobi_eig(C.c_int32(n), _p(w, C.c_double), _p(qt, C.c_double), _p(lam, C.c_double))
    return lam, qt.T.copy()


def dense_sign(a: np.ndarray, mu: float = 0.0) -> np.ndarray:
    """sign(a - mu I) of one dense symmetric matrix via Jacobi (Eq.(17), Eq.(12))."""
    n = a.shape[0]
    aa = _f64(a)
    s = np.zeros((n, n))
    lib().orc_dense_sign(C.c_int32(n), _p(aa, C.c_double), C.c_double(mu), _p(s, C.c_double), None)
    return s


def _run_groups(idx: Index, values, groups, mu, do_extract, want_eig, nthreads):
    groups = _i32(np.arange(idx.ngroups) if groups is None else groups)
    v = _f64(values)
    out = np.zeros_like(v) if do_extract else None
    lw_ptr = np.zeros(len(groups) + 1, dtype=np.int64)
    np.cumsum(idx.sub_dim[groups], out=lw_ptr[1:])
    lam = np.zeros(int(lw_ptr[-1])) if want_eig else None
    w = np.zeros(int(lw_ptr[-1])) if want_eig else None
    lib().orc_submatrix_groups(
        _p(idx.blk_size, C.c_int32), _p(idx.colptr, C.c_int64), _p(idx.rowidx, C.c_int32),
        _p(idx.val_off, C.c_int64), _p(v, C.c_double), _p(idx.grp_ptr, C.c_int32),
        _p(idx.grp_cols, C.c_int32), _p(idx.sub_ptr, C.c_int64), _p(idx.sub_blocks, C.c_int32),
        _p(idx.sub_off, C.c_int32), _p(idx.sub_dim, C.c_int32), _p(idx.gen_pos, C.c_int32),
        C.c_int32(len(groups)), _p(groups, C.c_int32), C.c_double(mu), C.c_int32(1 if do_extract else 0),
        _p(out, C.c_double), _p(lw_ptr, C.c_int64), _p(lam, C.c_double), _p(w, C.c_double),
        C.c_int32(nthreads))
    return out, lam, w, lw_ptr, groups


def density(idx: Index, values, mu: float, groups=None, nthreads: int = 0) -> np.ndarray:
    """D~ = 1/2 (I - sign(K~ - mu I)) by the submatrix method on the input pattern (L123-127).
    Only the block columns of the listed groups are filled (others stay 0)."""
    return _run_groups(idx, values, groups, mu, True, False, nthreads)[0]


def eig_groups(idx: Index, values, groups=None, nthreads: int = 0):
    """Eigenvalues lambda_{i,l} and weights w_{i,l} of the listed groups (Algorithm 1).
    Returns (lam, w, ptr, groups)."""
    _, lam, w, ptr, g = _run_groups(idx, values, groups, 0.0, False, True, nthreads)
    return lam, w, ptr, g


def nelec(idx: Index, lam, w, groups, mu: float) -> float:
    """Algorithm 1 inner loops for one mu."""
    ngen = float(idx.gen_width[groups].sum())
    return 0.5 * ngen - 0.5 * float(np.sum(w * np.sign(lam - mu)))


def occupation(lam, mu: float, kT: float = 0.0) -> np.ndarray:
    """Occupations f_l (L255, reading A18): Fermi function 1 / (1 + exp((lam - mu) / kT)) for kT > 0, else
    1/2 (1 - signum(lam - mu)).  Evaluated by the C oracle, element by element."""
    L = lib()
    return np.array([L.orc_occupation(float(x), float(mu), float(kT)) for x in np.atleast_1d(lam)])


def nelec_fermi(idx: Index, lam, w, groups, mu: float, kT: float) -> float:
    """Algorithm 1's count with the Fermi function in place of signum (L255): sum_i sum_l w_il f(lam_il)."""
    if kT <= 0.0:
        return nelec(idx, lam, w, groups, mu)
    return float(np.sum(w / (1.0 + np.exp((lam - mu) / kT))))


def density_fermi(idx: Index, values, mu: float, kT: float, groups=None, nthreads: int = 0) -> np.ndarray:
    """D~ = f(K~ - mu I) by the submatrix method at electronic temperature kT (L255): per submatrix
    Q f(Lambda) Q^T, generating columns copied back on the input pattern."""
    groups = _i32(np.arange(idx.ngroups) if groups is None else groups)
    v = _f64(values)
    out = np.zeros_like(v)
    lib().orc_submatrix_groups_fermi(
        _p(idx.blk_size, C.c_int32), _p(idx.colptr, C.c_int64), _p(idx.rowidx, C.c_int32),
        _p(idx.val_off, C.c_int64), _p(v, C.c_double), _p(idx.grp_ptr, C.c_int32),
        _p(idx.grp_cols, C.c_int32), _p(idx.sub_ptr, C.c_int64), _p(idx.sub_blocks, C.c_int32),
        _p(idx.sub_off, C.c_int32), _p(idx.sub_dim, C.c_int32), _p(idx.gen_pos, C.c_int32),
        C.c_int32(len(groups)), _p(groups, C.c_int32), C.c_double(mu), C.c_double(kT), _p(out, C.c_double),
        C.c_int32(nthreads))
    return out


def bisect_mu_fermi(idx: Index, lam, w, groups, n_target: float, mu0: float, lo: float, hi: float, tol_n: float,
                    kT: float, mu_tol: float = 1e-6, max_steps: int = 64):
    """Algorithm 1 (L272-276) with the rule of reading A11 on the finite-temperature count (continuous and
    strictly increasing in mu for kT > 0, so tol_n is reachable).  Same returns as bisect_mu."""
    trace = []
    mu = mu0
    best = None
    for _ in range(max_steps):
        ne = nelec_fermi(idx, lam, w, groups, mu, kT)
        g = ne - n_target
        trace.append((mu, ne))
        if best is None or abs(g) < abs(best[1]):
            best = (mu, g)
        if abs(g) <= tol_n:
            break
        if g < 0:
            lo = max(lo, mu)
        else:
            hi = min(hi, mu)
        if hi - lo <= mu_tol:
            break
        mu = 0.5 * (lo + hi)
    return best[0], best[1] + n_target, trace


def column_ids_of_groups(idx: Index, groups) -> np.ndarray:
    return np.concatenate([idx.grp_cols[idx.grp_ptr[g]:idx.grp_ptr[g + 1]] for g in groups]).astype(np.int32)


def traces(idx: Index, D, K, cols=None):
    """(tr D, tr D K) (Eq.(18), Eq.(10)); restricted to block columns `cols` if given."""
    td, tdk = C.c_double(0), C.c_double(0)
    D, K = _f64(D), _f64(K)
    cc = _i32(cols) if cols is not None else None
    lib().orc_traces(C.c_int32(idx.m.nb), _p(idx.blk_size, C.c_int32), _p(idx.colptr, C.c_int64),
                     _p(idx.rowidx, C.c_int32), _p(idx.val_off, C.c_int64), _p(D, C.c_double),
                     _p(K, C.c_double), C.c_int32(-1 if cc is None else len(cc)), _p(cc, C.c_int32),
                     C.byref(td), C.byref(tdk))
    return td.value, tdk.value


def flop_model(m, idx: "Index"):
    """PAPER.md Eq.(14) L201 and Eq.(15), written out: operations ~ sum_i n_i^3 for the given
    grouping; S = sum over single block columns c of n~_c^3 (n~_c = dimension of the submatrix that
    column c alone generates = total height of its stored blocks) divided by that."""
    ops = sum(int(n) ** 3 for n in idx.sub_dim)
    ops_cols = 0
    for c in range(m.nb):
        rows = m.rowidx[m.colptr[c]:m.colptr[c + 1]]
        ops_cols += int(m.blk_size[rows].sum()) ** 3
    return ops, ops_cols, (ops_cols / ops if ops else 0.0)


def partition_groups(sub_dim, world: int):
    """PAPER.md IV-E L235 (reading A19): consecutive chunks of submatrices; a rank is given the next submatrix
    "as long as" its load (sum of n^3 so far) "is expected to be lower than FLOP_total / #ranks", and
    "each rank obtains at least one submatrix" (so a rank also stops when only one submatrix per later rank
    is left); the last rank takes the rest.  Returns first[world + 1]."""
    n3 = [int(n) ** 3 for n in sub_dim]
    ng = len(n3)
    assert 1 <= world <= max(ng, 1)
    total = sum(n3)
    first, i = [], 0
    for r in range(world):
        first.append(i)
        if r == world - 1:
            i = ng
            break
        load = 0
        taken = 0
        while i < ng - (world - 1 - r) and (taken == 0 or load * world < total):
            load += n3[i]
            i += 1
            taken += 1
    first.append(ng)
    return first


def gershgorin_interval(m) -> tuple[float, float]:
    """Gershgorin interval of the whole block-sparse matrix: bracket for the mu loop (A11)."""
    cols = m.block_cols()
    voff = m.val_off()
    boff = m.blk_off()
    n = int(boff[-1])
    diag = np.zeros(n)
    rad = np.zeros(n)
    for b in range(m.nnzb):
        r, c = int(m.rowidx[b]), int(cols[b])
        br, bc = int(m.blk_size[r]), int(m.blk_size[c])
        blk = m.values[voff[b]:voff[b + 1]].reshape(bc, br)  # [q, e] column-major
        colsum = np.abs(blk).sum(axis=1)
        if r == c:
            d = np.diagonal(blk).copy()
            diag[boff[c]:boff[c] + bc] = d
            colsum = colsum - np.abs(d)
        rad[boff[c]:boff[c] + bc] += colsum
    return float((diag - rad).min()), float((diag + rad).max())


def sparse_matrix(m):
    """The block-sparse K~ as a scipy CSC matrix (block (r, c) stored column-major, bs[c] columns of
    bs[r] values each)."""
    import scipy.sparse as sp
    cols = m.block_cols()
    voff = m.val_off()
    boff = m.blk_off()
    n = int(boff[-1])
    ri, ci = [], []
    for b in range(m.nnzb):
        r, c = int(m.rowidx[b]), int(cols[b])
        br, bc = int(m.blk_size[r]), int(m.blk_size[c])
        ri.append(np.tile(np.arange(boff[r], boff[r] + br), bc))
        ci.append(np.repeat(np.arange(boff[c], boff[c] + bc), br))
    ri = np.concatenate(ri) if ri else np.zeros(0, dtype=np.int64)
    ci = np.concatenate(ci) if ci else np.zeros(0, dtype=np.int64)
    return sp.csc_matrix((np.asarray(m.values[:len(ri)], dtype=np.float64), (ri, ci)), shape=(n, n))


def lanczos_quadrature(m, steps: int = 24):
    """Reading A11d: `steps` steps of the plain Lanczos recurrence on K~ (no
    re-orthogonalisation) from the counter-based start vector v_i = +-1/sqrt(n) (sign = bit 0 of the
    integer hash h = i * 2654435761; h ^= h >> 15; h *= 2246822519; h ^= h >> 13 in 32-bit unsigned
    arithmetic).  Returns the Ritz values theta_j (eigenvalues of the tridiagonal T, ascending) and the
    Gauss quadrature weights w_j = (first component of T's j-th eigenvector)^2, for which
    v^T f(K~) v ~ sum_j w_j f(theta_j), exact for polynomials of degree < 2 steps."""
    A = sparse_matrix(m)
    n = A.shape[0]
    v = v_start_of(n)
    vp = np.zeros(n)
    al, be = [], []
    b = 0.0
    for _ in range(min(steps, n)):
        w = A @ v
        a = float(w @ v)
        w = w - a * v - b * vp
        b = float(np.sqrt(w @ w))
        al.append(a)
        be.append(b)
        if not b > 1e-300:
            break
        vp, v = v, w / b
    T = np.diag(al) + np.diag(be[:len(al) - 1], 1) + np.diag(be[:len(al) - 1], -1)
    th, U = np.linalg.eigh(T)
    return th, U[0] ** 2


def v_start_of(n: int) -> np.ndarray:
    """The start vector of lanczos_quadrature (for the moment pins)."""
    i = np.arange(n, dtype=np.uint64)
    h = (i * 2654435761) & 0xFFFFFFFF
    h ^= h >> 15
    h = (h * 2246822519) & 0xFFFFFFFF
    h ^= h >> 13
    return np.where(h & 1, 1.0, -1.0) / np.sqrt(n)


def lanczos_interval(th, margin: float = 0.03):
    """Reading A8: the extreme Ritz values widened by margin * spread (the interlacing interval)."""
    spread = float(th[-1] - th[0])
    return float(th[0]) - margin * spread, float(th[-1]) + margin * spread


def mu_guess_interval(th, w, frac: float):
    """Reading A11d: cum_j = sum_{l <= j} w_l estimates the fraction of eigenvalues of K~ at or below
    theta_j.  m = the node (last excluded) whose cum is nearest to the target filling `frac`; among the
    Ritz intervals (theta_i, theta_i+1), m-2 <= i <= m+2, the widest one is taken for the gap."""
    k = len(th)
    cum = np.cumsum(w) / np.sum(w)
    m = int(np.argmin(np.abs(cum[:k - 1] - frac)))
    best = max(0, m - 2)
    for i in range(best + 1, min(k - 2, m + 2) + 1):
        if th[i + 1] - th[i] > th[best + 1] - th[best]:
            best = i
    return float(th[best]), float(th[best + 1])


def mu_guess(th, w, frac: float) -> float:
    """Reading A11d: the midpoint of the Ritz interval taken for the gap."""
    a, b = mu_guess_interval(th, w, frac)
    return 0.5 * (a + b)


def mu_start(th, w, frac: float, mu0: float, lo: float, hi: float) -> float:
    """Reading A11e: the mu of step 0.  The caller's mu0 if it lies strictly inside the Ritz interval taken
    for the gap (it is then as good as the estimate), or if the estimate is not strictly inside the
    bracket [lo, hi]; otherwise the estimate of reading A11d."""
    a, b = mu_guess_interval(th, w, frac)
    guess = 0.5 * (a + b)
    if lo < guess < hi and not (a < mu0 < b):
        return guess
    return mu0


def bisect_mu(idx: Index, lam, w, groups, n_target: float, mu0: float, lo: float, hi: float,
              tol_n: float, mu_tol: float = 1e-6, max_steps: int = 64, mu_first: float | None = None):
    """Algorithm 1 (L272-276) with the update rule of reading A11: evaluate mu0, then
    midpoint bisection on g(mu) = n_elec(mu) - n_target inside [lo, hi] (raise mu if g < 0).
    Stops on |g| <= tol_n, bracket width <= mu_tol, or max_steps; returns the evaluated mu with
    the smallest |g| and the trace [(mu, n_elec), ...].  Reading A11d: if mu_first is given and lies
    strictly inside the bracket after step 0, step 1 evaluates it instead of the midpoint."""
    trace = []
    mu = mu0
    best = None
    for _ in range(max_steps):
        ne = nelec(idx, lam, w, groups, mu)
        g = ne - n_target
        trace.append((mu, ne))
        if best is None or abs(g) < abs(best[1]):
            best = (mu, g)
        if abs(g) <= tol_n:
            break
        if g < 0:
            lo = max(lo, mu)
        else:
            hi = min(hi, mu)
        if hi - lo <= mu_tol:
            break
        mu = 0.5 * (lo + hi)
        if len(trace) == 1 and mu_first is not None and lo < mu_first < hi:
            mu = mu_first
    return best[0], best[1] + n_target, trace
