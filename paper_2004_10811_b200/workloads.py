"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds NO arithmetic of the submatrix method (no index building, no
assembly, no sign function, no extraction).  It only fabricates inputs with the
shapes of the paper's liquid-water workloads (32-H2O cell
replicated, SZV-/DZVP-MOLOPT-SR-GTH; BASELINE.json `configs`) and packs them in
the block-sparse layout the C-ABI takes (include/submatrix.h):

* one block row/column per atom (DBCSR-style), atom order O,H,H;
* block-CSC pattern `colptr[nb+1]` (int64), `rowidx[nnzb]` (int32, ascending in
  each column) -- the paper's "COO sorted by columns and rows" (L180), so the
  position of a block in `rowidx` is its id;
* `values`: blocks in that order, each dense column-major `bs[r] x bs[c]`;
* `grp_ptr/grp_cols`: generating block-column groups, one per molecule (L199).

The recipe is BASELINE.json's, with the readings of
SURVEY.md section 8(d).  Random numbers come from numpy's counter-based Philox.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

RHO_MOLECULES_PER_A3 = 0.0334273  # 1 g/cm^3 of H2O
R_OH = 0.9572
ANGLE_HOH = math.radians(104.52)
BASIS = {
    "SZV": {"O": 4, "H": 1},
    "DZVP": {"O": 13, "H": 5},
}
N_OCC_PER_MOLECULE = 4  # the O atom's first four functions carry N(-1, 0.1)


@dataclasses.dataclass
class BlockSparseSym:
    """A structurally and numerically symmetric block-sparse matrix + groups."""

    nb: int
    blk_size: np.ndarray  # int32 [nb]
    colptr: np.ndarray  # int64 [nb+1]
    rowidx: np.ndarray  # int32 [nnzb]
    values: np.ndarray  # float64 [nnz]
    grp_ptr: np.ndarray  # int32 [ngroups+1]
    grp_cols: np.ndarray  # int32 [nb]
    n_occ: int = 0  # number of N(-1,.) on-site functions (target electron count)
    meta: dict = dataclasses.field(default_factory=dict)

    @property
    def ngroups(self) -> int:
        return len(self.grp_ptr) - 1

    @property
    def nnzb(self) -> int:
        return len(self.rowidx)

    @property
    def n_basis(self) -> int:
        return int(self.blk_size.sum())

    def blk_off(self) -> np.ndarray:
        o = np.zeros(self.nb + 1, dtype=np.int64)
        np.cumsum(self.blk_size, out=o[1:])
        return o

    def val_off(self) -> np.ndarray:
        """Exclusive prefix sum of bs[r]*bs[c] over blocks in storage order."""
        cols = np.repeat(np.arange(self.nb), np.diff(self.colptr))
        sz = self.blk_size[self.rowidx].astype(np.int64) * self.blk_size[cols]
        o = np.zeros(self.nnzb + 1, dtype=np.int64)
        np.cumsum(sz, out=o[1:])
        return o

    def block_cols(self) -> np.ndarray:
        return np.repeat(np.arange(self.nb, dtype=np.int32), np.diff(self.colptr))

    def to_dense(self, values: np.ndarray | None = None) -> np.ndarray:
        """Dense copy (small cases only; test helper, pure data movement)."""
        v = self.values if values is None else values
        off = self.blk_off()
        voff = self.val_off()
        n = int(off[-1])
        out = np.zeros((n, n))
        cols = self.block_cols()
        for b in range(self.nnzb):
            r, c = int(self.rowidx[b]), int(cols[b])
            br, bc = int(self.blk_size[r]), int(self.blk_size[c])
            out[off[r]:off[r] + br, off[c]:off[c] + bc] = (
                v[voff[b]:voff[b + 1]].reshape(bc, br).T)
        return out


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed, stream]))


def water_positions(n_mol: int, seed: int):
    """Jittered simple-cubic lattice of rigid waters at 1 g/cm^3 in a periodic cube.

    Returns (pos[3*n_mol,3] in atom order O,H,H per molecule, box length L)."""
    L = (n_mol / RHO_MOLECULES_PER_A3) ** (1.0 / 3.0)
    g = int(math.ceil(n_mol ** (1.0 / 3.0) - 1e-9))
    rng = _rng(seed, 0)
    sites = np.sort(rng.permutation(g ** 3)[:n_mol])  # ascending site order: locality (L188)
    ix, iy, iz = sites // (g * g), (sites // g) % g, sites % g
    a = L / g
    centre = (np.stack([ix, iy, iz], axis=1) + 0.5) * a
    centre += rng.uniform(-0.15, 0.15, size=(n_mol, 3)) * a
    # random rigid rotation per molecule (QR of a Gaussian, det fixed to +1)
    m = rng.standard_normal((n_mol, 3, 3))
    q, r = np.linalg.qr(m)
    q = q * np.sign(np.einsum("nii->ni", r))[:, None, :]
    q[:, :, 2] *= np.linalg.det(q)[:, None]
    h1 = np.array([R_OH, 0.0, 0.0])
    h2 = np.array([R_OH * math.cos(ANGLE_HOH), R_OH * math.sin(ANGLE_HOH), 0.0])
    pos = np.empty((n_mol, 3, 3))
    pos[:, 0] = centre
    pos[:, 1] = centre + q @ h1
    pos[:, 2] = centre + q @ h2
    pos = np.mod(pos.reshape(-1, 3), L)
    return pos, L


def _pairs_within(pos: np.ndarray, L: float, cutoff: float):
    """All atom pairs i<j with minimum-image distance < cutoff; each pair once."""
    n = len(pos)
    if n <= 6000 or cutoff >= 0.5 * L:
        out_i, out_j, out_d = [], [], []
        step = max(1, 4_000_000 // n)
        for s in range(0, n, step):
            d = pos[s:s + step, None, :] - pos[None, :, :]
            d -= L * np.round(d / L)
            dist = np.sqrt((d * d).sum(-1))
            ii, jj = np.nonzero(dist < cutoff)
            ii += s
            keep = ii < jj
            out_i.append(ii[keep]); out_j.append(jj[keep]); out_d.append(dist[ii[keep] - s, jj[keep]])
        i, j, d = np.concatenate(out_i), np.concatenate(out_j), np.concatenate(out_d)
    else:
        from scipy.spatial import cKDTree
        tree = cKDTree(pos, boxsize=L)
        pr = tree.query_pairs(cutoff, output_type="ndarray")
        i, j = pr.min(1), pr.max(1)
        dv = pos[i] - pos[j]
        dv -= L * np.round(dv / L)
        d = np.sqrt((dv * dv).sum(-1))
        keep = d < cutoff
        i, j, d = i[keep], j[keep], d[keep]
    order = np.lexsort((j, i))
    return i[order].astype(np.int64), j[order].astype(np.int64), d[order]


def water_like(n_mol: int, basis: str = "SZV", cutoff: float = 6.0, seed: int = 1,
               group: str = "molecule") -> BlockSparseSym:
    """BASELINE.json configs 0, 2, 3, 4: water-like orthogonalised Kohn-Sham matrix.

    On-site diagonal N(-1,0.1) for O's first four functions, N(+1,0.1) for every other
    function; inter-atomic blocks 0.3*exp(-d^2/4)*N(0,1)*f, kept iff d < cutoff, with
    f = sqrt(b_r^SZV b_c^SZV / (b_r b_c)) (=1 for SZV)."""
    pos, L = water_positions(n_mol, seed)
    nb = 3 * n_mol
    bO, bH = BASIS[basis]["O"], BASIS[basis]["H"]
    bs = np.tile(np.array([bO, bH, bH], dtype=np.int32), n_mol)
    bs_szv = np.tile(np.array([4, 1, 1], dtype=np.int64), n_mol)
    pi, pj, pd = _pairs_within(pos, L, cutoff)

    # pattern: both orientations + diagonal, sorted by (column, row)
    rows = np.concatenate([pi, pj, np.arange(nb)])
    cols = np.concatenate([pj, pi, np.arange(nb)])
    npair = len(pi)
    # source tag: 0..npair-1 = block (i,j) of pair, npair..2npair-1 = block (j,i), then diagonal
    tag = np.arange(len(rows))
    order = np.lexsort((rows, cols))
    rows, cols, tag = rows[order], cols[order], tag[order]
    colptr = np.zeros(nb + 1, dtype=np.int64)
    np.cumsum(np.bincount(cols, minlength=nb), out=colptr[1:])
    sz = bs[rows].astype(np.int64) * bs[cols]
    voff = np.zeros(len(rows) + 1, dtype=np.int64)
    np.cumsum(sz, out=voff[1:])
    values = np.zeros(int(voff[-1]))
    where = np.empty(len(rows), dtype=np.int64)  # tag -> block id
    where[tag] = np.arange(len(rows))

    # couplings: one flat normal stream, pair by pair in (i,j) order, row-major (bs_i x bs_j)
    rng = _rng(seed, 1)
    psz = bs[pi].astype(np.int64) * bs[pj]
    poff = np.zeros(npair + 1, dtype=np.int64)
    np.cumsum(psz, out=poff[1:])
    z = rng.standard_normal(int(poff[-1]))
    f = np.sqrt(bs_szv[pi] * bs_szv[pj] / (bs[pi].astype(np.float64) * bs[pj]))
    amp = 0.3 * np.exp(-pd * pd / 4.0) * f
    z *= np.repeat(amp, psz)
    for bi in np.unique(bs):
        for bj in np.unique(bs):
            sel = np.nonzero((bs[pi] == bi) & (bs[pj] == bj))[0]
            if len(sel) == 0:
                continue
            m = int(bi) * int(bj)
            seg = z[poff[sel][:, None] + np.arange(m)[None, :]]  # (npairs, bi*bj) row-major (i,j)
            # block (j,i) in column i is column-major (bj x bi) == row-major (bi x bj)
            dst_ji = voff[where[npair + sel]][:, None] + np.arange(m)[None, :]
            values[dst_ji] = seg
            # block (i,j) in column j is column-major (bi x bj) == transpose of the above
            dst_ij = voff[where[sel]][:, None] + np.arange(m)[None, :]
            values[dst_ij] = seg.reshape(-1, int(bi), int(bj)).transpose(0, 2, 1).reshape(-1, m)

    # on-site: diagonal only
    rng2 = _rng(seed, 2)
    n_basis = int(bs.sum())
    mean = np.ones(n_basis)
    boff = np.zeros(nb + 1, dtype=np.int64)
    np.cumsum(bs, out=boff[1:])
    o_start = boff[0::3][:n_mol]
    occ_idx = (o_start[:, None] + np.arange(N_OCC_PER_MOLECULE)[None, :]).ravel()
    mean[occ_idx] = -1.0
    onsite = mean + 0.1 * rng2.standard_normal(n_basis)
    dblk = where[2 * npair + np.arange(nb)]
    for b in np.unique(bs):
        sel = np.nonzero(bs == b)[0]
        k = np.arange(int(b))
        dst = voff[dblk[sel]][:, None] + (k * (int(b) + 1))[None, :]
        values[dst] = onsite[boff[sel][:, None] + k[None, :]]

    if group == "molecule":
        grp_ptr = (3 * np.arange(n_mol + 1)).astype(np.int32)
    elif group == "atom":
        grp_ptr = np.arange(nb + 1, dtype=np.int32)
    else:
        raise ValueError(group)
    grp_cols = np.arange(nb, dtype=np.int32)
    return BlockSparseSym(nb, bs, colptr, rows.astype(np.int32), values, grp_ptr, grp_cols,
                          n_occ=N_OCC_PER_MOLECULE * n_mol,
                          meta={"kind": "water_like", "n_mol": n_mol, "basis": basis, "cutoff": cutoff,
                                "seed": seed, "L": L, "positions": pos})


def haar_spectrum_batch(batch: int, n: int, seed: int = 1):
    """BASELINE.json config 1: A = Q diag(lam) Q^T, Haar Q, lam uniform in
    [-1,-0.05] U [0.05,1], half negative.  Returns (A[batch,n,n], Q, lam)."""
    rng = _rng(seed, 3)
    g = rng.standard_normal((batch, n, n))
    q, r = np.linalg.qr(g)
    q = q * np.sign(np.einsum("bii->bi", r))[:, None, :]
    mag = rng.uniform(0.05, 1.0, size=(batch, n))
    sgn = np.ones(n)
    sgn[: n // 2] = -1.0
    lam = mag * sgn[None, :]
    a = np.einsum("bik,bk,bjk->bij", q, lam, q)
    a = 0.5 * (a + a.transpose(0, 2, 1))
    return a, q, lam


def dense_batch_as_blocks(a: np.ndarray) -> BlockSparseSym:
    """Wrap a batch of dense symmetric matrices as a block-diagonal BlockSparseSym:
    block column i holds only block (i,i); one group per column, so submatrix i == a[i]."""
    batch, n, _ = a.shape
    bs = np.full(batch, n, dtype=np.int32)
    colptr = np.arange(batch + 1, dtype=np.int64)
    rowidx = np.arange(batch, dtype=np.int32)
    values = np.ascontiguousarray(a.transpose(0, 2, 1)).reshape(-1).copy()
    return BlockSparseSym(batch, bs, colptr, rowidx, values,
                          np.arange(batch + 1, dtype=np.int32), np.arange(batch, dtype=np.int32),
                          n_occ=int(batch * (n // 2)), meta={"kind": "dense_batch", "n": n})


def random_block_pattern(nb: int, density: float, max_bs: int, seed: int,
                         ngroups: int | None = None, contiguous_groups: bool = False) -> BlockSparseSym:
    """Small random structurally-symmetric block matrix with ragged block sizes and a
    random partition of the block columns into groups (edge-case / brute-force tests)."""
    rng = _rng(seed, 4)
    bs = rng.integers(1, max_bs + 1, size=nb).astype(np.int32)
    m = rng.random((nb, nb)) < density
    m = np.triu(m, 1)
    m = m | m.T | np.eye(nb, dtype=bool)
    cols, rows = np.nonzero(m.T)  # sorted by column then row
    colptr = np.zeros(nb + 1, dtype=np.int64)
    np.cumsum(np.bincount(cols, minlength=nb), out=colptr[1:])
    off = np.zeros(nb + 1, dtype=np.int64)
    np.cumsum(bs, out=off[1:])
    n = int(off[-1])
    dense = rng.standard_normal((n, n)) * 0.2
    dense = 0.5 * (dense + dense.T)
    dense[np.arange(n), np.arange(n)] += np.where(rng.random(n) < 0.5, -1.0, 1.0)
    vals = []
    for r, c in zip(rows, cols):
        vals.append(dense[off[r]:off[r + 1], off[c]:off[c + 1]].T.reshape(-1))
    values = np.concatenate(vals)
    if ngroups is None:
        ngroups = max(1, nb // 2)
    ngroups = min(ngroups, nb)
    if contiguous_groups:
        perm = np.arange(nb)
    else:
        perm = rng.permutation(nb)
    cuts = np.sort(rng.choice(np.arange(1, nb), size=ngroups - 1, replace=False)) if ngroups > 1 else np.array([], dtype=np.int64)
    grp_ptr = np.concatenate([[0], cuts, [nb]]).astype(np.int32)
    return BlockSparseSym(nb, bs, colptr, rows.astype(np.int32), values, grp_ptr,
                          perm.astype(np.int32), n_occ=0, meta={"kind": "random", "seed": seed})


CONFIGS = {
    # BASELINE.json `configs`, zero-indexed
    0: dict(kind="water", n_mol=32, basis="SZV", cutoff=6.0),
    1: dict(kind="haar", batch=512, n=256),
    2: dict(kind="water", n_mol=1024, basis="SZV", cutoff=6.0),
    3: dict(kind="water", n_mol=4096, basis="DZVP", cutoff=5.0),
    4: dict(kind="water", n_mol=20736, basis="SZV", cutoff=6.0),
    # "3b": BASELINE's prose for config 3 says ~1500-3000-dimensional submatrices, which the
    # literal 5 A cutoff does not give; 8 A does (n ~ 1700-2050).  512 molecules keep the workspace at ~45 GB.
    5: dict(kind="water", n_mol=512, basis="DZVP", cutoff=8.0),
}


def make_config(idx: int, seed: int = 1) -> BlockSparseSym:
    c = CONFIGS[idx]
    if c["kind"] == "water":
        return water_like(c["n_mol"], c["basis"], c["cutoff"], seed)
    a, q, lam = haar_spectrum_batch(c["batch"], c["n"], seed)
    m = dense_batch_as_blocks(a)
    m.meta.update(Q=q, lam=lam)
    return m
