/*
 * CPU ORACLE for the submatrix method -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct C (fp64) restatement of what the hot path computes,
 * written from /root/reference/PAPER.md only.  It shares no code, header, table or
 * helper with the CUDA path (paper_2004_10811_b200/csrc) and neither imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.
 *
 * What it follows, step by step (PAPER.md line numbers; "A<n>" = reading in DESIGN.md):
 *   index     L125  "principal submatrix a_i is assembled by removing all rows and columns j
 *                    where A_{j,i} = 0", applied per block column (L170, L196) and per group of
 *                    block columns (L199).  Row order inside a submatrix: ascending (A2).
 *   assemble  L125 / L187  copy the stored blocks of S_i x S_i, zero elsewhere (A4).
 *   shift     Eq.(16) L243 / Eq.(18): a_i - mu I.
 *   sign      Eq.(17): A = Q Lambda Q^T, Lambda' = signum(Lambda), sign(A) = Q Lambda' Q^T,
 *             with signum(0) = 0 (Eq.(12)).  Eigendecomposition by cyclic Jacobi rotations
 *             (the paper calls LAPACK dsyevd, L246; Jacobi is the textbook definition-level method).
 *   extract   L127 "values from the k-th column of f(a_i) are used to assemble the i-th column ...
 *             retaining the sparsity pattern", with D = 1/2 (I - sign(.)) (Eq.(16) inner factor).
 *   n_elec    Algorithm 1: n_elec += 1/2 - 1/2 sum_l Q_{k,l}^2 lambda'_l for the generating
 *             columns k; we return lambda_l and w_l = sum_{k in gen} Q_{k,l}^2 (L270) so that the
 *             mu loop of Algorithm 1 needs no new decomposition.
 *   energy    Eq.(10): Tr(D K).
 *   fermi     L255 "systems at finite temperature by replacing the signum function in Eq. (17) by the
 *             Fermi function": occupation f(lambda) = 1 / (1 + exp((lambda - mu) / kT)) in place of
 *             1/2 (1 - signum(lambda - mu)), i.e. signum(x) -> tanh(x / (2 kT)) (reading A18);
 *             D = Q f(Lambda) Q^T.  kT = 0 is the signum case.
 *
 * No blocking, fusion or reordering beyond the statements above.  OpenMP is used only ACROSS
 * submatrices (the paper does the same, L229).
 *
 * Parity pins: tests/test_oracle_pins.py.  Unpinned: none of the
 * functions here; the final mu of a bisection is pinned only up to its plateau (A12).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int cmp_i32(const void *a, const void *b) {
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* S_i = sorted set of block rows r with a stored block (r,c) for some c in G_i (L125, L199).
 * Algorithm: concatenate the row lists, qsort, drop duplicates. Returns |S_i|; out may be NULL. */
static int64_t union_rows(const int64_t *colptr, const int32_t *rowidx, const int32_t *gcols, int ng,
                          int32_t *out) {
    int64_t tot = 0;
    for (int g = 0; g < ng; ++g) tot += colptr[gcols[g] + 1] - colptr[gcols[g]];
    int32_t *tmp = (int32_t *)malloc((size_t)(tot > 0 ? tot : 1) * sizeof(int32_t));
    int64_t k = 0;
    for (int g = 0; g < ng; ++g)
        for (int64_t p = colptr[gcols[g]]; p < colptr[gcols[g] + 1]; ++p) tmp[k++] = rowidx[p];
    qsort(tmp, (size_t)tot, sizeof(int32_t), cmp_i32);
    int64_t m = 0;
    for (int64_t p = 0; p < tot; ++p)
        if (p == 0 || tmp[p] != tmp[p - 1]) {
            if (out) out[m] = tmp[p];
            ++m;
        }
    free(tmp);
    return m;
}

/* Step "index", pass 1: sub_ptr[ngroups+1] (exclusive prefix sum of |S_i|). Returns sum |S_i|. */
int64_t orc_index_count(int32_t nb, const int64_t *colptr, const int32_t *rowidx, int32_t ngroups,
                        const int32_t *grp_ptr, const int32_t *grp_cols, int64_t *sub_ptr) {
    (void)nb;
    sub_ptr[0] = 0;
    for (int i = 0; i < ngroups; ++i)
        sub_ptr[i + 1] = sub_ptr[i] + union_rows(colptr, rowidx, grp_cols + grp_ptr[i],
                                                 grp_ptr[i + 1] - grp_ptr[i], NULL);
    return sub_ptr[ngroups];
}

/* Step "index", pass 2: sub_blocks[sum|S_i|] (ascending per group), sub_off[sum|S_i|] (element
 * offset of each member inside a_i), sub_dim[ngroups] (n_i), gen_pos[len(grp_cols)] (position of
 * every generating column's block inside S_i; -1 if its diagonal block is not stored, A3). */
void orc_index_fill(int32_t nb, const int32_t *blk_size, const int64_t *colptr, const int32_t *rowidx,
                    int32_t ngroups, const int32_t *grp_ptr, const int32_t *grp_cols,
                    const int64_t *sub_ptr, int32_t *sub_blocks, int32_t *sub_off, int32_t *sub_dim,
                    int32_t *gen_pos) {
    (void)nb;
    for (int i = 0; i < ngroups; ++i) {
        int32_t *S = sub_blocks + sub_ptr[i];
        int64_t m = union_rows(colptr, rowidx, grp_cols + grp_ptr[i], grp_ptr[i + 1] - grp_ptr[i], S);
        int32_t off = 0;
        for (int64_t t = 0; t < m; ++t) {
            sub_off[sub_ptr[i] + t] = off;
            off += blk_size[S[t]];
        }
        sub_dim[i] = off;
        for (int g = grp_ptr[i]; g < grp_ptr[i + 1]; ++g) {
            gen_pos[g] = -1;
            for (int64_t t = 0; t < m; ++t)
                if (S[t] == grp_cols[g]) gen_pos[g] = (int32_t)t;
        }
    }
}

/* Step "assemble": dense column-major n x n principal submatrix over the block set S (L125).
 * val_off[b] = element offset of block b; block (r,c) is column-major bs[r] x bs[c]. */
void orc_assemble(const int32_t *blk_size, const int64_t *colptr, const int32_t *rowidx,
                  const int64_t *val_off, const double *vals, int64_t m, const int32_t *S,
                  const int32_t *S_off, int32_t n, double *a) {
    memset(a, 0, (size_t)n * n * sizeof(double));
    for (int64_t tc = 0; tc < m; ++tc) {
        int32_t c = S[tc];
        for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
            int32_t r = rowidx[p];
            int64_t tr = -1; /* linear search: is r a member of S? */
            for (int64_t t = 0; t < m; ++t)
                if (S[t] == r) { tr = t; break; }
            if (tr < 0) continue;
            int br = blk_size[r], bc = blk_size[c];
            for (int q = 0; q < bc; ++q)
                for (int e = 0; e < br; ++e)
                    a[(size_t)(S_off[tc] + q) * n + S_off[tr] + e] = vals[val_off[p] + (int64_t)q * br + e];
        }
    }
}

/* Cyclic Jacobi eigendecomposition of a symmetric n x n matrix (Eq.(17) first line).
 * In:  A (n x n, symmetric, overwritten).  Out: lam[n]; Qt[n x n] row l = eigenvector l
 * (i.e. Q_{k,l} = Qt[l*n + k]).  Returns the number of sweeps used.
 * Rotation (Golub & Van Loan, symmetric Schur 2x2): tau = (a_qq - a_pp) / (2 a_pq),
 * t = sign(tau) / (|tau| + sqrt(1 + tau^2)), c = 1/sqrt(1+t^2), s = t c. */
int orc_jacobi_eig(int32_t n, double *A, double *Qt, double *lam) {
    for (size_t i = 0; i < (size_t)n * n; ++i) Qt[i] = 0.0;
    for (int i = 0; i < n; ++i) Qt[(size_t)i * n + i] = 1.0;
    double fro2 = 0.0;
    for (size_t i = 0; i < (size_t)n * n; ++i) fro2 += A[i] * A[i];
    const double fro = sqrt(fro2);
    int sweep = 0;
    for (; sweep < 60; ++sweep) {
        double off2 = 0.0;
        for (int p = 0; p < n; ++p)
            for (int q = p + 1; q < n; ++q) off2 += 2.0 * A[(size_t)p * n + q] * A[(size_t)p * n + q];
        if (sqrt(off2) <= 1e-15 * fro) break;
        int rotated = 0;
        for (int p = 0; p < n - 1; ++p) {
            for (int q = p + 1; q < n; ++q) {
                double apq = A[(size_t)p * n + q];
                if (fabs(apq) <= 1e-300) continue;
                double app = A[(size_t)p * n + p], aqq = A[(size_t)q * n + q];
                /* rotation would not change anything representable */
                if (fabs(apq) < 1e-20 * (fabs(app) + fabs(aqq)) ) { A[(size_t)p*n+q] = 0.0; A[(size_t)q*n+p] = 0.0; continue; }
                double tau = (aqq - app) / (2.0 * apq);
                double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                rotated = 1;
                /* A <- J^T A J, J = [[c, s], [-s, c]] in the (p,q) plane */
                double *rp = A + (size_t)p * n, *rq = A + (size_t)q * n;
                for (int k = 0; k < n; ++k) { /* rows p, q */
                    double x = rp[k], y = rq[k];
                    rp[k] = c * x - s * y;
                    rq[k] = s * x + c * y;
                }
                for (int k = 0; k < n; ++k) { /* columns p, q */
                    double x = A[(size_t)k * n + p], y = A[(size_t)k * n + q];
                    A[(size_t)k * n + p] = c * x - s * y;
                    A[(size_t)k * n + q] = s * x + c * y;
                }
                A[(size_t)p * n + q] = 0.0;
                A[(size_t)q * n + p] = 0.0;
                /* Q <- Q J : columns p,q of Q = rows p,q of Qt */
                double *qp = Qt + (size_t)p * n, *qq = Qt + (size_t)q * n;
                for (int k = 0; k < n; ++k) {
                    double x = qp[k], y = qq[k];
                    qp[k] = c * x - s * y;
                    qq[k] = s * x + c * y;
                }
            }
        }
        if (!rotated) break;
    }
    for (int i = 0; i < n; ++i) lam[i] = A[(size_t)i * n + i];
    return sweep;
}

static double signum(double x) { return (x > 0.0) - (x < 0.0); } /* Eq.(9), Eq.(12): signum(0)=0 */

/* sign(A) = Q diag(signum(lam_l - shift)) Q^T (Eq.(17)); column-major n x n output (symmetric). */
void orc_sign_from_eig(int32_t n, const double *Qt, const double *lam, double shift, double *S) {
    memset(S, 0, (size_t)n * n * sizeof(double));
    for (int l = 0; l < n; ++l) {
        double sg = signum(lam[l] - shift);
        if (sg == 0.0) continue;
        const double *v = Qt + (size_t)l * n;
        for (int j = 0; j < n; ++j) {
            double f = sg * v[j];
            for (int i = 0; i < n; ++i) S[(size_t)j * n + i] += v[i] * f;
        }
    }
}

/* Dense sign of one symmetric matrix (convenience for the pins): S = sign(A - mu I). */
int orc_dense_sign(int32_t n, const double *A, double mu, double *S, double *lam_out) {
    double *W = (double *)malloc((size_t)n * n * sizeof(double));
    double *Qt = (double *)malloc((size_t)n * n * sizeof(double));
    double *lam = (double *)malloc((size_t)n * sizeof(double));
    memcpy(W, A, (size_t)n * n * sizeof(double));
    for (int i = 0; i < n; ++i) W[(size_t)i * n + i] -= mu; /* shift (Eq.(16)) */
    int sw = orc_jacobi_eig(n, W, Qt, lam);
    orc_sign_from_eig(n, Qt, lam, 0.0, S);
    if (lam_out) memcpy(lam_out, lam, (size_t)n * sizeof(double));
    free(W); free(Qt); free(lam);
    return sw;
}

/* The submatrix method for a list of groups (all steps, L123-127 + Eq.(16)):
 * for every listed group i: assemble a_i, shift by mu, sign by Jacobi, and write
 * D[r,c] = 1/2 (delta_rc I - sign(a_i)[loc r, loc c]) for every stored block (r,c) of every
 * generating column c of the group into vals_out (same layout as vals).  Blocks of groups not
 * listed are left untouched.  If lam_out/w_out are non-NULL they receive, at offset
 * lw_ptr[j] for the j-th listed group, the eigenvalues of a_i (UNshifted by mu... of a_i itself)
 * and the weights w_l = sum_{k in generating columns} Q_{k,l}^2 (Algorithm 1).
 * If do_extract == 0 only lam/w are produced. */
void orc_submatrix_groups(const int32_t *blk_size, const int64_t *colptr, const int32_t *rowidx,
                          const int64_t *val_off, const double *vals, const int32_t *grp_ptr,
                          const int32_t *grp_cols, const int64_t *sub_ptr, const int32_t *sub_blocks,
                          const int32_t *sub_off, const int32_t *sub_dim, const int32_t *gen_pos,
                          int32_t nlist, const int32_t *list, double mu, int32_t do_extract,
                          double *vals_out, const int64_t *lw_ptr, double *lam_out, double *w_out,
                          int32_t nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < nlist; ++j) {
        int i = list[j];
        int32_t n = sub_dim[i];
        int64_t m = sub_ptr[i + 1] - sub_ptr[i];
        const int32_t *S = sub_blocks + sub_ptr[i];
        const int32_t *So = sub_off + sub_ptr[i];
        double *a = (double *)malloc((size_t)n * n * sizeof(double));
        double *Qt = (double *)malloc((size_t)n * n * sizeof(double));
        double *sg = (double *)malloc((size_t)n * n * sizeof(double));
        double *lam = (double *)malloc((size_t)n * sizeof(double));
        orc_assemble(blk_size, colptr, rowidx, val_off, vals, m, S, So, n, a);
        /* eigendecomposition of a_i itself; the shift is applied to Lambda (Algorithm 1:
         * lambda' = signum(lambda - mu); identical to decomposing a_i - mu I, Eq.(16)) */
        orc_jacobi_eig(n, a, Qt, lam);
        if (lam_out) {
            for (int l = 0; l < n; ++l) {
                double w = 0.0;
                for (int g = grp_ptr[i]; g < grp_ptr[i + 1]; ++g) {
                    int t = gen_pos[g];
                    for (int e = 0; e < blk_size[grp_cols[g]]; ++e) {
                        double qkl = Qt[(size_t)l * n + So[t] + e];
                        w += qkl * qkl;
                    }
                }
                lam_out[lw_ptr[j] + l] = lam[l];
                w_out[lw_ptr[j] + l] = w;
            }
        }
        if (do_extract) {
            orc_sign_from_eig(n, Qt, lam, mu, sg);
            for (int g = grp_ptr[i]; g < grp_ptr[i + 1]; ++g) {
                int32_t c = grp_cols[g];
                int tc = gen_pos[g];
                int bc = blk_size[c];
                for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
                    int32_t r = rowidx[p];
                    int64_t tr = -1;
                    for (int64_t t = 0; t < m; ++t)
                        if (S[t] == r) { tr = t; break; }
                    int br = blk_size[r];
                    for (int q = 0; q < bc; ++q)
                        for (int e = 0; e < br; ++e) {
                            double delta = (r == c && q == e) ? 1.0 : 0.0;
                            vals_out[val_off[p] + (int64_t)q * br + e] =
                                0.5 * (delta - sg[(size_t)(So[tc] + q) * n + So[tr] + e]);
                        }
                }
            }
        }
        free(a); free(Qt); free(sg); free(lam);
    }
}

/* Occupation of one eigenvalue (L255, reading A18): Fermi function for kT > 0, else the zero-temperature
 * limit 1/2 (1 - signum(lambda - mu)) of Eq.(16)/(17) (1/2 exactly at lambda == mu, Eq.(12)). */
double orc_occupation(double lam, double mu, double kT) {
    if (kT > 0.0) return 1.0 / (1.0 + exp((lam - mu) / kT));
    return 0.5 * (1.0 - signum(lam - mu));
}

/* D = Q diag(f_l) Q^T, f_l = orc_occupation(lam_l, mu, kT); column-major n x n output (symmetric). */
void orc_occ_from_eig(int32_t n, const double *Qt, const double *lam, double mu, double kT, double *D) {
    memset(D, 0, (size_t)n * n * sizeof(double));
    for (int l = 0; l < n; ++l) {
        double f = orc_occupation(lam[l], mu, kT);
        if (f == 0.0) continue;
        const double *v = Qt + (size_t)l * n;
        for (int j = 0; j < n; ++j) {
            double fj = f * v[j];
            for (int i = 0; i < n; ++i) D[(size_t)j * n + i] += v[i] * fj;
        }
    }
}

/* The submatrix method at finite temperature (L255): as orc_submatrix_groups, with
 * D[r,c] = (Q f(Lambda) Q^T)[loc r, loc c] for the generating columns of every listed group. */
void orc_submatrix_groups_fermi(const int32_t *blk_size, const int64_t *colptr, const int32_t *rowidx,
                                const int64_t *val_off, const double *vals, const int32_t *grp_ptr,
                                const int32_t *grp_cols, const int64_t *sub_ptr, const int32_t *sub_blocks,
                                const int32_t *sub_off, const int32_t *sub_dim, const int32_t *gen_pos,
                                int32_t nlist, const int32_t *list, double mu, double kT, double *vals_out,
                                int32_t nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < nlist; ++j) {
        int i = list[j];
        int32_t n = sub_dim[i];
        int64_t m = sub_ptr[i + 1] - sub_ptr[i];
        const int32_t *S = sub_blocks + sub_ptr[i];
        const int32_t *So = sub_off + sub_ptr[i];
        double *a = (double *)malloc((size_t)n * n * sizeof(double));
        double *Qt = (double *)malloc((size_t)n * n * sizeof(double));
        double *D = (double *)malloc((size_t)n * n * sizeof(double));
        double *lam = (double *)malloc((size_t)n * sizeof(double));
        orc_assemble(blk_size, colptr, rowidx, val_off, vals, m, S, So, n, a);
        orc_jacobi_eig(n, a, Qt, lam);
        orc_occ_from_eig(n, Qt, lam, mu, kT, D);
        for (int g = grp_ptr[i]; g < grp_ptr[i + 1]; ++g) {
            int32_t c = grp_cols[g];
            int tc = gen_pos[g];
            int bc = blk_size[c];
            for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
                int32_t r = rowidx[p];
                int64_t tr = -1;
                for (int64_t t = 0; t < m; ++t)
                    if (S[t] == r) { tr = t; break; }
                int br = blk_size[r];
                for (int q = 0; q < bc; ++q)
                    for (int e = 0; e < br; ++e)
                        vals_out[val_off[p] + (int64_t)q * br + e] = D[(size_t)(So[tc] + q) * n + So[tr] + e];
            }
        }
        free(a); free(Qt); free(D); free(lam);
    }
}

/* Eq.(10) / Eq.(18): tr(D) over diagonal blocks and tr(D K) = sum over stored elements D o K
 * (valid because K is symmetric and D, K share the pattern).  Restricted to the block columns
 * listed in cols (ncols = -1: all nb columns). */
void orc_traces(int32_t nb, const int32_t *blk_size, const int64_t *colptr, const int32_t *rowidx,
                const int64_t *val_off, const double *D, const double *K, int32_t ncols,
                const int32_t *cols, double *tr_d, double *tr_dk) {
    double td = 0.0, tdk = 0.0;
    int nc = ncols < 0 ? nb : ncols;
    for (int ic = 0; ic < nc; ++ic) {
        int c = ncols < 0 ? ic : cols[ic];
        for (int64_t p = colptr[c]; p < colptr[c + 1]; ++p) {
            int r = rowidx[p];
            int64_t sz = (int64_t)blk_size[r] * blk_size[c];
            for (int64_t e = 0; e < sz; ++e) tdk += D[val_off[p] + e] * K[val_off[p] + e];
            if (r == c)
                for (int e = 0; e < blk_size[c]; ++e) td += D[val_off[p] + (int64_t)e * blk_size[c] + e];
        }
    }
    *tr_d = td;
    *tr_dk = tdk;
}
