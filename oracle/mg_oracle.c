/*
 * mg_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, obviously-correct FP64 CPU loops for the block kernels of the toroidal semi-coarsening
 * multigrid solve path of arXiv 2506.16676.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code with the CUDA
 * library under paper_2506_16676_b200/csrc and is never used by the product path.
 *
 * Every function is the written-out definition of the operation; no blocking, fusion or reordering.
 * OpenMP is used only to split independent block rows over host cores (each row's arithmetic and its
 * summation order are unchanged by the thread count).
 *
 * Layout (same arrays the library takes): block-CSR, row_ptr int64[n+1], col_idx int32[nnzb],
 * vals double[nnzb*b*b] with row-major b x b blocks, vectors double[n*b] with scalar index I*b + c.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* y = A x  -- definition of the matrix-vector product; "a sparse matrix vector product, the kernel of
 * MG"; block size b = 36 in the paper.
 * y[I*b+r] = sum_{p in row I} sum_{c<b} vals[p][r][c] * x[col_idx[p]*b + c], blocks in stored order, c inner. */
void orc_bsr_spmv(int64_t n_brows, int b, const int64_t *row_ptr, const int32_t *col_idx, const double *vals,
                  const double *x, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t I = 0; I < n_brows; ++I) {
        for (int r = 0; r < b; ++r) {
            double acc = 0.0;
            for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p) {
                const double *blk = vals + (size_t)p * b * b + (size_t)r * b;
                const double *xj = x + (size_t)col_idx[p] * b;
                for (int c = 0; c < b; ++c) acc += blk[c] * xj[c];
            }
            y[(size_t)I * b + r] = acc;
        }
    }
}

/* PBJ setup: Dinv_I = (A_II)^-1, "PBJ smoothers in PETSc compute explicit, dense inverses of these
 * diagonal blocks".  Gauss-Jordan elimination with partial (row) pivoting on [D | I].
 * Returns 0 on success, 1 + I for the first block row whose diagonal block is missing or has a zero pivot. */
int64_t orc_pbj_invert(int64_t n_brows, int b, const int64_t *row_ptr, const int32_t *col_idx, const double *vals,
                       double *dinv)
{
    int64_t bad = 0;
#pragma omp parallel for schedule(static)
    for (int64_t I = 0; I < n_brows; ++I) {
        int64_t pd = -1;
        for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p)
            if ((int64_t)col_idx[p] == I) pd = p;
        double *M = (double *)malloc(sizeof(double) * (size_t)b * 2 * b); /* [D | I], row-major b x 2b */
        int fail = (pd < 0);
        if (!fail) {
            const double *D = vals + (size_t)pd * b * b;
            for (int r = 0; r < b; ++r)
                for (int c = 0; c < b; ++c) {
                    M[r * 2 * b + c] = D[r * b + c];
                    M[r * 2 * b + b + c] = (r == c) ? 1.0 : 0.0;
                }
            for (int k = 0; k < b && !fail; ++k) {
                int piv = k;
                double best = fabs(M[k * 2 * b + k]);
                for (int r = k + 1; r < b; ++r)
                    if (fabs(M[r * 2 * b + k]) > best) { best = fabs(M[r * 2 * b + k]); piv = r; }
                if (best == 0.0 || best != best) { fail = 1; break; }
                if (piv != k)
                    for (int c = 0; c < 2 * b; ++c) {
                        double t = M[k * 2 * b + c]; M[k * 2 * b + c] = M[piv * 2 * b + c]; M[piv * 2 * b + c] = t;
                    }
                double inv = 1.0 / M[k * 2 * b + k];
                for (int c = 0; c < 2 * b; ++c) M[k * 2 * b + c] *= inv;
                for (int r = 0; r < b; ++r) {
                    if (r == k) continue;
                    double f = M[r * 2 * b + k];
                    if (f != 0.0)
                        for (int c = 0; c < 2 * b; ++c) M[r * 2 * b + c] -= f * M[k * 2 * b + c];
                }
            }
        }
        if (fail) {
#pragma omp critical
            { if (bad == 0 || I + 1 < bad) bad = I + 1; }
        } else {
            for (int r = 0; r < b; ++r)
                for (int c = 0; c < b; ++c) dinv[(size_t)I * b * b + r * b + c] = M[r * 2 * b + b + c];
        }
        free(M);
    }
    return bad;
}

/* PBJ apply: z_I = Dinv_I r_I, "applied effectively on GPUs with dense matrix-vector products". */
void orc_pbj_apply(int64_t n_brows, int b, const double *dinv, const double *r, double *z)
{
#pragma omp parallel for schedule(static)
    for (int64_t I = 0; I < n_brows; ++I)
        for (int rr = 0; rr < b; ++rr) {
            double acc = 0.0;
            const double *row = dinv + (size_t)I * b * b + (size_t)rr * b;
            for (int c = 0; c < b; ++c) acc += row[c] * r[(size_t)I * b + c];
            z[(size_t)I * b + rr] = acc;
        }
}

/* Galerkin coarse operator values, A_c = P^T A P with P = P_phi (x) I:
 *   A_c[(i,K),(j,M)] = sum_{k,m} P_phi[k,K] * P_phi[m,M] * A[(i,k),(j,m)]
 * written as the scatter of every fine block to every coarse pair with a non-zero weight.  The coarse
 * pattern (crow_ptr/ccol_idx, columns ascending) is built by the caller; pphi is the dense n_f x n_c
 * interpolation matrix in row-major order.  cvals must be zero on entry.  Serial on purpose: the scatter
 * has write conflicts between fine rows; the loop order is the summation order.
 * Returns 0, or 1 + p for the first fine block whose coarse target is missing from the pattern. */
int64_t orc_galerkin_numeric(int64_t n_pol, int n_f, int n_c, int b, const double *pphi, const int64_t *row_ptr,
                             const int32_t *col_idx, const double *vals, const int64_t *crow_ptr,
                             const int32_t *ccol_idx, double *cvals)
{
    const size_t bb = (size_t)b * b;
    for (int64_t I = 0; I < n_pol * n_f; ++I) {
        const int64_t k = I / n_pol, i = I % n_pol;
        for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p) {
            const int64_t J = col_idx[p], m = J / n_pol, j = J % n_pol;
            for (int K = 0; K < n_c; ++K) {
                const double wk = pphi[k * n_c + K];
                if (wk == 0.0) continue;
                for (int M = 0; M < n_c; ++M) {
                    const double wm = pphi[m * n_c + M];
                    if (wm == 0.0) continue;
                    const int64_t Ic = (int64_t)K * n_pol + i, Jc = (int64_t)M * n_pol + j;
                    int64_t q = -1;
                    for (int64_t t = crow_ptr[Ic]; t < crow_ptr[Ic + 1]; ++t)
                        if ((int64_t)ccol_idx[t] == Jc) { q = t; break; }
                    if (q < 0) return 1 + p;
                    const double w = wk * wm;
                    double *dst = cvals + (size_t)q * bb;
                    const double *src = vals + (size_t)p * bb;
                    for (size_t e = 0; e < bb; ++e) dst[e] += w * src[e];
                }
            }
        }
    }
    return 0;
}
