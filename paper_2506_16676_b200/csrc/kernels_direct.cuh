// kernels_direct.cuh -- direct solve of the coarsest level (the paper solves its coarsest grid with
// an LU factorisation, and applies block solvers as "explicit inverses and BLAS2").
//
// The block rows of the coarsest level are ordered by the level sets of a breadth-first search of its block graph: every
// block then couples only rows of the same or of adjacent level sets, i.e. the matrix is BLOCK TRIDIAGONAL with dense
// blocks D_k (n_k x n_k), L_k (n_k x n_{k-1}), U_k (n_k x n_{k+1}).  Setup (off the solve path) forms the inverses of the
// Schur complements explicitly,  S_0 = D_0,  M_k = L_k S_{k-1}^-1,  S_k = D_k - M_k U_{k-1},  and the solve is dense
// mat-vec streaming (bandwidth bound, 3 n_k^2 doubles per level set):
//      forward :  z_0 = b_0,             z_k = b_k - M_k z_{k-1}
//      backward:  x_q = S_q^-1 z_q,      x_k = S_k^-1 (z_k - U_k x_{k+1})
// All matrices are row-major FP64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

struct DirectTables {       // device arrays describing the level-set ordering
    const int32_t *inv;     // [n_brows] new position of block row I
    const int32_t *lev;     // [n_brows] level set of NEW position p
    const int32_t *off;     // [nlev + 1] first new position of every level set
    double *const *D;       // [nlev] dense blocks
    double *const *Lm;      // [nlev] (Lm[0] unused)
    double *const *U;       // [nlev] (U[nlev-1] unused)
};

// One CTA per stored block: scatter it into the dense block of its (level set of row, level set of column).
__global__ void __launch_bounds__(128) direct_assemble_kernel(const int64_t *__restrict__ row_of_block,
                                                              const int32_t *__restrict__ col_idx,
                                                              const double *__restrict__ vals, const int b, const DirectTables t,
                                                              int *__restrict__ bad) {
    const int64_t p = blockIdx.x;
    const int pi = t.inv[row_of_block[p]], pj = t.inv[col_idx[p]];
    const int li = t.lev[pi], lj = t.lev[pj];
    double *dst;
    if (lj == li) dst = t.D[li];
    else if (lj == li - 1) dst = t.Lm[li];
    else if (lj == li + 1) dst = t.U[li];
    else {
        if (threadIdx.x == 0) atomicExch(bad, 1);
        return;
    }
    const int ncols = (t.off[lj + 1] - t.off[lj]) * b;
    const size_t r0 = (size_t)(pi - t.off[li]) * b, c0 = (size_t)(pj - t.off[lj]) * b;
    const double *src = vals + (size_t)p * b * b;
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        dst[(r0 + r) * ncols + c0 + c] = src[e];
    }
}

// block row of every stored block (level 0 has no such array from the Galerkin setup)
__global__ void rows_of_blocks_kernel(const int64_t *__restrict__ row_ptr, const int64_t n_brows, int64_t *__restrict__ rob) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_brows) return;
    for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p) rob[p] = I;
}

// ---- in-place Gauss-Jordan inverse without pivoting (the Schur complements inherit a positive definite symmetric part)
// step p, part 1: save column p, scale row p
__global__ void gj_pivot_kernel(double *__restrict__ A, const int n, const int p, double *__restrict__ colp, int *__restrict__ bad) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double piv = A[(size_t)p * n + p];
    if (j == 0 && !(fabs(piv) > 0.0)) atomicExch(bad, 2);
    const double d = 1.0 / piv;
    colp[j] = (j == p) ? 0.0 : A[(size_t)j * n + p];   // column p (read) and row p (written) only meet in the pivot
    if (j != p) A[(size_t)p * n + j] *= d;
}
// step p, part 2: eliminate column p from every other row; column p becomes -colp * d, A[p][p] = d
__global__ void __launch_bounds__(256) gj_update_kernel(double *__restrict__ A, const int n, const int p,
                                                        const double *__restrict__ colp) {
    const int j = blockIdx.x * 256 + threadIdx.x;
    const int i0 = blockIdx.y * 16;
    if (j >= n) return;
    const double d = 1.0 / A[(size_t)p * n + p];   // pivot itself is still untouched (j == p is skipped in part 1)
    const double apj = A[(size_t)p * n + j];
    for (int i = i0; i < i0 + 16 && i < n; ++i) {
        if (i == p) continue;
        const double f = colp[i];
        if (j == p) A[(size_t)i * n + p] = -f * d;
        else A[(size_t)i * n + j] = fma(-f, apj, A[(size_t)i * n + j]);
    }
}
__global__ void gj_finish_pivot_kernel(double *__restrict__ A, const int n, const int p) {
    A[(size_t)p * n + p] = 1.0 / A[(size_t)p * n + p];
}

// ---- C (m x n) = beta * C0 + alpha * A (m x k) * B (k x n), all row-major; 32 x 32 tiles in shared memory
__global__ void __launch_bounds__(1024) dense_gemm_kernel(const double *__restrict__ A, const double *__restrict__ B,
                                                          const double *__restrict__ C0, double *__restrict__ C, const int m,
                                                          const int n, const int k, const double alpha, const double beta) {
    __shared__ double As[32][33], Bs[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int row = blockIdx.y * 32 + ty, col = blockIdx.x * 32 + tx;
    double acc = 0.0;
    for (int k0 = 0; k0 < k; k0 += 32) {
        As[ty][tx] = (row < m && k0 + tx < k) ? A[(size_t)row * k + k0 + tx] : 0.0;
        Bs[ty][tx] = (k0 + ty < k && col < n) ? B[(size_t)(k0 + ty) * n + col] : 0.0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 32; ++q) acc = fma(As[ty][q], Bs[q][tx], acc);
        __syncthreads();
    }
    if (row < m && col < n) C[(size_t)row * n + col] = (beta != 0.0 ? beta * C0[(size_t)row * n + col] : 0.0) + alpha * acc;
}

// ---- y = (y0 or 0) + sign * A x, A row-major rows x cols; one warp per row (the solve's only kernel: bandwidth bound)
__global__ void __launch_bounds__(256) dense_gemv_kernel(const double *__restrict__ A, const double *__restrict__ x,
                                                         const double *__restrict__ y0, double *__restrict__ y, const int rows,
                                                         const int cols, const double sign) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const double *a = A + (size_t)row * cols;
    double acc0 = 0.0, acc1 = 0.0;
    if ((cols & 1) == 0 && (reinterpret_cast<uintptr_t>(x) & 15) == 0 && (reinterpret_cast<uintptr_t>(a) & 15) == 0) {
        const double2 *a2 = reinterpret_cast<const double2 *>(a);
        const double2 *x2 = reinterpret_cast<const double2 *>(x);
#pragma unroll 4
        for (int c = lane; c < (cols >> 1); c += 32) {
            const double2 av = a2[c], xv = x2[c];
            acc0 = fma(av.x, xv.x, acc0);
            acc1 = fma(av.y, xv.y, acc1);
        }
    } else {
        for (int c = lane; c < cols; c += 32) acc0 = fma(a[c], x[c], acc0);
    }
    double s = acc0 + acc1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) y[row] = (y0 != nullptr ? y0[row] : 0.0) + sign * s;
}

// block-row permutation of a vector: dst[new p] = src[perm[p]] (gather) or dst[perm[p]] = src[p] (scatter)
__global__ void permute_blocks_kernel(const double *__restrict__ src, double *__restrict__ dst, const int32_t *__restrict__ perm,
                                      const int64_t n_brows, const int b, const int scatter) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_brows * b) return;
    const int64_t p = e / b;
    const int c = (int)(e - p * b);
    if (scatter) dst[(int64_t)perm[p] * b + c] = src[e];
    else dst[e] = src[(int64_t)perm[p] * b + c];
}

}  // namespace mgk
