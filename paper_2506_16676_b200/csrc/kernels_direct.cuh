// kernels_direct.cuh -- direct solve of the coarsest level (the paper solves its coarsest grid with
// an LU factorisation, and applies block solvers as "explicit inverses and BLAS2").
//
// The block rows of the coarsest level are ordered by the level sets of a breadth-first search of its block graph: every
// block then couples only rows of the same or of adjacent level sets, i.e. the matrix is BLOCK TRIDIAGONAL with dense
// diagonal blocks D_k (n_k x n_k) and SPARSE off-diagonal blocks L_k (n_k x n_{k-1}), U_k (n_k x n_{k+1}), which stay in
// the level's block-CSR storage.  Setup (off the solve path) forms the inverses of the Schur complements explicitly,
//      S_0 = D_0,   S_k = D_k - (L_k S_{k-1}^-1) U_{k-1},
// (only S_k^-1 is kept: sum_k n_k^2 doubles plus one n_k x n_{k-1} scratch) and the solve is dense mat-vec streaming
// (bandwidth bound, 2 n_k^2 doubles per level set) interleaved with small sparse products:
//      forward :  y_k = S_k^-1 (b_k - L_k y_{k-1})
//      backward:  x_q = y_q,      x_k = y_k - S_k^-1 (U_k x_{k+1})
// All dense matrices are row-major FP64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

struct DirectTables {       // device arrays describing the level-set ordering
    const int32_t *perm;    // [n_brows] block row at NEW position p
    const int32_t *inv;     // [n_brows] new position of block row I
    const int32_t *lev;     // [n_brows] level set of NEW position p
    const int32_t *off;     // [nlev + 1] first new position of every level set
    double *const *S;       // [nlev] dense diagonal blocks (D_k at assembly, then S_k, then S_k^-1)
};

// One CTA per stored block: the blocks inside a level set are scattered into its dense diagonal block.
__global__ void __launch_bounds__(128) direct_assemble_kernel(const int64_t *__restrict__ row_of_block,
                                                              const int32_t *__restrict__ col_idx,
                                                              const double *__restrict__ vals, const int b, const DirectTables t) {
    const int64_t p = blockIdx.x;
    const int pi = t.inv[row_of_block[p]], pj = t.inv[col_idx[p]];
    const int li = t.lev[pi];
    if (t.lev[pj] != li) return;
    double *dst = t.S[li];
    const int ncols = (t.off[li + 1] - t.off[li]) * b;
    const size_t r0 = (size_t)(pi - t.off[li]) * b, c0 = (size_t)(pj - t.off[li]) * b;
    const double *src = vals + (size_t)p * b * b;
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        dst[(r0 + r) * ncols + c0 + c] = src[e];
    }
}

// Sparse off-diagonal product of one level set with an adjacent one (L_k or U_k), one warp per scalar row:
//      out[local row] = (y0 or 0) + sign * sum_{u in list of the block row} A_{pos[u]} v[col[u] * b ...]
// list_ptr is indexed by the NEW position of the block row (first = first new position of the level set), list_pos holds
// positions in the block-CSR arrays and list_col the new position of the block column.  v is a whole vector in the
// permuted numbering; y0 / out are local to the level set.
constexpr int OD_MAXE = 8;   // listed blocks per row held in registers (more: generic loop)
__global__ void __launch_bounds__(128) direct_offdiag_kernel(const int64_t *__restrict__ list_ptr,
                                                             const int64_t *__restrict__ list_pos,
                                                             const int32_t *__restrict__ list_col,
                                                             const double *__restrict__ vals, const int b, const int first,
                                                             const int rows, const double *__restrict__ v,
                                                             const double *__restrict__ y0, double *__restrict__ out,
                                                             const double sign) {
    const int row = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    cudaTriggerProgrammaticLaunchCompletion();   // the dense mat-vec that follows may start prefetching its matrix
    if (row >= rows) {
        cudaGridDependencySynchronize();
        return;
    }
    const int pl = row / b, r = row - pl * b;
    const int64_t u0 = list_ptr[first + pl], u1 = list_ptr[first + pl + 1];   // setup data: independent of the chain
    const int ne = (int)(u1 - u0);
    double acc = 0.0;
    if (ne <= OD_MAXE && b <= 64) {
        // the row of every listed block (setup data too) is in registers before the previous kernel has finished
        double a0[OD_MAXE], a1[OD_MAXE];
        int col[OD_MAXE];
#pragma unroll
        for (int i = 0; i < OD_MAXE; ++i) {
            col[i] = 0;
            a0[i] = a1[i] = 0.0;
            if (i < ne) {
                col[i] = list_col[u0 + i];
                const double *a = vals + ((size_t)list_pos[u0 + i] * b + r) * b;
                if (lane < b) a0[i] = a[lane];
                if (lane + 32 < b) a1[i] = a[lane + 32];
            }
        }
        cudaGridDependencySynchronize();   // v, y0 come from the previous kernels
#pragma unroll
        for (int i = 0; i < OD_MAXE; ++i)
            if (i < ne) {
                const double *x = v + (size_t)col[i] * b;
                if (lane < b) acc = fma(a0[i], x[lane], acc);
                if (lane + 32 < b) acc = fma(a1[i], x[lane + 32], acc);
            }
    } else {
        cudaGridDependencySynchronize();
        for (int64_t u = u0; u < u1; ++u) {
            const double *a = vals + ((size_t)list_pos[u] * b + r) * b;
            const double *x = v + (size_t)list_col[u] * b;
            for (int c = lane; c < b; c += 32) acc = fma(a[c], x[c], acc);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) out[row] = (y0 != nullptr ? y0[row] : 0.0) + sign * acc;
}

// Setup: M (n_k x n_{k-1}) = L_k S_{k-1}^-1 with L_k read from the block-CSR storage.  grid (ceil(n_{k-1} / 128), block
// rows of level set k); thread = one column of M, 4 scalar rows at a time.
__global__ void __launch_bounds__(128) direct_lsinv_kernel(const int64_t *__restrict__ row_ptr,
                                                           const int32_t *__restrict__ col_idx,
                                                           const double *__restrict__ vals, const int b, const DirectTables t,
                                                           const int k, const double *__restrict__ Sprev, const int nprev,
                                                           double *__restrict__ M) {
    const int64_t I = t.perm[t.off[k] + blockIdx.y];
    const int c = blockIdx.x * 128 + threadIdx.x;
    if (c >= nprev) return;
    const int64_t p0 = row_ptr[I], p1 = row_ptr[I + 1];
    const int first_prev = t.off[k - 1];
    for (int r0 = 0; r0 < b; r0 += 4) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (int64_t p = p0; p < p1; ++p) {
            const int pj = t.inv[col_idx[p]];
            if (t.lev[pj] != k - 1) continue;
            const double *a = vals + (size_t)p * b * b;
            const double *s = Sprev + (size_t)(pj - first_prev) * b * nprev + c;
            for (int q = 0; q < b; ++q) {
                const double sv = s[(size_t)q * nprev];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (r0 + i < b) acc[i] = fma(a[(r0 + i) * b + q], sv, acc[i]);
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (r0 + i < b) M[((size_t)blockIdx.y * b + r0 + i) * nprev + c] = acc[i];
    }
}

// Setup: S_k -= M U_{k-1}.  The blocks of U_{k-1} in block column C of level set k are listed (positions in the block-CSR
// arrays) in ucsc_pos[ucsc_ptr[new position of C] ...].  grid (block columns of level set k, ceil(n_k / 32)).
__global__ void __launch_bounds__(128) direct_schur_kernel(const int64_t *__restrict__ ucsc_ptr,
                                                           const int64_t *__restrict__ ucsc_pos,
                                                           const int64_t *__restrict__ row_of_block,
                                                           const double *__restrict__ vals, const int b, const DirectTables t,
                                                           const int k, const double *__restrict__ M, const int nprev,
                                                           double *__restrict__ S, const int nk) {
    const int cnew = t.off[k] + blockIdx.x;
    const int first_prev = t.off[k - 1];
    const int64_t u0 = ucsc_ptr[cnew], u1 = ucsc_ptr[cnew + 1];
    for (int idx = threadIdx.x; idx < 32 * b; idx += blockDim.x) {
        const int m = blockIdx.y * 32 + idx / b, cc = idx % b;
        if (m >= nk) break;
        double acc = 0.0;
        for (int64_t u = u0; u < u1; ++u) {
            const int64_t p = ucsc_pos[u];
            const double *mrow = M + (size_t)m * nprev + (size_t)(t.inv[row_of_block[p]] - first_prev) * b;
            const double *a = vals + (size_t)p * b * b + cc;
            for (int q = 0; q < b; ++q) acc = fma(mrow[q], a[(size_t)q * b], acc);
        }
        S[(size_t)m * nk + (size_t)blockIdx.x * b + cc] -= acc;
    }
}

// block row of every stored block (level 0 has no such array from the Galerkin setup)
__global__ void rows_of_blocks_kernel(const int64_t *__restrict__ row_ptr, const int64_t n_brows, int64_t *__restrict__ rob) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_brows) return;
    for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p) rob[p] = I;
}

// ---- in-place BLOCKED Gauss-Jordan inverse without pivoting (the Schur complements inherit a positive definite symmetric
// part).  Panel K = [p0, p0 + w), w <= 32, three launches per panel:
//      1. Pinv = A[K,K]^-1                                           (one CTA, shared memory)
//      2. C = A[:,K] saved;  A[K,J] = Pinv A[K,J] (J != K),  A[K,K] = Pinv;  R = the new A[K,:]
//      3. A[I,J] = A[I,J] - C[I,:] R[:,J]  (I != K, J != K),   A[I,K] = -C[I,:] Pinv   (I != K)
// which is the scalar elimination (scale row p, eliminate column p, column p becomes -colp / pivot) taken w pivots at a
// time: the matrix is read and written n / w times instead of n times.
constexpr int GJ_W = 32;

__global__ void __launch_bounds__(GJ_W *GJ_W) gj_panel_inverse_kernel(const double *__restrict__ A, const int n, const int p0,
                                                                       const int w, double *__restrict__ Pinv,
                                                                       int *__restrict__ bad) {
    __shared__ double s[GJ_W][GJ_W + 1];
    const int j = threadIdx.x & (GJ_W - 1), i = threadIdx.x / GJ_W;
    const bool in = i < w && j < w;
    s[i][j] = in ? A[(size_t)(p0 + i) * n + p0 + j] : (i == j ? 1.0 : 0.0);
    __syncthreads();
    for (int p = 0; p < w; ++p) {
        const double piv = s[p][p], colp = s[i][p], rowp = s[p][j], aij = s[i][j];
        __syncthreads();
        if (threadIdx.x == 0 && !(fabs(piv) > 0.0 && fabs(piv) < 1.0e300)) atomicExch(bad, 2);
        const double d = 1.0 / piv;
        double v;
        if (i == p) v = (j == p) ? d : rowp * d;
        else if (j == p) v = -colp * d;
        else v = fma(-colp, rowp * d, aij);
        s[i][j] = v;
        __syncthreads();
    }
    if (in) Pinv[i * GJ_W + j] = s[i][j];
}

// one thread per column j of the row panel (and, as a row index, per row of the column panel that is saved)
__global__ void __launch_bounds__(256) gj_row_panel_kernel(double *__restrict__ A, const int n, const int p0, const int w,
                                                           const double *__restrict__ Pinv, double *__restrict__ C,
                                                           double *__restrict__ R) {
    __shared__ double sp[GJ_W][GJ_W + 1];
    for (int e = threadIdx.x; e < GJ_W * GJ_W; e += 256) {
        const int q = e / GJ_W, c = e - q * GJ_W;
        sp[q][c] = (q < w && c < w) ? Pinv[e] : 0.0;
    }
    __syncthreads();
    const int j = blockIdx.x * 256 + threadIdx.x;
    if (j >= n) return;
    if (j < p0 || j >= p0 + w)   // rows outside the panel: save A[j, K] (rows inside are not used by step 3)
        for (int q = 0; q < w; ++q) C[(size_t)j * GJ_W + q] = A[(size_t)j * n + p0 + q];
    double out[GJ_W];
    if (j >= p0 && j < p0 + w) {
#pragma unroll
        for (int q = 0; q < GJ_W; ++q) out[q] = sp[q][j - p0];
    } else {
        double a[GJ_W];
#pragma unroll
        for (int q = 0; q < GJ_W; ++q) a[q] = q < w ? A[(size_t)(p0 + q) * n + j] : 0.0;
#pragma unroll
        for (int q = 0; q < GJ_W; ++q) {
            double acc = 0.0;
#pragma unroll
            for (int c = 0; c < GJ_W; ++c) acc = fma(sp[q][c], a[c], acc);
            out[q] = acc;
        }
    }
#pragma unroll
    for (int q = 0; q < GJ_W; ++q)
        if (q < w) {
            A[(size_t)(p0 + q) * n + j] = out[q];
            R[(size_t)q * n + j] = out[q];
        }
}

// rank-w update, 64 x 64 tile per CTA, 4 x 4 outputs per thread (rows ty + 16 ii, columns tx + 16 jj)
__global__ void __launch_bounds__(256) gj_update_kernel(double *__restrict__ A, const int n, const int p0, const int w,
                                                        const double *__restrict__ C, const double *__restrict__ R) {
    __shared__ double Cs[64][GJ_W + 1], Rs[GJ_W][64];
    const int i0 = blockIdx.y * 64, j0 = blockIdx.x * 64;
    for (int e = threadIdx.x; e < 64 * GJ_W; e += 256) {
        const int i = e / GJ_W, q = e - i * GJ_W;
        const int gi = i0 + i;
        Cs[i][q] = (gi < n && q < w && (gi < p0 || gi >= p0 + w)) ? C[(size_t)gi * GJ_W + q] : 0.0;
    }
    for (int e = threadIdx.x; e < GJ_W * 64; e += 256) {
        const int q = e >> 6, j = e & 63;
        Rs[q][j] = (q < w && j0 + j < n) ? R[(size_t)q * n + j0 + j] : 0.0;
    }
    __syncthreads();
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[4][4];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = 0.0;
#pragma unroll 8
    for (int q = 0; q < GJ_W; ++q) {
        double c[4], r[4];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) c[ii] = Cs[ty + 16 * ii][q];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) r[jj] = Rs[q][tx + 16 * jj];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = fma(c[ii], r[jj], acc[ii][jj]);
    }
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) {
        const int gi = i0 + ty + 16 * ii;
        if (gi >= n || (gi >= p0 && gi < p0 + w)) continue;   // the rows of the panel are final after step 2
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            const int gj = j0 + tx + 16 * jj;
            if (gj >= n) continue;
            double *dst = A + (size_t)gi * n + gj;
            *dst = ((gj >= p0 && gj < p0 + w) ? 0.0 : *dst) - acc[ii][jj];
        }
    }
}

// ---- y = (y0 or 0) + sign * A x, A row-major rows x cols (the solve's dense kernel: bandwidth bound).  Two consecutive rows
// per CTA, walked together by all 256 threads (every step of the CTA reads 2 x 4 KB of consecutive matrix bytes, four
// 128-bit loads per thread in flight per row); the 8 warp sums of a row are combined in a fixed order.  For the few
// thousand rows of a level set this gives ~10 CTAs per SM, so the SMs stay evenly loaded.
constexpr int GEMV_ROWS = 2;
constexpr int GEMV_PREFETCH = 32768;   // leading bytes of the CTA's rows prefetched into L2 before the dependency wait
__global__ void __launch_bounds__(256) dense_gemv_kernel(const double *__restrict__ A, const double *__restrict__ x,
                                                         const double *__restrict__ y0, double *__restrict__ y, const int rows,
                                                         const int cols, const double sign) {
    __shared__ double part[GEMV_ROWS][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r0 = blockIdx.x * GEMV_ROWS;
    const bool two = r0 + 1 < rows;
    const double *a0 = A + (size_t)r0 * cols;
    const double *a1 = two ? a0 + cols : a0;
    // Programmatic dependent launch: the kernels of one direct solve form a chain; A is setup data, so the start of this
    // CTA's rows is pulled into L2 while the previous kernel is still running, then wait for x / y0.
    cudaTriggerProgrammaticLaunchCompletion();
    {
        const char *base = reinterpret_cast<const char *>(a0);
        const size_t bytes = min((size_t)cols * sizeof(double) * (two ? 2 : 1), (size_t)GEMV_PREFETCH);
        for (size_t o = (size_t)threadIdx.x * 128; o < bytes; o += 256 * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + o));
    }
    cudaGridDependencySynchronize();
    double s0 = 0.0, s1 = 0.0, t0 = 0.0, t1 = 0.0;   // row 0: s0 + s1, row 1: t0 + t1
    if ((cols & 1) == 0 && (reinterpret_cast<uintptr_t>(x) & 15) == 0 && (reinterpret_cast<uintptr_t>(A) & 15) == 0) {
        const double2 *p0 = reinterpret_cast<const double2 *>(a0);
        const double2 *p1 = reinterpret_cast<const double2 *>(a1);
        const double2 *x2 = reinterpret_cast<const double2 *>(x);
        const int n2 = cols >> 1;
        int c = threadIdx.x;
        for (; c + 768 < n2; c += 1024) {
            double2 u[4], v[4], xv[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) u[i] = p0[c + 256 * i];
#pragma unroll
            for (int i = 0; i < 4; ++i) v[i] = p1[c + 256 * i];
#pragma unroll
            for (int i = 0; i < 4; ++i) xv[i] = x2[c + 256 * i];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                s0 = fma(u[i].x, xv[i].x, s0);
                s1 = fma(u[i].y, xv[i].y, s1);
                t0 = fma(v[i].x, xv[i].x, t0);
                t1 = fma(v[i].y, xv[i].y, t1);
            }
        }
        for (; c < n2; c += 256) {
            const double2 u = p0[c], v = p1[c], xv = x2[c];
            s0 = fma(u.x, xv.x, s0);
            s1 = fma(u.y, xv.y, s1);
            t0 = fma(v.x, xv.x, t0);
            t1 = fma(v.y, xv.y, t1);
        }
    } else {
        for (int c = threadIdx.x; c < cols; c += 256) {
            const double xv = x[c];
            s0 = fma(a0[c], xv, s0);
            t0 = fma(a1[c], xv, t0);
        }
    }
    double s = s0 + s1, t = t0 + t1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s += __shfl_xor_sync(0xffffffffu, s, o);
        t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    if (lane == 0) {
        part[0][warp] = s;
        part[1][warp] = t;
    }
    __syncthreads();
    if (threadIdx.x < GEMV_ROWS && r0 + (int)threadIdx.x < rows) {
        const double *q = part[threadIdx.x];
        const double sum = ((q[0] + q[1]) + (q[2] + q[3])) + ((q[4] + q[5]) + (q[6] + q[7]));
        const int r = r0 + threadIdx.x;
        y[r] = (y0 != nullptr ? y0[r] : 0.0) + sign * sum;
    }
}

// block-row permutation of a vector: dst[new p] = src[perm[p]] (gather) or dst[perm[p]] = src[p] (scatter)
__global__ void permute_blocks_kernel(const double *__restrict__ src, double *__restrict__ dst, const int32_t *__restrict__ perm,
                                      const int64_t n_brows, const int b, const int scatter) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    cudaTriggerProgrammaticLaunchCompletion();
    cudaGridDependencySynchronize();
    if (e >= n_brows * b) return;
    const int64_t p = e / b;
    const int c = (int)(e - p * b);
    if (scatter) dst[(int64_t)perm[p] * b + c] = src[e];
    else dst[e] = src[(int64_t)perm[p] * b + c];
}

}  // namespace mgk
