// kernels_direct.cuh -- direct solve of the coarsest level (the paper solves its coarsest grid with
// an LU factorisation, and applies block solvers as "explicit inverses and BLAS2").
//
// The block rows of the coarsest level are ordered by the level sets of a breadth-first search of its block graph: every
// block then couples only rows of the same or of adjacent level sets, i.e. the matrix is BLOCK TRIDIAGONAL with dense
// diagonal blocks D_k (n_k x n_k) and SPARSE off-diagonal blocks L_k (n_k x n_{k-1}), U_k (n_k x n_{k+1}), which stay in
// the level's block-CSR storage.  The elimination runs from BOTH ends of the chain towards a middle level set m ("burn at
// both ends"): two independent recurrences, so every step of the solve has two level sets to work on -- twice the bytes per
// dependent step, which is what makes the solve bandwidth bound instead of latency bound.  Setup (off the solve path)
// forms the inverses of the Schur complements explicitly,
//      S_0 = D_0,  S_k = D_k - (L_k S_{k-1}^-1) U_{k-1}  (k < m);      S_q = D_q,  S_k = D_k - (U_k S_{k+1}^-1) L_{k+1}  (k > m);
//      S_m = D_m - (L_m S_{m-1}^-1) U_{m-1} - (U_m S_{m+1}^-1) L_{m+1},
// (only S_k^-1 is kept: sum_k n_k^2 doubles plus one n_k x n_{k+-1} scratch) and the solve is dense mat-vec streaming
// (2 n_k^2 doubles per level set) interleaved with small sparse products:
//      elimination:       y_k = S_k^-1 (b_k - L_k y_{k-1})  (k < m),    y_k = S_k^-1 (b_k - U_k y_{k+1})  (k > m),
//                         x_m = S_m^-1 (b_m - L_m y_{m-1} - U_m y_{m+1});
//      back-substitution: x_k = y_k - S_k^-1 (U_k x_{k+1})  (k < m),    x_k = y_k - S_k^-1 (L_k x_{k-1})  (k > m).
// Per NEW block row the blocks an elimination step multiplies ("elim" list) and those of the back-substitution ("back"
// list) are listed at setup.  All dense matrices are row-major FP64.
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
                                                             const int rows, const double *v, const double *y0, double *out,
                                                             const double sign) {   // v, y0, out: written by the preceding
                                                                                    // kernels of the chain -> no __restrict__
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

// Setup: M (n_k x n_kp) = (blocks of level set k with columns in the neighbouring level set kp) S_kp^-1, i.e. L_k S_{k-1}^-1 or
// U_k S_{k+1}^-1, read from the block-CSR storage.  grid (ceil(n_kp / 128), block rows of level set k); thread = one column
// of M, 4 scalar rows at a time.
__global__ void __launch_bounds__(128) direct_lsinv_kernel(const int64_t *__restrict__ row_ptr,
                                                           const int32_t *__restrict__ col_idx,
                                                           const double *__restrict__ vals, const int b, const DirectTables t,
                                                           const int k, const int kp, const double *__restrict__ Sprev,
                                                           const int nprev, double *__restrict__ M) {
    const int64_t I = t.perm[t.off[k] + blockIdx.y];
    const int c = blockIdx.x * 128 + threadIdx.x;
    if (c >= nprev) return;
    const int64_t p0 = row_ptr[I], p1 = row_ptr[I + 1];
    const int first_prev = t.off[kp];
    for (int r0 = 0; r0 < b; r0 += 4) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (int64_t p = p0; p < p1; ++p) {
            const int pj = t.inv[col_idx[p]];
            if (t.lev[pj] != kp) continue;
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

// Setup: S_k -= M X with X = the blocks (row in level set kp, column in level set k), i.e. U_{k-1} or L_{k+1}.  The blocks of X in
// block column C of level set k are listed (positions in the block-CSR arrays) in csc_pos[csc_ptr[new position of C] ...].
// grid (block columns of level set k, ceil(n_k / 32)).
__global__ void __launch_bounds__(128) direct_schur_kernel(const int64_t *__restrict__ ucsc_ptr,
                                                           const int64_t *__restrict__ ucsc_pos,
                                                           const int64_t *__restrict__ row_of_block,
                                                           const double *__restrict__ vals, const int b, const DirectTables t,
                                                           const int k, const int kp, const double *__restrict__ M,
                                                           const int nprev, double *__restrict__ S, const int nk) {
    const int cnew = t.off[k] + blockIdx.x;
    const int first_prev = t.off[kp];
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
__global__ void __launch_bounds__(256) dense_gemv_kernel(const double *__restrict__ A, const double *x, const double *y0, double *y,
                                                         const int rows, const int cols, const double sign) {   // x, y0, y: chain data
                                                                                    // (y0 may alias y): no __restrict__
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
__global__ void permute_blocks_kernel(const double *src, double *dst, const int32_t *__restrict__ perm,
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


// ================================================================================================ persistent direct solve
// ONE cooperative launch per coarsest-level direct solve instead of a chain of ~4 launches per level set.
//
//   * A STEP holds up to two independent jobs (one level set of the lower chain, one of the upper chain; see the top of
//     this file); a job is (A) the sparse off-diagonal product t = z_k - X y (elimination) or t = X x (back-substitution)
//     and (B) the dense product with S_k^-1.  The rows of a step's jobs are concatenated and split evenly over the CTAs.
//   * grid = one CTA per SM, co-resident (cooperative launch); CTA c owns a contiguous row range of every step: of the
//     dense inverses (contiguous spans of the row-major matrices) and of the off-diagonal block rows, which the numeric
//     phase packs row by row into a padded (ELL) array in the level-set ordering;
//   * hence the whole matrix stream of a solve is STATIC and contiguous per CTA and step: one producer warp walks it from
//     start to end with 1-D bulk async copies (TMA engine, SASS UBLKCP) into a shared-memory ring of DS_SEG-double stages,
//     gated only by the ring's "empty" barriers: it runs ahead across the steps while the consumers exchange vectors;
//   * NO grid barrier: the vectors the CTAs exchange (y of the elimination, x of the back-substitution, t of every step)
//     are written exactly once per solve into buffers that the host fills with a SENTINEL bit pattern (all ones, a NaN
//     no arithmetic produces) before the launch; a reader polls the values it needs until none is the sentinel (8-byte
//     accesses at the L2 coherence point).  A dependent step therefore costs two global round trips (y -> gathered by (A),
//     t -> read by (B)) instead of two barriers plus two round trips, and a CTA waits only for the values it really needs;
//   * 7 consumer warps per CTA.  (A): DS_TPR threads per scalar row, packed block rows out of the ring, only the gathered
//     y / x values come from global memory (the column lists were fetched during the preceding step);  (B): every CTA copies
//     the step's t into shared memory and its warps multiply the CTA's rows of S_k^-1 out of the ring (one row per warp at
//     a time, 128-bit shared-memory reads, fixed summation order), writing y_k / x_k.  The permutation of the right-hand
//     side and of the solution rides in (A) and (B).
// Measured and rejected: grid barriers between (A) and (B) (2.3 ms per C1 solve one-sided, 1.78 ms two-sided: a step is
// then ~12 us of dependent latency against 10-20 us of streaming); prefetching the stream into L2 ahead of the ring
// (cp.async.bulk.prefetch.L2, 48 / 160 stages ahead: 6 % / 50 % SLOWER, the L2 -> SM path is not faster than HBM here).
// Requirements (checked by the host, otherwise the launch chain above is used): b even (16-byte aligned rows for the bulk
// copies), 8 <= b <= 64, at most DS_MAXNE listed blocks per block row and list, the t vectors of a step + DS_PL ring stages +
// the step table fit the shared memory, the packed stages of one step of one CTA fit the ring together.
#ifndef MG_DS_SEG
#define MG_DS_SEG 1024
#endif
constexpr int DS_SEG = MG_DS_SEG;       // doubles per ring stage (8 KB)
constexpr int DS_WARPS = 7;             // consumer warps (+ 1 producer warp = 8: register allocation is per 4 warps)
constexpr int DS_THREADS = (DS_WARPS + 1) * 32;
constexpr int DS_PL = 16;               // producer lanes issuing copies in parallel
constexpr int DS_MAXNE = 16;            // listed blocks per block row and list (ELL width); DS_MAXNE * 64 <= DS_SEG
constexpr int DS_TPR = 8;               // threads per scalar row in the off-diagonal phase
constexpr int DS_NCOL = 8;              // listed blocks of a row handled out of registers (more: a second, slower pass)
struct DsJob {
    const double *S;        // S_k^-1, row-major n x n
    long long ell_off;      // offset (doubles) of the job's packed off-diagonal rows [n][ne][b]
    int n;                  // scalars in the level set (0: no job)
    int first;              // first NEW block position of the level set (scalar offset = first * b)
    int ne;                 // ELL width (0: no blocks)
    int phase;              // 0 elimination (t = z - X y, y = S^-1 t), 1 back-substitution (t = X x, x = y - S^-1 t)
    int final;              // the job's result is final: scatter it to the natural ordering (and, phase 0, copy it to xb)
    int toff;               // offset of the job's t in tb
};
struct DsStepDesc {
    DsJob j[2];
};
struct DirectSolveArgs {
    const DsStepDesc *steps;  // [nsteps]
    int nsteps, b;
    const double *ell;       // packed off-diagonal rows
    const int32_t *ell_col;  // [phase][new block row][DS_MAXNE] new block column or -1
    const int32_t *perm;     // block row at NEW position p
    const double *rhs;       // [n] natural ordering
    double *e;               // [n] natural ordering (solution)
    double *yb, *xb, *tb;    // [n] elimination results, [n] back-substitution results (permuted ordering), [sum of the steps' t];
                             // all SENTINEL-filled at launch, every entry written once
    int64_t n_brows;
    int stages, tcap;        // ring stages, capacity of the shared-memory copy of t (doubles)
};
inline size_t direct_smem_bytes(int stages, int tcap, int nsteps) {
    return sizeof(double) * ((size_t)stages * DS_SEG + (size_t)tcap) + sizeof(DsStepDesc) * (size_t)nsteps +
           sizeof(uint64_t) * 2 * (size_t)stages + sizeof(int) * (size_t)stages + 64;
}

// Numeric phase: pack the listed off-diagonal blocks of every block row (list 0 = elimination / 1 = back-substitution) into
// the ELL array of its level set.  grid (n_brows, 2); lev_ne / lev_off: [nlev][2].
__global__ void __launch_bounds__(128) direct_pack_ell_kernel(const int64_t *__restrict__ od_ptr0, const int64_t *__restrict__ od_pos0,
                                                              const int32_t *__restrict__ od_col0, const int64_t *__restrict__ od_ptr1,
                                                              const int64_t *__restrict__ od_pos1, const int32_t *__restrict__ od_col1,
                                                              const double *__restrict__ vals, const int b, const int32_t *__restrict__ lev,
                                                              const int32_t *__restrict__ off, const int *__restrict__ lev_ne,
                                                              const long long *__restrict__ lev_off, double *__restrict__ ell,
                                                              int32_t *__restrict__ ell_col, const int64_t n_brows) {
    const int64_t pn = blockIdx.x;
    const int side = blockIdx.y;
    const int k = lev[pn];
    const int ne = lev_ne[2 * k + side];
    const int64_t *optr = side ? od_ptr1 : od_ptr0, *opos = side ? od_pos1 : od_pos0;
    const int32_t *ocol = side ? od_col1 : od_col0;
    const int64_t u0 = optr[pn], cnt = optr[pn + 1] - u0;
    int32_t *cdst = ell_col + ((size_t)side * n_brows + pn) * DS_MAXNE;
    for (int i = threadIdx.x; i < DS_MAXNE; i += blockDim.x) cdst[i] = i < cnt ? ocol[u0 + i] : -1;
    if (ne == 0) return;
    double *dst = ell + lev_off[2 * k + side] + (size_t)(pn - off[k]) * b * ne * b;   // [r][i][c]
    for (int e = threadIdx.x; e < b * ne * b; e += blockDim.x) {
        const int r = e / (ne * b), rem = e - r * ne * b, i = rem / b, c = rem - i * b;
        dst[e] = i < cnt ? vals[((size_t)opos[u0 + i] * b + r) * b + c] : 0.0;
    }
}

__device__ __forceinline__ uint32_t ds_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ds_mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ds_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void ds_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ds_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ds_mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(ds_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool ds_mbar_try(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(ds_smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void ds_bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            ds_smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(ds_smem_u32(bar)), "l"(policy)
        : "memory");
}
// Sentinel-polled exchange: 8-byte accesses at the L2 coherence point (never L1).
__device__ __forceinline__ double ds_ld(const double *p) {
    double v;
    asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void ds_st(double *p, const double v) {
    asm volatile("st.relaxed.gpu.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}
__device__ __forceinline__ bool ds_missing(const double v) { return __double_as_longlong(v) == -1ll; }
// A poll gives up after this many tries (a fraction of a second): a right-hand side that itself holds the sentinel bit pattern (a NaN with an
// all-ones payload) must end in NaNs, not in a hang.
constexpr int DS_SPIN_MAX = 1 << 18;   // (a legitimate wait is a few hundred polls)

// One CTA's share of one step: per job the rows [ra, rb) of the level set.  Stream order: the packed off-diagonal rows of
// job 0 (`rps` rows per stage), those of job 1, then the rows of S^-1 of job 0 in segments of DS_SEG doubles, then job 1's.
struct DsPiece {
    const double *S, *ell;
    int n, first, ra, rb, nseg, rowlen, rps, nA, nB, toff, phase, final;
};
struct DsWork {
    DsPiece p[2];
    int nA, total, nt, t0;   // packed stages, all stages, scalars of t in the step, offset of the step's t in tb
};
__device__ __forceinline__ DsWork ds_work(const DirectSolveArgs &a, const DsStepDesc &sd, const int c, const int G) {
    DsWork w;
    const int n0 = sd.j[0].n, n1 = sd.j[1].n;
    const int nt = n0 + n1;
    const int lo = (int)((long long)nt * c / G), hi = (int)((long long)nt * (c + 1) / G);
    w.nt = nt;
    w.t0 = sd.j[0].toff;
    w.nA = 0;
    w.total = 0;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const DsJob &J = sd.j[q];
        DsPiece &P = w.p[q];
        const int base = q ? n0 : 0;
        P.S = J.S;
        P.n = J.n;
        P.first = J.first;
        P.ra = min(max(lo - base, 0), J.n);
        P.rb = min(max(hi - base, 0), J.n);
        P.nseg = (J.n + DS_SEG - 1) / DS_SEG;
        P.rowlen = J.ne * a.b;
        P.rps = P.rowlen > 0 ? DS_SEG / P.rowlen : 1;
        P.ell = a.ell + J.ell_off;
        P.nA = P.rowlen > 0 ? (P.rb - P.ra + P.rps - 1) / P.rps : 0;
        P.nB = (P.rb - P.ra) * P.nseg;
        P.toff = J.toff;
        P.phase = J.phase;
        P.final = J.final;
        w.nA += P.nA;
        w.total += P.nA + P.nB;
    }
    return w;
}
// source address and length (doubles) of stage i of a step's stream
__device__ __forceinline__ const double *ds_stage_src(const DsWork &w, int i, int &len) {
    if (i < w.nA) {
        DsPiece P = w.p[0];   // (copies selected field by field: an indexed reference would put the struct in local memory)
        if (i >= w.p[0].nA) {
            i -= w.p[0].nA;
            P = w.p[1];
        }
        const int r0 = P.ra + i * P.rps;
        len = min(P.rps, P.rb - r0) * P.rowlen;
        return P.ell + (size_t)r0 * P.rowlen;
    }
    i -= w.nA;
    DsPiece P = w.p[0];
    if (i >= w.p[0].nB) {
        i -= w.p[0].nB;
        P = w.p[1];
    }
    const int row = P.ra + i / P.nseg, sg = i - (i / P.nseg) * P.nseg;
    len = min(DS_SEG, P.n - sg * DS_SEG);
    return P.S + (size_t)row * P.n + (size_t)sg * DS_SEG;
}
// column list (first DS_NCOL entries) and permutation entry of NEW block row `pn`: static data
__device__ __forceinline__ void ds_load_cols(const DirectSolveArgs &a, const int phase, const int pn, const bool have, int (&ncol)[DS_NCOL],
                                             int &nperm) {
    const int32_t *cl = a.ell_col + ((size_t)phase * a.n_brows + pn) * DS_MAXNE;
#pragma unroll
    for (int w = 0; w < DS_NCOL; ++w) ncol[w] = have ? __ldg(cl + w) : -1;
    nperm = have ? __ldg(a.perm + pn) : 0;
}
// row q (0-based in the CTA's share of the step) -> piece index and row of the level set; false if q is beyond the share
__device__ __forceinline__ bool ds_row_of(const DsWork &w, const int q, int &pi, int &row) {
    const int r0 = w.p[0].rb - w.p[0].ra;
    pi = q < r0 ? 0 : 1;
    row = pi == 0 ? w.p[0].ra + q : w.p[1].ra + (q - r0);
    return q < r0 + (w.p[1].rb - w.p[1].ra);
}

#ifdef MG_DS_STAMP   // development probe (compiled out in the library): per-phase global-timer stamps of CTA 0
__device__ unsigned long long ds_stamps[16384];
#define DS_STAMP(slot) \
    if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && (threadIdx.x == 0 || threadIdx.x == DS_WARPS * 32) && s < 2000) { \
        unsigned long long t__; \
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t__)); \
        ds_stamps[s * 8 + (slot)] = t__; \
    }
#else
#define DS_STAMP(slot)
#endif

__global__ void __launch_bounds__(DS_THREADS, 1) direct_solve_persistent_kernel(const DirectSolveArgs a) {
    extern __shared__ __align__(128) unsigned char ds_smem[];
    double *ring = reinterpret_cast<double *>(ds_smem);
    double *tsm = ring + (size_t)a.stages * DS_SEG;
    DsStepDesc *steps = reinterpret_cast<DsStepDesc *>(tsm + a.tcap);
    uint64_t *full = reinterpret_cast<uint64_t *>(steps + a.nsteps);
    uint64_t *empty = full + a.stages;
    volatile int *round_of = reinterpret_cast<volatile int *>(empty + a.stages);   // rounds for which a stage has been issued
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x, b = a.b, ST = a.stages;
    const int nsteps = a.nsteps;
    if (tid == 0) {
        for (int s = 0; s < ST; ++s) {
            round_of[s] = 0;
            ds_mbar_init(&full[s], 1);
            ds_mbar_init(&empty[s], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {   // the step table (static) into shared memory: no global round trip at the start of a step
        const int words = (int)(sizeof(DsStepDesc) / sizeof(int)) * nsteps;
        const int *src = reinterpret_cast<const int *>(a.steps);
        int *dst = reinterpret_cast<int *>(steps);
        for (int i = tid; i < words; i += DS_THREADS) dst[i] = __ldg(src + i);
    }
    __syncthreads();

    if (warp == DS_WARPS) {
        // ---------------------------------------------------------------- producer: the CTA's static matrix stream
        uint64_t pol;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
        long long cnt = 0;
        for (int s = 0; s < nsteps; ++s) {
            const DsWork d = ds_work(a, steps[s], c, G);
            for (int base = 0; base < d.total; base += DS_PL) {
                const int i = base + lane;
                if (lane < DS_PL && i < d.total) {
                    const long long cc = cnt + i;
                    const int st = (int)(cc % ST);
                    const int round = (int)(cc / ST);
                    while (!ds_mbar_try(&empty[st], ((uint32_t)round & 1u) ^ 1u)) {
                    }
                    round_of[st] = round + 1;
                    int len;
                    const double *src = ds_stage_src(d, i, len);
                    ds_mbar_expect_tx(&full[st], (uint32_t)(len * sizeof(double)));
                    ds_bulk_g2s(ring + (size_t)st * DS_SEG, src, (uint32_t)(len * sizeof(double)), &full[st], pol);
                }
                __syncwarp();
            }
            cnt += d.total;
            DS_STAMP(7);
        }
        return;
    }

    // -------------------------------------------------------------------- consumers
    long long cnt = 0;
    constexpr int RPP = DS_WARPS * 32 / DS_TPR;   // rows per pass of phase (A)
    constexpr int NV = (64 + DS_TPR - 1) / DS_TPR;   // columns of a block per thread (b <= 64)
    const int sub = tid % DS_TPR;
    int ncol[DS_NCOL], nperm = 0;   // column list / permutation entry of this thread's row in the coming step (first pass)
    {
        const DsWork d0 = ds_work(a, steps[0], c, G);
        int pi, row;
        const bool have = ds_row_of(d0, tid / DS_TPR, pi, row);
        ds_load_cols(a, pi ? d0.p[1].phase : d0.p[0].phase, (pi ? d0.p[1].first : d0.p[0].first) + (have ? row : 0) / b, have, ncol, nperm);
    }
    for (int s = 0; s < nsteps; ++s) {
        const DsWork d = ds_work(a, steps[s], c, G);
        DS_STAMP(0);
        // ---- (A) t = z_k - X y   or   t = X x   for the CTA's rows: DS_TPR threads per scalar row; thread `sub` of a row takes
        // the columns sub, sub + DS_TPR, ... of every listed block, all its gathers in flight at once; a gathered value that
        // is still the sentinel has not been written yet and is loaded again
        {
            const int nr = (d.p[0].rb - d.p[0].ra) + (d.p[1].rb - d.p[1].ra);
            int released = 0;   // packed stages of this step handed back so far
            for (int q0 = 0; q0 < nr; q0 += RPP) {
                int pi, row;
                const bool have = ds_row_of(d, q0 + tid / DS_TPR, pi, row);
                DsPiece P = d.p[0];
                if (pi) P = d.p[1];
                if (!have) row = P.ra;
                const int pl = row / b, r = row - pl * b;
                if (q0 != 0) ds_load_cols(a, P.phase, P.first + pl, have, ncol, nperm);
                double acc = 0.0, zv = 0.0;
                if (have && P.phase == 0) zv = __ldg(a.rhs + (size_t)nperm * b + r);
                if (have && P.rowlen > 0) {
                    const double *src = P.phase == 0 ? a.yb : a.xb;
                    const int ne = P.rowlen / b;
                    double xv[DS_NCOL][NV];
#pragma unroll
                    for (int w = 0; w < DS_NCOL; ++w)
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            const int cx = sub + v * DS_TPR;
                            xv[w][v] = (w < ne && ncol[w] >= 0 && cx < b) ? ds_ld(src + (size_t)ncol[w] * b + cx) : 0.0;
                        }
                    bool again;
                    int spins = 0;
                    do {
                        again = false;
#pragma unroll
                        for (int w = 0; w < DS_NCOL; ++w)
#pragma unroll
                            for (int v = 0; v < NV; ++v)
                                if (ds_missing(xv[w][v])) {
                                    xv[w][v] = ds_ld(src + (size_t)ncol[w] * b + sub + v * DS_TPR);
                                    again = again || ds_missing(xv[w][v]);
                                }
                    } while (again && ++spins < DS_SPIN_MAX);
                    const int ql = row - P.ra;                       // row within the piece
                    const long long cc = cnt + (pi ? d.p[0].nA : 0) + ql / P.rps;
                    const int st = (int)(cc % ST);
                    const int round = (int)(cc / ST);
                    while (round_of[st] <= round) __nanosleep(100);
                    while (!ds_mbar_try(&full[st], (uint32_t)round & 1u)) {
                    }
                    const double *As = ring + (size_t)st * DS_SEG + (size_t)(ql - (ql / P.rps) * P.rps) * P.rowlen;
#pragma unroll
                    for (int w = 0; w < DS_NCOL; ++w)
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            const int cx = sub + v * DS_TPR;
                            if (w < ne && cx < b) acc = fma(As[w * b + cx], xv[w][v], acc);
                        }
                    for (int w = DS_NCOL; w < ne; ++w) {   // rows with more listed blocks than registers hold: the plain way
                        const int col = __ldg(a.ell_col + ((size_t)P.phase * a.n_brows + P.first + pl) * DS_MAXNE + w);
                        if (col >= 0)
                            for (int cx = sub; cx < b; cx += DS_TPR) {
                                double x1;
                                do x1 = ds_ld(src + (size_t)col * b + cx);
                                while (ds_missing(x1) && ++spins < DS_SPIN_MAX);
                                acc = fma(As[w * b + cx], x1, acc);
                            }
                    }
                }
#pragma unroll
                for (int o = DS_TPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (have && sub == 0) ds_st(a.tb + P.toff + row, P.phase == 0 ? zv - acc : acc);
                // the packed stages whose rows are all done (this pass and before) go back to the producer once every
                // consumer warp is here: a very wide level set has more packed stages than the ring holds
                asm volatile("bar.sync 1, %0;" ::"n"(DS_WARPS * 32) : "memory");
                {
                    const int qe = min(q0 + RPP, nr);   // rows [0, qe) of the CTA's share are done
                    const int nr0 = d.p[0].rb - d.p[0].ra;
                    const int d0 = qe >= nr0 ? d.p[0].nA : min(d.p[0].nA, qe / d.p[0].rps);   // (nA = 0 for a job without blocks)
                    const int d1 = qe >= nr ? d.p[1].nA : (qe > nr0 ? min(d.p[1].nA, (qe - nr0) / d.p[1].rps) : 0);
                    const int upto = d0 + d1;
                    for (int i = released + tid; i < upto; i += DS_WARPS * 32) ds_mbar_arrive(&empty[(int)((cnt + i) % ST)]);
                    released = upto;
                }
            }
        }
        cnt += d.nA;
        DS_STAMP(1);
        // ---- (B) rows of S_k^-1 times t: the step's t (written by all CTAs) into shared memory, polled until complete
        const int nr0 = d.p[0].rb - d.p[0].ra, nr1 = d.p[1].rb - d.p[1].ra;
        {
            constexpr int tbase = 0;
            const int tlen = d.nt;
            for (int i0 = 0; i0 < tlen; i0 += 16 * DS_WARPS * 32) {   // 16 independent loads in flight per thread
                double tv[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const int i = i0 + tid + u * DS_WARPS * 32;
                    tv[u] = i < tlen ? ds_ld(a.tb + d.t0 + tbase + i) : 0.0;
                }
                bool again;
                int spins = 0;
                do {
                    again = false;
#pragma unroll
                    for (int u = 0; u < 16; ++u)
                        if (ds_missing(tv[u])) {
                            tv[u] = ds_ld(a.tb + d.t0 + tbase + i0 + tid + u * DS_WARPS * 32);
                            again = again || ds_missing(tv[u]);
                        }
                } while (again && ++spins < DS_SPIN_MAX);
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const int i = i0 + tid + u * DS_WARPS * 32;
                    if (i < tlen) tsm[i] = tv[u];
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(DS_WARPS * 32) : "memory");
            DS_STAMP(3);
            for (int i = warp; i < nr0 + nr1; i += DS_WARPS) {
                const int pi = i < nr0 ? 0 : 1;
                DsPiece P = d.p[0];
                if (pi) P = d.p[1];
                const int il = pi ? i - nr0 : i;
                const int row = P.ra + il;
                const long long c0 = cnt + (pi ? d.p[0].nB : 0) + (long long)il * P.nseg;
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
                for (int sg = 0; sg < P.nseg; ++sg) {
                    const long long cc = c0 + sg;
                    const int st = (int)(cc % ST);
                    const int round = (int)(cc / ST);
                    while (round_of[st] <= round) __nanosleep(100);
                    while (!ds_mbar_try(&full[st], (uint32_t)round & 1u)) {
                    }
                    const int len2 = min(DS_SEG, P.n - sg * DS_SEG) >> 1;
                    const double2 *A2 = reinterpret_cast<const double2 *>(ring + (size_t)st * DS_SEG);
                    const double2 *t2 = reinterpret_cast<const double2 *>(tsm + (P.toff - d.t0 - tbase) + (size_t)sg * DS_SEG);
                    int e = lane;
                    for (; e + 32 < len2; e += 64) {
                        const double2 v0 = A2[e], v1 = A2[e + 32];
                        const double2 y0 = t2[e], y1 = t2[e + 32];
                        s0 = fma(v0.x, y0.x, s0);
                        s1 = fma(v0.y, y0.y, s1);
                        s2 = fma(v1.x, y1.x, s2);
                        s3 = fma(v1.y, y1.y, s3);
                    }
                    if (e < len2) {
                        const double2 v0 = A2[e], y0 = t2[e];
                        s0 = fma(v0.x, y0.x, s0);
                        s1 = fma(v0.y, y0.y, s1);
                    }
                    __syncwarp();
                    if (lane == 0) ds_mbar_arrive(&empty[st]);
                }
                double sum = (s0 + s1) + (s2 + s3);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
                if (lane == 0) {
                    const size_t gi = (size_t)P.first * b + row;
                    if (P.phase == 0) {
                        ds_st(a.yb + gi, sum);
                        if (P.final) ds_st(a.xb + gi, sum);   // the middle level set: its result is also the first x
                    } else {
                        int spins = 0;
                        double yk;                            // y_k of the elimination phase (written many steps ago, possibly
                        do yk = ds_ld(a.yb + gi);             // by another CTA: the steps pair the level sets differently)
                        while (ds_missing(yk) && ++spins < DS_SPIN_MAX);
                        sum = yk - sum;
                        ds_st(a.xb + gi, sum);
                    }
                    if (P.final) {   // final value of this row: scatter to the natural ordering
                        const int pl = row / b;
                        a.e[(size_t)__ldg(a.perm + P.first + pl) * b + (row - pl * b)] = sum;
                    }
                }
            }
        }
        cnt += d.p[0].nB + d.p[1].nB;
        DS_STAMP(4);
        if (s + 1 < nsteps) {   // static data of the coming step's first pass
            const DsWork dn = ds_work(a, steps[s + 1], c, G);
            int pi, row;
            const bool have = ds_row_of(dn, tid / DS_TPR, pi, row);
            ds_load_cols(a, pi ? dn.p[1].phase : dn.p[0].phase, (pi ? dn.p[1].first : dn.p[0].first) + (have ? row : 0) / b, have, ncol, nperm);
        }
        // tsm is rewritten in the next step: every warp must be done reading it
        asm volatile("bar.sync 1, %0;" ::"n"(DS_WARPS * 32) : "memory");
        DS_STAMP(6);
    }
}

}  // namespace mgk
