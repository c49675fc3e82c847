// kernels_setup.cuh -- mg_setup kernels: input validation, batched inversion of the
// diagonal blocks ("PBJ smoothers ... compute explicit, dense inverses of these diagonal blocks",
// PAPER.md:63) and the numeric Galerkin product A_{l+1} = P^T A_l P, which for
// P = P_phi (x) I is a weighted sum of fine blocks with weights in {1, 1/2, 1/4}: a gather, not an SpGEMM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

// err[0] = min over offending rows of (row + 1); 0 = pattern is valid.  Checks: ascending columns in range,
// diagonal block present; records its position.
__global__ void __launch_bounds__(256) check_pattern_kernel(const int64_t *__restrict__ row_ptr,
                                                            const int32_t *__restrict__ col_idx, const int64_t n,
                                                            int64_t *__restrict__ diag_pos,
                                                            unsigned long long *__restrict__ err_pattern,
                                                            unsigned long long *__restrict__ err_diag) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n) return;
    const int64_t p0 = row_ptr[I], p1 = row_ptr[I + 1];
    int64_t dp = -1;
    bool bad = p1 < p0;
    int64_t prev = -1;
    for (int64_t p = p0; p < p1; ++p) {
        const int64_t J = col_idx[p];
        if (J <= prev || J >= n) bad = true;
        prev = J;
        if (J == I) dp = p;
    }
    diag_pos[I] = dp;
    if (bad) atomicMin(err_pattern, (unsigned long long)(I + 1));
    if (dp < 0) atomicMin(err_diag, (unsigned long long)(I + 1));
}

// One CTA per diagonal block: Gauss-Jordan elimination with partial (row) pivoting on [D | I] held in shared
// memory (b x 2b doubles); first maximal entry wins ties.  A zero / NaN pivot reports the block row in err.
__global__ void __launch_bounds__(128) invert_blocks_kernel(const double *__restrict__ vals,
                                                            const int64_t *__restrict__ diag_pos, const int b,
                                                            double *__restrict__ dinv,
                                                            unsigned long long *__restrict__ err) {
    extern __shared__ double sm[];
    double *M = sm;                 // b x 2b
    double *fcol = sm + 2 * b * b;  // b
    __shared__ int piv_s;
    __shared__ double pivval_s;
    const int64_t I = blockIdx.x;
    const int w2 = 2 * b;
    const double *D = vals + (size_t)diag_pos[I] * b * b;
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        M[r * w2 + c] = D[e];
        M[r * w2 + b + c] = (r == c) ? 1.0 : 0.0;
    }
    __syncthreads();
    for (int k = 0; k < b; ++k) {
        if (threadIdx.x < 32) {
            double best = -1.0;
            int piv = k;
            for (int r = k + (int)threadIdx.x; r < b; r += 32) {
                const double v = fabs(M[r * w2 + k]);
                if (v > best || v != v) { best = v; piv = r; }
            }
            for (int o = 16; o > 0; o >>= 1) {
                const double ob = __shfl_xor_sync(0xffffffffu, best, o);
                const int op = __shfl_xor_sync(0xffffffffu, piv, o);
                if (ob > best || (ob == best && op < piv) || ob != ob) { best = ob; piv = op; }
            }
            if (threadIdx.x == 0) { piv_s = piv; pivval_s = best; }
        }
        __syncthreads();
        const int piv = piv_s;
        if (!(pivval_s > 0.0)) {  // zero or NaN pivot
            if (threadIdx.x == 0) atomicMin(err, (unsigned long long)(I + 1));
            return;
        }
        if (piv != k)
            for (int c = threadIdx.x; c < w2; c += blockDim.x) {
                const double t = M[k * w2 + c];
                M[k * w2 + c] = M[piv * w2 + c];
                M[piv * w2 + c] = t;
            }
        __syncthreads();
        const double inv = 1.0 / M[k * w2 + k];
        __syncthreads();
        for (int c = threadIdx.x; c < w2; c += blockDim.x) M[k * w2 + c] *= inv;
        for (int r = threadIdx.x; r < b; r += blockDim.x) fcol[r] = M[r * w2 + k];
        __syncthreads();
        for (int e = threadIdx.x; e < b * w2; e += blockDim.x) {
            const int r = e / w2, c = e - r * w2;
            if (r != k) M[e] -= fcol[r] * M[k * w2 + c];
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        dinv[(size_t)I * b * b + e] = M[r * w2 + b + c];
    }
}

// P_phi[k, K] for n_c = n_f/2 coarse planes, by the "+=" definition (periodic, coarse plane K on fine plane 2K).
__device__ __host__ __forceinline__ double pphi_entry(const int k, const int K, const int n_f) {
    const int n_c = n_f / 2;
    double w = 0.0;
    if (k == 2 * K) w += 1.0;
    if (k & 1) {
        if ((k - 1) / 2 == K) w += 0.5;
        if (((k + 1) / 2) % n_c == K) w += 0.5;
    }
    return w;
}

// One CTA per coarse block ((i,K),(j,M)): A_c = sum_{k,m} P_phi[k,K] P_phi[m,M] A[(i,k),(j,m)] over the (deduplicated)
// fine planes k in {2K-1, 2K, 2K+1}, m in {2M-1, 2M, 2M+1}; the fine block is found by binary search in row (i,k).
__global__ void __launch_bounds__(128) galerkin_numeric_kernel(const int64_t *__restrict__ row_ptr,
                                                               const int32_t *__restrict__ col_idx,
                                                               const double *__restrict__ vals,
                                                               const int64_t *__restrict__ crow_of_block,
                                                               const int32_t *__restrict__ ccol_idx,
                                                               double *__restrict__ cvals, const int n_pol, const int n_f,
                                                               const int b) {
    const int64_t q = blockIdx.x;
    const int64_t Ic = crow_of_block[q];
    const int64_t Jc = ccol_idx[q];
    const int K = (int)(Ic / n_pol), i = (int)(Ic % n_pol);
    const int M = (int)(Jc / n_pol), j = (int)(Jc % n_pol);
    const int bb = b * b;
    int ks[3] = {(2 * K - 1 + n_f) % n_f, 2 * K, (2 * K + 1) % n_f};
    int ms[3] = {(2 * M - 1 + n_f) % n_f, 2 * M, (2 * M + 1) % n_f};
    __shared__ int64_t src[9];
    __shared__ double wgt[9];
    __shared__ int nsrc;
    if (threadIdx.x == 0) {
        int cnt = 0;
        for (int a = 0; a < 3; ++a) {
            bool dupk = false;
            for (int a2 = 0; a2 < a; ++a2) dupk |= (ks[a2] == ks[a]);
            if (dupk) continue;
            const double wk = pphi_entry(ks[a], K, n_f);
            if (wk == 0.0) continue;
            const int64_t If = (int64_t)ks[a] * n_pol + i;
            for (int c = 0; c < 3; ++c) {
                bool dupm = false;
                for (int c2 = 0; c2 < c; ++c2) dupm |= (ms[c2] == ms[c]);
                if (dupm) continue;
                const double wm = pphi_entry(ms[c], M, n_f);
                if (wm == 0.0) continue;
                const int64_t Jf = (int64_t)ms[c] * n_pol + j;
                int64_t lo = row_ptr[If], hi = row_ptr[If + 1] - 1, found = -1;
                while (lo <= hi) {
                    const int64_t mid = (lo + hi) >> 1;
                    const int64_t cv = col_idx[mid];
                    if (cv == Jf) { found = mid; break; }
                    if (cv < Jf) lo = mid + 1; else hi = mid - 1;
                }
                if (found >= 0) { src[cnt] = found; wgt[cnt] = wk * wm; ++cnt; }
            }
        }
        nsrc = cnt;
    }
    __syncthreads();
    const int cnt = nsrc;
    for (int e = threadIdx.x; e < bb; e += blockDim.x) {
        double acc = 0.0;
        for (int s = 0; s < cnt; ++s) acc = fma(wgt[s], vals[(size_t)src[s] * bb + e], acc);
        cvals[(size_t)q * bb + e] = acc;
    }
}

// Ahat_p = A_p * Dinv_{col(p)}: the right-PBJ-preconditioned operator A D^-1 of the coarsest-level GMRES as ONE
// block-CSR matrix with A's pattern ("right-preconditioned ... M_c = D^-1").  A GMRES
// step is then a single SpMV instead of a PBJ apply followed by an SpMV.  One CTA per block; plain triple loop in
// FP64 (k innermost in stored order), b <= 64.
__global__ void __launch_bounds__(256) right_scale_blocks_kernel(const int32_t *__restrict__ col_idx,
                                                                 const double *__restrict__ vals,
                                                                 const double *__restrict__ dinv, double *__restrict__ out,
                                                                 const int b) {
    extern __shared__ double rs_sm[];
    const int bb = b * b;
    double *As = rs_sm, *Ds = rs_sm + bb;
    const int64_t p = blockIdx.x;
    const double *Ap = vals + (size_t)p * bb;
    const double *Dp = dinv + (size_t)col_idx[p] * bb;
    for (int e = threadIdx.x; e < bb; e += blockDim.x) {
        As[e] = Ap[e];
        Ds[e] = Dp[e];
    }
    __syncthreads();
    for (int e = threadIdx.x; e < bb; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        double acc = 0.0;
        for (int k = 0; k < b; ++k) acc = fma(As[r * b + k], Ds[k * b + c], acc);
        out[(size_t)p * bb + e] = acc;
    }
}

}  // namespace mgk
