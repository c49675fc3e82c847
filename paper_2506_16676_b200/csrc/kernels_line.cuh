// kernels_line.cuh -- toroidal-LINE block-Jacobi preconditioner of the Chebyshev smoother (the
// paper's outlook: "expanding the options for, and size of, the blocks in the PBJ smoothers that fit in a device's thread
// group ... line subdomains (e.g., in the toroidal direction)").
//
// The block of poloidal node i couples the planes k = 0..N-1 of that node: a PERIODIC BLOCK-TRIDIAGONAL matrix with b x b
// blocks D_k = A_{(i,k),(i,k)}, L_k = A_{(i,k),(i,k-1)}, U_k = A_{(i,k),(i,k+1)} (plane indices mod N; for N = 2 the two
// neighbours coincide and the pattern holds ONE off-diagonal block per row; N = 1: the point block).  In the spirit of the
// paper's PBJ ("explicit, dense inverses ... dense matrix-vector products") the setup stores explicit
// b x b inverses, so that an apply is nothing but b x b mat-vecs:
//   chain T = planes 0..C-1 (C = N-1), border = plane N-1:   [T u; v D_{N-1}],  u, v nonzero in block rows 0 and C-1;
//   block Thomas on T:  G_0 = D_0^-1,  G_k = (D_k - L_k G_{k-1} U_{k-1})^-1;
//   W = T^-1 u (C blocks),  S = D_{N-1} - v W,  stored S^-1.
// Apply z = M_line^-1 r:  y_0 = r_0, q_k = G_k y_k, y_k = r_k - L_k q_{k-1};  x_{C-1} = q_{C-1}, x_k = q_k - G_k (U_k x_{k+1});
//   z_{N-1} = S^-1 (r_{N-1} - v x);  z_k = x_k - W_k z_{N-1}.   L_k, U_k, u, v are read from the level's block-CSR values.
// Storage per level: 2 N - 1 blocks per node beside A (G: N blocks incl. S^-1, W: N - 1 blocks).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

// lpos[3 * I + {0,1,2}] = position of the blocks (i,k-1), (i,k), (i,k+1) of block row I = (i,k), or -1.  N = 2: row 0 keeps its
// single off-diagonal block as "upper", row 1 as "lower"; N = 1: none.  bad: set to 1 if a row couples its own node on a
// plane other than k-1, k, k+1 (the line block would not be tridiagonal) or lacks its diagonal block.
__global__ void __launch_bounds__(256) line_positions_kernel(const int64_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx,
                                                             const int n_pol, const int n_phi, int64_t *__restrict__ lpos,
                                                             int *__restrict__ bad) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= (int64_t)n_pol * n_phi) return;
    const int k = (int)(I / n_pol), i = (int)(I % n_pol);
    const int km = (k - 1 + n_phi) % n_phi, kp = (k + 1) % n_phi;
    int64_t lo = -1, di = -1, up = -1;
    for (int64_t p = row_ptr[I]; p < row_ptr[I + 1]; ++p) {
        const int64_t J = col_idx[p];
        if (J % n_pol != i) continue;
        const int m = (int)(J / n_pol);
        if (m == k) di = p;
        else if (n_phi == 2) {
            if (k == 0) up = p; else lo = p;
        } else if (m == km) lo = p;
        else if (m == kp) up = p;
        else atomicExch(bad, 1);
    }
    if (di < 0) atomicExch(bad, 1);
    lpos[3 * I + 0] = lo;
    lpos[3 * I + 1] = di;
    lpos[3 * I + 2] = up;
}

// ---- CTA-wide helpers of the setup kernel (128 threads, b x b row-major matrices in shared memory)
__device__ __forceinline__ void line_load(double *dst, const double *__restrict__ vals, const int64_t pos, const int bb) {
    for (int e = threadIdx.x; e < bb; e += blockDim.x) dst[e] = pos >= 0 ? vals[(size_t)pos * bb + e] : 0.0;
}
// C = (Cin ? Cin : 0) + sgn * A B;  C may alias Cin (element-wise), never A or B
__device__ __forceinline__ void line_mm(double *C, const double *Cin, const double sgn, const double *A, const double *B, const int b) {
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        double acc = 0.0;
        for (int q = 0; q < b; ++q) acc = fma(A[r * b + q], B[q * b + c], acc);
        C[e] = (Cin != nullptr ? Cin[e] : 0.0) + sgn * acc;
    }
}
// out = M^-1 by Gauss-Jordan with partial pivoting on [M | I] in `work` (b x 2b + b doubles); false on a zero / NaN pivot
__device__ bool line_inverse(const double *M, double *out, double *work, const int b) {
    const int w2 = 2 * b;
    double *fcol = work + 2 * b * b;
    __shared__ int piv_s;
    __shared__ double pivval_s;
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        work[r * w2 + c] = M[e];
        work[r * w2 + b + c] = (r == c) ? 1.0 : 0.0;
    }
    __syncthreads();
    for (int k = 0; k < b; ++k) {
        if (threadIdx.x < 32) {
            double best = -1.0;
            int piv = k;
            for (int r = k + (int)threadIdx.x; r < b; r += 32) {
                const double v = fabs(work[r * w2 + k]);
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
        if (!(pivval_s > 0.0)) return false;   // uniform: every thread reads the same shared value
        if (piv != k)
            for (int c = threadIdx.x; c < w2; c += blockDim.x) {
                const double t = work[k * w2 + c];
                work[k * w2 + c] = work[piv * w2 + c];
                work[piv * w2 + c] = t;
            }
        __syncthreads();
        const double inv = 1.0 / work[k * w2 + k];
        __syncthreads();
        for (int c = threadIdx.x; c < w2; c += blockDim.x) work[k * w2 + c] *= inv;
        for (int r = threadIdx.x; r < b; r += blockDim.x) fcol[r] = work[r * w2 + k];
        __syncthreads();
        for (int e = threadIdx.x; e < b * w2; e += blockDim.x) {
            const int r = e / w2, c = e - r * w2;
            if (r != k) work[e] -= fcol[r] * work[k * w2 + c];
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int r = e / b, c = e - r * b;
        out[e] = work[r * w2 + b + c];
    }
    __syncthreads();
    return true;
}

// One CTA per poloidal node: factorisation of its line block (see the top of the file).  G: [n_pol][N][b*b], W: [n_pol][max(N-1,1)][b*b]
// (W also holds the Y_k of the forward sweep until the backward sweep replaces them).  Shared memory: 7 b^2 + b doubles.
__global__ void __launch_bounds__(128) line_factor_kernel(const double *__restrict__ vals, const int64_t *__restrict__ lpos,
                                                          const int n_pol, const int N, const int b, double *__restrict__ G,
                                                          double *__restrict__ W, unsigned long long *__restrict__ err) {
    extern __shared__ double lf_sm[];
    const int bb = b * b;
    double *Gs = lf_sm;            // current G_k
    double *T1 = Gs + bb;          // L_k G_{k-1}
    double *Ys = T1 + bb;          // Y_{k-1} -> Y_k, later W_{k+1}
    double *B1 = Ys + bb;          // a loaded block
    double *B2 = B1 + bb;          // another / a product
    double *work = B2 + bb;        // 2 b^2 + b
    const int i = blockIdx.x;
    const int C = N - 1;
    auto pos = [&](int k, int which) { return lpos[3 * ((int64_t)k * n_pol + i) + which]; };
    double *Gi = G + (size_t)i * N * bb;
    double *Wi = W + (size_t)i * (C > 0 ? C : 1) * bb;
    auto fail = [&]() {
        if (threadIdx.x == 0) atomicMin(err, (unsigned long long)(i + 1));
    };
    if (C == 0) {   // one plane: the point block
        line_load(B1, vals, pos(0, 1), bb);
        __syncthreads();
        if (!line_inverse(B1, Gs, work, b)) { fail(); return; }
        for (int e = threadIdx.x; e < bb; e += blockDim.x) Gi[e] = Gs[e];
        return;
    }
    // ---- forward: G_k and Y_k = u_k - L_k G_{k-1} Y_{k-1}
    line_load(B1, vals, pos(0, 1), bb);   // D_0
    __syncthreads();
    if (!line_inverse(B1, Gs, work, b)) { fail(); return; }
    {   // u_0 = lower(0) (+ upper(0) if the chain has a single plane)
        line_load(Ys, vals, pos(0, 0), bb);
        __syncthreads();
        if (C == 1) {
            line_load(B1, vals, pos(0, 2), bb);
            __syncthreads();
            for (int e = threadIdx.x; e < bb; e += blockDim.x) Ys[e] += B1[e];
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < bb; e += blockDim.x) {
        Gi[e] = Gs[e];
        Wi[e] = Ys[e];
    }
    for (int k = 1; k < C; ++k) {
        line_load(B1, vals, pos(k, 0), bb);       // L_k
        __syncthreads();
        line_mm(T1, nullptr, 1.0, B1, Gs, b);     // T1 = L_k G_{k-1}
        __syncthreads();
        line_load(B2, vals, pos(k - 1, 2), bb);   // U_{k-1}
        line_load(B1, vals, pos(k, 1), bb);       // D_k
        __syncthreads();
        line_mm(B1, B1, -1.0, T1, B2, b);         // P_k = D_k - T1 U_{k-1}  (in place: element e reads only B1[e] of B1)
        __syncthreads();
        if (!line_inverse(B1, Gs, work, b)) { fail(); return; }
        // Y_k = u_k - T1 Y_{k-1}
        line_load(B1, vals, k == C - 1 ? pos(k, 2) : (int64_t)-1, bb);   // u_k = upper(C-1) on the last chain plane, else 0
        __syncthreads();
        line_mm(B2, B1, -1.0, T1, Ys, b);
        __syncthreads();
        for (int e = threadIdx.x; e < bb; e += blockDim.x) {
            Ys[e] = B2[e];
            Gi[(size_t)k * bb + e] = Gs[e];
            Wi[(size_t)k * bb + e] = B2[e];
        }
        __syncthreads();
    }
    // ---- backward: W_{C-1} = G_{C-1} Y_{C-1};  W_k = G_k (Y_k - U_k W_{k+1})
    line_mm(B2, nullptr, 1.0, Gs, Ys, b);
    __syncthreads();
    for (int e = threadIdx.x; e < bb; e += blockDim.x) {
        Ys[e] = B2[e];   // Ys = W_{k+1}
        Wi[(size_t)(C - 1) * bb + e] = B2[e];
    }
    __syncthreads();
    // S accumulates in T1: D_{N-1} - v_{C-1} W_{C-1} - v_0 W_0,  v_{C-1} = lower(N-1), v_0 = upper(N-1)
    line_load(T1, vals, pos(N - 1, 1), bb);
    line_load(B1, vals, pos(N - 1, 0), bb);
    __syncthreads();
    line_mm(B2, T1, -1.0, B1, Ys, b);
    __syncthreads();
    for (int e = threadIdx.x; e < bb; e += blockDim.x) T1[e] = B2[e];
    __syncthreads();
    for (int k = C - 2; k >= 0; --k) {
        line_load(B1, vals, pos(k, 2), bb);   // U_k
        for (int e = threadIdx.x; e < bb; e += blockDim.x) {
            Gs[e] = Gi[(size_t)k * bb + e];
            B2[e] = Wi[(size_t)k * bb + e];   // Y_k
        }
        __syncthreads();
        line_mm(work, B2, -1.0, B1, Ys, b);   // Y_k - U_k W_{k+1}   (work's first b^2 doubles as a temporary)
        __syncthreads();
        line_mm(Ys, nullptr, 1.0, Gs, work, b);   // W_k = G_k (Y_k - U_k W_{k+1})
        __syncthreads();
        for (int e = threadIdx.x; e < bb; e += blockDim.x) Wi[(size_t)k * bb + e] = Ys[e];
        __syncthreads();
    }
    if (C > 1) {   // - v_0 W_0 with v_0 = upper(N-1); (for C == 1 the single term above used lower(N-1) = v_0)
        line_load(B1, vals, pos(N - 1, 2), bb);
        __syncthreads();
        line_mm(B2, T1, -1.0, B1, Ys, b);
        __syncthreads();
        for (int e = threadIdx.x; e < bb; e += blockDim.x) T1[e] = B2[e];
        __syncthreads();
    }
    if (!line_inverse(T1, Gs, work, b)) { fail(); return; }
    for (int e = threadIdx.x; e < bb; e += blockDim.x) Gi[(size_t)(N - 1) * bb + e] = Gs[e];
}

// ---- apply: one warp per poloidal node; lane r owns rows r and r + 32 of every b x b mat-vec (b <= 64)
struct LineArgs {
    const double *vals;      // block-CSR values of the level (L_k, U_k, u, v)
    const int64_t *lpos;
    const double *G, *W;
    const double *rin;       // r
    const double *dold;      // may be nullptr (c_d = 0)
    double *dout;            // d' = c_d dold + c_z z; also the scratch of the recurrences (dout != rin, dout != dold)
    double *x;               // if non-null: x += d'
    double c_d, c_z;
    int n_pol, N, b;
    const int *done;
};
constexpr int LINE_WARPS = 4;

// (acc0, acc1) = rows lane, lane + 32 of M v;  M global row-major b x b (nullptr: zero), v in shared memory
__device__ __forceinline__ void line_matvec(const double *__restrict__ M, const double *v, const int b, const int lane, double &a0,
                                            double &a1) {
    a0 = a1 = 0.0;
    if (M == nullptr) return;
    if ((b & 1) == 0) {
        const double2 *v2 = reinterpret_cast<const double2 *>(v);
        if (lane < b) {
            const double2 *m = reinterpret_cast<const double2 *>(M + (size_t)lane * b);
            double s0 = 0.0, s1 = 0.0;
#pragma unroll 6
            for (int c = 0; c < b / 2; ++c) {
                const double2 mv = __ldg(m + c), x = v2[c];
                s0 = fma(mv.x, x.x, s0);
                s1 = fma(mv.y, x.y, s1);
            }
            a0 = s0 + s1;
        }
        if (lane + 32 < b) {
            const double2 *m = reinterpret_cast<const double2 *>(M + (size_t)(lane + 32) * b);
            double s0 = 0.0, s1 = 0.0;
#pragma unroll 6
            for (int c = 0; c < b / 2; ++c) {
                const double2 mv = __ldg(m + c), x = v2[c];
                s0 = fma(mv.x, x.x, s0);
                s1 = fma(mv.y, x.y, s1);
            }
            a1 = s0 + s1;
        }
    } else {
        if (lane < b)
            for (int c = 0; c < b; ++c) a0 = fma(__ldg(M + (size_t)lane * b + c), v[c], a0);
        if (lane + 32 < b)
            for (int c = 0; c < b; ++c) a1 = fma(__ldg(M + (size_t)(lane + 32) * b + c), v[c], a1);
    }
}

__global__ void __launch_bounds__(LINE_WARPS * 32) line_apply_kernel(const LineArgs a) {
    if (a.done != nullptr && *a.done != 0) return;
    __shared__ __align__(16) double sv[LINE_WARPS][2][64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * LINE_WARPS + warp;
    if (i >= a.n_pol) return;
    const int b = a.b, N = a.N, C = N - 1, bb = b * b;
    double *va = sv[warp][0], *vb = sv[warp][1];
    const double *Gi = a.G + (size_t)i * N * bb;
    const double *Wi = a.W + (size_t)i * (C > 0 ? C : 1) * bb;
    auto blk = [&](int k, int which) -> const double * {
        const int64_t p = a.lpos[3 * ((int64_t)k * a.n_pol + i) + which];
        return p >= 0 ? a.vals + (size_t)p * bb : nullptr;
    };
    auto idx = [&](int k, int r) { return ((size_t)k * a.n_pol + i) * b + r; };
    const bool r0ok = lane < b, r1ok = lane + 32 < b;
    double *z = a.dout;   // scratch: q_k, then x_k, then the final values
    double t0, t1, s0, s1;
    if (C > 0) {
        // ---- forward: y_0 = r_0, q_k = G_k y_k, y_k = r_k - L_k q_{k-1}
        if (r0ok) va[lane] = a.rin[idx(0, lane)];
        if (r1ok) va[lane + 32] = a.rin[idx(0, lane + 32)];
        __syncwarp();
        for (int k = 0; k < C; ++k) {
            if (k > 0) {
                line_matvec(blk(k, 0), vb, b, lane, t0, t1);   // L_k q_{k-1}   (vb = q_{k-1})
                __syncwarp();
                if (r0ok) va[lane] = a.rin[idx(k, lane)] - t0;
                if (r1ok) va[lane + 32] = a.rin[idx(k, lane + 32)] - t1;
                __syncwarp();
            }
            line_matvec(Gi + (size_t)k * bb, va, b, lane, s0, s1);   // q_k
            __syncwarp();
            if (r0ok) { vb[lane] = s0; z[idx(k, lane)] = s0; }
            if (r1ok) { vb[lane + 32] = s1; z[idx(k, lane + 32)] = s1; }
            __syncwarp();
        }
        // ---- backward: x_{C-1} = q_{C-1} (in vb); x_k = q_k - G_k (U_k x_{k+1})
        for (int k = C - 2; k >= 0; --k) {
            line_matvec(blk(k, 2), vb, b, lane, t0, t1);   // U_k x_{k+1}
            __syncwarp();
            if (r0ok) va[lane] = t0;
            if (r1ok) va[lane + 32] = t1;
            __syncwarp();
            line_matvec(Gi + (size_t)k * bb, va, b, lane, s0, s1);
            __syncwarp();
            if (r0ok) { const double xv = z[idx(k, lane)] - s0; vb[lane] = xv; z[idx(k, lane)] = xv; }
            if (r1ok) { const double xv = z[idx(k, lane + 32)] - s1; vb[lane + 32] = xv; z[idx(k, lane + 32)] = xv; }
            __syncwarp();
        }
        // ---- border: z_{N-1} = S^-1 (r_{N-1} - v_0 x_0 - v_{C-1} x_{C-1});  vb = x_0
        double c0, c1;
        if (C == 1) {   // v_0 = upper(N-1) + lower(N-1), one of them absent
            line_matvec(blk(N - 1, 0), vb, b, lane, t0, t1);
            line_matvec(blk(N - 1, 2), vb, b, lane, c0, c1);
            t0 += c0;
            t1 += c1;
        } else {
            line_matvec(blk(N - 1, 2), vb, b, lane, t0, t1);          // upper(N-1) x_0
            __syncwarp();
            if (r0ok) va[lane] = z[idx(C - 1, lane)];                  // x_{C-1}: written by this very lane
            if (r1ok) va[lane + 32] = z[idx(C - 1, lane + 32)];
            __syncwarp();
            line_matvec(blk(N - 1, 0), va, b, lane, c0, c1);          // lower(N-1) x_{C-1}
            t0 += c0;
            t1 += c1;
        }
        __syncwarp();
        if (r0ok) va[lane] = a.rin[idx(N - 1, lane)] - t0;
        if (r1ok) va[lane + 32] = a.rin[idx(N - 1, lane + 32)] - t1;
        __syncwarp();
    } else {
        if (r0ok) va[lane] = a.rin[idx(0, lane)];
        if (r1ok) va[lane + 32] = a.rin[idx(0, lane + 32)];
        __syncwarp();
    }
    line_matvec(Gi + (size_t)(N - 1) * bb, va, b, lane, s0, s1);   // z_{N-1}
    __syncwarp();
    if (r0ok) vb[lane] = s0;
    if (r1ok) vb[lane + 32] = s1;
    __syncwarp();
    // ---- final values and the Chebyshev update d' = c_d d + c_z z  (x += d')
    auto emit = [&](int k, int r, double zv) {
        const size_t g = idx(k, r);
        double dn = a.c_z * zv;
        if (a.dold != nullptr && a.c_d != 0.0) dn = fma(a.c_d, a.dold[g], dn);
        a.dout[g] = dn;
        if (a.x != nullptr) a.x[g] += dn;
    };
    if (r0ok) emit(N - 1, lane, s0);
    if (r1ok) emit(N - 1, lane + 32, s1);
    for (int k = 0; k < C; ++k) {
        line_matvec(Wi + (size_t)k * bb, vb, b, lane, t0, t1);   // W_k z_{N-1}
        if (r0ok) emit(k, lane, z[idx(k, lane)] - t0);
        if (r1ok) emit(k, lane + 32, z[idx(k, lane + 32)] - t1);
    }
}

}  // namespace mgk
