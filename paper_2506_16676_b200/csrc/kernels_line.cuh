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


// ================================================================================================ staged apply (b % 4 == 0)
// The same recurrences as line_apply_kernel, as a list of 5 (N - 1) mat-vec OPERATIONS per node executed by one CTA:
// thread t owns the b/4-element segment t % 4 of row t / 4 of every block (the mapping of the b = 36 TMA kernel: the four
// partial sums of a row meet by two shuffles).  The blocks an apply reads are STATIC, so thread 0 walks the operation list
// ahead of the arithmetic with 1-D bulk async copies (TMA engine, SASS UBLKCP) into a small ring of LS_STAGES block buffers: the
// block of an operation is in shared memory before the operation starts, and every global read of a block is one coalesced
// copy.  (line_apply_kernel walks the same ~5N dependent mat-vecs with per-lane row reads: 32 different lines per load
// instruction, 2.5 TB/s on C1's level 0.)
#ifndef MG_LS_STAGES
#define MG_LS_STAGES 2   /* measured on C1 level 0: 2 stages 249 us, 3: 285, 4: 293, 6: 325 (more CTAs per SM beat a deeper ring) */
#endif
constexpr int LS_STAGES = MG_LS_STAGES;
enum { LA_Q = 0, LA_Y, LA_T, LA_X, LA_B1, LA_B2, LA_ZN, LA_W };           // what the writer lanes do with the result t
enum { LV_Y = 0, LV_Q, LV_X, LV_T, LV_Y2, LV_ZN, LV_COUNT };               // vectors in shared memory (64 doubles each)
struct LineOp {
    const double *M;   // b x b block (nullptr: absent, t = 0)
    short src, act;    // source vector, action
    int k;             // plane the action refers to
};
inline size_t line_staged_smem(int b, int N) {
    const int nops = 5 * (N > 1 ? N - 1 : 0) + 1;
    return sizeof(double) * ((size_t)LS_STAGES * b * b + LV_COUNT * 64) + sizeof(LineOp) * (size_t)nops + sizeof(uint64_t) * LS_STAGES + 64;
}
__device__ __forceinline__ uint32_t ls_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ls_issue(double *dst, const double *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ls_smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(ls_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(ls_smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void ls_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(ls_smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}

// One CTA of 4 b threads per poloidal node.  Dynamic shared memory: line_staged_smem(b, N).
__global__ void line_apply_staged_kernel(const LineArgs a) {
    if (a.done != nullptr && *a.done != 0) return;
    extern __shared__ __align__(128) unsigned char ls_raw[];
    const int b = a.b, N = a.N, C = N - 1, bb = b * b, i = blockIdx.x, tid = threadIdx.x;
    double *ring = reinterpret_cast<double *>(ls_raw);
    double *vecs = ring + (size_t)LS_STAGES * bb;
    LineOp *ops = reinterpret_cast<LineOp *>(vecs + LV_COUNT * 64);
    const int nops = C > 0 ? 5 * C : 1;
    uint64_t *full = reinterpret_cast<uint64_t *>(ops + nops);
    const double *Gi = a.G + (size_t)i * N * bb;
    const double *Wi = a.W + (size_t)i * (C > 0 ? C : 1) * bb;
    auto blk = [&](int k, int which) -> const double * {
        const int64_t p = a.lpos[3 * ((int64_t)k * a.n_pol + i) + which];
        return p >= 0 ? a.vals + (size_t)p * bb : nullptr;
    };
    auto idx = [&](int k, int r) { return ((size_t)k * a.n_pol + i) * b + r; };
    // ---- the operation list (closed form; see the top of the file)
    for (int j = tid; j < nops; j += blockDim.x) {
        LineOp o;
        o.M = nullptr; o.src = LV_Y; o.act = LA_ZN; o.k = N - 1;
        if (C == 0) {
            o.M = Gi;                                                     // S^-1 = D_0^-1
        } else if (j < 2 * C - 1) {                                       // forward: G_0 | L_k, G_k
            const int k = (j + 1) / 2;
            if ((j & 1) == 0) { o.M = Gi + (size_t)k * bb; o.src = LV_Y; o.act = LA_Q; o.k = k; }
            else { o.M = blk(k, 0); o.src = LV_Q; o.act = LA_Y; o.k = k; }
        } else if (j < 4 * C - 3) {                                       // backward: U_k, G_k for k = C-2 .. 0
            const int m = j - (2 * C - 1), k = C - 2 - m / 2;
            if ((m & 1) == 0) { o.M = blk(k, 2); o.src = LV_X; o.act = LA_T; o.k = k; }
            else { o.M = Gi + (size_t)k * bb; o.src = LV_T; o.act = LA_X; o.k = k; }
        } else if (j < 4 * C) {                                           // border
            const int m = j - (4 * C - 3);
            if (m == 0) { o.M = blk(N - 1, 2); o.src = LV_X; o.act = LA_B1; }
            else if (m == 1) { o.M = blk(N - 1, 0); o.src = LV_Y2; o.act = LA_B2; }
            else { o.M = Gi + (size_t)(N - 1) * bb; o.src = LV_Y; o.act = LA_ZN; }
        } else {                                                          // z_k = x_k - W_k z_{N-1}
            const int k = j - 4 * C;
            o.M = Wi + (size_t)k * bb; o.src = LV_ZN; o.act = LA_W; o.k = k;
        }
        ops[j] = o;
    }
    if (tid == 0) {
        for (int s = 0; s < LS_STAGES; ++s)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ls_smem_u32(&full[s])) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int r = tid >> 2, h = tid & 3, seg = b >> 2;
    const bool active = r < b, writer = active && h == 0;
    if (writer) vecs[LV_Y * 64 + r] = a.rin[idx(0, r)];                   // y_0 = r_0 (N = 1: the only right-hand side)
    __syncthreads();
    // ---- thread 0 keeps LS_STAGES block copies in flight, in list order (absent blocks take no stage)
    int issue = 0, issued = 0;                                            // next list entry to look at / copies issued (thread 0)
    auto issue_next = [&]() {
        while (issue < nops && ops[issue].M == nullptr) ++issue;
        if (issue < nops) {
            ls_issue(ring + (size_t)(issued % LS_STAGES) * bb, ops[issue].M, (uint32_t)(bb * sizeof(double)), &full[issued % LS_STAGES]);
            ++issue;
            ++issued;
        }
    };
    if (tid == 0)
        for (int s = 0; s < LS_STAGES; ++s) issue_next();
    double *z = a.dout;
    int seq = 0;                                                          // copies consumed so far (every thread)
    for (int j = 0; j < nops; ++j) {
        const LineOp o = ops[j];
        // values the action needs from global memory: asked for before the block is waited for
        double g0 = 0.0;
        if (writer) {
            if (o.act == LA_Y) g0 = a.rin[idx(o.k, r)];
            else if (o.act == LA_X || o.act == LA_W) g0 = z[idx(o.k, r)];
            else if (o.act == LA_B2) g0 = a.rin[idx(N - 1, r)];
            else if (o.act == LA_B1 && C > 1) g0 = z[idx(C - 1, r)];
        }
        double t = 0.0;
        if (o.M != nullptr) {
            ls_wait(&full[seq % LS_STAGES], (uint32_t)(seq / LS_STAGES) & 1u);
            if (active) {
                const double *Mrow = ring + (size_t)(seq % LS_STAGES) * bb + (size_t)r * b + h * seg;
                const double *v = vecs + o.src * 64 + h * seg;
                double t0 = 0.0, t1 = 0.0;
                int cidx = 0;
                for (; cidx + 1 < seg; cidx += 2) {
                    t0 = fma(Mrow[cidx], v[cidx], t0);
                    t1 = fma(Mrow[cidx + 1], v[cidx + 1], t1);
                }
                if (cidx < seg) t0 = fma(Mrow[cidx], v[cidx], t0);
                t = t0 + t1;
            }
            t += __shfl_xor_sync(0xffffffffu, t, 1);
            t += __shfl_xor_sync(0xffffffffu, t, 2);
            ++seq;
        }
        if (writer) {
            double *V = vecs;
            switch (o.act) {
                case LA_Q: V[LV_Q * 64 + r] = t; V[LV_X * 64 + r] = t; z[idx(o.k, r)] = t; break;
                case LA_Y: V[LV_Y * 64 + r] = g0 - t; break;
                case LA_T: V[LV_T * 64 + r] = t; break;
                case LA_X: { const double xv = g0 - t; V[LV_X * 64 + r] = xv; z[idx(o.k, r)] = xv; } break;
                case LA_B1: V[LV_T * 64 + r] = t; V[LV_Y2 * 64 + r] = C > 1 ? g0 : V[LV_X * 64 + r]; break;
                case LA_B2: V[LV_Y * 64 + r] = g0 - V[LV_T * 64 + r] - t; break;
                default: {   // LA_ZN, LA_W: final values and the Chebyshev update d' = c_d d + c_z z (x += d')
                    const double zv = o.act == LA_ZN ? t : g0 - t;
                    if (o.act == LA_ZN) V[LV_ZN * 64 + r] = t;
                    const size_t g = idx(o.k, r);
                    double dn = a.c_z * zv;
                    if (a.dold != nullptr && a.c_d != 0.0) dn = fma(a.c_d, a.dold[g], dn);
                    a.dout[g] = dn;
                    if (a.x != nullptr) a.x[g] += dn;
                }
            }
        }
        __syncthreads();   // the action's vectors are visible; the block's stage is free
        if (tid == 0 && o.M != nullptr) issue_next();
    }
}

}  // namespace mgk
