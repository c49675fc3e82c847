// kernels_vec.cuh -- streaming vector kernels of the solve path: toroidal restriction / prolongation
// (stencil [1/2 1 1/2], 2:1, periodic), the orthogonalisation reductions of (F)GMRES
// (batched dots with warp-shuffle reductions, batched axpys) and the device-resident Givens/Hessenberg
// bookkeeping that lets a whole GMRES restart cycle run without a host round trip.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

#define MG_EARLY_EXIT(done) \
    if ((done) != nullptr && *(done) != 0) return

// ------------------------------------------------------------------------------------------------ transfer
// r_c[K] = r[2K] + (r[2K-1] + r[2K+1]) / 2, plane indices periodic.  For n_f = 2 both halves hit plane 1 and add
// up to weight 1, which is P_phi = [1; 1] (the "+=" reading, Q8).  plane = n_pol*b doubles.
__global__ void __launch_bounds__(256) restrict_kernel(const double *__restrict__ rf, double *__restrict__ rc,
                                                       const int64_t plane, const int n_f, const int *done) {
    MG_EARLY_EXIT(done);
    const int n_c = n_f / 2;
    const int64_t total = plane * n_c;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t K = e / plane, off = e - K * plane;
        const int64_t km = (2 * K - 1 + n_f) % n_f, kp = (2 * K + 1) % n_f;
        rc[e] = rf[2 * K * plane + off] + 0.5 * (rf[km * plane + off] + rf[kp * plane + off]);
    }
}

// x[2K] += e[K]; x[2K+1] += (e[K] + e[(K+1) mod n_c]) / 2; pe (optional) receives the prolonged correction P e.
__global__ void __launch_bounds__(256) prolong_add_kernel(const double *__restrict__ ec, double *__restrict__ xf,
                                                          double *__restrict__ pe, const int64_t plane, const int n_f,
                                                          const int *done) {
    MG_EARLY_EXIT(done);
    const int n_c = n_f / 2;
    const int64_t total = plane * n_f;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t k = e / plane, off = e - k * plane;
        const int64_t K = k >> 1;
        double v;
        if ((k & 1) == 0) v = ec[K * plane + off];
        else v = 0.5 * (ec[K * plane + off] + ec[((K + 1) % n_c) * plane + off]);
        xf[e] += v;
        if (pe != nullptr) pe[e] = v;
    }
}

// ------------------------------------------------------------------------------------------------ reductions
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum_256(double v, double *sh /* >= 8 doubles */) {
    v = warp_sum(v);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double t = (threadIdx.x < 8) ? sh[threadIdx.x] : 0.0;
    if (warp == 0) {
        t += __shfl_xor_sync(0xffffffffu, t, 4);
        t += __shfl_xor_sync(0xffffffffu, t, 2);
        t += __shfl_xor_sync(0xffffffffu, t, 1);
    }
    return t;  // valid in warp 0
}

// h[i] = <V_i, w>, i = 0..k-1 (gridDim.y = k; *kdev, if given, is the live count and rows >= it are skipped);
// V_i = V + i*stride.  Deterministic: per-CTA partials, the last CTA of row i (ticket counter) adds them in a
// fixed order.  partial: [k][gridDim.x]; counter: [k] zero-initialised, self-resetting.
__global__ void __launch_bounds__(256) dot_multi_kernel(const double *__restrict__ V, const int64_t stride,
                                                        const double *__restrict__ w, const int64_t n,
                                                        double *__restrict__ partial, unsigned *__restrict__ counter,
                                                        double *__restrict__ h, const int *done) {
    MG_EARLY_EXIT(done);
    __shared__ double sh[8];
    __shared__ bool last;
    const int i = blockIdx.y;
    const double *v = V + (size_t)i * stride;
    double acc = 0.0;
    const int64_t n2 = n >> 1;
    const double2 *v2 = reinterpret_cast<const double2 *>(v), *w2 = reinterpret_cast<const double2 *>(w);
    for (int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x; e < n2; e += (int64_t)gridDim.x * 256) {
        const double2 a = v2[e], b = w2[e];
        acc = fma(a.x, b.x, acc);
        acc = fma(a.y, b.y, acc);
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) acc = fma(v[n - 1], w[n - 1], acc);
    const double s = block_sum_256(acc, sh);
    if (threadIdx.x == 0) {
        partial[(size_t)i * gridDim.x + blockIdx.x] = s;
        __threadfence();
        const unsigned t = atomicAdd(counter + i, 1u);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (last) {
        __threadfence();
        double a2 = 0.0;
        for (int cidx = threadIdx.x; cidx < (int)gridDim.x; cidx += 256)
            a2 += *((volatile double *)(partial + (size_t)i * gridDim.x + cidx));
        const double tot = block_sum_256(a2, sh);
        if (threadIdx.x == 0) {
            h[i] = tot;
            counter[i] = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------ GMRES state
// Device-resident Arnoldi / Givens bookkeeping (one thread): nothing of a restart cycle needs the host.
struct GmresDev {
    double *H;     // (m+1) x m, column-major, leading dimension m+1 (upper triangular after rotations)
    double *cs, *sn, *g, *y;
    double *h1, *h2;   // the two classical Gram-Schmidt passes of the current column
    double *nrm2;      // ||w||^2 after orthogonalisation / ||r||^2 at cycle begin / ||rhs||^2
    double *hnext;     // h_{j+1,j} (or beta): divisor for the next basis vector
    double *tol;       // absolute tolerance rtol*||rhs||
    double *hist;      // hist[it] = residual estimate (absolute), it = 0..maxit
    int *status;       // [0] done, [1] j_used, [2] it, [3] converged
    int m, maxit;
};

// Column j: h = h1 + h2, h_{j+1,j} = ||w||, previous rotations, new rotation, residual estimate, stop test.
// One thread.  Runs at the tail of the second Gram-Schmidt update (axpy_multi_kernel, last CTA).
__device__ __forceinline__ void gmres_update_dev(const GmresDev &s, const int j) {
    if (s.status[0] != 0) return;
    double *col = s.H + (size_t)j * (s.m + 1);
    for (int i = 0; i <= j; ++i) col[i] = s.h1[i] + s.h2[i];
    const double hn = sqrt(fmax(*s.nrm2, 0.0));
    col[j + 1] = hn;
    *s.hnext = hn;
    for (int i = 0; i < j; ++i) {
        const double t = s.cs[i] * col[i] + s.sn[i] * col[i + 1];
        col[i + 1] = -s.sn[i] * col[i] + s.cs[i] * col[i + 1];
        col[i] = t;
    }
    const double denom = hypot(col[j], col[j + 1]);
    s.cs[j] = col[j] / denom;
    s.sn[j] = col[j + 1] / denom;
    col[j] = denom;
    col[j + 1] = 0.0;
    s.g[j + 1] = -s.sn[j] * s.g[j];
    s.g[j] = s.cs[j] * s.g[j];
    const int it = s.status[2] + 1;
    s.status[2] = it;
    s.status[1] = j + 1;
    const double est = fabs(s.g[j + 1]);
    s.hist[it] = est;
    const bool breakdown = (hn == 0.0);
    if (est <= *s.tol || breakdown) { s.status[0] = 1; s.status[3] = 1; }
    else if (it >= s.maxit) { s.status[0] = 1; }
}

// w += sign * sum_{i<k} coef[i] V_i ; optionally nrm2 = <w, w> of the result (same deterministic scheme).
// If kdev != nullptr the live count is min(k, *kdev).
__global__ void __launch_bounds__(256) axpy_multi_kernel(const double *__restrict__ V, const int64_t stride, const int k,
                                                         const int *__restrict__ kdev, const double *__restrict__ coef,
                                                         const double sign, double *__restrict__ w, const int64_t n,
                                                         double *__restrict__ partial, unsigned *__restrict__ counter,
                                                         double *__restrict__ nrm2, const int *done, const GmresDev upd,
                                                         const int upd_j /* >= 0: Hessenberg/Givens update of column j */) {
    MG_EARLY_EXIT(done);
    __shared__ double cf[128];
    __shared__ double sh[8];
    __shared__ bool last;
    int kk = k;
    if (kdev != nullptr) kk = min(kk, *kdev);
    const int64_t n2 = n >> 1;
    const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;  // one double2 per thread
    double2 acc = make_double2(0.0, 0.0);
    double tail = 0.0;
    const bool has = e < n2;
    const bool has_tail = (n & 1) && blockIdx.x == 0 && threadIdx.x == 0;
    for (int i0 = 0; i0 < kk; i0 += 128) {
        const int cnt = min(128, kk - i0);
        __syncthreads();
        if (threadIdx.x < cnt) cf[threadIdx.x] = coef[i0 + threadIdx.x];
        __syncthreads();
        if (has) {
            const double2 *v2 = reinterpret_cast<const double2 *>(V + (size_t)i0 * stride) + e;
#pragma unroll 4
            for (int i = 0; i < cnt; ++i) {
                const double2 a = *reinterpret_cast<const double2 *>(reinterpret_cast<const double *>(v2) + (size_t)i * stride);
                acc.x = fma(cf[i], a.x, acc.x);
                acc.y = fma(cf[i], a.y, acc.y);
            }
        }
        if (has_tail)
            for (int i = 0; i < cnt; ++i) tail = fma(cf[i], V[(size_t)(i0 + i) * stride + n - 1], tail);
    }
    double sq = 0.0;
    if (has) {
        double2 *w2 = reinterpret_cast<double2 *>(w) + e;
        double2 o = *w2;
        o.x = fma(sign, acc.x, o.x);
        o.y = fma(sign, acc.y, o.y);
        *w2 = o;
        sq = fma(o.x, o.x, o.y * o.y);
    }
    if (has_tail) {
        const double o = fma(sign, tail, w[n - 1]);
        w[n - 1] = o;
        sq = fma(o, o, sq);
    }
    if (nrm2 == nullptr) return;
    const double s = block_sum_256(sq, sh);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = s;
        __threadfence();
        const unsigned t = atomicAdd(counter, 1u);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (last) {
        __threadfence();
        double a2 = 0.0;
        for (int cidx = threadIdx.x; cidx < (int)gridDim.x; cidx += 256) a2 += *((volatile double *)(partial + cidx));
        const double tot = block_sum_256(a2, sh);
        if (threadIdx.x == 0) {
            *nrm2 = tot;
            *counter = 0;
            if (upd_j >= 0) gmres_update_dev(upd, upd_j);
        }
    }
}

// dst = src / *denom   (v_{j+1} = w / h_{j+1,j}); dst may equal src.
__global__ void __launch_bounds__(256) scale_div_kernel(const double *src, double *dst, const int64_t n,
                                                        const double *__restrict__ denom, const int *done) {
    MG_EARLY_EXIT(done);
    const double inv = 1.0 / *denom;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x)
        dst[e] = src[e] * inv;
}

// y = a*x + b*y
__global__ void __launch_bounds__(256) axpby_kernel(const double a, const double *__restrict__ x, const double bcoef,
                                                    double *__restrict__ y, const int64_t n) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x)
        y[e] = (bcoef == 0.0) ? a * x[e] : fma(a, x[e], bcoef * y[e]);
}

// v0[g] = ((g * 2654435761) mod 2^32) / 2^32 - 1/2: the bit-reproducible power-iteration start vector.
__global__ void __launch_bounds__(256) hashed_start_kernel(double *__restrict__ v, const int64_t n) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t hsh = ((uint64_t)e * 2654435761ull) & 0xffffffffull;
        v[e] = (double)hsh / 4294967296.0 - 0.5;
    }
}

__global__ void gmres_set_tol_kernel(GmresDev s, const double rtol) {
    *s.tol = rtol * sqrt(fmax(*s.nrm2, 0.0));
    s.status[0] = 0; s.status[1] = 0; s.status[2] = 0; s.status[3] = 0;
}

// Cycle begin: beta = ||r||; converged if beta <= tol; g = beta e_1.
__global__ void gmres_begin_kernel(GmresDev s) {
    s.status[1] = 0;
    if (s.status[0] != 0) return;
    const double beta = sqrt(fmax(*s.nrm2, 0.0));
    if (s.status[2] == 0) s.hist[0] = beta;
    if (beta <= *s.tol) { s.status[0] = 1; s.status[3] = 1; return; }
    if (s.status[2] >= s.maxit) { s.status[0] = 1; return; }
    s.g[0] = beta;
    *s.hnext = beta;
}

// Back substitution H y = g over the j_used columns of this cycle.
__global__ void gmres_solve_y_kernel(GmresDev s) {
    const int ju = s.status[1];
    for (int i = ju - 1; i >= 0; --i) {
        double t = s.g[i];
        for (int l = i + 1; l < ju; ++l) t -= s.H[(size_t)l * (s.m + 1) + i] * s.y[l];
        s.y[i] = t / s.H[(size_t)i * (s.m + 1) + i];
    }
}

}  // namespace mgk
