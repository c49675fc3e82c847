// kernels_vec.cuh -- streaming vector kernels of the solve path: toroidal restriction / prolongation
// (stencil [1/2 1 1/2], 2:1, periodic), the orthogonalisation reductions of (F)GMRES
// (batched dots with warp-shuffle reductions, batched axpys) and the device-resident Givens/Hessenberg
// bookkeeping that lets a whole GMRES restart cycle run without a host round trip.
#pragma once
#include <cooperative_groups.h>
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
    int *status;       // [0] done, [1] j_used, [2] it, [3] converged, [4] done as the latest Gram-Schmidt kernel saw it (the flag a
                       //     SpMV running BESIDE the deferred Givens update reads: nothing writes it while that SpMV runs)
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

// The same update by ONE WARP with three scratch arrays of j + 2 doubles in shared memory: the column, the rotations and the
// coefficients are fetched with coalesced independent loads and the rotation recurrence runs out of shared memory.  (The
// one-thread version above walks ~4 j dependent global loads: ~13 us at j = 50, a third of the whole Gram-Schmidt kernel.)
// Same arithmetic in the same order, so the results are bit-identical.
__device__ __forceinline__ void gmres_update_warp(const GmresDev &s, const int j, const int lane, double *sc, double *scs, double *ssn,
                                                  const bool write_hnext = true) {
    if (s.status[0] != 0) return;   // (uniform: every lane reads the same value)
    for (int i = lane; i <= j; i += 32) {
        sc[i] = __ldcg(s.h1 + i) + __ldcg(s.h2 + i);
        if (i < j) {
            scs[i] = __ldcg(s.cs + i);
            ssn[i] = __ldcg(s.sn + i);
        }
    }
    __syncwarp();
    if (lane == 0) {
        const double hn = sqrt(fmax(*s.nrm2, 0.0));
        sc[j + 1] = hn;
        if (write_hnext) *s.hnext = hn;
        for (int i = 0; i < j; ++i) {
            const double t = scs[i] * sc[i] + ssn[i] * sc[i + 1];
            sc[i + 1] = -ssn[i] * sc[i] + scs[i] * sc[i + 1];
            sc[i] = t;
        }
        const double denom = hypot(sc[j], sc[j + 1]);
        const double csj = sc[j] / denom, snj = sc[j + 1] / denom;
        s.cs[j] = csj;
        s.sn[j] = snj;
        sc[j] = denom;
        sc[j + 1] = 0.0;
        const double gj = s.g[j];
        s.g[j + 1] = -snj * gj;
        s.g[j] = csj * gj;
        const int it = s.status[2] + 1;
        s.status[2] = it;
        s.status[1] = j + 1;
        const double est = fabs(snj * gj);
        s.hist[it] = est;
        const bool breakdown = (hn == 0.0);
        if (est <= *s.tol || breakdown) { s.status[0] = 1; s.status[3] = 1; }
        else if (it >= s.maxit) { s.status[0] = 1; }
    }
    __syncwarp();
    double *col = s.H + (size_t)j * (s.m + 1);
    for (int i = lane; i <= j + 1; i += 32) col[i] = sc[i];
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

// ------------------------------------------------------------------------------------------------ fused CGS2
// One cooperative launch per Arnoldi step instead of four kernels: both classical Gram-Schmidt passes, the norm of
// the result and the Hessenberg/Givens update.  CTA c owns the slice [c*slice, (c+1)*slice) of the vectors: it
// keeps its slice of w in shared memory for the whole step and caches the slices of the first `cap` basis vectors
// there while it reads them for the first dots, so that the first update, the second dots and the second update
// run out of shared memory (the remaining vectors are re-read through L2).  The two global reductions (h1, h2)
// are grid-wide barriers; every CTA then sums the per-CTA partials itself, in a fixed order (deterministic).
struct OrthArgs {
    const double *V;
    int64_t stride;
    int j;                 // orthogonalise against V_0..V_j
    double *w;             // V_{j+1}, updated in place
    int64_t n;
    double *partial;       // [ORTH_REPLICAS][gridDim.x][ld]: every CTA reads all partials after the barrier; replicas at
                           // different addresses spread that hot spot over more L2 slices (CTA c reads replica c % R)
    double *nrm_partial;   // [gridDim.x]
    unsigned *counter;     // ticket of the final norm, zero-initialised, self-resetting
    GmresDev dev;
    const int *done;
    int slice;             // elements per CTA, even
    int cap;               // basis vectors cached in shared memory
    int ld;                // >= m + 1
    int defer_update;      // 1: the last CTA writes ||w||^2 and h_{j+1,j} only; the Hessenberg / Givens / stop-test update of
                           // column j runs in gmres_givens_kernel, beside the next SpMV (coarsest-level cycle)
    double eta2;           // selective reorthogonalisation (Daniel-Gragg-Kaufman-Stewart): the second pass is skipped
                           // when ||w - V h1||^2 >= eta2 ||w||^2, estimated as ||w||^2 - |h1|^2; 0 = always two passes
};
#ifdef MG_ORTH_STAMPS   // development probe (compiled out in the library): per-phase global-timer stamps of CTA 0, by step j
__device__ unsigned long long orth_stamps[16 * 256];
#define MG_ORTH_STAMP(k) \
    if (blockIdx.x == 0 && threadIdx.x == 0 && a.j < 256) { \
        unsigned long long t__; \
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t__)); \
        orth_stamps[a.j * 16 + (k)] = t__; \
    }
#else
#define MG_ORTH_STAMP(k)
#endif
constexpr int ORTH_THREADS = 512;
constexpr int ORTH_REPLICAS = 8;
constexpr int ORTH_MAX_GRID = 152;          // 8 * 19: the cross-CTA reduction unrolls over 19 loads per thread
constexpr int ORTH_SCRATCH = 8 * 64 + 32;   // doubles of reduction scratch (+ 2*ld for the half-slice dots)
inline size_t orth_smem_bytes(int slice, int ld, int cap) {
    return sizeof(double) * ((size_t)slice + 3 * (size_t)ld + ORTH_SCRATCH + (size_t)cap * slice);
}

// <src_slice, ws> over the double2 range [start, end), 8 independent 128-bit loads in flight per lane;
// optionally copies the source into the shared-memory cache on the way.
__device__ __forceinline__ double orth_dot_range(const double2 *__restrict__ src2, const double2 *__restrict__ ws2,
                                                 double2 *cache2, const int start, const int end, const int lane) {
    double acc0 = 0.0, acc1 = 0.0;
    for (int k0 = start + lane; k0 < end; k0 += 32 * 8) {
        double2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int e = k0 + 32 * u;
            v[u] = (e < end) ? src2[e] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int e = k0 + 32 * u;
            if (e < end) {
                if (cache2 != nullptr) cache2[e] = v[u];
                const double2 wv = ws2[e];
                acc0 = fma(v[u].x, wv.x, acc0);
                acc1 = fma(v[u].y, wv.y, acc1);
            }
        }
    }
    return acc0 + acc1;
}

__global__ void __launch_bounds__(ORTH_THREADS, 1) gmres_orth_fused_kernel(const OrthArgs a) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    if (a.done != nullptr && *a.done != 0) {   // written by an earlier kernel: every CTA takes the same branch
        if (a.defer_update && blockIdx.x == 0 && threadIdx.x == 0) a.dev.status[4] = 1;
        return;
    }
    extern __shared__ __align__(16) double orth_sm[];
    double *ws = orth_sm;                 // [slice]   this CTA's slice of w
    double *hs = ws + a.slice;            // [ld]      coefficients of the current pass
    double *hd = hs + a.ld;               // [2 * ld]  half-slice dot products
    double *red = hd + 2 * a.ld;          // [ORTH_SCRATCH]
    double *vc = red + ORTH_SCRATCH;      // [cap][slice] cached slices of V_0..V_{cap-1}
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = ORTH_THREADS / 32;
    const int G = gridDim.x;
    const int64_t e0 = (int64_t)blockIdx.x * a.slice;
    int len = 0;
    if (e0 < a.n) len = (int)((a.n - e0 < (int64_t)a.slice) ? (a.n - e0) : (int64_t)a.slice);
    const int len2 = len >> 1;            // 128-bit part; an odd last element (odd n only) is handled by one lane
    const int half2 = (len2 + 1) >> 1;
    const bool odd = (len & 1) != 0;
    const int slice2 = a.slice >> 1;
    const double2 *ws2 = reinterpret_cast<const double2 *>(ws);
    MG_ORTH_STAMP(0);
    for (int e = tid; e < len; e += ORTH_THREADS) ws[e] = a.w[e0 + e];
    __syncthreads();
    MG_ORTH_STAMP(1);
    const int nvec = a.j + 1;
    const int nc = nvec < a.cap ? nvec : a.cap;
    for (int pass = 0; pass < 2; ++pass) {
        // ---- dots of the slice with V_0..V_j: work item = (vector, half of the slice), one warp per item
        for (int item = warp; item < 2 * nvec; item += NW) {
            const int i = item >> 1, hf = item & 1;
            const bool cached = i < a.cap;
            const int start = hf * half2, end = (hf == 0) ? (half2 < len2 ? half2 : len2) : len2;
            const double *vg = a.V + (size_t)i * a.stride + e0;
            double *vs = vc + (size_t)(cached ? i : 0) * a.slice;
            const bool from_smem = (pass == 1 && cached);
            double s = orth_dot_range(reinterpret_cast<const double2 *>(from_smem ? vs : vg), ws2,
                                      (pass == 0 && cached) ? reinterpret_cast<double2 *>(vs) : nullptr, start, end, lane);
            if (odd && hf == 1 && lane == 0) {
                const double v = from_smem ? vs[len - 1] : vg[len - 1];
                if (pass == 0 && cached) vs[len - 1] = v;
                s = fma(v, ws[len - 1], s);
            }
            s = warp_sum(s);
            if (lane == 0) hd[item] = s;
        }
        // pass 0 also reduces <w, w> (entry nvec): it decides whether a second pass is needed
        const int nred = nvec + ((pass == 0 && a.eta2 > 0.0) ? 1 : 0);
        if (nred > nvec) {
            double sq = 0.0;
            for (int e = tid; e < len; e += ORTH_THREADS) sq = fma(ws[e], ws[e], sq);
            sq = warp_sum(sq);
            if (lane == 0) red[warp] = sq;
        }
        __syncthreads();
        const size_t rep_stride = (size_t)G * a.ld;
        if (nred > nvec && tid == 0) {
            double t = 0.0;
            for (int k = 0; k < NW; ++k) t += red[k];
            hd[2 * nvec] = t;
            hd[2 * nvec + 1] = 0.0;
        }
        __syncthreads();
        for (int i = tid; i < nred * ORTH_REPLICAS; i += ORTH_THREADS) {
            const int rep = i / nred, ii = i - rep * nred;
            a.partial[rep * rep_stride + (size_t)blockIdx.x * a.ld + ii] = hd[2 * ii] + hd[2 * ii + 1];
        }
        MG_ORTH_STAMP(2 + 4 * pass);
        grid.sync();
        MG_ORTH_STAMP(3 + 4 * pass);
        // ---- h_i = sum over CTAs: 8 interleaved sub-ranges in parallel (19 independent loads each), fixed order
        double *hout = (pass == 0) ? a.dev.h1 : a.dev.h2;
        for (int i0 = 0; i0 < nred; i0 += 64) {
            const int il = tid & 63, q = tid >> 6, i = i0 + il;
            double pv[ORTH_MAX_GRID / 8];
#pragma unroll
            for (int u = 0; u < ORTH_MAX_GRID / 8; ++u) {
                const int c = q + 8 * u;
                pv[u] = (i < nred && c < G) ? __ldcg(a.partial + (blockIdx.x % ORTH_REPLICAS) * rep_stride + (size_t)c * a.ld + i) : 0.0;
            }
            double s = 0.0;
#pragma unroll
            for (int u = 0; u < ORTH_MAX_GRID / 8; ++u) s += pv[u];
            red[q * 64 + il] = s;
            __syncthreads();
            if (q == 0 && i < nred) {
                double t = 0.0;
#pragma unroll
                for (int qq = 0; qq < 8; ++qq) t += red[qq * 64 + il];
                hs[i] = t;
                if (blockIdx.x == 0 && i < nvec) hout[i] = t;
            }
            __syncthreads();
        }
        // every CTA sums the same partials in the same order, so every CTA takes the same decision
        bool skip_second = false;
        if (nred > nvec) {
            if (tid == 0) {
                double s2 = 0.0;
                for (int i = 0; i < nvec; ++i) s2 = fma(hs[i], hs[i], s2);
                red[0] = (hs[nvec] - s2 >= a.eta2 * hs[nvec]) ? 1.0 : 0.0;
            }
            __syncthreads();
            skip_second = red[0] != 0.0;
        }
        MG_ORTH_STAMP(4 + 4 * pass);
        // ---- w_slice -= sum_i h_i V_i : one double2 per thread, two independent accumulator pairs
        for (int e = tid; e < len2; e += ORTH_THREADS) {
            double2 s0 = make_double2(0.0, 0.0), s1 = make_double2(0.0, 0.0);
            const double2 *c2 = reinterpret_cast<const double2 *>(vc) + e;
            int i = 0;
#pragma unroll 4
            for (; i + 1 < nc; i += 2) {
                const double2 v0 = c2[(size_t)i * slice2], v1 = c2[(size_t)(i + 1) * slice2];
                const double h0 = hs[i], h1 = hs[i + 1];
                s0.x = fma(h0, v0.x, s0.x); s0.y = fma(h0, v0.y, s0.y);
                s1.x = fma(h1, v1.x, s1.x); s1.y = fma(h1, v1.y, s1.y);
            }
            if (i < nc) {
                const double2 v0 = c2[(size_t)i * slice2];
                s0.x = fma(hs[i], v0.x, s0.x); s0.y = fma(hs[i], v0.y, s0.y);
            }
            const double2 *g2 = reinterpret_cast<const double2 *>(a.V + e0) + e;
            const size_t st2 = (size_t)(a.stride >> 1);
#pragma unroll 8
            for (i = nc; i < nvec; ++i) {
                const double2 v0 = __ldg(g2 + (size_t)i * st2);
                s1.x = fma(hs[i], v0.x, s1.x); s1.y = fma(hs[i], v0.y, s1.y);
            }
            double2 wv = reinterpret_cast<double2 *>(ws)[e];
            wv.x -= s0.x + s1.x;
            wv.y -= s0.y + s1.y;
            reinterpret_cast<double2 *>(ws)[e] = wv;
        }
        if (odd && tid == 0) {
            double acc = 0.0;
            for (int i = 0; i < nvec; ++i)
                acc = fma(hs[i], (i < a.cap) ? vc[(size_t)i * a.slice + len - 1] : a.V[(size_t)i * a.stride + e0 + len - 1], acc);
            ws[len - 1] -= acc;
        }
        __syncthreads();
        MG_ORTH_STAMP(5 + 4 * pass);
        if (skip_second) {
            if (blockIdx.x == 0)
                for (int i = tid; i < nvec; i += ORTH_THREADS) a.dev.h2[i] = 0.0;
            break;
        }
    }
    // ---- write back, ||w||^2, Hessenberg column / Givens / stop test in the last CTA
    double sq = 0.0;
    for (int e = tid; e < len; e += ORTH_THREADS) {
        const double v = ws[e];
        a.w[e0 + e] = v;
        sq = fma(v, v, sq);
    }
    sq = warp_sum(sq);
    if (lane == 0) red[warp] = sq;
    __syncthreads();
    __shared__ bool last;
    if (tid == 0) {
        double t = 0.0;
        for (int k = 0; k < NW; ++k) t += red[k];
        a.nrm_partial[blockIdx.x] = t;
        __threadfence();
        last = (atomicAdd(a.counter, 1u) == (unsigned)(G - 1));
    }
    __syncthreads();
    if (last && warp == 0) {
        __threadfence();
        double t = 0.0;
        for (int c = lane; c < G; c += 32) t += __ldcg(a.nrm_partial + c);
        t = warp_sum(t);
        if (lane == 0) {
            *a.dev.nrm2 = t;
            *a.counter = 0;
            if (a.defer_update) *a.dev.hnext = sqrt(fmax(t, 0.0));
        }
        __syncwarp();
        if (!a.defer_update)
            gmres_update_warp(a.dev, a.j, lane, hd, hd + a.ld, hs);   // hd [2 ld] and hs [ld] are free by now (ld >= m + 2)
    }
    MG_ORTH_STAMP(10);
}

// The deferred update of column j (OrthArgs::defer_update): one warp, launched on a side branch of the captured coarsest-level
// cycle, so that the serial rotation recurrence and the stop test run BESIDE the next SpMV -- which needs h_{j+1,j} and the new
// vector but nothing of the Givens state -- instead of in front of it.  That SpMV reads status[4], the `done` flag as the
// Gram-Schmidt kernel before it saw it (nothing writes it while the SpMV runs): after convergence it computes ONE vector nobody
// uses (the basis slot it writes is not part of the solution update).  The next Gram-Schmidt kernel is ordered after both.
__global__ void __launch_bounds__(32) gmres_givens_kernel(const GmresDev dev, const int j, const int ld) {
    extern __shared__ double givens_sm[];   // 3 ld doubles, ld >= m + 1
    gmres_update_warp(dev, j, (int)threadIdx.x, givens_sm, givens_sm + ld, givens_sm + 2 * ld, false);
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
    s.status[0] = 0; s.status[1] = 0; s.status[2] = 0; s.status[3] = 0; s.status[4] = 0;
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

// Back substitution H y = g over the j_used columns of this cycle.  One warp: the inner sum over l > i is split
// across the lanes (fixed lane -> l mapping and shuffle tree: deterministic).  Fast path (j_used <= 256): y lives in shared
// memory and the entries of row i-1 (which do not depend on y) are loaded while row i is reduced, so a row costs a shuffle
// tree and a division instead of two dependent global round trips (100 columns: ~150 -> ~35 us per restart cycle).  Same
// operations in the same order as the plain loop below: bit-identical y.
__global__ void __launch_bounds__(32) gmres_solve_y_kernel(GmresDev s) {
    const int ju = s.status[1];
    const int lane = threadIdx.x;
    constexpr int NL = 8;
    __shared__ double ys[32 * NL];
    const size_t ld = (size_t)s.m + 1;
    if (ju <= 32 * NL) {
        double hn[NL], gn = 0.0, dn = 1.0;
        {
            const int i = ju - 1;   // row ju-1 has no entries right of the diagonal
#pragma unroll
            for (int k = 0; k < NL; ++k) hn[k] = 0.0;
            if (lane == 0 && i >= 0) { gn = s.g[i]; dn = s.H[(size_t)i * ld + i]; }
        }
        for (int i = ju - 1; i >= 0; --i) {
            double hc[NL];
#pragma unroll
            for (int k = 0; k < NL; ++k) hc[k] = hn[k];
            const double gc = gn, dc = dn;
            if (i > 0) {
                const int ip = i - 1;
#pragma unroll
                for (int k = 0; k < NL; ++k) {
                    const int l = ip + 1 + lane + 32 * k;
                    hn[k] = (l < ju) ? s.H[(size_t)l * ld + ip] : 0.0;
                }
                if (lane == 0) { gn = s.g[ip]; dn = s.H[(size_t)ip * ld + ip]; }
            }
            double t = 0.0;
#pragma unroll
            for (int k = 0; k < NL; ++k) {
                const int l = i + 1 + lane + 32 * k;
                if (l < ju) t = fma(hc[k], ys[l], t);
            }
            t = warp_sum(t);
            if (lane == 0) {
                const double yi = (gc - t) / dc;
                ys[i] = yi;
                s.y[i] = yi;
            }
            __syncwarp();
        }
        return;
    }
    for (int i = ju - 1; i >= 0; --i) {
        double t = 0.0;
        for (int l = i + 1 + lane; l < ju; l += 32) t = fma(s.H[(size_t)l * ld + i], s.y[l], t);
        t = warp_sum(t);
        if (lane == 0) s.y[i] = (s.g[i] - t) / s.H[(size_t)i * ld + i];
        __syncwarp();
    }
}

}  // namespace mgk
