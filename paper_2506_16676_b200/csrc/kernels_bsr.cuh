// kernels_bsr.cuh -- block-CSR kernels of the solve path: SpMV, residual, PBJ apply and the fused
// PBJ-Chebyshev sweep ("explicit, dense inverses ... dense matrix-vector
// products", "a sparse matrix vector product, the kernel of MG").
//
// One kernel body, four modes, so that a smoother sweep reads the block row of A exactly once:
//   SPMV : out_I  = sum_J A_IJ vin_J
//   RESID: out_I  = rin_I - sum_J A_IJ vin_J
//   SWEEP: out_I  = rin_I - sum_J A_IJ vin_J          (new residual, may alias rin)
//          x_I   (+)= vin_I                           (flags SET_X / UPD_X)
//          z      = Dinv_I out_I ; dout_I = c_d vin_I + c_z z     (flag NEED_D; dout != vin)
//          x_I   += dout_I                            (flag FINAL_X)
//   PBJ  : z = Dinv_I rin_I ; dout_I = c_z z ; x_I += dout_I (flag FINAL_X)
//
// Thread mapping (fast path, compile-time B): a group of EPB = B*B/VEC threads owns one block row; thread q
// owns element q (VEC = 2 doubles, one 128-bit load) of every block of the row, so consecutive threads read
// consecutive 16-byte words of the contiguous value span of the row: fully coalesced, 128-bit vectorised.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mgk {

enum { MODE_SPMV = 0, MODE_RESID = 1, MODE_SWEEP = 2, MODE_PBJ = 3 };
enum { F_UPD_X = 1, F_SET_X = 2, F_NEED_D = 4, F_FINAL_X = 8 };

struct BsrArgs {
    const int64_t *row_ptr;
    const int32_t *col_idx;
    const double *vals;
    const double *dinv;
    const double *vin;
    const double *rin;
    double *out;
    double *x;
    double *dout;
    double c_d, c_z;
    int64_t n_brows;
    int mode;
    int flags;
    const int *done;  // optional device flag: the kernel is a no-op when *done != 0
};

__device__ __forceinline__ double2 ld_stream2(const double *p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_stream1(const double *p) {
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}

template <int B>
struct BsrCfg {
    static constexpr int VEC = (B % 2 == 0) ? 2 : 1;
    static constexpr int EPB = B * B / VEC;  // VEC-wide elements per block
    static constexpr int EPR = B / VEC;      // elements per row of a block
    static constexpr int G = (EPB >= 256) ? 1 : (256 / EPB);  // block rows (groups) per CTA
    static constexpr int THREADS = ((G * EPB + 31) / 32) * 32;
    static constexpr int RESIDENT = 2048 / THREADS;   // CTAs per SM the small-block kernel is compiled for (32 registers;
                                                      // 5 / 6 CTAs with 48 / 40 registers measured 8-20 % slower)
};

// Small blocks are occupancy bound (ncu: 44 registers allowed 5 CTAs of 224 threads per SM, 55 % occupancy, DRAM at
// 48 %): capping the kernel at 32 registers (full occupancy, 17 words of spill) raised b = 12 from 0.54 to 0.72 and
// b = 6 from 0.53 to 0.62 of 8 TB/s.
// One group of G block rows (row group `rg`) by one CTA; every return below is CTA-uniform.
template <int B>
__device__ __forceinline__ void bsr_fused_rowgroup(const BsrArgs &a, const int64_t rg, double (*part)[BsrCfg<B>::EPB],
                                                   double (*vec)[B]) {
    using C = BsrCfg<B>;
    constexpr int VEC = C::VEC, EPB = C::EPB, EPR = C::EPR, G = C::G, BB = B * B;
    const int tid = threadIdx.x;
    const int g = tid / EPB;
    const int q = tid - g * EPB;
    const int64_t I = rg * G + g;
    const bool valid = (g < G) && (I < a.n_brows);
    const int c = (q * VEC) % B;  // first column this thread multiplies

    double acc0 = 0.0, acc1 = 0.0;
    double2 dv = make_double2(0.0, 0.0);
    if (valid) {
        if (a.mode == MODE_PBJ || (a.mode == MODE_SWEEP && (a.flags & F_NEED_D))) {
            const double *dp = a.dinv + (size_t)I * BB + (size_t)q * VEC;
            if (VEC == 2) dv = ld_stream2(dp); else dv.x = ld_stream1(dp);
        }
        if (a.mode != MODE_PBJ) {
            int64_t p = a.row_ptr[I];
            const int64_t p1 = a.row_ptr[I + 1];
            const double *ap = a.vals + (size_t)p * BB + (size_t)q * VEC;
            const double *xin = a.vin + c;
            if (VEC == 2) {
                for (; p + 4 <= p1; p += 4) {
                    const double2 v0 = ld_stream2(ap), v1 = ld_stream2(ap + BB), v2 = ld_stream2(ap + 2 * BB),
                                  v3 = ld_stream2(ap + 3 * BB);
                    const int j0 = __ldg(a.col_idx + p), j1 = __ldg(a.col_idx + p + 1), j2 = __ldg(a.col_idx + p + 2),
                              j3 = __ldg(a.col_idx + p + 3);
                    const double2 x0 = __ldg(reinterpret_cast<const double2 *>(xin + (size_t)j0 * B));
                    const double2 x1 = __ldg(reinterpret_cast<const double2 *>(xin + (size_t)j1 * B));
                    const double2 x2 = __ldg(reinterpret_cast<const double2 *>(xin + (size_t)j2 * B));
                    const double2 x3 = __ldg(reinterpret_cast<const double2 *>(xin + (size_t)j3 * B));
                    acc0 = fma(v0.x, x0.x, acc0); acc1 = fma(v0.y, x0.y, acc1);
                    acc0 = fma(v1.x, x1.x, acc0); acc1 = fma(v1.y, x1.y, acc1);
                    acc0 = fma(v2.x, x2.x, acc0); acc1 = fma(v2.y, x2.y, acc1);
                    acc0 = fma(v3.x, x3.x, acc0); acc1 = fma(v3.y, x3.y, acc1);
                    ap += 4 * BB;
                }
                for (; p < p1; ++p) {
                    const double2 v0 = ld_stream2(ap);
                    const int j0 = __ldg(a.col_idx + p);
                    const double2 x0 = __ldg(reinterpret_cast<const double2 *>(xin + (size_t)j0 * B));
                    acc0 = fma(v0.x, x0.x, acc0); acc1 = fma(v0.y, x0.y, acc1);
                    ap += BB;
                }
            } else {
                for (; p < p1; ++p) {
                    const double v0 = ld_stream1(ap);
                    const int j0 = __ldg(a.col_idx + p);
                    acc0 = fma(v0, __ldg(xin + (size_t)j0 * B), acc0);
                    ap += BB;
                }
            }
        }
    }
    if (a.mode != MODE_PBJ) {
        if (g < G) part[g][q] = acc0 + acc1;
        __syncthreads();
    }
    double rnew = 0.0;
    if (valid && q < B) {
        const size_t gi = (size_t)I * B + q;
        if (a.mode == MODE_PBJ) {
            rnew = a.rin[gi];
        } else {
            double t = 0.0;
#pragma unroll
            for (int e = 0; e < EPR; ++e) t += part[g][q * EPR + e];
            if (a.mode == MODE_SPMV) {
                a.out[gi] = t;
            } else {
                rnew = a.rin[gi] - t;
                a.out[gi] = rnew;
            }
        }
        vec[g][q] = rnew;
    }
    const bool second = (a.mode == MODE_PBJ) || (a.mode == MODE_SWEEP && (a.flags & F_NEED_D));
    if (a.mode == MODE_SWEEP && !second) {
        if (valid && q < B) {
            const size_t gi = (size_t)I * B + q;
            const double dold = a.vin[gi];
            if (a.flags & F_SET_X) a.x[gi] = dold;
            else if (a.flags & F_UPD_X) a.x[gi] += dold;
        }
        return;
    }
    if (!second) return;
    __syncthreads();
    if (g < G) {
        double s = dv.x * vec[g][c];
        if (VEC == 2) s = fma(dv.y, vec[g][c + 1], s);
        part[g][q] = s;
    }
    __syncthreads();
    if (valid && q < B) {
        const size_t gi = (size_t)I * B + q;
        double z = 0.0;
#pragma unroll
        for (int e = 0; e < EPR; ++e) z += part[g][q * EPR + e];
        double dnew = a.c_z * z;
        double xv = 0.0;
        const bool touch_x = (a.flags & (F_UPD_X | F_SET_X | F_FINAL_X)) != 0;
        if (a.mode == MODE_SWEEP) {
            const double dold = a.vin[gi];
            if (a.c_d != 0.0) dnew = fma(a.c_d, dold, dnew);
            if (a.flags & F_SET_X) xv = dold;
            else {
                if (touch_x) xv = a.x[gi];
                if (a.flags & F_UPD_X) xv += dold;
            }
        } else if (touch_x) {
            xv = a.x[gi];
        }
        a.dout[gi] = dnew;
        if (a.flags & F_FINAL_X) xv += dnew;
        if (touch_x) a.x[gi] = xv;
    }
}

// The kernel: a grid-stride loop over the row groups.  Small blocks are launched with a RESIDENT grid (SM count x CTAs per SM):
// a CTA lives for ~3 dependent load rounds per row group, so one CTA per group spent ~5-7 % of the launch on CTA turnover
// (round 2, C4: b = 6 SpMV 4.88-4.93 -> 5.16-5.21 TB/s, sweep 4.67 -> 4.98-5.02; b = 12 SpMV 5.73-5.82 -> 5.86-6.08, sweep
// 5.22-5.27 -> 5.55-5.62).
template <int B>
__global__ void __launch_bounds__(BsrCfg<B>::THREADS, (B <= 12 ? BsrCfg<B>::RESIDENT : 0)) bsr_fused_kernel(const BsrArgs a) {
    using C = BsrCfg<B>;
    if (a.done != nullptr && *a.done != 0) return;
    __shared__ double part[C::G][C::EPB];
    __shared__ double vec[C::G][B];
    const int64_t ngroups = (a.n_brows + C::G - 1) / C::G;
    for (int64_t rg = blockIdx.x; rg < ngroups; rg += gridDim.x) {
        bsr_fused_rowgroup<B>(a, rg, part, vec);
        __syncthreads();   // part / vec are reused by the next row group
    }
}

// Generic block size (1 <= b <= 64, run time): one warp per block row, lane r (and r + 32) owns row r of every
// block.  Correct for any b; not tuned (the configs use b in {6, 12, 36}, which take the path above).
__global__ void __launch_bounds__(128) bsr_fused_generic_kernel(const BsrArgs a, const int b) {
    if (a.done != nullptr && *a.done != 0) return;
    __shared__ double vec[4][64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t I = (int64_t)blockIdx.x * 4 + warp;
    const bool valid = I < a.n_brows;
    const int bb = b * b;
    double t[2] = {0.0, 0.0};
    if (valid && a.mode != MODE_PBJ) {
        for (int64_t p = a.row_ptr[I]; p < a.row_ptr[I + 1]; ++p) {
            const double *blk = a.vals + (size_t)p * bb;
            const double *xj = a.vin + (size_t)a.col_idx[p] * b;
            for (int h = 0; h < 2; ++h) {
                const int r = lane + 32 * h;
                if (r < b)
                    for (int cc = 0; cc < b; ++cc) t[h] = fma(blk[r * b + cc], xj[cc], t[h]);
            }
        }
    }
    double rnew[2] = {0.0, 0.0};
    if (valid)
        for (int h = 0; h < 2; ++h) {
            const int r = lane + 32 * h;
            if (r >= b) continue;
            const size_t gi = (size_t)I * b + r;
            if (a.mode == MODE_PBJ) rnew[h] = a.rin[gi];
            else if (a.mode == MODE_SPMV) a.out[gi] = t[h];
            else { rnew[h] = a.rin[gi] - t[h]; a.out[gi] = rnew[h]; }
            vec[warp][r] = rnew[h];
        }
    const bool second = (a.mode == MODE_PBJ) || (a.mode == MODE_SWEEP && (a.flags & F_NEED_D));
    __syncwarp();
    if (!valid || a.mode == MODE_SPMV || a.mode == MODE_RESID) return;
    const bool touch_x = (a.flags & (F_UPD_X | F_SET_X | F_FINAL_X)) != 0;
    for (int h = 0; h < 2; ++h) {
        const int r = lane + 32 * h;
        if (r >= b) continue;
        const size_t gi = (size_t)I * b + r;
        double dnew = 0.0;
        if (second) {
            const double *drow = a.dinv + (size_t)I * bb + (size_t)r * b;
            double z = 0.0;
            for (int cc = 0; cc < b; ++cc) z = fma(drow[cc], vec[warp][cc], z);
            dnew = a.c_z * z;
        }
        double xv = 0.0;
        if (a.mode == MODE_SWEEP) {
            const double dold = a.vin[gi];
            if (second && a.c_d != 0.0) dnew = fma(a.c_d, dold, dnew);
            if (a.flags & F_SET_X) xv = dold;
            else {
                if (touch_x) xv = a.x[gi];
                if (a.flags & F_UPD_X) xv += dold;
            }
        } else if (touch_x) {
            xv = a.x[gi];
        }
        if (second) {
            a.dout[gi] = dnew;
            if (a.flags & F_FINAL_X) xv += dnew;
        }
        if (touch_x) a.x[gi] = xv;
    }
}

}  // namespace mgk
