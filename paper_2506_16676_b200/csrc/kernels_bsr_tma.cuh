// kernels_bsr_tma.cuh -- block-CSR kernels of the solve path for b = 36 on sm_100a: SpMV, residual, PBJ apply
// and the fused PBJ-Chebyshev sweep as ONE persistent kernel whose
// matrix stream is moved by the TMA engine.
//
// Why: every step is a scan with 0.25 flop/byte, so the only thing that matters is keeping HBM busy.  The first
// kernel of this library (kernels_bsr.cuh: one CTA per block row, 128-bit loads into registers) moved exactly the
// algorithmic bytes but was latency bound at 72 % of the measured copy rate (profiles/r01_baseline_ldg_kernel.md:
// 2 CTAs per SM, every CTA drains its loads before it reduces).  Here loading and arithmetic are decoupled:
//
//   * grid = one persistent CTA per SM; CTA k owns a CONTIGUOUS range of block rows holding ~nnzb/grid blocks
//     (partition table built in mg_setup), hence one contiguous span of `vals`;
//   * a producer warp streams that span block by block (b*b*8 = 10,368 B) with 1-D bulk async copies
//     (cp.async.bulk -> SASS UBLKCP) into a ring of STAGES shared-memory stages, and with each block the x_J it
//     multiplies (288 B, an L2 hit), both completing on the stage's "full" mbarrier.  STAGES * 10.6 KB ~ 213 KB are
//     in flight per SM whatever the consumers do;
//   * NG consumer groups of 160 threads take the CTA's rows round-robin.  Thread t < 144 of a group owns the
//     9-element segment [9t, 9t+9) of every block of its row (row t/4, columns 9(t%4)..): shared-memory reads at a
//     9-double stride are bank-conflict free, the 4 partial sums of a row meet by two warp shuffles, blocks are
//     added in stored order (deterministic).  After the last read of a stage each consumer warp arrives on the
//     stage's "empty" mbarrier, which hands it back to the producer;
//   * the row epilogue is the fused part: residual, x update, z = Dinv_I r_I, Chebyshev direction update --
//     kernels_bsr.cuh documents the modes.  In a sweep Dinv_I rides in the SAME ring: the producer appends it to the
//     stream after the last block of every owned row, and the consumers multiply it by r_I exactly as they multiply a
//     block of A by x_J (round 1 fetched it with 72-byte per-thread loads into registers: the sweep then ran 4-5 %
//     below the SpMV pass in GB/s).
//
// PBJ apply alone is the same kernel on the implicit block-diagonal matrix `dinv` (row I = block I = column I).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels_bsr.cuh"

namespace mgk {

struct TmaCfg {
    static constexpr int B = 36, BB = B * B;
    static constexpr int SEGL = 9;                    // segment length (doubles) owned by one thread
    static constexpr int SEG = B / SEGL;              // 4 segments per block row
    static constexpr int ACTIVE = B * SEG;            // 144 working threads per group
    static constexpr int GROUP = 160;                 // 5 warps per group (16 idle lanes)
    static constexpr int GWARPS = GROUP / 32;
    static constexpr int NG = 4;                      // consumer groups per CTA (3: -8 %, 5: no gain)
    static constexpr int STAGES = 20;
    static constexpr int THREADS = NG * GROUP + 32;   // + 1 producer warp
    static constexpr int VECPAD = 40;                 // per group and row parity: the new residual r_I for the Dinv product
    static constexpr unsigned POLL_NS = 1000;         // sleep between polls of the producer's per-stage round counters
    static constexpr unsigned SWEEP_MBAR_NS = 100;    // back-off of the full-barrier wait in the fused sweep
    static constexpr size_t SMEM = sizeof(double) * ((size_t)STAGES * (BB + B) + 2 * NG * VECPAD) + sizeof(uint64_t) * (3 * STAGES);
};

// extra arguments of the TMA kernel (the common ones are BsrArgs)
struct TmaExtra {
    const int64_t *part;      // [2*(gridDim.x + 1)] per CTA k: {first block P_k, first OWNED block row Ra_k} (nullptr: uniform
                              // split of the implicit block-diagonal matrix).  A CTA owns the rows that START in [P_k, P_k+1).
                              // When P_k falls inside a row (balanced split), CTA k multiplies the row's remaining blocks first
                              // and hands the 36 partial sums to the owner CTA k-1 through frag_part / frag_flag.
    double *frag_part;        // [gridDim.x][36]
    int *frag_flag;           // [gridDim.x] zero-initialised; set by the fragment's CTA, cleared by the owner
    const double *scale_div;  // SPMV mode, optional: the input vector is vin / *scale_div (out = A vin / *scale_div)
    double *vout;             // SPMV mode, optional: vout_I = vin_I / *scale_div (the normalised input; vout != vin)
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
// Same, with a back-off between polls (ns = 0: none).  Waiting consumer warps otherwise compete with the producer warp
// and with the group that is in its row epilogue for issue slots (measured: see DESIGN.md 5.1).
__device__ __forceinline__ void mbar_wait_backoff(uint64_t *bar, uint32_t parity, unsigned ns) {
    uint32_t ok;
    while (true) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (ok) break;
        if (ns) __nanosleep(ns);
    }
}
// 1-D bulk async copy global -> shared, completing `bytes` on the mbarrier (TMA engine; SASS UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void group_bar(int g) {
    asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "n"(TmaCfg::GROUP) : "memory");
}

// max over block rows of the number of stored blocks
__global__ void max_row_blocks_kernel(const int64_t *__restrict__ row_ptr, const int64_t n_brows, int *__restrict__ out) {
    int m = 0;
    for (int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; I < n_brows; I += (int64_t)gridDim.x * blockDim.x)
        m = max(m, (int)(row_ptr[I + 1] - row_ptr[I]));
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// split != 0: P_k = k*nnzb/nparts exactly (equal block counts; a row may straddle two CTAs); split == 0: P_k is moved up to
// the next row start (row-aligned ranges, +-1 row of imbalance).  part[2k] = P_k, part[2k+1] = Ra_k = first row with
// row_ptr >= P_k.
__global__ void partition_rows_kernel(const int64_t *__restrict__ row_ptr, const int64_t n_brows, const int64_t nnzb,
                                      const int nparts, const int split, int64_t *__restrict__ part) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > nparts) return;
    if (k == nparts) {
        part[2 * k] = nnzb;
        part[2 * k + 1] = n_brows;
        return;
    }
    const int64_t target = (int64_t)(((__int128)nnzb * k) / nparts);
    int64_t lo = 0, hi = n_brows;  // first I in [0, n_brows] with row_ptr[I] >= target
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (row_ptr[mid] >= target) hi = mid; else lo = mid + 1;
    }
    part[2 * k] = split ? target : row_ptr[lo];
    part[2 * k + 1] = lo;
}

__global__ void __launch_bounds__(TmaCfg::THREADS, 1) bsr_tma_kernel(const BsrArgs a, const TmaExtra ex) {
    using C = TmaCfg;
    constexpr int B = C::B, BB = C::BB;
    if (a.done != nullptr && *a.done != 0) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sA = reinterpret_cast<double *>(smem_raw);
    double *sX = sA + (size_t)C::STAGES * BB;
    double *sVec = sX + C::STAGES * B;
    uint64_t *full = reinterpret_cast<uint64_t *>(sVec + 2 * C::NG * C::VECPAD);
    uint64_t *empty = full + C::STAGES;
    // round_of[s] = number of rounds for which stage s has been issued.  A consumer group may be more than one ring
    // round ahead of the stage it wants next (its row starts >= STAGES blocks after the oldest block still in flight);
    // an mbarrier parity wait is only meaningful for the current or the preceding phase, so the group first waits
    // until its block has been ISSUED (then the stage's previous round is consumed and its phase is the current one).
    volatile int *round_of = reinterpret_cast<volatile int *>(empty + C::STAGES);   // [STAGES]

    const bool diag = (a.mode == MODE_PBJ);             // implicit block-diagonal matrix `dinv`, x block = rin_I
    const double *stream = diag ? a.dinv : a.vals;
    const double *xsrc = diag ? a.rin : a.vin;
    int64_t R0, R1, P0, P1;   // owned rows [R0, R1), streamed blocks [P0, P1)
    if (ex.part != nullptr) {
        P0 = ex.part[2 * blockIdx.x];
        R0 = ex.part[2 * blockIdx.x + 1];
        P1 = ex.part[2 * blockIdx.x + 2];
        R1 = ex.part[2 * blockIdx.x + 3];
    } else {
        R0 = a.n_brows * blockIdx.x / gridDim.x;
        R1 = a.n_brows * (blockIdx.x + 1) / gridDim.x;
        P0 = R0;
        P1 = R1;
    }
    if (P0 >= P1) return;
    // head fragment: blocks [P0, row_ptr[R0]) belong to row R0-1, owned by the previous CTA
    const bool head = !diag && (a.row_ptr[R0] > P0);
    const int nitems = (int)(R1 - R0) + (head ? 1 : 0);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < C::STAGES; ++s) round_of[s] = 0;
        for (int s = 0; s < C::STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], C::GWARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == C::NG * C::GWARPS) {
        // ------------------------------------------------------------------ producer warp: stream blocks P0..P1
        const uint64_t pol = policy_evict_first();
        // Sweep with the Dinv product: the stream is [head fragment blocks] then, per owned row I, its blocks inside
        // [P0, P1) followed by Dinv_I; ring counter of row I's first block: f(I) = row_ptr[I] - P0 + (I - R0).
        const bool with_dinv = (a.mode == MODE_SWEEP) && (a.flags & F_NEED_D);
        const int total = (int)(P1 - P0) + (with_dinv ? (int)(R1 - R0) : 0);
        // Every lane < PL issues its own stage: the waits on the stages' "empty" barriers and the issue latencies
        // overlap (one issuing thread was the pacing element of the whole kernel: +5-7 % on levels 1-3).  round_of[s]
        // tells the consumers that stage s has been (re)issued for round k, see above.
        constexpr int PL = 16;
        int64_t Icur = R0;   // row cursor of this lane (with_dinv): largest owned row with f(I) <= i so far
        for (int base = 0; base < total; base += PL) {
            const int i = base + lane;
            if (lane < PL && i < total) {
                int64_t pblk = P0 + i;   // block to copy, or -1: Dinv of row Icur
                if (with_dinv) {
                    const int64_t fR0 = __ldg(a.row_ptr + R0) - P0;
                    if (i >= fR0 && R1 > R0) {
                        while (Icur + 1 < R1 && __ldg(a.row_ptr + Icur + 1) - P0 + (Icur + 1 - R0) <= i) ++Icur;
                        const int64_t rp = __ldg(a.row_ptr + Icur);
                        const int64_t o = i - (rp - P0 + (Icur - R0));
                        const int64_t nblk = min(__ldg(a.row_ptr + Icur + 1), P1) - rp;
                        pblk = o < nblk ? rp + o : -1;
                    }
                }
                const int s = i % C::STAGES, k = i / C::STAGES;
                mbar_wait(&empty[s], ((uint32_t)k & 1u) ^ 1u);
                round_of[s] = k + 1;
                if (pblk < 0) {   // Dinv_I: multiplied by the residual the consumers hold, no x block
                    mbar_expect_tx(&full[s], (uint32_t)(BB * sizeof(double)));
                    bulk_g2s(sA + (size_t)s * BB, a.dinv + (size_t)Icur * BB, BB * sizeof(double), &full[s]);
                } else {
                    const int j = diag ? (int)pblk : __ldg(a.col_idx + pblk);
                    mbar_expect_tx(&full[s], (uint32_t)((BB + B) * sizeof(double)));
                    // the matrix stream is read once per launch: evict-first keeps the vectors, the Krylov basis and (on small
                    // levels) Dinv resident in the 126 MB L2; Dinv itself is loaded with the default policy
                    if (diag) bulk_g2s(sA + (size_t)s * BB, stream + (size_t)pblk * BB, BB * sizeof(double), &full[s]);
                    else bulk_g2s_hint(sA + (size_t)s * BB, stream + (size_t)pblk * BB, BB * sizeof(double), &full[s], pol);
                    bulk_g2s(sX + s * B, xsrc + (size_t)j * B, B * sizeof(double), &full[s]);
                }
            }
            __syncwarp();
        }
        return;
    }

    // ---------------------------------------------------------------------- consumer groups: rows R0+g, R0+g+NG, ...
    const int g = tid / C::GROUP, t = tid - g * C::GROUP;
    const bool active = t < C::ACTIVE;
    const int r = t >> 2, h = t & 3;
    const bool writer = active && h == 0;
    const int flags = a.flags;
    const bool sweep = (a.mode == MODE_SWEEP);
    const bool need_d = sweep && (flags & F_NEED_D);
    const bool touch_x = (flags & (F_UPD_X | F_SET_X | F_FINAL_X)) != 0;
    double *vecbase = sVec + 2 * g * C::VECPAD;
    double inv_scale = 1.0;
    const bool spmv_scaled = (a.mode == MODE_SPMV) && ex.scale_div != nullptr;
    if (spmv_scaled) inv_scale = 1.0 / *ex.scale_div;

    const unsigned mbar_ns = need_d ? C::SWEEP_MBAR_NS : 0u;   // back off only when row epilogues are heavy
    // work items of this CTA: [the head fragment,] then the owned rows; group g takes items g, g+NG, ...
    int it = g;
    int64_t I = R0 + it - (head ? 1 : 0);
    int64_t p0 = 0, p1 = 0;
    if (it < nitems) {
        p0 = diag ? I : a.row_ptr[I];
        p1 = diag ? I + 1 : a.row_ptr[I + 1];
    }
    for (; it < nitems; it += C::NG, I += C::NG) {
        // next row's extent (off the critical path)
        const int64_t In = I + C::NG;
        int64_t p0n = 0, p1n = 0;
        if (it + C::NG < nitems) {
            p0n = diag ? In : a.row_ptr[In];
            p1n = diag ? In + 1 : a.row_ptr[In + 1];
        }
        const bool frag = head && it == 0;     // the tail of row R0-1: partial sums go to the owner CTA
        const bool open = p1 > P1;             // this row continues in the next CTA, which publishes its part
        if (frag) p0 = P0;
        if (open) p1 = P1;
        const size_t gi = (size_t)I * B + r;
        double rin_v = 0.0, dold = 0.0, xold = 0.0;
        if (active && !frag) {
            if (a.mode == MODE_RESID || sweep) rin_v = a.rin[gi];
            if (sweep || (spmv_scaled && ex.vout != nullptr)) dold = a.vin[gi];
            if (touch_x && !(flags & F_SET_X)) xold = a.x[gi];
        }
        // ring counter of the item's first block (with Dinv stages in the stream: one per owned row before this one)
        int n = (int)(p0 - P0) + ((need_d && !frag) ? (int)(I - R0) : 0);
        int s = n % C::STAGES;
        uint32_t ph = (uint32_t)(n / C::STAGES) & 1u;
        double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;
        for (int64_t p = p0; p < p1; ++p, ++n) {
            // not (re)issued for this round yet: sleep instead of spinning on shared memory (5-6 % on every level)
            while (round_of[s] <= n / C::STAGES) __nanosleep(C::POLL_NS);
            mbar_wait_backoff(&full[s], ph, mbar_ns);
            if (active) {
                const double *A = sA + (size_t)s * BB + C::SEGL * t;
                const double *xs = sX + s * B + C::SEGL * h;
                acc0 = fma(A[0], xs[0], acc0);
                acc1 = fma(A[1], xs[1], acc1);
                acc2 = fma(A[2], xs[2], acc2);
                acc0 = fma(A[3], xs[3], acc0);
                acc1 = fma(A[4], xs[4], acc1);
                acc2 = fma(A[5], xs[5], acc2);
                acc0 = fma(A[6], xs[6], acc0);
                acc1 = fma(A[7], xs[7], acc1);
                acc2 = fma(A[8], xs[8], acc2);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
            if (++s == C::STAGES) {
                s = 0;
                ph ^= 1u;
            }
        }
        double acc = (acc0 + acc1) + acc2;
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);

        if (frag) {
            // publish the 36 partial sums of the straddling row to its owner (CTA blockIdx.x - 1), then go on
            if (writer) ex.frag_part[(size_t)blockIdx.x * B + r] = acc;
            __threadfence();
            group_bar(g);
            if (t == 0) {
                __threadfence();
                atomicExch(ex.frag_flag + blockIdx.x, 1);
            }
            p0 = p0n;
            p1 = p1n;
            continue;
        }
        if (open) {
            // the rest of this row was multiplied by CTA blockIdx.x + 1 as its FIRST work item: it is there by now
            if (t == 0) {
                while (atomicAdd(ex.frag_flag + blockIdx.x + 1, 0) == 0) {
                }
                __threadfence();
            }
            group_bar(g);
            if (active) acc += __ldcg(ex.frag_part + (size_t)(blockIdx.x + 1) * B + r);
            group_bar(g);
            if (t == 0) atomicExch(ex.frag_flag + blockIdx.x + 1, 0);   // ready for the next launch
        }

        if (a.mode == MODE_SPMV) {
            if (writer) {
                a.out[gi] = spmv_scaled ? acc * inv_scale : acc;
                if (spmv_scaled && ex.vout != nullptr) ex.vout[gi] = dold * inv_scale;   // the normalised input vector
            }
        } else if (a.mode == MODE_RESID) {
            if (writer) a.out[gi] = rin_v - acc;
        } else if (diag) {
            const double dnew = a.c_z * acc;
            if (writer) {
                a.dout[gi] = dnew;
                if (flags & F_FINAL_X) a.x[gi] = xold + dnew;
            }
        } else {
            const double rnew = rin_v - acc;
            if (writer) a.out[gi] = rnew;
            if (!need_d) {
                if (writer) {
                    if (flags & F_SET_X) a.x[gi] = dold;
                    else if (flags & F_UPD_X) a.x[gi] = xold + dold;
                }
            } else {
                // z = Dinv_I r': Dinv_I is the next stage of the ring (s, ph, n already point at it); r' goes through a
                // per-group buffer, double-buffered by row parity so that one group barrier per row suffices
                double *vec = vecbase + (((it - g) / C::NG) & 1) * C::VECPAD;
                if (writer) vec[r] = rnew;
                group_bar(g);
                while (round_of[s] <= n / C::STAGES) __nanosleep(C::POLL_NS);
                mbar_wait_backoff(&full[s], ph, mbar_ns);
                double z = 0.0;
                if (active) {
                    const double *D = sA + (size_t)s * BB + C::SEGL * t;
                    const double *vs = vec + C::SEGL * h;
                    double z0 = 0.0, z1 = 0.0, z2 = 0.0;
                    z0 = fma(D[0], vs[0], z0);
                    z1 = fma(D[1], vs[1], z1);
                    z2 = fma(D[2], vs[2], z2);
                    z0 = fma(D[3], vs[3], z0);
                    z1 = fma(D[4], vs[4], z1);
                    z2 = fma(D[5], vs[5], z2);
                    z0 = fma(D[6], vs[6], z0);
                    z1 = fma(D[7], vs[7], z1);
                    z2 = fma(D[8], vs[8], z2);
                    z = (z0 + z1) + z2;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
                z += __shfl_xor_sync(0xffffffffu, z, 1);
                z += __shfl_xor_sync(0xffffffffu, z, 2);
                if (writer) {
                    double dnew = a.c_z * z;
                    if (a.c_d != 0.0) dnew = fma(a.c_d, dold, dnew);
                    double xv;
                    if (flags & F_SET_X) xv = dold;
                    else {
                        xv = xold;
                        if (flags & F_UPD_X) xv += dold;
                    }
                    a.dout[gi] = dnew;
                    if (flags & F_FINAL_X) xv += dnew;
                    if (touch_x) a.x[gi] = xv;
                }
            }
        }
        p0 = p0n;
        p1 = p1n;
    }
}

}  // namespace mgk
