// mg_toroidal.cu -- C-ABI library (include/mg_toroidal.h): handle, setup, V-cycle, coarse GMRES, FGMRES.
// Host code only orchestrates; every step of the path runs in the kernels of kernels_*.cuh.
#include "../../include/mg_toroidal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <queue>
#include <string>
#include <vector>

#include "kernels_bsr.cuh"
#include "kernels_bsr_tma.cuh"
#include "kernels_direct.cuh"
#include "kernels_line.cuh"
#include "kernels_setup.cuh"
#include "kernels_vec.cuh"

using namespace mgk;

namespace {

thread_local std::string g_last_cuda_error;

// ---- mg_dot_noalloc: scratch of the deterministic dot product in a file-scope device array (no cudaMalloc anywhere on that
// path).  Layout: [0, 8192) 1,024 per-CTA partial sums (double), [8192, 8196) the ticket counter (unsigned).  In HOST code this
// name is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress, once per device.
constexpr int NOALLOC_MAX_GRID = 1024;
static __device__ __align__(256) unsigned char mg_noalloc_scratch[MG_NOALLOC_SCRATCH_BYTES];
static_assert(MG_NOALLOC_SCRATCH_BYTES >= NOALLOC_MAX_GRID * 8 + 4, "scratch holds the partial sums and the counter");
constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned char *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};   // device address of mg_noalloc_scratch per device ordinal
std::mutex g_noalloc_mutex;

struct Level {
    int index = 0;
    int n_phi = 0;
    int64_t n_brows = 0, nnzb = 0, nvec = 0;
    const int64_t *row_ptr = nullptr;
    const int32_t *col_idx = nullptr;
    const double *vals = nullptr;
    int64_t *diag_pos = nullptr;
    int64_t *row_of_block = nullptr;  // coarse levels: block row of every stored block (Galerkin numeric phase)
    unsigned long long *err_flag = nullptr;  // device flag of the batched inverse (first singular block, or ~0)
    double *dinv = nullptr;
    int64_t *part = nullptr;  // TMA kernel: first block row of each persistent CTA (tma_grid + 1 entries)
    int tma_grid = 0;
    double rho_est = 0.0, lam_min = 0.0, lam_max = 0.0;
    // toroidal-line block Jacobi (opt.smoother = 2): block positions, explicit inverses G (N per node), W (N - 1 per node)
    int64_t *lpos = nullptr;
    double *lineG = nullptr, *lineW = nullptr;
    bool line_ready = false;   // factorised for the current values
    bool rho_is_line = false;  // rho_est was estimated with the line preconditioner
    double *x = nullptr, *r = nullptr, *d[2] = {nullptr, nullptr}, *pe = nullptr, *rhs = nullptr;
    std::vector<int64_t> h_row_ptr;  // host copies of the pattern (Galerkin symbolic phase)
    std::vector<int32_t> h_col_idx;
};

struct ProfPair {
    cudaEvent_t e0, e1;
    int level, kind;
};
struct ProfAcc {
    int64_t launches = 0;  // every launch since the last reset (graph replays included)
    int64_t timed = 0;     // launches bracketed by events while profiling was on
    double ms = 0.0;       // their summed device time
};

struct Gmres {
    GmresDev dev{};
    int m = 0, maxit = 0;
    int64_t n = 0, stride = 0;
    double *V = nullptr, *Z = nullptr;
    double *partial = nullptr;
    unsigned *counter = nullptr;
    int red_grid = 0;
    bool flexible = false;
    bool ready = false;
    int level = 0;  // level whose vectors this engine orthogonalises (profiling only)
    // fused cooperative CGS2 step (gmres_orth_fused_kernel)
    bool fused_ok = false;
    int orth_grid = 0, orth_slice = 0, orth_cap = 0, orth_ld = 0;
    size_t orth_smem = 0;
    double *orth_partial = nullptr, *orth_nrm = nullptr;
    unsigned *orth_counter = nullptr;
};

// Direct solve of the coarsest level (kernels_direct.cuh): level-set ordering, dense blocks, explicit Schur inverses.
struct DirectCoarse {
    bool symbolic = false, numeric = false;
    int nlev = 0;
    std::vector<int> nk;        // dense dimension of every level set
    std::vector<int> voff;      // offset of every level set in the permuted vector (scalars)
    std::vector<double *> S;    // device; D_k at assembly, then the Schur complement S_k, then S_k^-1
    double *Mtmp = nullptr;     // scratch of the numeric phase: L_k S_{k-1}^-1
    int32_t *perm = nullptr, *inv = nullptr, *lev = nullptr, *off = nullptr;   // device
    double **dS = nullptr;      // device pointer table
    int mid = 0;                // middle level set: elimination runs 0 -> mid and nlev-1 -> mid
    int64_t *csc_ptr[2] = {nullptr, nullptr}, *csc_pos[2] = {nullptr, nullptr};   // by block column (new numbering): 0 = blocks of U_{k-1}
                                // (row one level set down), 1 = blocks of L_{k+1} (row one level set up): the Schur updates
    int64_t *od_ptr[2] = {nullptr, nullptr}, *od_pos[2] = {nullptr, nullptr};   // by block row (new numbering): 0 = the blocks an
    int32_t *od_col[2] = {nullptr, nullptr};   // elimination step multiplies, 1 = those of the back-substitution; new columns
    struct Job { int level, phase, final; };
    std::vector<std::vector<Job>> steps;       // the solve: steps of up to two independent jobs
    int64_t *rob = nullptr;     // block row of every stored block
    double *zb = nullptr, *yb = nullptr, *tb = nullptr;
    double *pinv = nullptr, *cpanel = nullptr, *rpanel = nullptr;   // blocked Gauss-Jordan: pivot-block inverse, saved panels
    int *bad = nullptr;
    int maxn = 0;
    int64_t bytes = 0;
    // persistent cooperative solve kernel (direct_solve_persistent_kernel); the launch chain is the fallback
    bool persist = false;
    DsStepDesc *stepdev = nullptr;
    double *xchg = nullptr;       // yb | xb | tb of the persistent kernel, one allocation (sentinel-filled before every launch)
    int64_t xchg_doubles = 0, tb_doubles = 0;
    int ds_grid = 0, ds_stages = 0, ds_tcap = 0;
    size_t ds_smem = 0;
    std::vector<int32_t> first;   // first new block position of every level set
    int64_t offdiag_blocks = 0;   // stored blocks of all L_k and U_k
    double *ell = nullptr;        // packed (ELL) off-diagonal block rows in the level-set ordering, both sides
    int32_t *ell_col = nullptr;   // [2][n_brows][DS_MAXNE]
    int *lev_ne = nullptr;        // device [nlev][2]
    long long *lev_off = nullptr; // device [nlev][2]
    int64_t ell_doubles = 0;
};

}  // namespace

struct mg_handle {
    mg_options opt{};
    int b = 0, n_pol = 0, n_phi = 0, n_levels = 0;
    int sm_count = 148;
    bool coop_ok = false;    // cooperative launches available and gmres_orth_fused_kernel's shared memory opted in
    bool coop_launch = false;  // the device supports cooperative launches
    double *frag_part = nullptr;  // TMA kernel: partial sums of rows that straddle two CTAs (sm_count x 36)
    int *frag_flag = nullptr;
    bool tma_ready = false;  // b == 36 and the kernel's shared-memory attribute is set
    size_t line_smem_set = 0;  // dynamic shared memory line_apply_staged_kernel has been opted in for
    cudaStream_t stream = nullptr;      // active stream: the caller's, or cap_stream while a graph is captured
    cudaStream_t cap_stream = nullptr;  // internal non-default stream (the legacy default stream cannot capture)
    cudaStream_t side_stream = nullptr; // captured side branch: the deferred Givens kernel of the coarsest-level cycle
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bool join_pending = false;
    std::vector<Level> lev;
    std::vector<void *> owned;
    std::vector<size_t> owned_bytes;   // parallel to `owned`
    int64_t dev_bytes = 0;
    int64_t launches = 0;
    int *pinned = nullptr;        // 8 ints + 4 doubles of pinned host scratch
    double *pinned_d = nullptr;
    // scratch reduction (power iteration, norms)
    double *red_partial = nullptr, *red_out = nullptr;
    unsigned *red_counter = nullptr;
    Gmres coarse, outer;
    DirectCoarse direct;
    std::vector<Gmres> smooth_g;         // per level: Arnoldi engine of the GMRES-PBJ smoother (opt.smoother = 1)
    const double *outer_vals = nullptr;  // values of the operator FGMRES solves with (mg_set_operator); NULL = level 0's
    double *coarse_ahat = nullptr;       // A D^-1 of the coarsest level as one block-CSR matrix (fused coarse GMRES)
    double *coarse_stage[2] = {nullptr, nullptr};  // unnormalised Arnoldi vectors between the SpMV and the CGS2 kernel
    cudaGraphExec_t coarse_graph = nullptr;
    int64_t coarse_graph_kernels = 0;
    bool capturing = false;
    int64_t capture_count = 0;
    double *d_rhs_host = nullptr, *d_x_host = nullptr;  // device staging for mg_solve_host
    int coarse_iters_total = 0, coarse_iters_last = 0;
    cudaEvent_t ev_solve[2] = {nullptr, nullptr};        // device time of the last mg_solve
    // profiling (mg_profile_enable): every launch is bracketed by an event pair and booked per (level, kind)
    bool profiling = false;
    int cur_level = 0, cur_kind = MG_KIND_OTHER;
    std::vector<ProfPair> prof_pending;
    std::vector<cudaEvent_t> prof_free;
    ProfAcc prof[MG_PROFILE_MAX_LEVELS][MG_KIND_COUNT];
    int64_t graph_hist[MG_PROFILE_MAX_LEVELS][MG_KIND_COUNT] = {};  // kernel nodes of the captured coarse cycle
};

namespace {

int cuda_fail(cudaError_t e, const char *what) {
    g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
    return MG_ECUDA;
}
#define CU(expr)                                            \
    do {                                                    \
        cudaError_t e__ = (expr);                           \
        if (e__ != cudaSuccess) return cuda_fail(e__, #expr); \
    } while (0)
#define MG(expr)                  \
    do {                          \
        int rc__ = (expr);        \
        if (rc__ != MG_OK) return rc__; \
    } while (0)

inline void count_launch(mg_handle *h) {
    const int lv = std::min(h->cur_level, MG_PROFILE_MAX_LEVELS - 1);
    if (h->capturing) {
        h->capture_count++;
        h->graph_hist[lv][h->cur_kind]++;
    } else {
        h->launches++;
        h->prof[lv][h->cur_kind].launches++;
    }
}

// Profiling: resolve the pending event pairs into the per-(level, kind) accumulators (synchronises the stream).
void prof_flush(mg_handle *h) {
    if (h->prof_pending.empty()) return;
    cudaStreamSynchronize(h->stream);
    for (const ProfPair &pp : h->prof_pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, pp.e0, pp.e1) == cudaSuccess) {
            ProfAcc &a = h->prof[std::min(pp.level, MG_PROFILE_MAX_LEVELS - 1)][pp.kind];
            a.timed++;
            a.ms += ms;
        }
        h->prof_free.push_back(pp.e0);
        h->prof_free.push_back(pp.e1);
    }
    h->prof_pending.clear();
}
inline cudaEvent_t prof_event(mg_handle *h) {
    if (!h->prof_free.empty()) {
        cudaEvent_t e = h->prof_free.back();
        h->prof_free.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
inline bool prof_begin(mg_handle *h, ProfPair &pp) {
    if (!h->profiling || h->capturing) return false;
    if (h->prof_pending.size() >= 2048) prof_flush(h);
    pp.e0 = prof_event(h);
    pp.e1 = prof_event(h);
    pp.level = h->cur_level;
    pp.kind = h->cur_kind;
    cudaEventRecord(pp.e0, h->stream);
    return true;
}
inline void prof_end(mg_handle *h, ProfPair &pp) {
    cudaEventRecord(pp.e1, h->stream);
    h->prof_pending.push_back(pp);
}
#define LAUNCH(h, kern, grid, block, smem, ...)                     \
    do {                                                            \
        ProfPair pp__;                                              \
        const bool prof__ = prof_begin(h, pp__);                    \
        kern<<<(grid), (block), (smem), (h)->stream>>>(__VA_ARGS__); \
        if (prof__) prof_end(h, pp__);                              \
        count_launch(h);                                            \
    } while (0)
// Programmatic dependent launch (the kernel calls cudaGridDependencySynchronize() before it touches data of the previous
// kernel in the stream): the launch latency and the prologue overlap the tail of that kernel.
template <typename... KArgs, typename... Args>
inline void launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#define LAUNCH_PDL(h, kern, grid, block, smem, ...)                                \
    do {                                                                           \
        ProfPair pp__;                                                             \
        const bool prof__ = prof_begin(h, pp__);                                   \
        launch_pdl(kern, dim3(grid), dim3(block), (smem), (h)->stream, __VA_ARGS__); \
        if (prof__) prof_end(h, pp__);                                             \
        count_launch(h);                                                           \
    } while (0)
struct KindScope {  // books the launches of one scope under (level, kind)
    mg_handle *h;
    int level0, kind0;
    KindScope(mg_handle *hh, int level, int kind) : h(hh), level0(hh->cur_level), kind0(hh->cur_kind) {
        h->cur_level = level;
        h->cur_kind = kind;
    }
    ~KindScope() {
        h->cur_level = level0;
        h->cur_kind = kind0;
    }
};

int dalloc(mg_handle *h, void **p, size_t bytes) {
    bytes = std::max<size_t>(bytes, 16);
    void *q = nullptr;
    if (h->opt.alloc) {
        q = h->opt.alloc(bytes, h->opt.alloc_ctx);
        if (!q) return MG_ENOMEM;
    } else {
        cudaError_t e = cudaMalloc(&q, bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return MG_ENOMEM;
        }
    }
    h->owned.push_back(q);
    h->owned_bytes.push_back(bytes);
    h->dev_bytes += (int64_t)bytes;
    *p = q;
    return MG_OK;
}
template <typename T>
int dalloc_t(mg_handle *h, T **p, size_t count) {
    return dalloc(h, reinterpret_cast<void **>(p), count * sizeof(T));
}
// Release one allocation of the handle before mg_destroy (buffers that are re-sized: the Krylov bases).
template <typename T>
void dfree_t(mg_handle *h, T *&p) {
    if (p == nullptr) return;
    auto it = std::find(h->owned.begin(), h->owned.end(), static_cast<void *>(p));
    if (it != h->owned.end()) {
        const size_t idx = (size_t)(it - h->owned.begin());
        h->dev_bytes -= (int64_t)h->owned_bytes[idx];
        h->owned_bytes.erase(h->owned_bytes.begin() + idx);
        h->owned.erase(it);
        if (h->opt.free) h->opt.free(p, h->opt.alloc_ctx);
        else if (!h->opt.alloc) cudaFree(p);
    }
    p = nullptr;
}

inline int grid_for(int64_t n, int per_block, int cap = 148 * 16) {
    int64_t g = (n + per_block - 1) / per_block;
    return (int)std::max<int64_t>(1, std::min<int64_t>(g, cap));
}

// ------------------------------------------------------------------------------------------------ BSR launch
int launch_bsr(mg_handle *h, const Level &L, BsrArgs a, TmaExtra ex = TmaExtra{}) {
    a.row_ptr = L.row_ptr;
    a.col_idx = L.col_idx;
    a.vals = L.vals;
    a.dinv = L.dinv;
    a.n_brows = L.n_brows;
    if (L.n_brows == 0) return MG_OK;
    const int kind = a.mode == MODE_SPMV ? MG_KIND_SPMV : a.mode == MODE_RESID ? MG_KIND_RESID : a.mode == MODE_PBJ ? MG_KIND_PBJ
                     : (a.flags & F_NEED_D) ? MG_KIND_SWEEP : MG_KIND_SWEEP_NOD;
    KindScope scope(h, L.index, kind);
    if (h->tma_ready && h->opt.kernel_variant == 0 && L.part != nullptr) {
        int grid = L.tma_grid;
        ex.part = L.part;
        ex.frag_part = h->frag_part;
        ex.frag_flag = h->frag_flag;
        if (a.mode == MODE_PBJ) {  // implicit block-diagonal stream: uniform split
            ex.part = nullptr;
            grid = (int)std::min<int64_t>(h->sm_count, L.n_brows);
        }
        LAUNCH(h, bsr_tma_kernel, grid, TmaCfg::THREADS, TmaCfg::SMEM, a, ex);
        CU(cudaGetLastError());
        return MG_OK;
    }
    if (ex.scale_div != nullptr || ex.vout != nullptr) return MG_EINVAL;  // fused scaling exists in the TMA kernel only
    switch (h->b) {
#define BSR_CASE(B)                                                                                          \
    case B: {                                                                                                \
        int grid = (int)((L.n_brows + BsrCfg<B>::G - 1) / BsrCfg<B>::G);                                      \
        if (B <= 12 && a.mode != MODE_PBJ) grid = std::min(grid, h->sm_count * BsrCfg<B>::RESIDENT); /* resident grid, row groups in a loop (not for the one-load-round PBJ apply: 15 % slower there) */ \
        LAUNCH(h, bsr_fused_kernel<B>, grid, BsrCfg<B>::THREADS, 0, a);                                       \
        break;                                                                                               \
    }
        BSR_CASE(6)
        BSR_CASE(12)
        BSR_CASE(36)
#undef BSR_CASE
        default: {
            const int grid = (int)((L.n_brows + 3) / 4);
            LAUNCH(h, bsr_fused_generic_kernel, grid, 128, 0, a, h->b);
        }
    }
    CU(cudaGetLastError());
    return MG_OK;
}

int spmv(mg_handle *h, const Level &L, const double *x, double *y, const int *done = nullptr) {
    BsrArgs a{};
    a.mode = MODE_SPMV;
    a.vin = x;
    a.out = y;
    a.done = done;
    return launch_bsr(h, L, a);
}
int residual(mg_handle *h, const Level &L, const double *rhs, const double *x, double *r, const int *done = nullptr) {
    BsrArgs a{};
    a.mode = MODE_RESID;
    a.vin = x;
    a.rin = rhs;
    a.out = r;
    a.done = done;
    return launch_bsr(h, L, a);
}
// dout = c_z * Dinv rin ; if xacc: xacc += dout
int pbj(mg_handle *h, const Level &L, const double *rin, double *dout, double c_z, double *xacc = nullptr,
        const int *done = nullptr) {
    BsrArgs a{};
    a.mode = MODE_PBJ;
    a.rin = rin;
    a.dout = dout;
    a.c_z = c_z;
    a.x = xacc;
    a.flags = xacc ? F_FINAL_X : 0;
    a.done = done;
    return launch_bsr(h, L, a);
}
int sweep(mg_handle *h, const Level &L, const double *vin, const double *rin, double *rout, double *x, double *dout,
          double c_d, double c_z, int flags) {
    BsrArgs a{};
    a.mode = MODE_SWEEP;
    a.vin = vin;
    a.rin = rin;
    a.out = rout;
    a.x = x;
    a.dout = dout;
    a.c_d = c_d;
    a.c_z = c_z;
    a.flags = flags;
    return launch_bsr(h, L, a);
}

// ------------------------------------------------------------------------------------------------ line blocks (NEXT-4)
inline bool line_mode(const mg_handle *h, const Level &L) { return h->opt.smoother == 2 && L.line_ready; }

// dout = c_d dold + c_z M_line^-1 rin ; if xacc: xacc += dout.   dout must differ from rin and dold.
int line_apply(mg_handle *h, const Level &L, const double *rin, const double *dold, double *dout, double c_d, double c_z,
               double *xacc = nullptr) {
    if (L.n_brows == 0) return MG_OK;
    KindScope scope(h, L.index, MG_KIND_LINE);
    LineArgs a{};
    a.vals = L.vals;
    a.lpos = L.lpos;
    a.G = L.lineG;
    a.W = L.lineW;
    a.rin = rin;
    a.dold = dold;
    a.dout = dout;
    a.x = xacc;
    a.c_d = c_d;
    a.c_z = c_z;
    a.n_pol = h->n_pol;
    a.N = L.n_phi;
    a.b = h->b;
    a.done = nullptr;
    const size_t smem = line_staged_smem(a.b, a.N);
    if (a.b % 4 == 0 && smem <= 200 * 1024 && h->opt.kernel_variant == 0) {   // blocks staged through shared memory by bulk copies
        if (smem > 48 * 1024 && smem > h->line_smem_set) {
            CU(cudaFuncSetAttribute(line_apply_staged_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            h->line_smem_set = smem;
        }
        LAUNCH(h, line_apply_staged_kernel, h->n_pol, (4 * a.b + 31) / 32 * 32, smem, a);
    } else {
        LAUNCH(h, line_apply_kernel, (h->n_pol + LINE_WARPS - 1) / LINE_WARPS, LINE_WARPS * 32, 0, a);
    }
    CU(cudaGetLastError());
    return MG_OK;
}

// Positions (once) and factorisation (setup and every refresh) of the line blocks of one level.
int setup_level_line(mg_handle *h, Level &L) {
    const int b = h->b, N = L.n_phi;
    const size_t bb = (size_t)b * b;
    L.line_ready = false;
    if (L.n_brows == 0) return MG_OK;
    if (L.lpos == nullptr) {
        MG(dalloc_t(h, &L.lpos, 3 * (size_t)L.n_brows));
        MG(dalloc_t(h, &L.lineG, (size_t)h->n_pol * N * bb));
        MG(dalloc_t(h, &L.lineW, (size_t)h->n_pol * std::max(N - 1, 1) * bb));
        int *bad = nullptr;
        MG(dalloc_t(h, &bad, 4));
        CU(cudaMemsetAsync(bad, 0, sizeof(int), h->stream));
        LAUNCH(h, line_positions_kernel, grid_for(L.n_brows, 256, 1 << 30), 256, 0, L.row_ptr, L.col_idx, h->n_pol, N, L.lpos, bad);
        int hbad = 0;
        CU(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        dfree_t(h, bad);
        if (hbad) return MG_EINVAL;   // a node couples itself beyond the neighbouring planes: not a tridiagonal line block
    }
    const size_t smem = sizeof(double) * (7 * bb + b);
    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(line_factor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU(cudaMemsetAsync(L.err_flag, 0xff, sizeof(unsigned long long), h->stream));
    LAUNCH(h, line_factor_kernel, (unsigned)h->n_pol, 128, smem, L.vals, L.lpos, h->n_pol, N, b, L.lineG, L.lineW, L.err_flag);
    CU(cudaGetLastError());
    unsigned long long herr = 0;
    CU(cudaMemcpyAsync(&herr, L.err_flag, sizeof(herr), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (herr != ~0ull) return MG_ESINGULAR;
    L.line_ready = true;
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ reductions
// out[0] = <a, b> via the handle's scratch reduction (device result).
int dot_dev(mg_handle *h, const double *a, const double *b, int64_t n, double *out) {
    const int grid = grid_for(n / 2 + 1, 256 * 4, 1024);
    LAUNCH(h, dot_multi_kernel, dim3(grid, 1), 256, 0, a, (int64_t)0, b, n, h->red_partial, h->red_counter, out,
           (const int *)nullptr);
    CU(cudaGetLastError());
    return MG_OK;
}
int dot_host(mg_handle *h, const double *a, const double *b, int64_t n, double *result) {
    MG(dot_dev(h, a, b, n, h->red_out));
    CU(cudaMemcpyAsync(h->pinned_d, h->red_out, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    *result = h->pinned_d[0];
    return MG_OK;
}
int scale_div(mg_handle *h, const double *src, double *dst, int64_t n, const double *denom, const int *done) {
    LAUNCH(h, scale_div_kernel, grid_for(n, 256), 256, 0, src, dst, n, denom, done);
    CU(cudaGetLastError());
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ smoothers
struct Cheb {
    double theta, delta, sigma1;
};
inline Cheb cheb_of(const Level &L) {
    Cheb c;
    c.theta = 0.5 * (L.lam_max + L.lam_min);
    c.delta = 0.5 * (L.lam_max - L.lam_min);
    c.sigma1 = c.theta / c.delta;
    return c;
}

// nu >= 0 sweeps from a zero guess: x = x_nu, L.r = rhs - A x_nu (the residual carried by the recurrence).
int presmooth(mg_handle *h, Level &L, const double *rhs, double *x, int nu) {
    const size_t bytes = (size_t)L.nvec * sizeof(double);
    if (nu <= 0) {
        CU(cudaMemsetAsync(x, 0, bytes, h->stream));
        CU(cudaMemcpyAsync(L.r, rhs, bytes, cudaMemcpyDeviceToDevice, h->stream));
        return MG_OK;
    }
    const Cheb c = cheb_of(L);
    if (line_mode(h, L)) {   // the same recurrence with D := the toroidal-line blocks; their solve is a kernel of its own
        MG(line_apply(h, L, rhs, nullptr, L.d[0], 0.0, 1.0 / c.theta));
        double rho = 1.0 / c.sigma1;
        for (int k = 0; k < nu; ++k) {
            const double rho_new = 1.0 / (2.0 * c.sigma1 - rho);
            MG(sweep(h, L, L.d[k & 1], k == 0 ? rhs : L.r, L.r, x, nullptr, 0.0, 0.0, (k == 0) ? F_SET_X : F_UPD_X));
            if (k < nu - 1) MG(line_apply(h, L, L.r, L.d[k & 1], L.d[(k + 1) & 1], rho_new * rho, 2.0 * rho_new / c.delta));
            rho = rho_new;
        }
        return MG_OK;
    }
    MG(pbj(h, L, rhs, L.d[0], 1.0 / c.theta));  // d_0 = D^-1 r_0 / theta, r_0 = rhs
    double rho = 1.0 / c.sigma1;
    for (int k = 0; k < nu; ++k) {
        const double rho_new = 1.0 / (2.0 * c.sigma1 - rho);
        int flags = (k == 0) ? F_SET_X : F_UPD_X;
        if (k < nu - 1) flags |= F_NEED_D;
        MG(sweep(h, L, L.d[k & 1], k == 0 ? rhs : L.r, L.r, x, L.d[(k + 1) & 1], rho_new * rho, 2.0 * rho_new / c.delta,
                 flags));
        rho = rho_new;
    }
    return MG_OK;
}

// nu >= 1 sweeps from the guess x whose residual update is L.r - A v (v = correction just added to x, or x itself
// with L.r = rhs).  v must not alias x.
int postsmooth(mg_handle *h, Level &L, const double *v, double *x, int nu) {
    if (nu <= 0) return MG_OK;
    const Cheb c = cheb_of(L);
    if (line_mode(h, L)) {
        MG(sweep(h, L, v, L.r, L.r, x, nullptr, 0.0, 0.0, 0));   // r -= A v
        MG(line_apply(h, L, L.r, nullptr, L.d[0], 0.0, 1.0 / c.theta, nu == 1 ? x : nullptr));
        double rho = 1.0 / c.sigma1;
        for (int k = 0; k + 1 < nu; ++k) {
            const double rho_new = 1.0 / (2.0 * c.sigma1 - rho);
            MG(sweep(h, L, L.d[k & 1], L.r, L.r, x, nullptr, 0.0, 0.0, F_UPD_X));
            MG(line_apply(h, L, L.r, L.d[k & 1], L.d[(k + 1) & 1], rho_new * rho, 2.0 * rho_new / c.delta, k == nu - 2 ? x : nullptr));
            rho = rho_new;
        }
        return MG_OK;
    }
    MG(sweep(h, L, v, L.r, L.r, x, L.d[0], 0.0, 1.0 / c.theta, F_NEED_D | (nu == 1 ? F_FINAL_X : 0)));
    double rho = 1.0 / c.sigma1;
    for (int k = 0; k + 1 < nu; ++k) {
        const double rho_new = 1.0 / (2.0 * c.sigma1 - rho);
        const int flags = F_UPD_X | F_NEED_D | (k == nu - 2 ? F_FINAL_X : 0);
        MG(sweep(h, L, L.d[k & 1], L.r, L.r, x, L.d[(k + 1) & 1], rho_new * rho, 2.0 * rho_new / c.delta, flags));
        rho = rho_new;
    }
    return MG_OK;
}

int restrict_to(mg_handle *h, int l, const double *rf, double *rc) {
    const Level &L = h->lev[l];
    const int64_t plane = (int64_t)h->n_pol * h->b;
    KindScope scope(h, l, MG_KIND_RESTRICT);
    LAUNCH(h, restrict_kernel, grid_for(plane * (L.n_phi / 2), 256), 256, 0, rf, rc, plane, L.n_phi, (const int *)nullptr);
    CU(cudaGetLastError());
    return MG_OK;
}
int prolong_add(mg_handle *h, int l, const double *ec, double *xf, double *pe) {
    const Level &L = h->lev[l];
    const int64_t plane = (int64_t)h->n_pol * h->b;
    KindScope scope(h, l, MG_KIND_PROLONG);
    LAUNCH(h, prolong_add_kernel, grid_for(plane * L.n_phi, 256), 256, 0, ec, xf, pe, plane, L.n_phi, (const int *)nullptr);
    CU(cudaGetLastError());
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ GMRES engine
// Frees the buffers of a previous gmres_alloc (restart length or iteration cap changed): without this every change of
// `restart` / `maxit` leaked a whole Krylov basis until mg_destroy.
void gmres_release(mg_handle *h, Gmres &G) {
    if (!G.ready) return;
    cudaStreamSynchronize(h->stream);   // kernels in flight may still use the old buffers
    dfree_t(h, G.V);
    dfree_t(h, G.Z);
    dfree_t(h, G.partial);
    dfree_t(h, G.counter);
    GmresDev &d = G.dev;
    dfree_t(h, d.H);
    dfree_t(h, d.cs);
    dfree_t(h, d.sn);
    dfree_t(h, d.g);
    dfree_t(h, d.y);
    dfree_t(h, d.h1);
    dfree_t(h, d.h2);
    dfree_t(h, d.nrm2);
    dfree_t(h, d.hnext);
    dfree_t(h, d.tol);
    dfree_t(h, d.hist);
    dfree_t(h, d.status);
    dfree_t(h, G.orth_partial);
    dfree_t(h, G.orth_nrm);
    dfree_t(h, G.orth_counter);
    G.ready = false;
}

int gmres_alloc(mg_handle *h, Gmres &G, int64_t n, int m, int maxit, bool flexible) {
    if (G.ready && G.n == n && G.m == m && G.flexible == flexible) {   // only the iteration cap changed: the history buffer
        dfree_t(h, G.dev.hist);
        G.maxit = maxit;
        G.dev.maxit = maxit;
        MG(dalloc_t(h, &G.dev.hist, (size_t)maxit + 2));
        return MG_OK;
    }
    gmres_release(h, G);
    G.n = n;
    G.m = m;
    G.maxit = maxit;
    G.flexible = flexible;
    G.stride = (n + 31) / 32 * 32;
    G.red_grid = grid_for(n / 2 + 1, 256 * 4, 256);
    MG(dalloc_t(h, &G.V, (size_t)G.stride * (m + 1)));
    if (flexible) MG(dalloc_t(h, &G.Z, (size_t)G.stride * m));
    const int axpy_grid = (int)((n / 2 + 256) / 256);
    MG(dalloc_t(h, &G.partial, (size_t)std::max((m + 1) * G.red_grid, axpy_grid)));
    MG(dalloc_t(h, &G.counter, (size_t)(m + 2)));
    CU(cudaMemsetAsync(G.counter, 0, sizeof(unsigned) * (m + 2), h->stream));
    GmresDev &d = G.dev;
    d.m = m;
    d.maxit = maxit;
    MG(dalloc_t(h, &d.H, (size_t)(m + 1) * m));
    MG(dalloc_t(h, &d.cs, (size_t)m));
    MG(dalloc_t(h, &d.sn, (size_t)m));
    MG(dalloc_t(h, &d.g, (size_t)m + 1));
    MG(dalloc_t(h, &d.y, (size_t)m));
    MG(dalloc_t(h, &d.h1, (size_t)m + 1));
    MG(dalloc_t(h, &d.h2, (size_t)m + 1));
    MG(dalloc_t(h, &d.nrm2, 1));
    MG(dalloc_t(h, &d.hnext, 1));
    MG(dalloc_t(h, &d.tol, 1));
    MG(dalloc_t(h, &d.hist, (size_t)maxit + 2));
    MG(dalloc_t(h, &d.status, 8));
    CU(cudaMemsetAsync(d.status, 0, 8 * sizeof(int), h->stream));
    // fused CGS2 step: one persistent CTA per SM, the slice of w (and as many basis slices as fit) in shared memory
    G.fused_ok = false;
    if (h->coop_ok && n > 0) {
        const size_t budget = 220 * 1024;
        G.orth_grid = (int)std::min<int64_t>(std::min(h->sm_count, ORTH_MAX_GRID), (n + 1) / 2);
        G.orth_slice = (int)(((n + G.orth_grid - 1) / G.orth_grid + 1) / 2 * 2);
        G.orth_grid = (int)((n + G.orth_slice - 1) / G.orth_slice);
        G.orth_ld = (m + 2) / 2 * 2;
        if (orth_smem_bytes(G.orth_slice, G.orth_ld, 0) <= budget) {
            const size_t left = budget - orth_smem_bytes(G.orth_slice, G.orth_ld, 0);
            G.orth_cap = (int)std::min<size_t>(left / (sizeof(double) * G.orth_slice), (size_t)m + 1);
            G.orth_smem = orth_smem_bytes(G.orth_slice, G.orth_ld, G.orth_cap);
            MG(dalloc_t(h, &G.orth_partial, (size_t)ORTH_REPLICAS * G.orth_grid * G.orth_ld));
            MG(dalloc_t(h, &G.orth_nrm, (size_t)G.orth_grid));
            MG(dalloc_t(h, &G.orth_counter, 2));
            CU(cudaMemsetAsync(G.orth_counter, 0, 2 * sizeof(unsigned), h->stream));
            G.fused_ok = true;
        }
    }
    G.ready = true;
    return MG_OK;
}

// tol = rtol * ||rhs||, iteration counters reset.
int gmres_start(mg_handle *h, Gmres &G, const double *rhs, double rtol) {
    KindScope scope(h, G.level, MG_KIND_ORTH);
    LAUNCH(h, dot_multi_kernel, dim3(G.red_grid, 1), 256, 0, rhs, (int64_t)0, rhs, G.n, G.partial, G.counter,
           G.dev.nrm2, (const int *)nullptr);
    LAUNCH(h, gmres_set_tol_kernel, 1, 1, 0, G.dev, rtol);
    CU(cudaGetLastError());
    return MG_OK;
}
// V[0] holds the residual r: beta = ||r||, stop test, g = beta e_1, V[0] /= beta.
int gmres_cycle_begin(mg_handle *h, Gmres &G, bool normalize = true) {
    KindScope scope(h, G.level, MG_KIND_ORTH);
    const int *done = G.dev.status;
    LAUNCH(h, dot_multi_kernel, dim3(G.red_grid, 1), 256, 0, G.V, (int64_t)0, G.V, G.n, G.partial, G.counter, G.dev.nrm2,
           done);
    LAUNCH(h, gmres_begin_kernel, 1, 1, 0, G.dev);
    if (normalize) MG(scale_div(h, G.V, G.V, G.n, G.dev.hnext, done));
    return MG_OK;
}
// V[j+1] holds w = A M v_j: two classical Gram-Schmidt passes against V[0..j]; the tail of the second update
// kernel does the Hessenberg column / Givens / stop test.  normalize: v_{j+1} = w / h_{j+1,j} here (otherwise the
// caller folds the division into its next kernel).
#ifndef MG_DEFER_GIVENS
#define MG_DEFER_GIVENS 1
#endif
int join_side_branch(mg_handle *h) {
    if (h->join_pending) {
        CU(cudaStreamWaitEvent(h->stream, h->ev_join, 0));
        h->join_pending = false;
    }
    return MG_OK;
}
int gmres_orth(mg_handle *h, Gmres &G, int j, bool normalize = true, double *w_override = nullptr, bool defer_update = false) {
    KindScope scope(h, G.level, MG_KIND_ORTH);
    const int *done = G.dev.status;
    double *w = w_override ? w_override : G.V + (size_t)(j + 1) * G.stride;
    if (G.fused_ok && h->opt.kernel_variant == 0) {
        OrthArgs oa{};
        oa.V = G.V;
        oa.stride = G.stride;
        oa.j = j;
        oa.w = w;
        oa.n = G.n;
        oa.partial = G.orth_partial;
        oa.nrm_partial = G.orth_nrm;
        oa.counter = G.orth_counter;
        oa.dev = G.dev;
        oa.done = done;
        oa.slice = G.orth_slice;
        oa.cap = G.orth_cap;
        oa.ld = G.orth_ld;
        oa.eta2 = h->opt.orth_eta * h->opt.orth_eta;
        oa.defer_update = defer_update ? 1 : 0;
        void *params[] = {&oa};
        MG(join_side_branch(h));
        ProfPair pp;
        const bool prof = prof_begin(h, pp);
        CU(cudaLaunchCooperativeKernel((const void *)gmres_orth_fused_kernel, dim3(G.orth_grid), dim3(ORTH_THREADS), params,
                                       G.orth_smem, h->stream));
        if (prof) prof_end(h, pp);
        count_launch(h);
        if (defer_update) {  // column j's Givens / stop-test update: a one-warp kernel the next SpMV runs beside
            const size_t gsm = sizeof(double) * 3 * G.orth_ld;
            if (h->capturing) {   // a side branch of the captured graph, joined before the next Gram-Schmidt kernel
                if (!h->side_stream) {
                    CU(cudaStreamCreateWithFlags(&h->side_stream, cudaStreamNonBlocking));
                    CU(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
                    CU(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
                }
                CU(cudaEventRecord(h->ev_fork, h->stream));
                CU(cudaStreamWaitEvent(h->side_stream, h->ev_fork, 0));
                gmres_givens_kernel<<<1, 32, gsm, h->side_stream>>>(G.dev, j, G.orth_ld);
                count_launch(h);
                CU(cudaEventRecord(h->ev_join, h->side_stream));
                h->join_pending = true;
            } else {
                LAUNCH(h, gmres_givens_kernel, 1, 32, gsm, G.dev, j, G.orth_ld);
            }
        }
        if (normalize) MG(scale_div(h, w, w, G.n, G.dev.hnext, done));
        return MG_OK;
    }
    const int axpy_grid = (int)((G.n / 2 + 256) / 256);
    for (int pass = 0; pass < 2; ++pass) {
        double *hh = pass == 0 ? G.dev.h1 : G.dev.h2;
        LAUNCH(h, dot_multi_kernel, dim3(G.red_grid, j + 1), 256, 0, G.V, G.stride, w, G.n, G.partial, G.counter, hh,
               done);
        LAUNCH(h, axpy_multi_kernel, axpy_grid, 256, 0, G.V, G.stride, j + 1, (const int *)nullptr, hh, -1.0, w, G.n,
               G.partial, G.counter + G.m + 1, pass == 1 ? G.dev.nrm2 : (double *)nullptr, done, G.dev, pass == 1 ? j : -1);
    }
    if (normalize) MG(scale_div(h, w, w, G.n, G.dev.hnext, done));
    CU(cudaGetLastError());
    return MG_OK;
}
// y = H^-1 g ; out += sum_i y_i B_i  (B = Z for flexible, V otherwise)
int gmres_cycle_end(mg_handle *h, Gmres &G, double *out) {
    KindScope scope(h, G.level, MG_KIND_ORTH);
    LAUNCH(h, gmres_solve_y_kernel, 1, 32, 0, G.dev);
    const int axpy_grid = (int)((G.n / 2 + 256) / 256);
    LAUNCH(h, axpy_multi_kernel, axpy_grid, 256, 0, G.flexible ? G.Z : G.V, G.stride, G.m, G.dev.status + 1, G.dev.y, 1.0,
           out, G.n, G.partial, G.counter + G.m + 1, (double *)nullptr, (const int *)nullptr, G.dev, -1);
    CU(cudaGetLastError());
    return MG_OK;
}
int read_status(mg_handle *h, Gmres &G, int st[4]) {
    CU(cudaMemcpyAsync(h->pinned, G.dev.status, 4 * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    for (int i = 0; i < 4; ++i) st[i] = h->pinned[i];
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ coarse solve
// Fused coarse cycle (TMA kernel + fused CGS2): GMRES on the precomputed operator Ahat = A D^-1.  Two launches per
// Arnoldi step.  S[0], S[1] alternate as the unnormalised Arnoldi vector: the SpMV of step j gathers S[j&1], writes
// v_j = S[j&1] / h (the normalised basis vector) and S[(j+1)&1] = Ahat v_j; the CGS2 kernel orthogonalises
// S[(j+1)&1] against V_0..V_j in place and leaves h_{j+1,j} for the next division.
int coarse_cycle_enqueue_fused(mg_handle *h) {
    Level &L = h->lev.back();
    Gmres &G = h->coarse;
    const int *done = G.dev.status;
    MG(residual(h, L, L.rhs, L.x, h->coarse_stage[0], done));
    {
        KindScope scope(h, G.level, MG_KIND_ORTH);
        LAUNCH(h, dot_multi_kernel, dim3(G.red_grid, 1), 256, 0, h->coarse_stage[0], (int64_t)0, h->coarse_stage[0], G.n, G.partial,
               G.counter, G.dev.nrm2, done);
        LAUNCH(h, gmres_begin_kernel, 1, 1, 0, G.dev);
    }
    Level Lhat = L;            // same pattern and partition, values A D^-1
    Lhat.vals = h->coarse_ahat;
    for (int j = 0; j < G.m; ++j) {
        double *sj = h->coarse_stage[j & 1], *sn = h->coarse_stage[(j + 1) & 1];
        BsrArgs a{};
        a.mode = MODE_SPMV;
        a.vin = sj;
        a.out = sn;
        a.done = done;
        TmaExtra ex{};
        ex.scale_div = G.dev.hnext;
        ex.vout = G.V + (size_t)j * G.stride;
        // the Givens / stop-test update of column j-1 is deferred to a one-warp kernel on a side branch of the graph: this SpMV
        // runs beside it (measured on C1: 119.9 -> 117.1 us per step, same counts; as a programmatic dependent launch: 117.9)
        const bool defer = MG_DEFER_GIVENS && G.fused_ok && h->opt.kernel_variant == 0 && h->tma_ready && G.orth_ld <= 2048;
        if (defer && j > 0) a.done = done + 4;   // stable while the Givens kernel of column j-1 runs (GmresDev::status)
        MG(launch_bsr(h, Lhat, a, ex));
        MG(gmres_orth(h, G, j, false, sn, defer));
    }
    MG(join_side_branch(h));
    CU(cudaMemsetAsync(L.d[1], 0, (size_t)L.nvec * sizeof(double), h->stream));
    MG(gmres_cycle_end(h, G, L.d[1]));
    MG(pbj(h, L, L.d[1], L.d[0], 1.0, L.x));  // e += D^-1 (V y)
    return MG_OK;
}

int coarse_cycle_enqueue(mg_handle *h) {
    Level &L = h->lev.back();
    Gmres &G = h->coarse;
    const int *done = G.dev.status;
    if (h->coarse_ahat != nullptr && h->opt.kernel_variant == 0 && G.fused_ok) return coarse_cycle_enqueue_fused(h);
    MG(residual(h, L, L.rhs, L.x, G.V, done));
    MG(gmres_cycle_begin(h, G, true));
    for (int j = 0; j < G.m; ++j) {
        MG(pbj(h, L, G.V + (size_t)j * G.stride, L.d[0], 1.0, nullptr, done));
        MG(spmv(h, L, L.d[0], G.V + (size_t)(j + 1) * G.stride, done));
        MG(gmres_orth(h, G, j, true));
    }
    CU(cudaMemsetAsync(L.d[1], 0, (size_t)L.nvec * sizeof(double), h->stream));
    MG(gmres_cycle_end(h, G, L.d[1]));
    MG(pbj(h, L, L.d[1], L.d[0], 1.0, L.x));  // e += D^-1 (V y)
    return MG_OK;
}

// Ahat = A D^-1 of the coarsest level (values only; the pattern is A's).
int refresh_coarse_ahat(mg_handle *h) {
    Level &L = h->lev.back();
    if (h->coarse_ahat == nullptr || L.nnzb == 0) return MG_OK;
    const int b = h->b;
    LAUNCH(h, right_scale_blocks_kernel, (unsigned)L.nnzb, 256, sizeof(double) * 2 * b * b, L.col_idx, L.vals, L.dinv,
           h->coarse_ahat, b);
    CU(cudaGetLastError());
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ direct coarse solve
// Symbolic part (once per hierarchy): BFS level sets of the coarsest level's block graph, permutation, dense storage.
int direct_symbolic(mg_handle *h) {
    Level &L = h->lev.back();
    DirectCoarse &dc = h->direct;
    const int b = h->b;
    const int64_t n = L.n_brows;
    if (n <= 0 || n > (int64_t)1 << 30) return MG_EINVAL;
    if (L.h_row_ptr.empty()) {
        L.h_row_ptr.resize((size_t)n + 1);
        L.h_col_idx.resize((size_t)L.nnzb);
        CU(cudaMemcpyAsync(L.h_row_ptr.data(), L.row_ptr, sizeof(int64_t) * (n + 1), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(L.h_col_idx.data(), L.col_idx, sizeof(int32_t) * L.nnzb, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    // BFS from `start`; returns the level of every block row (every component is appended after the previous ones)
    auto bfs = [&](int64_t start, std::vector<int> &lvl) {
        lvl.assign((size_t)n, -1);
        int maxl = 0;
        int64_t last = start;
        std::queue<int64_t> q;
        auto run = [&](int64_t s0, int l0) {
            lvl[s0] = l0;
            q.push(s0);
            while (!q.empty()) {
                const int64_t u = q.front();
                q.pop();
                last = u;
                maxl = std::max(maxl, lvl[u]);
                for (int64_t p = L.h_row_ptr[u]; p < L.h_row_ptr[u + 1]; ++p) {
                    const int64_t v = L.h_col_idx[p];
                    if (lvl[v] < 0) {
                        lvl[v] = lvl[u] + 1;
                        q.push(v);
                    }
                }
            }
        };
        run(start, 0);
        for (int64_t s0 = 0; s0 < n; ++s0)
            if (lvl[s0] < 0) run(s0, maxl + 2);   // another component: its own level sets, never adjacent to the previous ones
        return last;
    };
    std::vector<int> lvl;
    const int64_t far = bfs(0, lvl);
    bfs(far, lvl);   // pseudo-peripheral start: narrower level sets
    // compress level numbers (gaps between components) and order rows by level
    std::vector<int> used;
    {
        std::vector<int> sorted(lvl);
        std::sort(sorted.begin(), sorted.end());
        sorted.erase(std::unique(sorted.begin(), sorted.end()), sorted.end());
        used = sorted;
    }
    dc.nlev = (int)used.size();
    std::vector<int32_t> lev_of_old((size_t)n), perm((size_t)n), inv((size_t)n), lev_new((size_t)n), off((size_t)dc.nlev + 1, 0);
    for (int64_t i = 0; i < n; ++i) lev_of_old[i] = (int32_t)(std::lower_bound(used.begin(), used.end(), lvl[i]) - used.begin());
    for (int64_t i = 0; i < n; ++i) off[lev_of_old[i] + 1]++;
    for (int k = 0; k < dc.nlev; ++k) off[k + 1] += off[k];
    {
        std::vector<int32_t> cur(off.begin(), off.end() - 1);
        for (int64_t i = 0; i < n; ++i) {   // stable within a level set: ascending old index
            const int32_t pnew = cur[lev_of_old[i]]++;
            perm[pnew] = (int32_t)i;
            inv[i] = pnew;
            lev_new[pnew] = lev_of_old[i];
        }
    }
    // every block must couple equal or adjacent level sets (true for a structurally symmetric pattern)
    for (int64_t i = 0; i < n; ++i)
        for (int64_t p = L.h_row_ptr[i]; p < L.h_row_ptr[i + 1]; ++p) {
            const int d = lev_of_old[L.h_col_idx[p]] - lev_of_old[i];
            if (d > 1 || d < -1) return MG_EINVAL;
        }
    // Two-sided elimination: level sets 0 .. mid-1 are eliminated upwards, nlev-1 .. mid+1 downwards, mid last.
    dc.mid = dc.nlev / 2;
    const int mid = dc.mid;
    // blocks by block column for the Schur updates: list 0 = (row one level set DOWN, i.e. U_{k-1}), 1 = (row one level set UP, L_{k+1})
    std::vector<int64_t> csc_ptr[2], csc_pos[2];
    for (int dir = 0; dir < 2; ++dir) {
        const int want = dir == 0 ? 1 : -1;   // lev(col) - lev(row)
        csc_ptr[dir].assign((size_t)n + 1, 0);
        for (int64_t i = 0; i < n; ++i)
            for (int64_t p = L.h_row_ptr[i]; p < L.h_row_ptr[i + 1]; ++p) {
                const int64_t j = L.h_col_idx[p];
                if (lev_of_old[j] - lev_of_old[i] == want) csc_ptr[dir][inv[j] + 1]++;
            }
        for (int64_t i = 0; i < n; ++i) csc_ptr[dir][i + 1] += csc_ptr[dir][i];
        csc_pos[dir].resize((size_t)std::max<int64_t>(csc_ptr[dir][n], 1));
        std::vector<int64_t> cur(csc_ptr[dir].begin(), csc_ptr[dir].end() - 1);
        for (int64_t i = 0; i < n; ++i)
            for (int64_t p = L.h_row_ptr[i]; p < L.h_row_ptr[i + 1]; ++p) {
                const int64_t j = L.h_col_idx[p];
                if (lev_of_old[j] - lev_of_old[i] == want) csc_pos[dir][cur[inv[j]]++] = p;
            }
    }
    // row-wise lists of the off-diagonal blocks for the solve: list 0 = elimination (columns in the level set eliminated just
    // before: k-1 below mid, k+1 above, both at mid), list 1 = back-substitution (the other neighbour; none at mid)
    std::vector<int64_t> od_ptr[2], od_pos[2];
    std::vector<int32_t> od_col[2];
    dc.offdiag_blocks = 0;
    for (int side = 0; side < 2; ++side) {
        od_ptr[side].assign((size_t)n + 1, 0);
        for (int64_t pn = 0; pn < n; ++pn) {
            const int64_t i = perm[pn];
            const int k = lev_of_old[i];
            for (int64_t p = L.h_row_ptr[i]; p < L.h_row_ptr[i + 1]; ++p) {
                const int64_t j = L.h_col_idx[p];
                const int d = lev_of_old[j] - k;
                if (d == 0) continue;
                const bool elim = (k < mid && d == -1) || (k > mid && d == 1) || k == mid;
                if ((side == 0) != elim) continue;
                od_pos[side].push_back(p);
                od_col[side].push_back(inv[j]);
            }
            od_ptr[side][pn + 1] = (int64_t)od_pos[side].size();
        }
        dc.offdiag_blocks += (int64_t)od_pos[side].size();
        if (od_pos[side].empty()) {
            od_pos[side].push_back(0);
            od_col[side].push_back(0);
        }
    }
    // steps of the solve: elimination from both ends, the middle level set, back-substitution outwards
    dc.steps.clear();
    {
        const int q = dc.nlev - 1;
        for (int j = 0; j < std::max(mid, q - mid); ++j) {
            std::vector<DirectCoarse::Job> st;
            if (j < mid) st.push_back({j, 0, 0});
            if (q - j > mid) st.push_back({q - j, 0, 0});
            dc.steps.push_back(st);
        }
        dc.steps.push_back({{mid, 0, 1}});
        for (int j = 1; j <= std::max(mid, q - mid); ++j) {
            std::vector<DirectCoarse::Job> st;
            if (mid - j >= 0) st.push_back({mid - j, 1, 1});
            if (mid + j <= q) st.push_back({mid + j, 1, 1});
            dc.steps.push_back(st);
        }
    }
    dc.nk.resize(dc.nlev);
    dc.voff.assign(dc.nlev + 1, 0);
    dc.maxn = 0;
    int64_t bytes = 0, mtmp = 1;
    for (int k = 0; k < dc.nlev; ++k) {
        dc.nk[k] = (off[k + 1] - off[k]) * b;
        dc.voff[k + 1] = dc.voff[k] + dc.nk[k];
        dc.maxn = std::max(dc.maxn, dc.nk[k]);
        bytes += (int64_t)sizeof(double) * dc.nk[k] * dc.nk[k];
    }
    for (int k = 1; k < dc.nlev; ++k) mtmp = std::max(mtmp, (int64_t)dc.nk[k] * dc.nk[k - 1]);
    bytes += (int64_t)sizeof(double) * mtmp;
    size_t free_b = 0, total_b = 0;
    CU(cudaMemGetInfo(&free_b, &total_b));
    if ((double)bytes > 0.9 * (double)free_b) return MG_ENOMEM;
    dc.bytes = bytes;
    dc.S.assign(dc.nlev, nullptr);
    for (int k = 0; k < dc.nlev; ++k) MG(dalloc_t(h, &dc.S[k], (size_t)dc.nk[k] * dc.nk[k]));
    MG(dalloc_t(h, &dc.Mtmp, (size_t)mtmp));
    MG(dalloc_t(h, &dc.perm, (size_t)n));
    MG(dalloc_t(h, &dc.inv, (size_t)n));
    MG(dalloc_t(h, &dc.lev, (size_t)n));
    MG(dalloc_t(h, &dc.off, (size_t)dc.nlev + 1));
    MG(dalloc_t(h, &dc.dS, (size_t)dc.nlev));
    for (int side = 0; side < 2; ++side) {
        MG(dalloc_t(h, &dc.csc_ptr[side], (size_t)n + 1));
        MG(dalloc_t(h, &dc.csc_pos[side], csc_pos[side].size()));
        CU(cudaMemcpyAsync(dc.csc_ptr[side], csc_ptr[side].data(), sizeof(int64_t) * (n + 1), cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemcpyAsync(dc.csc_pos[side], csc_pos[side].data(), sizeof(int64_t) * csc_pos[side].size(), cudaMemcpyHostToDevice,
                           h->stream));
        MG(dalloc_t(h, &dc.od_ptr[side], (size_t)n + 1));
        MG(dalloc_t(h, &dc.od_pos[side], od_pos[side].size()));
        MG(dalloc_t(h, &dc.od_col[side], od_col[side].size()));
        CU(cudaMemcpyAsync(dc.od_ptr[side], od_ptr[side].data(), sizeof(int64_t) * (n + 1), cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemcpyAsync(dc.od_pos[side], od_pos[side].data(), sizeof(int64_t) * od_pos[side].size(), cudaMemcpyHostToDevice,
                           h->stream));
        CU(cudaMemcpyAsync(dc.od_col[side], od_col[side].data(), sizeof(int32_t) * od_col[side].size(), cudaMemcpyHostToDevice,
                           h->stream));
    }
    MG(dalloc_t(h, &dc.zb, (size_t)L.nvec + 2));
    MG(dalloc_t(h, &dc.yb, (size_t)L.nvec + 2));
    MG(dalloc_t(h, &dc.tb, (size_t)2 * dc.maxn + 2));
    MG(dalloc_t(h, &dc.pinv, (size_t)GJ_W * GJ_W));
    MG(dalloc_t(h, &dc.cpanel, (size_t)dc.maxn * GJ_W + 2));
    MG(dalloc_t(h, &dc.rpanel, (size_t)dc.maxn * GJ_W + 2));
    MG(dalloc_t(h, &dc.bad, 4));
    CU(cudaMemcpyAsync(dc.perm, perm.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(dc.inv, inv.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(dc.lev, lev_new.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(dc.off, off.data(), sizeof(int32_t) * (dc.nlev + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(dc.dS, dc.S.data(), sizeof(double *) * dc.nlev, cudaMemcpyHostToDevice, h->stream));
    if (L.row_of_block != nullptr) dc.rob = L.row_of_block;
    else {
        MG(dalloc_t(h, &dc.rob, (size_t)std::max<int64_t>(L.nnzb, 1)));
        LAUNCH(h, rows_of_blocks_kernel, grid_for(n, 256, 1 << 30), 256, 0, L.row_ptr, n, dc.rob);
    }
    // persistent solve kernel: needs 16-byte aligned rows (b even), b <= 64, ELL width <= DS_MAXNE, t and >= DS_PL ring stages
    // in shared memory, and the packed stages of one step of one CTA must fit the ring together
    dc.first.assign(off.begin(), off.end());
    dc.persist = false;
    {
        std::vector<int> lev_ne((size_t)2 * dc.nlev, 0);
        std::vector<long long> lev_off((size_t)2 * dc.nlev, 0);
        int ne_max = 0;
        for (int side = 0; side < 2; ++side)
            for (int64_t pn = 0; pn < n; ++pn) {
                const int cnt = (int)(od_ptr[side][pn + 1] - od_ptr[side][pn]);
                int &m = lev_ne[2 * lev_new[pn] + side];
                m = std::max(m, cnt);
                ne_max = std::max(ne_max, cnt);
            }
        long long ell_doubles = 0;
        for (int k = 0; k < dc.nlev; ++k)
            for (int side = 0; side < 2; ++side) {
                lev_off[2 * k + side] = ell_doubles;
                ell_doubles += (long long)dc.nk[k] * lev_ne[2 * k + side] * b;
            }
        const int nsteps = (int)dc.steps.size();
        int tcap = 2;
        for (const auto &st : dc.steps) {
            int nt = 0;
            for (const auto &j : st) nt += dc.nk[j.level];
            tcap = std::max(tcap, (nt + 1) / 2 * 2);
        }
        const size_t budget = 227 * 1024;
        // (level sets so wide that the t of a step leaves fewer than DS_PL ring stages -- C3: 2 x 8,496 scalars -- take the
        // launch chain: measured 10.06 ms against 10.32 ms per C3 coarse solve for a persistent variant with one job's t at a time)
        int stages = 0;
        if (direct_smem_bytes(DS_PL, tcap, nsteps) <= budget)
            stages = (int)std::min<size_t>(64, (budget - direct_smem_bytes(0, tcap, nsteps)) /
                                                   (sizeof(double) * DS_SEG + 2 * sizeof(uint64_t) + sizeof(int)));
        bool fits = (b % 2 == 0) && b >= DS_TPR && b <= 64 && ne_max <= DS_MAXNE && stages >= DS_PL && h->coop_launch;
        for (int k = 0; fits && k < dc.nlev; ++k)   // the packed stages of one pass of phase (A) are handed back together
            for (int side = 0; side < 2; ++side) {
                const int rowlen = lev_ne[2 * k + side] * b;
                if (rowlen == 0) continue;
                const int rps = DS_SEG / rowlen, rpp = DS_WARPS * 32 / DS_TPR;
                if (rps < 1 || (rpp + rps - 1) / rps + 2 > stages - 1) fits = false;
            }
        int per_sm = 0;
        if (fits &&
            cudaFuncSetAttribute(direct_solve_persistent_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)direct_smem_bytes(stages, tcap, nsteps)) == cudaSuccess &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, direct_solve_persistent_kernel, DS_THREADS,
                                                          direct_smem_bytes(stages, tcap, nsteps)) == cudaSuccess && per_sm >= 1) {
            dc.ds_stages = stages;
            dc.ds_tcap = tcap;
            dc.ds_smem = direct_smem_bytes(stages, tcap, nsteps);
            dc.ds_grid = h->sm_count;
            dc.ell_doubles = ell_doubles;
            MG(dalloc_t(h, &dc.stepdev, (size_t)nsteps));
            MG(dalloc_t(h, &dc.ell, (size_t)std::max<long long>(ell_doubles, 2)));
            MG(dalloc_t(h, &dc.ell_col, (size_t)2 * n * DS_MAXNE));
            MG(dalloc_t(h, &dc.lev_ne, (size_t)2 * dc.nlev));
            MG(dalloc_t(h, &dc.lev_off, (size_t)2 * dc.nlev));
            std::vector<DsStepDesc> sd((size_t)nsteps);
            std::memset(sd.data(), 0, sizeof(DsStepDesc) * sd.size());
            int64_t toff = 0;
            for (int si = 0; si < nsteps; ++si)
                for (size_t ji = 0; ji < 2; ++ji) {
                    if (ji >= dc.steps[si].size()) {
                        sd[si].j[ji].toff = (int)toff;
                        continue;
                    }
                    const auto &j = dc.steps[si][ji];
                    DsJob &J = sd[si].j[ji];
                    J.S = dc.S[j.level];
                    J.ell_off = lev_off[2 * j.level + j.phase];
                    J.n = dc.nk[j.level];
                    J.first = off[j.level];
                    J.ne = lev_ne[2 * j.level + j.phase];
                    J.phase = j.phase;
                    J.final = j.final;
                    J.toff = (int)toff;
                    toff += J.n;
                }
            dc.tb_doubles = toff;
            dc.xchg_doubles = 2 * (int64_t)L.nvec + toff;
            MG(dalloc_t(h, &dc.xchg, (size_t)dc.xchg_doubles + 2));
            CU(cudaMemcpyAsync(dc.stepdev, sd.data(), sizeof(DsStepDesc) * nsteps, cudaMemcpyHostToDevice, h->stream));
            CU(cudaMemcpyAsync(dc.lev_ne, lev_ne.data(), sizeof(int) * 2 * dc.nlev, cudaMemcpyHostToDevice, h->stream));
            CU(cudaMemcpyAsync(dc.lev_off, lev_off.data(), sizeof(long long) * 2 * dc.nlev, cudaMemcpyHostToDevice, h->stream));
            CU(cudaStreamSynchronize(h->stream));
            dc.persist = true;
        } else {
            cudaGetLastError();
        }
    }
    CU(cudaStreamSynchronize(h->stream));   // the host vectors above are locals
    dc.symbolic = true;
    return MG_OK;
}

int dense_inverse_inplace(mg_handle *h, double *A, int n) {
    DirectCoarse &dc = h->direct;
    for (int p0 = 0; p0 < n; p0 += GJ_W) {
        const int w = std::min(GJ_W, n - p0);
        LAUNCH(h, gj_panel_inverse_kernel, 1, GJ_W * GJ_W, 0, A, n, p0, w, dc.pinv, dc.bad);
        LAUNCH(h, gj_row_panel_kernel, (n + 255) / 256, 256, 0, A, n, p0, w, dc.pinv, dc.cpanel, dc.rpanel);
        LAUNCH(h, gj_update_kernel, dim3((n + 63) / 64, (n + 63) / 64), 256, 0, A, n, p0, w, dc.cpanel, dc.rpanel);
    }
    CU(cudaGetLastError());
    return MG_OK;
}

int direct_solve(mg_handle *h, const double *rhs, double *e);

// Numeric part (setup and every refresh): assemble the dense diagonal blocks, then S_k = D_k - (L_k S_{k-1}^-1) U_{k-1}
// and its inverse, level set by level set.
int direct_numeric(mg_handle *h) {
    Level &L = h->lev.back();
    DirectCoarse &dc = h->direct;
    KindScope scope(h, L.index, MG_KIND_OTHER);
    const int b = h->b;
    for (int k = 0; k < dc.nlev; ++k) CU(cudaMemsetAsync(dc.S[k], 0, sizeof(double) * (size_t)dc.nk[k] * dc.nk[k], h->stream));
    CU(cudaMemsetAsync(dc.bad, 0, sizeof(int), h->stream));
    DirectTables t{dc.perm, dc.inv, dc.lev, dc.off, dc.dS};
    if (L.nnzb > 0) LAUNCH(h, direct_assemble_kernel, (unsigned)L.nnzb, 128, 0, dc.rob, L.col_idx, L.vals, b, t);
    CU(cudaGetLastError());
    // S_k -= (blocks of level set k with columns in kp) S_kp^-1 (blocks with rows in kp and columns in k); S_kp^-1 is final
    auto schur_update = [&](int k, int kp) -> int {
        const int nk = dc.nk[k], np = dc.nk[kp];
        const int dir = kp < k ? 0 : 1;
        LAUNCH(h, direct_lsinv_kernel, dim3((np + 127) / 128, nk / b), 128, 0, L.row_ptr, L.col_idx, L.vals, b, t, k, kp, dc.S[kp], np,
               dc.Mtmp);
        LAUNCH(h, direct_schur_kernel, dim3(nk / b, (nk + 31) / 32), 128, 0, dc.csc_ptr[dir], dc.csc_pos[dir], dc.rob, L.vals, b, t, k, kp,
               dc.Mtmp, np, dc.S[k], nk);
        CU(cudaGetLastError());
        return MG_OK;
    };
    for (int k = 0; k < dc.mid; ++k) {            // lower chain, upwards
        if (k > 0) MG(schur_update(k, k - 1));
        MG(dense_inverse_inplace(h, dc.S[k], dc.nk[k]));
    }
    for (int k = dc.nlev - 1; k > dc.mid; --k) {  // upper chain, downwards
        if (k < dc.nlev - 1) MG(schur_update(k, k + 1));
        MG(dense_inverse_inplace(h, dc.S[k], dc.nk[k]));
    }
    if (dc.mid > 0) MG(schur_update(dc.mid, dc.mid - 1));
    if (dc.mid < dc.nlev - 1) MG(schur_update(dc.mid, dc.mid + 1));
    MG(dense_inverse_inplace(h, dc.S[dc.mid], dc.nk[dc.mid]));
    if (dc.persist) {   // off-diagonal block rows in the level-set ordering, one contiguous span per level set and side
        LAUNCH(h, direct_pack_ell_kernel, dim3((unsigned)L.n_brows, 2), 128, 0, dc.od_ptr[0], dc.od_pos[0], dc.od_col[0], dc.od_ptr[1],
               dc.od_pos[1], dc.od_col[1], L.vals, b, dc.lev, dc.off, dc.lev_ne, dc.lev_off, dc.ell, dc.ell_col, L.n_brows);
        CU(cudaGetLastError());
    }
    int bad = 0;
    CU(cudaMemcpyAsync(&bad, dc.bad, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (bad == 2) return MG_ESINGULAR;
    dc.numeric = true;
    // The Schur complements are inverted WITHOUT pivoting (fine for operators with a positive definite symmetric part, which
    // the Galerkin hierarchy of the paper's elliptic systems has): one probe solve checks the factorisation, so that a small
    // pivot on some other operator is an error code and not a silently inaccurate coarse solve.
    {
        LAUNCH(h, hashed_start_kernel, grid_for(L.nvec, 256), 256, 0, L.d[0], L.nvec);
        const int rc = direct_solve(h, L.d[0], L.d[1]);
        if (rc != MG_OK) { dc.numeric = false; return rc; }
        MG(residual(h, L, L.d[0], L.d[1], L.pe));
        double rr = 0.0, bb = 0.0;
        MG(dot_host(h, L.pe, L.pe, L.nvec, &rr));
        MG(dot_host(h, L.d[0], L.d[0], L.nvec, &bb));
        if (!(rr <= 1e-12 * bb)) {   // relative residual above 1e-6 (or NaN)
            dc.numeric = false;
            return MG_ESINGULAR;
        }
    }
    return MG_OK;
}

// e = A_c^-1 rhs by block forward / backward substitution: dense mat-vec streaming of the S_k^-1 interleaved with the
// sparse off-diagonal products, no host synchronisation.
int direct_solve(mg_handle *h, const double *rhs, double *e) {
    Level &L = h->lev.back();
    DirectCoarse &dc = h->direct;
    KindScope scope(h, L.index, MG_KIND_DIRECT);
    const int b = h->b;
    if (dc.persist && h->opt.kernel_variant == 0) {
        DirectSolveArgs a{};
        a.steps = dc.stepdev;
        a.nsteps = (int)dc.steps.size();
        a.b = b;
        a.ell = dc.ell;
        a.ell_col = dc.ell_col;
        a.n_brows = L.n_brows;
        a.perm = dc.perm;
        a.rhs = rhs;
        a.e = e;
        a.yb = dc.xchg;
        a.xb = dc.xchg + L.nvec;
        a.tb = dc.xchg + 2 * L.nvec;
        a.stages = dc.ds_stages;
        a.tcap = dc.ds_tcap;
        CU(cudaMemsetAsync(dc.xchg, 0xff, sizeof(double) * (size_t)dc.xchg_doubles, h->stream));   // the sentinel: all ones
        void *params[] = {&a};
        ProfPair pp;
        const bool prof = prof_begin(h, pp);
        CU(cudaLaunchCooperativeKernel((const void *)direct_solve_persistent_kernel, dim3(dc.ds_grid), dim3(DS_THREADS), params,
                                       dc.ds_smem, h->stream));
        if (prof) prof_end(h, pp);
        count_launch(h);
        return MG_OK;
    }
    // launch chain: the same steps, one job after the other (jobs of a step are independent)
    LAUNCH_PDL(h, permute_blocks_kernel, grid_for(L.nvec, 256, 1 << 30), 256, 0, rhs, dc.zb, dc.perm, L.n_brows, b, 0);
    for (const auto &st : dc.steps)
        for (const auto &j : st) {
            const int k = j.level, nk = dc.nk[k];
            if (j.phase == 0) {   // y_k = S_k^-1 (z_k - X y)
                LAUNCH_PDL(h, direct_offdiag_kernel, (nk + 3) / 4, 128, 0, dc.od_ptr[0], dc.od_pos[0], dc.od_col[0], L.vals, b, dc.voff[k] / b,
                           nk, dc.yb, dc.zb + dc.voff[k], dc.tb, -1.0);
                LAUNCH_PDL(h, dense_gemv_kernel, (nk + GEMV_ROWS - 1) / GEMV_ROWS, 256, 0, dc.S[k], dc.tb, (const double *)nullptr,
                           dc.yb + dc.voff[k], nk, nk, 1.0);
            } else {              // x_k = y_k - S_k^-1 (X x); the solution is built in place in yb
                LAUNCH_PDL(h, direct_offdiag_kernel, (nk + 3) / 4, 128, 0, dc.od_ptr[1], dc.od_pos[1], dc.od_col[1], L.vals, b, dc.voff[k] / b,
                           nk, dc.yb, (const double *)nullptr, dc.tb, 1.0);
                LAUNCH_PDL(h, dense_gemv_kernel, (nk + GEMV_ROWS - 1) / GEMV_ROWS, 256, 0, dc.S[k], dc.tb, dc.yb + dc.voff[k],
                           dc.yb + dc.voff[k], nk, nk, -1.0);
            }
        }
    LAUNCH_PDL(h, permute_blocks_kernel, grid_for(L.nvec, 256, 1 << 30), 256, 0, dc.yb, e, dc.perm, L.n_brows, b, 1);
    CU(cudaGetLastError());
    return MG_OK;
}

// Solve A_{L-1} x = rhs on the coarsest level's own buffers (L.rhs -> L.x), zero guess.
int coarse_solve_internal(mg_handle *h) {
    Level &L = h->lev.back();
    if (h->opt.coarse_mode == 2) {
        if (!h->direct.symbolic) MG(direct_symbolic(h));
        if (!h->direct.numeric) MG(direct_numeric(h));
        h->coarse_iters_last = 0;
        return direct_solve(h, L.rhs, L.x);
    }
    if (h->opt.coarse_mode == 1) {
        h->coarse_iters_last = h->opt.coarse_fixed_sweeps;
        h->coarse_iters_total += h->coarse_iters_last;
        return presmooth(h, L, L.rhs, L.x, h->opt.coarse_fixed_sweeps);
    }
    Gmres &G = h->coarse;
    if (!G.ready || G.m != h->opt.coarse_restart || G.maxit != h->opt.coarse_maxit) {
        if (h->coarse_graph) {
            cudaGraphExecDestroy(h->coarse_graph);
            h->coarse_graph = nullptr;
        }
        MG(gmres_alloc(h, G, L.nvec, h->opt.coarse_restart, h->opt.coarse_maxit, false));
        G.level = L.index;
        if (h->tma_ready && L.part != nullptr && G.fused_ok && h->coarse_ahat == nullptr && L.nnzb > 0) {
            const int b = h->b;
            MG(dalloc_t(h, &h->coarse_ahat, (size_t)L.nnzb * b * b));
            MG(dalloc_t(h, &h->coarse_stage[0], (size_t)L.nvec + 2));
            MG(dalloc_t(h, &h->coarse_stage[1], (size_t)L.nvec + 2));
            MG(refresh_coarse_ahat(h));
        }
    }
    CU(cudaMemsetAsync(L.x, 0, (size_t)L.nvec * sizeof(double), h->stream));
    MG(gmres_start(h, G, L.rhs, h->opt.coarse_rtol));
    const bool use_graph = h->opt.use_graphs && !h->profiling;
    for (int attempt = 0; use_graph && !h->coarse_graph && attempt < 2; ++attempt) {
        cudaGraph_t graph = nullptr;
        if (!h->cap_stream) CU(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
        cudaStream_t user_stream = h->stream;
        CU(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
        h->stream = h->cap_stream;
        h->capturing = true;
        h->join_pending = false;   // (a failed earlier attempt may have left its side branch open)
        h->capture_count = 0;
        std::memset(h->graph_hist, 0, sizeof(h->graph_hist));
        const int rc = coarse_cycle_enqueue(h);
        h->capturing = false;
        h->stream = user_stream;
        cudaError_t e = cudaStreamEndCapture(h->cap_stream, &graph);
        if (e == cudaSuccess && rc == MG_OK) {
            h->coarse_graph_kernels = h->capture_count;
            e = cudaGraphInstantiate(&h->coarse_graph, graph, 0);
        }
        if (graph) cudaGraphDestroy(graph);
        if (e == cudaSuccess && rc == MG_OK) break;
        cudaGetLastError();
        h->coarse_graph = nullptr;
        if (attempt == 0 && G.fused_ok) {  // a cooperative node the graph cannot hold: capture the four-kernel CGS2 instead
            G.fused_ok = false;
            continue;
        }
        if (rc != MG_OK) return rc;
        return cuda_fail(e, "capture of the coarse GMRES cycle");
    }
    int st[4] = {0, 0, 0, 0};
    do {
        if (use_graph) {
            CU(cudaGraphLaunch(h->coarse_graph, h->stream));
            h->launches += h->coarse_graph_kernels;
            for (int lv = 0; lv < MG_PROFILE_MAX_LEVELS; ++lv)
                for (int k = 0; k < MG_KIND_COUNT; ++k) h->prof[lv][k].launches += h->graph_hist[lv][k];
        } else {
            MG(coarse_cycle_enqueue(h));
        }
        MG(read_status(h, G, st));
    } while (!st[0]);
    h->coarse_iters_last = st[2];
    h->coarse_iters_total += st[2];
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ GMRES smoother
// The paper's level smoother (App. B 421-424): nu iterations of GMRES preconditioned (on the right) with
// PBJ, no convergence test, no restart: x <- argmin ||rhs - A x|| over x0 + D^-1 K_nu(A D^-1, r0).  Everything stays on
// the device: the Arnoldi/Givens state is GmresDev, the tolerance is 0, nothing is read back.
int gmres_smooth(mg_handle *h, Level &L, const double *rhs, double *x, int nu, bool zero_guess) {
    const size_t bytes = (size_t)L.nvec * sizeof(double);
    if (zero_guess) CU(cudaMemsetAsync(x, 0, bytes, h->stream));
    if (nu <= 0 || L.nvec == 0) return MG_OK;
    if ((int)h->smooth_g.size() != h->n_levels) h->smooth_g.resize(h->n_levels);
    Gmres &G = h->smooth_g[L.index];
    if (!G.ready || G.m < nu) {
        const int m = std::max(nu, std::max(h->opt.nu_pre, h->opt.nu_post));
        MG(gmres_alloc(h, G, L.nvec, m, m, false));  // maxit = m: the stop flag can only rise after the last step
        G.level = L.index;
    }
    const int *done = G.dev.status;
    MG(gmres_start(h, G, rhs, 0.0));
    if (zero_guess) CU(cudaMemcpyAsync(G.V, rhs, bytes, cudaMemcpyDeviceToDevice, h->stream));
    else MG(residual(h, L, rhs, x, G.V));
    MG(gmres_cycle_begin(h, G, true));
    for (int j = 0; j < nu; ++j) {
        MG(pbj(h, L, G.V + (size_t)j * G.stride, L.d[0], 1.0, nullptr, done));
        MG(spmv(h, L, L.d[0], G.V + (size_t)(j + 1) * G.stride, done));
        MG(gmres_orth(h, G, j, true));
    }
    CU(cudaMemsetAsync(L.d[1], 0, bytes, h->stream));
    MG(gmres_cycle_end(h, G, L.d[1]));
    MG(pbj(h, L, L.d[1], L.d[0], 1.0, x));  // x += D^-1 (V y)
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ V-cycle
int vcycle_internal(mg_handle *h, const double *r, double *z) {
    const int Lc = h->n_levels - 1;
    if (Lc == 0) {
        Level &L = h->lev[0];
        CU(cudaMemcpyAsync(L.rhs, r, (size_t)L.nvec * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
        MG(coarse_solve_internal(h));
        CU(cudaMemcpyAsync(z, L.x, (size_t)L.nvec * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
        return MG_OK;
    }
    const bool gsm = (h->opt.smoother == 1);
    for (int l = 0; l < Lc; ++l) {
        Level &L = h->lev[l];
        const double *rhs = (l == 0) ? r : L.rhs;
        double *x = (l == 0) ? z : L.x;
        if (gsm) {
            MG(gmres_smooth(h, L, rhs, x, h->opt.nu_pre, true));
            MG(residual(h, L, rhs, x, L.r));
        } else {
            MG(presmooth(h, L, rhs, x, h->opt.nu_pre));
        }
        MG(restrict_to(h, l, L.r, h->lev[l + 1].rhs));
    }
    MG(coarse_solve_internal(h));
    for (int l = Lc - 1; l >= 0; --l) {
        Level &L = h->lev[l];
        double *x = (l == 0) ? z : L.x;
        if (gsm) {
            MG(prolong_add(h, l, h->lev[l + 1].x, x, nullptr));
            MG(gmres_smooth(h, L, (l == 0) ? r : L.rhs, x, h->opt.nu_post, false));
        } else {
            MG(prolong_add(h, l, h->lev[l + 1].x, x, h->opt.nu_post > 0 ? L.pe : nullptr));
            MG(postsmooth(h, L, L.pe, x, h->opt.nu_post));
        }
    }
    return MG_OK;
}

// ------------------------------------------------------------------------------------------------ setup pieces
int power_rho(mg_handle *h, Level &L, int iters, double *rho_out) {
    LAUNCH(h, hashed_start_kernel, grid_for(L.nvec, 256), 256, 0, L.x, L.nvec);
    double nrm2 = 0.0;
    MG(dot_host(h, L.x, L.x, L.nvec, &nrm2));
    if (!(nrm2 > 0.0)) {
        *rho_out = 1.0;
        return MG_OK;
    }
    LAUNCH(h, axpby_kernel, grid_for(L.nvec, 256), 256, 0, 1.0 / std::sqrt(nrm2), L.x, 0.0, L.x, L.nvec);
    double rho = 0.0;
    L.rho_is_line = line_mode(h, L);
    for (int it = 0; it < iters; ++it) {
        MG(spmv(h, L, L.x, L.r));
        if (L.rho_is_line) MG(line_apply(h, L, L.r, nullptr, L.d[0], 0.0, 1.0));
        else MG(pbj(h, L, L.r, L.d[0], 1.0));
        MG(dot_host(h, L.d[0], L.d[0], L.nvec, &nrm2));
        rho = std::sqrt(nrm2);
        if (!(rho > 0.0)) break;
        LAUNCH(h, axpby_kernel, grid_for(L.nvec, 256), 256, 0, 1.0 / rho, L.d[0], 0.0, L.x, L.nvec);
    }
    CU(cudaGetLastError());
    *rho_out = rho;
    return MG_OK;
}

void set_bounds(mg_handle *h, Level &L) {
    L.lam_min = h->opt.cheb_lo * L.rho_est;
    L.lam_max = h->opt.cheb_hi * L.rho_est;
}

// Host symbolic phase of the Galerkin product: the coarse pattern in closed form from the fine pattern.
void galerkin_symbolic(const Level &F, int n_pol, std::vector<int64_t> &crow_ptr, std::vector<int32_t> &ccol,
                       std::vector<int64_t> &crow_of_block) {
    const int n_f = F.n_phi, n_c = n_f / 2;
    crow_ptr.assign((size_t)n_c * n_pol + 1, 0);
    ccol.clear();
    crow_of_block.clear();
    std::vector<int64_t> cand;
    for (int K = 0; K < n_c; ++K) {
        int ks[3] = {(2 * K - 1 + n_f) % n_f, 2 * K, (2 * K + 1) % n_f};
        int nk = 0, kk[3];
        for (int a = 0; a < 3; ++a) {
            bool dup = false;
            for (int a2 = 0; a2 < nk; ++a2) dup |= (kk[a2] == ks[a]);
            if (!dup) kk[nk++] = ks[a];
        }
        for (int i = 0; i < n_pol; ++i) {
            cand.clear();
            for (int a = 0; a < nk; ++a) {
                const int64_t If = (int64_t)kk[a] * n_pol + i;
                for (int64_t p = F.h_row_ptr[If]; p < F.h_row_ptr[If + 1]; ++p) {
                    const int64_t J = F.h_col_idx[p];
                    const int m = (int)(J / n_pol);
                    const int64_t j = J % n_pol;
                    if ((m & 1) == 0) {
                        cand.push_back((int64_t)(m / 2) * n_pol + j);
                    } else {
                        cand.push_back((int64_t)((m - 1) / 2) * n_pol + j);
                        cand.push_back((int64_t)(((m + 1) / 2) % n_c) * n_pol + j);
                    }
                }
            }
            std::sort(cand.begin(), cand.end());
            cand.erase(std::unique(cand.begin(), cand.end()), cand.end());
            const int64_t Ic = (int64_t)K * n_pol + i;
            for (int64_t c : cand) {
                ccol.push_back((int32_t)c);
                crow_of_block.push_back(Ic);
            }
            crow_ptr[Ic + 1] = (int64_t)ccol.size();
        }
    }
}

// TMA kernel (b = 36): contiguous row ranges with equal block counts, one per persistent CTA.
int setup_level_partition(mg_handle *h, Level &L) {
    if (!h->tma_ready || L.n_brows == 0) return MG_OK;
    L.tma_grid = (int)std::min<int64_t>(h->sm_count, L.n_brows);
    MG(dalloc_t(h, &L.part, 2 * ((size_t)L.tma_grid + 1)));
    // equal block counts per CTA (a row may straddle two CTAs) when every CTA's range holds at least two whole rows;
    // otherwise row-aligned ranges
    int *d_max = nullptr;
    MG(dalloc_t(h, &d_max, 4));
    CU(cudaMemsetAsync(d_max, 0, sizeof(int), h->stream));
    LAUNCH(h, max_row_blocks_kernel, grid_for(L.n_brows, 256, 1024), 256, 0, L.row_ptr, L.n_brows, d_max);
    int hmax = 0;
    CU(cudaMemcpyAsync(&hmax, d_max, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    const int split = (hmax > 0 && L.nnzb / L.tma_grid >= 3 * (int64_t)hmax) ? 1 : 0;
    LAUNCH(h, partition_rows_kernel, (L.tma_grid + 1 + 127) / 128, 128, 0, L.row_ptr, L.n_brows, L.nnzb, L.tma_grid, split, L.part);
    CU(cudaGetLastError());
    if (h->frag_part == nullptr) {
        MG(dalloc_t(h, &h->frag_part, (size_t)h->sm_count * TmaCfg::B));
        MG(dalloc_t(h, &h->frag_flag, (size_t)h->sm_count));
        CU(cudaMemsetAsync(h->frag_flag, 0, sizeof(int) * h->sm_count, h->stream));
    }
    return MG_OK;
}

int alloc_level_vectors(mg_handle *h, Level &L) {
    const size_t n = (size_t)L.nvec + 2;
    MG(dalloc_t(h, &L.x, n));
    MG(dalloc_t(h, &L.r, n));
    MG(dalloc_t(h, &L.d[0], n));
    MG(dalloc_t(h, &L.d[1], n));
    MG(dalloc_t(h, &L.pe, n));
    MG(dalloc_t(h, &L.rhs, n));
    return MG_OK;
}

int invert_level_blocks(mg_handle *h, Level &L);

int setup_level_pbj(mg_handle *h, Level &L) {
    const int b = h->b;
    MG(dalloc_t(h, &L.diag_pos, (size_t)L.n_brows));
    unsigned long long *err = nullptr;
    MG(dalloc_t(h, &err, 2));
    CU(cudaMemsetAsync(err, 0xff, 2 * sizeof(unsigned long long), h->stream));
    LAUNCH(h, check_pattern_kernel, grid_for(L.n_brows, 256, 1 << 30), 256, 0, L.row_ptr, L.col_idx, L.n_brows, L.diag_pos,
           err, err + 1);
    unsigned long long herr[2];
    CU(cudaMemcpyAsync(herr, err, sizeof(herr), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (herr[0] != ~0ull) return MG_EINVAL;
    if (herr[1] != ~0ull) return MG_ESINGULAR;
    MG(dalloc_t(h, &L.dinv, (size_t)L.n_brows * b * b));
    MG(dalloc_t(h, &L.err_flag, 1));
    return invert_level_blocks(h, L);
}

// Batched inverse of the diagonal blocks of one level into L.dinv; MG_ESINGULAR on a zero pivot.
int invert_level_blocks(mg_handle *h, Level &L) {
    const int b = h->b;
    unsigned long long *err = L.err_flag;
    unsigned long long herr[1];
    CU(cudaMemsetAsync(err, 0xff, sizeof(unsigned long long), h->stream));
    const size_t smem = sizeof(double) * (size_t)(2 * b * b + b);
    if (smem > 48 * 1024)
        CU(cudaFuncSetAttribute(invert_blocks_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (L.n_brows > 0) LAUNCH(h, invert_blocks_kernel, (unsigned)L.n_brows, 128, smem, L.vals, L.diag_pos, b, L.dinv, err);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(herr, err, sizeof(herr), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (herr[0] != ~0ull) return MG_ESINGULAR;
    return MG_OK;
}

// Numeric phase of A_{l+1} = P^T A_l P into the existing pattern of level l+1 (mg_setup and mg_update_values).
int galerkin_numeric(mg_handle *h, int l) {
    Level &F = h->lev[l];
    Level &C = h->lev[l + 1];
    if (C.nnzb > 0)
        LAUNCH(h, galerkin_numeric_kernel, (unsigned)C.nnzb, 128, 0, F.row_ptr, F.col_idx, F.vals, C.row_of_block, C.col_idx,
               const_cast<double *>(C.vals), h->n_pol, F.n_phi, h->b);
    CU(cudaGetLastError());
    return MG_OK;
}

int build_coarse_level(mg_handle *h, int l) {
    Level &F = h->lev[l];
    Level &C = h->lev[l + 1];
    const int b = h->b;
    if (F.h_row_ptr.empty()) {
        F.h_row_ptr.resize((size_t)F.n_brows + 1);
        F.h_col_idx.resize((size_t)F.nnzb);
        CU(cudaMemcpyAsync(F.h_row_ptr.data(), F.row_ptr, sizeof(int64_t) * (F.n_brows + 1), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(F.h_col_idx.data(), F.col_idx, sizeof(int32_t) * F.nnzb, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    std::vector<int64_t> crow_of_block;
    galerkin_symbolic(F, h->n_pol, C.h_row_ptr, C.h_col_idx, crow_of_block);
    C.n_phi = F.n_phi / 2;
    C.n_brows = (int64_t)C.n_phi * h->n_pol;
    C.nvec = C.n_brows * b;
    C.nnzb = (int64_t)C.h_col_idx.size();
    int64_t *d_rp = nullptr, *d_rob = nullptr;
    int32_t *d_ci = nullptr;
    double *d_v = nullptr;
    MG(dalloc_t(h, &d_rp, (size_t)C.n_brows + 1));
    MG(dalloc_t(h, &d_ci, (size_t)C.nnzb));
    MG(dalloc_t(h, &d_v, (size_t)C.nnzb * b * b));
    MG(dalloc_t(h, &d_rob, (size_t)std::max<int64_t>(C.nnzb, 1)));
    CU(cudaMemcpyAsync(d_rp, C.h_row_ptr.data(), sizeof(int64_t) * (C.n_brows + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(d_ci, C.h_col_idx.data(), sizeof(int32_t) * C.nnzb, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(d_rob, crow_of_block.data(), sizeof(int64_t) * C.nnzb, cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));  // crow_of_block is a local
    C.row_ptr = d_rp;
    C.col_idx = d_ci;
    C.vals = d_v;
    C.row_of_block = d_rob;
    return galerkin_numeric(h, l);
}

bool level_ok(mg_handle *h, int level) { return h && level >= 0 && level < h->n_levels; }
// Vectors and matrix arrays must be 16-byte aligned: the TMA kernels issue bulk copies from them (a misaligned pointer
// would be a device fault, not an error code).
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

// ================================================================================================ C ABI
extern "C" {

int mg_options_default(mg_options *o) {
    if (!o) return MG_EINVAL;
    std::memset(o, 0, sizeof(*o));
    o->nu_pre = 2;
    o->nu_post = 2;
    o->cheb_lo = 0.1;
    o->cheb_hi = 1.1;
    o->eig_iters = 20;
    o->coarse_mode = 0;
    o->coarse_rtol = 1e-10;
    o->coarse_restart = 100;
    o->coarse_maxit = 20000;
    o->coarse_fixed_sweeps = 8;
    o->restart = 100;
    o->maxit = 400;
    o->use_graphs = 1;
    o->kernel_variant = 0;
    o->smoother = 0;
    o->orth_eta = 0.25;
    return MG_OK;
}

size_t mg_sizeof_options(void) { return sizeof(mg_options); }
size_t mg_sizeof_solve_info(void) { return sizeof(mg_solve_info); }

static int validate_options(const mg_options &o) {
    if (o.nu_pre < 0 || o.nu_post < 0 || o.eig_iters < 1) return MG_EINVAL;
    if (!(o.cheb_lo > 0.0) || !(o.cheb_hi > o.cheb_lo)) return MG_EINVAL;
    if (o.coarse_mode < 0 || o.coarse_mode > 2 || !(o.coarse_rtol > 0.0)) return MG_EINVAL;
    if (o.coarse_restart < 1 || o.coarse_maxit < 1 || o.coarse_fixed_sweeps < 0) return MG_EINVAL;
    if (o.restart < 1 || o.maxit < 1) return MG_EINVAL;
    if (o.kernel_variant < 0 || o.kernel_variant > 1) return MG_EINVAL;
    if (o.smoother < 0 || o.smoother > 2) return MG_EINVAL;
    if (!(o.orth_eta >= 0.0) || o.orth_eta >= 1.0) return MG_EINVAL;
    return MG_OK;
}

int mg_destroy(mg_handle *h) {
    if (!h) return MG_EINVAL;
    cudaStreamSynchronize(h->stream);
    if (h->coarse_graph) cudaGraphExecDestroy(h->coarse_graph);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->side_stream) cudaStreamDestroy(h->side_stream);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    for (const ProfPair &pp : h->prof_pending) {
        cudaEventDestroy(pp.e0);
        cudaEventDestroy(pp.e1);
    }
    for (cudaEvent_t e : h->prof_free) cudaEventDestroy(e);
    for (cudaEvent_t e : h->ev_solve)
        if (e) cudaEventDestroy(e);
    for (void *p : h->owned) {
        if (h->opt.free) h->opt.free(p, h->opt.alloc_ctx);
        else if (!h->opt.alloc) cudaFree(p);
    }
    if (h->pinned) cudaFreeHost(h->pinned);
    if (h->pinned_d) cudaFreeHost(h->pinned_d);
    delete h;
    return MG_OK;
}

int mg_setup(mg_handle **out, const int64_t *row_ptr, const int32_t *col_idx, const double *vals, int b, int n_pol,
             int n_phi, int levels, const mg_options *opt, void *cuda_stream) {
    if (!out) return MG_EINVAL;
    *out = nullptr;
    if (!row_ptr || !col_idx || !vals || !aligned16(vals)) return MG_EINVAL;
    if (b < 1 || b > 64 || n_pol < 1 || n_phi < 1 || levels < 1 || levels > 30) return MG_EINVAL;
    if (opt && opt->smoother == 2 && b > 48) return MG_EINVAL;   // shared memory of the line factorisation
    if (n_phi % (1 << (levels - 1)) != 0) return MG_EINVAL;
    mg_options o;
    if (opt) o = *opt; else mg_options_default(&o);
    if (validate_options(o) != MG_OK) return MG_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g_last_cuda_error = "no CUDA device: libmgtoroidal has no CPU fallback";
        return MG_ECUDA;
    }
    mg_handle *h = new mg_handle();
    h->opt = o;
    h->b = b;
    h->n_pol = n_pol;
    h->n_phi = n_phi;
    h->n_levels = levels;
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    h->lev.resize(levels);
    for (int l = 0; l < levels; ++l) h->lev[l].index = l;
    int rc = MG_OK;
    auto fail = [&](int code) {
        mg_destroy(h);
        return code;
    };
    if (cudaMallocHost(&h->pinned, 8 * sizeof(int)) != cudaSuccess || cudaMallocHost(&h->pinned_d, 8 * sizeof(double)) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "cudaMallocHost"));
    if ((rc = dalloc_t(h, &h->red_partial, 2048)) != MG_OK) return fail(rc);
    if ((rc = dalloc_t(h, &h->red_out, 8)) != MG_OK) return fail(rc);
    if ((rc = dalloc_t(h, &h->red_counter, 8)) != MG_OK) return fail(rc);
    if (cudaMemsetAsync(h->red_counter, 0, 8 * sizeof(unsigned), h->stream) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "cudaMemsetAsync"));

    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            h->sm_count = sms;
        int coop = 0;
        if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop) h->coop_launch = true;
        if (h->coop_launch &&
            cudaFuncSetAttribute(gmres_orth_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) == cudaSuccess)
            h->coop_ok = true;
        else
            cudaGetLastError();
        if (b == TmaCfg::B) {
            if (cudaFuncSetAttribute(bsr_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TmaCfg::SMEM) != cudaSuccess)
                return fail(cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(bsr_tma_kernel)"));
            h->tma_ready = true;
        }
    }
    Level &L0 = h->lev[0];
    L0.n_phi = n_phi;
    L0.n_brows = (int64_t)n_pol * n_phi;
    L0.nvec = L0.n_brows * b;
    L0.row_ptr = row_ptr;
    L0.col_idx = col_idx;
    L0.vals = vals;
    int64_t ends[2] = {0, 0};
    if (cudaMemcpyAsync(&ends[0], row_ptr, sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(&ends[1], row_ptr + L0.n_brows, sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaStreamSynchronize(h->stream) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "read row_ptr"));
    if (ends[0] != 0 || ends[1] < L0.n_brows) return fail(MG_EINVAL);
    L0.nnzb = ends[1];

    for (int l = 0; l < levels; ++l) {
        Level &L = h->lev[l];
        if ((rc = setup_level_pbj(h, L)) != MG_OK) return fail(rc);
        if ((rc = setup_level_partition(h, L)) != MG_OK) return fail(rc);
        if ((rc = alloc_level_vectors(h, L)) != MG_OK) return fail(rc);
        if (o.smoother == 2 && l + 1 < levels && (rc = setup_level_line(h, L)) != MG_OK) return fail(rc);
        if ((rc = power_rho(h, L, o.eig_iters, &L.rho_est)) != MG_OK) return fail(rc);
        set_bounds(h, L);
        if (l + 1 < levels && (rc = build_coarse_level(h, l)) != MG_OK) return fail(rc);
    }
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "setup sync"));
    *out = h;
    return MG_OK;
}

int mg_update_options(mg_handle *h, const mg_options *opt) {
    if (!h || !opt) return MG_EINVAL;
    mg_options o = *opt;
    o.alloc = h->opt.alloc;
    o.free = h->opt.free;
    o.alloc_ctx = h->opt.alloc_ctx;
    o.eig_iters = h->opt.eig_iters;
    if (validate_options(o) != MG_OK) return MG_EINVAL;
    const bool bounds = (o.cheb_lo != h->opt.cheb_lo) || (o.cheb_hi != h->opt.cheb_hi);
    if ((o.kernel_variant != h->opt.kernel_variant || o.orth_eta != h->opt.orth_eta) && h->coarse_graph) {  // the captured cycle holds the old kernels
        cudaStreamSynchronize(h->stream);
        cudaGraphExecDestroy(h->coarse_graph);
        h->coarse_graph = nullptr;
    }
    if (o.smoother == 2 && h->b > 48) return MG_EINVAL;
    h->opt = o;
    // the Chebyshev interval belongs to the preconditioner (point or line blocks): re-estimate where it changed
    for (int l = 0; l + 1 < h->n_levels; ++l) {
        Level &L = h->lev[l];
        if (o.smoother == 2 && !L.line_ready) MG(setup_level_line(h, L));
        if (L.rho_is_line != (o.smoother == 2)) {
            MG(power_rho(h, L, o.eig_iters, &L.rho_est));
            set_bounds(h, L);
        }
    }
    if (bounds)
        for (auto &L : h->lev) set_bounds(h, L);
    return MG_OK;
}

int mg_update_values(mg_handle *h, const double *vals) {
    if (!h || !vals) return MG_EINVAL;
    if (!aligned16(vals)) return MG_EINVAL;
    if (h->coarse_graph && h->n_levels == 1) {   // the captured coarse cycle holds level 0's old (borrowed) values pointer
        cudaStreamSynchronize(h->stream);
        cudaGraphExecDestroy(h->coarse_graph);
        h->coarse_graph = nullptr;
    }
    h->lev[0].vals = vals;
    h->outer_vals = nullptr;
    for (int l = 0; l < h->n_levels; ++l) {
        Level &L = h->lev[l];
        MG(invert_level_blocks(h, L));
        L.line_ready = false;
        if (h->opt.smoother == 2 && l + 1 < h->n_levels) MG(setup_level_line(h, L));
        MG(power_rho(h, L, h->opt.eig_iters, &L.rho_est));
        set_bounds(h, L);
        if (l + 1 < h->n_levels) MG(galerkin_numeric(h, l));
    }
    MG(refresh_coarse_ahat(h));
    h->direct.numeric = false;   // the dense Schur inverses of the direct coarse solve are rebuilt on first use
    CU(cudaStreamSynchronize(h->stream));
    return MG_OK;
}

int mg_set_operator(mg_handle *h, const double *vals) {
    if (!h || !aligned16(vals)) return MG_EINVAL;
    h->outer_vals = vals;
    return MG_OK;
}

int mg_vcycle(mg_handle *h, const double *r, double *z) {
    if (!h || !r || !z || r == z || !aligned16(r) || !aligned16(z)) return MG_EINVAL;
    return vcycle_internal(h, r, z);
}

int mg_solve(mg_handle *h, const double *rhs, double *x, double rtol, int x_is_initial_guess, mg_solve_info *info) {
    if (!h || !rhs || !x || rhs == x || !(rtol > 0.0) || !aligned16(rhs) || !aligned16(x)) return MG_EINVAL;
    Level L = h->lev[0];  // the operator of the Krylov iteration: level 0's pattern with the current operator values
    L.h_row_ptr.clear();
    L.h_col_idx.clear();
    if (h->outer_vals != nullptr) L.vals = h->outer_vals;
    Gmres &G = h->outer;
    const int64_t n = L.nvec;
    const size_t bytes = (size_t)n * sizeof(double);
    if (!G.ready || G.m != h->opt.restart || G.maxit != h->opt.maxit)
        MG(gmres_alloc(h, G, n, h->opt.restart, h->opt.maxit, true));
    h->coarse_iters_total = 0;
    if (!h->ev_solve[0]) {
        CU(cudaEventCreate(&h->ev_solve[0]));
        CU(cudaEventCreate(&h->ev_solve[1]));
    }
    CU(cudaEventRecord(h->ev_solve[0], h->stream));
    if (!x_is_initial_guess) CU(cudaMemsetAsync(x, 0, bytes, h->stream));
    MG(gmres_start(h, G, rhs, rtol));
    CU(cudaMemcpyAsync(h->pinned_d, G.dev.nrm2, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    const double bnorm = std::sqrt(std::max(h->pinned_d[0], 0.0));
    int st[4] = {0, 0, 0, 0};
    if (bnorm == 0.0) {
        CU(cudaMemsetAsync(x, 0, bytes, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        if (info) {
            info->iters = 0;
            info->converged = 1;
            info->solve_ms = 0.0;
            info->rel_res = 0.0;
            info->coarse_iters_total = 0;
            if (info->hist && info->hist_len > 0) info->hist[0] = 0.0;
            info->hist_len = (info->hist && info->hist_len > 0) ? 1 : 0;
        }
        return MG_OK;
    }
    while (true) {
        MG(residual(h, L, rhs, x, G.V));
        MG(gmres_cycle_begin(h, G));
        MG(read_status(h, G, st));
        if (st[0]) break;
        for (int j = 0; j < G.m; ++j) {
            double *zj = G.Z + (size_t)j * G.stride;
            MG(vcycle_internal(h, G.V + (size_t)j * G.stride, zj));
            MG(spmv(h, L, zj, G.V + (size_t)(j + 1) * G.stride));
            MG(gmres_orth(h, G, j));
            MG(read_status(h, G, st));
            if (st[0]) break;
        }
        MG(gmres_cycle_end(h, G, x));
        if (st[0]) break;
    }
    // true residual
    MG(residual(h, L, rhs, x, L.r));
    double rn2 = 0.0;
    MG(dot_host(h, L.r, L.r, n, &rn2));
    CU(cudaEventRecord(h->ev_solve[1], h->stream));
    CU(cudaEventSynchronize(h->ev_solve[1]));
    float solve_ms = 0.f;
    CU(cudaEventElapsedTime(&solve_ms, h->ev_solve[0], h->ev_solve[1]));
    if (info) {
        info->solve_ms = solve_ms;
        info->iters = st[2];
        info->converged = st[3];
        info->rel_res = std::sqrt(std::max(rn2, 0.0)) / bnorm;
        info->coarse_iters_total = h->coarse_iters_total;
        int cnt = 0;
        if (info->hist && info->hist_len > 0) {
            cnt = std::min(info->hist_len, st[2] + 1);
            CU(cudaMemcpy(info->hist, G.dev.hist, sizeof(double) * cnt, cudaMemcpyDeviceToHost));
            for (int i = 0; i < cnt; ++i) info->hist[i] /= bnorm;
        }
        info->hist_len = cnt;
    }
    return MG_OK;
}

int mg_solve_host(mg_handle *h, const double *rhs_host, double *x_host, double rtol, int x_is_initial_guess,
                  mg_solve_info *info) {
    if (!h || !rhs_host || !x_host) return MG_EINVAL;
    Level &L = h->lev[0];
    const size_t bytes = (size_t)L.nvec * sizeof(double);
    if (!h->d_rhs_host) {
        MG(dalloc_t(h, &h->d_rhs_host, (size_t)L.nvec + 2));
        MG(dalloc_t(h, &h->d_x_host, (size_t)L.nvec + 2));
    }
    CU(cudaMemcpyAsync(h->d_rhs_host, rhs_host, bytes, cudaMemcpyHostToDevice, h->stream));
    if (x_is_initial_guess) CU(cudaMemcpyAsync(h->d_x_host, x_host, bytes, cudaMemcpyHostToDevice, h->stream));
    MG(mg_solve(h, h->d_rhs_host, h->d_x_host, rtol, x_is_initial_guess, info));
    CU(cudaMemcpyAsync(x_host, h->d_x_host, bytes, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return MG_OK;
}

int mg_spmv(mg_handle *h, int level, const double *x, double *y) {
    if (!level_ok(h, level) || !x || !y || x == y || !aligned16(x) || !aligned16(y)) return MG_EINVAL;
    return spmv(h, h->lev[level], x, y);
}

int mg_residual(mg_handle *h, int level, const double *rhs, const double *x, double *r) {
    if (!level_ok(h, level) || !rhs || !x || !r || x == r || !aligned16(rhs) || !aligned16(x) || !aligned16(r)) return MG_EINVAL;
    return residual(h, h->lev[level], rhs, x, r);
}

int mg_pbj_apply(mg_handle *h, int level, const double *r, double *z) {
    if (!level_ok(h, level) || !r || !z || !aligned16(r) || !aligned16(z)) return MG_EINVAL;
    return pbj(h, h->lev[level], r, z, 1.0);
}

int mg_smooth(mg_handle *h, int level, const double *rhs, double *x, int nu, int zero_guess) {
    if (!level_ok(h, level) || !rhs || !x || nu < 0 || rhs == x || !aligned16(rhs) || !aligned16(x)) return MG_EINVAL;
    Level &L = h->lev[level];
    if (h->opt.smoother == 1) return gmres_smooth(h, L, rhs, x, nu, zero_guess != 0);
    if (zero_guess) return presmooth(h, L, rhs, x, nu);
    if (nu == 0) return MG_OK;
    const size_t bytes = (size_t)L.nvec * sizeof(double);
    CU(cudaMemcpyAsync(L.pe, x, bytes, cudaMemcpyDeviceToDevice, h->stream));   // v = x_0 (gathered copy)
    CU(cudaMemcpyAsync(L.r, rhs, bytes, cudaMemcpyDeviceToDevice, h->stream));  // r = rhs, then r -= A x_0
    return postsmooth(h, L, L.pe, x, nu);
}

int mg_restrict(mg_handle *h, int level, const double *r_fine, double *r_coarse) {
    if (!level_ok(h, level) || level + 1 >= h->n_levels || !r_fine || !r_coarse) return MG_EINVAL;
    return restrict_to(h, level, r_fine, r_coarse);
}

int mg_prolong_add(mg_handle *h, int level, const double *e_coarse, double *x_fine) {
    if (!level_ok(h, level) || level + 1 >= h->n_levels || !e_coarse || !x_fine) return MG_EINVAL;
    return prolong_add(h, level, e_coarse, x_fine, nullptr);
}

int mg_coarse_solve(mg_handle *h, const double *r, double *e, int *iters) {
    if (!h || !r || !e || !aligned16(r) || !aligned16(e)) return MG_EINVAL;
    Level &L = h->lev.back();
    const size_t bytes = (size_t)L.nvec * sizeof(double);
    CU(cudaMemcpyAsync(L.rhs, r, bytes, cudaMemcpyDeviceToDevice, h->stream));
    MG(coarse_solve_internal(h));
    CU(cudaMemcpyAsync(e, L.x, bytes, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (iters) *iters = h->coarse_iters_last;
    return MG_OK;
}

int mg_direct_info(mg_handle *h, int *level_sets, int64_t *dense_bytes, int64_t *offdiag_bytes, int *max_n, int *persistent) {
    if (!h || !h->direct.symbolic) return MG_EINVAL;
    const DirectCoarse &dc = h->direct;
    int64_t dense = 0;
    for (int k = 0; k < dc.nlev; ++k) dense += (int64_t)sizeof(double) * dc.nk[k] * dc.nk[k];
    if (level_sets) *level_sets = dc.nlev;
    if (dense_bytes) *dense_bytes = dense;
    if (offdiag_bytes) *offdiag_bytes = dc.offdiag_blocks * (int64_t)sizeof(double) * h->b * h->b;   // (the packed copy is padded)
    if (max_n) *max_n = dc.maxn;
    if (persistent) *persistent = (dc.persist && h->opt.kernel_variant == 0) ? 1 : 0;
    return MG_OK;
}

int mg_get_level(mg_handle *h, int level, int64_t *n_brows, int64_t *nnzb, const int64_t **row_ptr,
                 const int32_t **col_idx, const double **vals, const double **dinv, double *rho_est, double *lam_min,
                 double *lam_max) {
    if (!level_ok(h, level)) return MG_EINVAL;
    const Level &L = h->lev[level];
    if (n_brows) *n_brows = L.n_brows;
    if (nnzb) *nnzb = L.nnzb;
    if (row_ptr) *row_ptr = L.row_ptr;
    if (col_idx) *col_idx = L.col_idx;
    if (vals) *vals = L.vals;
    if (dinv) *dinv = L.dinv;
    if (rho_est) *rho_est = L.rho_est;
    if (lam_min) *lam_min = L.lam_min;
    if (lam_max) *lam_max = L.lam_max;
    return MG_OK;
}

int mg_copy_level_to_host(mg_handle *h, int level, int64_t *row_ptr_host, int32_t *col_idx_host, double *vals_host,
                          double *dinv_host) {
    if (!level_ok(h, level)) return MG_EINVAL;
    const Level &L = h->lev[level];
    const size_t bb = (size_t)h->b * h->b;
    if (row_ptr_host)
        CU(cudaMemcpyAsync(row_ptr_host, L.row_ptr, sizeof(int64_t) * (L.n_brows + 1), cudaMemcpyDeviceToHost, h->stream));
    if (col_idx_host && L.nnzb > 0)
        CU(cudaMemcpyAsync(col_idx_host, L.col_idx, sizeof(int32_t) * L.nnzb, cudaMemcpyDeviceToHost, h->stream));
    if (vals_host && L.nnzb > 0)
        CU(cudaMemcpyAsync(vals_host, L.vals, sizeof(double) * L.nnzb * bb, cudaMemcpyDeviceToHost, h->stream));
    if (dinv_host && L.n_brows > 0)
        CU(cudaMemcpyAsync(dinv_host, L.dinv, sizeof(double) * L.n_brows * bb, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return MG_OK;
}

int mg_set_cheb_bounds(mg_handle *h, int level, double lam_min, double lam_max) {
    if (!level_ok(h, level) || !(lam_min > 0.0) || !(lam_max > lam_min)) return MG_EINVAL;
    h->lev[level].lam_min = lam_min;
    h->lev[level].lam_max = lam_max;
    return MG_OK;
}

int mg_profile_enable(mg_handle *h, int on) {
    if (!h) return MG_EINVAL;
    prof_flush(h);
    h->profiling = (on != 0);
    return MG_OK;
}

int mg_profile_reset(mg_handle *h) {
    if (!h) return MG_EINVAL;
    prof_flush(h);
    for (auto &row : h->prof)
        for (auto &a : row) a = ProfAcc();
    return MG_OK;
}

int mg_profile_get(mg_handle *h, int level, int kind, int64_t *launches, int64_t *timed, double *ms) {
    if (!h || level < 0 || level >= MG_PROFILE_MAX_LEVELS || kind < 0 || kind >= MG_KIND_COUNT) return MG_EINVAL;
    prof_flush(h);
    if (launches) *launches = h->prof[level][kind].launches;
    if (timed) *timed = h->prof[level][kind].timed;
    if (ms) *ms = h->prof[level][kind].ms;
    return MG_OK;
}

int64_t mg_launch_count(mg_handle *h) { return h ? h->launches : -1; }
int64_t mg_device_bytes(mg_handle *h) { return h ? h->dev_bytes : -1; }

int mg_dot(mg_handle *h, int level, const double *a, const double *b, double *out) {
    if (!level_ok(h, level) || !a || !b || !out || !aligned16(a) || !aligned16(b)) return MG_EINVAL;
    return dot_dev(h, a, b, h->lev[level].nvec, out);
}

int mg_dot_noalloc(const double *a, const double *b, int64_t n, double *out, void *cuda_stream) {
    if (!a || !b || !out || n < 0 || !aligned16(a) || !aligned16(b)) return MG_EINVAL;
    if (n > MG_NOALLOC_MAX_N) return MG_ETOOLARGE;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return MG_EINVAL;
    unsigned char *scratch = nullptr;
    {   // once per device, with that device current: the device address of the file-scope array
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (g_noalloc_ptr[dev] == nullptr) {
            void *p = nullptr;
            CU(cudaGetSymbolAddress(&p, mg_noalloc_scratch));
            g_noalloc_ptr[dev] = static_cast<unsigned char *>(p);
        }
        scratch = g_noalloc_ptr[dev];
    }
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    double *partial = reinterpret_cast<double *>(scratch);
    unsigned *counter = reinterpret_cast<unsigned *>(scratch + NOALLOC_MAX_GRID * sizeof(double));
    // the array keeps the last call's contents: the ticket must start at zero (the partials are written before they are read)
    CU(cudaMemsetAsync(counter, 0, sizeof(unsigned), stream));
    const int grid = grid_for(n / 2 + 1, 256 * 4, NOALLOC_MAX_GRID);   // the launch shape of dot_dev: same sums, same order
    dot_multi_kernel<<<dim3(grid, 1), 256, 0, stream>>>(a, (int64_t)0, b, n, partial, counter, out, (const int *)nullptr);
    CU(cudaGetLastError());
    return MG_OK;
}

const char *mg_strerror(int code) {
    switch (code) {
        case MG_OK: return "ok";
        case MG_EINVAL: return "invalid argument (shape, ordering, divisibility, NULL or aliased pointer, unsupported b)";
        case MG_ENOMEM: return "out of memory";
        case MG_ESINGULAR: return "a diagonal block is missing or singular";
        case MG_ECUDA: return g_last_cuda_error.empty() ? "CUDA error" : g_last_cuda_error.c_str();
        case MG_ETOOLARGE: return "mg_dot_noalloc: n exceeds MG_NOALLOC_MAX_N (2^26 doubles), the capacity of the fixed scratch array";
        default: return "unknown error code";
    }
}

#ifdef MG_ORTH_STAMPS
int mg_debug_orth_stamps(unsigned long long *host, int n) {
    return cudaMemcpyFromSymbol(host, mgk::orth_stamps, sizeof(unsigned long long) * n) == cudaSuccess ? 0 : -1;
}
#endif
#ifdef MG_DS_STAMP
int mg_debug_ds_stamps(unsigned long long *host, int n) {
    return cudaMemcpyFromSymbol(host, mgk::ds_stamps, sizeof(unsigned long long) * n) == cudaSuccess ? 0 : -1;
}
#endif

const char *mg_version(void) { return "mg_toroidal 0.2.0 (sm_100a)"; }

}  // extern "C"
