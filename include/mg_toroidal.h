/*
 * mg_toroidal.h -- C ABI of libmgtoroidal.so: the solve phase of the toroidal semi-coarsening geometric
 * multigrid preconditioned FGMRES of arXiv 2506.16676 ("Fast solvers for tokamak fluid models with
 * PETSc"), hand-written CUDA for NVIDIA B200 (sm_100a), one GPU, FP64.
 *
 * Citations are lines of the paper text PAPER.md (section in brackets).
 *
 * PROBLEM.  A x = b with A an FP64 block-CSR matrix of b x b node blocks (b = 36 = 12 derivative DoFs x 3
 * fields in the paper, PAPER.md:45, 63 [2.1, 2.3]) on a 2-D poloidal mesh of n_pol nodes extruded over
 * n_phi periodic toroidal planes (PAPER.md:27 [1]).  Block row I = k*n_pol + i (plane k, node i;
 * "blocks group DoFs on planes of constant toroidal coordinate"); scalar index I*b + c.
 *
 * METHOD.  FGMRES (PAPER.md:51, 372 [2.2, App. B]) right-preconditioned by one V(nu_pre, nu_post) cycle
 * (PAPER.md:63 [2.3]) over a hierarchy built by geometric 2:1 coarsening of the toroidal direction with
 * the 3-point prolongation stencil [1/2 1 1/2] and Galerkin operators A_{l+1} = P^T A_l P (PAPER.md:51,
 * 59).  Level smoother: point-block-Jacobi (explicit dense inverses of the diagonal blocks applied as
 * dense mat-vecs) preconditioned Chebyshev (BASELINE.json north_star; reading Q1).
 * Coarsest level: PBJ-preconditioned restarted GMRES to coarse_rtol (BASELINE.json configs[1]).
 * Convergence: rtol = |b - A x| / |b| (PAPER.md:57 [2.2]).
 *
 * CONVENTIONS.
 *  - Unless a parameter says "host", every array pointer is a DEVICE pointer on the current CUDA device,
 *    16-byte aligned, FP64 vectors of n_brows(level)*b doubles.
 *  - All work is enqueued on the cudaStream_t given to mg_setup (pass PyTorch's current stream); calls
 *    return after enqueueing except where a host decision is needed (mg_setup, mg_solve, mg_coarse_solve
 *    synchronise that stream on a few scalars).
 *  - Ownership: the library BORROWS row_ptr / col_idx / vals of the fine matrix for the life of the handle
 *    (never writes or copies them); everything it allocates comes from mg_options.alloc (or cudaMalloc)
 *    and is released by mg_destroy.  Output arrays are caller-owned.
 *  - Errors: every call returns MG_OK (0) or a negative code; no exceptions, no exit().  Non-convergence is
 *    a status (info->converged = 0, return MG_OK), cf. the paper's separate converged_reason reporting
 *    (PAPER.md:365, 437-438).
 *  - Level 0 is the finest level (the paper's A_i -> A_{i+1} numbering).
 *  - There is no CPU fallback: without a CUDA device every entry point that computes returns MG_ECUDA.
 */
#ifndef MG_TOROIDAL_H
#define MG_TOROIDAL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MG_OK 0
#define MG_EINVAL (-1)    /* bad shape, ordering, divisibility, NULL pointer, unsupported b (1..64) */
#define MG_ENOMEM (-2)    /* device or host allocation failed */
#define MG_ESINGULAR (-3) /* a diagonal block is missing or has a zero pivot (PBJ inverse undefined) */
#define MG_ECUDA (-4)     /* CUDA runtime error; mg_strerror gives the last CUDA message */
#define MG_ETOOLARGE (-5) /* mg_dot_noalloc: n exceeds MG_NOALLOC_MAX_N, the capacity of the library's fixed scratch array */

typedef struct mg_handle mg_handle; /* opaque */

/* Device allocator hooks (e.g. PyTorch's caching allocator).  alloc returns a device pointer aligned to
 * at least 256 bytes or NULL; free releases it.  Called from the host thread inside mg_setup /
 * mg_destroy (and lazily on the first mg_solve / mg_coarse_solve for the Krylov bases). */
typedef void *(*mg_alloc_fn)(size_t bytes, void *ctx);
typedef void (*mg_free_fn)(void *ptr, void *ctx);

typedef struct mg_options {
    int nu_pre, nu_post;     /* Chebyshev degree (= number of D^-1 applications) per pre/post smoothing;
                                default 2, 2 ("2 Chebyshev-PBJ sweeps", configs[0]); V(pre,post) */
    double cheb_lo, cheb_hi; /* Chebyshev interval [cheb_lo, cheb_hi] * rho_est(D^-1 A); default 0.1, 1.1 */
    int eig_iters;           /* power iterations for rho_est; default 20 */
    int coarse_mode;         /* 0: PBJ-GMRES(coarse_restart) to coarse_rtol (default);
                                1: coarse_fixed_sweeps Chebyshev-PBJ sweeps (a fixed polynomial: parity mode);
                                2: direct solve (the paper's LU on the coarsest level):
                                   block rows ordered by BFS level sets => block tridiagonal, dense diagonal blocks, sparse
                                   off-diagonal blocks; explicit inverses of the Schur complements at setup/refresh (blocked
                                   Gauss-Jordan), dense mat-vec streaming per solve.  Memory sum_k n_k^2 doubles (n_k = size
                                   of level set k) plus one n_k x n_{k-1} scratch: MG_ENOMEM if it does not fit, MG_EINVAL
                                   if the block pattern is not structurally symmetric */
    double coarse_rtol;      /* default 1e-10 (configs[1]) */
    int coarse_restart, coarse_maxit, coarse_fixed_sweeps; /* defaults 100, 20000, 8 (restart: DESIGN.md Q9) */
    int restart, maxit;      /* outer FGMRES restart length and iteration cap; defaults 100, 400
                                (paper: 200 / 200) */
    int use_graphs;          /* 1 (default): the coarse GMRES restart cycle is replayed as a CUDA graph */
    int kernel_variant;      /* launch mechanics only (same arithmetic up to summation order): 0 (default) the
                                persistent TMA-ring block-CSR kernel where it exists (b = 36), 1 the one-CTA-per-row
                                128-bit-load kernel for every b (kept for A/B measurement) */
    int smoother;            /* 0 (default): PBJ-Chebyshev (BASELINE.json north_star); 1: nu iterations of right-PBJ-
                                preconditioned GMRES without a convergence test -- the paper's own level smoother,
                                "one iteration of GMRES preconditioned with PBJ", V(1,1) / V(6,6);
                                2: Chebyshev preconditioned by toroidal-LINE block Jacobi (the paper's
                                outlook): the block of a poloidal node couples all its planes, a periodic
                                block-tridiagonal system factorised at setup / refresh into explicit b x b inverses.  Needs
                                b <= 48 and same-node couplings on planes k-1, k, k+1 only (MG_EINVAL otherwise); 2N-1 extra
                                blocks per node and level.  The coarsest-level GMRES keeps PBJ. */
    double orth_eta;         /* Gram-Schmidt in (F)GMRES: 0 = classical Gram-Schmidt with a second pass on every step
                                (CGS2); eta in (0,1) = the second pass only when ||w - V V^T w|| < eta ||w|| (selective
                                reorthogonalisation, Daniel-Gragg-Kaufman-Stewart).  Same Arnoldi relation either way.
                                Default 0.25 (orthogonality kept to ~4 eps per step). */
    mg_alloc_fn alloc;       /* NULL => cudaMalloc */
    mg_free_fn free;         /* NULL => cudaFree */
    void *alloc_ctx;
} mg_options;

typedef struct mg_solve_info {
    int iters;              /* outer FGMRES iterations = number of V-cycle applications */
    int converged;          /* 1 if the Arnoldi residual estimate reached rtol*|b| */
    double solve_ms;        /* device time of the solve (CUDA events on the stream, inputs resident in HBM) */
    double rel_res;         /* true |b - A x| / |b| recomputed after the solve */
    int coarse_iters_total; /* coarsest-level GMRES iterations summed over all V-cycles */
    int hist_len;           /* in: capacity of hist; out: entries written (iters + 1, clipped) */
    double *hist;           /* HOST array, caller-owned, may be NULL: hist[k] = estimate_k / |b| */
} mg_solve_info;

/* Fill *opt with the defaults above.  Returns MG_EINVAL if opt is NULL. */
int mg_options_default(mg_options *opt);
/* sizeof(mg_options) / sizeof(mg_solve_info) as this library was compiled: a binding checks its own layout against them. */
size_t mg_sizeof_options(void);
size_t mg_sizeof_solve_info(void);

/* mg_setup -- build the hierarchy ("the batched diagonal-block inversion and ... the Galerkin coarse
 * operators", north_star).  Per level: locate and invert every diagonal block
 * (Gauss-Jordan, partial pivoting), estimate rho(D^-1 A) by eig_iters power iterations from the start
 * vector v0[g] = ((g*2654435761) mod 2^32)/2^32 - 1/2, and form A_{l+1} = P^T A_l P.
 *   row_ptr  int64[n_brows+1], col_idx int32[nnzb] (ascending within a row), vals double[nnzb*b*b]
 *   (ROW-MAJOR b x b blocks, the only layout: the fine matrix is borrowed, never copied, so a column-major input
 *   (SURVEY 8b proposed a flag) would need a transposed copy of up to 55 GB; the caller transposes instead):
 *   the fine matrix, DEVICE pointers, borrowed until mg_destroy.
 *   n_brows = n_pol*n_phi; levels >= 1; n_phi divisible by 2^(levels-1); 1 <= b <= 64.
 *   levels == 1 is legal: mg_vcycle is then the coarsest-level solve on the fine matrix.
 *   opt may be NULL (defaults).  cuda_stream is a cudaStream_t (NULL = legacy default stream).
 * Errors: MG_EINVAL (arguments, unsorted columns, column out of range), MG_ESINGULAR, MG_ENOMEM, MG_ECUDA. */
int mg_setup(mg_handle **h, const int64_t *row_ptr, const int32_t *col_idx, const double *vals, int b, int n_pol,
             int n_phi, int levels, const mg_options *opt, void *cuda_stream);

/* Replace the solve-phase options (nu, Chebyshev interval factors, coarse_*, restart, maxit) without
 * rebuilding the hierarchy; alloc/free/eig_iters are ignored. */
int mg_update_options(mg_handle *h, const mg_options *opt);

/* Lagged preconditioner ("one new Jacobian per time step ... the preconditioner
 * is lagged, refreshed every `refresh period` steps"; refresh cost: Table 4).
 * mg_update_values -- REFRESH: new fine-level values with the SAME pattern (device pointer, borrowed from now on in
 *   place of the old one): recomputes the block inverses, the Chebyshev bounds and the Galerkin operators into the
 *   existing patterns and allocations (no symbolic phase).  Also resets the solve operator to these values.
 *   Errors: MG_EINVAL, MG_ESINGULAR, MG_ECUDA.  Synchronises the stream.
 * mg_set_operator -- LAG: mg_solve iterates on A_new = (level-0 pattern, `vals`) while the V-cycle keeps the
 *   hierarchy of the last setup/refresh.  vals: device pointer, borrowed; NULL = back to the hierarchy's own matrix. */
int mg_update_values(mg_handle *h, const double *vals);
int mg_set_operator(mg_handle *h, const double *vals);

/* mg_vcycle -- z = M(r): one V(nu_pre,nu_post) cycle from a zero guess.  r, z: level-0
 * vectors; r is not modified, z is overwritten.  Asynchronous in coarse_mode 1. */
int mg_vcycle(mg_handle *h, const double *r, double *z);

/* mg_solve -- FGMRES(restart) on A x = rhs preconditioned by mg_vcycle, stopping when the residual
 * estimate <= rtol*|rhs| or after maxit iterations.  x is the initial guess if
 * x_is_initial_guess != 0, else it is ignored and the guess is zero; x receives the solution.
 * info may be NULL.  Synchronises the stream. */
int mg_solve(mg_handle *h, const double *rhs, double *x, double rtol, int x_is_initial_guess, mg_solve_info *info);

/* Same solve with HOST buffers: copies rhs (and x if it is the guess) to the device, solves, copies x back.
 * rhs_host, x_host: host arrays of n_brows*b doubles (pinned memory makes the copies asynchronous). */
int mg_solve_host(mg_handle *h, const double *rhs_host, double *x_host, double rtol, int x_is_initial_guess,
                  mg_solve_info *info);

int mg_destroy(mg_handle *h);

/* ---- per-kernel entry points (parity tests and roofline measurements) ---------------------------------- */
/* y = A_level x                                           (block-CSR SpMV, "the kernel of MG") */
int mg_spmv(mg_handle *h, int level, const double *x, double *y);
/* r = rhs - A_level x */
int mg_residual(mg_handle *h, int level, const double *rhs, const double *x, double *r);
/* z = D_level^-1 r                                        (PBJ apply) */
int mg_pbj_apply(mg_handle *h, int level, const double *r, double *z);
/* nu sweeps (polynomial degree nu = nu applications of D^-1) of PBJ-Chebyshev on A_level x = rhs; x is the
 * initial guess unless zero_guess != 0 (then x is overwritten from a zero guess).  rhs must not alias x. */
int mg_smooth(mg_handle *h, int level, const double *rhs, double *x, int nu, int zero_guess);
/* r_coarse = P^T r_fine, from level to level+1           (stencil [1/2 1 1/2]) */
int mg_restrict(mg_handle *h, int level, const double *r_fine, double *r_coarse);
/* x_fine += P e_coarse, from level+1 to level */
int mg_prolong_add(mg_handle *h, int level, const double *e_coarse, double *x_fine);
/* Coarsest-level solve A_{L-1} e = r from a zero guess (mode per options); iters may be NULL. Synchronises. */
int mg_coarse_solve(mg_handle *h, const double *r, double *e, int *iters);

/* Direct coarsest-level solve (coarse_mode = 2), after its first use: number of BFS level sets, bytes of the dense Schur
 * inverses (sum_k n_k^2 doubles), bytes of the off-diagonal blocks L_k, U_k read per solve, widest level set (scalars) and
 * whether the persistent cooperative kernel is in use (else the launch chain).  One solve streams 2 * dense_bytes +
 * offdiag_bytes.  Any out pointer may be NULL.  MG_EINVAL before the first direct solve. */
int mg_direct_info(mg_handle *h, int *level_sets, int64_t *dense_bytes, int64_t *offdiag_bytes, int *max_n, int *persistent);

/* Borrowed DEVICE pointers and sizes of one level (any out pointer may be NULL). */
int mg_get_level(mg_handle *h, int level, int64_t *n_brows, int64_t *nnzb, const int64_t **row_ptr,
                 const int32_t **col_idx, const double **vals, const double **dinv, double *rho_est,
                 double *lam_min, double *lam_max);
/* Copy one level's arrays into caller-owned HOST buffers (any may be NULL): row_ptr int64[n_brows+1],
 * col_idx int32[nnzb], vals double[nnzb*b*b], dinv double[n_brows*b*b].  Synchronises the stream. */
int mg_copy_level_to_host(mg_handle *h, int level, int64_t *row_ptr_host, int32_t *col_idx_host, double *vals_host,
                          double *dinv_host);
/* Override the Chebyshev interval of one level (parity tests inject the oracle's bounds). */
int mg_set_cheb_bounds(mg_handle *h, int level, double lam_min, double lam_max);
/* ---- dot products (the reduction of the orthogonalisation: deterministic, warp-shuffle + fixed-order sums) -- */
/* out[0] = <a, b> over the n_brows(level)*b entries of two level vectors; out is a DEVICE pointer (1 double), written on
 * the handle's stream.  Scratch: the handle's own (allocated in mg_setup). */
int mg_dot(mg_handle *h, int level, const double *a, const double *b, double *out);

/* mg_dot_noalloc -- the same reduction (same kernel, same launch shape, hence the same bits as mg_dot) for callers that
 * must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It needs NO
 * handle and calls no cudaMalloc / cudaFree / allocating routine: the per-CTA partial sums and the ticket counter live in a
 * file-scope `static __device__` array of the library (MG_NOALLOC_SCRATCH_BYTES = 8,448 bytes; every GPU that loads the
 * library holds it until exit), whose device address is taken once per device with cudaGetSymbolAddress.
 *   a, b: DEVICE vectors of n doubles (16-byte aligned), out: DEVICE pointer to 1 double, cuda_stream: a cudaStream_t.
 *   n <= MG_NOALLOC_MAX_N, else MG_ETOOLARGE (nothing is launched).  n == 0 gives 0.
 * Every call shares the one scratch array: the ticket counter is cleared on the stream before each launch, the partial
 * sums are overwritten before they are read.  Calls that OVERLAP on the GPU (different streams, or several host threads
 * on one device) RACE on it: serialise them (one stream, or events).  Errors: MG_EINVAL, MG_ETOOLARGE, MG_ECUDA. */
#define MG_NOALLOC_MAX_N ((int64_t)1 << 26)      /* 67,108,864 doubles = 512 MiB per vector (the configs' largest: 9,216,000) */
#define MG_NOALLOC_SCRATCH_BYTES (1024 * 8 + 256)
int mg_dot_noalloc(const double *a, const double *b, int64_t n, double *out, void *cuda_stream);

/* ---- profiling: per-(level, kind) device time of the library's own kernel launches --------------------- */
#define MG_KIND_SPMV 0      /* y = A x */
#define MG_KIND_RESID 1     /* r = rhs - A x */
#define MG_KIND_SWEEP 2     /* fused PBJ-Chebyshev sweep: r -= A d, z = D^-1 r, d' = c_d d + c_z z, x update */
#define MG_KIND_SWEEP_NOD 3 /* last pre-smoothing sweep: r -= A d, x += d (no D^-1 pass) */
#define MG_KIND_PBJ 4       /* z = D^-1 r */
#define MG_KIND_RESTRICT 5
#define MG_KIND_PROLONG 6
#define MG_KIND_ORTH 7      /* (F)GMRES dots / axpys / Givens bookkeeping */
#define MG_KIND_OTHER 8
#define MG_KIND_CYCLE 9     /* one whole coarsest-level GMRES restart cycle in a single persistent kernel */
#define MG_KIND_DIRECT 10   /* direct coarsest-level solve: the persistent cooperative kernel (or its launch-chain fallback) */
#define MG_KIND_LINE 11     /* toroidal-line block solve + Chebyshev direction update (smoother = 2) */
#define MG_KIND_COUNT 12
#define MG_PROFILE_MAX_LEVELS 32
/* Launches are always counted per (level, kind).  on != 0 additionally brackets every kernel launch with a
 * CUDA event pair on the stream and books its duration; CUDA-graph replay is bypassed while that is on. */
int mg_profile_enable(mg_handle *h, int on);
int mg_profile_reset(mg_handle *h);
/* One (level, kind) class since the last reset: launches (all), timed (launches that were event-bracketed)
 * and ms (their summed device milliseconds).  Any out pointer may be NULL.  Synchronises the stream. */
int mg_profile_get(mg_handle *h, int level, int kind, int64_t *launches, int64_t *timed, double *ms);

/* Number of CUDA kernels this handle has launched so far (graph replays count their kernel nodes). */
int64_t mg_launch_count(mg_handle *h);
/* Bytes of device memory the handle has allocated. */
int64_t mg_device_bytes(mg_handle *h);
const char *mg_strerror(int code);
const char *mg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_TOROIDAL_H */
