/*
 * coarse_mrhs.h -- C ABI of the B200-native coarse-grid multi-RHS operator and block CG
 * (data-parallel hot path of the multiple right-hand-side HDCG method, arXiv:2409.03904).
 *
 * Citations are PAPER.md:<line> (the paper text) plus section / equation.
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 *  - "dev" pointers are CUDA device pointers owned by the CALLER (e.g. torch tensors); "host" pointers
 *    are ordinary host memory owned by the caller.  The library never frees or keeps a caller pointer
 *    beyond the call, except where stated (coarse_op_create copies A).
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *  - Every function returns a status code (COARSE_OK = 0, negative = error); no exceptions cross the ABI.
 *    On COARSE_INVALID_ARG / COARSE_UNSUPPORTED the outputs are untouched.  coarse_last_error() returns a
 *    thread-local, human-readable description of the last failure.
 *  - There is NO CPU fallback: every entry point that computes runs CUDA kernels on the current device
 *    and fails with COARSE_CUDA_ERROR when there is none.
 *
 * Canonical (boundary) layouts
 * ----------------------------
 *  lattice site     x = x0 + L0*(x1 + L1*(x2 + L2*x3)),  dims = {L0, L1, L2, L3}, dims[0] fastest
 *  stencil point    p = (d0+1) + 3*(d1+1) + 9*(d2+1) + 27*(d3+1),  d_k in {-1,0,1}; centre p = 40,
 *                   opposite point 80-p.  81 points = all relative shifts (-1..1)^4.
 *  stencil matrices A : [V][81][nbasis][nbasis], row-major blocks, interleaved (re, im)
 *  vector blocks    X, Y, B : [V][nbasis][nrhs], right-hand-side index fastest, interleaved (re, im)
 *                   ("N_basis x N_rhs" per coarse site; the RHS index is the paper's
 *                   fictitious fifth dimension)
 *  dtype            COARSE_C64: float re/im pairs; COARSE_C128: double re/im pairs
 *  boundary         periodic: neighbour = (x_k + d_k + L_k) mod L_k.  With L_k = 1 or 2 several stencil
 *                   points address the same neighbour; their contributions ADD.
 */
#ifndef COARSE_MRHS_H
#define COARSE_MRHS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct coarse_op coarse_op_t; /* opaque, library-owned */

enum { COARSE_C64 = 0, COARSE_C128 = 1 };

enum {
    COARSE_OK = 0,
    COARSE_INVALID_ARG = -1,
    COARSE_UNSUPPORTED = -2,   /* shape outside 1 <= nbasis <= 64, 1 <= nrhs <= 64 */
    COARSE_CUDA_ERROR = -3,
    COARSE_OUT_OF_MEMORY = -4,
    COARSE_NOT_CONVERGED = -5, /* block_cg_solve hit maxiter; outputs are valid */
    COARSE_BREAKDOWN = -6      /* a Gram matrix was not positive definite (no column deflation) */
};

/* create-time flags */
enum {
    COARSE_FLAG_FORCE_GENERIC = 1u << 0, /* always use the generic (untiled) stencil kernel: test / debugging aid */
    COARSE_FLAG_NO_TENSOR = 1u << 1,     /* never select a tensor-core kernel variant */
    COARSE_FLAG_TENSOR_ONLY = 1u << 2,   /* complex64 shapes the tensor-core kernel covers: keep only its layout of A (one
                                            internal copy instead of two); apply / solve with an nrhs that kernel does not
                                            cover (not a multiple of 8) then return COARSE_UNSUPPORTED */
    COARSE_FLAG_TF32 = 1u << 3,          /* complex64, nbasis 32: use the split-TF32 tensor kernel (operator kept as float32)
                                            instead of the default split-FP16 kernel (operator stored pre-split as two
                                            binary16 numbers per real: 22-23 significant bits, elements below 2^-29 of the
                                            operator's largest element lose relative precision) */
    COARSE_FLAG_UNFUSED_LINALG = 1u << 4, /* block_cg_*: run the block rotations and Gram products of an iteration as six
                                            separate kernels instead of the two fused passes (cross-check / debugging aid) */
    COARSE_FLAG_H16X = 1u << 5,          /* complex64, nbasis 32: keep the operator in the layout of the split-FP16 kernel that
                                            holds the X operand in tensor memory (stencil_h16x: the default for nbasis 8, 16, 24)
                                            instead of the paired-site kernel's (stencil_h16) */
    COARSE_FLAG_TENSOR_LINALG = 1u << 6, /* complex64: run the block rotations and Gram products of widths 16 to 32 on the tensor
                                            cores too (split-FP16, as the stencil kernels); widths >= 40 always do, unless
                                            COARSE_FLAG_NO_TENSOR */
    COARSE_FLAG_H16X_WIDE = 1u << 7,     /* complex64, nbasis 32, nrhs_max > 48: keep BOTH split-FP16 layouts of the operator (one more
                                            internal copy): stencil_h16 serves nrhs <= 48, stencil_h16x the wider blocks, where it
                                            is the faster kernel (7.4 vs 7.8 ms at BASELINE configs[3], nrhs 64) */
    COARSE_FLAG_NO_GRAPH = 1u << 8       /* block_cg_*: never replay an iteration as a CUDA graph (by default small, launch-bound blocks --
                                            V * nbasis * nrhs <= 2^22 -- do, from the second iteration of a solve on) */
};

#define COARSE_MAX_NRHS 64
#define COARSE_MAX_NBASIS 64
#define COARSE_MAX_NEV 4096 /* eigenvectors of coarse_deflate (the paper: several hundred to 1000) */

/*
 * coarse_op_create -- build the operator object.  "The coarse matrix coefficients are stored entirely
 * internal to this object" and the neighbour addressing is precomputed once.
 *   out       : receives the handle
 *   dims      : host, 4 extents, each >= 1
 *   nbasis    : 1..64 (rows/cols of each stencil matrix)
 *   nrhs_max  : 1..64, largest nrhs later passed to apply / solve; sizes the block-CG workspace
 *   dtype     : COARSE_C64 or COARSE_C128 (storage and multiply precision of A, X, Y)
 *   A_dev     : device, canonical layout; COPIED (re-laid-out for the kernels) -- may be freed after return
 *   flags     : COARSE_FLAG_*
 * Allocates device memory: one internal copy of A (two for complex64 shapes the tensor-core kernel covers, unless
 * COARSE_FLAG_TENSOR_ONLY or COARSE_FLAG_NO_TENSOR), V*81 int32 neighbour table, 6 vector blocks of
 * V*nbasis*nrhs_max elements plus O(grid * nrhs_max^2) reduction scratch.  Synchronises `stream`.
 */
int coarse_op_create(coarse_op_t **out, const int32_t dims[4], int32_t nbasis, int32_t nrhs_max,
                     int32_t dtype, const void *A_dev, uint32_t flags, void *stream);

int coarse_op_destroy(coarse_op_t *op);

/*
 * coarse_op_apply -- Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p) for all sites, one launch
 * (Eq. 19 summed over the stencil; the paper issues 81 batched GEMMs).
 *   X_dev, Y_dev : device, [V][nbasis][nrhs], dtype of the operator, 16-byte aligned; Y must not alias X
 *   nrhs         : 1..nrhs_max
 * Asynchronous on `stream`; allocates nothing.  Kernel selection (coarse_op_kernel_name tells which): complex64 with nbasis 32
 * and nrhs 4 or a multiple of 8 -> stencil_h16 (tcgen05, split FP16, paired sites); complex64 with nbasis 8, 16, 24 and nrhs >= 4
 * (nbasis 32 with COARSE_FLAG_H16X, or above nrhs 48 with COARSE_FLAG_H16X_WIDE) -> stencil_h16x (tcgen05, split FP16, X operand
 * in tensor memory); COARSE_FLAG_TF32 -> stencil_tc; complex128 with nbasis and nrhs multiples of 8 -> stencil_dmma (mma.sync
 * f64); otherwise a tiled SIMT variant or the generic kernel.  The split-FP16 kernels first run two short pre-pass kernels that
 * write the scaled, split copy of X into a scratch block OWNED BY THE HANDLE, so applies on one handle must be ordered (same
 * stream, or externally synchronised) although the handle is passed as const; distinct handles are independent.
 */
int coarse_op_apply(const coarse_op_t *op, const void *X_dev, void *Y_dev, int32_t nrhs, void *stream);

/* Same operation with HOST buffers: copies X host->device, applies, copies Y device->host, synchronises.
 * Uses the operator's own workspace blocks (the paper's "import/export to preallocated arrays"). */
int coarse_op_apply_host(coarse_op_t *op, const void *X_host, void *Y_host, int32_t nrhs, void *stream);

/*
 * block_cg_solve -- BlockCGrQ (Fig. 2 left) for H X = B with the operator above:
 *   R = B - H X0;  Q C = R (Cholesky QR);  D = Q;  loop:  Z = H D;  M = (D^H Z)^-1;
 *   X += D M C;  Q S = Q - Z M;  D = Q + D S^H;  C = S C;  stop when max_r ||C[:,r]|| / ||B[:,r]|| <= tol.
 * (X update carries C_k: DESIGN.md reading R1.)
 *   B_dev   : device, sources, [V][nbasis][nrhs]
 *   X_dev   : device, in: initial guess X0, out: solution
 *   res     : host; iterations = number of H.D products in the loop; rel_res_recursive[r] from C,
 *             rel_res_true[r] = ||B - H X||/||B|| from one extra apply; history[k] = max_r recursive
 *             relative residual after k iterations (k <= COARSE_MAX_HISTORY-1)
 * Returns COARSE_OK, COARSE_NOT_CONVERGED or COARSE_BREAKDOWN (res->status holds the same).
 * Synchronises `stream` (one scalar is read back per iteration for the stop test).
 */
#define COARSE_MAX_HISTORY 256
typedef struct {
    int32_t iterations;
    int32_t status;
    double rel_res_recursive[COARSE_MAX_NRHS];
    double rel_res_true[COARSE_MAX_NRHS];
    double history[COARSE_MAX_HISTORY];
    double seconds; /* wall time of the solve, host clock, stream synchronised on both sides */
} block_cg_result;

int block_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol,
                   int32_t maxiter, block_cg_result *res, void *stream);

/*
 * The same solve in three calls, for callers that drive the iteration themselves (bench.py times exactly K
 * iterations on the device this way; block_cg_solve is begin + {step, read stop scalar} + end):
 *   block_cg_begin : R = B - H X0, Q C = R, D = Q (statements 4-6 of Fig. 2 left).  Synchronises
 *                    (reads the initial residual into *rel_res0, may be NULL).  Returns COARSE_NOT_CONVERGED when
 *                    iterations are needed (the normal case), COARSE_OK when X0 already meets tol, or an error.
 *                    B_dev and X_dev must stay valid until block_cg_end.
 *   block_cg_step  : `count` iterations (statements 8-13); asynchronous, no host read, no stop test.
 *   block_cg_end   : one extra apply for the true residual; fills res (status OK or BREAKDOWN); synchronises.
 */
int block_cg_begin(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, double *rel_res0,
                   void *stream);
int block_cg_step(coarse_op_t *op, int32_t count, void *stream);
int block_cg_end(coarse_op_t *op, block_cg_result *res, void *stream);

/*
 * coarse_cheby_apply -- stationary polynomial coarse solve  X = P(H) B,  P = "Chebyshev approximation to 1/x over
 * eigenspan [lo, hi]" of the given order, "coefficients ... at the Chebyshev interpolation points from the target function
 * 1/x" (section 2.3; the paper's tuned coarse solve is [lo, hi, order] = [0.02, 40, 120], its smoother
 * [2.0, 92.0] order 8).  Reading (R16): `order` = number of coefficients (degree order - 1), interpolation at the
 * first-kind Chebyshev points of [lo, hi]; P(H) B by the three-term recurrence on blocks: order - 1 applications of the
 * operator, each followed by ONE fused elementwise pass (T_{j+1} = 2 (a H T_j + b T_j) - T_{j-1}; X += c_{j+1} T_{j+1}),
 * no reductions, no host synchronisation.
 *   B_dev, X_dev : [V][nb][nrhs] device blocks of the operator's dtype, X_dev != B_dev; B is not modified
 *   lo, hi       : 0 < lo < hi;  order >= 1;  coefficients are computed on the host in double precision
 * Asynchronous on `stream`; uses the handle's block-CG workspace (do not interleave with a begin/step/end solve).
 * Errors: COARSE_INVALID_ARG (NULL, aliasing, lo/hi/order/nrhs out of range), kernel launch errors.
 */
int coarse_cheby_apply(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double lo, double hi, int32_t order,
                       void *stream);

/*
 * coarse_deflate -- multi-RHS deflation with n_ev eigenpairs of the operator (Eq. 7-10; "applied to
 * multiple right-hand sides"):  C = Vev^H B;  QBpar = Vev (C / lambda) = (sum_i |i><i| / lambda_i) b;
 * Bperp = B - Vev C = (1 - sum_i |i><i|) b.  Tall-skinny products, eigenvectors taken in chunks of 64
 * columns (chunk j projects the running Bperp: the columns are orthonormal): per chunk a deterministic two-stage reduction
 * (complex128 sums) and one pass over the chunk and the block.  The FIRST call on a handle allocates the scratch for the
 * 64 x nrhs_max coefficients and their per-CTA partials (about 1 MiB per right-hand side; freed by coarse_op_destroy).
 *   Vev_dev     : [V*nbasis][nev] device block of the operator's dtype, eigenvector index fastest, orthonormal columns
 *   lambda_host : [nev] HOST doubles, all > 0;  1 <= nev <= COARSE_MAX_NEV (the paper deflates with 192-1000 vectors)
 *   B_dev       : [V][nb][nrhs];  QBpar_dev, Bperp_dev: outputs of the same shape, QBpar != B, QBpar != Bperp (Bperp may alias B)
 * coarse_cheby_defl_solve -- the paper's stationary coarse solve  X = Defl(b_par) + P^Cheby(b_perp)  (Eq. 11-12), P as in
 * coarse_cheby_apply.  Asynchronous on `stream`; both use the handle's block-CG workspace.
 * Errors: COARSE_INVALID_ARG (NULL, aliasing, nev / nrhs / lambda / lo / hi / order out of range), COARSE_OUT_OF_MEMORY (first call), launch errors.
 */
int coarse_deflate(coarse_op_t *op, const void *Vev_dev, const double *lambda_host, int32_t nev, const void *B_dev,
                   void *QBpar_dev, void *Bperp_dev, int32_t nrhs, void *stream);
int coarse_cheby_defl_solve(coarse_op_t *op, const void *Vev_dev, const double *lambda_host, int32_t nev, const void *B_dev,
                            void *X_dev, int32_t nrhs, double lo, double hi, int32_t order, void *stream);

/*
 * pblock_cg_solve -- Preconditioned BlockCGrQ (Fig. 2 right) for H X = B with a STATIONARY Hermitian
 * positive definite preconditioner M^-1: the Chebyshev polynomial of H (coarse_cheby_apply) or the
 * deflated Chebyshev solve (coarse_cheby_defl_solve).  Statement by statement as printed, with the two readings of
 * DESIGN.md (the update is X += D_k N_k C_k; one Cholesky factor S per iteration, S^H S = T^H t).  Both the unpreconditioned
 * (q, z, t) and the preconditioned (Q, Z, T) blocks are rotated; Gram products in the M inner product are Z^H z, D^H z, T^H t.
 * Stop test: the Euclidean residual r_{k+1} = q_{k+1} C_{k+1} = t_k C_k, max_r ||r[:,r]|| / ||B[:,r]|| <= tol (one extra Gram
 * t^H t per iteration), taken BEFORE the factorisation of T^H t: once converged that matrix is rounding noise.
 *   B_dev, X_dev : as block_cg_solve (X in: X_0, out: solution);  M: host struct, its pointers as in coarse_deflate
 *   res          : host; rel_res_recursive = the stop quantity at the last iteration, rel_res_true from one extra apply
 * Synchronises the stream every iteration (stop scalar).  Allocates five more workspace blocks on first use.
 * Returns COARSE_OK, COARSE_NOT_CONVERGED (outputs valid), COARSE_BREAKDOWN, COARSE_INVALID_ARG, COARSE_OUT_OF_MEMORY.
 */
enum { COARSE_PRECOND_CHEBY = 0, COARSE_PRECOND_DEFL_CHEBY = 1 };
typedef struct {
    int32_t kind;                 /* COARSE_PRECOND_* */
    int32_t order;                /* Chebyshev order (number of coefficients) */
    double lo, hi;                /* Chebyshev interval */
    const void *Vev_dev;          /* DEFL_CHEBY: [V*nbasis][nev] eigenvectors (device), else NULL */
    const double *lambda_host;    /* DEFL_CHEBY: [nev] eigenvalues (host), else NULL */
    int32_t nev;
} coarse_precond;
int pblock_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter,
                    const coarse_precond *M, block_cg_result *res, void *stream);

/*
 * stacked_cg_solve -- the coarse solve "as an enlarged five dimensional system with a single Krylov solve, albeit with a
 * block diagonal structure": plain conjugate gradients on (I_nrhs (x) H) vec(X) = vec(B), ONE alpha and
 * ONE beta per iteration from Frobenius inner products over all right-hand sides.  Per iteration: one apply, two fused
 * elementwise passes (X += alpha P, R -= alpha Z with <R,R>;  P = R + beta P), one inner product; scalars stay on the device,
 * one stop scalar goes to the host.  Stop: ||R||_F / ||B||_F <= tol (R18); res->history holds that quantity,
 * rel_res_recursive its last value in every column, rel_res_true the per-column true residuals from one extra apply.
 * Arguments and return codes as block_cg_solve.
 */
int stacked_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter,
                     block_cg_result *res, void *stream);

/*
 * coarse_block_project / coarse_block_promote -- multi-RHS transfer between grids (section 2.5.1), "one
 * matrix multiply for each coarse lattice site":
 *   project (Eq. 14):  C[x] (nbasis x nrhs) = Basis[x]^dagger (nbasis x vblock) . F[x] (vblock x nrhs)
 *   promote (Eq. 15):  F[x] (vblock x nrhs) = Basis[x] (vblock x nbasis) . C[x] (nbasis x nrhs)
 * Layouts (device, row-major, interleaved complex of `dtype`): Basis [Vc][vblock][nbasis], fine vectors [Vc][vblock][nrhs]
 * (the fine field block by block -- the paper's "BLAS ready layout"), coarse vectors [Vc][nbasis][nrhs] (the layout of
 * coarse_op_apply).  Stateless (no handle), asynchronous on `stream`, allocate nothing.  nbasis, nrhs <= 64.
 * Errors: COARSE_INVALID_ARG, launch errors.
 * Kernels: SIMT.  nbasis and nrhs multiples of 4 (Table 6's 64 x 12 and the coarse operator's shapes) take register-tiled,
 * pipelined kernels (project: bulk-copied row tiles, several sites per CTA; promote: padded cp.async tiles) at 2.2-3.0 TB/s
 * = 22-32 TFLOP/s on B200 -- both shapes are bound by the FP32 pipe, not by HBM; other shapes take a plain kernel (1.3-1.5 TB/s).
 * Sums: project adds runs of <= 32 rows in `dtype` into the site's accumulator (double for complex128, float for complex64:
 * error <= (32 + vblock/32) eps); promote sums its nbasis terms in `dtype`.
 */
int coarse_block_project(const void *Basis_dev, const void *F_dev, void *C_dev, int64_t Vc, int32_t vblock, int32_t nbasis,
                         int32_t nrhs, int32_t dtype, void *stream);
int coarse_block_promote(const void *Basis_dev, const void *C_dev, void *F_dev, int64_t Vc, int32_t vblock, int32_t nbasis,
                         int32_t nrhs, int32_t dtype, void *stream);

/* Same with HOST buffers for B (in) and X (in: X0, out: solution). */
int block_cg_solve_host(coarse_op_t *op, const void *B_host, void *X_host, int32_t nrhs, double tol,
                        int32_t maxiter, block_cg_result *res, void *stream);

/* The same two solves with options.  COARSE_SOLVE_ZERO_GUESS: "X arbitrary" taken as X_0 = 0 -- X is an output
 * only (its contents on entry are ignored; the host variant does not copy it to the device), R_0 = B and the application of
 * the operator to X_0 is skipped.  Unknown flag bits: COARSE_INVALID_ARG.
 * The host variants start the device->host copy of the solution as soon as the iteration has stopped, on a stream of the
 * handle's own, so that it overlaps the extra apply of the true residual; they return after both have finished. */
enum { COARSE_SOLVE_ZERO_GUESS = 1u << 0 };
int block_cg_solve_ex(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter, uint32_t flags,
                      block_cg_result *res, void *stream);
int block_cg_solve_host_ex(coarse_op_t *op, const void *B_host, void *X_host, int32_t nrhs, double tol, int32_t maxiter,
                           uint32_t flags, block_cg_result *res, void *stream);

/*
 * The block-CG building blocks, exported so that each can be checked against the oracle on its own.
 * n = number of rows (V*nbasis), s = nrhs (1..64); blocks are [n][s] in `dtype`; s x s matrices are
 * ALWAYS complex128, row-major, on the device.
 *
 * coarse_block_gram   : G = U^H W  (Table 6 "ThinQR" shape).
 *                       Deterministic two-stage reduction; products in `dtype`, partial sums in double.
 * coarse_small_cholesky: G = S^H S, S upper triangular with positive diagonal (G symmetrised first);
 *                       optionally S^-1.  info_dev (int32, device) = 0 or COARSE_BREAKDOWN.
 * coarse_small_hpd_inverse: M = G^-1 through the Cholesky factor (M_k = [D^H Z]^-1).
 * coarse_block_rotate : W = beta*W + U K, K s x s (the "block rotations" X += D M C, Q - Z M, T S^-1,
 *                       Q + D S^H of PAPER.md:145-149); beta in {0,1} or any real; W may alias neither U.
 */
int coarse_block_gram(coarse_op_t *op, const void *U_dev, const void *W_dev, void *G_dev, int64_t n,
                      int32_t s, void *stream);
/*
 * coarse_block_gram_noalloc -- the same G = U^H W for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it) and so cannot hold a handle (coarse_op_create allocates).
 * It takes no handle and allocates nothing: no cudaMalloc / cudaFree / allocating library routine on any call, the first
 * included.  The per-CTA partial sums of the two-stage reduction live in a file-scope device array of
 * COARSE_NOALLOC_SCRATCH_BYTES (4 MiB) that every GPU holds from the moment it loads the library until the process exits.
 *   dtype        : COARSE_C64 or COARSE_C128 (U, W: [n][s] in dtype, device, 16-byte aligned; caller-owned, read only)
 *   G_dev        : [s][s] complex128, row-major, device, 16-byte aligned; caller-owned, overwritten
 *   n >= 1, 1 <= s <= COARSE_NOALLOC_MAX_NRHS (32).  A larger s returns COARSE_UNSUPPORTED with a message naming the limit
 *                  and leaves G untouched; use coarse_block_gram for it.
 *   stream       : the two kernels are launched on it; nothing synchronises.
 * EVERY call on a device shares the one array: calls that overlap on the GPU (different streams, different host threads)
 * race -- order them on one stream or with events.  The array keeps the last call's contents; nothing in it has to be
 * zero (each launch overwrites every partial it later reads).  Deterministic; SIMT kernels only (widths <= 32 never take
 * the tensor path of coarse_block_gram either), same arithmetic as coarse_block_gram up to the order of the partial sums.
 * Errors: COARSE_INVALID_ARG (NULL, dtype, n, s < 1, alignment), COARSE_UNSUPPORTED (s beyond the limit), CUDA errors.
 */
#define COARSE_NOALLOC_MAX_NRHS 32
#define COARSE_NOALLOC_SCRATCH_BYTES (256 * 32 * 32 * 16)
int coarse_block_gram_noalloc(int32_t dtype, const void *U_dev, const void *W_dev, void *G_dev, int64_t n, int32_t s,
                              void *stream);
int coarse_small_cholesky(const void *G_dev, void *S_dev, void *Sinv_dev /* may be NULL */, int32_t s,
                          int32_t *info_dev, void *stream);
int coarse_small_hpd_inverse(const void *G_dev, void *M_dev, int32_t s, int32_t *info_dev, void *stream);
int coarse_block_rotate(coarse_op_t *op, const void *U_dev, const void *K_dev, void *W_dev, double beta,
                        int64_t n, int32_t s, void *stream);

/*
 * Bench convenience (input generation, not part of the method): fills A_dev (canonical layout) with the
 * seeded synthetic Hermitian positive definite operator of DESIGN.md "Synthetic inputs" -- the same
 * counter-based hash as inputs/synth.py, implemented independently on the device.
 *   c_factor : diagonal shift c = c_factor * max_x [ ||Hrand(x)||_F + sum_{p != 40} ||A_p(x)||_F ]
 *   c_out    : host, receives c (float32-exact)
 * coarse_fill_block fills a [V][nbasis][nrhs] block with complex N(0,1) values of stream `tag`.
 */
int coarse_op_fill_synthetic(void *A_dev, const int32_t dims[4], int32_t nbasis, int32_t dtype,
                             uint64_t seed, double c_factor, double *c_out, void *stream);
int coarse_fill_block(void *X_dev, const int32_t dims[4], int32_t nbasis, int32_t nrhs, int32_t dtype,
                      uint64_t seed, int32_t tag, void *stream);

/* Introspection: name of the stencil kernel variant coarse_op_apply would launch for `nrhs`
 * (static string), bytes of device memory owned by the handle, and the number of kernels this library
 * has launched in this process so far (monotonic; used for bench.py's gpu_launches). */
const char *coarse_op_kernel_name(const coarse_op_t *op, int32_t nrhs);
int64_t coarse_op_device_bytes(const coarse_op_t *op);
/*
 * coarse_measure_peaks -- bench helper: roofline denominators measured on the current device.
 *   out_host[0] read-only HBM stream GB/s (the stencil operator is read once and never written: a copy is the wrong roof),
 *   out_host[1] FFMA, [2] packed FFMA2, [3] DFMA, [4] DMMA (mma.sync m8n8k4) TFLOP/s of register-resident loops.
 *   nout >= 5; scratch_dev: device block of scratch_bytes >= 256 MiB (larger than L2 for a meaningful stream figure; its
 *   contents are read, its first 256 bytes may be written).  Synchronises `stream`.  Nothing on the product path calls it.
 */
int coarse_measure_peaks(double *out_host, int32_t nout, void *scratch_dev, int64_t scratch_bytes, void *stream);

int64_t coarse_launch_count(void);

/* Per-launch device timing of the stencil kernel (measurement aid for bench.py's roofline object):
 * while enabled, every coarse_op_apply -- including those inside block_cg_* -- is bracketed by a CUDA event
 * pair on its launch stream (at most 64 pairs are kept).  coarse_op_profile_read synchronises on the events,
 * writes the durations in milliseconds to ms[0..*count) (host) and clears the list. */
int coarse_op_profile(coarse_op_t *op, int32_t enable);
int coarse_op_profile_read(coarse_op_t *op, double *ms, int32_t capacity, int32_t *count);

const char *coarse_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* COARSE_MRHS_H */
