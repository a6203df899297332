/*
 * CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct implementation of the data-parallel hot path of the multiple
 * right-hand-side HDCG method of arXiv:2409.03904, written from /root/reference/PAPER.md:
 *
 *   - oracle_apply*      : the coarse-grid operator applied to a block of Nrhs vectors,
 *                          Y(x) = sum_p A^p(x) . X(x + delta_p)         (Eq. 19;
 *                          81-point stencil of relative shifts (-1..1)^4)
 *   - oracle_gram        : the s x s block inner product U^H W           (Table 6 "ThinQR")
 *   - oracle_cholesky_upper, oracle_upper_inverse, oracle_hpd_inverse :
 *                          the small dense algebra of BlockCGrQ
 *   - oracle_block_rotate: the block rotation W = beta W + U K
 *   - oracle_block_cg    : BlockCGrQ, Fig. 2 (left), step by step in the paper's
 *                          order and notation, with the X-update read as X + D M C (reading R1).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or constant with the CUDA path (paper_2409_03904_b200/csrc) and
 * neither includes the other.  All arithmetic is complex128 (double re/im pairs), whatever the
 * storage type of A.  Parallelism: OpenMP over lattice sites (apply) / columns (Gram); no blocking,
 * fusion or reordering beyond the loop nests written here.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): dense brute-force matrix on tiny lattices,
 * pure-shift closed form, Fourier symbol closed form, Hermiticity invariant, scipy BSR product,
 * numpy.linalg.solve for block CG, s=1 reduction to textbook CG, O'Leary block-CG iterates,
 * per-iteration invariants (Q^H Q = I, R = Q C), Chebyshev convergence bound.  No function here is
 * "parity unpinned".
 *
 * Layouts (canonical boundary layouts):
 *   site index   x = x0 + L0*(x1 + L1*(x2 + L2*x3))
 *   stencil pt   p = (d0+1) + 3(d1+1) + 9(d2+1) + 27(d3+1)
 *   A : [site][81][nb][nb]   row-major nb x nb blocks, interleaved (re, im); float or double storage
 *   X, Y : [site][nb][s]     column index r fastest; interleaved (re, im) doubles
 *   s x s matrices : row-major, interleaved doubles
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_NOT_CONVERGED (-5)
#define ORACLE_BREAKDOWN (-6)
#define ORACLE_A_C64 0
#define ORACLE_A_C128 1

typedef struct { double re, im; } zd;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* x + delta_p with periodic wrap (PAPER.md:298 relative shifts; single-GPU build wraps periodically,
 * DESIGN.md reading R7).  Coordinate arithmetic, no table. */
int64_t oracle_neighbour(const int32_t dims[4], int64_t x, int32_t p)
{
    int64_t y = 0, stride = 1, rem = x;
    int32_t q = p;
    for (int k = 0; k < 4; ++k) {
        int64_t L = dims[k];
        int64_t c = rem % L;
        rem /= L;
        int64_t d = (q % 3) - 1;
        q /= 3;
        int64_t cn = (c + d + L) % L;
        y += cn * stride;
        stride *= L;
    }
    return y;
}

static inline zd load_a(const void *A, int a_dtype, int64_t e)
{
    zd v;
    if (a_dtype == ORACLE_A_C64) {
        const float *f = (const float *)A;
        v.re = (double)f[2 * e];
        v.im = (double)f[2 * e + 1];
    } else {
        const double *d = (const double *)A;
        v.re = d[2 * e];
        v.im = d[2 * e + 1];
    }
    return v;
}

/*
 * Y[k] = sum_{p=0}^{80} A[k][p] . X[nbr(site_k, p)]   for the listed sites.   (Eq. 19 summed over p)
 *   A_sub : matrices of the listed sites only, [n_sites][81][nb][nb]
 *   X     : the whole block, [V][nb][s]
 *   Y_sub : [n_sites][nb][s]
 *   sites : the n_sites site indices, or NULL for sites 0..n_sites-1
 *   p_only: -1 for the full stencil, else accumulate only that stencil point (tests)
 */
void oracle_apply_sites(const int32_t dims[4], int32_t nb, int32_t s, int32_t a_dtype,
                        const void *A_sub, const double *X, double *Y_sub,
                        int64_t n_sites, const int64_t *sites, int32_t p_only)
{
    const zd *Xz = (const zd *)X;
    zd *Yz = (zd *)Y_sub;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n_sites; ++k) {
        int64_t x = sites ? sites[k] : k;
        zd *y = Yz + k * (int64_t)nb * s;
        for (int64_t e = 0; e < (int64_t)nb * s; ++e) { y[e].re = 0.0; y[e].im = 0.0; }
        for (int32_t p = 0; p < 81; ++p) {
            if (p_only >= 0 && p != p_only) continue;
            int64_t nbr = oracle_neighbour(dims, x, p);
            const zd *xin = Xz + nbr * (int64_t)nb * s;
            int64_t abase = (k * 81 + p) * (int64_t)nb * nb;
            for (int32_t i = 0; i < nb; ++i)
                for (int32_t j = 0; j < nb; ++j) {
                    zd a = load_a(A_sub, a_dtype, abase + (int64_t)i * nb + j);
                    for (int32_t r = 0; r < s; ++r) {
                        zd b = xin[(int64_t)j * s + r];
                        y[(int64_t)i * s + r].re += a.re * b.re - a.im * b.im;
                        y[(int64_t)i * s + r].im += a.re * b.im + a.im * b.re;
                    }
                }
        }
    }
}

void oracle_apply(const int32_t dims[4], int32_t nb, int32_t s, int32_t a_dtype,
                  const void *A, const double *X, double *Y)
{
    int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    oracle_apply_sites(dims, nb, s, a_dtype, A, X, Y, V, NULL, -1);
}

/* G = U^H W : G[a][b] = sum_k conj(U[k][a]) W[k][b],  U, W : [n][s], G : [s][s] */
void oracle_gram(int64_t n, int32_t s, const double *U, const double *W, double *G)
{
    const zd *Uz = (const zd *)U, *Wz = (const zd *)W;
    zd *Gz = (zd *)G;
#pragma omp parallel for schedule(static) collapse(2)
    for (int32_t a = 0; a < s; ++a)
        for (int32_t b = 0; b < s; ++b) {
            double re = 0.0, im = 0.0;
            for (int64_t k = 0; k < n; ++k) {
                zd u = Uz[k * s + a], w = Wz[k * s + b];
                re += u.re * w.re + u.im * w.im;
                im += u.re * w.im - u.im * w.re;
            }
            Gz[a * s + b].re = re;
            Gz[a * s + b].im = im;
        }
}

/* W = U . K  (n x s times s x s) */
static void block_times_small(int64_t n, int32_t s, const zd *U, const zd *K, zd *W)
{
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k)
        for (int32_t b = 0; b < s; ++b) {
            double re = 0.0, im = 0.0;
            for (int32_t a = 0; a < s; ++a) {
                zd u = U[k * s + a], m = K[a * s + b];
                re += u.re * m.re - u.im * m.im;
                im += u.re * m.im + u.im * m.re;
            }
            W[k * s + b].re = re;
            W[k * s + b].im = im;
        }
}

/* Block rotation as one exported call (the "block rotations" of PAPER.md:145-149):
 * W = beta * W + U . K, U, W : [n][s], K : [s][s].  Same loop nest as block_times_small above. */
void oracle_block_rotate(int64_t n, int32_t s, const double *U, const double *K, double beta, double *W)
{
    zd *tmp = (zd *)malloc(sizeof(zd) * (size_t)n * s);
    zd *Wz = (zd *)W;
    block_times_small(n, s, (const zd *)U, (const zd *)K, tmp);
    for (int64_t e = 0; e < n * s; ++e) {
        Wz[e].re = beta * Wz[e].re + tmp[e].re;
        Wz[e].im = beta * Wz[e].im + tmp[e].im;
    }
    free(tmp);
}

static void small_matmul(int32_t s, const zd *P, const zd *Q, zd *R) /* R = P Q */
{
    for (int32_t a = 0; a < s; ++a)
        for (int32_t b = 0; b < s; ++b) {
            double re = 0.0, im = 0.0;
            for (int32_t c = 0; c < s; ++c) {
                zd u = P[a * s + c], v = Q[c * s + b];
                re += u.re * v.re - u.im * v.im;
                im += u.re * v.im + u.im * v.re;
            }
            R[a * s + b].re = re;
            R[a * s + b].im = im;
        }
}

static void small_adjoint(int32_t s, const zd *P, zd *R) /* R = P^H */
{
    for (int32_t a = 0; a < s; ++a)
        for (int32_t b = 0; b < s; ++b) {
            R[a * s + b].re = P[b * s + a].re;
            R[a * s + b].im = -P[b * s + a].im;
        }
}

/*
 * Cholesky factorisation in the form the paper keeps explicit: G = S^H S with S upper
 * triangular and a real positive diagonal (unique).  G is symmetrised (G + G^H)/2 first.  Returns
 * ORACLE_BREAKDOWN if a pivot is not positive (reading R12: no column deflation).
 * Textbook row-by-row algorithm:  S[a][a] = sqrt(G[a][a] - sum_{c<a} |S[c][a]|^2),
 *                                 S[a][b] = (G[a][b] - sum_{c<a} conj(S[c][a]) S[c][b]) / S[a][a],  b > a.
 */
int oracle_cholesky_upper(int32_t s, const double *G, double *S)
{
    const zd *Gz = (const zd *)G;
    zd *Sz = (zd *)S;
    for (int32_t e = 0; e < s * s; ++e) { Sz[e].re = 0.0; Sz[e].im = 0.0; }
    for (int32_t a = 0; a < s; ++a) {
        double d = Gz[a * s + a].re;
        for (int32_t c = 0; c < a; ++c)
            d -= Sz[c * s + a].re * Sz[c * s + a].re + Sz[c * s + a].im * Sz[c * s + a].im;
        if (!(d > 0.0) || !isfinite(d)) return ORACLE_BREAKDOWN;
        double saa = sqrt(d);
        Sz[a * s + a].re = saa;
        for (int32_t b = a + 1; b < s; ++b) {
            double re = 0.5 * (Gz[a * s + b].re + Gz[b * s + a].re);
            double im = 0.5 * (Gz[a * s + b].im - Gz[b * s + a].im);
            for (int32_t c = 0; c < a; ++c) {
                zd u = Sz[c * s + a], v = Sz[c * s + b]; /* conj(u) * v */
                re -= u.re * v.re + u.im * v.im;
                im -= u.re * v.im - u.im * v.re;
            }
            Sz[a * s + b].re = re / saa;
            Sz[a * s + b].im = im / saa;
        }
    }
    return ORACLE_OK;
}

/* Inverse of an upper triangular matrix by back substitution, column by column: S . Sinv = I. */
void oracle_upper_inverse(int32_t s, const double *S, double *Sinv)
{
    const zd *Sz = (const zd *)S;
    zd *Iz = (zd *)Sinv;
    for (int32_t e = 0; e < s * s; ++e) { Iz[e].re = 0.0; Iz[e].im = 0.0; }
    for (int32_t b = 0; b < s; ++b)
        for (int32_t a = b; a >= 0; --a) {
            double re = (a == b) ? 1.0 : 0.0, im = 0.0;
            for (int32_t c = a + 1; c <= b; ++c) {
                zd u = Sz[a * s + c], v = Iz[c * s + b];
                re -= u.re * v.re - u.im * v.im;
                im -= u.re * v.im + u.im * v.re;
            }
            zd d = Sz[a * s + a];
            double den = d.re * d.re + d.im * d.im;
            Iz[a * s + b].re = (re * d.re + im * d.im) / den;
            Iz[a * s + b].im = (im * d.re - re * d.im) / den;
        }
}

/* Inverse of a Hermitian positive definite s x s matrix through its Cholesky factor:
 * G = S^H S  =>  G^{-1} = S^{-1} S^{-H}.  (M_k = [D_k^H Z_k]^{-1}) */
int oracle_hpd_inverse(int32_t s, const double *G, double *Ginv)
{
    zd *S = (zd *)malloc(sizeof(zd) * s * s), *Si = (zd *)malloc(sizeof(zd) * s * s),
       *SiH = (zd *)malloc(sizeof(zd) * s * s);
    int st = oracle_cholesky_upper(s, G, (double *)S);
    if (st == ORACLE_OK) {
        oracle_upper_inverse(s, (const double *)S, (double *)Si);
        small_adjoint(s, Si, SiH);
        small_matmul(s, Si, SiH, (zd *)Ginv);
    }
    free(S); free(Si); free(SiH);
    return st;
}

/* ------------------------------------------------------------------------------------------------
 * BlockCGrQ  (Fig. 2 left), statement by statement.
 *
 *   4.  R_0 = B - H X_0
 *   5.  Q_0 C_0 = R_0            thin QR by Cholesky: C_0^H C_0 = R_0^H R_0, Q_0 = R_0 C_0^{-1}
 *   6.  D_0 = Q_0
 *   7.  for k = 0, 1, 2, ...
 *   8.      Z_k = H D_k
 *   9.      M_k = [D_k^H Z_k]^{-1}
 *   10.     X_{k+1} = X_k + D_k M_k C_k      (the listing prints "X_k + D_k M_k"; the C_k factor is
 *                                             forced by R_k = Q_k C_k and C_{k+1} = S_{k+1} C_k:
 *                                             DESIGN.md reading R1)
 *   11.     Q_{k+1} S_{k+1} = Q_k - Z_k M_k   thin QR by Cholesky of T^H T, T = Q_k - Z_k M_k
 *   12.     D_{k+1} = Q_{k+1} + D_k S_{k+1}^H
 *   13.     C_{k+1} = S_{k+1} C_k
 *   stop when max_r ||C_{k+1}[:,r]||_2 / ||B[:,r]||_2 <= tol   (R = Q C, Q^H Q = I => ||R[:,r]|| = ||C[:,r]||;
 *                                                               DESIGN.md reading R4)
 *
 *   B, X : [n][s] with n = V*nb (X in: X_0, out: solution);  history : [(maxiter+1)][s] recursive
 *   relative residuals (row 0 = initial);  true_rel : [s] ||B - H X||/||B|| from one extra apply.
 *   callback (may be NULL) is called with (k, X_k, Q_k, D_k, C_k) for k = 0 (after step 6) and after
 *   every iteration -- tests use it to check invariants of the iterates.
 *   Returns ORACLE_OK, ORACLE_NOT_CONVERGED (maxiter hit; outputs valid) or ORACLE_BREAKDOWN.
 * ------------------------------------------------------------------------------------------------ */
typedef void (*oracle_bcg_callback)(int32_t k, const double *X, const double *Q, const double *D,
                                    const double *C, void *user);

static void column_norms(int64_t n, int32_t s, const zd *U, double *out)
{
    for (int32_t r = 0; r < s; ++r) {
        double acc = 0.0;
        for (int64_t k = 0; k < n; ++k) acc += U[k * s + r].re * U[k * s + r].re + U[k * s + r].im * U[k * s + r].im;
        out[r] = sqrt(acc);
    }
}

int oracle_block_cg(const int32_t dims[4], int32_t nb, int32_t s, int32_t a_dtype, const void *A,
                    const double *B, double *X, double tol, int32_t maxiter,
                    int32_t *iterations, double *history, double *true_rel,
                    oracle_bcg_callback callback, void *user)
{
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    const int64_t n = V * nb, ns = n * s;
    const zd *Bz = (const zd *)B;
    zd *Xz = (zd *)X;
    zd *Q = (zd *)malloc(sizeof(zd) * ns), *D = (zd *)malloc(sizeof(zd) * ns), *Z = (zd *)malloc(sizeof(zd) * ns),
       *T = (zd *)malloc(sizeof(zd) * ns), *W = (zd *)malloc(sizeof(zd) * ns);
    zd *G = (zd *)malloc(sizeof(zd) * s * s), *C = (zd *)malloc(sizeof(zd) * s * s), *S = (zd *)malloc(sizeof(zd) * s * s),
       *M = (zd *)malloc(sizeof(zd) * s * s), *K1 = (zd *)malloc(sizeof(zd) * s * s), *K2 = (zd *)malloc(sizeof(zd) * s * s);
    double *bnorm = (double *)malloc(sizeof(double) * s), *cn = (double *)malloc(sizeof(double) * s);
    int status = ORACLE_NOT_CONVERGED;
    int32_t its = 0;

    column_norms(n, s, Bz, bnorm);
    for (int32_t r = 0; r < s; ++r) if (bnorm[r] == 0.0) bnorm[r] = 1.0;   /* zero source: absolute residual */

    /* 4. R_0 = B - H X_0   (R is held in T) */
    oracle_apply(dims, nb, s, a_dtype, A, X, (double *)T);
    for (int64_t e = 0; e < ns; ++e) { T[e].re = Bz[e].re - T[e].re; T[e].im = Bz[e].im - T[e].im; }
    /* 5. Q_0 C_0 = R_0 */
    oracle_gram(n, s, (const double *)T, (const double *)T, (double *)G);
    double worst = 0.0;
    for (int32_t r = 0; r < s; ++r) {
        double rel = sqrt(fmax(G[r * s + r].re, 0.0)) / bnorm[r];
        history[r] = rel;
        if (rel > worst) worst = rel;
    }
    if (worst <= tol) { status = ORACLE_OK; goto finish; }
    if (oracle_cholesky_upper(s, (const double *)G, (double *)C) != ORACLE_OK) { status = ORACLE_BREAKDOWN; goto finish; }
    oracle_upper_inverse(s, (const double *)C, (double *)K1);
    block_times_small(n, s, T, K1, Q);
    /* 6. D_0 = Q_0 */
    memcpy(D, Q, sizeof(zd) * ns);
    if (callback) callback(0, X, (const double *)Q, (const double *)D, (const double *)C, user);

    for (int32_t k = 0; k < maxiter; ++k) {
        /* 8. Z_k = H D_k */
        oracle_apply(dims, nb, s, a_dtype, A, (const double *)D, (double *)Z);
        /* 9. M_k = [D_k^H Z_k]^{-1} */
        oracle_gram(n, s, (const double *)D, (const double *)Z, (double *)G);
        if (oracle_hpd_inverse(s, (const double *)G, (double *)M) != ORACLE_OK) { status = ORACLE_BREAKDOWN; its = k; goto finish; }
        /* 10. X_{k+1} = X_k + D_k (M_k C_k) */
        small_matmul(s, M, C, K1);
        block_times_small(n, s, D, K1, W);
        for (int64_t e = 0; e < ns; ++e) { Xz[e].re += W[e].re; Xz[e].im += W[e].im; }
        /* 11. Q_{k+1} S_{k+1} = Q_k - Z_k M_k */
        block_times_small(n, s, Z, M, W);
        for (int64_t e = 0; e < ns; ++e) { T[e].re = Q[e].re - W[e].re; T[e].im = Q[e].im - W[e].im; }
        oracle_gram(n, s, (const double *)T, (const double *)T, (double *)G);
        if (oracle_cholesky_upper(s, (const double *)G, (double *)S) != ORACLE_OK) { status = ORACLE_BREAKDOWN; its = k + 1; goto finish; }
        oracle_upper_inverse(s, (const double *)S, (double *)K1);
        block_times_small(n, s, T, K1, Q);
        /* 12. D_{k+1} = Q_{k+1} + D_k S_{k+1}^H */
        small_adjoint(s, S, K1);
        block_times_small(n, s, D, K1, W);
        for (int64_t e = 0; e < ns; ++e) { D[e].re = Q[e].re + W[e].re; D[e].im = Q[e].im + W[e].im; }
        /* 13. C_{k+1} = S_{k+1} C_k */
        small_matmul(s, S, C, K2);
        memcpy(C, K2, sizeof(zd) * s * s);
        its = k + 1;
        /* stop test on the recursive residual ||C[:,r]|| / ||B[:,r]|| */
        worst = 0.0;
        for (int32_t r = 0; r < s; ++r) {
            double acc = 0.0;
            for (int32_t a = 0; a < s; ++a) acc += C[a * s + r].re * C[a * s + r].re + C[a * s + r].im * C[a * s + r].im;
            double rel = sqrt(acc) / bnorm[r];
            history[(int64_t)(k + 1) * s + r] = rel;
            if (rel > worst) worst = rel;
        }
        if (callback) callback(k + 1, X, (const double *)Q, (const double *)D, (const double *)C, user);
        if (worst <= tol) { status = ORACLE_OK; break; }
    }

finish:
    *iterations = its;
    /* true residual ||B - H X|| / ||B|| per column, one extra apply */
    oracle_apply(dims, nb, s, a_dtype, A, X, (double *)W);
    for (int64_t e = 0; e < ns; ++e) { W[e].re = Bz[e].re - W[e].re; W[e].im = Bz[e].im - W[e].im; }
    column_norms(n, s, W, cn);
    for (int32_t r = 0; r < s; ++r) true_rel[r] = cn[r] / bnorm[r];
    free(Q); free(D); free(Z); free(T); free(W); free(G); free(C); free(S); free(M); free(K1); free(K2);
    free(bnorm); free(cn);
    return status;
}
