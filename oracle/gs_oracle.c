/*
 * gs_oracle.c -- plain, slow, obviously-correct CPU oracle.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the CUDA path
 * (paper_2502_02460_b200/csrc, include/gs.h) and neither includes the other.
 *
 * What it computes ("Solving the generalized eigenproblem"):
 *   1. Cholesky decomposition  S = U^T U, U upper triangular              (step 1)
 *   2. Inversion of the upper triangular matrix  U -> U^-1                (step 2)
 *   3. two matrix products  H~ = (U^-1)^T H U^-1                          (step 3)
 *   4. back-transformation  C = U^-1 C~
 *   "A^T corresponds to the transpose or conjugate-transpose of a real- or complex-valued matrix"
 *   (PAPER.md:67), so the complex routines use the conjugate transpose throughout.
 * plus, off the GPU hot path, a cyclic Jacobi eigensolver for the standard problem
 *   H~ C~ = eps C~ so that eigen-level checks do not need a library.
 *
 * Steps 1-4 are exact direct methods; the oracle is their plain definition: unblocked Cholesky,
 * substitution-based inversion, triple-loop products (BASELINE.json north_star).  No blocking, no
 * fusion, no BLAS/LAPACK.  The only liberties, none of which changes which numbers are multiplied
 * and added:
 *   - loops skip operands that are exactly zero by triangularity;
 *   - loop nests are ordered so the innermost index runs down a column (column-major storage);
 *   - `#pragma omp parallel for` over independent output columns only.
 *
 * Layout: column-major, leading dimension N (C~ and C: N x nev, ld N); complex = C99 double _Complex
 * (interleaved re,im).  All pointers are HOST pointers.  Readings of silent points:
 * Q1 unique factor with real positive diagonal; Q4 only the upper triangle of S / U is read, the
 * strictly-lower part of U and U^-1 is written as zero; Q6 non-positive (or NaN) pivot -> return
 * its 1-based index, no regularisation.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): diagonal pencil closed form, S = I, the
 * tridiag(-1,2,-1) closed forms for U, U^-1, H~ and eps, 2x2 quadratic, Sturm/inertia brute force
 * at tiny N, planted factor, complex = real (x) phase identity, scipy/LAPACK cross-checks; the density
 * matrix (O7): hand-computed case fixing the conjugate, electron count sum_ij P_ij S_ij = sum_l f_l,
 * projector identity, numpy einsum (tests/test_oracle_density.py).
 * NEXT-4 helpers (the standard eigenproblem between steps 3 and 4, whose stages the paper's
 * Table 1 calls "Tridiag. / Solve / Back"): the oracle for eps and C~ stays the Jacobi
 * method above; O8/O9 (Sturm count and bisection on a symmetric tridiagonal matrix) check the INTERMEDIATE
 * tridiagonal matrix a GPU tridiagonalisation emits (same eigenvalues as H~), and O10 (inertia of A - sigma I
 * by LDL^H without pivoting) proves that a set of computed eigenvalues is the LOWEST nev with none missing.
 * Pins (tests/test_oracle_tridiag.py): closed-form spectrum of tridiag(-1,2,-1), diagonal and 2 x 2 cases,
 * Jacobi on the same matrix, inertia against brute-force eigenvalue counts and a hand-computed LDL^T.
 * (5) truncated-basis route for an ill-conditioned S: O11 plain triple-loop products C = A^H B and
 * C = A B; the route itself is assembled from O5 (Jacobi on S and on H_r) and O11 in oracle/__init__.py,
 * step by step in the paper's order.  Pins (tests/test_oracle_truncated.py): commuting pencil with planted
 * near-null directions (closed form eps_i = h_i / sigma_i on the kept directions), delta = 0 reproduces the
 * Cholesky route's eigenvalues, numpy products.
 * No function here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex zdouble;
#define AT(a, i, j) ((a)[(size_t)(i) + (size_t)(j) * (size_t)N])

/* ------------------------------------------------------------------------------------------ */
/* O1. Unblocked Cholesky S = U^H U.  In place: on entry the upper triangle of S, */
/* on exit U in the upper triangle and zeros below.  Row-by-row (Crout) form:                   */
/*   U(j,j) = sqrt( S(j,j) - sum_{k<j} |U(k,j)|^2 )                                             */
/*   U(j,i) = ( S(j,i) - sum_{k<j} conj(U(k,j)) U(k,i) ) / U(j,j),   i > j                      */
/* Returns 0, or the 1-based index j+1 of the first pivot that is not > 0 (also catches NaN).   */
/* ------------------------------------------------------------------------------------------ */
int64_t orc_cholesky_d(int64_t N, double *S)
{
    for (int64_t j = 0; j < N; ++j) {
        double d = AT(S, j, j);
        for (int64_t k = 0; k < j; ++k) d -= AT(S, k, j) * AT(S, k, j);
        if (!(d > 0.0)) return j + 1;
        const double ujj = sqrt(d);
        AT(S, j, j) = ujj;
#pragma omp parallel for schedule(static)
        for (int64_t i = j + 1; i < N; ++i) {
            double s = AT(S, j, i);
            for (int64_t k = 0; k < j; ++k) s -= AT(S, k, j) * AT(S, k, i);
            AT(S, j, i) = s / ujj;
        }
    }
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = j + 1; i < N; ++i) AT(S, i, j) = 0.0;
    return 0;
}

int64_t orc_cholesky_z(int64_t N, zdouble *S)
{
    for (int64_t j = 0; j < N; ++j) {
        double d = creal(AT(S, j, j));
        for (int64_t k = 0; k < j; ++k) {
            const zdouble u = AT(S, k, j);
            d -= creal(u) * creal(u) + cimag(u) * cimag(u);
        }
        if (!(d > 0.0)) return j + 1;
        const double ujj = sqrt(d);
        AT(S, j, j) = ujj; /* real, positive (reading Q1) */
#pragma omp parallel for schedule(static)
        for (int64_t i = j + 1; i < N; ++i) {
            zdouble s = AT(S, j, i);
            for (int64_t k = 0; k < j; ++k) s -= conj(AT(S, k, j)) * AT(S, k, i);
            AT(S, j, i) = s / ujj;
        }
    }
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = j + 1; i < N; ++i) AT(S, i, j) = 0.0;
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* O2. Substitution-based inversion U -> V = U^-1.  Solves U V = I one column at  */
/* a time by back substitution (column-oriented form): for column j, b = e_j;                   */
/*   for k = j .. 0:  V(k,j) = b_k / U(k,k);  b_i -= U(i,k) V(k,j)  for i < k.                  */
/* Only the upper triangle of U is read; strictly-lower part of V is zero.                      */
/* Returns 0, or 1-based index of a zero diagonal entry.                                        */
/* ------------------------------------------------------------------------------------------ */
int64_t orc_invert_upper_d(int64_t N, const double *U, double *V)
{
    for (int64_t k = 0; k < N; ++k)
        if (AT(U, k, k) == 0.0) return k + 1;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j) {
        double *b = &AT(V, 0, j);
        for (int64_t i = 0; i < N; ++i) b[i] = 0.0;
        b[j] = 1.0;
        for (int64_t k = j; k >= 0; --k) {
            const double x = b[k] / AT(U, k, k);
            b[k] = x;
            for (int64_t i = 0; i < k; ++i) b[i] -= AT(U, i, k) * x;
        }
    }
    return 0;
}

int64_t orc_invert_upper_z(int64_t N, const zdouble *U, zdouble *V)
{
    for (int64_t k = 0; k < N; ++k)
        if (AT(U, k, k) == 0.0) return k + 1;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j) {
        zdouble *b = &AT(V, 0, j);
        for (int64_t i = 0; i < N; ++i) b[i] = 0.0;
        b[j] = 1.0;
        for (int64_t k = j; k >= 0; --k) {
            const zdouble x = b[k] / AT(U, k, k);
            b[k] = x;
            for (int64_t i = 0; i < k; ++i) b[i] -= AT(U, i, k) * x;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* O3. Two matrix products H~ = V^H H V, V = U^-1 upper triangular.               */
/*   W(i,j)  = sum_{k<=j} H(i,k) V(k,j)             (all i,j; V(k,j) = 0 for k > j)             */
/*   H~(i,j) = sum_{k<=i} conj(V(k,i)) W(k,j)       (all i,j -- BOTH triangles are computed     */
/*             independently, so symmetry of the result is a check, not an assumption)          */
/* W is caller-provided scratch (N x N).  All of H is read (both triangles), upper triangle of V.*/
/* ------------------------------------------------------------------------------------------ */
void orc_to_standard_d(int64_t N, const double *H, const double *V, double *W, double *Ht)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j) {
        double *w = &AT(W, 0, j);
        for (int64_t i = 0; i < N; ++i) w[i] = 0.0;
        for (int64_t k = 0; k <= j; ++k) {
            const double v = AT(V, k, j);
            const double *h = &AT(H, 0, k);
            for (int64_t i = 0; i < N; ++i) w[i] += h[i] * v;
        }
    }
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) {
            double s = 0.0;
            for (int64_t k = 0; k <= i; ++k) s += AT(V, k, i) * AT(W, k, j);
            AT(Ht, i, j) = s;
        }
}

void orc_to_standard_z(int64_t N, const zdouble *H, const zdouble *V, zdouble *W, zdouble *Ht)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j) {
        zdouble *w = &AT(W, 0, j);
        for (int64_t i = 0; i < N; ++i) w[i] = 0.0;
        for (int64_t k = 0; k <= j; ++k) {
            const zdouble v = AT(V, k, j);
            const zdouble *h = &AT(H, 0, k);
            for (int64_t i = 0; i < N; ++i) w[i] += h[i] * v;
        }
    }
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) {
            zdouble s = 0.0;
            for (int64_t k = 0; k <= i; ++k) s += conj(AT(V, k, i)) * AT(W, k, j);
            AT(Ht, i, j) = s;
        }
}

/* ------------------------------------------------------------------------------------------ */
/* O4. Back-transformation C = V C~, V = U^-1 upper, C~ and C are N x nev (ld N): */
/*   C(i,j) = sum_{k>=i} V(i,k) C~(k,j).   No conjugation (reading Q2).                         */
/* ------------------------------------------------------------------------------------------ */
void orc_backtransform_d(int64_t N, int64_t nev, const double *V, const double *Ct, double *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < nev; ++j) {
        double *c = &AT(C, 0, j);
        for (int64_t i = 0; i < N; ++i) c[i] = 0.0;
        for (int64_t k = 0; k < N; ++k) {
            const double x = AT(Ct, k, j);
            const double *v = &AT(V, 0, k);
            for (int64_t i = 0; i <= k; ++i) c[i] += v[i] * x;
        }
    }
}

void orc_backtransform_z(int64_t N, int64_t nev, const zdouble *V, const zdouble *Ct, zdouble *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < nev; ++j) {
        zdouble *c = &AT(C, 0, j);
        for (int64_t i = 0; i < N; ++i) c[i] = 0.0;
        for (int64_t k = 0; k < N; ++k) {
            const zdouble x = AT(Ct, k, j);
            const zdouble *v = &AT(V, 0, k);
            for (int64_t i = 0; i <= k; ++i) c[i] += v[i] * x;
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O5. Cyclic Jacobi for the standard problem A Q = Q diag(eps) ("H~ C~ = eps C~"). */
/* Off the GPU hot path.  Textbook method (Golub & Van Loan, Matrix Computations, sec. 8.5):    */
/* row-cyclic sweeps over p < q; for each pair, with a = A(p,q) = |a| e^{i phi},                */
/*   theta = (A(q,q) - A(p,p)) / (2|a|),  t = sign(theta) / (|theta| + sqrt(theta^2 + 1)),      */
/*   c = 1/sqrt(1+t^2),  s = t c,                                                               */
/* and the unitary R = I except R(p,p) = c, R(p,q) = s e^{i phi}, R(q,p) = -s e^{-i phi},       */
/* R(q,q) = c;  A <- R^H A R annihilates A(p,q);  Q <- Q R.  (Real case: e^{i phi} = +-1.)      */
/* A: full Hermitian N x N on entry (both triangles), destroyed.  Q: N x N out (eigenvectors as */
/* columns).  eps: N eigenvalues ascending; columns of Q ordered alike.            */
/* Stops when a whole sweep rotates nothing (every |A(p,q)| <= 2^-52 ||A||_F / N).  Returns the  */
/* number of sweeps used, or -1 if 60 sweeps did not suffice.                                   */
/* ------------------------------------------------------------------------------------------ */
static void sort_eigs_d(int64_t N, double *eps, double *Q)
{
    /* stable insertion sort on eps, moving columns of Q alike */
    double *col = (double *)malloc(sizeof(double) * (size_t)N);
    for (int64_t a = 1; a < N; ++a) {
        const double e = eps[a];
        memcpy(col, &AT(Q, 0, a), sizeof(double) * (size_t)N);
        int64_t b = a - 1;
        while (b >= 0 && eps[b] > e) {
            eps[b + 1] = eps[b];
            memcpy(&AT(Q, 0, b + 1), &AT(Q, 0, b), sizeof(double) * (size_t)N);
            --b;
        }
        eps[b + 1] = e;
        memcpy(&AT(Q, 0, b + 1), col, sizeof(double) * (size_t)N);
    }
    free(col);
}

int64_t orc_jacobi_d(int64_t N, double *A, double *eps, double *Q)
{
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) AT(Q, i, j) = (i == j) ? 1.0 : 0.0;
    double fro = 0.0;
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) fro += AT(A, i, j) * AT(A, i, j);
    fro = sqrt(fro);
    const double tol = ldexp(1.0, -52) * fro / (double)(N > 0 ? N : 1);
    int64_t sweeps = 0;
    for (; sweeps < 60; ++sweeps) {
        int64_t rotations = 0;
        for (int64_t p = 0; p < N - 1; ++p)
            for (int64_t q = p + 1; q < N; ++q) {
                const double apq = AT(A, p, q);
                if (!(fabs(apq) > tol)) continue;
                ++rotations;
                const double theta = (AT(A, q, q) - AT(A, p, p)) / (2.0 * apq);
                const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                /* columns p,q:  A <- A R */
                for (int64_t i = 0; i < N; ++i) {
                    const double aip = AT(A, i, p), aiq = AT(A, i, q);
                    AT(A, i, p) = c * aip - s * aiq;
                    AT(A, i, q) = s * aip + c * aiq;
                }
                /* rows p,q:  A <- R^T A */
                for (int64_t j = 0; j < N; ++j) {
                    const double apj = AT(A, p, j), aqj = AT(A, q, j);
                    AT(A, p, j) = c * apj - s * aqj;
                    AT(A, q, j) = s * apj + c * aqj;
                }
                AT(A, p, q) = 0.0;
                AT(A, q, p) = 0.0;
                for (int64_t i = 0; i < N; ++i) {
                    const double qip = AT(Q, i, p), qiq = AT(Q, i, q);
                    AT(Q, i, p) = c * qip - s * qiq;
                    AT(Q, i, q) = s * qip + c * qiq;
                }
            }
        if (rotations == 0) break;
    }
    if (sweeps == 60) return -1;
    for (int64_t i = 0; i < N; ++i) eps[i] = AT(A, i, i);
    sort_eigs_d(N, eps, Q);
    return sweeps + 1;
}

static void sort_eigs_z(int64_t N, double *eps, zdouble *Q)
{
    zdouble *col = (zdouble *)malloc(sizeof(zdouble) * (size_t)N);
    for (int64_t a = 1; a < N; ++a) {
        const double e = eps[a];
        memcpy(col, &AT(Q, 0, a), sizeof(zdouble) * (size_t)N);
        int64_t b = a - 1;
        while (b >= 0 && eps[b] > e) {
            eps[b + 1] = eps[b];
            memcpy(&AT(Q, 0, b + 1), &AT(Q, 0, b), sizeof(zdouble) * (size_t)N);
            --b;
        }
        eps[b + 1] = e;
        memcpy(&AT(Q, 0, b + 1), col, sizeof(zdouble) * (size_t)N);
    }
    free(col);
}

int64_t orc_jacobi_z(int64_t N, zdouble *A, double *eps, zdouble *Q)
{
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) AT(Q, i, j) = (i == j) ? 1.0 : 0.0;
    double fro = 0.0;
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) {
            const zdouble a = AT(A, i, j);
            fro += creal(a) * creal(a) + cimag(a) * cimag(a);
        }
    fro = sqrt(fro);
    const double tol = ldexp(1.0, -52) * fro / (double)(N > 0 ? N : 1);
    int64_t sweeps = 0;
    for (; sweeps < 60; ++sweeps) {
        int64_t rotations = 0;
        for (int64_t p = 0; p < N - 1; ++p)
            for (int64_t q = p + 1; q < N; ++q) {
                const zdouble apq = AT(A, p, q);
                const double alpha = cabs(apq);
                if (!(alpha > tol)) continue;
                ++rotations;
                const zdouble ph = apq / alpha; /* e^{i phi} */
                const double theta = (creal(AT(A, q, q)) - creal(AT(A, p, p))) / (2.0 * alpha);
                const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                const zdouble rpq = s * ph;        /* R(p,q) =  s e^{ i phi} */
                const zdouble rqp = -s * conj(ph); /* R(q,p) = -s e^{-i phi} */
                /* A <- A R : col p = c*col p + rqp*col q ; col q = rpq*col p + c*col q */
                for (int64_t i = 0; i < N; ++i) {
                    const zdouble aip = AT(A, i, p), aiq = AT(A, i, q);
                    AT(A, i, p) = c * aip + rqp * aiq;
                    AT(A, i, q) = rpq * aip + c * aiq;
                }
                /* A <- R^H A : row p = c*row p + conj(rqp)*row q ; row q = conj(rpq)*row p + c*row q */
                for (int64_t j = 0; j < N; ++j) {
                    const zdouble apj = AT(A, p, j), aqj = AT(A, q, j);
                    AT(A, p, j) = c * apj + conj(rqp) * aqj;
                    AT(A, q, j) = conj(rpq) * apj + c * aqj;
                }
                AT(A, p, q) = 0.0;
                AT(A, q, p) = 0.0;
                AT(A, p, p) = creal(AT(A, p, p));
                AT(A, q, q) = creal(AT(A, q, q));
                for (int64_t i = 0; i < N; ++i) {
                    const zdouble qip = AT(Q, i, p), qiq = AT(Q, i, q);
                    AT(Q, i, p) = c * qip + rqp * qiq;
                    AT(Q, i, q) = rpq * qip + c * qiq;
                }
            }
        if (rotations == 0) break;
    }
    if (sweeps == 60) return -1;
    for (int64_t i = 0; i < N; ++i) eps[i] = creal(AT(A, i, i));
    sort_eigs_z(N, eps, Q);
    return sweeps + 1;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* O7 (NEXT-1, off the four-step path). Single-particle density matrix:            */
/*   P_ij = sum_l f_l c*_li c_lj,   c_li = C(i,l) (eigenvectors stored as columns)  */
/* Plain triple loop over all i, j (both triangles computed independently).                     */
/* ------------------------------------------------------------------------------------------ */
void orc_density_d(int64_t N, int64_t nev, const double *C, const double *f, double *P)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) {
            double s = 0.0;
            for (int64_t l = 0; l < nev; ++l) s += f[l] * AT(C, i, l) * AT(C, j, l);
            AT(P, i, j) = s;
        }
}

void orc_density_z(int64_t N, int64_t nev, const zdouble *C, const double *f, zdouble *P)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < N; ++i) {
            zdouble s = 0.0;
            for (int64_t l = 0; l < nev; ++l) s += f[l] * conj(AT(C, i, l)) * AT(C, j, l);
            AT(P, i, j) = s;
        }
}

/* ------------------------------------------------------------------------------------------ */
/* O8. Sturm count: the number of eigenvalues of the real symmetric tridiagonal matrix          */
/* T = tridiag(e, d, e) (d: n diagonal, e: n-1 off-diagonal entries) that are < x.              */
/* Sylvester's law of inertia applied to T - x I = L D L^T (Golub & Van Loan sec. 8.4.2;        */
/* Parlett, The Symmetric Eigenvalue Problem, sec. 3.3):                                        */
/*   q_0 = d_0 - x,   q_i = d_i - x - e_{i-1}^2 / q_{i-1},   count = #{ i : q_i < 0 }.          */
/* A pivot that is exactly zero is replaced by -tiny (the usual convention: it counts as        */
/* negative, i.e. an eigenvalue equal to x is counted as "< x" only through rounding).          */
/* ------------------------------------------------------------------------------------------ */
int64_t orc_sturm_count(int64_t n, const double *d, const double *e, double x)
{
    int64_t count = 0;
    double q = 1.0;
    for (int64_t i = 0; i < n; ++i) {
        const double off = (i == 0) ? 0.0 : e[i - 1] * e[i - 1] / q;
        q = d[i] - x - off;
        if (q == 0.0) q = -1e-300;
        if (q < 0.0) ++count;
    }
    return count;
}

/* O9. The k-th smallest eigenvalue (k = 0 .. n-1) of T by bisection on the Gershgorin interval:   */
/* invariant count(lo) <= k < count(hi); stops when the interval cannot be halved any more in FP64. */
double orc_tridiag_eigenvalue(int64_t n, const double *d, const double *e, int64_t k)
{
    double lo = d[0], hi = d[0];
    for (int64_t i = 0; i < n; ++i) {
        const double r = (i > 0 ? fabs(e[i - 1]) : 0.0) + (i + 1 < n ? fabs(e[i]) : 0.0);
        if (d[i] - r < lo) lo = d[i] - r;
        if (d[i] + r > hi) hi = d[i] + r;
    }
    const double pad = 2.0 * ldexp(1.0, -52) * (fabs(lo) > fabs(hi) ? fabs(lo) : fabs(hi)) * (double)n + 1e-300;
    lo -= pad;
    hi += pad;
    for (int it = 0; it < 2000; ++it) {
        const double mid = lo + 0.5 * (hi - lo);
        if (!(mid > lo && mid < hi)) break;
        if (orc_sturm_count(n, d, e, mid) <= k) lo = mid; else hi = mid;
    }
    return lo + 0.5 * (hi - lo);
}

void orc_tridiag_eigenvalues(int64_t n, const double *d, const double *e, int64_t nev, double *eps)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < nev; ++k) eps[k] = orc_tridiag_eigenvalue(n, d, e, k);
}

/* ------------------------------------------------------------------------------------------ */
/* O10. Inertia: the number of eigenvalues of the Hermitian matrix A that are < sigma, as the    */
/* number of negative pivots of A - sigma I = L D L^H (symmetric Gaussian elimination WITHOUT    */
/* pivoting; Sylvester's law of inertia).  A: full N x N on entry (the upper triangle is read),  */
/* destroyed.  Returns -1 if a pivot is exactly zero (sigma hit an eigenvalue of a leading       */
/* block: choose another sigma).  Independent of Cholesky, Jacobi and of any tridiagonalisation. */
/*   for j: p_j = A(j,j);  for i > j: l = conj(A(j,i)) / p_j;  A(i, c) -= l A(j, c), c >= i.      */
/* ------------------------------------------------------------------------------------------ */
int64_t orc_inertia_d(int64_t N, double *A, double sigma)
{
    int64_t neg = 0;
    for (int64_t j = 0; j < N; ++j) AT(A, j, j) -= sigma;
    for (int64_t j = 0; j < N; ++j) {
        const double p = AT(A, j, j);
        if (p == 0.0 || p != p) return -1;
        if (p < 0.0) ++neg;
#pragma omp parallel for schedule(static)
        for (int64_t c = j + 1; c < N; ++c) {
            const double ajc = AT(A, j, c);
            if (ajc == 0.0) continue;
            for (int64_t i = j + 1; i <= c; ++i) AT(A, i, c) -= (AT(A, j, i) / p) * ajc;
        }
    }
    return neg;
}

int64_t orc_inertia_z(int64_t N, zdouble *A, double sigma)
{
    int64_t neg = 0;
    for (int64_t j = 0; j < N; ++j) AT(A, j, j) = creal(AT(A, j, j)) - sigma;
    for (int64_t j = 0; j < N; ++j) {
        const double p = creal(AT(A, j, j));
        if (p == 0.0 || p != p) return -1;
        if (p < 0.0) ++neg;
#pragma omp parallel for schedule(static)
        for (int64_t c = j + 1; c < N; ++c) {
            const zdouble ajc = AT(A, j, c);
            if (ajc == 0.0) continue;
            for (int64_t i = j + 1; i <= c; ++i) AT(A, i, c) -= (conj(AT(A, j, i)) / p) * ajc;
            AT(A, c, c) = creal(AT(A, c, c));
        }
    }
    return neg;
}

/* ------------------------------------------------------------------------------------------ */
/* O11. Plain triple-loop products (column-major, leading dimensions = row counts):             */
/*   orc_matmul_hn:  C (M x N) = A^H B,  A is K x M, B is K x N                                 */
/*   orc_matmul_nn:  C (M x N) = A B,    A is M x K, B is K x N                                 */
/* Used by the truncated-basis route of PAPER.md:73 (H_r = X^H H X, C = X y).                   */
/* ------------------------------------------------------------------------------------------ */
void orc_matmul_hn_d(int64_t M, int64_t N, int64_t K, const double *A, const double *B, double *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < M; ++i) {
            double s = 0.0;
            for (int64_t k = 0; k < K; ++k) s += A[k + i * K] * B[k + j * K];
            C[i + j * M] = s;
        }
}

void orc_matmul_hn_z(int64_t M, int64_t N, int64_t K, const zdouble *A, const zdouble *B, zdouble *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < M; ++i) {
            zdouble s = 0.0;
            for (int64_t k = 0; k < K; ++k) s += conj(A[k + i * K]) * B[k + j * K];
            C[i + j * M] = s;
        }
}

void orc_matmul_nn_d(int64_t M, int64_t N, int64_t K, const double *A, const double *B, double *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < M; ++i) {
            double s = 0.0;
            for (int64_t k = 0; k < K; ++k) s += A[i + k * M] * B[k + j * K];
            C[i + j * M] = s;
        }
}

void orc_matmul_nn_z(int64_t M, int64_t N, int64_t K, const zdouble *A, const zdouble *B, zdouble *C)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < M; ++i) {
            zdouble s = 0.0;
            for (int64_t k = 0; k < K; ++k) s += A[i + k * M] * B[k + j * K];
            C[i + j * M] = s;
        }
}
