/*
 * hpsd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation (complex FP64) of the
 * Euclidean projection of a Hermitian matrix onto the PSD cone,
 *
 *     X = V diag(lambda) V^H   ->   P(X) = V diag(max(lambda,0)) V^H ,
 *
 * "computing an eigendecomposition and setting all negative eigenvalues to
 * zero", on the real-vector encoding vec_R of Eq. (D10)
 * (PAPER.md:1220-1226).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code,
 * header, table or helper with the CUDA path under paper_2606_20519_b200/.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed form on
 * Q diag(lam) Q^H inputs, analytic 2x2, brute force n<=4 via the matrix sign
 * function, projection invariants (PSD, idempotent, Moreau PAPER.md:1345,
 * orthogonality), special cases, covariances, numpy eigh (complex and the
 * 2n x 2n real embedding) as third opinion.  Nothing here is "parity unpinned".
 *
 * Algorithm, step by step; textbook methods restated:
 *   1. unpack   svec -> full Hermitian array                (D10 inverse, mat_R)
 *   2. Householder tridiagonalisation with Hermitian reflectors
 *        H = I - 2 u u^H/(u^H u),  u = x + e^{i arg x_0} ||x|| e_1
 *      (Golub & Van Loan, Hermitian tridiagonalisation), Q <- Q H
 *   3. phase fix: D = diag(d_k), d_0 = 1, d_{k+1} = d_k e_k/|e_k|, so that
 *      D^H T D has the real sub-diagonal |e_k|; fold D into Q
 *   4. implicit QL with Wilkinson shift on the real (d, e), the real Givens
 *      rotations applied to the complex columns of Q (EISPACK tql2 scheme).
 *      e_m is negligible when |e_m| <= eps (|d_m| + |d_{m+1}|)  or
 *      |e_m| <= eps max_i(|d_i| + |e_i|): the second, norm-wise test (the one
 *      tql2's running `tst1` amounts to) is needed for rank-deficient inputs
 *      such as P(P(X)), whose null-space block is pure rounding noise on which
 *      the relative test alone never fires.  The paper fixes no eigensolver
 *      tolerance; both tests keep the backward error at
 *      O(n eps ||X||), which is what the pins check.
 *   5. clamp    lambda_+ = max(lambda, 0)
 *   6. rebuild  P_ij = sum_{lambda_l > 0} lambda_l z_il conj(z_jl)  (lower)
 *   7. pack     vec_R                                       (D10)
 *
 * svec layout (the library's own): block b starts at
 * sum_{c<b} n_c^2.  Inside a block the lower triangle is stored column by
 * column; column j starts at off(j) = j (2n - j) and holds
 *   [ X_jj, sqrt2 Re X_{j+1,j}, sqrt2 Im X_{j+1,j}, ..., sqrt2 Re X_{n-1,j}, sqrt2 Im X_{n-1,j} ].
 *
 * The loops over rows are spread over OpenMP threads when nthreads > 1; every
 * output element is still produced by one thread with the same operation
 * order, so the result does not depend on the thread count.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex zc;

#define A_(i, j) A[(size_t)(j) * n + (i)]
#define Q_(i, j) Q[(size_t)(j) * n + (i)]

static const double SQRT2 = 1.4142135623730951; /* nearest double to sqrt(2) */

/* ---- (D10) and its inverse ------------------------------------------------ */

/* off(j) = j (2n - j): start of column j of the lower triangle in the svec. */
static size_t col_off(int n, int j) { return (size_t)j * (size_t)(2 * n - j); }

/* mat_R: svec (n^2 doubles) -> full Hermitian n x n, column-major. */
void orc_unpack(int n, const double *sv, zc *A)
{
    for (int j = 0; j < n; ++j) {
        const double *c = sv + col_off(n, j);
        A_(j, j) = c[0];
        for (int i = j + 1; i < n; ++i) {
            double re = c[1 + 2 * (i - j - 1)] / SQRT2;
            double im = c[2 + 2 * (i - j - 1)] / SQRT2;
            A_(i, j) = re + im * I;
            A_(j, i) = re - im * I;
        }
    }
}

/* vec_R: lower triangle of a Hermitian n x n (column-major) -> svec. */
void orc_pack(int n, const zc *A, double *sv)
{
    for (int j = 0; j < n; ++j) {
        double *c = sv + col_off(n, j);
        c[0] = creal(A_(j, j));
        for (int i = j + 1; i < n; ++i) {
            c[1 + 2 * (i - j - 1)] = SQRT2 * creal(A_(i, j));
            c[2 + 2 * (i - j - 1)] = SQRT2 * cimag(A_(i, j));
        }
    }
}

/* ---- step 2+3: A = Q T Q^H with T real symmetric tridiagonal --------------- */

/* On exit d[0..n-1], e[0..n-2] hold T (e[n-1] = 0) and Q (n x n, column-major)
 * the unitary with X = Q T Q^H.  A is destroyed. */
static void tridiagonalise(int n, zc *A, zc *Q, double *d, double *e, zc *u, zc *p)
{
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) Q_(i, j) = (i == j) ? 1.0 : 0.0;

    for (int k = 0; k + 2 < n; ++k) {
        int m = n - k - 1;             /* length of x = A[k+1:, k] */
        double tail2 = 0.0;            /* ||x[1:]||^2 */
        for (int i = k + 2; i < n; ++i) {
            zc a = A_(i, k);
            tail2 += creal(a) * creal(a) + cimag(a) * cimag(a);
        }
        if (tail2 == 0.0) continue;    /* column already tridiagonal */
        zc x0 = A_(k + 1, k);
        double ax0 = cabs(x0);
        double nx = sqrt(ax0 * ax0 + tail2);
        zc phase = (ax0 > 0.0) ? x0 / ax0 : 1.0;   /* arg 0 := 0 */
        /* u = x + phase ||x|| e_1 */
        for (int i = 0; i < m; ++i) u[i] = A_(k + 1 + i, k);
        u[0] += phase * nx;
        double uu = 0.0;
        for (int i = 0; i < m; ++i) uu += creal(u[i]) * creal(u[i]) + cimag(u[i]) * cimag(u[i]);

        /* p = 2 A22 u / (u^H u),  A22 = A[k+1:, k+1:] */
#pragma omp parallel for schedule(static) if (m >= 128)
        for (int i = 0; i < m; ++i) {
            zc s = 0.0;
            for (int j = 0; j < m; ++j) s += A_(k + 1 + i, k + 1 + j) * u[j];
            p[i] = 2.0 * s / uu;
        }
        /* q = p - (u^H p / u^H u) u   (stored back in p) */
        zc up = 0.0;
        for (int i = 0; i < m; ++i) up += conj(u[i]) * p[i];
        zc kk = up / uu;
        for (int i = 0; i < m; ++i) p[i] -= kk * u[i];
        /* A22 -= u q^H + q u^H */
#pragma omp parallel for schedule(static) if (m >= 128)
        for (int j = 0; j < m; ++j) {
            zc qj = conj(p[j]), uj = conj(u[j]);
            for (int i = 0; i < m; ++i) A_(k + 1 + i, k + 1 + j) -= u[i] * qj + p[i] * uj;
        }
        /* column/row k: H x = -phase ||x|| e_1 */
        A_(k + 1, k) = -phase * nx;
        A_(k, k + 1) = conj(A_(k + 1, k));
        for (int i = k + 2; i < n; ++i) { A_(i, k) = 0.0; A_(k, i) = 0.0; }

        /* Q <- Q H on columns k+1.. :  Q[:,k+1:] -= (Q[:,k+1:] u) (2/uu) u^H */
#pragma omp parallel for schedule(static) if (n >= 128)
        for (int i = 0; i < n; ++i) {
            zc s = 0.0;
            for (int j = 0; j < m; ++j) s += Q_(i, k + 1 + j) * u[j];
            s *= 2.0 / uu;
            for (int j = 0; j < m; ++j) Q_(i, k + 1 + j) -= s * conj(u[j]);
        }
    }

    /* step 3: phase fix.  T has complex sub-diagonal t_k = A[k+1,k].  With
     * D = diag(ph_k), ph_0 = 1, ph_{k+1} = ph_k t_k/|t_k|, D^H T D is real with
     * sub-diagonal |t_k|;  X = (Q D) (D^H T D) (Q D)^H. */
    zc ph = 1.0;
    for (int k = 0; k < n; ++k) {
        d[k] = creal(A_(k, k));
        if (k > 0) {
            zc t = A_(k, k - 1);
            double at = cabs(t);
            e[k - 1] = at;
            if (at > 0.0) ph = ph * (t / at);
            double aph = cabs(ph);          /* keep |ph| = 1 against drift */
            ph /= aph;
#pragma omp parallel for schedule(static) if (n >= 1024)
            for (int i = 0; i < n; ++i) Q_(i, k) *= ph;
        }
    }
    if (n > 0) e[n - 1] = 0.0;
}

/* ---- step 4: implicit QL with Wilkinson shift ------------------------------ */

static double sign_of(double a, double b) { return (b >= 0.0) ? fabs(a) : -fabs(a); }

/* Returns 0 on success, l+1 if eigenvalue l did not converge in 60 iterations. */
static int implicit_ql(int n, double *d, double *e, zc *Q, double *cs, double *sn)
{
    const double eps = 2.220446049250313e-16; /* 2^-52 */
    double anorm = 0.0;
    for (int i = 0; i < n; ++i) {
        double t = fabs(d[i]) + (i < n - 1 ? fabs(e[i]) : 0.0);
        if (t > anorm) anorm = t;
    }
    for (int l = 0; l < n; ++l) {
        int iter = 0;
        for (;;) {
            int m;
            for (m = l; m < n - 1; ++m) {
                double dd = fabs(d[m]) + fabs(d[m + 1]);
                if (fabs(e[m]) <= eps * dd || fabs(e[m]) <= eps * anorm) break;
            }
            if (m == l) break;
            if (++iter > 60) return l + 1;
            double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
            double r = hypot(g, 1.0);
            g = d[m] - d[l] + e[l] / (g + sign_of(r, g));
            double s = 1.0, c = 1.0, p = 0.0;
            int i, underflow = 0;
            for (i = m - 1; i >= l; --i) {
                double f = s * e[i], b = c * e[i];
                r = hypot(f, g);
                e[i + 1] = r;
                if (r == 0.0) { d[i + 1] -= p; e[m] = 0.0; underflow = 1; break; }
                s = f / r; c = g / r;
                g = d[i + 1] - p;
                r = (d[i] - g) * s + 2.0 * c * b;
                p = s * r;
                d[i + 1] = g + p;
                g = c * r - b;
                cs[i] = c; sn[i] = s;
            }
            int ilo = underflow ? i + 1 : l;
            /* rotate columns (i, i+1) of Q for i = m-1 .. ilo, in that order */
#pragma omp parallel for schedule(static) if (n >= 512)
            for (int k = 0; k < n; ++k) {
                for (int ii = m - 1; ii >= ilo; --ii) {
                    zc f = Q_(k, ii + 1);
                    Q_(k, ii + 1) = sn[ii] * Q_(k, ii) + cs[ii] * f;
                    Q_(k, ii) = cs[ii] * Q_(k, ii) - sn[ii] * f;
                }
            }
            if (underflow) continue;
            d[l] -= p; e[l] = g; e[m] = 0.0;
        }
    }
    return 0;
}

/* ---- public entry points --------------------------------------------------- */

/* Full eigendecomposition of one block given as svec.  lam[n] (unsorted, as QL
 * leaves them) and Z (n x n column-major, X = Z diag(lam) Z^H).  Returns 0, or
 * >0 on QL non-convergence, or -1 on allocation failure. */
int orc_eigh_svec(int n, const double *sv, double *lam, zc *Z, int nthreads)
{
    if (n <= 0) return 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    size_t nn = (size_t)n * n;
    zc *A = malloc(nn * sizeof(zc));
    zc *u = malloc((size_t)n * sizeof(zc)), *p = malloc((size_t)n * sizeof(zc));
    double *e = malloc((size_t)n * sizeof(double));
    double *cs = malloc((size_t)n * sizeof(double)), *sn = malloc((size_t)n * sizeof(double));
    int rc = -1;
    if (A && u && p && e && cs && sn) {
        orc_unpack(n, sv, A);
        tridiagonalise(n, A, Z, lam, e, u, p);
        rc = implicit_ql(n, lam, e, Z, cs, sn);
    }
    free(A); free(u); free(p); free(e); free(cs); free(sn);
    return rc;
}

/* Projection of one block: svec in -> svec out. */
int orc_project_block(int n, const double *in, double *out, int nthreads)
{
    if (n <= 0) return 0;
    size_t nn = (size_t)n * n;
    double *lam = malloc((size_t)n * sizeof(double));
    zc *Z = malloc(nn * sizeof(zc));
    zc *P = malloc(nn * sizeof(zc));
    int rc = -1;
    if (lam && Z && P) {
        rc = orc_eigh_svec(n, in, lam, Z, nthreads);
        if (rc == 0) {
            /* step 5 + 6: clamp and rebuild the lower triangle */
#pragma omp parallel for schedule(dynamic, 8) if (n >= 128)
            for (int j = 0; j < n; ++j) {
                for (int i = j; i < n; ++i) {
                    zc s = 0.0;
                    for (int l = 0; l < n; ++l) {
                        double lp = lam[l] > 0.0 ? lam[l] : 0.0;
                        if (lp > 0.0) s += lp * Z[(size_t)l * n + i] * conj(Z[(size_t)l * n + j]);
                    }
                    P[(size_t)j * n + i] = s;
                }
            }
            orc_pack(n, P, out); /* step 7 */
        }
    }
    free(lam); free(Z); free(P);
    return rc;
}

/* Projection of a block list, same signature shape as the library's
 * hpsd_project but on HOST pointers.  Returns 0 or the first failing code. */
int orc_project(int n_blocks, const int *sizes, const double *in, double *out, int nthreads)
{
    size_t off = 0;
    for (int b = 0; b < n_blocks; ++b) {
        int n = sizes[b];
        if (n < 0) return -2;
        int rc = orc_project_block(n, in + off, out + off, nthreads);
        if (rc != 0) return rc;
        off += (size_t)n * n;
    }
    return 0;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
