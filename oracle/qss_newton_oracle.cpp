/* CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * NEXT-2: the dense direct solve of the Newton system that consumes the chemical Jacobian
 * ("relying on forming and inverting the chemical Jacobian of phi ... to advance the Newton step", Eq. 7;
 * L397 "a dense direct linear solve from the MAGMA library which uses an analytic Jacobian").  The paper does not write the
 * matrix; reading G20: the Newton matrix of an implicit multistep method (CVODE's form),
 *     M_c = I - gamma_c J_c,      J_c the (N+1) x (N+1) Jacobian of cell c over phi = {C_1..C_N, T} (Eq. 7),
 * rows 0..N-1 from the species block (jac), row N the energy row (erow); gamma_c = h_c * beta is per cell (every cell has
 * its own step size).  Solve M_c x_c = b_c.
 *
 * The oracle is the textbook definition written out: Gaussian elimination with partial pivoting (row interchanges, the
 * largest |entry| of the column at or below the diagonal, the first one on ties), multipliers by division, then forward
 * and back substitution -- one cell at a time, no blocking.  In double, or in __float128 rounded at the end (referee).
 * With erow == NULL the system is the N x N species block (columns 0..N-1 of jac; constant temperature).
 *
 * Layout as in qss_oracle.h: jac[(i*(N+1) + j)*ld + c], erow[j*ld + c], gamma[c], b[i*ld + c], x[i*ld + c], i < n.
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>

#include <vector>

namespace {

template <class S> S s_abs(S v) { return v < S(0) ? -v : v; }

/* A: n x n row-major (destroyed), rhs: n (overwritten by the solution).  Returns 0, or k+1 when the pivot of step k is 0. */
template <class S>
int lu_solve(int n, std::vector<S> &A, std::vector<S> &rhs) {
    int info = 0;
    for (int k = 0; k < n; ++k) {
        int p = k;
        S best = s_abs(A[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i) {
            const S v = s_abs(A[(size_t)i * n + k]);
            if (v > best) { best = v; p = i; }
        }
        if (p != k) {
            for (int j = 0; j < n; ++j) { const S t = A[(size_t)k * n + j]; A[(size_t)k * n + j] = A[(size_t)p * n + j]; A[(size_t)p * n + j] = t; }
            const S t = rhs[k]; rhs[k] = rhs[p]; rhs[p] = t;
        }
        const S piv = A[(size_t)k * n + k];
        if (piv == S(0) && info == 0) info = k + 1;
        for (int i = k + 1; i < n; ++i) {
            const S l = A[(size_t)i * n + k] / piv;
            A[(size_t)i * n + k] = l;
            for (int j = k + 1; j < n; ++j) A[(size_t)i * n + j] -= l * A[(size_t)k * n + j];
            rhs[i] -= l * rhs[k];
        }
    }
    for (int k = n - 1; k >= 0; --k) {
        S s = rhs[k];
        for (int j = k + 1; j < n; ++j) s -= A[(size_t)k * n + j] * rhs[j];
        rhs[k] = s / A[(size_t)k * n + k];
    }
    return info;
}

template <class S>
int solve_cell(int N, int n, int64_t c, int64_t ld, const double *jac, const double *erow, double g, const double *b, double *x,
               std::vector<S> &A, std::vector<S> &r) {
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) {
            const double J = i < N ? jac[((size_t)i * (N + 1) + j) * ld + c] : erow[(size_t)j * ld + c];
            A[(size_t)i * n + j] = (i == j ? S(1) : S(0)) - S(g) * S(J);
        }
        r[i] = S(b[(size_t)i * ld + c]);
    }
    const int info = lu_solve<S>(n, A, r);
    for (int i = 0; i < n; ++i) x[(size_t)i * ld + c] = (double)r[i];
    return info;
}

}  // namespace

/* N: transported species.  erow may be NULL (n = N), else n = N + 1.  info: NULL, or [ncells] (0, or k+1: zero pivot at step k).
 * quad != 0: arithmetic in __float128.  Returns 0, or -1 on a bad argument. */
extern "C" int oracle_newton_solve(int N, int64_t ncells, int64_t ld, const double *jac, const double *erow, const double *gamma,
                                   const double *b, double *x, int32_t *info, int quad) {
    if (N < 1 || ncells < 0 || ld < ncells || !jac || !gamma || !b || !x) return -1;
    const int n = erow ? N + 1 : N;
#pragma omp parallel
    {
        std::vector<double> Ad((size_t)n * n), rd(n);
        std::vector<__float128> Aq(quad ? (size_t)n * n : 0), rq(quad ? n : 0);
#pragma omp for schedule(static)
        for (int64_t c = 0; c < ncells; ++c) {
            const int rc = quad ? solve_cell<__float128>(N, n, c, ld, jac, erow, gamma[c], b, x, Aq, rq)
                                : solve_cell<double>(N, n, c, ld, jac, erow, gamma[c], b, x, Ad, rd);
            if (info) info[c] = rc;
        }
    }
    return 0;
}
