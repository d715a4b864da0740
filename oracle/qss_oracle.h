/* CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct fp64 (and float128 / dual-number / complex-step) evaluation of the
 * per-cell QSS chemistry of arXiv 2405.05974: rate constants -> algebraic QSS closure
 * (Eq. 4, Eq. 6) -> net production rates (Eq. 2-3) -> analytical Jacobian d wdot / d[C,T] with the
 * chain rule through the closure (Eq. 7, Eq. 9).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call this.
 * It shares no code, header, table or helper with the CUDA path (paper_2405_05974_b200/, include/).
 *
 * Layout: SoA, cell innermost.  C[k*ld + c] (k < N transported), T[c], wdot[i*ld + c],
 * cqss[m*ld + c], S[i*ld + c], jac[(i*(N+1) + j)*ld + c] (row i: species rate, column j < N: C_j,
 * column N: T), jscale same shape as jac.  All pointers are HOST pointers.
 * Units: mol, m^3, s, K, J.  R = 8.31446261815324 J/(mol K), P0 = 101325 Pa.
 */
#ifndef QSS_ORACLE_H
#define QSS_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t n_nqss, n_qss, n_reac;
    const double  *nasa_T;            /* [n_sp*3]  Tlow Tmid Thigh                           */
    const double  *nasa_lo, *nasa_hi; /* [n_sp*7]  a1..a7 below / at-or-above Tmid            */
    const int32_t *rtype;             /* [n_reac]  0 Arrhenius 1 third-body 2 Troe falloff    */
    const uint8_t *dir_mask;          /* [n_reac]  bit0 forward enabled, bit1 reverse enabled */
    const int32_t *reac_ptr, *reac_sp, *reac_nu;   /* CSR reactants, nu' > 0 */
    const int32_t *prod_ptr, *prod_sp, *prod_nu;   /* CSR products,  nu'' > 0 */
    const double  *arr;               /* [n_reac*3] A, beta, Ea[J/mol] (k_inf for type 2)     */
    const double  *arr_low;           /* [n_reac*3] k_0 parameters, type 2                    */
    const double  *troe;              /* [n_reac*4] alpha, T***, T*, T**, type 2              */
    const int32_t *eff_ptr, *eff_sp;  /* CSR non-unity third-body efficiencies                */
    const double  *eff_val;
} oracle_mech_t;

enum {
    ORACLE_EXPLICIT_F64   = 0,  /* explicit formulas, double (the reference values and the timed CPU baseline) */
    ORACLE_EXPLICIT_F128  = 1,  /* same formulas in __float128, rounded to double at the end (referee)         */
    ORACLE_JAC_DUAL       = 2,  /* Jacobian by forward-mode dual numbers through the wdot routine              */
    ORACLE_JAC_CSTEP      = 3,  /* Jacobian by complex step (h = 1e-30) through the wdot routine               */
    ORACLE_JAC_CONST_QSS  = 4,  /* explicit formulas with the chain term W_y*Y_x dropped        */
    ORACLE_JAC_ZERO_QSS   = 5   /* chain term dropped AND C_QSS := 0 in the partials ("zero QSS AJ") */
};

/* Any output pointer may be NULL (skipped). Returns 0, or -1 on a bad argument.
 * wdot/cqss/S are always from the explicit routine in the precision `mode` implies. */
int oracle_eval(const oracle_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                double *wdot, double *cqss, double *S, double *jac, double *jscale, int mode, int nthreads);

/* NEXT-1 (Eq. 7): temperature right-hand side of the adiabatic constant-volume reactor,
 *   tdot[c] = -T sum_i (h_i/RT - 1) wdot_i / sum_i C_i (cp_i/R - 1)   (sums over the transported species, reading G17),
 * and the energy row of the (N+1) x (N+1) Jacobian, erow[k*ld + c] = d Tdot / d C_k (k < N), d Tdot / d T (k = N);
 * escale: running-error scale of the row (explicit modes only).  mode: ORACLE_EXPLICIT_F64 / _F128 / _JAC_DUAL / _JAC_CSTEP. */
int oracle_eval_energy(const oracle_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                       double *tdot, double *erow, double *escale, int mode, int nthreads);

/* NEXT-2 (reading G20): x_c = (I - gamma_c J_c)^-1 b_c by Gaussian elimination with partial
 * pivoting, J_c the (N+1) x (N+1) Jacobian (rows 0..N-1 jac, row N erow), or its N x N species block when erow == NULL.
 * gamma [ncells], b and x [n*ld], info NULL or [ncells] (0, or k+1: zero pivot at step k).  quad != 0: __float128 arithmetic.
 * (qss_newton_oracle.cpp) */
int oracle_newton_solve(int N, int64_t ncells, int64_t ld, const double *jac, const double *erow, const double *gamma,
                        const double *b, double *x, int32_t *info, int quad);

/* One cell: effective forward / reverse rate constants (k including the third-body or fall-off factor,
 * kb = k / Kc; 0 for a disabled direction). kf, kb: [n_reac]. */
int oracle_rate_constants(const oracle_mech_t *m, const double *C, double T, double *kf, double *kb);

/* One cell: QSS closure residual g_m = sum_n P[m][n] y_n - D_m y_m + p0_m and the sum of |terms|. */
int oracle_closure_check(const oracle_mech_t *m, const double *C, double T, double *y, double *res,
                         double *res_scale);

int oracle_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
