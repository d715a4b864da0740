/* qss.h -- C-ABI of libqss: batched per-cell evaluation of QSS-reduced chemistry on one B200 (sm_100a).
 *
 * What is computed (PAPER.md = arXiv 2405.05974; readings G1..G15 are listed in DESIGN.md):
 *   - mass-action rates  Q_j = kf_j prod C^nu' - kb_j prod C^nu''           PAPER.md Eq. 2 (L59)
 *   - net production     wdot_i = sum_j nu_ij Q_j                             PAPER.md Eq. 3 (L64)
 *   - QSS closure        dC_q/dt = 0 for the N_q QSS species, a linear system
 *                        A C_QSS = b solved per cell, group by group          PAPER.md Eq. 4 (L71), Eq. 6 (L150-157),
 *                                                                             ordering L159-173, App. B
 *   - analytical Jacobian J_ik = d wdot_i / d phi_k, phi = {C_1..C_N, T},
 *                        with the chain rule through the closure              PAPER.md Eq. 7 (L185), Eq. 9 (L224)
 *   Rate-constant forms (Arrhenius, third body, Troe fall-off, reverse rates from NASA-7 equilibrium
 *   constants) are the standard CHEMKIN forms the paper leaves implicit (L278, L461); DESIGN.md "Readings" G4.
 *
 * Layout (all DEVICE buffers are SoA, cell innermost; `ld` is the cell stride, ld >= ncells; a stride that is not a power of two,
 * e.g. ncells rounded up to a multiple of 32 plus 64, avoids rows that start exact MiB apart: measured up to 9 % faster):
 *   C[k*ld + c]      k < N transported species, mol/m^3        T[c]   K
 *   wdot[i*ld + c]   i < N, mol/(m^3 s)                         cqss[q*ld + c]  q < N_q, mol/m^3
 *   jac[(i*(N+1) + k)*ld + c]   row i < N: species whose rate is differentiated,
 *                               column k < N: d/dC_k, column k = N: d/dT        (N x (N+1) block, reading G5)
 * Units: mol, m^3, s, K, J.  R = 8.31446261815324 J/(mol K), P0 = 101325 Pa.  Pressure is not an input.
 *
 * Ownership: the caller owns every device buffer including `workspace` (size from qss_mech_info); the
 * library owns only the handle and its device tables (allocated in qss_mech_create on `device`, freed in
 * qss_mech_destroy).  The arrays of qss_mech_desc_t are HOST pointers borrowed for the duration of
 * qss_mech_create only.
 *
 * Execution: qss_eval_* enqueue kernels on `stream` (a cudaStream_t passed as void*) and return; they do
 * not synchronise, allocate, or touch the default stream, and may be captured in a CUDA graph.
 *
 * Errors: every function returns QSS_OK (0) or a negative qss_status; nothing throws or aborts across the
 * ABI.  qss_last_error() returns a thread-local message for the last failure.
 * Preconditions NOT checked on the hot path: T > 0, C >= 0, every QSS species has a positive consumption
 * coefficient, third-body concentration > 0 for fall-off reactions.  NaN/Inf propagate.
 * There is no CPU fallback: without a CUDA device qss_mech_create fails with QSS_E_CUDA.
 *
 * Run-time specialisation: for mechanisms of up to 60 species, qss_mech_create generates
 * CUDA source for this mechanism (every size a compile-time constant; closure and Jacobian columns as straight-line code)
 * and compiles it with NVRTC (libnvrtc.so.12, opened with dlopen; seconds per mechanism, then read from an on-disk cache of
 * device images: $QSS_CACHE_DIR, else $XDG_CACHE_HOME/libqss, else ~/.cache/libqss; QSS_CACHE=0 switches it off).
 * Optional: without NVRTC the table-driven kernels compute the same thing (qss_mech_info.kernel_variant_jac tells which
 * one runs).  Environment read at qss_mech_create by the release build: QSS_VARIANT=0..3 (force a variant, fail when it does
 * not apply), QSS_JIT=0 (no run-time compilation) / 2 (failed compilation is an error), QSS_CACHE, QSS_CACHE_DIR,
 * QSS_CS_GLOBAL (test knob of variant 1).  Nothing is read on the launch path.
 *
 * Threads: a handle may be used from several host threads; the device calls only enqueue work on the caller's stream (the
 * caller orders kernels that share a workspace); qss_eval_jac_host serialises on a mutex of the handle.  qss_mech_destroy
 * synchronises the device before it frees the tables, so work still in flight on any stream finishes first.
 */
#ifndef QSS_H
#define QSS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    QSS_OK = 0,
    QSS_E_INVALID = -1,      /* null pointer, bad size / index / alignment, ld < ncells, workspace too small */
    QSS_E_QUADRATIC = -2,    /* an enabled direction consumes >= 2 QSS molecules (linearise first, L77) */
    QSS_E_QSS_FANOUT = -3,   /* an enabled direction produces >= 2 QSS molecules                                  */
    QSS_E_NO_SINK = -4,      /* a QSS species cannot reach a transported species: closure structurally singular  */
    QSS_E_UNSUPPORTED = -5,  /* reaction type outside {0,1,2}, non-positive stoichiometric coefficient          */
    QSS_E_CUDA = -6,         /* a CUDA runtime call failed (message in qss_last_error)                         */
    QSS_E_UNBALANCED = -7    /* strict_balance: a reaction does not conserve an element (needs comp)          */
} qss_status;

typedef struct qss_mech qss_mech_t;   /* opaque */

/* Mechanism description. All pointers are HOST pointers. Species 0..n_nqss-1 are transported,
 * n_nqss..n_nqss+n_qss-1 are QSS. */
typedef struct {
    int32_t n_elem, n_nqss, n_qss, n_reac;
    const double  *elem_weight;            /* [n_elem] g/mol (may be NULL; not used on the hot path)          */
    const int32_t *comp;                   /* [(n_nqss+n_qss)*n_elem] species-major (may be NULL)             */
    const double  *nasa_T;                 /* [n_sp*3]  Tlow, Tmid, Thigh                                     */
    const double  *nasa_lo, *nasa_hi;      /* [n_sp*7]  a1..a7 for T < Tmid / T >= Tmid (reading G9)           */
    const int32_t *type;                   /* [n_reac]  0 Arrhenius, 1 third-body, 2 Troe fall-off            */
    const uint8_t *dir_mask;               /* [n_reac]  bit0 forward enabled, bit1 reverse enabled (G10)      */
    const int32_t *reac_ptr, *reac_sp, *reac_nu;   /* CSR reactants, nu' positive integers (G11)              */
    const int32_t *prod_ptr, *prod_sp, *prod_nu;   /* CSR products,  nu''                                     */
    const double  *arr;                    /* [n_reac*3] A, beta, Ea[J/mol]; high-pressure limit for type 2   */
    const double  *arr_low;                /* [n_reac*3] low-pressure limit, read for type 2 only             */
    const double  *troe;                   /* [n_reac*4] alpha, T***, T*, T**, read for type 2 only           */
    const int32_t *eff_ptr, *eff_sp;       /* CSR non-unity third-body efficiencies, transported species only */
    const double  *eff_val;                /*   (third-body concentration M = sum_{k<N} alpha_k C_k, G7)      */
    int32_t strict_balance;                /* != 0: qss_mech_create / _validate check sum_s nu_s comp[s][e] = 0 for every
                                            * reaction and element and fail with QSS_E_UNBALANCED (comp must be given);
                                            * the conservation pins of wdot and of the Jacobian's null space rest on it */
} qss_mech_desc_t;

typedef struct {
    int32_t n_nqss, n_qss, n_reac;
    int32_t n_groups, max_group;           /* QSS coupling groups (SCCs of the QSS digraph)  */
    int32_t n_levels;                      /* depth of the condensed DAG of groups                             */
    int32_t group_size[64];                /* sizes of the first min(n_groups, 64) groups, in solve order      */
    /* algorithmic cost per cell of the sparse method: fp64-pipe instruction slots
     * (add = mul = fma = 1, exp 18, log 30, division 24, reciprocal 22) and bytes (inputs read once, outputs
     * written once) */
    double  slots_wdot, slots_jac;
    double  bytes_wdot, bytes_jac;
    /* workspace the caller must supply to qss_eval_wdot / qss_eval_jac (device memory, 256-byte aligned);
     * independent of ncells */
    size_t  workspace_bytes_wdot, workspace_bytes_jac;
    /* which kernel the library selected: 0 general slab kernel, 1 slab-smem kernel (table
     * interpreter), 2 slab-smem kernel with the Jacobian sweep specialised for this mechanism at qss_mech_create,
     * 3 the kernel generated for this mechanism as a whole, rate phases with lane = reaction (NVRTC; images cached
     * on disk; 2 and 3 fall back to 1 when NVRTC is missing) */
    int32_t kernel_variant_wdot, kernel_variant_jac;
} qss_mech_info_t;

/* Validate `desc`, order the QSS groups (Tarjan SCC + topological order), build the static elimination
 * schedules and gather tables, and upload them to `device`.  On success *out receives the handle. */
int qss_mech_create(const qss_mech_desc_t *desc, int device, qss_mech_t **out);
int qss_mech_destroy(qss_mech_t *mech);
int qss_mech_info(const qss_mech_t *mech, qss_mech_info_t *out);

/* Solve order of the QSS species: order[i] is the local QSS index (0..n_qss-1) solved i-th, group_of[i]
 * the group it belongs to (groups numbered in solve order).  HOST arrays of n_qss entries. For tests. */
int qss_mech_qss_order(const qss_mech_t *mech, int32_t *order, int32_t *group_of);

/* Host-only part of qss_mech_create (no CUDA call): validates `desc` and reports the QSS solve order.
 * n_groups, order[n_qss], group_of[n_qss] may each be NULL. Same return codes as qss_mech_create. */
int qss_mech_validate(const qss_mech_desc_t *desc, int32_t *n_groups, int32_t *order, int32_t *group_of);

/* Host-only check of the run-time specialisation (no CUDA call, no device needed): validates `desc`, generates the
 * mechanism-specialised source of the Jacobian kernel (the paper's generated-code idea,
 * PAPER.md L324-326, applied to pass A of the sweep) and compiles it with NVRTC for compute capability
 * cc_major.cc_minor (10.0 = B200).  *image_bytes (may be NULL) receives the size of the device image.
 * Returns QSS_OK; QSS_E_UNSUPPORTED when the mechanism does not fit kernel variant 1 (nothing to specialise);
 * QSS_E_CUDA when NVRTC is missing or the compilation fails (qss_last_error() holds the compiler log). */
int qss_mech_specialise_check(const qss_mech_desc_t *desc, int cc_major, int cc_minor, size_t *image_bytes);

/* wdot (and optionally the closure's C_QSS) for ncells cells.  C, T, wdot, cqss_or_null, workspace are
 * DEVICE pointers, 16-byte aligned; stream is a cudaStream_t.  ncells == 0 is a no-op. */
int qss_eval_wdot(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T,
                  double *wdot, double *cqss_or_null, void *workspace, size_t workspace_bytes, void *stream);

/* Analytical Jacobian d wdot / d[C,T] (and optionally wdot in the same pass). */
int qss_eval_jac(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T,
                 double *jac, double *wdot_or_null, void *workspace, size_t workspace_bytes, void *stream);

/* The paper's simplified Jacobians (Table 5a), cheap modes of the same kernel:
 *   QSS_JAC_EXACT      the exact analytical Jacobian of qss_eval_jac (Eq. 9)
 *   QSS_JAC_CONST_QSS  "constant QSS AJ": the second term of Eq. 9 (chain rule through the closure) is dropped
 *   QSS_JAC_ZERO_QSS   "zero QSS AJ": additionally the QSS concentrations are nullified in every partial derivative
 * Same layout and workspace as qss_eval_jac; wdot is not produced.  Returns QSS_E_UNSUPPORTED when the handle does not run
 * kernel variant 3 (qss_mech_info.kernel_variant_jac != 3). */
typedef enum { QSS_JAC_EXACT = 0, QSS_JAC_CONST_QSS = 1, QSS_JAC_ZERO_QSS = 2 } qss_jac_mode;
int qss_eval_jac_approx(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac,
                        int mode, void *workspace, size_t workspace_bytes, void *stream);

/* NEXT-1 of the build plan: the last row of the paper's (N+1) x (N+1) Jacobian (Eq. 7; state {C, T} L181) and the
 * temperature right-hand side, for the adiabatic constant-volume reactor the paper integrates (L190), "simply obtained from
 * the species production rates" (L278) and the NASA-7 polynomials (reading G17; sums over the transported species):
 *   tdot[c]        = -T sum_i (h_i/RT - 1) wdot_i / sum_i C_i (cp_i/R - 1)                      K/s
 *   erow[k*ld + c] = d tdot / d C_k (k < N),  d tdot / d T (k = N)
 * Inputs: the state and the outputs wdot, jac of qss_eval_jac for the same cells (DEVICE pointers, same layout, 16-byte
 * aligned); outputs tdot [ld], erow [(N+1)*ld].  One kernel on `stream`, bound by reading jac once.  N <= 430. */
int qss_eval_energy(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T, const double *wdot,
                    const double *jac, double *tdot, double *erow, void *stream);

/* NEXT-2: the dense direct solve of the Newton system that consumes the Jacobian (Eq. 7:
 * "forming and inverting the chemical Jacobian ... to advance the Newton step"; L397: the MAGMA batched dense direct solve of
 * Case 3).  The paper does not write the matrix; reading G20: the Newton matrix of an implicit multistep method,
 *   x_c = (I - gamma_c J_c)^-1 b_c        per cell c, by Gaussian elimination with partial pivoting,
 * J_c the (N+1) x (N+1) Jacobian of Eq. 7: rows 0..N-1 = jac (output of qss_eval_jac), row N = erow (output of qss_eval_energy).
 * With erow == NULL the system is the N x N species block (columns 0..N-1 of jac; temperature frozen).  n = N + 1 or N.
 * DEVICE pointers, 8-byte aligned, SoA cell innermost: jac [N*(N+1)*ld], erow [(N+1)*ld], gamma [ncells] (= h_c * beta: every
 * cell has its own step size), b and x [n*ld]; x may alias b.  Nothing else is written.  A singular matrix gives non-finite x
 * (no error).  One kernel on `stream`, no workspace; the matrix is read once from HBM.  n <= 40 (QSS_E_UNSUPPORTED above: the matrix
 * is held in the registers of one warp).  The kernel is compiled for n with NVRTC on the FIRST call per handle and shape (seconds,
 * or milliseconds from the on-disk cache; that first call must not be inside a stream capture; QSS_E_CUDA without NVRTC).
 * qss_newton_specialise_check compiles the kernel for a compute capability without a device (build check). */
int qss_newton_solve(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *jac, const double *erow_or_null,
                     const double *gamma, const double *b, double *x, void *stream);
int qss_newton_specialise_check(int n_species, int with_energy, int cc_major, int cc_minor, size_t *image_bytes_or_null);

/* Mapping micro-benchmark, NOT part of the path (north_star subsystem 3: cell-to-thread vs cell-to-warp with warp shuffles for the
 * species-parallel reductions): wdot[i*ld + c] = sum_j nu_ij Q[j*ld + c] (Eq. 3) for i < N from given rates of progress Q [M*ld]
 * (DEVICE pointers), mode 0: lane = cell, every species' reaction list walked per lane; mode 1: a warp per cell, lane = reaction,
 * contributions scattered per lane and every species reduced over the lanes by a SHFL butterfly.  Same staging of Q through shared
 * memory and same coalesced output in both.  QSS_E_UNSUPPORTED when the slab does not fit one SM's shared memory.
 * has the measurement that decided the mapping of the kernels. */
int qss_bench_species_sums(const qss_mech_t *mech, int mode, int64_t ncells, int64_t ld, const double *Q, double *wdot, void *stream);

/* Allocation-free variant of qss_eval_wdot, for callers that cannot provide (or allocate) a workspace: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc.  Same inputs, outputs, layout and results as qss_eval_wdot; the
 * workspace is a static device array of QSS_STATIC_SCRATCH_BYTES bytes inside the library, which every GPU that loads the library
 * holds until the process exits (its device address is taken once per device at qss_mech_create).  The call launches the general
 * slab kernel (kernel variant 0, whatever variant the handle selected for qss_eval_wdot) with as many persistent blocks as fit the
 * array, and calls no allocating routine.  Limit: a mechanism whose ONE-block workspace exceeds the array is rejected with
 * QSS_E_UNSUPPORTED (more than 32 768 doubles of per-cell workspace, roughly 7 000 reactions; the BASELINE configs need
 * 0.03-2.3 MB per block); any ncells is accepted.  Every call on a device shares the array: calls that overlap on the GPU (two streams, two handles, two threads) race;
 * order them on one stream.  Nothing in the array has to start at zero: the kernel writes every row before it reads it. */
#define QSS_STATIC_SCRATCH_BYTES (8u << 20)
int qss_eval_wdot_static(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T, double *wdot,
                         double *cqss_or_null, void *stream);

/* NEXT-1 in one call: the full (N+1) x (N+1) Jacobian of Eq. 7 (L185) and both right-hand sides: the outputs of qss_eval_jac (jac,
 * wdot) AND of qss_eval_energy (tdot, erow) for the same cells; all four are required.  Two launches on `stream` (the Jacobian
 * kernel, then the energy-row kernel at 0.81 of the HBM peak).  Arguments, layout and workspace as qss_eval_jac. */
int qss_eval_jac_full(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac, double *wdot,
                      double *tdot, double *erow, void *workspace, size_t workspace_bytes, void *stream);

/* NEXT-3: sparsity (Table 4: fraction of non-zero entries of the AJ; the chain term of Eq. 9 roughly doubles it).
 * qss_mech_jac_pattern: host only, no device: pattern[i*(N+1) + k] = 1 when entry (row i, column k; k = N: T) of the Jacobian of
 * `mode` (qss_jac_mode) can be non-zero for some state, else 0 -- those entries are exactly 0.0 in the output of qss_eval_jac /
 * qss_eval_jac_approx for every state.  The description is validated as in qss_mech_create.
 * qss_jac_pack: packed[e*ld + c] = jac[idx[e]*ld + c] for e < nnz: the rows idx[e] (= i*(N+1) + k of the wanted entries; DEVICE array)
 * of the dense SoA Jacobian gathered into nnz consecutive rows, the layout a batched sparse solver takes with the pattern as its
 * index arrays.  DEVICE pointers, 16-byte aligned, ld even; one kernel on `stream`. */
int qss_mech_jac_pattern(const qss_mech_desc_t *desc, int mode, uint8_t *pattern);
int qss_jac_pack(const qss_mech_t *mech, int64_t ncells, int64_t ld, int32_t nnz, const int32_t *idx, const double *jac,
                 double *packed, void *stream);

/* NEXT-2, output layout for external batched solvers (the Jacobian goes to a batched dense direct solver, which
 * wants one contiguous matrix per cell).  qss_jac_to_aos: out[c][i][j] = J_c[i][j] for the cells c < ncells, rows i < N from `jac`
 * (layout of qss_eval_jac), and, when erow != NULL, row N from `erow` (layout of qss_eval_energy): rows = N or N + 1, cols = N + 1;
 * row-major out[(c*rows + i)*cols + j], or column-major (LAPACK) out[(c*cols + j)*rows + i] when col_major != 0.  `out`: DEVICE,
 * ncells*rows*cols doubles, 8-byte aligned, written completely for c < ncells; must not overlap the inputs.  Pure data movement
 * (bit-exact), one kernel on `stream`, no workspace.  Errors: QSS_E_INVALID (NULL pointer, ncells < 0, ld < ncells). */
int qss_jac_to_aos(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *jac, const double *erow_or_null, int col_major,
                   double *out, void *stream);

/* NEXT-3: the paper's own treatment of the temperature column (d wdot / dT "via finite difference by computing the
 * species' production rate twice at different temperatures"; L234: central differences, perturbation 1e-4; reading G22).
 * Same outputs as qss_eval_jac, except that column N of jac is
 *     (wdot(C, T+) - wdot(C, T-)) / (T+ - T-),     dT = 1e-4 T,  T+ = T + dT,  T- = T - dT   (every operation rounded on its own)
 * instead of the analytic derivative (which this library computes by default, reading G6).  Four launches of the library's kernels
 * (Jacobian, two wdot evaluations, two element-wise kernels) on `stream`.  workspace: qss_jac_fdt_workspace_bytes(mech, ld) bytes of
 * device memory, 256-byte aligned; ld even.  A comparison mode: slower and less accurate than the analytic column. */
size_t qss_jac_fdt_workspace_bytes(const qss_mech_t *mech, int64_t ld);
int qss_eval_jac_fdt(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac,
                     double *wdot_or_null, void *workspace, size_t workspace_bytes, void *stream);

/* NEXT-4 (first half): 0-D constant-volume integrator, the paper's validation workload (the
 * interval "divided into substeps over which the chemical state is advanced ... to mimic timestepping in a fluid simulation";
 * L183-188: implicit scheme, Newton method with the chemical Jacobian).  The paper integrates with CVODE (variable order, variable
 * step), which it does not specify; reading G21: `nsub` backward-Euler substeps of size dt[c] PER CELL, each solved by
 * `newton_iters` full Newton iterations with the exact (N+1) x (N+1) Jacobian re-evaluated in every iteration:
 *     phi = (C, T), f = (wdot, Tdot);  F(phi_m) = phi_m - phi^n - h f(phi_m);  (I - h J(phi_m)) delta = -F(phi_m);
 *     phi_{m+1} = phi_m + delta, C := max(C, 0)
 * No step-size control and no convergence test: the launch sequence is fixed (2 kernels per Newton iteration: the Jacobian kernel,
 * then ONE kernel that forms the energy row and the right-hand side in shared memory, solves and updates (C, T) in place -- neither
 * the energy row nor the right-hand side reaches HBM; without run-time compilation of that kernel the five calls qss_eval_jac,
 * qss_eval_energy, residual, qss_newton_solve, update; 2 copies per substep), nothing synchronises, and the call can be captured
 * in a CUDA graph after one warm-up call (run-time compilation).  C [N*ld] and T [ld] are updated IN PLACE (DEVICE
 * pointers, 16-byte aligned, ld even); dt [ncells]; `workspace`: qss_bdf1_workspace_bytes(mech, ld) bytes of device memory, 256-byte
 * aligned (holds the Jacobian: 8 N (N+1) ld bytes).  N + 1 <= 40 (limit of qss_newton_solve). */
size_t qss_bdf1_workspace_bytes(const qss_mech_t *mech, int64_t ld);
int qss_bdf1_advance(const qss_mech_t *mech, int64_t ncells, int64_t ld, double *C, double *T, const double *dt, int nsub,
                     int newton_iters, void *workspace, size_t workspace_bytes, void *stream);

/* NEXT-4, adaptive form with ignition time (the integrator "employs its own variable size time-stepping strategy";
 * L126: ignition delay = "the earliest time after which the initial temperature increased by at least 400K"; reading G23).
 * `n_attempts` attempts per cell, each one backward-Euler step of size h = min(dt[c], t_end - t[c]) (0 once t_end is reached: the
 * identity) solved by `newton_iters` full Newton iterations as in qss_bdf1_advance; with delta the LAST Newton update the attempt is
 * ACCEPTED when  max( max_i |delta_i| / (atol_C + rtol |C_i|), |delta_T| / (atol_T + rtol |T|) ) <= 1  and the new state is finite with
 * T > 0:  t[c] += h, dt[c] *= 1.5, and t_ign[c] = t[c] if it is still NaN and T - T0[c] >= dT_ign;  else REJECTED: (C, T) of the start
 * of the attempt are restored and dt[c] *= 0.25.  C, T, dt, t, t_ign are DEVICE arrays updated in place (t_ign, T0 may be NULL; fill
 * t_ign with NaN before the first call); the launch sequence is fixed (2 kernels per Newton iteration, 2 copies per attempt), nothing
 * synchronises.  Workspace as qss_bdf1_advance; ld even; N + 1 <= 40.  Needs run-time compilation (QSS_E_CUDA without NVRTC). */
int qss_ignition_advance(const qss_mech_t *mech, int64_t ncells, int64_t ld, double *C, double *T, double *dt, double *t, double t_end,
                         double *t_ign_or_null, const double *T0_or_null, double dT_ign, int n_attempts, int newton_iters, double rtol,
                         double atol_C, double atol_T, void *workspace, size_t workspace_bytes, void *stream);

/* Host-buffer convenience used for end-to-end timing: copies C and T to the device (in `dev_scratch`, which
 * must hold qss_host_scratch_bytes() bytes), evaluates, copies the Jacobian (and wdot if not NULL) back to
 * the HOST buffers, and synchronises `stream`.  Host buffers should be pinned for full copy bandwidth.  Large batches are
 * pipelined in chunks of cells: kernels run on `stream`, the copies back run on a stream owned by the handle (created by
 * qss_mech_create, released by qss_mech_destroy), so this call is not capturable in a CUDA graph; concurrent calls on one
 * handle are serialised by a mutex of the handle.  On an error both streams are synchronised before the call returns. */
size_t qss_host_scratch_bytes(const qss_mech_t *mech, int64_t ncells, int64_t ld);
int qss_eval_jac_host(const qss_mech_t *mech, int64_t ncells, int64_t ld, const double *C_host,
                      const double *T_host, double *jac_host, double *wdot_host_or_null,
                      void *dev_scratch, size_t dev_scratch_bytes, void *stream);

/* fp64 FMA-pipe micro-benchmark used as the roofline denominator: launches
 * `blocks` x 256 threads each running `iters` rounds of 8 independent dependent-chain DFMAs.
 * Returns the number of DFMA lane-operations issued in *n_fma (time it with CUDA events on `stream`). */
int qss_bench_dfma(int blocks, int iters, double *sink_dev, double *n_fma, void *stream);

const char *qss_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
