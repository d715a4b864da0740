// Internal: launch descriptor of kernel variant 3 (qss_kernel_v3.cu), shared by the host (qss_gen3.cpp, qss_api.cu,
// qss_jit.cpp) and the kernel source, which exists only as a run-time compiled (NVRTC) program: every size, row and offset
// of the mechanism is a compile-time constant of the generated header `qss_gen3.h`.  Not part of the public ABI.
#ifndef QSS_V3_H
#define QSS_V3_H
#include "qss_stdint.h"

// doubles / ints per rate-task slot in the parameter blobs (slot = 32 * group + lane: one reaction; layout [param][slot])
#define QSS3_NDP 91
#define QSS3_NIP 14
#define QSS3_MAX_EFF 8           // non-unity third-body efficiencies per reaction held in registers
#define QSS3_MAX_CORR 8          // distinct NASA-7 breakpoints Tmid among the species of one reaction

// double parameters
#define QSS3_D_LNA 0             // ln A, beta, Ea/R (high-pressure limit for fall-off reactions)
#define QSS3_D_BETA 1
#define QSS3_D_EAR 2
#define QSS3_D_TMID 3            // smallest NASA-7 range breakpoint Tmid among the species of the reaction
#define QSS3_D_ELO 4             // [7] coefficients of -ln Kc below it: e0 + e1 lnT + T(e2 + T(e3 + T(e4 + T e5))) + e6/T
#define QSS3_D_EHI 11            // [7] the same at and above the LARGEST Tmid of the reaction's species
#define QSS3_D_LNA0 18           // low-pressure limit ln A0, beta0, E0/R
#define QSS3_D_BETA0 19
#define QSS3_D_E0R 20
#define QSS3_D_ALPHA 21          // Troe alpha, 1/T***, 1/T*, T**
#define QSS3_D_I3 22
#define QSS3_D_I1 23
#define QSS3_D_T2S 24
#define QSS3_D_EFFV 25           // [8] alpha_k - 1
#define QSS3_D_TMAX 33           // largest Tmid among the species of the reaction (= QSS3_D_TMID when they share one)
#define QSS3_D_CORR 34           // [8 + 7 x 7] reactions whose species have different Tmid: up to 6 breakpoints strictly between TMID and TMAX
                                 // (ascending, rows 0..5), then one coefficient set of -ln Kc per interval between consecutive breakpoints
                                 // (set i at rows 8 + 7 i .. 8 + 7 i + 6, i = number of inner breakpoints <= T)
// int parameters
#define QSS3_I_FLAGS 0           // mask (bits 0-1) | type << 2 | valid << 4 | n_eff << 8
#define QSS3_I_KAP 1             // byte offset of the k_f / kappa_f / Q_j row (the reverse row follows G_M rows later)
#define QSS3_I_TB 2              // index among the third-body / fall-off reactions, -1: none
#define QSS3_I_QF 3              // byte offset of the V row of the QSS reactant of the forward direction (none: the 1.0 row)
#define QSS3_I_QB 4
#define QSS3_I_EFFS 5            // [8] byte offsets of the V rows of the species with non-unity efficiency
#define QSS3_I_NCORR 13          // inner breakpoints in QSS3_D_CORR

struct QssV3 {
    const double *C, *T;
    double *wdot, *cqss, *jac, *scratch;
    int64_t ncells, ld, scratch_stride;          // scratch_stride: doubles per block
    const double *dP;                            // [QSS3_NDP][n_slot]
    const int32_t *iP;                           // [QSS3_NIP][n_slot]
    long long *timing;                           // NULL, or 16 phase counters (images built with -DQSS3_TIMING=1 only)
    int32_t mode;                                // 0 exact Jacobian; 1 constant-QSS AJ (no chain term); 2 zero-QSS AJ (also C_QSS := 0)
};

#endif
