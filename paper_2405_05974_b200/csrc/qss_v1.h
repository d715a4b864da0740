// Internal: launch descriptor of kernel variant 1 ("slab-smem"), shared by the host mechanism compiler
// (qss_compile.cpp) and the kernel (qss_kernel_v1.cu).  Not part of the public ABI.
//
// Variant 1 processes a slab of 32 consecutive cells per thread block, lane = cell (so every table read is
// warp-uniform and every per-cell array access is a conflict-free 256-byte row), one block per SM.  The hot
// per-cell state lives in shared memory, one Jacobian column at a time lives in REGISTERS (scatter through a
// uniform indexed branch), the interpreter tables live in the kernel-parameter constant bank (`h`), and only
// the write-once / read-once per-direction arrays (k_d, kappa_d, dlnk/dT) go to an L2-resident scratch slab.
// DESIGN.md "Kernels" gives the layout and the reasons.
#ifndef QSS_V1_H
#define QSS_V1_H
#include <stdint.h>

#define QSS_V1_HMAX 7600        // 32-bit words of hot tables carried in the kernel parameters (<= 32 KB total)
#define QSS_V1_NT 36            // max transported species (register column rows)
#define QSS_V1_NQ 20            // max QSS species
#define QSS_V1_RREC 8           // int32 words per reaction record

struct QssV1 {
    // ---- filled at launch
    const double *C, *T;
    double *wdot, *cqss, *jac, *scratch;
    int64_t ncells, ld, scratch_stride;          // scratch_stride: doubles per block
    // ---- global tables (the QssTab blobs)
    const int32_t *gI;
    const double *gD;
    int32_t d_thermo, d_rate, d_effm1, i_eff_ptr, i_eff_sp, i_rrec;
    // ---- sizes
    int32_t N, Nq, M, nsp, n_tb, nw, n_groups, n_levels, n_centry, n_xp, n_wy;
    // ---- shared-memory rows (one row = 32 doubles, lane = cell)
    int32_t s_V;        // [N+1+Nq]  C_0..C_{N-1}, 1.0, y_0..y_{Nq-1}
    int32_t s_CT;       // [1]       sum_k C_k
    int32_t s_CL;       // [cl_size] closure storage: per group P[g*g], leak[g], p0[g], 1/D[g]
    int32_t s_XP;       // [n_xp]    cross-group couplings
    int32_t s_TV;       // [nsp]     third-body vector  sum_j nu_sj dQ_j/dM
    int32_t s_QM;       // [n_tb]    d ln k / dM, then dQ/dM
    int32_t s_WY;       // [n_wy]    W_y entries, row-major            } region R, time-shared with
    int32_t s_YC;       // [nw*Nq]   per-warp dy/dx_k column           }   s_G, s_H (thermo, rate phases)
    int32_t s_G, s_H;   // [nsp+1]   g/RT, h/RT (+ a zero row)          }   s_Q, s_QT (net rates phase)
    int32_t s_Q, s_QT;  // [M]       Q_j, dQ_j/dT at fixed y, M; s_QT < 0: kept in the scratch DC rows
    int32_t smem_rows;
    // ---- scratch rows
    int32_t g_K, g_KAP; // [2M]      k_d, kappa_d
    int32_t g_DF, g_DC; // [M]       dlnk/dT, dlnKc/dT
    int32_t g_ET;       // [nsp]     T-column vector sum_j nu_sj dQ_j/dT
    int32_t scratch_rows;
    // ---- hot tables (offsets into h)
    int32_t h_ce_ptr, h_ce_dst, h_ce_dir;            // closure gather
    int32_t h_xp_ptr, h_xp_dir, h_xp_m, h_xp_n;      // cross-group gather
    int32_t h_group, h_gmember, h_level_ptr;         // group records (8 words), members, levels
    int32_t h_q;                                     // [M] qf | qb<<8 | (tb+1)<<16  (V rows of the QSS reactants)
    int32_t h_ssw_ptr, h_ssw;                        // species assigned to each warp (balanced)
    int32_t h_ss_ptr, h_ss;                          // species incidence: j | nucode<<12 | (tb+1)<<16
    int32_t h_wya_ptr, h_wya;                        // W_y assembly: dir | nucode<<12
    int32_t h_cw_ptr, h_cw;                          // Jacobian columns assigned to each warp (balanced)
    int32_t h_col_ptr, h_inc;                        // column incidences: d | o1<<12 | o2<<20
    int32_t h_net_ptr, h_net;                        // net stoichiometry by reaction: slot | nucode<<8
    int32_t h_effc_ptr, h_effc, h_effc_val;          // (alpha-1) corrections by column: j | tb<<12 ; double values
    int32_t h_wyrow_ptr, h_wyq;                      // W_y rows: QSS index of each entry
    int32_t h_nulut;                                 // 16 doubles: nucode -> nu (nucode = nu + 8)
    int32_t h_used;
    int32_t h[QSS_V1_HMAX];
};

#endif
