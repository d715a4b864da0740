// Internal: launch descriptor of kernel variant 1 ("slab-smem"), shared by the host mechanism compiler
// (qss_compile.cpp) and the kernel (qss_kernel_v1.cu).  Not part of the public ABI.
//
// Variant 1 processes a slab of 32 consecutive cells per thread block, lane = cell (so every table read is
// warp-uniform and every per-cell array access is a conflict-free 256-byte row), one block of QSS_V1_NW warps per
// SM.  The hot per-cell state lives in shared memory; the Jacobian is swept in rounds of QSS_V1_NW columns: each
// warp builds one column of [W_x; G_x] in its shared-memory column buffer and solves for dy/dx_k in place,
// then the warps switch to rows and add W_y * dy/dx for the whole round from a register tile.  The interpreter
// tables live in the kernel-parameter constant bank (`h`); the write-once / read-few per-direction arrays go to an
// L2-resident scratch slab.  DESIGN.md "Kernels" gives the layout and the reasons.
#ifndef QSS_V1_H
#define QSS_V1_H
#include "qss_stdint.h"

#define QSS_V1_HMAX 8000        // 32-bit words of hot tables carried in the kernel parameters (<= 32 KB total)
#define QSS_V1_NW 12            // warps per block = Jacobian columns per round
#define QSS_V1_RREC 8           // int32 words per reaction record

struct QssV1 {
    // ---- filled at launch
    const double *C, *T;
    double *wdot, *cqss, *jac, *scratch;
    int64_t ncells, ld, scratch_stride;          // scratch_stride: doubles per block
    long long *timing;                           // NULL, or 16 counters for the phase timing (QSS_TIMING=1, debugging aid)
    // ---- global tables (the QssTab blobs)
    const int32_t *gI;
    const double *gD;
    int32_t d_thermo, d_rate_r, d_effm1, i_eff_ptr, i_eff_sp, i_rrec;   // d_rate_r: rate records in processing order
    int32_t d_effv;                                  // (alpha - 1) values of the column streams
    int32_t i_wya_ptr, n_tab_words;                  // W_y assembly lists: [n_wy + 1] pointers, then byte offset of kappa_d | sign bit
    // ---- sizes
    int32_t N, Nq, M, nsp, n_tb, nw, n_groups, n_levels, n_centry, n_xp, n_wy, n_rounds, n_sp_ops;
    // ---- shared-memory rows (one row = 32 doubles = 256 bytes, lane = cell)
    int32_t s_V;        // [N+1+Nq]  C_0..C_{N-1}, 1.0, y_0..y_{Nq-1}      (must start at row 0)
    int32_t s_CT;       // [1]       sum_k C_k
    int32_t s_CL;       // [cl_size] closure storage: per group P[g*g], leak[g], p0[g], 1/D[g]
    int32_t s_XP;       // [n_xp]    cross-group couplings
    int32_t s_TV;       // [nsp]     third-body vector  sum_j nu_sj dQ_j/dM
    int32_t s_Z0;       // [1]       zeros (padding of the fixed-format solve operations)
    int32_t s_YC;       // [Nq*nw]   dy/dx of the round's columns, row q*nw + w   } region R, time-shared with
    int32_t s_WX;       // [N*nw]    W_x of the round's columns, row i*nw + w     }   s_G, s_H (thermo, rate phases)
    int32_t s_KAP;      // [2M]      kappa_d; then in place Q_j (row 2j), dQ_j/dT (row 2j+1) }   (phases P2-P6)
    int32_t s_G, s_H;   // [nsp+1]   g/RT, h/RT (+ a zero row), after s_KAP                  }   (phases P1-P2)
    int32_t s_TAB;      // staged once per block (n_tab_words int32): the W_y assembly lists, then the closure gather lists
    int32_t t_q;                                     //   offset of [M] qf | qb<<8 | (tb+1)<<16 (V rows of the QSS reactants) in it
    int32_t t_ce_ptr, t_ce_dst, t_ce_dir;            //   offsets of the closure gather pointers / destinations / kappa rows in it
    int32_t smem_rows;
    // ---- scratch rows
    int32_t g_K;        // [2M]      k_d
    int32_t g_DF, g_DC; // [M]       dlnk/dT, dlnKc/dT
    int32_t g_ET;       // [nsp]     T-column vector sum_j nu_sj dQ_j/dT
    int32_t g_QM;       // [n_tb]    d ln k / dM, then dQ/dM
    int32_t g_WY;       // [n_wy]    W_y entries, row-major
    int32_t scratch_rows;
    // ---- hot tables (offsets into h)
    int32_t h_xp_ptr, h_xp_dir, h_xp_m, h_xp_n;      // cross-group gather
    int32_t h_group, h_gmember, h_level_ptr;         // group records (8 words), members, levels
    int32_t h_ssw_ptr, h_ssw;                        // species assigned to each warp (balanced)
    int32_t h_ss_ptr, h_ss;                          // species incidence: byte offset of Q_j in s_KAP | sign bit
    int32_t h_st_ptr, h_st;                          // third-body incidence: index of dQ_j/dM | sign bit
    int32_t h_eff_val, h_eff_off;                    // third-body (alpha - 1) doubles; V-row byte offsets, two 16-bit per word
    int32_t h_cw;                                    // [n_rounds*nw] Jacobian column of (round, warp), -1: none
    int32_t h_cs_ptr, h_cs;                          // column streams (see qss_compile.cpp "column stream"); h_cs is an offset into
    int32_t cs_global;                               //   h, or into the global int blob when cs_global (tables too large for h)
    int32_t h_sp;                                    // dy/dx solve program: n_sp_ops pairs of fixed-format row operations
    int32_t h_wr_ptr;                                // [N+1] W_y rows: index of the first entry of each row
    int32_t h_rw;                                    // [nw][3] Jacobian rows of each warp's pass-B tile (-1: none)
    int32_t h_tile_ptr, h_tile;                      // per warp: q | row mask << 8 over the union of the rows' W_y columns
    int32_t h_used;
    alignas(8) int32_t h[QSS_V1_HMAX];
};

#endif
