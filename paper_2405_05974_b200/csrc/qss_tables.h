// Internal: device-table layout shared by the host mechanism compiler (qss_compile.cpp) and the kernels
// (qss_kernels.cu).  Not part of the public ABI (include/qss.h).
//
// A compiled mechanism is two flat blobs on the device -- `I` (int32) and `D` (double) -- plus this struct
// of offsets into them, passed to the kernels by value.  All lists are CSR: ptr arrays have n+1 entries.
//
// Index conventions: species s < N transported, s >= N QSS (q = s - N).  Direction d = 2*j + dir,
// dir 0 = forward (reactants = the reaction's reactant side), dir 1 = reverse (reactants = product side).
#ifndef QSS_TABLES_H
#define QSS_TABLES_H
#include "qss_stdint.h"

#define QSS_TH_STRIDE 24   // doubles per species in the thermo table
#define QSS_RD_STRIDE 12   // doubles per reaction in the rate table
#define QSS_RI_STRIDE 8    // ints per reaction
#define QSS_GI_STRIDE 8    // ints per QSS group

struct QssTab {
    const int32_t *I;
    const double *D;
    int32_t N, Nq, M, nsp;
    int32_t n_tb;            // reactions of type 1 or 2
    int32_t n_groups, n_levels, max_group;
    // ---- double blob offsets
    int32_t d_thermo;        // [nsp][QSS_TH_STRIDE]: Tmid, then per range {h: a1,a2/2,a3/3,a4/4,a5/5,a6 ; s: a2,a3/2,a4/3,a5/4,a7}
    int32_t d_rate;          // [M][QSS_RD_STRIDE]: lnA, beta, Ea/R, lnA0, beta0, E0/R, alpha, 1/T3, 1/T1, T2, dnu
    int32_t d_effm1;         // eff CSR values (alpha - 1), by reaction
    int32_t d_effc;          // eff CSR values (alpha - 1), by column (species)
    // ---- int blob offsets
    int32_t i_reac;          // [M][QSS_RI_STRIDE]: type, dir_mask, tb index (-1), qss reactant fwd (-1), qss reactant rev (-1), order slot
    int32_t i_side_ptr;      // [2M+1] CSR over directions: reactant list of direction d
    int32_t i_side_sp, i_side_nu;
    int32_t i_net_ptr;       // [M+1] CSR: net stoichiometry (all species with nu_net != 0)
    int32_t i_net_sp, i_net_nu;
    int32_t i_eff_ptr;       // [M+1] CSR third-body efficiencies by reaction
    int32_t i_eff_sp;
    int32_t i_rorder;        // [M] reaction processing order (expensive types first)
    // closure
    int32_t i_group;         // [n_groups][QSS_GI_STRIDE]: size, member offset, storage offset, level, xp_begin, xp_end
    int32_t i_gmember;       // [Nq] local QSS indices, group by group in solve order
    int32_t i_level_ptr;     // [n_levels+1] groups of each level (groups are sorted by level)
    int32_t n_centry;        // closure gather entries (P, leak, p0 slots that receive at least one kappa)
    int32_t i_ce_ptr;        // [n_centry+1]
    int32_t i_ce_dst;        // [n_centry] destination offset in the per-cell closure storage
    int32_t i_ce_dir;        // direction ids
    int32_t n_xp;            // cross-group couplings P[m][n], n in an earlier group
    int32_t i_xp_ptr;        // [n_xp+1] gather lists
    int32_t i_xp_dir;
    int32_t i_xp_m, i_xp_n;  // [n_xp] m: position of the target inside its group, n: source local QSS index
    int32_t cl_size;         // per-cell closure storage, doubles
    // species incidence
    int32_t i_sp_ptr;        // [nsp+1] CSR: reactions with nu_net(s) != 0
    int32_t i_sp_reac, i_sp_nu;
    // W_y
    int32_t n_wy;            // non-zero entries of W_y
    int32_t i_wy_ptr;        // [n_wy+1] gather lists: (direction, coefficient)
    int32_t i_wy_dir, i_wy_coef;
    int32_t i_wyrow_ptr;     // [N+1] CSR rows: (q, entry)
    int32_t i_wyrow_q, i_wyrow_e;
    // Jacobian columns
    int32_t i_col_ptr;       // [N+1] CSR: incidences (direction, position of the variable in that direction's reactant list)
    int32_t i_col_dir, i_col_pos;
    int32_t i_effc_ptr;      // [N+1] CSR: third-body reactions in which species k has a non-unity efficiency
    int32_t i_effc_reac;
    // ---- per-cell workspace offsets (units of doubles per cell; the slab holds 32 cells per item)
    int32_t w_G, w_H, w_K, w_KAP, w_DF, w_DC, w_DLM, w_MM, w_CL, w_XP, w_Y, w_Q, w_QT, w_QM, w_ET, w_TV, w_WY, w_COL;
    int32_t ws_wdot, ws_jac_base;   // doubles per cell without the per-warp column buffers (w_COL starts at ws_jac_base)
};

#endif
