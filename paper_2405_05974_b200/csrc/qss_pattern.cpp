// NEXT-3: structural sparsity pattern of the N x (N+1) Jacobian block (Table 4: "fraction of
// non-zero entries in the first N rows and N columns of the AJ"; the chain term of Eq. 9 "increases the number of non-zero entries by
// a factor of about 2").  Host only, from the mechanism description: entry (i, k) can be non-zero when
//   W_x:   an enabled direction d of a reaction with nu_i != 0 depends on x_k directly: k is a transported reactant molecule of d,
//          or the reaction has a third body / fall-off factor (M = sum alpha_k C_k, alpha_k != 0), or k = T;
//   chain: (exact mode only) d has a QSS reactant q and y_q depends on x_k: x_k enters a direction of the balance of a QSS species
//          that can reach q in the coupling digraph (its own group and every group upstream of it).
// Modes as in qss_jac_mode: constant-QSS drops the chain part, zero-QSS also every direction with a QSS reactant.
#include <cstdint>
#include <vector>

#include "../../include/qss.h"

int qss_pattern_build(const qss_mech_desc_t *d, int mode, uint8_t *pat /* [N * (N+1)] row-major */) {
    const int N = d->n_nqss, Nq = d->n_qss, M = d->n_reac, NC = N + 1;
    std::vector<uint8_t> out((size_t)N * NC, 0);
    // variables a direction depends on directly (bit vector over N + 1), per direction 2 j + dir
    std::vector<std::vector<uint8_t>> dep(2 * M, std::vector<uint8_t>(NC, 0));
    std::vector<int> qreact(2 * M, -1);                                // the QSS reactant of the direction (at most one: validated)
    std::vector<std::vector<int>> qprod(2 * M);                        // QSS species the direction produces
    std::vector<uint8_t> on(2 * M, 0);
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
        const int dd = 2 * j + dir;
        on[dd] = (d->dir_mask[j] >> dir) & 1;
        if (!on[dd]) continue;
        const int32_t *rp = dir == 0 ? d->reac_ptr : d->prod_ptr, *rs = dir == 0 ? d->reac_sp : d->prod_sp;
        const int32_t *pp = dir == 0 ? d->prod_ptr : d->reac_ptr, *ps = dir == 0 ? d->prod_sp : d->reac_sp;
        for (int t = rp[j]; t < rp[j + 1]; ++t) { if (rs[t] < N) dep[dd][rs[t]] = 1; else qreact[dd] = rs[t] - N; }
        for (int t = pp[j]; t < pp[j + 1]; ++t) if (ps[t] >= N) qprod[dd].push_back(ps[t] - N);
        dep[dd][N] = 1;                                                // every rate constant depends on T
        if (d->type[j] != 0) {
            std::vector<double> alpha(N, 1.0);
            for (int t = d->eff_ptr[j]; t < d->eff_ptr[j + 1]; ++t) if (d->eff_sp[t] < N) alpha[d->eff_sp[t]] = d->eff_val[t];
            for (int k = 0; k < N; ++k) if (alpha[k] != 0.0) dep[dd][k] = 1;
        }
    }
    // net stoichiometry per reaction over the transported species
    std::vector<std::vector<int>> rows(M);
    for (int j = 0; j < M; ++j) {
        std::vector<int> nu(N, 0);
        for (int t = d->reac_ptr[j]; t < d->reac_ptr[j + 1]; ++t) if (d->reac_sp[t] < N) nu[d->reac_sp[t]] -= d->reac_nu[t];
        for (int t = d->prod_ptr[j]; t < d->prod_ptr[j + 1]; ++t) if (d->prod_sp[t] < N) nu[d->prod_sp[t]] += d->prod_nu[t];
        for (int i = 0; i < N; ++i) if (nu[i]) rows[j].push_back(i);
    }
    // y_q depends on: the direct dependencies of every direction in the balance of q (producing or consuming q), and -- through
    // P[m][n] != 0 (a direction consuming n produces m) -- on everything the species that reach q depend on (transitive closure)
    std::vector<std::vector<uint8_t>> ydep(Nq, std::vector<uint8_t>(NC, 0));
    std::vector<std::vector<uint8_t>> reach(Nq, std::vector<uint8_t>(Nq, 0));      // reach[m][n]: y_n enters the equation of y_m
    for (int dd = 0; dd < 2 * M; ++dd) if (on[dd]) {
        if (qreact[dd] >= 0) for (int k = 0; k < NC; ++k) ydep[qreact[dd]][k] |= dep[dd][k];
        for (int m : qprod[dd]) {
            for (int k = 0; k < NC; ++k) ydep[m][k] |= dep[dd][k];
            if (qreact[dd] >= 0) reach[m][qreact[dd]] = 1;
        }
    }
    for (int q = 0; q < Nq; ++q) reach[q][q] = 1;
    for (int v = 0; v < Nq; ++v) for (int a = 0; a < Nq; ++a) if (reach[a][v]) for (int b = 0; b < Nq; ++b) if (reach[v][b]) reach[a][b] = 1;      // Warshall
    std::vector<std::vector<uint8_t>> yfull(Nq, std::vector<uint8_t>(NC, 0));
    for (int m = 0; m < Nq; ++m) for (int n2 = 0; n2 < Nq; ++n2) if (reach[m][n2]) for (int k = 0; k < NC; ++k) yfull[m][k] |= ydep[n2][k];
    for (int dd = 0; dd < 2 * M; ++dd) if (on[dd]) {
        const int j = dd >> 1;
        if (mode == QSS_JAC_ZERO_QSS && qreact[dd] >= 0) continue;
        for (int i : rows[j]) {
            for (int k = 0; k < NC; ++k) if (dep[dd][k]) out[(size_t)i * NC + k] = 1;
            if (mode == QSS_JAC_EXACT && qreact[dd] >= 0)
                for (int k = 0; k < NC; ++k) if (yfull[qreact[dd]][k]) out[(size_t)i * NC + k] = 1;
        }
    }
    for (size_t x = 0; x < out.size(); ++x) pat[x] = out[x];
    return QSS_OK;
}
