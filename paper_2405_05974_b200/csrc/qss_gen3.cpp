// Kernel variant 3: host side.  Emits, for ONE mechanism, the header `qss_gen3.h` that specialises qss_kernel_v3.cu
// (compiled at qss_mech_create with NVRTC) and the parameter blobs of its reaction-per-lane phases.
//
// Mapping: one persistent block of 12 warps per SM works on a slab of 32 cells whose per-cell
// state lives in shared memory as rows of 33 doubles (row pitch 264 bytes), so that BOTH access directions are free of
// bank conflicts: "lane = cell" (a warp reads one row) and "lane = item" (the lanes of a warp read the same cell of 32
// consecutive rows).
//   - rate constants (Eq. 2): lane = REACTION.  The reaction's parameters (Arrhenius, the NASA-7 sums of ln Kc
//     folded into seven coefficients per temperature range, fall-off, efficiencies) are per-lane registers, loaded once per
//     task; the lane loops over cells and writes k_f, k_b into 32 consecutive rows.  No table decoding, no thermo phase.
//   - direction coefficients kappa_d = k_d prod C (Eq. 6): lane = cell, a compact table loop; k_d leaves for the
//     scratch slab on the way (coalesced rows: a lane = reaction store to a [row][cell] array would touch 32 lines).
//   - net rates Q_j and dQ_j/dT after the closure: lane = reaction again.
//   - closure gather, closure solve, species sums, Jacobian columns: lane = cell, straight-line code generated here
//     (as in variant 2), the column of [W_x; G_x] in registers.
#include "qss_compile.h"
#include "qss_ctx.h"
#include "qss_devtools.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <limits>
#include <stdexcept>

namespace qssc {

namespace {

struct Gen {
    std::string s;
    void operator()(const char *f, ...) {
        char b[512];
        va_list ap;
        va_start(ap, f);
        const int n = std::vsnprintf(b, sizeof b, f, ap);
        va_end(ap);
        if (n < 0 || n >= (int)sizeof b) throw std::runtime_error("qss_gen3: generated line exceeds the line buffer");
        s += b;
    }
};

// longest-processing-time assignment of items (cost) to `nbin` bins; returns the bin of each item
std::vector<int> lpt(const std::vector<double> &cost, int nbin, std::vector<double> *load_out = nullptr) {
    std::vector<int> idx(cost.size()), bin(cost.size(), 0);
    for (size_t i = 0; i < idx.size(); ++i) idx[i] = (int)i;
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    std::vector<double> load(nbin, 0.0);
    for (int i : idx) { const int b = (int)(std::min_element(load.begin(), load.end()) - load.begin()); bin[i] = b; load[b] += cost[i]; }
    if (load_out) *load_out = load;
    return bin;
}

}  // namespace

bool build_v3(const V1Ctx &c, QssCompiled &out, std::string &why) {
    const int N = c.N, Nq = c.Nq, M = c.M, nsp = c.nsp, ntb = c.n_tb;
    const std::vector<Reaction> &R = *c.R;
    const qss_mech_desc_t *d = c.desc;
    QssV3Host &v = out.v3;
    v = QssV3Host();
    int NW = 12;                        // warps per block in every phase but the column sweep
    if (const char *e = qss_devenv("QSS3_NW")) NW = std::atoi(e);
    // registers per thread: at launch (all phases but the sweep), of the idle warps and of the column warps during the sweep
    const int reg_base = std::min(255, 65536 / (NW * 32)) / 8 * 8, reg_idle = 24;
    const int reg_col = NW > 12 ? reg_base + (NW - 12) * (reg_base - reg_idle) / 12 / 8 * 8 : reg_base;
    const int NWC = 12, PITCH = 264, MAXROWS = (227 * 1024) / PITCH;      // NWC: column warps (one Jacobian column in ~160 registers each)
    if (M < 1) { why = "no reactions"; return false; }
    if (nsp > 60) { why = "more than 60 species: one Jacobian column does not fit the registers of a thread"; return false; }
    for (int j = 0; j < M; ++j)
        for (int s = 0; s < 2; ++s) { int n = 0; for (const Term &x : R[j].side[s]) n += x.nu; if (n > 3) { why = "a reaction side has more than 3 molecules"; return false; } }
    // ---- shared-memory rows (pitch 264 bytes) ---------------------------------------------------------------------
    int rows = 0;
    auto take = [&](int n) { const int r = rows; rows += n; return r; };
    const int R_V = take(N + 1 + Nq), R_ONE = R_V + N, R_Y = R_V + N + 1;
    const int R_T = take(1), R_LNT = take(1), R_INVT = take(1), R_CT = take(1);
    const int R_CL = take(c.cl_size), R_XP = take((int)c.xpl->size());
    const int R_TV = take(nsp), R_DLM = take(ntb);
    // reactions that consume a QSS species: kappa_d of those directions is kept for the chain-rule product W_y dy/dx
    struct KqRec { int j, q[2], idx[2]; std::vector<std::pair<int, int>> tgt; };      // tgt: (transported species, nu_net)
    std::vector<KqRec> kq;
    std::vector<int> kq_row(2 * M, -1);
    int n_kq = 0;
    for (int j = 0; j < M; ++j) {
        KqRec r{j, {-1, -1}, {-1, -1}, {}};
        for (const Term &x : R[j].net) if (x.sp < N) r.tgt.push_back({x.sp, x.nu});
        if (r.tgt.empty()) continue;
        for (int dir = 0; dir < 2; ++dir)
            if (((R[j].mask >> dir) & 1) && R[j].q[dir] >= 0) { r.q[dir] = R[j].q[dir]; r.idx[dir] = n_kq; kq_row[2 * j + dir] = n_kq++; }
        if (r.idx[0] >= 0 || r.idx[1] >= 0) kq.push_back(r);
    }
    // kappa_d of the QSS-consuming directions comes back for the column sweep as PAIRS per lane ([pair][lane][2], 528 bytes
    // per pair, 16-byte aligned): one 16-byte read brings two of them
    const int kq_rows = n_kq + 2;
    // k_d / kappa_d / Q_j rows: forward rows, one row that stays zero, reverse rows, one zero row (row stride MS between the two
    // directions of a reaction; the zero rows pad the species-sum lists to multiples of four terms)
    const int MS = M + 1;
    const int region = std::max(2 * MS, kq_rows + N + NW);
    const int R_KAP = take(region), R_KQ = R_KAP, R_STAGE = R_KAP + kq_rows;
    const int KQ_BASE = R_KQ * PITCH + ((R_KQ * PITCH) % 16);          // byte offset of pair 0 (PITCH = 8 mod 16)
    if (rows > MAXROWS) { why = "per-cell state does not fit the shared memory of one SM"; return false; }
    std::vector<std::vector<int>> slots(2 * M);            // species of each molecule of the reactant side of direction d
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir)
        for (const Term &x : R[j].side[dir]) for (int u = 0; u < x.nu; ++u) slots[2 * j + dir].push_back(x.sp);
    // ---- rate-task groups: reactions of one type, at most 32 per group (lane = reaction) -----------------------------
    std::vector<int> order(M);
    for (int j = 0; j < M; ++j) order[j] = j;
    auto nslot = [&](int j, int s) { return (int)slots[2 * j + s].size(); };
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
        if (R[a].type != R[b].type) return R[a].type > R[b].type;
        const int sa = std::max(nslot(a, 0), nslot(a, 1)), sb = std::max(nslot(b, 0), nslot(b, 1));
        return sa > sb;
    });
    struct Group { int type, first, count; };
    std::vector<Group> groups;
    for (int t = 2; t >= 0; --t) {
        int first = 0, n = 0;
        for (int r = 0; r < M; ++r) if (R[order[r]].type == t) { if (!n) first = r; ++n; }
        if (!n) continue;
        const int ng = (n + 31) / 32;
        for (int g = 0, o = first; g < ng; ++g) { const int cnt = n / ng + (g < n % ng ? 1 : 0); groups.push_back({t, o, cnt}); o += cnt; }
    }
    // rows of the rate constants / kappa_d / Q_j: in task order, so that the 32 lanes of a task own 32 consecutive rows
    // (forward rows R_KAP + pos, reverse rows R_KAP + MS + pos); direction index e = dir * MS + pos
    std::vector<int> pos(M);
    for (int r = 0; r < M; ++r) pos[order[r]] = r;
    auto erow = [&](int dd) { return (dd & 1) * MS + pos[dd >> 1]; };           // dd = 2 j + dir
    const int n_slot = 32 * (int)groups.size();
    // ---- scratch rows (256 bytes: 32 cells, lane = cell): k_d (read by the column records), kappa_d of the QSS-consuming
    //      directions (saved while the kappa rows are reused for Q_j), the T-column vector; d ln k/dT and d ln Kc/dT are
    //      exchanged between two lane = reaction phases and therefore stored [cell][2 n_slot] (2 n_slot "rows" of 32 doubles)
    int srows = 0;
    auto stake = [&](int n) { const int r = srows; srows += n; return r; };
    const int S_K = stake(2 * MS), S_KQ = stake(n_kq), S_ET = stake(nsp), S_DT = stake(2 * n_slot);
    v.dP.assign((size_t)QSS3_NDP * n_slot, 0.0);
    v.iP.assign((size_t)QSS3_NIP * n_slot, 0);
    auto DP = [&](int p, int slot) -> double & { return v.dP[(size_t)p * n_slot + slot]; };
    auto IP = [&](int p, int slot) -> int32_t & { return v.iP[(size_t)p * n_slot + slot]; };
    auto vrow = [&](int sp) { return sp < N ? R_V + sp : R_ONE; };                 // a QSS molecule reads 1.0 (y is not known yet)
    const double RGAS = 8.31446261815324;
    const long double LNP0R = std::log((long double)101325.0 / (long double)RGAS);
    bool has_corr = false;                  // some reaction's species have different NASA-7 mid temperatures
    for (size_t g = 0; g < groups.size(); ++g) for (int l = 0; l < 32; ++l) {
        const int slot = 32 * (int)g + l;
        // a padding lane computes a harmless reaction and stores nothing
        IP(QSS3_I_KAP, slot) = R_KAP * PITCH; IP(QSS3_I_TB, slot) = -1;
        IP(QSS3_I_QF, slot) = IP(QSS3_I_QB, slot) = R_ONE * PITCH;
        for (int u = 0; u < QSS3_MAX_EFF; ++u) IP(QSS3_I_EFFS + u, slot) = R_ONE * PITCH;
        DP(QSS3_D_TMID, slot) = DP(QSS3_D_TMAX, slot) = 1000.0; DP(QSS3_D_I3, slot) = 1.0; DP(QSS3_D_I1, slot) = 1.0; DP(QSS3_D_ALPHA, slot) = 0.5;
        if (l >= groups[g].count) continue;
        const int j = order[groups[g].first + l];
        const Reaction &r = R[j];
        const double A = d->arr[3 * j];
        DP(QSS3_D_LNA, slot) = std::log(A); DP(QSS3_D_BETA, slot) = d->arr[3 * j + 1]; DP(QSS3_D_EAR, slot) = d->arr[3 * j + 2] / RGAS;
        if (r.type == 2) {
            DP(QSS3_D_LNA0, slot) = std::log(d->arr_low[3 * j]); DP(QSS3_D_BETA0, slot) = d->arr_low[3 * j + 1]; DP(QSS3_D_E0R, slot) = d->arr_low[3 * j + 2] / RGAS;
            DP(QSS3_D_ALPHA, slot) = d->troe[4 * j]; DP(QSS3_D_I3, slot) = 1.0 / d->troe[4 * j + 1]; DP(QSS3_D_I1, slot) = 1.0 / d->troe[4 * j + 2];
            DP(QSS3_D_T2S, slot) = d->troe[4 * j + 3];
        }
        // -ln Kc = sum nu g/RT - dnu ln(P0/RT) as seven coefficients per NASA-7 range (reading G4; g/RT =
        // a1 (1 - lnT) - a2 T/2 - a3 T^2/6 - a4 T^3/12 - a5 T^4/20 + a6/T - a7).  ELO holds below the smallest Tmid of the
        // reaction's species, EHI at and above the largest; between them (real thermodynamic data: every species has its own
        // Tmid) there is one more set per interval between consecutive breakpoints, fetched by the kernel when a cell needs it.
        DP(QSS3_D_TMAX, slot) = DP(QSS3_D_TMID, slot);
        if (r.mask & 2) {
            double tmin = 0.0, tmax = 0.0; bool have = false;
            for (const Term &x : r.net) {
                const double tm = d->nasa_T[3 * x.sp + 1];
                tmin = have ? std::min(tmin, tm) : tm; tmax = have ? std::max(tmax, tm) : tm; have = true;
            }
            DP(QSS3_D_TMID, slot) = have ? tmin : 1000.0;
            DP(QSS3_D_TMAX, slot) = have ? tmax : 1000.0;
            const size_t st = (size_t)n_slot;
            auto fold = [&](const long double (&As)[7], long double dnu, double *e) {
                e[0 * st] = (double)(As[0] - As[6] - dnu * LNP0R);
                e[1 * st] = (double)(-As[0] + dnu);
                e[2 * st] = (double)(-As[1] / 2.0L); e[3 * st] = (double)(-As[2] / 6.0L); e[4 * st] = (double)(-As[3] / 12.0L); e[5 * st] = (double)(-As[4] / 20.0L);
                e[6 * st] = (double)As[5];
            };
            for (int rg = 0; rg < 2; ++rg) {
                long double As[7] = {0, 0, 0, 0, 0, 0, 0};
                for (const Term &x : r.net) { const double *a = (rg == 0 ? d->nasa_lo : d->nasa_hi) + 7 * x.sp; for (int i = 0; i < 7; ++i) As[i] += (long double)x.nu * (long double)a[i]; }
                fold(As, (long double)r.dnu, &DP((rg == 0 ? QSS3_D_ELO : QSS3_D_EHI), slot));
            }
            if (have && tmin != tmax) {
                std::vector<double> bp;                       // distinct breakpoints, ascending
                for (const Term &x : r.net) bp.push_back(d->nasa_T[3 * x.sp + 1]);
                std::sort(bp.begin(), bp.end());
                bp.erase(std::unique(bp.begin(), bp.end()), bp.end());
                if (bp.size() > (size_t)QSS3_MAX_CORR) { why = "the species of a reaction have more than 8 different NASA-7 mid temperatures"; return false; }
                const int nb = (int)bp.size() - 2;            // inner breakpoints
                for (int i = 0; i < nb; ++i) DP(QSS3_D_CORR + i, slot) = bp[i + 1];
                for (int iv = 0; iv <= nb; ++iv) {            // interval [bp[iv], bp[iv + 1]): species s is in its high range iff Tmid_s <= bp[iv]
                    long double As[7] = {0, 0, 0, 0, 0, 0, 0};
                    for (const Term &x : r.net) {
                        const double *a = (d->nasa_T[3 * x.sp + 1] <= bp[iv] ? d->nasa_hi : d->nasa_lo) + 7 * x.sp;
                        for (int i = 0; i < 7; ++i) As[i] += (long double)x.nu * (long double)a[i];
                    }
                    fold(As, (long double)r.dnu, &DP(QSS3_D_CORR + 8 + 7 * iv, slot));
                }
                IP(QSS3_I_NCORR, slot) = nb;
                has_corr = true;
            }
        }
        int ne = 0;
        if (r.type >= 1) for (int k = 0; k < N; ++k) for (auto &e : (*c.effc)[k]) if (e.first == j) {
            if (ne >= QSS3_MAX_EFF) { why = "a reaction has more than 8 non-unity third-body efficiencies"; return false; }
            IP(QSS3_I_EFFS + ne, slot) = (R_V + k) * PITCH; DP(QSS3_D_EFFV + ne, slot) = e.second; ++ne;
        }
        IP(QSS3_I_FLAGS, slot) = r.mask | (r.type << 2) | (1 << 4) | (ne << 8);
        IP(QSS3_I_KAP, slot) = (R_KAP + pos[j]) * PITCH;
        IP(QSS3_I_TB, slot) = r.tb;
        IP(QSS3_I_QF, slot) = (r.q[0] >= 0 ? R_Y + r.q[0] : R_ONE) * PITCH;
        IP(QSS3_I_QB, slot) = (r.q[1] >= 0 ? R_Y + r.q[1] : R_ONE) * PITCH;
    }
    if (!has_corr) v.dP.resize((size_t)QSS3_D_TMAX * n_slot);      // (the rows behind the efficiencies are read by images with G_HAS_CORR only)
    // ---- tasks: (group, cell chunk) dealt to the warps by cost -------------------------------------------------------
    // A warp takes a CONTIGUOUS stretch of the line "group 0 cells 0..31, group 1 cells 0..31, ..." of equal cost, so that it
    // loads the parameters of at most two or three groups per slab and every group is loaded about once per block.
    struct Task { int type, slot0, c0, c1; };
    auto partition = [&](const double (&per_cell)[3], int gran, std::vector<Task> &out_tasks, std::vector<int> &ptr) {
        double total = 0.0;
        for (const Group &g : groups) total += 32.0 * per_cell[g.type];
        out_tasks.clear(); ptr.assign(NW + 1, 0);
        double acc = 0.0;
        int w = 0;
        for (size_t g = 0; g < groups.size(); ++g) {
            int c0 = 0;
            for (int cidx = 0; cidx < 32; cidx += gran) {
                acc += gran * per_cell[groups[g].type];
                const bool last_cell = cidx + gran >= 32;
                const bool cut = w + 1 < NW && acc >= total * (w + 1) / NW - 1e-9;
                if (cut || last_cell) {
                    out_tasks.push_back({groups[g].type, 32 * (int)g, c0, cidx + gran});
                    c0 = cidx + gran;
                    if (cut) ptr[++w] = (int)out_tasks.size();
                }
            }
        }
        while (w < NW) ptr[++w] = (int)out_tasks.size();
    };
    std::vector<Task> rsorted, nsorted;
    std::vector<int> rptr, nptr;
    {
        double rate_cost[3] = {130.0, 200.0, 700.0};      // per cell and group, fitted to the measured per-warp times (with the table exponential)
        const double net_cost[3] = {1.0, 1.1, 1.1};
        if (const char *e = qss_devenv("QSS3_W")) std::sscanf(e, "%lf,%lf,%lf", &rate_cost[0], &rate_cost[1], &rate_cost[2]);
        partition(rate_cost, 2, rsorted, rptr);
        partition(net_cost, 4, nsorted, nptr);
    }
    // ---- Jacobian column records ----------------------------------------------------------------------------------
    // column k of [W_x; G_x] (Eq. 9 first parenthesis): one record per (enabled direction, reactant molecule that
    // is species k): value = k_d times the OTHER molecules of the side (valid at C_k = 0, reading G12), scattered with the
    // signed net stoichiometry; one per non-unity third-body efficiency: value = dQ_j/dM (alpha_jk - 1)
    struct Rec { int src; bool from_smem; int f1, f2; double lit; std::vector<std::pair<int, int>> tgt; };    // f1, f2: V byte offsets or -1
    std::vector<std::vector<Rec>> rec(N);
    auto vrow_y = [&](int sp) { return sp < N ? R_V + sp : R_Y + (sp - N); };
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
        if (!((R[j].mask >> dir) & 1)) continue;
        const std::vector<int> &sl = slots[2 * j + dir];
        for (size_t p = 0; p < sl.size(); ++p) {
            const int k = sl[p];
            if (k >= N) continue;
            int o[2] = {-1, -1}, no = 0;
            for (size_t q = 0; q < sl.size(); ++q) if (q != p) o[no++] = vrow_y(sl[q]) * PITCH;
            Rec r{(S_K + erow(2 * j + dir)) * 256, false, o[0], o[1], 1.0, {}};
            for (const Term &x : R[j].net) r.tgt.push_back({x.sp, dir == 0 ? x.nu : -x.nu});
            if (!r.tgt.empty()) rec[k].push_back(r);
        }
    }
    for (int k = 0; k < N; ++k) for (auto &e : (*c.effc)[k]) if (R[e.first].mask) {
        Rec r{(R_DLM + R[e.first].tb) * PITCH, true, -1, -1, e.second, {}};
        for (const Term &x : R[e.first].net) r.tgt.push_back({x.sp, x.nu});
        if (!r.tgt.empty()) rec[k].push_back(r);
    }
    // ---- dy/dx solve: row operations y[a] = (y[a] + sum F y[b]) * S on the QSS rows of the column ----------------------
    struct Op { int a; std::vector<std::pair<int, int>> terms; int scale; };           // (F row, QSS index b); scale row or -1
    std::vector<std::vector<Op>> gops(c.n_groups);
    for (int g = 0; g < c.n_groups; ++g) {
        const std::vector<int> &mem = (*c.members)[g];
        const int sz = (int)mem.size(), base = R_CL + (*c.gbase)[g];
        for (int x = (*c.xp_begin)[g]; x < (*c.xp_end)[g]; ++x) gops[g].push_back({(*c.xpl)[x].first.first, {{R_XP + x, (*c.xpl)[x].first.second}}, -1});
        for (int m = sz - 2; m >= 0; --m) {
            Op o{mem[m], {}, -1};
            for (int k = m + 1; k < sz; ++k) o.terms.push_back({base + m * sz + k, mem[k]});
            gops[g].push_back(o);
        }
        for (int k = 0; k < sz; ++k) {
            Op o{mem[k], {}, base + sz * sz + 2 * sz + k};
            for (int jj = 0; jj < k; ++jj) o.terms.push_back({base + k * sz + jj, mem[jj]});
            gops[g].push_back(o);
        }
    }
    // =================================================================================================================
    Gen G;
    G("// generated by qss_gen3.cpp for one mechanism (%d + %d species, %d reactions); compiled with qss_kernel_v3.cu\n", N, Nq, M);
    G("#define G_N %d\n#define G_NQ %d\n#define G_M %d\n#define G_NSP %d\n#define G_MS %d\n#define G_NTB %d\n#define G_NW %d\n#define G_NWC %d\n#define G_REG_BASE %d\n#define G_REG_IDLE %d\n#define G_REG_COL %d\n#define G_PITCH %d\n#define G_NSLOT %d\n",
      N, Nq, M, nsp, MS, ntb, NW, NWC, reg_base, reg_idle, reg_col, PITCH, n_slot);
    G("#define R_V %d\n#define R_ONE %d\n#define R_Y %d\n#define R_T %d\n#define R_LNT %d\n#define R_INVT %d\n#define R_CT %d\n#define R_CL %d\n#define R_XP %d\n#define R_TV %d\n#define R_DLM %d\n#define R_KAP %d\n#define R_KQ %d\n#define R_STAGE %d\n",
      R_V, R_ONE, R_Y, R_T, R_LNT, R_INVT, R_CT, R_CL, R_XP, R_TV, R_DLM, R_KAP, R_KQ, R_STAGE);
    G("#define KQ_BASE %d\n", KQ_BASE);
    G("#define G_HAS_CORR %d\n", has_corr ? 1 : 0);
    G("#define S_K %d\n#define S_KQ %d\n#define S_ET %d\n#define S_DT %d\n#define G_NKQ %d\n#define G_KQ_PER_WARP %d\n#define G_SROWS %d\n", S_K, S_KQ, S_ET, S_DT, n_kq,
      std::max(1, (n_kq + NW - 1) / NW), srows);
    // ---- interpreter tables (int32 words, appended to the int parameter blob, staged in shared memory once per block)
    std::vector<int32_t> tabw;
    auto tput = [&](const char *name, const std::vector<int32_t> &a) { G("#define %s %d\n", name, (int)tabw.size()); tabw.insert(tabw.end(), a.begin(), a.end()); };
    {   // kappa pass (lane = cell): per direction e the V rows of its (up to 3) reactant molecules (a QSS molecule or an empty
        // slot reads the 1.0 row), 6 bits each, and (index + 1) << 18 of the scratch row that keeps kappa_d for the chain-rule
        // product; the two zero rows are directions without reactants
        std::vector<int32_t> w(2 * MS, R_ONE | (R_ONE << 6) | (R_ONE << 12));
        for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
            int rr[3] = {R_ONE, R_ONE, R_ONE};
            const std::vector<int> &sl = slots[2 * j + dir];
            for (size_t u = 0; u < sl.size(); ++u) rr[u] = vrow(sl[u]);
            if (rr[0] >= 64 || rr[1] >= 64 || rr[2] >= 64 || n_kq >= (1 << 13)) { why = "rows beyond the packed fields of the kappa table"; return false; }
            w[erow(2 * j + dir)] = rr[0] | (rr[1] << 6) | (rr[2] << 12) | ((kq_row[2 * j + dir] + 1) << 18);
        }
        while (w.size() % 4) w.push_back(R_ONE | (R_ONE << 6) | (R_ONE << 12));
        tput("T_KAP", w);
    }
    {
        std::vector<int32_t> a2(rptr.begin(), rptr.end()), b2, c2(nptr.begin(), nptr.end()), d2;
        for (const Task &t : rsorted) { b2.push_back(t.type); b2.push_back(t.slot0); b2.push_back(t.c0); b2.push_back(t.c1); }
        for (const Task &t : nsorted) { d2.push_back(t.slot0); d2.push_back(t.c0); d2.push_back(t.c1); d2.push_back(0); }
        tput("T_RT_PTR", a2); tput("T_RT", b2); tput("T_NT_PTR", c2); tput("T_NT", d2);
        // 2^(j/64), j = 0..63, for the table form of the exponential (qss_math.h qss_exp_tab): 64 doubles as 128 words, 8-byte aligned
        while (tabw.size() % 2) tabw.push_back(0);
        std::vector<int32_t> ex(128);
        for (int j = 0; j < 64; ++j) { const double v = (double)exp2l((long double)j / 64.0L); std::memcpy(&ex[2 * j], &v, 8); }
        tput("T_EXP", ex);
    }
    // ---- species sums: per species the added terms, then the subtracted terms, one table word (byte offset of the row) per
    //      unit of |nu| (two 16-bit row numbers per 32-bit word), each list padded to a multiple of four words with the row that stays zero; T_SS_PTR: the Q_j lists
    //      (wdot, T-column vector), T_ST_PTR: the dQ_j/dM lists (third-body vector), both index the same word array
    {
        std::vector<std::vector<int32_t>> sp(nsp), sm(nsp), tp(nsp), tm(nsp);
        for (int j = 0; j < M; ++j) if (R[j].mask) for (const Term &x : R[j].net) for (int u = 0; u < std::abs(x.nu); ++u) {
            (x.nu > 0 ? sp : sm)[x.sp].push_back(R_KAP + pos[j]);
            if (R[j].tb >= 0) (x.nu > 0 ? tp : tm)[x.sp].push_back(R_DLM + R[j].tb);
        }
        std::vector<double> cost(nsp);
        for (int s2 = 0; s2 < nsp; ++s2) cost[s2] = 16.0 + sp[s2].size() + sm[s2].size() + 0.6 * (tp[s2].size() + tm[s2].size());
        const std::vector<int> bin = lpt(cost, NW);
        std::vector<int32_t> ptr, all, tptr, wptr{0}, wall;
        auto lists = [&](std::vector<std::vector<int32_t>> &a, std::vector<std::vector<int32_t>> &b2, std::vector<int32_t> &pp) {
            pp.push_back((int32_t)all.size());
            for (int s2 = 0; s2 < nsp; ++s2) for (auto *l : {&a[s2], &b2[s2]}) {
                all.insert(all.end(), l->begin(), l->end());
                while (all.size() % 4) all.push_back(R_KAP + M);
                pp.push_back((int32_t)all.size());
            }
        };
        lists(sp, sm, ptr);
        lists(tp, tm, tptr);
        for (int u = 0; u < 8; ++u) all.push_back(R_KAP + M);      // (the software pipeline reads two steps past a list)
        // two 16-bit row numbers per word; the pointers count terms
        std::vector<int32_t> packed;
        for (size_t i = 0; i < all.size(); i += 2) packed.push_back(all[i] | (all[i + 1] << 16));
        for (int w = 0; w < NW; ++w) { for (int s2 = 0; s2 < nsp; ++s2) if (bin[s2] == w) wall.push_back(s2); wptr.push_back((int32_t)wall.size()); }
        while (tabw.size() % 2) tabw.push_back(0);
        tput("T_SS", packed); tput("T_SS_PTR", ptr); tput("T_ST_PTR", tptr); tput("T_SSW_PTR", wptr); tput("T_SSW", wall);
    }
    {
        if (rows & 1) ++rows;                                 // (the tables are read 16 bytes at a time)
        const int R_TAB = rows, tab_rows = ((int)tabw.size() * 4 + PITCH - 1) / PITCH;
        rows += tab_rows;
        if (rows > MAXROWS) { why = "per-cell state and the staged tables do not fit the shared memory of one SM"; return false; }
        G("#define R_TAB %d\n#define G_NTAB %d\n", R_TAB, (int)tabw.size());
        v.iP.insert(v.iP.end(), tabw.begin(), tabw.end());
    }
    // ---- P3: closure slots and cross-group couplings as signed sums of kappa rows ------------------------------------
    {
        struct Ent { int dst; std::vector<int> terms; };
        std::vector<Ent> ents;
        for (auto &kv : *c.ce) { Ent e{(R_CL + kv.first) * PITCH, {}}; for (int dd : kv.second) e.terms.push_back((R_KAP + erow(dd)) * PITCH); ents.push_back(e); }
        for (size_t x = 0; x < c.xpl->size(); ++x) { Ent e{(R_XP + (int)x) * PITCH, {}}; for (int dd : (*c.xpl)[x].second) e.terms.push_back((R_KAP + erow(dd)) * PITCH); ents.push_back(e); }
        std::vector<double> cost;
        for (const Ent &e : ents) cost.push_back(2.0 + e.terms.size());
        const std::vector<int> bin = lpt(cost, NW);
        G("__device__ __forceinline__ void qss_gen_gather(const int warp, const unsigned sml) {\n    switch (warp) {\n");
        for (int w = 0; w < NW; ++w) {
            G("    case %d:\n", w);
            for (size_t i = 0; i < ents.size(); ++i) if (bin[i] == w) {
                G("        sS<%d>(sml, ", ents[i].dst);
                if (ents[i].terms.empty()) G("0.0");
                for (size_t t = 0; t < ents[i].terms.size(); ++t) G("%slS<%d>(sml)", t ? " + " : "", ents[i].terms[t]);
                G(");\n");
            }
            G("        break;\n");
        }
        G("    default: break;\n    }\n}\n");
    }
    // ---- P2c and P6 as straight-line code (one part per warp): kappa_d = k_d prod C, and the species sums.  MEASURED AND NOT USED
    //      (development builds, QSS3_EXP bits 8 / 16): the table loops spend 4-6x as many instructions on the same work, but the
    //      7.6 k instructions of once-per-slab code arrive at ~4.5 bytes per clock and SM: 12.2 / 12.7 ms against 11.5 ms.
    int exp_bits = 0;
    if (const char *e = qss_devenv("QSS3_EXP")) exp_bits = std::atoi(e);
    if (exp_bits & 24) {
    {
        std::vector<std::vector<int>> fac(2 * MS);                      // V rows of the transported reactant molecules per direction row
        std::vector<int> kqe(2 * MS, -1);
        for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
            const int e = erow(2 * j + dir);
            for (int sp2 : slots[2 * j + dir]) if (vrow(sp2) != R_ONE) fac[e].push_back(vrow(sp2));
            kqe[e] = kq_row[2 * j + dir];
        }
        std::vector<double> cost(2 * MS);
        for (int e = 0; e < 2 * MS; ++e) cost[e] = 4.0 + 2.0 * fac[e].size() + (kqe[e] >= 0 ? 1.0 : 0.0);
        // contiguous ranges of rows per warp (neighbouring rows: the same shared-memory banks pattern as the table loop)
        double total = 0.0; for (double x : cost) total += x;
        G("__device__ __forceinline__ void qss_gen_kappa(const int warp, const unsigned sml, double *sc) {\n    switch (warp) {\n");
        int e = 0; double acc = 0.0;
        for (int w = 0; w < NW; ++w) {
            G("    case %d:\n", w);
            const double upto = total * (w + 1) / NW;
            while (e < 2 * MS && (acc + 0.5 * cost[e] <= upto || w == NW - 1)) {
                G("        { const double k = lS<%d>(sml); const double kp = k", (R_KAP + e) * PITCH);
                for (int r : fac[e]) G(" * lS<%d>(sml)", r * PITCH);
                G("; sS<%d>(sml, kp);", (R_KAP + e) * PITCH);
                G("\n#if QSS3_JAC\n          sc[%d] = k;", (S_K + e) * 32);
                if (kqe[e] >= 0) G(" sc[%d] = kp;", (S_KQ + kqe[e]) * 32);
                G("\n#endif\n        }\n");
                acc += cost[e]; ++e;
            }
            G("        break;\n");
        }
        G("    default: break;\n    }\n}\n");
    }
    {
        std::vector<std::vector<int>> sp(nsp), sm(nsp), tp(nsp), tm(nsp);
        for (int j = 0; j < M; ++j) if (R[j].mask) for (const Term &x : R[j].net) for (int u = 0; u < std::abs(x.nu); ++u) {
            (x.nu > 0 ? sp : sm)[x.sp].push_back((R_KAP + pos[j]) * PITCH);
            if (R[j].tb >= 0) (x.nu > 0 ? tp : tm)[x.sp].push_back((R_DLM + R[j].tb) * PITCH);
        }
        std::vector<double> cost(nsp);
        for (int s2 = 0; s2 < nsp; ++s2) cost[s2] = 6.0 + 2.0 * (sp[s2].size() + sm[s2].size()) + (tp[s2].size() + tm[s2].size());
        const std::vector<int> bin = lpt(cost, NW);
        // a signed sum with four partial sums: name = (sum of plus rows + off) - (sum of minus rows + off)
        auto emit_sum = [&](const char *name, const std::vector<int> &plus, const std::vector<int> &minus, int off) {
            for (int sign = 0; sign < 2; ++sign) {
                const std::vector<int> &l = sign ? minus : plus;
                const char *pre = sign ? "m" : "p";
                const int na = (int)std::min<size_t>(4, l.size());
                for (int a = 0; a < na; ++a) G("            double %s%s%d = lS<%d>(sml);\n", name, pre, a, l[a] + off);
                for (size_t t = 4; t < l.size(); ++t) G("            %s%s%d += lS<%d>(sml);\n", name, pre, (int)(t % 4), l[t] + off);
                G("            const double %s%s = ", name, pre);
                if (na == 0) G("0.0");
                else if (na == 1) G("%s%s0", name, pre);
                else if (na == 2) G("%s%s0 + %s%s1", name, pre, name, pre);
                else if (na == 3) G("(%s%s0 + %s%s1) + %s%s2", name, pre, name, pre, name, pre);
                else G("(%s%s0 + %s%s1) + (%s%s2 + %s%s3)", name, pre, name, pre, name, pre, name, pre);
                G(";\n");
            }
            G("            const double %s = %sp - %sm;\n", name, name, name);
        };
        G("__device__ __forceinline__ void qss_gen_sums(const int warp, const unsigned sml, double *sc, double *wdot, const long long ld, const bool active) {\n    switch (warp) {\n");
        for (int w = 0; w < NW; ++w) {
            G("    case %d:\n", w);
            for (int s2 = 0; s2 < nsp; ++s2) if (bin[s2] == w) {
                G("        {\n");
                emit_sum("w", sp[s2], sm[s2], 0);
                if (s2 < N) G("            if (wdot && active) wdot[%d * ld] = w;\n", s2);
                G("#if QSS3_JAC\n");
                emit_sum("et", sp[s2], sm[s2], MS * PITCH);
                emit_sum("tv", tp[s2], tm[s2], 0);
                G("            sS<%d>(sml, tv); sc[%d] = et;\n", (R_TV + s2) * PITCH, (S_ET + s2) * 32);
                G("#endif\n        }\n");
            }
            G("        break;\n");
        }
        G("    default: break;\n    }\n}\n");
    }
    }
    // ---- P4: closure solve of every group with its matrix in registers (subtraction-free elimination, Eq. 6
    //      L150-157, L159-171; readings G2, G8), level by level of the condensed DAG; also prepares U = P / D for dy/dx
    {
        G("__device__ __forceinline__ void qss_gen_closure(const int warp, const unsigned sml) {\n");
        std::vector<std::vector<int>> by_level(c.n_levels);
        for (int gi = 0; gi < c.n_groups; ++gi) by_level[(*c.lvl_of_group)[gi]].push_back(gi);
        for (int l = 0; l < c.n_levels; ++l) {
            G("    switch (warp) {\n");
            std::vector<std::vector<int>> bw(NW);
            for (size_t i = 0; i < by_level[l].size(); ++i) bw[i % NW].push_back(by_level[l][i]);
            for (int w = 0; w < NW; ++w) {
                if (bw[w].empty()) continue;
                G("    case %d: {\n", w);
                for (int gi : bw[w]) {
                    const std::vector<int> &mem = (*c.members)[gi];
                    const int sz = (int)mem.size(), base = R_CL + (*c.gbase)[gi];
                    const int oL = base + sz * sz, oP0 = oL + sz, oID = oP0 + sz;
                    G("        {\n");
                    for (int m = 0; m < sz; ++m) for (int j = 0; j < sz; ++j) if (m != j) G("            double a%d_%d = lS<%d>(sml);\n", m, j, (base + m * sz + j) * PITCH);
                    for (int k = 0; k < sz; ++k) G("            double L%d = lS<%d>(sml), q%d = lS<%d>(sml), d%d;\n", k, (oL + k) * PITCH, k, (oP0 + k) * PITCH, k);
                    for (int x = (*c.xp_begin)[gi]; x < (*c.xp_end)[gi]; ++x)
                        G("            q%d += lS<%d>(sml) * lS<%d>(sml);\n", (*c.pos_in_grp)[(*c.xpl)[x].first.first], (R_XP + x) * PITCH, (R_Y + (*c.xpl)[x].first.second) * PITCH);
                    for (int k = sz - 1; k >= 1; --k) {
                        G("            {   const double lk = L%d;\n                double Dk = lk;\n", k);
                        for (int m = 0; m < k; ++m) G("                Dk += a%d_%d;\n", m, k);
                        G("                const double iD = qss_rcp(Dk);\n                d%d = iD;\n", k);
                        for (int jj = 0; jj < k; ++jj) {
                            G("                {   const double f = a%d_%d * iD;\n                    L%d += f * lk;\n", k, jj, jj);
                            for (int m = 0; m < k; ++m) if (m != jj) G("                    a%d_%d += a%d_%d * f;\n", m, jj, m, k);
                            G("                }\n");
                        }
                        G("            }\n");
                    }
                    G("            d0 = qss_rcp(L0);\n");
                    for (int k = sz - 1; k >= 1; --k) {
                        G("            {   const double iD = d%d, tk = q%d * iD;\n", k, k);
                        for (int m = 0; m < k; ++m) G("                {   const double pmk = a%d_%d; a%d_%d = pmk * iD; q%d += pmk * tk; }\n", m, k, m, k, m);
                        G("            }\n");
                    }
                    for (int k = 0; k < sz; ++k) {
                        G("            {   double acc = q%d;\n", k);
                        for (int jj = 0; jj < k; ++jj) G("                acc += a%d_%d * q%d;\n", k, jj, jj);
                        G("                acc *= d%d;\n                q%d = acc;\n                sS<%d>(sml, acc);\n            }\n", k, k, (R_Y + mem[k]) * PITCH);
                    }
                    for (int m = 0; m < sz; ++m) for (int j = 0; j < sz; ++j) if (m != j) G("            sS<%d>(sml, a%d_%d);\n", (base + m * sz + j) * PITCH, m, j);
                    for (int k = 0; k < sz; ++k) G("            sS<%d>(sml, d%d);\n", (oID + k) * PITCH, k);
                    G("        }\n");
                }
                G("    } break;\n");
            }
            G("    default: break;\n    }\n    __syncthreads();\n");
        }
        G("}\n");
    }
    // ---- P8: one Jacobian column in registers: init, records, dy/dx solve, W_y dy/dx, stores --------------------------
    {
        int dist = 12, fdist = 4, sdist = 3, pdist = 8;      // loads run this many items ahead of their use
        if (const char *e = qss_devenv("QSS3_DIST")) std::sscanf(e, "%d,%d,%d,%d", &dist, &fdist, &sdist, &pdist);
        G("__device__ __forceinline__ void qss_gen_column(const int k, const int mode, const unsigned sml, const unsigned sml2, const double *sc, double *jc, const long long rs, const bool active) {\n    double ");
        for (int s = 0; s < nsp; ++s) G("c%d%s", s, s + 1 < nsp ? ", " : ";\n");
        G("    if (k < %d) {\n", N);
        for (int s = 0; s < nsp; ++s) G("        c%d = lS<%d>(sml);\n", s, (R_TV + s) * PITCH);
        G("    } else {\n");
        for (int s = 0; s < nsp; ++s) G("        c%d = lG<%d>(sc);\n", s, (S_ET + s) * 256);
        G("    }\n    switch (k) {\n");
        for (int k = 0; k < N; ++k) {
            const std::vector<Rec> &rr = rec[k];
            const int n = (int)rr.size();
            if (!n) continue;
            G("    case %d: {\n", k);
            auto load_A = [&](int i) { if (i < n) { if (rr[i].from_smem) G("        const double A%d = lS<%d>(sml);\n", i, rr[i].src); else G("        const double A%d = lG<%d>(sc);\n", i, rr[i].src); } };
            auto load_F = [&](int i) {
                if (i >= n) return;
                if (rr[i].f1 >= 0) G("        const double f%d = lS<%d>(sml);\n", i, rr[i].f1);
                if (rr[i].f2 >= 0) G("        const double h%d = lS<%d>(sml);\n", i, rr[i].f2);
            };
            for (int i = 0; i < dist; ++i) load_A(i);
            for (int i = 0; i < fdist; ++i) load_F(i);
            for (int i = 0; i < n; ++i) {
                load_A(i + dist);
                load_F(i + fdist);
                const Rec &r = rr[i];
                if (r.from_smem) G("        const double p%d = vmul(A%d, %.17g)", i, i, r.lit);
                else if (r.f1 >= 0) G("        const double p%d = vmul(A%d, f%d)", i, i, i);
                else G("        const double p%d = A%d", i, i);
                if (r.f2 >= 0) G(" * h%d", i);
                G(";");
                for (auto &t : r.tgt) {
                    const int a = std::abs(t.second);
                    if (a == 1) G(" c%d %s= p%d;", t.first, t.second > 0 ? "+" : "-", i);
                    else G(" c%d = fma(%s%d.0, p%d, c%d);", t.first, t.second > 0 ? "" : "-", a, i, t.first);
                }
                G("\n");
            }
            G("    } break;\n");
        }
        G("    default: break;\n    }\n");
        // the chain-rule term (dy/dx solve, W_y dy/dx) belongs to the exact Jacobian only; the constant-QSS and zero-QSS
        // approximations of PAPER.md L232 (mode 1, 2) stop at W_x
        G("    if (mode == 0) {\n");
        {   // dy/dx solve; the operations of independent groups are interleaved (two chains)
            std::vector<const Op *> ch[2];
            size_t len[2] = {0, 0};
            for (int gi = 0; gi < c.n_groups; ++gi) {
                const int w = c.xpl->empty() ? (len[0] <= len[1] ? 0 : 1) : 0;
                for (const Op &o : gops[gi]) { ch[w].push_back(&o); len[w] += 1 + o.terms.size(); }
            }
            std::vector<const Op *> seq;
            for (size_t i = 0; i < std::max(ch[0].size(), ch[1].size()); ++i) {
                if (i < ch[0].size()) seq.push_back(ch[0][i]);
                if (i < ch[1].size()) seq.push_back(ch[1][i]);
            }
            // (the shared-memory reads of operation i + sdist are issued before operation i is applied: ptxas keeps the order of
            //  the pinned loads and does not hoist them by itself when registers are short)
            auto load_op = [&](int i) {
                if (i >= (int)seq.size()) return;
                const Op &o = *seq[i];
                for (size_t t = 0; t < o.terms.size(); ++t) G("    const double u%d_%d = lS<%d>(sml);\n", i, (int)t, o.terms[t].first * PITCH);
                if (o.scale >= 0) G("    const double u%d_s = lS<%d>(sml);\n", i, o.scale * PITCH);
            };
            for (int i = 0; i < sdist; ++i) load_op(i);
            for (int i = 0; i < (int)seq.size(); ++i) {
                load_op(i + sdist);
                const Op &o = *seq[i];
                const int a = N + o.a;
                // (the first operation of every step is a pinned instruction: it keeps its place after the loads issued above)
                for (size_t t = 0; t < o.terms.size(); ++t) {
                    if (t == 0) G("    vfma(c%d, u%d_%d, c%d);\n", a, i, (int)t, N + o.terms[t].second);
                    else G("    c%d = fma(u%d_%d, c%d, c%d);\n", a, i, (int)t, N + o.terms[t].second, a);
                }
                if (o.scale >= 0) { if (o.terms.empty()) G("    c%d = vmul(c%d, u%d_s);\n", a, a, i); else G("    c%d *= u%d_s;\n", a, i); }
            }
        }
        // J[:, k] = W_x[:, k] + W_y dy/dx_k (Eq. 7), reaction by reaction: the QSS-consuming directions of reaction j
        // change its rate by t = kappa_f dy_qf - kappa_b dy_qb, scattered once with the net stoichiometry
        {
            // pair p (two consecutive kappa rows) is read by one 16-byte load before the first reaction that needs it
            std::vector<int> first_use((n_kq + 1) / 2, -1);
            for (int i = 0; i < (int)kq.size(); ++i) for (int dir = 0; dir < 2; ++dir)
                if (kq[i].idx[dir] >= 0 && first_use[kq[i].idx[dir] / 2] < 0) first_use[kq[i].idx[dir] / 2] = i;
            auto load_k = [&](int i) {
                if (i >= (int)kq.size()) return;
                for (size_t pp = 0; pp < first_use.size(); ++pp) if (first_use[pp] == i) G("    const double2 kq%d = lS2<%d>(sml2);\n", (int)pp, KQ_BASE + (int)pp * 528);
            };
            for (int i = 0; i < pdist; ++i) load_k(i);
            for (int i = 0; i < (int)kq.size(); ++i) {
                load_k(i + pdist);
                const KqRec &r = kq[i];
                if (r.idx[0] >= 0 && r.idx[1] >= 0) {
                    G("    {   const double t = vfms(kq%d.%c, c%d, kq%d.%c * c%d);", r.idx[0] / 2, r.idx[0] % 2 ? 'y' : 'x', N + r.q[0], r.idx[1] / 2, r.idx[1] % 2 ? 'y' : 'x', N + r.q[1]);
                    for (auto &t : r.tgt) {
                        const int a = std::abs(t.second);
                        if (a == 1) G(" c%d %s= t;", t.first, t.second > 0 ? "+" : "-");
                        else G(" c%d = fma(%s%d.0, t, c%d);", t.first, t.second > 0 ? "" : "-", a, t.first);
                    }
                } else {
                    // one direction: c_t += (+-nu_t) kappa dy_q; the first unit-coefficient target is the pinned instruction
                    const int dir = r.idx[0] >= 0 ? 0 : 1, sg = dir == 0 ? 1 : -1;
                    char kn[32];
                    std::snprintf(kn, sizeof kn, "kq%d.%c", r.idx[dir] / 2, r.idx[dir] % 2 ? 'y' : 'x');
                    int anchor = -1;
                    for (size_t u = 0; u < r.tgt.size(); ++u) if (std::abs(r.tgt[u].second) == 1) { anchor = (int)u; break; }
                    G("    {  ");
                    if (anchor < 0) G(" const double t = vmul(%s, c%d);", kn, N + r.q[dir]);
                    else G(" %s(c%d, %s, c%d);", sg * r.tgt[anchor].second > 0 ? "vfma" : "vfnma", r.tgt[anchor].first, kn, N + r.q[dir]);
                    for (size_t u = 0; u < r.tgt.size(); ++u) {
                        if ((int)u == anchor) continue;
                        const int sv = sg * r.tgt[u].second, a = std::abs(sv);
                        if (anchor < 0) G(" c%d = fma(%s%d.0, t, c%d);", r.tgt[u].first, sv > 0 ? "" : "-", a, r.tgt[u].first);
                        else if (a == 1) G(" c%d = fma(%s%s, c%d, c%d);", r.tgt[u].first, sv > 0 ? "" : "-", kn, N + r.q[dir], r.tgt[u].first);
                        else G(" c%d = fma(%s%d.0 * %s, c%d, c%d);", r.tgt[u].first, sv > 0 ? "" : "-", a, kn, N + r.q[dir], r.tgt[u].first);
                    }
                }
                G(" }\n");
            }
        }
        G("    }\n");
        G("    if (active) {\n");
        for (int i = 0; i < N; ++i) G("        __stcs(jc + %d * rs, c%d);\n", i, i);
        G("    }\n}\n");
        // columns of each warp: longest-processing-time assignment (the warps do not meet between columns)
        std::vector<double> cost(N + 1);
        double prod_cost = 0.0;
        for (const KqRec &r : kq) prod_cost += 3.0 + r.tgt.size();
        for (int k = 0; k <= N; ++k) {
            cost[k] = 150.0 + prod_cost;
            if (k < N) for (const Rec &r : rec[k]) cost[k] += 6.0 * (3.0 + r.tgt.size());       // (stream code is fetched, not cached)
        }
        const std::vector<int> bin = lpt(cost, NWC);
        size_t depth = 0;
        std::vector<std::vector<int>> cols(NWC);
        for (int k = 0; k <= N; ++k) cols[bin[k]].push_back(k);
        for (auto &cw : cols) { std::stable_sort(cw.begin(), cw.end(), [&](int a, int b) { return cost[a] > cost[b]; }); depth = std::max(depth, cw.size()); }
        // every other warp takes its columns in the opposite order, so that the fetch-bound record streams of one half of the
        // warps run against the shared-memory-bound products of the other half
        for (int w = 1; w < NWC; w += 2) std::reverse(cols[w].begin(), cols[w].end());
        G("#define QSS_GEN_DEPTH %d\n__constant__ int qss_gen_cols[] = {", (int)depth);
        for (int w = 0; w < NWC; ++w) for (size_t dd = 0; dd < depth; ++dd) G("%d, ", dd < cols[w].size() ? cols[w][dd] : -1);
        G("-1};\n");
    }
    v.gen = G.s;
    v.nw = NW; v.smem_bytes = rows * PITCH; v.scratch_rows = srows; v.n_slot = n_slot;
    v.n_pp = 0; v.n_kq = n_kq; v.n_groups = (int)groups.size();
    return true;
}

}  // namespace qssc
