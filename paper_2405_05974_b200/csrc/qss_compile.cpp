// Host-side mechanism compiler: qss_mech_desc_t -> flat device tables (QssTab).
//
// This is the run-time replacement of the paper's offline pre-processing (section 2.3;
// App. B): validate the linear-coupling premise (L73-77, L146), build the QSS dependency digraph,
// find its strongly connected components with Tarjan's algorithm, order the condensed DAG, and emit static
// gather / elimination schedules.  No symbolic expressions are generated (the paper's sympy + CSE path,
// L262-276, is prior art here): the kernels interpret these tables.
#include "qss_compile.h"
#include "qss_ctx.h"
#include "qss_devtools.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <cstring>
#include <map>
#include <stdexcept>

using namespace qssc;

namespace {

std::string fmt(const char *f, int a = 0, int b = 0, int c = 0) {
    char buf[256];
    std::snprintf(buf, sizeof buf, f, a, b, c);
    return buf;
}

// Tarjan's SCC algorithm on the QSS digraph (App. B): one DFS, adjacency lists.
// Returns component id per vertex; components are numbered in the order they are completed, which is a
// reverse topological order of the condensed DAG (a component is completed after everything it reaches).
int tarjan(int n, const std::vector<std::vector<int>> &adj, std::vector<int> &comp) {
    std::vector<int> index(n, -1), low(n, 0), stack;
    std::vector<char> on(n, 0);
    comp.assign(n, -1);
    int counter = 0, ncomp = 0;
    // iterative DFS (mechanisms may have hundreds of QSS species)
    struct Frame { int v; size_t e; };
    for (int root = 0; root < n; ++root) {
        if (index[root] != -1) continue;
        std::vector<Frame> call;
        call.push_back({root, 0});
        index[root] = low[root] = counter++;
        stack.push_back(root); on[root] = 1;
        while (!call.empty()) {
            Frame &f = call.back();
            int v = f.v;
            if (f.e < adj[v].size()) {
                int w = adj[v][f.e++];
                if (index[w] == -1) {
                    index[w] = low[w] = counter++;
                    stack.push_back(w); on[w] = 1;
                    call.push_back({w, 0});
                } else if (on[w]) {
                    low[v] = std::min(low[v], index[w]);
                }
            } else {
                if (low[v] == index[v]) {
                    for (;;) {
                        int w = stack.back(); stack.pop_back(); on[w] = 0;
                        comp[w] = ncomp;
                        if (w == v) break;
                    }
                    ++ncomp;
                }
                call.pop_back();
                if (!call.empty()) low[call.back().v] = std::min(low[call.back().v], low[v]);
            }
        }
    }
    return ncomp;
}


// ---------------------------------------------------------------------------------------------------------
// Kernel variant 1 ("slab-smem", qss_kernel_v1.cu): hot tables for the kernel-parameter constant bank, reaction
// records, shared-memory / scratch layout.  Applies when the mechanism is small enough (see the checks below);
// otherwise the general variant 0 is used.
// ---------------------------------------------------------------------------------------------------------
bool build_v1(const V1Ctx &c, QssCompiled &out, std::string &why) {
    const int N = c.N, Nq = c.Nq, M = c.M, nsp = c.nsp;
    const std::vector<Reaction> &R = *c.R;
    QssV1 &v = out.v1;
    v = QssV1();
    if (nsp > 126) { why = "more species than the one-byte row index of the column stream holds"; return false; }
    if (2 * M > 4096 || c.n_tb + 1 >= 4096) { why = "too many reactions for the packed tables of variant 1"; return false; }
    for (int j = 0; j < M; ++j) {
        for (int s = 0; s < 2; ++s) { int n = 0; for (const Term &x : R[j].side[s]) n += x.nu; if (n > 3) { why = "a reaction side has more than 3 molecules"; return false; } }
        for (const Term &x : R[j].net) if (x.nu < -7 || x.nu > 7) { why = "net stoichiometric coefficient out of range"; return false; }
    }
    std::vector<int32_t> H, ce_tab, cs_words;
    auto at = [&]() { return (int32_t)H.size(); };
    // closure gather
    {
        std::vector<int32_t> ptr{0}, dst, dir;
        for (auto &kv : *c.ce) { dst.push_back(kv.first); dir.insert(dir.end(), kv.second.begin(), kv.second.end()); ptr.push_back((int32_t)dir.size()); }
        v.n_centry = (int32_t)dst.size();
        // staged in shared memory with the W_y lists (t_ce_* are offsets into that table): pointers, destinations, kappa rows
        ce_tab.insert(ce_tab.end(), ptr.begin(), ptr.end());
        ce_tab.insert(ce_tab.end(), dst.begin(), dst.end());
        ce_tab.insert(ce_tab.end(), dir.begin(), dir.end());
    }
    {
        std::vector<int32_t> ptr{0}, dir, xm, xn;
        for (auto &e : *c.xpl) {
            xm.push_back((*c.pos_in_grp)[e.first.first]); xn.push_back(e.first.second);
            dir.insert(dir.end(), e.second.begin(), e.second.end()); ptr.push_back((int32_t)dir.size());
        }
        v.n_xp = (int32_t)xm.size();
        v.h_xp_ptr = at(); H.insert(H.end(), ptr.begin(), ptr.end());
        v.h_xp_dir = at(); H.insert(H.end(), dir.begin(), dir.end());
        v.h_xp_m = at(); H.insert(H.end(), xm.begin(), xm.end());
        v.h_xp_n = at(); H.insert(H.end(), xn.begin(), xn.end());
    }
    {
        v.h_group = at();
        int moff = 0;
        for (int g = 0; g < c.n_groups; ++g) {
            const int sz = (int)(*c.members)[g].size();
            int32_t rec[QSS_GI_STRIDE] = {sz, moff, (*c.gbase)[g], (*c.lvl_of_group)[g], (*c.xp_begin)[g], (*c.xp_end)[g], 0, 0};
            H.insert(H.end(), rec, rec + QSS_GI_STRIDE);
            moff += sz;
        }
        v.h_gmember = at();
        for (int g = 0; g < c.n_groups; ++g) H.insert(H.end(), (*c.members)[g].begin(), (*c.members)[g].end());
        std::vector<int32_t> lp(c.n_levels + 1, 0);
        for (int g = 0; g < c.n_groups; ++g) lp[(*c.lvl_of_group)[g] + 1]++;
        for (int l = 0; l < c.n_levels; ++l) lp[l + 1] += lp[l];
        v.h_level_ptr = at(); H.insert(H.end(), lp.begin(), lp.end());
    }
    // V rows: transported s -> s, the constant 1 -> N, QSS q -> N + 1 + q
    auto vrow = [&](int sp) { return sp < N ? sp : N + 1 + (sp - N); };
    std::vector<int32_t> q_tab;                            // per reaction: V rows of the QSS reactant of each direction (or the
    for (int j = 0; j < M; ++j) {                          //   1.0 row), third-body index; staged in shared memory
        const int qf = R[j].q[0] >= 0 ? N + 1 + R[j].q[0] : N, qb = R[j].q[1] >= 0 ? N + 1 + R[j].q[1] : N;
        q_tab.push_back(qf | (qb << 8) | ((R[j].tb + 1) << 16));
    }
    const int nw = QSS_V1_NW;
    // species incidence lists (their balanced assignment to warps follows below): one entry per unit of |nu|,
    //   h_ss: byte offset of Q_j (row 2j of s_KAP, dQ_j/dT follows at +256) | sign bit;  h_st: scratch row of dQ_j/dM | sign bit
    std::vector<std::vector<int32_t>> ss(nsp), st(nsp);
    for (int j = 0; j < M; ++j) if (R[j].mask) for (const Term &x : R[j].net) for (int u = 0; u < std::abs(x.nu); ++u) {
        const int32_t sgn = x.nu < 0 ? (int32_t)0x80000000 : 0;
        ss[x.sp].push_back((j * 512) | sgn);
        if (R[j].tb >= 0) st[x.sp].push_back(R[j].tb | sgn);
    }
    {
        std::vector<int32_t> ptr{0}, all, tptr{0}, tall;
        for (int s = 0; s < nsp; ++s) {
            all.insert(all.end(), ss[s].begin(), ss[s].end()); ptr.push_back((int32_t)all.size());
            tall.insert(tall.end(), st[s].begin(), st[s].end()); tptr.push_back((int32_t)tall.size());
        }
        v.h_ss_ptr = at(); H.insert(H.end(), ptr.begin(), ptr.end());
        v.h_ss = at(); H.insert(H.end(), all.begin(), all.end());
        H.push_back(0); H.push_back(0);                      // (the kernel's software pipeline reads two words past a list)
        v.h_st_ptr = at(); H.insert(H.end(), tptr.begin(), tptr.end());
        v.h_st = at(); H.insert(H.end(), tall.begin(), tall.end());
    }
    // W_y entries, row-major (i, then q): gather lists over the directions consuming q (lists go to the global blob)
    std::map<std::pair<int, int>, std::vector<int32_t>> wy;
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
        if (!((R[j].mask >> dir) & 1) || R[j].q[dir] < 0) continue;
        for (const Term &x : R[j].net) if (x.sp < N) {        // one word per unit of |nu|: byte offset of kappa_d in s_KAP | sign bit
            const int e = dir == 0 ? x.nu : -x.nu;
            for (int u = 0; u < std::abs(e); ++u) wy[{x.sp, R[j].q[dir]}].push_back(((2 * j + dir) * 256) | (e < 0 ? (int32_t)0x80000000 : 0));
        }
    }
    // the same sum direction by direction (specialised build): W_y dy/dx = sum over the enabled directions d that consume a QSS
    // species q(d) of kappa_d dy_q(d)/dx nu_d -- one shared-memory read per DIRECTION instead of one per W_y entry
    struct GenDir { int d, q; std::vector<std::pair<int, int>> tgt; };           // (transported species, signed coefficient)
    std::vector<GenDir> gdir;
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
        if (!((R[j].mask >> dir) & 1) || R[j].q[dir] < 0) continue;
        GenDir gd{2 * j + dir, R[j].q[dir], {}};
        for (const Term &x : R[j].net) if (x.sp < N) gd.tgt.push_back({x.sp, dir == 0 ? x.nu : -x.nu});
        if (!gd.tgt.empty()) gdir.push_back(gd);
    }
    std::vector<int32_t> wya_ptr{0}, wya_all;
    {
        std::vector<int32_t> rptr{0}, roff;
        int row = 0;
        for (auto &kv : wy) {
            while (row < kv.first.first) { rptr.push_back((int32_t)roff.size()); ++row; }
            roff.push_back(kv.first.second * nw * 256);          // byte offset of dy_q/dx rows inside the s_YC region
            wya_all.insert(wya_all.end(), kv.second.begin(), kv.second.end()); wya_ptr.push_back((int32_t)wya_all.size());
        }
        while (row < N) { rptr.push_back((int32_t)roff.size()); ++row; }
        v.n_wy = (int32_t)roff.size();
        v.h_wr_ptr = at(); H.insert(H.end(), rptr.begin(), rptr.end());
    }
    // ---- shared-memory layout (rows of 256 bytes) and scratch layout
    int rows_fixed = 0;
    auto take = [&](int n) { int r = rows_fixed; rows_fixed += n; return r; };
    v.s_V = take(N + 1 + Nq); v.s_CT = take(1); v.s_CL = take(c.cl_size); v.s_XP = take(v.n_xp); v.s_TV = take(nsp); v.s_Z0 = take(1);
    const int max_rows = (227 * 1024) / 256;
    const int region = std::max((nsp + 1) * nw, 2 * M + 2 * (nsp + 1));    // round buffers: nsp rows + 1 junk row per column
    if (c.n_tb > 2 * (nsp + 1)) { why = "more third-body reactions than the shared-memory rows that hold dQ/dM for the species sums"; return false; }
    if (rows_fixed + region > max_rows) { why = "per-cell state does not fit the shared memory of one SM"; return false; }
    v.nw = nw;
    v.s_WX = rows_fixed; v.s_YC = rows_fixed + N * nw;       // one column buffer: row (species) r of column w at r * nw + w
    v.s_KAP = rows_fixed; v.s_G = rows_fixed + 2 * M; v.s_H = v.s_G + nsp + 1;
    // the W_y assembly lists are staged once per block in the spare shared memory behind the per-cell rows
    v.t_ce_ptr = (int32_t)(wya_ptr.size() + wya_all.size()); v.t_ce_dst = v.t_ce_ptr + v.n_centry + 1; v.t_ce_dir = v.t_ce_dst + v.n_centry;
    v.t_q = (int32_t)(wya_ptr.size() + wya_all.size() + ce_tab.size());
    v.n_tab_words = v.t_q + (int32_t)q_tab.size();
    v.s_TAB = rows_fixed + region;
    v.smem_rows = v.s_TAB + (v.n_tab_words * 4 + 255) / 256;
    if (v.smem_rows > max_rows) { why = "per-cell state and staged tables do not fit the shared memory of one SM"; return false; }
    {
        int o = 0;
        auto tk = [&](int n) { int r = o; o += n; return r; };
        v.g_K = tk(2 * M); v.g_DF = tk(M); v.g_DC = tk(M); v.g_ET = tk(nsp); v.g_QM = tk(c.n_tb); v.g_WY = tk(v.n_wy);
        v.scratch_rows = o;
        if (o > 65535) { why = "scratch rows beyond the 16-bit offsets of variant 1"; return false; }
    }
    // ---- column stream: everything that is scattered into column k of [W_x; G_x], as records
    //   w0 = scratch row of A | n_entries << 16 | has_val << 20 | |nu| << 21 | own << 24      part = |nu| * A * V[o1] * V[o2] (* val)
    //        own: the contribution to the column's own row k (almost every record has one) is kept in a register: 1 add, 2 subtract
    //   w1 = byte offset of V row o1 | byte offset of V row o2 << 16        (has_val: index of val in the double blob)
    //   w2, w3 = up to 8 targets (bytes): species row of the column buffer | 0x80 if the term is subtracted; nsp = none (junk row)
    // One record per (enabled direction, molecule slot holding species k): A = k_d, o1/o2 = the other two slots
    // (Eq. 9 first parenthesis); one per non-unity third-body efficiency: A = dQ_j/dM, val = alpha_jk - 1.
    auto voff = [&](int vr) { return (v.s_V + vr) * 256; };
    std::vector<std::vector<int32_t>> cs(N);
    std::vector<double> effv;                              // (alpha - 1) values, read from the double blob
    bool cs_ok = true;
    // the same records, unpacked, for the run-time specialised pass A (qss_gen_pass_a below)
    struct GenRec { int rowA, o1, o2, mag; bool has_val; double val; std::vector<std::pair<int, int>> tgt; };   // tgt: (species row, +1 / -1)
    std::vector<std::vector<GenRec>> grec(N);
    auto push_record = [&](int k, int rowA, int o1, int o2, const std::vector<Term> &net, int sgn, bool has_val, double val) {
        for (int mag = 1; mag <= 7; ++mag) {                 // one record per magnitude |nu| (almost always only 1)
            std::vector<int> idx;
            int own = 0;                                     // the column's own row k is accumulated in a register: 1 add, 2 subtract
            GenRec gr{rowA, o1, o2, mag, has_val, val, {}};
            for (const Term &x : net) if (std::abs(x.nu) == mag) {
                gr.tgt.push_back({x.sp, sgn * x.nu < 0 ? -1 : 1});
                if (x.sp == k) own = sgn * x.nu < 0 ? 2 : 1;
                else idx.push_back(x.sp | (sgn * x.nu < 0 ? 0x80 : 0));
            }
            if (idx.empty() && !own) continue;
            grec[k].push_back(gr);
            if (idx.size() > 8) { cs_ok = false; return; }
            const uint32_t none = (uint32_t)nsp * 0x01010101u;   // the junk row of the column buffer
            uint32_t w[2] = {none, none};
            for (size_t u = 0; u < idx.size(); ++u) { w[u / 4] &= ~(0xFFu << (8 * (u % 4))); w[u / 4] |= (uint32_t)idx[u] << (8 * (u % 4)); }
            cs[k].push_back(rowA | ((int)idx.size() << 16) | ((has_val ? 1 : 0) << 20) | (mag << 21) | (own << 24));
            if (has_val) { cs[k].push_back((int32_t)effv.size()); effv.push_back(val); }
            else cs[k].push_back(o1 | (o2 << 16));
            cs[k].push_back((int32_t)w[0]); cs[k].push_back((int32_t)w[1]);
        }
    };
    for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
        if (!((R[j].mask >> dir) & 1)) continue;
        std::vector<int> slots;                              // species of each molecule of the reactant side
        for (const Term &x : R[j].side[dir]) for (int u = 0; u < x.nu; ++u) slots.push_back(x.sp);
        for (size_t pp = 0; pp < slots.size(); ++pp) {
            if (slots[pp] >= N) continue;
            int o[2] = {N, N}, no = 0;
            for (size_t q = 0; q < slots.size(); ++q) if (q != pp) o[no++] = vrow(slots[q]);
            push_record(slots[pp], v.g_K + 2 * j + dir, voff(o[0]), voff(o[1]), R[j].net, dir == 0 ? 1 : -1, false, 0.0);
        }
    }
    for (int k = 0; k < N; ++k)
        for (auto &e : (*c.effc)[k]) if (R[e.first].mask) push_record(k, v.g_QM + R[e.first].tb, voff(N), voff(N), R[e.first].net, 1, true, e.second);
    if (!cs_ok) { why = "a reaction changes more than 8 molecules (scatter record of variant 1)"; return false; }
    if (voff(N + Nq) > 65535) { why = "V rows beyond the 16-bit offsets of variant 1"; return false; }
    {
        if (H.size() & 1) H.push_back(0);
        // records are applied two at a time (the kernel issues the row loads of both together), so they are packed into
        // PAIRS with disjoint target rows; a record without a partner gets the null record
        const uint32_t junk4 = (uint32_t)nsp * 0x01010101u;
        const int32_t null_rec[4] = {v.g_K, voff(N) | (voff(N) << 16), (int32_t)junk4, (int32_t)junk4};
        auto rows_of = [&](const int32_t *r) {
            uint64_t m0 = 0, m1 = 0;
            for (int u = 0; u < 8; ++u) { const int row = ((uint32_t)r[2 + u / 4] >> (8 * (u % 4))) & 127; if (row != nsp) (row < 64 ? m0 : m1) |= 1ull << (row & 63); }
            return std::make_pair(m0, m1);
        };
        std::vector<int32_t> ptr{0}, all;
        for (int k = 0; k < N; ++k) {
            std::vector<const int32_t *> pending;
            for (size_t o = 0; o < cs[k].size(); o += 4) {
                const int32_t *r = &cs[k][o];
                const auto mr = rows_of(r);
                size_t hit = pending.size();
                for (size_t q = 0; q < pending.size(); ++q) { const auto mq = rows_of(pending[q]); if (!(mq.first & mr.first) && !(mq.second & mr.second)) { hit = q; break; } }
                if (hit == pending.size()) { pending.push_back(r); continue; }
                all.insert(all.end(), pending[hit], pending[hit] + 4); all.insert(all.end(), r, r + 4);
                pending.erase(pending.begin() + hit);
            }
            for (const int32_t *r : pending) { all.insert(all.end(), r, r + 4); all.insert(all.end(), null_rec, null_rec + 4); }
            ptr.push_back((int32_t)all.size());
        }
        ptr.push_back((int32_t)all.size());                  // the T column has an empty stream
        // two harmless sentinel pairs: the kernel's software pipeline fetches two pairs ahead of the one it applies
        for (int u = 0; u < 4; ++u) all.insert(all.end(), null_rec, null_rec + 4);
        cs_words = all;                                      // placed at the end: constant bank if it fits, else global memory
        v.h_cs_ptr = at(); H.insert(H.end(), ptr.begin(), ptr.end());
    }
    struct GenOp { int a; std::vector<std::pair<int, int>> terms; int scale; };     // y[a] = (y[a] + sum F y[b]) * S; (F row, QSS index b); scale -1: none
    std::vector<std::vector<GenOp>> ggops;
    // ---- dy/dx solve program: fixed-format row operations on the warp's dy/dx column,
    //          y[a] = (y[a] + F0 y[b0] + F1 y[b1] + F2 y[b2]) * S
    //      in the order cross-group terms, back-elimination (with U[m][k] = P[m][k] / D_k), forward substitution (S = 1/D),
    //      longer rows chained over several operations; unused terms read the zero row, unused scales the 1.0 row.
    //   4 words: a | n_terms << 12 | b0 << 16 ; b1 | b2 << 16 ; F0 | F1 << 16 ; F2 | S << 16   (a, b: rows relative to the warp's dy/dx
    //   column; F, S: absolute shared-memory rows).  Independent groups are dealt to TWO chains that the kernel
    //   advances together (one operation of each per step), which halves the length of the dependent chain.
    {
        const int one = v.s_V + N, zero = v.s_Z0, junk = (nsp - N) * nw;       // junk: the column's spare row, relative to dy/dx
        auto yoff = [&](int q) { return q * nw; };
        typedef std::vector<int32_t> Ops;
        auto emit = [&](Ops &o, int a, std::vector<std::pair<int, int>> terms, int scale) {   // terms: (F row, b row)
            size_t t = 0;
            do {
                int f[3] = {zero, zero, zero}, bb[3] = {a, a, a}, nt = 0;
                for (int u = 0; u < 3 && t < terms.size(); ++u, ++t, ++nt) { f[u] = terms[t].first; bb[u] = terms[t].second; }
                const int sc_ = t >= terms.size() ? scale : one;
                o.push_back(a | (nt << 12) | (bb[0] << 16)); o.push_back(bb[1] | (bb[2] << 16)); o.push_back(f[0] | (f[1] << 16)); o.push_back(f[2] | (sc_ << 16));
            } while (t < terms.size());
        };
        std::vector<Ops> gops(c.n_groups);
        ggops.assign(c.n_groups, {});
        for (int g = 0; g < c.n_groups; ++g) {
            const std::vector<int> &mem = (*c.members)[g];
            const int sz = (int)mem.size(), base = v.s_CL + (*c.gbase)[g];
            for (int x = (*c.xp_begin)[g]; x < (*c.xp_end)[g]; ++x) {
                const auto &e = (*c.xpl)[x];
                emit(gops[g], yoff(e.first.first), {{v.s_XP + x, yoff(e.first.second)}}, one);
                ggops[g].push_back({e.first.first, {{v.s_XP + x, e.first.second}}, -1});
            }
            for (int m = sz - 2; m >= 0; --m) {
                std::vector<std::pair<int, int>> t, tq;
                for (int k = m + 1; k < sz; ++k) { t.push_back({base + m * sz + k, yoff(mem[k])}); tq.push_back({base + m * sz + k, mem[k]}); }
                emit(gops[g], yoff(mem[m]), t, one);
                if (!tq.empty()) ggops[g].push_back({mem[m], tq, -1});
            }
            for (int k = 0; k < sz; ++k) {
                std::vector<std::pair<int, int>> t, tq;
                for (int jj = 0; jj < k; ++jj) { t.push_back({base + k * sz + jj, yoff(mem[jj])}); tq.push_back({base + k * sz + jj, mem[jj]}); }
                emit(gops[g], yoff(mem[k]), t, base + sz * sz + 2 * sz + k);
                ggops[g].push_back({mem[k], tq, base + sz * sz + 2 * sz + k});
            }
        }
        Ops chain[2];
        for (int g = 0; g < c.n_groups; ++g) {               // groups coupled across (n_xp > 0) stay in order on one chain
            Ops &dst = v.n_xp > 0 ? chain[0] : (chain[0].size() <= chain[1].size() ? chain[0] : chain[1]);
            dst.insert(dst.end(), gops[g].begin(), gops[g].end());
        }
        if ((Nq + 1) * nw >= 4096) { why = "dy/dx rows beyond the 12-bit field of the solve operations"; return false; }
        const int32_t nop[4] = {junk | (junk << 16), junk | (junk << 16), zero | (zero << 16), zero | (one << 16)};
        while (chain[0].size() < chain[1].size()) chain[0].insert(chain[0].end(), nop, nop + 4);
        while (chain[1].size() < chain[0].size()) chain[1].insert(chain[1].end(), nop, nop + 4);
        if (H.size() & 1) H.push_back(0);
        v.n_sp_ops = (int32_t)chain[0].size() / 4;
        v.h_sp = at();
        for (int i = 0; i < v.n_sp_ops; ++i) { H.insert(H.end(), chain[0].begin() + 4 * i, chain[0].begin() + 4 * i + 4); H.insert(H.end(), chain[1].begin() + 4 * i, chain[1].begin() + 4 * i + 4); }
    }
    // ---- species sums: balanced (longest-processing-time) assignment to warps
    {
        std::vector<int> idx(nsp);
        for (int s = 0; s < nsp; ++s) idx[s] = s;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return ss[a].size() > ss[b].size(); });
        std::vector<std::vector<int32_t>> bin(nw);
        std::vector<double> load(nw, 0.0);
        for (int i : idx) { int b = (int)(std::min_element(load.begin(), load.end()) - load.begin()); bin[b].push_back(i); load[b] += 6.0 + ss[i].size(); }
        std::vector<int32_t> ptr{0}, all;
        for (int w = 0; w < nw; ++w) { all.insert(all.end(), bin[w].begin(), bin[w].end()); ptr.push_back((int32_t)all.size()); }
        v.h_ssw_ptr = at(); H.insert(H.end(), ptr.begin(), ptr.end());
        v.h_ssw = at(); H.insert(H.end(), all.begin(), all.end());
    }
    {   // pass B tiles: every warp owns up to 3 Jacobian rows (balanced by their number of W_y entries) and sweeps the union
        // of their W_y columns once per round: h_tile word = q | row mask << 8, in ascending q (the W_y entries of a row are
        // stored in the same order, so a running index per row finds them)
        if (N > 3 * nw) { why = "more than 3 Jacobian rows per warp (register tile of pass B)"; return false; }
        std::vector<int> idx(N), cnt(N, 0);
        std::vector<std::vector<int>> qs(N);
        for (auto &kv : wy) { cnt[kv.first.first]++; qs[kv.first.first].push_back(kv.first.second); }
        for (int i = 0; i < N; ++i) idx[i] = i;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cnt[a] > cnt[b]; });
        std::vector<std::vector<int32_t>> bin(nw);
        std::vector<double> load(nw, 0.0);
        for (int i : idx) {
            int best = -1;
            for (int w = 0; w < nw; ++w) if (bin[w].size() < 3 && (best < 0 || load[w] < load[best])) best = w;
            bin[best].push_back(i); load[best] += 14.0 + cnt[i];
        }
        std::vector<int32_t> rows, tptr{0}, tile;
        for (int w = 0; w < nw; ++w) {
            for (int r = 0; r < 3; ++r) rows.push_back(r < (int)bin[w].size() ? bin[w][r] : -1);
            for (int q = 0; q < Nq; ++q) {
                int mask = 0;
                for (int r = 0; r < (int)bin[w].size(); ++r) if (std::find(qs[bin[w][r]].begin(), qs[bin[w][r]].end(), q) != qs[bin[w][r]].end()) mask |= 1 << r;
                if (mask) tile.push_back(q | (mask << 8));
            }
            tptr.push_back((int32_t)tile.size());
        }
        v.h_rw = at(); H.insert(H.end(), rows.begin(), rows.end());
        v.h_tile_ptr = at(); H.insert(H.end(), tptr.begin(), tptr.end());
        v.h_tile = at(); H.insert(H.end(), tile.begin(), tile.end());
    }
    // ---- Jacobian columns: rounds of nw columns of similar cost (the warps meet at a barrier after every round)
    {
        std::vector<int> idx(N + 1);
        for (int k = 0; k <= N; ++k) idx[k] = k;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return (a < N ? cs[a].size() : 0) > (b < N ? cs[b].size() : 0); });
        v.n_rounds = (N + 1 + nw - 1) / nw;
        v.h_cw = at();
        for (int i = 0; i < v.n_rounds * nw; ++i) H.push_back(i <= N ? idx[i] : -1);
    }
    // ---- third-body efficiencies (alpha - 1) by reaction, in the constant bank: the rate phase walks them for every
    //      third-body / fall-off reaction, and a walk through global memory is a chain of ~700-cycle L2 reads
    std::vector<int> eff_first(M, 0), eff_count(M, 0);
    {
        std::vector<double> val; std::vector<uint32_t> off;
        for (int j = 0; j < M; ++j) {
            eff_first[j] = (int)val.size();
            if (R[j].type >= 1) for (int k = 0; k < N; ++k) for (auto &e : (*c.effc)[k]) if (e.first == j) { val.push_back(e.second); off.push_back((uint32_t)voff(k)); }
            eff_count[j] = (int)val.size() - eff_first[j];
        }
        if (val.size() > 65535) { why = "too many third-body efficiencies for variant 1"; return false; }
        if (H.size() & 1) H.push_back(0);
        v.h_eff_val = at();
        for (double x : val) { int32_t w[2]; std::memcpy(w, &x, 8); H.push_back(w[0]); H.push_back(w[1]); }
        v.h_eff_off = at();
        for (size_t i = 0; i < off.size(); i += 2) H.push_back((int32_t)(off[i] | ((i + 1 < off.size() ? off[i + 1] : 0u) << 16)));
    }
    // the column streams are the largest table: they go to the constant bank when they fit, otherwise to global memory (the
    // kernel's software pipeline fetches them two pairs ahead, so the L2 latency is covered); QSS_CS_GLOBAL=1 forces the latter
    if (H.size() & 1) H.push_back(0);
    v.cs_global = ((int)(H.size() + cs_words.size()) > QSS_V1_HMAX || std::getenv("QSS_CS_GLOBAL")) ? 1 : 0;
    if (!v.cs_global) { v.h_cs = at(); H.insert(H.end(), cs_words.begin(), cs_words.end()); }
    if ((int)H.size() > QSS_V1_HMAX) { why = "hot tables exceed the kernel-parameter budget of variant 1"; return false; }
    v.h_used = (int32_t)H.size();
    std::memcpy(v.h, H.data(), H.size() * sizeof(int32_t));
    // ---- W_y assembly lists (appended to the int blob)
    {
        std::vector<int32_t> &I = out.I;
        v.i_wya_ptr = (int32_t)I.size(); I.insert(I.end(), wya_ptr.begin(), wya_ptr.end());   // [n_wy + 1] then the words
        I.insert(I.end(), wya_all.begin(), wya_all.end());
        I.insert(I.end(), ce_tab.begin(), ce_tab.end());
        I.insert(I.end(), q_tab.begin(), q_tab.end());       // (everything up to here is staged contiguously in shared memory)
        if (v.cs_global) { while (I.size() & 3) I.push_back(0); v.h_cs = (int32_t)I.size(); I.insert(I.end(), cs_words.begin(), cs_words.end()); }
    }
    // ---- reaction records (appended to the int blob), in processing order
    {
        std::vector<int32_t> &I = out.I;
        while (I.size() & 3) I.push_back(0);               // records are read as 16-byte vectors
        v.i_rrec = (int32_t)I.size();
        for (int r = 0; r < M; ++r) {
            const int j = (*c.rorder)[r];
            // w0 = j | type << 12 | mask << 14 | (tb + 1) << 16; w1..w3 = six 16-bit byte offsets of the V rows of the
            // reactant / product molecules (QSS and empty slots -> the 1.0 row); w4..w6 = six byte offsets (relative to
            // s_G) of their g/RT rows (empty slots -> the zero row); w7 = first third-body efficiency | count << 16
            int32_t rec[QSS_V1_RREC] = {j | (R[j].type << 12) | (R[j].mask << 14) | ((R[j].tb + 1) << 16), 0, 0, 0, 0, 0, 0, 0};
            uint32_t kap[6], gr[6];
            for (int s = 0; s < 2; ++s) {
                int n = 0;
                for (int u = 0; u < 3; ++u) { kap[3 * s + u] = (uint32_t)(v.s_V + N) * 256u; gr[3 * s + u] = (uint32_t)nsp * 256u; }
                for (const Term &x : R[j].side[s]) for (int u = 0; u < x.nu; ++u) {
                    kap[3 * s + n] = (uint32_t)(v.s_V + (x.sp < N ? x.sp : N)) * 256u; gr[3 * s + n] = (uint32_t)x.sp * 256u; ++n;
                }
            }
            for (int u = 0; u < 3; ++u) { rec[1 + u] = (int32_t)(kap[2 * u] | (kap[2 * u + 1] << 16)); rec[4 + u] = (int32_t)(gr[2 * u] | (gr[2 * u + 1] << 16)); }
            rec[7] = eff_first[j] | (eff_count[j] << 16);        // third-body efficiencies of this reaction in h_eff_*
            I.insert(I.end(), rec, rec + QSS_V1_RREC);
        }
    }
    v.N = N; v.Nq = Nq; v.M = M; v.nsp = nsp; v.n_tb = c.n_tb; v.n_groups = c.n_groups; v.n_levels = c.n_levels;
    v.d_thermo = out.tab.d_thermo; v.d_effm1 = out.tab.d_effm1;
    v.d_effv = (int32_t)out.D.size();
    out.D.insert(out.D.end(), effv.begin(), effv.end());
    {   // rate records again, in processing order (so that a warp can prefetch the next one without knowing j)
        std::vector<double> &Dd = out.D;
        v.d_rate_r = (int32_t)Dd.size();
        for (int r = 0; r < M; ++r) {
            const size_t src = (size_t)out.tab.d_rate + (size_t)(*c.rorder)[r] * QSS_RD_STRIDE;
            for (int u = 0; u < QSS_RD_STRIDE; ++u) Dd.push_back(Dd[src + u]);
        }
    }
    v.i_eff_ptr = out.tab.i_eff_ptr; v.i_eff_sp = out.tab.i_eff_sp;
    // ---- run-time specialised pass A (compiled with NVRTC by qss_jit.cpp and included by qss_kernel_v1.cu under QSS_GEN):
    //      the column lives in REGISTERS c0..c{nsp-1}; every record of the column stream becomes straight-line code with
    //      immediate offsets (1 L2 read of A fetched `dist` records ahead, <= 2 shared-memory factors, 2 multiplications,
    //      one add per target row); the dy/dx solve is the same row operations on registers; the column is then written
    //      to the round buffer for pass B.  Same operations in the same order per row as the interpreter, except that the
    //      interpreter applies the records of a column in paired order (rounding-order difference only).
    if (v.n_wy + N + nw <= region) {                         // (W_y and the staged inputs of the next slab must fit the time-shared region)
        std::string &g = out.v1_gen;
        char b[256];
        auto P = [&](const char *f, auto... a) {
            const int n_ = std::snprintf(b, sizeof b, f, a...);
            if (n_ < 0 || n_ >= (int)sizeof b) throw std::runtime_error("generated line exceeds the line buffer");
            g += b;
        };
        const int one = voff(N), dist = 12;
        g += "// generated by qss_compile.cpp for one mechanism: pass A of the Jacobian sweep (see qss_kernel_v1.cu)\n";
        g += "__device__ __forceinline__ void qss_gen_column(const int k, const unsigned sml, const double *sc, double *jc, const long long rs, const bool active) {\n";
        g += "    double ";
        for (int s = 0; s < nsp; ++s) P("c%d%s", s, s + 1 < nsp ? ", " : ";\n");
        P("    if (k < %d) {\n", N);
        for (int s = 0; s < nsp; ++s) P("        c%d = lS<%d>(sml);\n", s, (v.s_TV + s) * 256);
        g += "    } else {\n";
        for (int s = 0; s < nsp; ++s) P("        c%d = lG<%d>(sc);\n", s, (v.g_ET + s) * 256);
        g += "    }\n    switch (k) {\n";
        for (int k = 0; k < N; ++k) {
            const std::vector<GenRec> &rr = grec[k];
            const int n = (int)rr.size();
            if (!n) continue;
            P("    case %d: {\n", k);
            auto load_A = [&](int i) { if (i < n) P("        const double A%d = lG<%d>(sc);\n", i, rr[i].rowA * 256); };
            auto load_F = [&](int i) {
                if (i >= n || rr[i].has_val) return;
                if (rr[i].o1 != one) P("        const double f%d = lS<%d>(sml);\n", i, rr[i].o1);
                if (rr[i].o2 != one) P("        const double h%d = lS<%d>(sml);\n", i, rr[i].o2);
            };
            for (int i = 0; i < dist; ++i) load_A(i);
            load_F(0); load_F(1);
            for (int i = 0; i < n; ++i) {
                load_A(i + dist);
                load_F(i + 2);
                const GenRec &r = rr[i];
                P("        const double p%d = A%d", i, i);
                if (r.has_val) P(" * %.17g", r.val * r.mag);
                else {
                    if (r.o1 != one) P(" * f%d", i);
                    if (r.o2 != one) P(" * h%d", i);
                    if (r.mag > 1) P(" * %d.0", r.mag);
                }
                g += ";";
                for (auto &t : r.tgt) P(" c%d %s= p%d;", t.first, t.second > 0 ? "+" : "-", i);
                g += "\n";
            }
            g += "    } break;\n";
        }
        g += "    default: break;\n    }\n";
        // dy/dx solve on the QSS rows c{N+q}; the operations of independent groups are interleaved
        {
            std::vector<const GenOp *> ch[2];
            size_t len[2] = {0, 0};
            for (int gi = 0; gi < c.n_groups; ++gi) {
                const int w = v.n_xp > 0 ? 0 : (len[0] <= len[1] ? 0 : 1);
                for (const GenOp &o : ggops[gi]) { ch[w].push_back(&o); len[w] += 1 + o.terms.size(); }
            }
            int uid = 0;
            auto emit_op = [&](const GenOp &o) {
                const int a = N + o.a;
                for (size_t t = 0; t < o.terms.size(); ++t) P("    const double u%d_%d = lS<%d>(sml);\n", uid, (int)t, o.terms[t].first * 256);
                if (o.scale >= 0) P("    const double u%d_s = lS<%d>(sml);\n", uid, o.scale * 256);
                for (size_t t = 0; t < o.terms.size(); ++t) P("    c%d = fma(u%d_%d, c%d, c%d);\n", a, uid, (int)t, N + o.terms[t].second, a);
                if (o.scale >= 0) P("    c%d *= u%d_s;\n", a, uid);
                ++uid;
            };
            for (size_t i = 0; i < std::max(ch[0].size(), ch[1].size()); ++i) {
                if (i < ch[0].size()) emit_op(*ch[0][i]);
                if (i < ch[1].size()) emit_op(*ch[1][i]);
            }
        }
        // J[:, k] = W_x[:, k] + W_y dy/dx_k (Eq. 7) in place on the registers of the column: W_y (per cell, n_wy rows,
        // row-major, ascending q within a row) was copied to shared memory behind the fixed state; then 35 coalesced stores
        //   (by direction when that needs fewer rows than W_y has entries: kappa_d of the QSS-consuming directions was copied instead)
        const bool by_dir = (int)gdir.size() <= v.n_wy && !qss_devenv("QSS_GEN_WY");
        if (by_dir) {
            for (size_t r = 0; r < gdir.size(); ++r) {
                P("    {   const double kd = lS<%d>(sml);\n", (v.s_KAP + (int)r) * 256);
                for (auto &t : gdir[r].tgt) {
                    const int a = std::abs(t.second);
                    if (a == 1) P("        c%d = fma(%skd, c%d, c%d);\n", t.first, t.second < 0 ? "-" : "", N + gdir[r].q, t.first);
                    else P("        c%d = fma(%skd * %d.0, c%d, c%d);\n", t.first, t.second < 0 ? "-" : "", a, N + gdir[r].q, t.first);
                }
                g += "    }\n";
            }
        } else {
            int e = 0;
            for (auto &kv : wy) { P("    c%d = fma(lS<%d>(sml), c%d, c%d);\n", kv.first.first, (v.s_KAP + e) * 256, N + kv.first.second, kv.first.first); ++e; }
        }
        P("#define QSS_GEN_NROWS %d\n", by_dir ? (int)gdir.size() : v.n_wy);
        g += "    if (active) {\n";
        for (int i = 0; i < N; ++i) P("        __stcs(jc + %d * rs, c%d);\n", i, i);
        g += "    }\n}\n";
        // columns of each warp: longest-processing-time assignment (the warps do not meet between columns)
        {
            std::vector<int> idx(N + 1);
            for (int k = 0; k <= N; ++k) idx[k] = k;
            auto cost = [&](int k) { return 300.0 + 2.0 * v.n_wy + (k < N ? 8.0 * grec[k].size() : 0.0); };
            std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cost(a) > cost(b); });
            std::vector<std::vector<int>> bin(nw);
            std::vector<double> load(nw, 0.0);
            for (int k : idx) { const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin()); bin[w].push_back(k); load[w] += cost(k); }
            size_t depth = 0;
            for (auto &bb : bin) depth = std::max(depth, bb.size());
            P("#define QSS_GEN_DEPTH %d\n", (int)depth);
            g += "__constant__ int qss_gen_cols[] = {";
            for (int w = 0; w < nw; ++w) for (size_t d = 0; d < depth; ++d) P("%d, ", d < bin[w].size() ? bin[w][d] : -1);
            g += "-1};\n";
        }
        // ---- P4 specialised: the closure solve of every group with its matrix in REGISTERS (the interpreter walks it through
        //      shared memory: a chain of dependent ~30-cycle reads on one warp per group).  Same operations in the same order
        //      as the interpreter (subtraction-free elimination, U = P / D for the dy/dx solves, forward substitution).
        {
            g += "__device__ __forceinline__ void qss_gen_closure(const int warp, const unsigned sml) {\n";
            std::vector<std::vector<int>> by_level(c.n_levels);
            for (int gi = 0; gi < c.n_groups; ++gi) by_level[(*c.lvl_of_group)[gi]].push_back(gi);
            for (int l = 0; l < c.n_levels; ++l) {
                g += "    switch (warp) {\n";
                std::vector<std::vector<int>> bw(nw);
                for (size_t i = 0; i < by_level[l].size(); ++i) bw[i % nw].push_back(by_level[l][i]);
                for (int w = 0; w < nw; ++w) {
                    if (bw[w].empty()) continue;
                    P("    case %d: {\n", w);
                    for (int gi : bw[w]) {
                        const std::vector<int> &mem = (*c.members)[gi];
                        const int sz = (int)mem.size(), base = v.s_CL + (*c.gbase)[gi];
                        const int oL = base + sz * sz, oP0 = oL + sz, oID = oP0 + sz;
                        g += "        {\n";
                        for (int m = 0; m < sz; ++m) for (int j = 0; j < sz; ++j) if (m != j) P("            double a%d_%d = lS<%d>(sml);\n", m, j, (base + m * sz + j) * 256);
                        for (int k = 0; k < sz; ++k) P("            double L%d = lS<%d>(sml), q%d = lS<%d>(sml), d%d;\n", k, (oL + k) * 256, k, (oP0 + k) * 256, k);
                        for (int x = (*c.xp_begin)[gi]; x < (*c.xp_end)[gi]; ++x)
                            P("            q%d += lS<%d>(sml) * lS<%d>(sml);\n", (*c.pos_in_grp)[(*c.xpl)[x].first.first], (v.s_XP + x) * 256, voff(N + 1 + (*c.xpl)[x].first.second));
                        for (int k = sz - 1; k >= 1; --k) {
                            P("            {   const double lk = L%d;\n                double Dk = lk;\n", k);
                            for (int m = 0; m < k; ++m) P("                Dk += a%d_%d;\n", m, k);
                            P("                const double iD = qss_rcp(Dk);\n                d%d = iD;\n", k);
                            for (int jj = 0; jj < k; ++jj) {
                                P("                {   const double f = a%d_%d * iD;\n                    L%d += f * lk;\n", k, jj, jj);
                                for (int m = 0; m < k; ++m) if (m != jj) P("                    a%d_%d += a%d_%d * f;\n", m, jj, m, k);
                                g += "                }\n";
                            }
                            g += "            }\n";
                        }
                        g += "            d0 = qss_rcp(L0);\n";
                        for (int k = sz - 1; k >= 1; --k) {
                            P("            {   const double iD = d%d, tk = q%d * iD;\n", k, k);
                            for (int m = 0; m < k; ++m) P("                {   const double pmk = a%d_%d; a%d_%d = pmk * iD; q%d += pmk * tk; }\n", m, k, m, k, m);
                            g += "            }\n";
                        }
                        for (int k = 0; k < sz; ++k) {
                            P("            {   double acc = q%d;\n", k);
                            for (int jj = 0; jj < k; ++jj) P("                acc += a%d_%d * q%d;\n", k, jj, jj);
                            P("                acc *= d%d;\n                q%d = acc;\n                sS<%d>(sml, acc);\n            }\n", k, k, voff(N + 1 + mem[k]));
                        }
                        for (int m = 0; m < sz; ++m) for (int j = 0; j < sz; ++j) if (m != j) P("            sS<%d>(sml, a%d_%d);\n", (base + m * sz + j) * 256, m, j);
                        for (int k = 0; k < sz; ++k) P("            sS<%d>(sml, d%d);\n", (oID + k) * 256, k);
                        g += "        }\n";
                    }
                    g += "    } break;\n";
                }
                g += "    default: break;\n    }\n    __syncthreads();\n";
            }
            g += "}\n";
        }
        // ---- P3 + P7 specialised: every closure slot, cross-group coupling and W_y entry is a signed sum of kappas (8-10
        //      interpreter instructions per term, a dependent table -> kappa -> add chain); as straight-line code it is one
        //      shared-memory read and one add per term (45 KB for cfg2: 8x fewer instructions, which pays for the instruction fetch)
        {
            struct Ent { std::string dst; std::vector<std::pair<int, int>> terms; };     // (byte offset of kappa, sign)
            std::vector<Ent> ents;
            for (auto &kv : *c.ce) {
                Ent e; std::snprintf(b, sizeof b, "sS<%d>(sml, ", (v.s_CL + kv.first) * 256); e.dst = b;
                for (int d : kv.second) e.terms.push_back({(v.s_KAP + d) * 256, 1});
                ents.push_back(e);
            }
            for (size_t x = 0; x < c.xpl->size(); ++x) {
                Ent e; std::snprintf(b, sizeof b, "sS<%d>(sml, ", (v.s_XP + (int)x) * 256); e.dst = b;
                for (int d : (*c.xpl)[x].second) e.terms.push_back({(v.s_KAP + d) * 256, 1});
                ents.push_back(e);
            }
            if (by_dir) {
                for (size_t r = 0; r < gdir.size(); ++r) {       // kappa_d of the QSS-consuming directions -> scratch (kappa is overwritten by P5)
                    Ent e; std::snprintf(b, sizeof b, "sG<%d>(sc, ", (v.g_WY + (int)r) * 256); e.dst = b;
                    e.terms.push_back({(v.s_KAP + gdir[r].d) * 256, 1});
                    ents.push_back(e);
                }
            } else {
                int eidx = 0;
                for (auto &kv : wy) {
                    Ent e; std::snprintf(b, sizeof b, "sG<%d>(sc, ", (v.g_WY + eidx) * 256); e.dst = b; ++eidx;
                    for (int32_t w : kv.second) e.terms.push_back({v.s_KAP * 256 + (int)(w & 0x7fffffff), w < 0 ? -1 : 1});
                    ents.push_back(e);
                }
            }
            std::vector<int> idx(ents.size());
            for (size_t i = 0; i < ents.size(); ++i) idx[i] = (int)i;
            std::stable_sort(idx.begin(), idx.end(), [&](int a, int c2) { return ents[a].terms.size() > ents[c2].terms.size(); });
            std::vector<std::vector<int>> bin(nw);
            std::vector<double> load(nw, 0.0);
            for (int i : idx) { const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin()); bin[w].push_back(i); load[w] += 2.0 + ents[i].terms.size(); }
            g += "__device__ __forceinline__ void qss_gen_gather(const int warp, const unsigned sml, double *sc) {\n    switch (warp) {\n";
            for (int w = 0; w < nw; ++w) {
                P("    case %d:\n", w);
                for (int i : bin[w]) {
                    g += "        " + ents[i].dst;
                    if (ents[i].terms.empty()) g += "0.0";
                    for (size_t t = 0; t < ents[i].terms.size(); ++t) {
                        const auto &tm = ents[i].terms[t];
                        P("%slS<%d>(sml)", t == 0 ? (tm.second < 0 ? "-" : "") : (tm.second < 0 ? " - " : " + "), tm.first);
                    }
                    g += ");\n";
                }
                g += "        break;\n";
            }
            g += "    default: break;\n    }\n}\n";
        }
    }
    return true;
}

}  // namespace

int qss_compile(const qss_mech_desc_t *d, QssCompiled &out, std::string &err) {
    if (!d) { err = "desc is NULL"; return QSS_E_INVALID; }
    const int N = d->n_nqss, Nq = d->n_qss, M = d->n_reac, nsp = N + Nq;
    if (N < 1 || Nq < 0 || M < 0) { err = "n_nqss must be >= 1, n_qss and n_reac >= 0"; return QSS_E_INVALID; }
    if (!d->nasa_T || !d->nasa_lo || !d->nasa_hi) { err = "NASA-7 tables are NULL"; return QSS_E_INVALID; }
    if (M > 0 && (!d->type || !d->dir_mask || !d->reac_ptr || !d->prod_ptr || !d->arr)) {
        err = "reaction arrays are NULL"; return QSS_E_INVALID;
    }
    // ---------------------------------------------------------------- reactions: parse + validate
    std::vector<Reaction> R(M);
    int n_tb = 0;
    for (int j = 0; j < M; ++j) {
        Reaction &r = R[j];
        r.type = d->type[j]; r.mask = d->dir_mask[j] & 3;
        if (r.type < 0 || r.type > 2) { err = fmt("reaction %d: unsupported type %d", j, r.type); return QSS_E_UNSUPPORTED; }
        if (r.type == 2 && (!d->arr_low || !d->troe)) { err = fmt("reaction %d: fall-off without arr_low/troe", j); return QSS_E_INVALID; }
        r.tb = r.type >= 1 ? n_tb++ : -1;
        const int32_t *ptr[2] = {d->reac_ptr, d->prod_ptr}, *sp[2] = {d->reac_sp, d->prod_sp}, *nu[2] = {d->reac_nu, d->prod_nu};
        std::map<int, int> net;
        r.dnu = 0;
        for (int s = 0; s < 2; ++s) {
            if (ptr[s][j + 1] < ptr[s][j]) { err = fmt("reaction %d: CSR pointers decrease", j); return QSS_E_INVALID; }
            int nq = 0;
            r.q[s] = -1;
            for (int p = ptr[s][j]; p < ptr[s][j + 1]; ++p) {
                if (!sp[s] || !nu[s]) { err = "species CSR arrays are NULL"; return QSS_E_INVALID; }
                Term t{sp[s][p], nu[s][p]};
                if (t.sp < 0 || t.sp >= nsp) { err = fmt("reaction %d: species index %d out of range", j, t.sp); return QSS_E_INVALID; }
                if (t.nu < 1) { err = fmt("reaction %d: stoichiometric coefficient %d < 1", j, t.nu); return QSS_E_UNSUPPORTED; }
                for (const Term &o : r.side[s]) if (o.sp == t.sp) { err = fmt("reaction %d: species %d listed twice on one side", j, t.sp); return QSS_E_INVALID; }
                r.side[s].push_back(t);
                net[t.sp] += s == 0 ? -t.nu : t.nu;
                r.dnu += s == 0 ? -t.nu : t.nu;
                if (t.sp >= N) { nq += t.nu; r.q[s] = t.sp - N; }
            }
            if (nq > 1) {
                // side s is consumed by direction s and produced by direction 1-s
                if (r.mask & (1 << s)) { err = fmt("reaction %d: an enabled direction consumes %d QSS molecules (quadratic coupling)", j, nq); return QSS_E_QUADRATIC; }
                if (r.mask & (1 << (1 - s))) { err = fmt("reaction %d: an enabled direction produces %d QSS molecules", j, nq); return QSS_E_QSS_FANOUT; }
            }
        }
        for (auto &kv : net) if (kv.second != 0) r.net.push_back({kv.first, kv.second});
        if (d->eff_ptr && (d->eff_ptr[j + 1] < d->eff_ptr[j] || d->eff_ptr[j] < 0)) { err = fmt("reaction %d: efficiency CSR pointers decrease", j); return QSS_E_INVALID; }
        if (r.type >= 1 && d->eff_ptr) {
            if (d->eff_ptr[j + 1] > d->eff_ptr[j] && (!d->eff_sp || !d->eff_val)) { err = "efficiency arrays are NULL"; return QSS_E_INVALID; }
            for (int p = d->eff_ptr[j]; p < d->eff_ptr[j + 1]; ++p) {
                if (d->eff_sp[p] < 0 || d->eff_sp[p] >= N) { err = fmt("reaction %d: third-body efficiency on species %d (must be transported)", j, d->eff_sp[p]); return QSS_E_INVALID; }
                if (!std::isfinite(d->eff_val[p])) { err = fmt("reaction %d: non-finite third-body efficiency", j); return QSS_E_INVALID; }
                for (int q = d->eff_ptr[j]; q < p; ++q)
                    if (d->eff_sp[q] == d->eff_sp[p]) { err = fmt("reaction %d: third-body efficiency of species %d given twice", j, d->eff_sp[p]); return QSS_E_INVALID; }
            }
        }
        if (r.type == 2) {
            // fall-off parameters: alpha finite, T*** and T* positive (CHEMKIN placeholders such as 1e-30 / 1e30 are fine: the
            // kernels saturate the exponentials), T** finite
            const double *tp = d->troe + 4 * j;
            if (!std::isfinite(tp[0]) || !(tp[1] > 0.0) || !(tp[2] > 0.0) || !std::isfinite(tp[1]) || !std::isfinite(tp[2]) || !std::isfinite(tp[3])) {
                err = fmt("reaction %d: Troe parameters need finite alpha and T**, and finite positive T***, T*", j); return QSS_E_INVALID;
            }
        }
    }
    if (d->strict_balance) {                 // optional strict mode (SURVEY.md 8(b) "Errors"): every reaction conserves every element
        if (!d->comp || d->n_elem < 1) { err = "strict_balance needs the element compositions (comp, n_elem)"; return QSS_E_INVALID; }
        for (int j = 0; j < M; ++j) for (int e = 0; e < d->n_elem; ++e) {
            long bal = 0;
            for (const Term &x : R[j].net) bal += (long)x.nu * d->comp[(size_t)x.sp * d->n_elem + e];
            if (bal != 0) { err = fmt("reaction %d does not conserve element %d (imbalance %d)", j, e, (int)bal); return QSS_E_UNBALANCED; }
        }
    }
    auto enabled = [&](int j, int dir) { return (R[j].mask >> dir) & 1; };

    // ---------------------------------------------------------------- QSS digraph, SCCs, levels
    // edge n -> m iff an enabled direction consumes QSS n and produces QSS m != n
    std::vector<std::vector<int>> adj(Nq);
    std::vector<char> has_leak(Nq, 0);
    for (int j = 0; j < M; ++j)
        for (int dir = 0; dir < 2; ++dir) {
            if (!enabled(j, dir)) continue;
            int n = R[j].q[dir], m = R[j].q[1 - dir];
            if (n < 0) continue;
            if (m >= 0 && m != n) adj[n].push_back(m);
            else if (m < 0) has_leak[n] = 1;
        }
    for (auto &a : adj) { std::sort(a.begin(), a.end()); a.erase(std::unique(a.begin(), a.end()), a.end()); }
    // every QSS species must reach a leak, else the closure matrix is structurally singular
    {
        std::vector<std::vector<int>> radj(Nq);
        for (int n = 0; n < Nq; ++n) for (int m : adj[n]) radj[m].push_back(n);
        std::vector<char> ok(has_leak);
        std::vector<int> st;
        for (int n = 0; n < Nq; ++n) if (ok[n]) st.push_back(n);
        while (!st.empty()) { int v = st.back(); st.pop_back(); for (int u : radj[v]) if (!ok[u]) { ok[u] = 1; st.push_back(u); } }
        for (int n = 0; n < Nq; ++n) if (!ok[n]) { err = fmt("QSS species %d (index %d) has no path to a transported species", n, N + n); return QSS_E_NO_SINK; }
    }
    std::vector<int> comp;
    const int ncomp = tarjan(Nq, adj, comp);
    // level of a component = longest chain of components feeding it (its sources must be solved first)
    std::vector<int> level(ncomp, 0);
    // Tarjan numbers components in reverse topological order: comp id larger => earlier in the DAG.
    for (int c = ncomp - 1; c >= 0; --c)
        for (int n = 0; n < Nq; ++n) if (comp[n] == c)
            for (int m : adj[n]) if (comp[m] != c) level[comp[m]] = std::max(level[comp[m]], level[c] + 1);
    std::vector<int> gorder(ncomp);
    for (int c = 0; c < ncomp; ++c) gorder[c] = c;
    std::stable_sort(gorder.begin(), gorder.end(), [&](int a, int b) {
        if (level[a] != level[b]) return level[a] < level[b];
        return a > b;
    });
    std::vector<int> gid(ncomp);             // component -> group number in solve order
    for (int g = 0; g < ncomp; ++g) gid[gorder[g]] = g;
    const int n_groups = ncomp;
    int n_levels = 0;
    for (int c = 0; c < ncomp; ++c) n_levels = std::max(n_levels, level[c] + 1);
    std::vector<std::vector<int>> members(n_groups);
    for (int n = 0; n < Nq; ++n) members[gid[comp[n]]].push_back(n);     // natural order inside a group
    std::vector<int> grp_of_q(Nq), pos_in_grp(Nq);
    int max_group = 0;
    for (int g = 0; g < n_groups; ++g) {
        max_group = std::max(max_group, (int)members[g].size());
        for (size_t p = 0; p < members[g].size(); ++p) { grp_of_q[members[g][p]] = g; pos_in_grp[members[g][p]] = (int)p; }
    }

    // ---------------------------------------------------------------- closure storage + gather lists
    // per group of size g: P[g*g] (P[m*g+n] = production of m from n), leak[g], p0[g], invD[g]
    std::vector<int> gbase(n_groups);
    int cl_size = 0;
    for (int g = 0; g < n_groups; ++g) { int sz = (int)members[g].size(); gbase[g] = cl_size; cl_size += sz * sz + 3 * sz; }
    std::map<int, std::vector<int>> ce;                    // closure slot -> directions
    std::map<std::pair<int, int>, std::vector<int>> xp;    // (m, n) cross-group -> directions
    for (int j = 0; j < M; ++j)
        for (int dir = 0; dir < 2; ++dir) {
            if (!enabled(j, dir)) continue;
            const int n = R[j].q[dir], m = R[j].q[1 - dir], dd = 2 * j + dir;
            if (n >= 0) {
                const int g = grp_of_q[n], sz = (int)members[g].size();
                if (m >= 0 && m != n && grp_of_q[m] == g) ce[gbase[g] + pos_in_grp[m] * sz + pos_in_grp[n]].push_back(dd);
                else if (m >= 0 && m != n) { ce[gbase[g] + sz * sz + pos_in_grp[n]].push_back(dd); xp[{m, n}].push_back(dd); }
                else if (m < 0) ce[gbase[g] + sz * sz + pos_in_grp[n]].push_back(dd);
            } else if (m >= 0) {
                const int g = grp_of_q[m], sz = (int)members[g].size();
                ce[gbase[g] + sz * sz + sz + pos_in_grp[m]].push_back(dd);
            }
        }
    for (int g = 0; g < n_groups; ++g) {                    // every P / leak / p0 slot is written, even when no direction feeds it
        const int sz = (int)members[g].size();
        for (int o = 0; o < sz * sz + 2 * sz; ++o) ce[gbase[g] + o];
    }
    // cross entries sorted by the group of their target m
    std::vector<std::pair<std::pair<int, int>, std::vector<int>>> xpl(xp.begin(), xp.end());
    std::stable_sort(xpl.begin(), xpl.end(), [&](const auto &a, const auto &b) { return grp_of_q[a.first.first] < grp_of_q[b.first.first]; });
    std::vector<int> xp_begin(n_groups, 0), xp_end(n_groups, 0);
    for (int g = 0, p = 0; g < n_groups; ++g) {
        xp_begin[g] = p;
        while (p < (int)xpl.size() && grp_of_q[xpl[p].first.first] == g) ++p;
        xp_end[g] = p;
    }

    // ---------------------------------------------------------------- blobs
    std::vector<int32_t> &I = out.I; std::vector<double> &D = out.D;
    I.clear(); D.clear();
    QssTab &t = out.tab;
    t = QssTab();
    t.N = N; t.Nq = Nq; t.M = M; t.nsp = nsp; t.n_tb = n_tb;
    t.n_groups = n_groups; t.n_levels = n_levels; t.max_group = max_group; t.cl_size = cl_size;
    auto atI = [&]() { return (int32_t)I.size(); };
    auto atD = [&]() { return (int32_t)D.size(); };

    // thermo (NASA-7; the h and s polynomials pre-divided as in the definition, reading G4)
    t.d_thermo = atD();
    for (int s = 0; s < nsp; ++s) {
        double rec[QSS_TH_STRIDE] = {0};
        rec[0] = d->nasa_T[3 * s + 1];
        for (int rg = 0; rg < 2; ++rg) {
            const double *a = (rg == 0 ? d->nasa_lo : d->nasa_hi) + 7 * s;
            double *o = rec + 1 + 11 * rg;
            o[0] = a[0]; o[1] = a[1] / 2.0; o[2] = a[2] / 3.0; o[3] = a[3] / 4.0; o[4] = a[4] / 5.0; o[5] = a[5];
            o[6] = a[1]; o[7] = a[2] / 2.0; o[8] = a[3] / 3.0; o[9] = a[4] / 4.0; o[10] = a[6];
        }
        D.insert(D.end(), rec, rec + QSS_TH_STRIDE);
    }
    const double RGAS = 8.31446261815324;
    t.d_rate = atD();
    for (int j = 0; j < M; ++j) {
        double rec[QSS_RD_STRIDE] = {0};
        const double A = d->arr[3 * j];
        if (!(A > 0)) { err = fmt("reaction %d: pre-exponential factor must be > 0", j); return QSS_E_INVALID; }
        rec[0] = std::log(A); rec[1] = d->arr[3 * j + 1]; rec[2] = d->arr[3 * j + 2] / RGAS;
        if (R[j].type == 2) {
            const double A0 = d->arr_low[3 * j];
            if (!(A0 > 0)) { err = fmt("reaction %d: low-pressure pre-exponential factor must be > 0", j); return QSS_E_INVALID; }
            rec[3] = std::log(A0); rec[4] = d->arr_low[3 * j + 1]; rec[5] = d->arr_low[3 * j + 2] / RGAS;
            rec[6] = d->troe[4 * j]; rec[7] = 1.0 / d->troe[4 * j + 1]; rec[8] = 1.0 / d->troe[4 * j + 2]; rec[9] = d->troe[4 * j + 3];
        }
        rec[10] = (double)R[j].dnu;
        D.insert(D.end(), rec, rec + QSS_RD_STRIDE);
    }
    // reaction order: fall-off first, then third-body, then Arrhenius (balances the warps of a block)
    std::vector<int> rorder(M);
    for (int j = 0; j < M; ++j) rorder[j] = j;
    std::stable_sort(rorder.begin(), rorder.end(), [&](int a, int b) { return R[a].type > R[b].type; });
    t.i_reac = atI();
    for (int j = 0; j < M; ++j) {
        int32_t rec[QSS_RI_STRIDE] = {R[j].type, R[j].mask, R[j].tb, R[j].q[0], R[j].q[1], 0, 0, 0};
        I.insert(I.end(), rec, rec + QSS_RI_STRIDE);
    }
    t.i_rorder = atI(); I.insert(I.end(), rorder.begin(), rorder.end());
    // direction reactant lists
    {
        std::vector<int32_t> ptr{0}, sp, nu;
        for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
            for (const Term &x : R[j].side[dir]) { sp.push_back(x.sp); nu.push_back(x.nu); }
            ptr.push_back((int32_t)sp.size());
        }
        t.i_side_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_side_sp = atI(); I.insert(I.end(), sp.begin(), sp.end());
        t.i_side_nu = atI(); I.insert(I.end(), nu.begin(), nu.end());
    }
    {   // net stoichiometry by reaction
        std::vector<int32_t> ptr{0}, sp, nu;
        for (int j = 0; j < M; ++j) { for (const Term &x : R[j].net) { sp.push_back(x.sp); nu.push_back(x.nu); } ptr.push_back((int32_t)sp.size()); }
        t.i_net_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_net_sp = atI(); I.insert(I.end(), sp.begin(), sp.end());
        t.i_net_nu = atI(); I.insert(I.end(), nu.begin(), nu.end());
    }
    std::vector<std::vector<std::pair<int, double>>> effc(N);
    {   // efficiencies by reaction
        std::vector<int32_t> ptr{0}, sp; std::vector<double> val;
        for (int j = 0; j < M; ++j) {
            if (R[j].type >= 1 && d->eff_ptr)
                for (int p = d->eff_ptr[j]; p < d->eff_ptr[j + 1]; ++p) {
                    sp.push_back(d->eff_sp[p]); val.push_back(d->eff_val[p] - 1.0);
                    effc[d->eff_sp[p]].push_back({j, d->eff_val[p] - 1.0});
                }
            ptr.push_back((int32_t)sp.size());
        }
        t.i_eff_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_eff_sp = atI(); I.insert(I.end(), sp.begin(), sp.end());
        t.d_effm1 = atD(); D.insert(D.end(), val.begin(), val.end());
    }
    {   // efficiencies by column
        std::vector<int32_t> ptr{0}, rj; std::vector<double> val;
        for (int k = 0; k < N; ++k) { for (auto &e : effc[k]) { rj.push_back(e.first); val.push_back(e.second); } ptr.push_back((int32_t)rj.size()); }
        t.i_effc_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_effc_reac = atI(); I.insert(I.end(), rj.begin(), rj.end());
        t.d_effc = atD(); D.insert(D.end(), val.begin(), val.end());
    }
    // groups
    std::vector<int> lvl_of_group(n_groups);
    for (int c = 0; c < ncomp; ++c) lvl_of_group[gid[c]] = level[c];
    {
        t.i_group = atI();
        int moff = 0;
        for (int g = 0; g < n_groups; ++g) {
            int32_t rec[QSS_GI_STRIDE] = {(int32_t)members[g].size(), moff, gbase[g], lvl_of_group[g], xp_begin[g], xp_end[g], 0, 0};
            I.insert(I.end(), rec, rec + QSS_GI_STRIDE);
            moff += (int)members[g].size();
        }
        t.i_gmember = atI();
        for (int g = 0; g < n_groups; ++g) I.insert(I.end(), members[g].begin(), members[g].end());
        std::vector<int32_t> lp(n_levels + 1, 0);
        for (int g = 0; g < n_groups; ++g) lp[lvl_of_group[g] + 1]++;
        for (int l = 0; l < n_levels; ++l) lp[l + 1] += lp[l];
        t.i_level_ptr = atI(); I.insert(I.end(), lp.begin(), lp.end());
        out.order.clear(); out.group_of.clear(); out.group_size.clear();
        for (int g = 0; g < n_groups; ++g) {
            out.group_size.push_back((int)members[g].size());
            for (int q : members[g]) { out.order.push_back(q); out.group_of.push_back(g); }
        }
    }
    {   // closure gather entries
        std::vector<int32_t> ptr{0}, dst, dir;
        for (auto &kv : ce) { dst.push_back(kv.first); dir.insert(dir.end(), kv.second.begin(), kv.second.end()); ptr.push_back((int32_t)dir.size()); }
        t.n_centry = (int32_t)dst.size();
        t.i_ce_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_ce_dst = atI(); I.insert(I.end(), dst.begin(), dst.end());
        t.i_ce_dir = atI(); I.insert(I.end(), dir.begin(), dir.end());
    }
    {   // cross-group couplings
        std::vector<int32_t> ptr{0}, dir, xm, xn;
        for (auto &e : xpl) {
            xm.push_back(pos_in_grp[e.first.first]); xn.push_back(e.first.second);
            dir.insert(dir.end(), e.second.begin(), e.second.end()); ptr.push_back((int32_t)dir.size());
        }
        t.n_xp = (int32_t)xm.size();
        t.i_xp_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_xp_dir = atI(); I.insert(I.end(), dir.begin(), dir.end());
        t.i_xp_m = atI(); I.insert(I.end(), xm.begin(), xm.end());
        t.i_xp_n = atI(); I.insert(I.end(), xn.begin(), xn.end());
    }
    size_t n_inc = 0;
    {   // species incidence
        std::vector<std::vector<Term>> inc(nsp);     // (reaction, nu_net)
        for (int j = 0; j < M; ++j) if (R[j].mask) for (const Term &x : R[j].net) inc[x.sp].push_back({j, x.nu});
        std::vector<int32_t> ptr{0}, rj, nu;
        for (int s = 0; s < nsp; ++s) { for (const Term &x : inc[s]) { rj.push_back(x.sp); nu.push_back(x.nu); } ptr.push_back((int32_t)rj.size()); }
        n_inc = rj.size();
        t.i_sp_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_sp_reac = atI(); I.insert(I.end(), rj.begin(), rj.end());
        t.i_sp_nu = atI(); I.insert(I.end(), nu.begin(), nu.end());
    }
    size_t n_wy_terms = 0;
    {   // W_y[i][q] = sum over directions consuming q of (+-) nu_net(i) kappa_d
        std::map<std::pair<int, int>, std::vector<std::pair<int, int>>> wy;
        for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
            if (!enabled(j, dir) || R[j].q[dir] < 0) continue;
            for (const Term &x : R[j].net) if (x.sp < N) wy[{x.sp, R[j].q[dir]}].push_back({2 * j + dir, dir == 0 ? x.nu : -x.nu});
        }
        std::vector<int32_t> ptr{0}, dir, coef, rptr{0}, rq, re;
        int e = 0, row = 0;
        for (auto &kv : wy) {
            while (row < kv.first.first) { rptr.push_back((int32_t)rq.size()); ++row; }
            rq.push_back(kv.first.second); re.push_back(e++);
            for (auto &dc : kv.second) { dir.push_back(dc.first); coef.push_back(dc.second); }
            ptr.push_back((int32_t)dir.size());
        }
        while (row < N) { rptr.push_back((int32_t)rq.size()); ++row; }
        n_wy_terms = dir.size();
        t.n_wy = e;
        t.i_wy_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_wy_dir = atI(); I.insert(I.end(), dir.begin(), dir.end());
        t.i_wy_coef = atI(); I.insert(I.end(), coef.begin(), coef.end());
        t.i_wyrow_ptr = atI(); I.insert(I.end(), rptr.begin(), rptr.end());
        t.i_wyrow_q = atI(); I.insert(I.end(), rq.begin(), rq.end());
        t.i_wyrow_e = atI(); I.insert(I.end(), re.begin(), re.end());
    }
    size_t n_colinc = 0, n_scatter = 0;
    {   // Jacobian column incidences
        std::vector<std::vector<std::pair<int, int>>> col(N);
        for (int j = 0; j < M; ++j) for (int dir = 0; dir < 2; ++dir) {
            if (!enabled(j, dir)) continue;
            for (size_t p = 0; p < R[j].side[dir].size(); ++p)
                if (R[j].side[dir][p].sp < N) { col[R[j].side[dir][p].sp].push_back({2 * j + dir, (int)p}); n_scatter += R[j].net.size(); }
        }
        std::vector<int32_t> ptr{0}, dir, pos;
        for (int k = 0; k < N; ++k) { for (auto &x : col[k]) { dir.push_back(x.first); pos.push_back(x.second); } ptr.push_back((int32_t)dir.size()); }
        n_colinc = dir.size();
        t.i_col_ptr = atI(); I.insert(I.end(), ptr.begin(), ptr.end());
        t.i_col_dir = atI(); I.insert(I.end(), dir.begin(), dir.end());
        t.i_col_pos = atI(); I.insert(I.end(), pos.begin(), pos.end());
    }
    // ---------------------------------------------------------------- per-cell workspace layout (doubles)
    {
        int o = 0;
        auto take = [&](int n) { int r = o; o += n; return r; };
        t.w_G = take(nsp); t.w_H = take(nsp); t.w_K = take(2 * M); t.w_KAP = take(2 * M);
        t.w_MM = take(n_tb); t.w_CL = take(cl_size); t.w_XP = take(t.n_xp); t.w_Y = take(Nq); t.w_Q = take(M);
        t.ws_wdot = o;
        t.w_DF = take(M); t.w_DC = take(M); t.w_DLM = take(n_tb);
        t.w_QT = take(M); t.w_QM = take(n_tb); t.w_ET = take(nsp); t.w_TV = take(nsp); t.w_WY = take(t.n_wy);
        t.w_COL = o; t.ws_jac_base = o;
    }
    // ---------------------------------------------------------------- algorithmic cost
    {
        const double EXP = 18, LOG = 30, DIV = 24, RCP = 22;
        double s = 0;
        s += LOG + RCP + 6 + N;                                   // lnT, 1/T, powers of T, ln(P0/RT), Ctot
        s += nsp * 13.0;                                          // NASA-7 h and g
        size_t n_eff = 0, n_side = 0, n_net = 0;
        int n_troe = 0, n_rev = 0;
        for (int j = 0; j < M; ++j) {
            n_side += R[j].side[0].size() + R[j].side[1].size(); n_net += R[j].net.size();
            if (R[j].type == 2) ++n_troe;
            if (R[j].mask & 2) ++n_rev;
            if (R[j].type >= 1 && d->eff_ptr) n_eff += d->eff_ptr[j + 1] - d->eff_ptr[j];
        }
        s += M * (2.0 + EXP);                                     // Arrhenius
        s += n_rev * (EXP + 2.0) + (double)n_side;                // Kc: sum nu g, dnu ln(P0/RT), exp, multiply
        s += (double)n_eff + n_tb;                                // third-body concentrations
        s += n_troe * (2.0 + EXP + 3 * EXP + 4 + 2 * LOG + 12 + 2 * DIV + EXP + DIV + 3);   // k0, Fcent, F, Pr/(1+Pr)
        s += (double)n_side + 2.0 * M;                            // kappa_d products, r_d
        for (auto &kv : ce) s += kv.second.size();                // closure assembly
        for (auto &e : xpl) s += e.second.size() + 1;
        for (int g = 0; g < n_groups; ++g) { double sz = (double)members[g].size(); s += sz * sz * sz / 3.0 + 2 * sz * sz + sz * RCP; }
        s += M + (double)n_inc;                                   // Q_j and wdot_i
        out.slots_wdot = s;
        double jx = 0;
        jx += nsp * 6.0 + M * 4.0 + n_rev * ((double)n_side / std::max(M, 1) + 3.0);   // h/RT sums, dlnk/dT, dlnKc/dT
        jx += n_troe * (40.0 + 3 * DIV);                          // fall-off derivatives
        jx += 3.0 * M + 2.0 * n_inc;                              // QT, QM, ET, t vectors
        jx += (double)n_wy_terms;                                 // W_y assembly
        jx += 3.0 * n_colinc + (double)n_scatter;                 // partials (product of others) + scatter
        for (int k = 0; k < N; ++k) for (auto &e : effc[k]) jx += 1.0 + R[e.first].net.size();   // (alpha-1) corrections
        jx += (double)nsp * N;                                    // rank-1 third-body term added to every species column
        double sg2 = 0;
        for (int g = 0; g < n_groups; ++g) sg2 += (double)members[g].size() * members[g].size();
        jx += (sg2 + Nq + t.n_xp) * (N + 1);                      // Y_x solves
        jx += (double)t.n_wy * (N + 1);                           // W_y * Y_x
        out.slots_jac = s + jx;
        out.bytes_wdot = 8.0 * (N + 1) + 8.0 * N;
        out.bytes_jac = 8.0 * (N + 1) + 8.0 * N * (N + 1);
    }
    {
        V1Ctx vc{N, Nq, M, nsp, n_tb, n_groups, n_levels, cl_size, &R, &members, &gbase, &xp_begin, &xp_end, &lvl_of_group,
                 &pos_in_grp, &rorder, &ce, &xpl, &effc, d};
        out.v1_ok = build_v1(vc, out, out.v1_why);
        out.v3_ok = build_v3(vc, out, out.v3_why);
        if (const char *dump = qss_devenv("QSS_GEN_DUMP")) {            // debugging aid: the generated source (variant 3, else variant 2)
            const std::string &g = out.v3_ok ? out.v3.gen : out.v1_gen;
            if (FILE *f = std::fopen(dump, "w")) { std::fwrite(g.data(), 1, g.size(), f); std::fclose(f); }
        }
        if (qss_devenv("QSS_DEBUG")) std::fprintf(stderr, "[qss] variant 3: %s%s\n", out.v3_ok ? "ok" : "not applicable: ", out.v3_ok ? "" : out.v3_why.c_str());
        if (qss_devenv("QSS_DEBUG"))
            std::fprintf(stderr, "[qss] variant 1: %s%s (hot table %d/%d words, smem rows %d, scratch rows %d, rounds %d, solve ops %d)\n",
                         out.v1_ok ? "ok" : "not applicable: ", out.v1_ok ? "" : out.v1_why.c_str(), out.v1.h_used, QSS_V1_HMAX,
                         out.v1.smem_rows, out.v1.scratch_rows, out.v1.n_rounds, out.v1.n_sp_ops);
    }
    err.clear();
    return QSS_OK;
}
