// Internal: the parsed mechanism and its QSS closure structure, as the host compiler (qss_compile.cpp) hands them to the
// kernel-variant builders (build_v1 in qss_compile.cpp, build_v3 in qss_gen3.cpp).  Not part of the public ABI.
#ifndef QSS_CTX_H
#define QSS_CTX_H
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "../../include/qss.h"

struct QssCompiled;

namespace qssc {

struct Term { int sp, nu; };

struct Reaction {
    int type, mask;
    std::vector<Term> side[2];     // side[0] reactants, side[1] products (as given)
    std::vector<Term> net;         // nu'' - nu', non-zero only
    int q[2];                      // local QSS index consumed by direction 0 / 1, or -1
    int dnu;
    int tb;                        // index among third-body / fall-off reactions, or -1
};

struct V1Ctx {
    int N, Nq, M, nsp, n_tb, n_groups, n_levels, cl_size;
    const std::vector<Reaction> *R;
    const std::vector<std::vector<int>> *members;       // [group] local QSS indices in solve order
    const std::vector<int> *gbase, *xp_begin, *xp_end, *lvl_of_group, *pos_in_grp, *rorder;
    const std::map<int, std::vector<int>> *ce;          // closure slot -> directions feeding it
    const std::vector<std::pair<std::pair<int, int>, std::vector<int>>> *xpl;    // cross-group couplings (m, n) -> directions
    const std::vector<std::vector<std::pair<int, double>>> *effc;                // [species k] (reaction, alpha - 1)
    const qss_mech_desc_t *desc;                        // the caller's description (thermo and rate parameters)
};

// Kernel variant 3 (qss_gen3.cpp): fills out.v3 and returns true when the mechanism fits it.
bool build_v3(const V1Ctx &c, QssCompiled &out, std::string &why);

}  // namespace qssc

#endif
