// Internal: host-side mechanism compiler interface (qss_compile.cpp -> qss_api.cu).
#ifndef QSS_COMPILE_H
#define QSS_COMPILE_H
#include <string>
#include <vector>

#include "../../include/qss.h"
#include "qss_tables.h"
#include "qss_v1.h"
#include "qss_v3.h"

// Host side of kernel variant 3 (qss_gen3.cpp): the generated header, the parameter blobs of the reaction-per-lane
// phases and the launch geometry.
struct QssV3Host {
    std::string gen;               // text of qss_gen3.h for this mechanism
    std::vector<double> dP;        // [QSS3_NDP][n_slot]
    std::vector<int32_t> iP;       // [QSS3_NIP][n_slot]
    int nw = 0, smem_bytes = 0, scratch_rows = 0, n_slot = 0, n_pp = 0, n_kq = 0, n_groups = 0;
};

struct QssCompiled {
    QssTab tab;                    // offsets filled in; I / D pointers are set after upload
    std::vector<int32_t> I;        // host image of the int blob
    std::vector<double> D;         // host image of the double blob
    std::vector<int32_t> order;    // [Nq] local QSS index solved i-th
    std::vector<int32_t> group_of; // [Nq] group (in solve order) of order[i]
    std::vector<int32_t> group_size;
    double slots_wdot = 0, slots_jac = 0, bytes_wdot = 0, bytes_jac = 0;
    QssV1 v1;                      // launch descriptor of kernel variant 1 (valid iff v1_ok)
    bool v1_ok = false;
    std::string v1_why;            // why variant 1 does not apply
    std::string v1_gen;            // CUDA source of the mechanism-specialised pass A (qss_gen_pass_a), compiled at run time
    QssV3Host v3;                  // kernel variant 3 (valid iff v3_ok)
    bool v3_ok = false;
    std::string v3_why;
};

// Validates `desc` and builds the tables. Returns QSS_OK or a negative qss_status with `err` set.
int qss_compile(const qss_mech_desc_t *desc, QssCompiled &out, std::string &err);

#endif
