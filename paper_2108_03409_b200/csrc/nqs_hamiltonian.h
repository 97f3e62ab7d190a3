// Host-side compiled Hamiltonian (step a0 of DESIGN.md): validation, grouping of terms by flip
// set, per-column data for the product-form kernels.  Eq. 39: every term of a
// group maps s to the same s', so their matrix elements are summed (reading Q4).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/nqs.h"

namespace nqs {

struct HostGroup {
    int32_t f0, f1;           // flip set, f0 < f1, f1 = -1 for a single flip
    int32_t term_first, term_count;  // range into gt_* arrays
    int32_t col[2];           // table column for parity +1 / -1 (pair) ; col[0] for single; -1 = none
};

struct HostCompiled {
    int32_t N = 0, T = 0;
    // diagonal terms (empty flip set): c * s[z0] * s[z1], z = -1 means factor 1
    std::vector<int32_t> diag_z0, diag_z1;
    std::vector<nqs_c64> diag_c;
    // flip groups, in order of first appearance
    std::vector<HostGroup> groups;
    // terms of the groups: element = gt_c * s[gt_z0] * s[gt_z1]  (coefficient already carries (-i)^nY)
    std::vector<int32_t> gt_z0, gt_z1;
    std::vector<nqs_c64> gt_c;
    // table columns: V_j = W[j,ci] + cp * W[j,ck] (ck = -1: single flip), sign = spin at ci
    std::vector<int32_t> col_i, col_k, col_p, col_group;
};

// returns NQS_OK or NQS_ERR_INVALID_TERM / NQS_ERR_INVALID_ARG with a message in err
int compile_hamiltonian(int32_t N, int32_t T, const int32_t* sites, const uint8_t* paulis,
                        const nqs_c64* coeffs, HostCompiled& out, std::string& err);

}  // namespace nqs
