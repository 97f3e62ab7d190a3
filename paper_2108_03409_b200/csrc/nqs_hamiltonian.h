// Host-side compiled Hamiltonian (step a0 of DESIGN.md): validation, grouping of terms by flip
// set, per-column data for the a5 kernels.  Eq. 39: every term of a
// group maps s to the same s', so their matrix elements are summed (reading Q4).
// Terms are Pauli strings on K slots (K = 2: the north_star's "at most 2-site terms"; K up to 8 with at
// most four flipping sites: the k-site strings of SURVEY.md 8(f) item 4).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/nqs.h"

namespace nqs {

constexpr int HAM_MAX_SLOTS = 8;   // operators per term
constexpr int HAM_MAX_FLIPS = 4;   // X / Y factors per term (a flip set of m sites has 2^(m-1) sign columns)

struct HostGroup {
    int32_t f[HAM_MAX_FLIPS];        // flip set, ascending, -1 = unused
    int32_t nf;
    int32_t term_first, term_count;  // range into gt_* arrays
};

struct HostCompiled {
    int32_t N = 0, T = 0;
    // diagonal terms (empty flip set): c * prod_z s[z]; the first two z sites in z0, z1 (-1 = factor 1),
    // any further ones in the zx list (range zx_off[t] .. zx_off[t+1])
    std::vector<int32_t> diag_z0, diag_z1, diag_zx_off, diag_zx;
    std::vector<nqs_c64> diag_c;
    // flip groups, in order of first appearance
    std::vector<HostGroup> groups;
    // terms of the groups: element = gt_c * prod_z s[z]  (coefficient already carries (-i)^nY)
    std::vector<int32_t> gt_z0, gt_z1, gt_zx_off, gt_zx;
    std::vector<nqs_c64> gt_c;
    // table columns: V_j = W[j,ci] + cp W[j,ck] + p2 W[j,s2] + p3 W[j,s3] (ck, s2, s3 = -1: absent); the sign of
    // the column's amplitude is the spin at ci, the column is active for a sample iff s[ck] s[ci] = cp etc.
    std::vector<int32_t> col_i, col_k, col_p, col_s2, col_p2, col_s3, col_p3, col_group;
    bool has_zx = false;
};

// sites, paulis: [T,K].  returns NQS_OK or NQS_ERR_INVALID_TERM / NQS_ERR_INVALID_ARG / NQS_ERR_UNSUPPORTED with a
// message in err
int compile_hamiltonian(int32_t N, int32_t T, int32_t K, const int32_t* sites, const uint8_t* paulis,
                        const nqs_c64* coeffs, HostCompiled& out, std::string& err);

}  // namespace nqs
