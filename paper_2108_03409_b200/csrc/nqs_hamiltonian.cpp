// Host-side Hamiltonian compiler.  See nqs_hamiltonian.h.
//
// Matrix elements in the row convention (reading Q3), s_k = spin of the ROW config:
//   <s|X_k|s'> = 1      (s' = s with k flipped)
//   <s|Y_k|s'> = -i s_k (s' = s with k flipped)
//   <s|Z_k|s > = s_k
// A term with n_Y sigma^y factors therefore has element c * (-i)^{n_Y} * prod_{k in Y,Z slots} s_k.
#include "nqs_hamiltonian.h"

#include <algorithm>
#include <map>
#include <utility>

namespace nqs {

static inline nqs_c64 cmul(nqs_c64 a, nqs_c64 b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }

int compile_hamiltonian(int32_t N, int32_t T, const int32_t* sites, const uint8_t* paulis,
                        const nqs_c64* coeffs, HostCompiled& out, std::string& err) {
    if (N <= 0 || T < 0 || (T > 0 && (!sites || !paulis || !coeffs))) {
        err = "compile_hamiltonian: bad N/T or NULL term arrays";
        return NQS_ERR_INVALID_ARG;
    }
    out = HostCompiled();
    out.N = N;
    out.T = T;

    struct Parsed { int32_t f[2]; int nf; int32_t z[2]; int nz; nqs_c64 c; };
    std::vector<Parsed> parsed(T);
    for (int t = 0; t < T; ++t) {
        Parsed p{{-1, -1}, 0, {-1, -1}, 0, coeffs[t]};
        int32_t s0 = sites[2 * t], s1 = sites[2 * t + 1];
        if (s0 >= 0 && s0 == s1) {
            err = "term " + std::to_string(t) + ": the same site in both slots";
            return NQS_ERR_INVALID_TERM;
        }
        for (int k = 0; k < 2; ++k) {
            int32_t site = sites[2 * t + k];
            uint8_t pk = paulis[2 * t + k];
            if (pk > 3) {
                err = "term " + std::to_string(t) + ": Pauli code > 3";
                return NQS_ERR_INVALID_TERM;
            }
            if (site < 0) {
                if (site != -1 || pk != NQS_I) {
                    err = "term " + std::to_string(t) + ": non-identity Pauli on an unused slot (or site < -1)";
                    return NQS_ERR_INVALID_TERM;
                }
                continue;
            }
            if (site >= N) {
                err = "term " + std::to_string(t) + ": site out of range";
                return NQS_ERR_INVALID_TERM;
            }
            if (pk == NQS_X || pk == NQS_Y) p.f[p.nf++] = site;
            if (pk == NQS_Y) p.c = cmul(p.c, nqs_c64{0.f, -1.f});
            if (pk == NQS_Y || pk == NQS_Z) p.z[p.nz++] = site;
        }
        if (p.nf == 2 && p.f[0] > p.f[1]) std::swap(p.f[0], p.f[1]);
        parsed[t] = p;
    }

    // group by flip set, in order of first appearance
    std::map<std::pair<int32_t, int32_t>, int> index;
    std::vector<std::vector<int>> members;
    for (int t = 0; t < T; ++t) {
        const Parsed& p = parsed[t];
        if (p.nf == 0) {
            out.diag_z0.push_back(p.z[0]);
            out.diag_z1.push_back(p.z[1]);
            out.diag_c.push_back(p.c);
            continue;
        }
        auto key = std::make_pair(p.f[0], p.f[1]);
        auto it = index.find(key);
        if (it == index.end()) {
            it = index.emplace(key, (int)out.groups.size()).first;
            out.groups.push_back(HostGroup{p.f[0], p.f[1], 0, 0, {-1, -1}});
            members.emplace_back();
        }
        members[it->second].push_back(t);
    }
    for (size_t g = 0; g < out.groups.size(); ++g) {
        HostGroup& G = out.groups[g];
        G.term_first = (int32_t)out.gt_c.size();
        G.term_count = (int32_t)members[g].size();
        for (int t : members[g]) {
            out.gt_z0.push_back(parsed[t].z[0]);
            out.gt_z1.push_back(parsed[t].z[1]);
            out.gt_c.push_back(parsed[t].c);
        }
        if (G.f1 < 0) {  // single flip: one column
            G.col[0] = (int32_t)out.col_i.size();
            out.col_i.push_back(G.f0);
            out.col_k.push_back(-1);
            out.col_p.push_back(+1);
            out.col_group.push_back((int32_t)g);
        } else {
            // pair flip: every term has both slots flipping, so the summed element is a function of
            // (s_f0, s_f1) only.  Emit the parity column p = s_f0 * s_f1 only if some spin pair of
            // that parity has a non-zero element (":458 non-zero matrix elements", reading Q5).
            for (int pi = 0; pi < 2; ++pi) {
                int par = pi == 0 ? +1 : -1;
                bool any = false;
                for (int sa = -1; sa <= 1; sa += 2) {
                    int sb = par * sa;
                    float mr = 0.f, mi = 0.f;
                    for (int q = 0; q < G.term_count; ++q) {
                        int idx = G.term_first + q;
                        float f = 1.f;
                        for (int32_t z : {out.gt_z0[idx], out.gt_z1[idx]}) {
                            if (z == G.f0) f *= (float)sa;
                            else if (z == G.f1) f *= (float)sb;
                        }
                        mr += out.gt_c[idx].re * f;
                        mi += out.gt_c[idx].im * f;
                    }
                    if (mr != 0.f || mi != 0.f) any = true;
                }
                if (any) {
                    G.col[pi] = (int32_t)out.col_i.size();
                    out.col_i.push_back(G.f0);
                    out.col_k.push_back(G.f1);
                    out.col_p.push_back(par);
                    out.col_group.push_back((int32_t)g);
                }
            }
        }
    }
    return NQS_OK;
}

}  // namespace nqs
