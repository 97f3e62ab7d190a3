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

int compile_hamiltonian(int32_t N, int32_t T, int32_t K, const int32_t* sites, const uint8_t* paulis,
                        const nqs_c64* coeffs, HostCompiled& out, std::string& err) {
    if (N <= 0 || T < 0 || K < 1 || K > HAM_MAX_SLOTS || (T > 0 && (!sites || !paulis || !coeffs))) {
        err = "compile_hamiltonian: bad N / T / K (1..8 slots per term) or NULL term arrays";
        return NQS_ERR_INVALID_ARG;
    }
    out = HostCompiled();
    out.N = N;
    out.T = T;

    struct Parsed { std::vector<int32_t> f, z; nqs_c64 c; };
    std::vector<Parsed> parsed(T);
    for (int t = 0; t < T; ++t) {
        Parsed p{{}, {}, coeffs[t]};
        for (int k = 0; k < K; ++k) {
            const int32_t site = sites[(size_t)t * K + k];
            const uint8_t pk = paulis[(size_t)t * K + k];
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
            for (int k2 = 0; k2 < k; ++k2)
                if (sites[(size_t)t * K + k2] == site) {
                    err = "term " + std::to_string(t) + ": the same site in two slots";
                    return NQS_ERR_INVALID_TERM;
                }
            if (pk == NQS_X || pk == NQS_Y) p.f.push_back(site);
            if (pk == NQS_Y) p.c = cmul(p.c, nqs_c64{0.f, -1.f});
            if (pk == NQS_Y || pk == NQS_Z) p.z.push_back(site);
        }
        if ((int)p.f.size() > HAM_MAX_FLIPS) {
            err = "term " + std::to_string(t) + ": more than four X / Y factors (flip sets of up to 4 sites are supported)";
            return NQS_ERR_UNSUPPORTED;
        }
        std::sort(p.f.begin(), p.f.end());
        parsed[t] = std::move(p);
    }

    auto push_z = [&](const Parsed& p, std::vector<int32_t>& z0, std::vector<int32_t>& z1, std::vector<int32_t>& zx) {
        z0.push_back(p.z.size() > 0 ? p.z[0] : -1);
        z1.push_back(p.z.size() > 1 ? p.z[1] : -1);
        for (size_t q = 2; q < p.z.size(); ++q) zx.push_back(p.z[q]);
        if (p.z.size() > 2) out.has_zx = true;
    };

    // group by flip set, in order of first appearance
    std::map<std::vector<int32_t>, int> index;
    std::vector<std::vector<int>> members;
    out.diag_zx_off.push_back(0);
    for (int t = 0; t < T; ++t) {
        const Parsed& p = parsed[t];
        if (p.f.empty()) {
            push_z(p, out.diag_z0, out.diag_z1, out.diag_zx);
            out.diag_zx_off.push_back((int32_t)out.diag_zx.size());
            out.diag_c.push_back(p.c);
            continue;
        }
        auto it = index.find(p.f);
        if (it == index.end()) {
            it = index.emplace(p.f, (int)out.groups.size()).first;
            HostGroup G{{-1, -1, -1, -1}, (int32_t)p.f.size(), 0, 0};
            for (size_t q = 0; q < p.f.size(); ++q) G.f[q] = p.f[q];
            out.groups.push_back(G);
            members.emplace_back();
        }
        members[it->second].push_back(t);
    }
    out.gt_zx_off.push_back(0);
    for (size_t g = 0; g < out.groups.size(); ++g) {
        HostGroup& G = out.groups[g];
        G.term_first = (int32_t)out.gt_c.size();
        G.term_count = (int32_t)members[g].size();
        bool outside = false;  // some term has a z factor on a site outside the flip set
        for (int t : members[g]) {
            push_z(parsed[t], out.gt_z0, out.gt_z1, out.gt_zx);
            out.gt_zx_off.push_back((int32_t)out.gt_zx.size());
            out.gt_c.push_back(parsed[t].c);
            for (int32_t z : parsed[t].z)
                if (std::find(G.f, G.f + G.nf, z) == G.f + G.nf) outside = true;
        }
        // one column per pattern of relative signs p_q = s[f_q] s[f_0], q = 1 .. nf-1 (2^(nf-1) patterns).  A
        // pattern is dropped only if the summed element is zero for both values of s[f_0] and no term looks at a
        // spin outside the flip set (":458 non-zero matrix elements", reading Q5): the antiparallel-only column
        // of the Heisenberg bonds.
        for (int pat = 0; pat < (1 << (G.nf - 1)); ++pat) {
            int sign[HAM_MAX_FLIPS] = {1, 1, 1, 1};
            for (int q = 1; q < G.nf; ++q) sign[q] = (pat >> (q - 1)) & 1 ? -1 : 1;
            bool any = outside;
            for (int sa = -1; sa <= 1 && !any; sa += 2) {
                float mr = 0.f, mi = 0.f;
                for (int t : members[g]) {
                    float f = 1.f;
                    for (int32_t z : parsed[t].z) {
                        const int q = (int)(std::find(G.f, G.f + G.nf, z) - G.f);
                        f *= (float)(sa * sign[q]);
                    }
                    mr += parsed[t].c.re * f;
                    mi += parsed[t].c.im * f;
                }
                if (mr != 0.f || mi != 0.f) any = true;
            }
            if (!any) continue;
            out.col_i.push_back(G.f[0]);
            out.col_k.push_back(G.nf > 1 ? G.f[1] : -1);
            out.col_p.push_back(sign[1]);
            out.col_s2.push_back(G.nf > 2 ? G.f[2] : -1);
            out.col_p2.push_back(sign[2]);
            out.col_s3.push_back(G.nf > 3 ? G.f[3] : -1);
            out.col_p3.push_back(sign[3]);
            out.col_group.push_back((int32_t)g);
        }
    }
    return NQS_OK;
}

}  // namespace nqs
