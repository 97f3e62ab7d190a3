// C ABI of libnqs_b200.so (declared in include/nqs.h): argument checks, workspace, launches.
// Every step of the path runs in the kernels of nqs_kernels.cuh; there is no CPU fallback.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <list>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/nqs.h"
#include "nqs_hamiltonian.h"
#include "nqs_kernels.cuh"
#include "nqs_forces.cuh"
#include "nqs_microbench.cuh"
#include "nqs_sampler.cuh"
#include "nqs_theta_mma.cuh"

using namespace nqs;

// ----------------------------------------------------------------------------------------
// errors
// ----------------------------------------------------------------------------------------
static thread_local std::string g_err;

static int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
#define NQS_CUDA(call)                                                                             \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail(NQS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__));        \
    } while (0)

extern "C" const char* nqs_last_error(void) { return g_err.c_str(); }
extern "C" const char* nqs_version(void) { return "0.1.0 sm_100a"; }

// ----------------------------------------------------------------------------------------
// handle
// ----------------------------------------------------------------------------------------
struct nqs_hamiltonian {
    HostCompiled hc;
    int device = -1;       // -1: host-only compile
    void* d_blob = nullptr;
    DevHam dev{};
    int C = 0;
    // launch plan (static for the handle): column tiling of the a5 kernel
    int WC = 1, WS = 2, TC = 16, nTiles = 1, C_pad = 16;
};

static constexpr int KJ = 16;
static constexpr int MAX_WC = 5;

static void plan_tiles(nqs_hamiltonian* h) {
    const int C = (int)h->hc.col_i.size();
    h->C = C;
    const int slices = C > 0 ? (C + 15) / 16 : 1;
    // least padded work divided by the measured efficiency of the block shape: a CTA has 2 WC warps, and
    // narrow CTAs leave the SM short of warps (measured per 16-column slice on configs 3 and 4, B200)
    static const double eff[MAX_WC + 1] = {0.0, 0.36, 0.54, 0.55, 0.68, 0.64};
    int best = 1;
    double best_cost = 1e30;
    for (int wc = 1; wc <= MAX_WC; ++wc) {
        const int tiles = (slices + wc - 1) / wc;
        const double cost = (double)tiles * wc / eff[wc];
        if (cost < best_cost - 1e-9) {
            best_cost = cost;
            best = wc;
        }
    }
    if (const char* e = getenv("NQS_WC")) {  // A/B experiments
        const int v = atoi(e);
        if (v >= 1 && v <= MAX_WC) best = v;
    }
    h->WC = best;
    h->WS = 2;
    h->TC = 16 * best;
    h->nTiles = (slices + best - 1) / best;
    h->C_pad = h->nTiles * h->TC;
}

static int upload(nqs_hamiltonian* h) {
    const HostCompiled& hc = h->hc;
    const int G = (int)hc.groups.size(), Td = (int)hc.diag_c.size(), Tg = (int)hc.gt_c.size();
    const int C_pad = h->C_pad;
    // blob layout: ints then float2s
    std::vector<int> ints;
    auto push = [&](const std::vector<int32_t>& v) {
        size_t o = ints.size();
        ints.insert(ints.end(), v.begin(), v.end());
        return o;
    };
    std::vector<int32_t> f0(G), f1(G), first(G), count(G);
    for (int g = 0; g < G; ++g) {
        f0[g] = hc.groups[g].f0;
        f1[g] = hc.groups[g].f1;
        first[g] = hc.groups[g].term_first;
        count[g] = hc.groups[g].term_count;
    }
    std::vector<int32_t> ci(C_pad, 0), ck(C_pad, -1), cp(C_pad, 1), cg(C_pad, -1);
    for (int c = 0; c < h->C; ++c) {
        ci[c] = hc.col_i[c];
        ck[c] = hc.col_k[c];
        cp[c] = hc.col_p[c];
        cg[c] = hc.col_group[c];
    }
    const size_t o_dz0 = push(hc.diag_z0), o_dz1 = push(hc.diag_z1);
    const size_t o_f0 = push(f0), o_f1 = push(f1), o_first = push(first), o_count = push(count);
    const size_t o_gz0 = push(hc.gt_z0), o_gz1 = push(hc.gt_z1);
    const size_t o_ci = push(ci), o_ck = push(ck), o_cp = push(cp), o_cg = push(cg);
    size_t int_bytes = (ints.size() * sizeof(int) + 15) / 16 * 16;
    std::vector<nqs_c64> cs;
    cs.insert(cs.end(), hc.diag_c.begin(), hc.diag_c.end());
    cs.insert(cs.end(), hc.gt_c.begin(), hc.gt_c.end());
    const size_t total = int_bytes + cs.size() * sizeof(nqs_c64) + 16;
    std::vector<unsigned char> blob(total, 0);
    if (!ints.empty()) memcpy(blob.data(), ints.data(), ints.size() * sizeof(int));
    if (!cs.empty()) memcpy(blob.data() + int_bytes, cs.data(), cs.size() * sizeof(nqs_c64));
    NQS_CUDA(cudaGetDevice(&h->device));
    NQS_CUDA(cudaMalloc(&h->d_blob, total));
    NQS_CUDA(cudaMemcpy(h->d_blob, blob.data(), total, cudaMemcpyHostToDevice));
    const int* di = reinterpret_cast<const int*>(h->d_blob);
    const float2* dc = reinterpret_cast<const float2*>(reinterpret_cast<const unsigned char*>(h->d_blob) + int_bytes);
    DevHam& D = h->dev;
    D.N = hc.N;
    D.G = G;
    D.C = h->C;
    D.Td = Td;
    D.Tg = Tg;
    D.diag_z0 = di + o_dz0;
    D.diag_z1 = di + o_dz1;
    D.diag_c = dc;
    D.grp_f0 = di + o_f0;
    D.grp_f1 = di + o_f1;
    D.grp_first = di + o_first;
    D.grp_count = di + o_count;
    D.gt_z0 = di + o_gz0;
    D.gt_z1 = di + o_gz1;
    D.gt_c = dc + Td;
    D.col_i = di + o_ci;
    D.col_k = di + o_ck;
    D.col_p = di + o_cp;
    D.col_group = di + o_cg;
    return NQS_OK;
}

static int create_impl(int32_t N, int32_t T, const int32_t* s, const uint8_t* p, const nqs_c64* c, bool device,
                       nqs_hamiltonian** out) {
    if (!out) return fail(NQS_ERR_INVALID_ARG, "nqs_hamiltonian_create: out is NULL");
    *out = nullptr;
    auto* h = new nqs_hamiltonian();
    std::string err;
    int rc = compile_hamiltonian(N, T, s, p, c, h->hc, err);
    if (rc != NQS_OK) {
        delete h;
        return fail(rc, err);
    }
    plan_tiles(h);
    if (device) {
        rc = upload(h);
        if (rc != NQS_OK) {
            if (h->d_blob) cudaFree(h->d_blob);
            delete h;
            return rc;
        }
    }
    *out = h;
    return NQS_OK;
}

extern "C" int nqs_hamiltonian_create(int32_t N, int32_t T, const int32_t* h_sites, const uint8_t* h_paulis,
                                      const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, h_sites, h_paulis, h_coeffs, true, out);
}
extern "C" int nqs_hamiltonian_compile_host(int32_t N, int32_t T, const int32_t* h_sites, const uint8_t* h_paulis,
                                            const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, h_sites, h_paulis, h_coeffs, false, out);
}
extern "C" int nqs_hamiltonian_destroy(nqs_hamiltonian* h) {
    if (!h) return NQS_OK;
    if (h->d_blob) cudaFree(h->d_blob);
    delete h;
    return NQS_OK;
}
extern "C" int nqs_hamiltonian_info(const nqs_hamiltonian* h, int32_t info[5], int32_t* flip_sites) {
    if (!h || !info) return fail(NQS_ERR_INVALID_ARG, "nqs_hamiltonian_info: NULL argument");
    info[0] = (int32_t)h->hc.groups.size();
    info[1] = (int32_t)h->hc.col_i.size();
    info[2] = (int32_t)h->hc.diag_c.size();
    info[3] = (int32_t)h->hc.gt_c.size();
    info[4] = h->hc.N;
    if (flip_sites)
        for (size_t g = 0; g < h->hc.groups.size(); ++g) {
            flip_sites[2 * g] = h->hc.groups[g].f0;
            flip_sites[2 * g + 1] = h->hc.groups[g].f1;
        }
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// cache of compiled Hamiltonians for the term-list entry points
// ----------------------------------------------------------------------------------------
struct CacheEntry {
    int device, N, T;
    std::vector<unsigned char> key;
    nqs_hamiltonian* h;
};
static std::mutex g_cache_mu;
static std::list<CacheEntry> g_cache;

static int cached_hamiltonian(int32_t N, int32_t T, const int32_t* s, const uint8_t* p, const nqs_c64* c,
                              nqs_hamiltonian** out) {
    if (T < 0 || (T > 0 && (!s || !p || !c))) return fail(NQS_ERR_INVALID_ARG, "term arrays are NULL or T < 0");
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    std::vector<unsigned char> key((size_t)T * (8 + 2 + 8));
    if (T > 0) {
        memcpy(key.data(), s, (size_t)T * 8);
        memcpy(key.data() + (size_t)T * 8, p, (size_t)T * 2);
        memcpy(key.data() + (size_t)T * 10, c, (size_t)T * 8);
    }
    std::lock_guard<std::mutex> lk(g_cache_mu);
    for (auto it = g_cache.begin(); it != g_cache.end(); ++it)
        if (it->device == dev && it->N == N && it->T == T && it->key == key) {
            g_cache.splice(g_cache.begin(), g_cache, it);
            *out = g_cache.front().h;
            return NQS_OK;
        }
    nqs_hamiltonian* h = nullptr;
    int rc = nqs_hamiltonian_create(N, T, s, p, c, &h);
    if (rc != NQS_OK) return rc;
    g_cache.push_front(CacheEntry{dev, N, T, std::move(key), h});
    if (g_cache.size() > 8) {
        // an evicted handle may still be in use by kernels in flight on some stream
        cudaDeviceSynchronize();
        nqs_hamiltonian_destroy(g_cache.back().h);
        g_cache.pop_back();
    }
    *out = h;
    return NQS_OK;
}

extern "C" int nqs_release(void) {
    std::lock_guard<std::mutex> lk(g_cache_mu);
    if (!g_cache.empty()) cudaDeviceSynchronize();
    for (auto& e : g_cache) nqs_hamiltonian_destroy(e.h);
    g_cache.clear();
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// optional per-kernel timing (bench.py's roofline leg): CUDA events recorded on the caller's
// stream around the four kernels of the most recent nqs_local_energy* call
// ----------------------------------------------------------------------------------------
static bool g_prof_on = false;
static cudaEvent_t g_prof_ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
static bool g_prof_valid = false;

extern "C" int nqs_profile_enable(int on) {
    if (on && !g_prof_ev[0])
        for (auto& e : g_prof_ev) NQS_CUDA(cudaEventCreate(&e));
    g_prof_on = on != 0;
    g_prof_valid = false;
    return NQS_OK;
}
extern "C" int nqs_profile_last(float ms[4]) {
    if (!ms) return fail(NQS_ERR_INVALID_ARG, "ms is NULL");
    if (!g_prof_valid) return fail(NQS_ERR_INVALID_ARG, "no profiled call recorded");
    NQS_CUDA(cudaEventSynchronize(g_prof_ev[4]));
    for (int k = 0; k < 4; ++k) NQS_CUDA(cudaEventElapsedTime(&ms[k], g_prof_ev[k], g_prof_ev[k + 1]));
    return NQS_OK;
}
#define NQS_PROF(k, st)                                            \
    do {                                                           \
        if (g_prof_on) NQS_CUDA(cudaEventRecord(g_prof_ev[k], st)); \
    } while (0)

// ----------------------------------------------------------------------------------------
// device checks, workspace
// ----------------------------------------------------------------------------------------
static int check_device() {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        cudaGetLastError();
        return fail(NQS_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
    }
    static std::once_flag once;
    std::call_once(once, [&] {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long thr = ~0ull;  // keep freed workspace cached in the pool
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
    });
    return NQS_OK;
}

static inline long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }

static int launch_theta_simt(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad, const nqs_c64* d_a,
                             const nqs_c64* d_b, const nqs_c64* d_W, float4* tp, long long nPairsPad,
                             nqs_c64* d_logpsi, cudaStream_t st, bool raw_theta) {
    const long long rows = tp ? nPairsPad * 2 : B;
    const unsigned grid = (unsigned)((rows + 63) / 64);
    static bool attr_set = false;
    if (!attr_set) {
        NQS_CUDA(cudaFuncSetAttribute(theta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TH_SMEM));
        attr_set = true;
    }
    theta_kernel<<<grid, 256, TH_SMEM, st>>>(d_spins, (long long)B, N, M, M_pad, (const float2*)d_a, (const float2*)d_b,
                                       (const float2*)d_W, tp, nPairsPad, (float2*)d_logpsi, raw_theta ? 1 : 0);
    NQS_CUDA(cudaGetLastError());
    return NQS_OK;
}

// a2 on the tensor cores: pack spins and the int8 digits of W, then theta_mma_kernel (tcgen05).
static int launch_theta_mma(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad, const nqs_c64* d_a,
                            const nqs_c64* d_b, const nqs_c64* d_W, float4* tp, long long nPairsPad,
                            nqs_c64* d_logpsi, cudaStream_t st, bool raw_theta) {
    const long long rows = tp ? nPairsPad * 2 : B;
    const long long nMT = (rows + TM_M - 1) / TM_M;
    const int K_pad = (int)round_up(N, TM_KC), K16 = K_pad / 16;
    const int nNT = (M_pad + TM_JT - 1) / TM_JT;
    uint4 *A_packed = nullptr, *B_packed = nullptr;
    float* scale = nullptr;
    NQS_CUDA(cudaMallocAsync(&A_packed, sizeof(uint4) * (size_t)nMT * K16 * TM_M, st));
    NQS_CUDA(cudaMallocAsync(&B_packed, sizeof(uint4) * (size_t)nNT * K16 * TM_N, st));
    NQS_CUDA(cudaMallocAsync(&scale, sizeof(float) * (size_t)nNT * TM_JT, st));
    const long long a_items = nMT * K16 * TM_M;
    const unsigned agrid = (unsigned)((a_items + 255) / 256 < 148 * 16 ? (a_items + 255) / 256 : 148 * 16);
    pack_spins_kernel<<<agrid, 256, 0, st>>>(d_spins, (long long)B, N, K16, nMT, A_packed);
    NQS_CUDA(cudaGetLastError());
    pack_w_kernel<<<(unsigned)(nNT * TM_JT), 128, 0, st>>>((const float2*)d_W, N, M, K16, B_packed, scale);
    NQS_CUDA(cudaGetLastError());
    const size_t smem = theta_mma_smem_bytes(K_pad);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        NQS_CUDA(cudaFuncSetAttribute(theta_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_smem = smem;
    }
    ThetaMmaParams p;
    p.A_packed = A_packed;
    p.B_packed = B_packed;
    p.scale = scale;
    p.bvec = (const float2*)d_b;
    p.a = (const float2*)d_a;
    p.spins = d_spins;
    p.B = B;
    p.N = N;
    p.M = M;
    p.M_pad = M_pad;
    p.K16 = K16;
    p.nNT = nNT;
    p.tp = tp;
    p.nPairsPad = nPairsPad;
    p.logpsi = (float2*)d_logpsi;
    p.raw_theta = raw_theta ? 1 : 0;
    theta_mma_kernel<<<(unsigned)nMT, TM_THREADS, smem, st>>>(p);
    NQS_CUDA(cudaGetLastError());
    NQS_CUDA(cudaFreeAsync(A_packed, st));
    NQS_CUDA(cudaFreeAsync(B_packed, st));
    NQS_CUDA(cudaFreeAsync(scale, st));
    return NQS_OK;
}

// NQS_THETA=simt forces the FP32 SIMT kernel (A/B comparisons); the tensor-core kernel covers N <= 512.
static bool theta_use_mma(int32_t N) {
    static const bool force_simt = [] {
        const char* e = getenv("NQS_THETA");
        return e && strcmp(e, "simt") == 0;
    }();
    return !force_simt && round_up(N, TM_KC) <= TM_MAX_KPAD;
}

static int launch_theta(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad, const nqs_c64* d_a,
                        const nqs_c64* d_b, const nqs_c64* d_W, float4* tp, long long nPairsPad, nqs_c64* d_logpsi,
                        cudaStream_t st, bool raw_theta = false) {
    if (theta_use_mma(N))
        return launch_theta_mma(d_spins, B, N, M, M_pad, d_a, d_b, d_W, tp, nPairsPad, d_logpsi, st, raw_theta);
    return launch_theta_simt(d_spins, B, N, M, M_pad, d_a, d_b, d_W, tp, nPairsPad, d_logpsi, st, raw_theta);
}

template <int WC, int WS>
static int launch_eloc_t(const ElocParams& p, long long nBlocksY, cudaStream_t st) {
    using Cfg = ElocCfg<WC, WS, KJ>;
    static bool attr_set = false;
    if (!attr_set) {
        NQS_CUDA(cudaFuncSetAttribute(eloc_kernel<WC, WS, KJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)Cfg::SMEM));
        attr_set = true;
    }
    dim3 grid((unsigned)p.nTiles, (unsigned)nBlocksY);
    eloc_kernel<WC, WS, KJ><<<grid, Cfg::NT, Cfg::SMEM, st>>>(p);
    NQS_CUDA(cudaGetLastError());
    return NQS_OK;
}

static int launch_eloc(const nqs_hamiltonian* h, const ElocParams& p, long long B_pad, cudaStream_t st) {
    const long long nby = B_pad / (32 * h->WS);
    switch (h->WC) {
        case 1: return launch_eloc_t<1, 2>(p, nby, st);
        case 2: return launch_eloc_t<2, 2>(p, nby, st);
        case 3: return launch_eloc_t<3, 2>(p, nby, st);
        case 4: return launch_eloc_t<4, 2>(p, nby, st);
        case 5: return launch_eloc_t<5, 2>(p, nby, st);
    }
    return fail(NQS_ERR_UNSUPPORTED, "unsupported column tiling");
}

static int check_common(const void* spins, int64_t B, int32_t N, int32_t M, const void* a, const void* b,
                        const void* W) {
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "B < 0");
    if (N <= 0 || M <= 0) return fail(NQS_ERR_INVALID_ARG, "N and M must be positive");
    if (B > 0 && (!spins || !a || !b || !W)) return fail(NQS_ERR_INVALID_ARG, "NULL spins/parameter pointer");
    if ((long long)B * N > (1ll << 40)) return fail(NQS_ERR_UNSUPPORTED, "B*N too large");
    return NQS_OK;
}

extern "C" int nqs_log_psi(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                           const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_logpsi, void* stream) {
    int rc = check_common(d_spins, B, N, M, d_a, d_b, d_W);
    if (rc) return rc;
    if (B > 0 && !d_logpsi) return fail(NQS_ERR_INVALID_ARG, "d_logpsi is NULL");
    if ((rc = check_device())) return rc;
    if (B == 0) return NQS_OK;
    return launch_theta(d_spins, B, N, M, (int)round_up(M, KJ), d_a, d_b, d_W, nullptr, 0, d_logpsi,
                        (cudaStream_t)stream);
}

// keep_tp != NULL: tanh(theta) ([M_pad][B_pad/2] float4, stream-ordered allocation) is handed to the
// caller (who frees it with cudaFreeAsync) instead of being released -- nqs_local_energy_forces_h.
static int local_energy_impl(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M,
                             const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_eloc,
                             nqs_c64* d_logpsi, void* stream, float4** keep_tp) {
    if (!h) return fail(NQS_ERR_INVALID_ARG, "hamiltonian handle is NULL");
    const int N = h->hc.N;
    int rc = check_common(d_spins, B, N, M, d_a, d_b, d_W);
    if (rc) return rc;
    if (B > 0 && !d_eloc) return fail(NQS_ERR_INVALID_ARG, "d_eloc is NULL");
    if ((rc = check_device())) return rc;
    if (h->device < 0) return fail(NQS_ERR_INVALID_ARG, "handle was compiled host-only (nqs_hamiltonian_compile_host)");
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    if (dev != h->device) return fail(NQS_ERR_INVALID_ARG, "handle belongs to another device");
    if (B == 0) return NQS_OK;
    cudaStream_t st = (cudaStream_t)stream;

    const int M_pad = (int)round_up(M, KJ);
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;
    const int nTiles = h->nTiles, TC = h->TC, C_pad = h->C_pad;

    float4 *tp = nullptr, *tab = nullptr, *rho = nullptr;
    float2* partial = nullptr;
    const bool have_cols = h->C > 0;
    if (have_cols || keep_tp) NQS_CUDA(cudaMallocAsync(&tp, sizeof(float4) * (size_t)M_pad * nPairsPad, st));
    if (have_cols) {
        NQS_CUDA(cudaMallocAsync(&tab, sizeof(float4) * (size_t)nTiles * M_pad * TC, st));
        NQS_CUDA(cudaMallocAsync(&rho, sizeof(float4) * (size_t)C_pad, st));
        NQS_CUDA(cudaMallocAsync(&partial, sizeof(float2) * (size_t)B * nTiles, st));
        NQS_PROF(0, st);
        const long long total = (long long)M_pad * C_pad;
        const unsigned tgrid = (unsigned)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
        table_kernel<<<tgrid, 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad, h->C, TC, nTiles,
                                            h->dev.col_i, h->dev.col_k, h->dev.col_p, tab, rho);
        NQS_CUDA(cudaGetLastError());
    }
    if (have_cols) NQS_PROF(1, st);
    if (have_cols || d_logpsi || keep_tp) {
        rc = launch_theta(d_spins, B, N, M, M_pad, d_a, d_b, d_W, tp, nPairsPad, d_logpsi, st);
        if (rc) return rc;
    }
    if (have_cols) {
        NQS_PROF(2, st);
        ElocParams p;
        p.tp = tp;
        p.nPairsPad = nPairsPad;
        p.tab = tab;
        p.rho = rho;
        p.spins = d_spins;
        p.B = B;
        p.N = N;
        p.M_pad = M_pad;
        p.nTiles = nTiles;
        p.H = h->dev;
        p.partial = partial;
        rc = launch_eloc(h, p, B_pad, st);
        if (rc) return rc;
        NQS_PROF(3, st);
    }
    finalize_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(d_spins, (long long)B, N, h->dev, partial,
                                                                 have_cols ? nTiles : 0, (float2*)d_eloc);
    NQS_CUDA(cudaGetLastError());
    if (have_cols) {
        NQS_PROF(4, st);
        g_prof_valid = g_prof_on;
        NQS_CUDA(cudaFreeAsync(tab, st));
        NQS_CUDA(cudaFreeAsync(rho, st));
        NQS_CUDA(cudaFreeAsync(partial, st));
    }
    if (keep_tp)
        *keep_tp = tp;
    else if (tp)
        NQS_CUDA(cudaFreeAsync(tp, st));
    return NQS_OK;
}

extern "C" int nqs_local_energy_h(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M,
                                  const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_eloc,
                                  nqs_c64* d_logpsi, void* stream) {
    return local_energy_impl(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream, nullptr);
}

extern "C" int nqs_local_energy(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                                const nqs_c64* d_b, const nqs_c64* d_W, int32_t T, const int32_t* h_sites,
                                const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_c64* d_eloc,
                                nqs_c64* d_logpsi, void* stream) {
    int rc = check_common(d_spins, B, N, M, d_a, d_b, d_W);
    if (rc) return rc;
    if ((rc = check_device())) return rc;
    nqs_hamiltonian* h = nullptr;
    if ((rc = cached_hamiltonian(N, T, h_sites, h_paulis, h_coeffs, &h))) return rc;
    return nqs_local_energy_h(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream);
}

extern "C" int nqs_enumerate_connected(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B,
                                       int8_t* d_sprime, nqs_c64* d_mel, void* stream) {
    if (!h) return fail(NQS_ERR_INVALID_ARG, "hamiltonian handle is NULL");
    if (B < 0 || (B > 0 && (!d_spins || !d_sprime || !d_mel))) return fail(NQS_ERR_INVALID_ARG, "bad arguments");
    int rc = check_device();
    if (rc) return rc;
    if (h->device < 0) return fail(NQS_ERR_INVALID_ARG, "handle was compiled host-only");
    if (B == 0) return NQS_OK;
    const long long total = (long long)B * (h->dev.G + 1);
    const unsigned grid = (unsigned)((total + 127) / 128 < 65535 ? (total + 127) / 128 : 65535);
    enumerate_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(d_spins, (long long)B, h->hc.N, h->dev, d_sprime,
                                                             (float2*)d_mel);
    NQS_CUDA(cudaGetLastError());
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// host-buffer entry points (end-to-end: H2D, kernels, D2H, synchronise)
// ----------------------------------------------------------------------------------------
struct HostStage {
    cudaStream_t st = nullptr;
    std::vector<void*> bufs;
    ~HostStage() {
        for (void* b : bufs) cudaFreeAsync(b, st);
        if (st) {
            cudaStreamSynchronize(st);
            cudaStreamDestroy(st);
        }
    }
    int init() {
        NQS_CUDA(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
        return NQS_OK;
    }
    int to_device(const void* h, size_t bytes, void** d) {
        NQS_CUDA(cudaMallocAsync(d, bytes ? bytes : 16, st));
        bufs.push_back(*d);
        if (bytes) NQS_CUDA(cudaMemcpyAsync(*d, h, bytes, cudaMemcpyHostToDevice, st));
        return NQS_OK;
    }
    int alloc(size_t bytes, void** d) {
        NQS_CUDA(cudaMallocAsync(d, bytes ? bytes : 16, st));
        bufs.push_back(*d);
        return NQS_OK;
    }
};

extern "C" int nqs_local_energy_host(const int8_t* h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* h_a,
                                     const nqs_c64* h_b, const nqs_c64* h_W, int32_t T, const int32_t* h_sites,
                                     const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_c64* h_eloc,
                                     nqs_c64* h_logpsi) {
    int rc = check_common(h_spins, B, N, M, h_a, h_b, h_W);
    if (rc) return rc;
    if (B > 0 && !h_eloc) return fail(NQS_ERR_INVALID_ARG, "h_eloc is NULL");
    if ((rc = check_device())) return rc;
    nqs_hamiltonian* h = nullptr;
    if ((rc = cached_hamiltonian(N, T, h_sites, h_paulis, h_coeffs, &h))) return rc;
    if (B == 0) return NQS_OK;
    HostStage S;
    if ((rc = S.init())) return rc;
    void *ds, *da, *db, *dW, *de, *dl = nullptr;
    if ((rc = S.to_device(h_spins, (size_t)B * N, &ds))) return rc;
    if ((rc = S.to_device(h_a, sizeof(nqs_c64) * N, &da))) return rc;
    if ((rc = S.to_device(h_b, sizeof(nqs_c64) * M, &db))) return rc;
    if ((rc = S.to_device(h_W, sizeof(nqs_c64) * (size_t)M * N, &dW))) return rc;
    if ((rc = S.alloc(sizeof(nqs_c64) * B, &de))) return rc;
    if (h_logpsi && (rc = S.alloc(sizeof(nqs_c64) * B, &dl))) return rc;
    rc = nqs_local_energy_h(h, (const int8_t*)ds, B, M, (const nqs_c64*)da, (const nqs_c64*)db, (const nqs_c64*)dW,
                            (nqs_c64*)de, (nqs_c64*)dl, S.st);
    if (rc) return rc;
    NQS_CUDA(cudaMemcpyAsync(h_eloc, de, sizeof(nqs_c64) * B, cudaMemcpyDeviceToHost, S.st));
    if (h_logpsi) NQS_CUDA(cudaMemcpyAsync(h_logpsi, dl, sizeof(nqs_c64) * B, cudaMemcpyDeviceToHost, S.st));
    NQS_CUDA(cudaStreamSynchronize(S.st));
    return NQS_OK;
}

extern "C" int nqs_log_psi_host(const int8_t* h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* h_a,
                                const nqs_c64* h_b, const nqs_c64* h_W, nqs_c64* h_logpsi) {
    int rc = check_common(h_spins, B, N, M, h_a, h_b, h_W);
    if (rc) return rc;
    if (B > 0 && !h_logpsi) return fail(NQS_ERR_INVALID_ARG, "h_logpsi is NULL");
    if ((rc = check_device())) return rc;
    if (B == 0) return NQS_OK;
    HostStage S;
    if ((rc = S.init())) return rc;
    void *ds, *da, *db, *dW, *dl;
    if ((rc = S.to_device(h_spins, (size_t)B * N, &ds))) return rc;
    if ((rc = S.to_device(h_a, sizeof(nqs_c64) * N, &da))) return rc;
    if ((rc = S.to_device(h_b, sizeof(nqs_c64) * M, &db))) return rc;
    if ((rc = S.to_device(h_W, sizeof(nqs_c64) * (size_t)M * N, &dW))) return rc;
    if ((rc = S.alloc(sizeof(nqs_c64) * B, &dl))) return rc;
    rc = nqs_log_psi((const int8_t*)ds, B, N, M, (const nqs_c64*)da, (const nqs_c64*)db, (const nqs_c64*)dW,
                     (nqs_c64*)dl, S.st);
    if (rc) return rc;
    NQS_CUDA(cudaMemcpyAsync(h_logpsi, dl, sizeof(nqs_c64) * B, cudaMemcpyDeviceToHost, S.st));
    NQS_CUDA(cudaStreamSynchronize(S.st));
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// pipe-rate micro-benchmarks (measured peaks for the roofline)
// ----------------------------------------------------------------------------------------
template <int KIND>
static void launch_microbench(float* out, unsigned grid, int iters, cudaStream_t st) {
    microbench_kernel<KIND><<<grid, 320, 0, st>>>(out, iters, 1e-3f, 0.999f);
}

extern "C" int nqs_microbench(int32_t kind, int32_t iters, double* lane_ops_per_s, float* ms_out) {
    if (kind < 0 || kind >= MB_KINDS || iters <= 0 || !lane_ops_per_s)
        return fail(NQS_ERR_INVALID_ARG, "nqs_microbench: bad kind / iters / NULL output");
    int rc = check_device();
    if (rc) return rc;
    int dev = 0, sms = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    NQS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const unsigned grid = 2u * (unsigned)sms;
    float* out = nullptr;
    cudaStream_t st = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    NQS_CUDA(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    NQS_CUDA(cudaMalloc(&out, sizeof(float) * (size_t)grid * 320));
    NQS_CUDA(cudaEventCreate(&e0));
    NQS_CUDA(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up; best of the rest
        NQS_CUDA(cudaEventRecord(e0, st));
        switch (kind) {
            case MB_FFMA: launch_microbench<MB_FFMA>(out, grid, iters, st); break;
            case MB_FFMA2: launch_microbench<MB_FFMA2>(out, grid, iters, st); break;
            case MB_BODY_PACKED: launch_microbench<MB_BODY_PACKED>(out, grid, iters, st); break;
            case MB_BODY_SCALAR: launch_microbench<MB_BODY_SCALAR>(out, grid, iters, st); break;
            default: launch_microbench<MB_MUFU_EX2>(out, grid, iters, st); break;
        }
        NQS_CUDA(cudaGetLastError());
        NQS_CUDA(cudaEventRecord(e1, st));
        NQS_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        NQS_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    cudaStreamDestroy(st);
    *lane_ops_per_s = (double)grid * 320.0 * iters * mb_ops_per_iter(kind) / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// batch statistics and the force vector
// ----------------------------------------------------------------------------------------
static int launch_stats(const nqs_c64* d_x, const float* d_w, int64_t B, double* d_stats, cudaStream_t st) {
    double* partial = nullptr;
    const int nblk = (int)((B + 255) / 256 < ST_BLOCKS ? (B + 255) / 256 : ST_BLOCKS);
    NQS_CUDA(cudaMallocAsync(&partial, sizeof(double) * 4 * ST_BLOCKS, st));
    stats_partial_kernel<<<nblk, 256, 0, st>>>((const float2*)d_x, d_w, (long long)B, partial);
    NQS_CUDA(cudaGetLastError());
    stats_final_kernel<<<1, 32, 0, st>>>(partial, nblk, d_stats);
    NQS_CUDA(cudaGetLastError());
    NQS_CUDA(cudaFreeAsync(partial, st));
    return NQS_OK;
}

extern "C" int nqs_energy_stats(const nqs_c64* d_x, const float* d_weights, int64_t B, double* d_stats,
                                void* stream) {
    if (B <= 0 || !d_x || !d_stats) return fail(NQS_ERR_INVALID_ARG, "nqs_energy_stats: B <= 0 or NULL pointer");
    int rc = check_device();
    if (rc) return rc;
    return launch_stats(d_x, d_weights, B, d_stats, (cudaStream_t)stream);
}

// tp_in != NULL: tanh(theta) of this batch from local_energy_impl (ownership passes to this function)
static int forces_impl(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                       const nqs_c64* d_b, const nqs_c64* d_W, const nqs_c64* d_eloc, const float* d_weights,
                       nqs_c64* d_F, double* d_stats, void* stream, float4* tp_in) {
    int rc = check_common(d_spins, B, N, M, d_a, d_b, d_W);
    if (rc) return rc;
    if (B <= 0 || !d_eloc || !d_F) return fail(NQS_ERR_INVALID_ARG, "nqs_forces: B <= 0 or NULL d_eloc / d_F");
    if (B > (1ll << 25)) return fail(NQS_ERR_UNSUPPORTED, "nqs_forces: B > 2^25 (int32 accumulation range)");
    if ((rc = check_device())) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int M_pad = (int)round_up(M, KJ);
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;
    const int K16 = (int)(B_pad / 16);
    const int nIT = (N + 1 + TM_M - 1) / TM_M, nJT = (M + 1 + TM_JT - 1) / TM_JT;

    float4* tp = tp_in;
    float2* cb = nullptr;
    double* stats = nullptr;
    int* gexp = nullptr;
    uint4 *A_packed = nullptr, *B_packed = nullptr;
    if (!tp) NQS_CUDA(cudaMallocAsync(&tp, sizeof(float4) * (size_t)M_pad * nPairsPad, st));
    NQS_CUDA(cudaMallocAsync(&cb, sizeof(float2) * (size_t)B_pad, st));
    NQS_CUDA(cudaMallocAsync(&stats, sizeof(double) * 4, st));
    NQS_CUDA(cudaMallocAsync(&gexp, sizeof(int) * (size_t)nJT * TM_JT, st));
    NQS_CUDA(cudaMallocAsync(&A_packed, sizeof(uint4) * (size_t)nIT * K16 * TM_M, st));
    NQS_CUDA(cudaMallocAsync(&B_packed, sizeof(uint4) * (size_t)nJT * K16 * TM_N, st));

    if ((rc = launch_stats(d_eloc, d_weights, B, stats, st))) return rc;
    if (d_stats) NQS_CUDA(cudaMemcpyAsync(d_stats, stats, sizeof(double) * 4, cudaMemcpyDeviceToDevice, st));
    force_coef_kernel<<<(unsigned)((B_pad + 255) / 256), 256, 0, st>>>((const float2*)d_eloc, d_weights, (long long)B,
                                                                       B_pad, stats, cb);
    NQS_CUDA(cudaGetLastError());
    if (!tp_in && (rc = launch_theta(d_spins, B, N, M, M_pad, d_a, d_b, d_W, tp, nPairsPad, nullptr, st))) return rc;
    force_gscale_kernel<<<(unsigned)(nJT * TM_JT), 256, 0, st>>>(tp, nPairsPad, cb, M, gexp);
    NQS_CUDA(cudaGetLastError());
    force_pack_g_kernel<<<148 * 8, 256, 0, st>>>(tp, nPairsPad, cb, M, K16, nJT, gexp, B_packed);
    NQS_CUDA(cudaGetLastError());
    force_pack_spins_kernel<<<148 * 8, 256, 0, st>>>(d_spins, (long long)B, N, K16, nIT, A_packed);
    NQS_CUDA(cudaGetLastError());
    static bool attr_set = false;
    if (!attr_set) {
        NQS_CUDA(cudaFuncSetAttribute(force_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FM_SMEM));
        attr_set = true;
    }
    ForceMmaParams p;
    p.A_packed = A_packed;
    p.B_packed = B_packed;
    p.gexp = gexp;
    p.N = N;
    p.M = M;
    p.K16 = K16;
    p.F = (float2*)d_F;
    force_mma_kernel<<<dim3((unsigned)nIT, (unsigned)nJT), FM_THREADS, FM_SMEM, st>>>(p);
    NQS_CUDA(cudaGetLastError());
    NQS_CUDA(cudaFreeAsync(tp, st));
    NQS_CUDA(cudaFreeAsync(cb, st));
    NQS_CUDA(cudaFreeAsync(stats, st));
    NQS_CUDA(cudaFreeAsync(gexp, st));
    NQS_CUDA(cudaFreeAsync(A_packed, st));
    NQS_CUDA(cudaFreeAsync(B_packed, st));
    return NQS_OK;
}

extern "C" int nqs_forces(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                          const nqs_c64* d_b, const nqs_c64* d_W, const nqs_c64* d_eloc, const float* d_weights,
                          nqs_c64* d_F, double* d_stats, void* stream) {
    return forces_impl(d_spins, B, N, M, d_a, d_b, d_W, d_eloc, d_weights, d_F, d_stats, stream, nullptr);
}

// One VMC evaluation step: E_loc, its statistics and the force vector of the same batch, with
// theta / tanh(theta) computed once and shared by the two halves.
extern "C" int nqs_local_energy_forces_h(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M,
                                         const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W,
                                         const float* d_weights, nqs_c64* d_eloc, nqs_c64* d_logpsi, nqs_c64* d_F,
                                         double* d_stats, void* stream) {
    if (B <= 0 || !d_F) return fail(NQS_ERR_INVALID_ARG, "nqs_local_energy_forces_h: B <= 0 or NULL d_F");
    float4* tp = nullptr;
    int rc = local_energy_impl(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream, &tp);
    if (rc) return rc;
    return forces_impl(d_spins, B, h->hc.N, M, d_a, d_b, d_W, d_eloc, d_weights, d_F, d_stats, stream, tp);
}

// ----------------------------------------------------------------------------------------
// Metropolis chains
// ----------------------------------------------------------------------------------------
template <int CPB>
static int launch_metropolis_t(const MetroParams& p, size_t smem, cudaStream_t st) {
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        NQS_CUDA(cudaFuncSetAttribute(metropolis_kernel<CPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_smem = smem;
    }
    metropolis_kernel<CPB><<<(unsigned)((p.C + CPB - 1) / CPB), CPB * 32, smem, st>>>(p);
    NQS_CUDA(cudaGetLastError());
    return NQS_OK;
}

extern "C" int nqs_metropolis(int8_t* d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64* d_a,
                              const nqs_c64* d_b, const nqs_c64* d_W, int32_t S, const int32_t* d_sites,
                              const float* d_u, int32_t* d_accepted, void* stream) {
    int rc = check_common(d_spins, C, N, M, d_a, d_b, d_W);
    if (rc) return rc;
    if (S < 0 || (S > 0 && C > 0 && (!d_sites || !d_u))) return fail(NQS_ERR_INVALID_ARG, "nqs_metropolis: S < 0 or NULL sites / u");
    if ((rc = check_device())) return rc;
    if (C == 0) return NQS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const int M_pad = (int)round_up(M, KJ);
    const long long C_pad = round_up(C, 256);
    const long long nPairsPad = C_pad / 2;
    int cpb = 16;
    while (cpb > 2 && metropolis_smem_bytes(cpb, N, M_pad) > 220 * 1024) cpb >>= 1;
    const size_t smem = metropolis_smem_bytes(cpb, N, M_pad);
    if (smem > 220 * 1024) return fail(NQS_ERR_UNSUPPORTED, "nqs_metropolis: M too large for the shared-memory chain state");

    float4 *tp = nullptr, *Gp = nullptr, *Gm = nullptr;
    float* lk2 = nullptr;
    NQS_CUDA(cudaMallocAsync(&tp, sizeof(float4) * (size_t)M_pad * nPairsPad, st));
    NQS_CUDA(cudaMallocAsync(&Gp, sizeof(float4) * (size_t)N * (M_pad / 2), st));
    NQS_CUDA(cudaMallocAsync(&Gm, sizeof(float4) * (size_t)N * (M_pad / 2), st));
    NQS_CUDA(cudaMallocAsync(&lk2, sizeof(float) * (size_t)N, st));
    site_table_kernel<<<(unsigned)N, 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad, Gp, Gm, lk2);
    NQS_CUDA(cudaGetLastError());
    MetroParams p;
    p.spins = d_spins;
    p.C = C;
    p.N = N;
    p.M = M;
    p.M_pad = M_pad;
    p.tp = tp;
    p.nPairsPad = nPairsPad;
    p.Gp = Gp;
    p.Gm = Gm;
    p.lk2 = lk2;
    p.accepted = d_accepted;
    // chunks of two sweeps; tanh(theta) is recomputed from the current spins before each chunk
    const int chunk = 2 * N;
    for (int s0 = 0; s0 == 0 || s0 < S; s0 += chunk) {
        if ((rc = launch_theta(d_spins, C, N, M, M_pad, d_a, d_b, d_W, tp, nPairsPad, nullptr, st, true))) return rc;
        p.S = S - s0 < chunk ? S - s0 : chunk;
        p.sites = d_sites + (long long)s0 * C;
        p.u = d_u + (long long)s0 * C;
        p.accumulate = s0 > 0;
        switch (cpb) {
            case 16: rc = launch_metropolis_t<16>(p, smem, st); break;
            case 8: rc = launch_metropolis_t<8>(p, smem, st); break;
            case 4: rc = launch_metropolis_t<4>(p, smem, st); break;
            default: rc = launch_metropolis_t<2>(p, smem, st); break;
        }
        if (rc) return rc;
    }
    if (rc) return rc;
    NQS_CUDA(cudaFreeAsync(tp, st));
    NQS_CUDA(cudaFreeAsync(Gp, st));
    NQS_CUDA(cudaFreeAsync(Gm, st));
    NQS_CUDA(cudaFreeAsync(lk2, st));
    return NQS_OK;
}
