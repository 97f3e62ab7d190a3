// C ABI of libnqs_b200.so (declared in include/nqs.h): argument checks, workspace, launches.
// Every step of the path runs in the kernels of nqs_kernels.cuh / nqs_series.cuh / nqs_theta_mma.cuh /
// nqs_forces.cuh / nqs_fisher.cuh / nqs_sampler.cuh; there is no CPU fallback.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <list>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/nqs.h"
#include "nqs_hamiltonian.h"
#include "nqs_kernels.cuh"
#include "nqs_fisher.cuh"
#include "nqs_forces.cuh"
#include "nqs_microbench.cuh"
#include "nqs_sampler.cuh"
#include "nqs_series.cuh"
#include "nqs_small.cuh"
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
#define NQS_TRY(expr)              \
    do {                           \
        int rc__ = (expr);         \
        if (rc__) return rc__;     \
    } while (0)

// every kernel launch of the library is counted (bench.py reports the launches of its timed region)
static std::atomic<long long> g_launches{0};
#define NQS_LAUNCHED()                  \
    do {                                \
        NQS_CUDA(cudaGetLastError());   \
        g_launches.fetch_add(1);        \
    } while (0)
extern "C" int nqs_launch_count(int64_t* out) {
    if (!out) return fail(NQS_ERR_INVALID_ARG, "out is NULL");
    *out = g_launches.load();
    return NQS_OK;
}

extern "C" const char* nqs_last_error(void) { return g_err.c_str(); }
extern "C" const char* nqs_version(void) { return "0.2.0 sm_100a"; }

// ----------------------------------------------------------------------------------------
// options (include/nqs.h: nqs_set_option)
// ----------------------------------------------------------------------------------------
static std::atomic<int> g_opt[NQS_OPT_COUNT] = {};
constexpr int HOST_MAX_CHUNKS = 16;  // nqs_local_energy_host
constexpr size_t SMALL_SMEM_MAX = 200 * 1024;  // shared memory of small_eloc_kernel above which the multi-launch path runs
#ifdef NQS_SERIES_TIMELINE
static long long* g_series_timeline = nullptr;
#endif

extern "C" int nqs_set_option(int32_t key, int32_t value) {
    if (key < 0 || key >= NQS_OPT_COUNT) return fail(NQS_ERR_INVALID_ARG, "nqs_set_option: unknown key");
    const int hi = key == NQS_OPT_A5_PATH ? 3 : key == NQS_OPT_HOST_CHUNKS ? HOST_MAX_CHUNKS : 1;  // the others: 0 / 1
    if (value < 0 || value > hi) return fail(NQS_ERR_INVALID_ARG, "nqs_set_option: value out of range");
    g_opt[key].store(value);
    return NQS_OK;
}
extern "C" int nqs_get_option(int32_t key, int32_t* value) {
    if (key < 0 || key >= NQS_OPT_COUNT || !value) return fail(NQS_ERR_INVALID_ARG, "nqs_get_option: bad key / NULL");
    *value = g_opt[key].load();
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// per-device state: a private stream-ordered memory pool for scratch (trimmed by nqs_release),
// a small status block, and the dynamic-shared-memory opt-in of every kernel
// ----------------------------------------------------------------------------------------
constexpr int MAX_DEVICES = 64;
struct DeviceState {
    bool ready = false;
    cudaMemPool_t pool = nullptr;
    int* status = nullptr;  // [4]: guard flag, failed samples, path tag of the last call (1 series, 2 product), -
    int* tags = nullptr;    // [4] constant {0, 1, 2, 3}: device-side source of the path tag
    std::atomic<int> last_tag{0};  // path tag the most recent call enqueued
    std::map<const void*, size_t> smem_optin;
    int sms = 148;  // multiprocessors of the device
    // host-buffer entry points (nqs_local_energy_host): a copy stream, a compute stream and the events between them,
    // made on first use and kept; host_mu serialises those entry points per device
    cudaStream_t host_copy = nullptr, host_comp = nullptr;
    cudaEvent_t host_ev[HOST_MAX_CHUNKS + 1] = {};
    std::mutex host_mu;
    // refusal latches of the automatic a5 path: LATCH_SLOTS records of four ints in pinned, device-mapped host memory,
    // one per live handle, written by series_latch_kernel and read by the host without synchronising; never freed
    // (a kernel of a handle that has since been destroyed may still write its slot: sequence numbers tell the
    // records of the slot's next owner from it)
    int* latch_host = nullptr;
    int* latch_dev = nullptr;
    std::vector<int> latch_free;
};
constexpr int LATCH_SLOTS = 64;
constexpr int LATCH_SKIP0 = 8, LATCH_SKIP_MAX = 64;  // product-form calls after a refusal before the series is probed again
static std::atomic<int> g_latch_seq{0};
static DeviceState g_dev[MAX_DEVICES];
static std::mutex g_dev_mu;

static int device_state(DeviceState** out) {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        cudaGetLastError();
        return fail(NQS_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
    }
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(NQS_ERR_UNSUPPORTED, "device ordinal >= 64");
    std::lock_guard<std::mutex> lk(g_dev_mu);
    DeviceState& D = g_dev[dev];
    if (!D.ready) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        NQS_CUDA(cudaMemPoolCreate(&D.pool, &props));
        unsigned long long thr = ~0ull;  // freed scratch stays in THIS pool until nqs_release() trims it
        NQS_CUDA(cudaMemPoolSetAttribute(D.pool, cudaMemPoolAttrReleaseThreshold, &thr));
        NQS_CUDA(cudaMalloc(&D.status, 8 * sizeof(int)));
        const int init[8] = {0, 0, 0, 0, 0, 1, 2, 3};
        NQS_CUDA(cudaMemcpy(D.status, init, sizeof(init), cudaMemcpyHostToDevice));
        D.tags = D.status + 4;
        NQS_CUDA(cudaHostAlloc((void**)&D.latch_host, LATCH_SLOTS * 4 * sizeof(int), cudaHostAllocMapped));
        memset(D.latch_host, 0, LATCH_SLOTS * 4 * sizeof(int));
        NQS_CUDA(cudaHostGetDevicePointer((void**)&D.latch_dev, D.latch_host, 0));
        for (int k = LATCH_SLOTS - 1; k >= 0; --k) D.latch_free.push_back(k);
        NQS_CUDA(cudaDeviceGetAttribute(&D.sms, cudaDevAttrMultiProcessorCount, dev));
        D.ready = true;
    }
    *out = &D;
    return NQS_OK;
}

// cudaFuncSetAttribute is per device: remember the largest opt-in per (kernel, device)
template <class K>
static int ensure_smem(DeviceState* D, K kernel, size_t bytes) {
    std::lock_guard<std::mutex> lk(g_dev_mu);
    size_t& cur = D->smem_optin[(const void*)kernel];
    if (bytes > cur) {
        NQS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        cur = bytes;
    }
    return NQS_OK;
}

// stream-ordered scratch, returned to the pool on every exit path
struct Scratch {
    cudaStream_t st;
    cudaMemPool_t pool;
    std::vector<void*> ptrs;
    Scratch(DeviceState* D, cudaStream_t s) : st(s), pool(D->pool) {}
    Scratch(const Scratch&) = delete;
    Scratch& operator=(const Scratch&) = delete;
    ~Scratch() {
        for (void* q : ptrs) cudaFreeAsync(q, st);
    }
    template <class T>
    int get(T** out, size_t count) {
        void* q = nullptr;
        const size_t bytes = count * sizeof(T);
        NQS_CUDA(cudaMallocFromPoolAsync(&q, bytes ? bytes : 16, pool, st));
        ptrs.push_back(q);
        *out = static_cast<T*>(q);
        return NQS_OK;
    }
    void adopt(void* q) { ptrs.push_back(q); }
    void disown(void* q) {
        for (auto it = ptrs.begin(); it != ptrs.end(); ++it)
            if (*it == q) {
                ptrs.erase(it);
                return;
            }
    }
};

// ----------------------------------------------------------------------------------------
// handle
// ----------------------------------------------------------------------------------------
struct nqs_hamiltonian {
    HostCompiled hc;
    int device = -1;       // -1: host-only compile
    void* d_blob = nullptr;
    bool pooled = false;   // blob came from the device pool (cache entries): freed in stream order
    // cache entries are shared between streams: `uploaded` marks the end of the stream-ordered upload (a hit on
    // another stream waits for it), `uses` holds one last-use event per stream that has read the blob (the free waits
    // for all of them); beyond MAX_USE_STREAMS streams the free falls back to a synchronising cudaFree
    static constexpr size_t MAX_USE_STREAMS = 16;
    cudaEvent_t uploaded = nullptr;
    mutable std::mutex use_mu;
    mutable std::vector<std::pair<cudaStream_t, cudaEvent_t>> uses;
    mutable bool uses_overflow = false;
    // refusal latch (automatic a5 path): after a call whose series was refused by the guard, the next `skip_left`
    // calls with this handle go straight to the product form, then the series is probed again; the skip length
    // doubles from LATCH_SKIP0 to LATCH_SKIP_MAX while the probes keep failing and resets when one passes
    int latch_slot = -1;  // record in DeviceState::latch_host, -1: none (no latch)
    mutable int seq_first = 0, seq_last = 0, seq_seen = 0, skip_left = 0, skip_len = 8;
    DevHam dev{};
    int C = 0;
    // launch plan (static for the handle): column tiling of the product-form a5 kernel ...
    int WC = 1, WS = 2, TC = 16, nTiles = 1, C_pad = 16;
    // ... and of the tensor-core series kernel: narrow tiles (NB <= 128, all four accumulator ranges in TMEM) and, where
    // that makes fewer tiles and fits in shared memory, wide ones (NB <= 224, two passes; NBw = 0: not available)
    int NB = 16, nNT = 1;
    int NBw = 0, nNTw = 0;
};

static constexpr int KJ = 16;
static constexpr int MAX_WC = 5;

static void plan_tiles(nqs_hamiltonian* h) {
    const int C = (int)h->hc.col_i.size();
    h->C = C;
    const int slices = C > 0 ? (C + 15) / 16 : 1;
    // least padded work divided by the efficiency of the block shape: a CTA has 2 WC warps, and narrow CTAs
    // leave the SM short of warps (per 16-column slice, measured on B200 at config-3 / config-4 shapes;
    // only the ORDER of these numbers matters to the choice)
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
    h->WC = best;
    h->WS = 2;
    h->TC = 16 * best;
    h->nTiles = (slices + best - 1) / best;
    h->C_pad = h->nTiles * h->TC;
    // series kernel: column tiles of NB <= 128 (4 NB TMEM columns), NB a multiple of 16
    h->nNT = C > 0 ? (C + 127) / 128 : 1;
    const int per = C > 0 ? (C + h->nNT - 1) / h->nNT : 16;
    h->NB = (per + 15) / 16 * 16;
    h->NBw = h->nNTw = 0;
    if (C > 128) {
        const int ntw = (C + SR_WIDE_MAX_NB - 1) / SR_WIDE_MAX_NB;
        const int nbw = ((C + ntw - 1) / ntw + 15) / 16 * 16;
        if (ntw < h->nNT && h->hc.N <= SR_MAX_N && series_gemm_smem_bytes(nbw, h->hc.N, true) <= 227 * 1024)
            h->NBw = nbw, h->nNTw = ntw;
    }
}

static int upload(nqs_hamiltonian* h, DeviceState* D, bool pooled, cudaStream_t st) {
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
    std::vector<int32_t> f0(G), f1(G), f2(G), f3(G), first(G), count(G);
    for (int g = 0; g < G; ++g) {
        f0[g] = hc.groups[g].f[0];
        f1[g] = hc.groups[g].f[1];
        f2[g] = hc.groups[g].f[2];
        f3[g] = hc.groups[g].f[3];
        first[g] = hc.groups[g].term_first;
        count[g] = hc.groups[g].term_count;
    }
    std::vector<int32_t> ci(C_pad, 0), ck(C_pad, -1), cp(C_pad, 1), cg(C_pad, -1);
    std::vector<int32_t> cs2(C_pad, -1), cp2(C_pad, 1), cs3(C_pad, -1), cp3(C_pad, 1);
    for (int c = 0; c < h->C; ++c) {
        ci[c] = hc.col_i[c];
        ck[c] = hc.col_k[c];
        cp[c] = hc.col_p[c];
        cs2[c] = hc.col_s2[c];
        cp2[c] = hc.col_p2[c];
        cs3[c] = hc.col_s3[c];
        cp3[c] = hc.col_p3[c];
        cg[c] = hc.col_group[c];
    }
    const size_t o_dz0 = push(hc.diag_z0), o_dz1 = push(hc.diag_z1);
    const size_t o_f0 = push(f0), o_f1 = push(f1), o_first = push(first), o_count = push(count);
    const size_t o_gz0 = push(hc.gt_z0), o_gz1 = push(hc.gt_z1);
    const size_t o_ci = push(ci), o_ck = push(ck), o_cp = push(cp), o_cg = push(cg);
    const size_t o_f2 = push(f2), o_f3 = push(f3);
    const size_t o_cs2 = push(cs2), o_cp2 = push(cp2), o_cs3 = push(cs3), o_cp3 = push(cp3);
    const size_t o_dxo = push(hc.diag_zx_off), o_dx = push(hc.diag_zx), o_gxo = push(hc.gt_zx_off), o_gx = push(hc.gt_zx);
    size_t int_bytes = (ints.size() * sizeof(int) + 15) / 16 * 16;
    std::vector<nqs_c64> cs;
    cs.insert(cs.end(), hc.diag_c.begin(), hc.diag_c.end());
    cs.insert(cs.end(), hc.gt_c.begin(), hc.gt_c.end());
    const size_t total = int_bytes + cs.size() * sizeof(nqs_c64) + 16;
    std::vector<unsigned char> blob(total, 0);
    if (!ints.empty()) memcpy(blob.data(), ints.data(), ints.size() * sizeof(int));
    if (!cs.empty()) memcpy(blob.data() + int_bytes, cs.data(), cs.size() * sizeof(nqs_c64));
    NQS_CUDA(cudaGetDevice(&h->device));
    {
        std::lock_guard<std::mutex> lk(g_dev_mu);
        if (!D->latch_free.empty()) {
            h->latch_slot = D->latch_free.back();
            D->latch_free.pop_back();
        }
    }
    if (pooled) {
        // pageable source: the runtime stages the bytes before cudaMemcpyAsync returns, so `blob` may die
        NQS_CUDA(cudaMallocFromPoolAsync(&h->d_blob, total, D->pool, st));
        h->pooled = true;
        NQS_CUDA(cudaMemcpyAsync(h->d_blob, blob.data(), total, cudaMemcpyHostToDevice, st));
        NQS_CUDA(cudaEventCreateWithFlags(&h->uploaded, cudaEventDisableTiming));
        NQS_CUDA(cudaEventRecord(h->uploaded, st));
    } else {
        NQS_CUDA(cudaMalloc(&h->d_blob, total));
        NQS_CUDA(cudaMemcpy(h->d_blob, blob.data(), total, cudaMemcpyHostToDevice));
    }
    const int* di = reinterpret_cast<const int*>(h->d_blob);
    const float2* dc = reinterpret_cast<const float2*>(reinterpret_cast<const unsigned char*>(h->d_blob) + int_bytes);
    DevHam& Dv = h->dev;
    Dv.N = hc.N;
    Dv.G = G;
    Dv.C = h->C;
    Dv.Td = Td;
    Dv.Tg = Tg;
    Dv.diag_z0 = di + o_dz0;
    Dv.diag_z1 = di + o_dz1;
    Dv.diag_c = dc;
    Dv.grp_f0 = di + o_f0;
    Dv.grp_f1 = di + o_f1;
    Dv.grp_first = di + o_first;
    Dv.grp_count = di + o_count;
    Dv.gt_z0 = di + o_gz0;
    Dv.gt_z1 = di + o_gz1;
    Dv.gt_c = dc + Td;
    Dv.col_i = di + o_ci;
    Dv.col_k = di + o_ck;
    Dv.col_p = di + o_cp;
    Dv.col_group = di + o_cg;
    Dv.grp_f2 = di + o_f2;
    Dv.grp_f3 = di + o_f3;
    Dv.col_s2 = di + o_cs2;
    Dv.col_p2 = di + o_cp2;
    Dv.col_s3 = di + o_cs3;
    Dv.col_p3 = di + o_cp3;
    Dv.has_zx = hc.has_zx ? 1 : 0;
    Dv.diag_zx_off = di + o_dxo;
    Dv.diag_zx = di + o_dx;
    Dv.gt_zx_off = di + o_gxo;
    Dv.gt_zx = di + o_gx;
    return NQS_OK;
}

// frees a handle; pooled blobs are freed in stream order after the most recent use on EVERY stream that read them
static void destroy_handle(nqs_hamiltonian* h) {
    if (!h) return;
    int cur = -1;
    const bool switch_dev = h->device >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != h->device;
    if (switch_dev) cudaSetDevice(h->device);  // an evicted entry may belong to another device than the caller's
    if (h->d_blob) {
        if (h->pooled && !h->uses_overflow) {
            if (h->uploaded) cudaStreamWaitEvent(nullptr, h->uploaded, 0);
            for (auto& u : h->uses) cudaStreamWaitEvent(nullptr, u.second, 0);
            cudaFreeAsync(h->d_blob, nullptr);
        } else {
            cudaFree(h->d_blob);  // waits for the device: kernels still reading the blob finish first
        }
    }
    if (h->uploaded) cudaEventDestroy(h->uploaded);
    for (auto& u : h->uses) cudaEventDestroy(u.second);
    if (h->latch_slot >= 0 && h->device >= 0 && h->device < MAX_DEVICES) {
        std::lock_guard<std::mutex> lk(g_dev_mu);
        g_dev[h->device].latch_free.insert(g_dev[h->device].latch_free.begin(), h->latch_slot);  // reused last
    }
    if (switch_dev) cudaSetDevice(cur);
    delete h;
}

// mode 0 host only, 1 blocking upload (user handle), 2 pooled, stream-ordered upload (cache entry)
static int create_impl(int32_t N, int32_t T, int32_t K, const int32_t* s, const uint8_t* p, const nqs_c64* c, int mode,
                       cudaStream_t st, nqs_hamiltonian** out) {
    if (!out) return fail(NQS_ERR_INVALID_ARG, "nqs_hamiltonian_create: out is NULL");
    *out = nullptr;
    auto* h = new nqs_hamiltonian();
    std::string err;
    int rc = compile_hamiltonian(N, T, K, s, p, c, h->hc, err);
    if (rc != NQS_OK) {
        delete h;
        return fail(rc, err);
    }
    plan_tiles(h);
    if (mode != 0) {
        DeviceState* D = nullptr;
        rc = device_state(&D);
        if (rc == NQS_OK) rc = upload(h, D, mode == 2, st);
        if (rc != NQS_OK) {
            destroy_handle(h);
            return rc;
        }
    }
    *out = h;
    return NQS_OK;
}

extern "C" int nqs_hamiltonian_create(int32_t N, int32_t T, const int32_t* h_sites, const uint8_t* h_paulis,
                                      const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, 2, h_sites, h_paulis, h_coeffs, 1, nullptr, out);
}
extern "C" int nqs_hamiltonian_compile_host(int32_t N, int32_t T, const int32_t* h_sites, const uint8_t* h_paulis,
                                            const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, 2, h_sites, h_paulis, h_coeffs, 0, nullptr, out);
}
extern "C" int nqs_hamiltonian_create_k(int32_t N, int32_t T, int32_t K, const int32_t* h_sites, const uint8_t* h_paulis,
                                        const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, K, h_sites, h_paulis, h_coeffs, 1, nullptr, out);
}
extern "C" int nqs_hamiltonian_compile_host_k(int32_t N, int32_t T, int32_t K, const int32_t* h_sites,
                                              const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_hamiltonian** out) {
    return create_impl(N, T, K, h_sites, h_paulis, h_coeffs, 0, nullptr, out);
}
extern "C" int nqs_hamiltonian_destroy(nqs_hamiltonian* h) {
    destroy_handle(h);
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
            flip_sites[2 * g] = h->hc.groups[g].f[0];
            flip_sites[2 * g + 1] = h->hc.groups[g].f[1];
        }
    return NQS_OK;
}
extern "C" int nqs_hamiltonian_info_k(const nqs_hamiltonian* h, int32_t info[5], int32_t* flip_sites4) {
    NQS_TRY(nqs_hamiltonian_info(h, info, nullptr));
    if (flip_sites4)
        for (size_t g = 0; g < h->hc.groups.size(); ++g)
            for (int q = 0; q < 4; ++q) flip_sites4[4 * g + q] = h->hc.groups[g].f[q];
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// cache of compiled Hamiltonians for the term-list entry points.  Entries are reference counted: a
// call holds its entry for as long as it enqueues work, eviction and nqs_release() only drop the
// cache's own reference, and the device blob is freed in stream order (never a device synchronise).
// ----------------------------------------------------------------------------------------
using HamRef = std::shared_ptr<nqs_hamiltonian>;
struct CacheEntry {
    int device, N, T, K;
    std::vector<unsigned char> key;
    HamRef h;
};
static std::mutex g_cache_mu;
static std::list<CacheEntry> g_cache;

static int cached_hamiltonian(int32_t N, int32_t T, int32_t K, const int32_t* s, const uint8_t* p, const nqs_c64* c,
                              cudaStream_t st, HamRef* out) {
    if (T < 0 || K < 1 || K > HAM_MAX_SLOTS || (T > 0 && (!s || !p || !c)))
        return fail(NQS_ERR_INVALID_ARG, "term arrays are NULL, T < 0 or K outside 1..8");
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    std::vector<unsigned char> key((size_t)T * (4 * K + K + 8));
    if (T > 0) {
        memcpy(key.data(), s, (size_t)T * 4 * K);
        memcpy(key.data() + (size_t)T * 4 * K, p, (size_t)T * K);
        memcpy(key.data() + (size_t)T * 5 * K, c, (size_t)T * 8);
    }
    std::lock_guard<std::mutex> lk(g_cache_mu);
    for (auto it = g_cache.begin(); it != g_cache.end(); ++it)
        if (it->device == dev && it->N == N && it->T == T && it->K == K && it->key == key) {
            g_cache.splice(g_cache.begin(), g_cache, it);
            *out = g_cache.front().h;
            // the blob was uploaded in the order of the stream that missed: any other stream waits for that copy
            // (no cost when `st` is that stream or the copy has long finished)
            if ((*out)->uploaded) NQS_CUDA(cudaStreamWaitEvent(st, (*out)->uploaded, 0));
            return NQS_OK;
        }
    nqs_hamiltonian* h = nullptr;
    NQS_TRY(create_impl(N, T, K, s, p, c, 2, st, &h));
    HamRef ref(h, destroy_handle);
    g_cache.push_front(CacheEntry{dev, N, T, K, std::move(key), ref});
    if (g_cache.size() > 8) g_cache.pop_back();  // the blob goes when the last holder lets go
    *out = ref;
    return NQS_OK;
}

// records that work reading the blob has been enqueued on `st` (one event per stream, re-recorded at every use)
static void mark_use(const nqs_hamiltonian* h, cudaStream_t st) {
    if (!h->pooled) return;  // user handles are freed with a synchronising cudaFree
    std::lock_guard<std::mutex> lk(h->use_mu);
    if (h->uses_overflow) return;
    for (auto& u : h->uses)
        if (u.first == st) {
            cudaEventRecord(u.second, st);
            return;
        }
    cudaEvent_t ev = nullptr;
    if (h->uses.size() >= nqs_hamiltonian::MAX_USE_STREAMS ||
        cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) {
        h->uses_overflow = true;
        return;
    }
    cudaEventRecord(ev, st);
    h->uses.emplace_back(st, ev);
}

extern "C" int nqs_release(void) {
    {
        std::lock_guard<std::mutex> lk(g_cache_mu);
        g_cache.clear();
    }
    std::lock_guard<std::mutex> lk(g_dev_mu);
    for (int d = 0; d < MAX_DEVICES; ++d)
        if (g_dev[d].ready) cudaMemPoolTrimTo(g_dev[d].pool, 0);
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// optional per-kernel timing (bench.py's roofline leg): CUDA events recorded on the caller's
// stream around the kernels of the most recent nqs_local_energy* call
// ----------------------------------------------------------------------------------------
static bool g_prof_on = false;
static cudaEvent_t g_prof_ev[NQS_PROFILE_SEGMENTS + 1] = {};
static bool g_prof_valid = false;

extern "C" int nqs_profile_enable(int on) {
    if (on && !g_prof_ev[0])
        for (auto& e : g_prof_ev) NQS_CUDA(cudaEventCreate(&e));
    g_prof_on = on != 0;
    g_prof_valid = false;
    return NQS_OK;
}
extern "C" int nqs_profile_last(float ms[NQS_PROFILE_SEGMENTS]) {
    if (!ms) return fail(NQS_ERR_INVALID_ARG, "ms is NULL");
    if (!g_prof_valid) return fail(NQS_ERR_INVALID_ARG, "no profiled call recorded");
    NQS_CUDA(cudaEventSynchronize(g_prof_ev[NQS_PROFILE_SEGMENTS]));
    for (int k = 0; k < NQS_PROFILE_SEGMENTS; ++k)
        NQS_CUDA(cudaEventElapsedTime(&ms[k], g_prof_ev[k], g_prof_ev[k + 1]));
    return NQS_OK;
}
#define NQS_PROF(k, st)                                            \
    do {                                                           \
        if (g_prof_on) NQS_CUDA(cudaEventRecord(g_prof_ev[k], st)); \
    } while (0)

// ----------------------------------------------------------------------------------------
// argument checks, NQS_VALIDATE
// ----------------------------------------------------------------------------------------
static inline long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }

static int check_common(const void* spins, int64_t B, int32_t N, int32_t M, const void* a, const void* b,
                        const void* W) {
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "B < 0");
    if (N <= 0 || M <= 0) return fail(NQS_ERR_INVALID_ARG, "N and M must be positive");
    if (B > 0 && (!spins || !a || !b || !W)) return fail(NQS_ERR_INVALID_ARG, "NULL spins/parameter pointer");
    if ((long long)B * N > (1ll << 40)) return fail(NQS_ERR_UNSUPPORTED, "B*N too large");
    if (B > (1ll << 31)) return fail(NQS_ERR_UNSUPPORTED, "B > 2^31");
    return NQS_OK;
}

__global__ void validate_spins_kernel(const int8_t* __restrict__ spins, long long total, int* __restrict__ bad) {
    int n = 0;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int v = spins[idx];
        n += (v != 1 && v != -1);
    }
    if (n) atomicAdd(bad, n);
}

// NQS_VALIDATE=1 (environment, read at every call): every spin must be +1 or -1.  Debug mode: the check
// synchronises `stream`.
static int validate_spins(DeviceState* D, const int8_t* d_spins, int64_t B, int32_t N, cudaStream_t st) {
    const char* e = getenv("NQS_VALIDATE");
    if (!e || e[0] != '1' || B == 0) return NQS_OK;
    Scratch S(D, st);
    int* bad = nullptr;
    NQS_TRY(S.get(&bad, 1));
    NQS_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), st));
    const long long total = (long long)B * N;
    const unsigned grid = (unsigned)((total + 255) / 256 < D->sms * 8 ? (total + 255) / 256 : D->sms * 8);
    validate_spins_kernel<<<grid, 256, 0, st>>>(d_spins, total, bad);
    NQS_LAUNCHED();
    int h_bad = 0;
    NQS_CUDA(cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    NQS_CUDA(cudaStreamSynchronize(st));
    if (h_bad)
        return fail(NQS_ERR_INVALID_ARG, "NQS_VALIDATE: " + std::to_string(h_bad) + " spin values other than +1/-1");
    return NQS_OK;
}

// ----------------------------------------------------------------------------------------
// a2 / a3 launches
// ----------------------------------------------------------------------------------------
// what one pass of the theta kernel writes
struct ThetaOut {
    float4* tp = nullptr;        // tanh(theta) (or theta itself with raw) as [M_pad][nPairsPad] pair records
    nqs_c64* logpsi = nullptr;   // [B]
    bool raw = false;
    uint4* sA = nullptr;         // series operand planes (tensor-core kernel only), with rown / rowmax
    bool sA_wide = false;        // their layout (series_plane_index)
    float4* rown = nullptr;
    float* rowmax = nullptr;
    const int* gate = nullptr;   // device word: run only if (gate[0] & 1)
    int S = 1;                   // tensor-core kernel, series path: hidden-unit tiles of a sample tile split over S CTAs
    double2* lp_part = nullptr;  // [S][rows] partial log psi (S > 1)
};

// how many CTAs share the hidden units of one sample tile: the split that needs the fewest waves of the 2 x SMs CTA slots
// (each extra CTA reloads the tile's spins and pays its own set-up: ~3 % per split)
static int theta_split(long long nMT, int nNT, int sms) {
    int best = 1;
    double best_cost = 1e30;
    for (int S = 1; S <= 8 && nNT / S >= 4; S *= 2) {
        const long long waves = (nMT * S + 2ll * sms - 1) / (2ll * sms);
        const double cost = (double)waves / S * (1.0 + 0.03 * (S - 1));
        if (cost < best_cost - 1e-9) best_cost = cost, best = S;
    }
    return best;
}

static int launch_theta_simt(DeviceState* D, const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad,
                             const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, long long nPairsPad,
                             const ThetaOut& o, cudaStream_t st) {
    const long long rows = o.tp ? nPairsPad * 2 : B;
    const unsigned grid = (unsigned)((rows + 63) / 64);
    NQS_TRY(ensure_smem(D, theta_kernel, TH_SMEM));
    theta_kernel<<<grid, 256, TH_SMEM, st>>>(d_spins, (long long)B, N, M, M_pad, (const float2*)d_a, (const float2*)d_b,
                                             (const float2*)d_W, o.tp, nPairsPad, (float2*)o.logpsi, o.raw ? 1 : 0,
                                             o.gate);
    NQS_LAUNCHED();
    return NQS_OK;
}

// a2 on the tensor cores: pack spins and the int8 digits of W, then theta_mma_kernel (tcgen05); all three
// kernels honour o.gate.
static int launch_theta_mma(DeviceState* D, const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad,
                            const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, long long nPairsPad,
                            const ThetaOut& o, cudaStream_t st) {
    const long long rows = (o.tp || o.sA) ? nPairsPad * 2 : B;
    const long long nMT = (rows + TM_M - 1) / TM_M;
    const int K_pad = (int)round_up(N, TM_KC), K16 = K_pad / 16;
    const int nNT = (M_pad + TH_JT - 1) / TH_JT;
    Scratch S(D, st);
    uint4 *A_packed = nullptr, *B_packed = nullptr;
    float* scale = nullptr;
    NQS_TRY(S.get(&A_packed, (size_t)nMT * K16 * TM_M));
    NQS_TRY(S.get(&B_packed, (size_t)nNT * K16 * TH_N));
    NQS_TRY(S.get(&scale, (size_t)nNT * TH_JT));
    const long long a_items = nMT * K16 * TM_M;
    const unsigned agrid = (unsigned)((a_items + 255) / 256 < D->sms * 16 ? (a_items + 255) / 256 : D->sms * 16);
    pack_spins_kernel<<<agrid, 256, 0, st>>>(d_spins, (long long)B, N, K16, nMT, A_packed, o.gate);
    NQS_LAUNCHED();
    pack_w_kernel<<<(unsigned)(nNT * TH_JT), 128, 0, st>>>((const float2*)d_W, N, M, K16, B_packed, scale, o.gate);
    NQS_LAUNCHED();
    const size_t smem = theta_mma_smem_bytes(K_pad);
    NQS_TRY(ensure_smem(D, theta_mma_kernel, smem));
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
    p.nPairsPad = nPairsPad;
    p.tp = o.tp;
    p.logpsi = (float2*)o.logpsi;
    p.raw_theta = o.raw ? 1 : 0;
    p.sA = o.sA;
    p.sA_wide = o.sA_wide ? 1 : 0;
    p.sA_tiles = nMT;
    p.rown = o.rown;
    p.rowmax = o.rowmax;
    p.gate = o.gate;
    p.S = o.S;
    p.lp_part = o.lp_part;
    p.rows = nMT * TM_M;
    theta_mma_kernel<<<(unsigned)(nMT * o.S), TM_THREADS, smem, st>>>(p);
    NQS_LAUNCHED();
    return NQS_OK;
}

// the tensor-core kernel covers N <= 512; NQS_OPT_THETA_PATH = 1 forces the FP32 SIMT kernel
static bool theta_use_mma(int32_t N) {
    return g_opt[NQS_OPT_THETA_PATH].load() == 0 && round_up(N, TM_KC) <= TM_MAX_KPAD;
}

static int launch_theta(DeviceState* D, const int8_t* d_spins, int64_t B, int32_t N, int32_t M, int M_pad,
                        const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, long long nPairsPad,
                        const ThetaOut& o, cudaStream_t st) {
    if (theta_use_mma(N)) return launch_theta_mma(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st);
    if (o.sA) return fail(NQS_ERR_UNSUPPORTED, "series planes need the tensor-core theta kernel");
    return launch_theta_simt(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st);
}

template <int WC, int WS>
static int launch_eloc_t(DeviceState* D, const ElocParams& p, long long nBlocksY, cudaStream_t st) {
    using Cfg = ElocCfg<WC, WS, KJ>;
    NQS_TRY(ensure_smem(D, eloc_kernel<WC, WS, KJ>, Cfg::SMEM));
    const long long blocks = (long long)p.nTiles * nBlocksY;
    if (blocks > 0x7fffffffll) return fail(NQS_ERR_UNSUPPORTED, "B x column tiles exceeds the grid limit");
    eloc_kernel<WC, WS, KJ><<<(unsigned)blocks, Cfg::NT, Cfg::SMEM, st>>>(p);
    NQS_LAUNCHED();
    return NQS_OK;
}

static int launch_eloc(DeviceState* D, const nqs_hamiltonian* h, const ElocParams& p, long long B_pad, cudaStream_t st) {
    const long long nby = B_pad / (32 * h->WS);
    switch (h->WC) {
        case 1: return launch_eloc_t<1, 2>(D, p, nby, st);
        case 2: return launch_eloc_t<2, 2>(D, p, nby, st);
        case 3: return launch_eloc_t<3, 2>(D, p, nby, st);
        case 4: return launch_eloc_t<4, 2>(D, p, nby, st);
        case 5: return launch_eloc_t<5, 2>(D, p, nby, st);
    }
    return fail(NQS_ERR_UNSUPPORTED, "unsupported column tiling");
}

extern "C" int nqs_log_psi(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                           const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_logpsi, void* stream) {
    NQS_TRY(check_common(d_spins, B, N, M, d_a, d_b, d_W));
    if (B > 0 && !d_logpsi) return fail(NQS_ERR_INVALID_ARG, "d_logpsi is NULL");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (B == 0) return NQS_OK;
    NQS_TRY(validate_spins(D, d_spins, B, N, (cudaStream_t)stream));
    ThetaOut o;
    o.logpsi = d_logpsi;
    return launch_theta(D, d_spins, B, N, M, (int)round_up(M, KJ), d_a, d_b, d_W, 0, o, (cudaStream_t)stream);
}

// ----------------------------------------------------------------------------------------
// a1 .. a6.  a5 runs on the tensor cores as a guarded series (nqs_series.cuh) when the problem is large
// enough to pay for its operand packing, with the FP32 product form behind it: eloc_kernel and
// finalize_kernel are always enqueued and return at once unless the guard raised status[0].
// keep_tp != NULL: tanh(theta) ([M_pad][B_pad/2] float4) is handed to `keeper` instead of being
// released when this function returns -- nqs_local_energy_forces_h.
// ----------------------------------------------------------------------------------------
static int local_energy_impl(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M,
                             const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_eloc,
                             nqs_c64* d_logpsi, void* stream, float4** keep_tp, Scratch* keeper) {
    if (!h) return fail(NQS_ERR_INVALID_ARG, "hamiltonian handle is NULL");
    const int N = h->hc.N;
    NQS_TRY(check_common(d_spins, B, N, M, d_a, d_b, d_W));
    if (B > 0 && !d_eloc) return fail(NQS_ERR_INVALID_ARG, "d_eloc is NULL");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (h->device < 0) return fail(NQS_ERR_INVALID_ARG, "handle was compiled host-only (nqs_hamiltonian_compile_host)");
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    if (dev != h->device) return fail(NQS_ERR_INVALID_ARG, "handle belongs to another device");
    if (B == 0) return NQS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    NQS_TRY(validate_spins(D, d_spins, B, N, st));

    const int M_pad = (int)round_up(M, KJ);
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;
    const int nTiles = h->nTiles, TC = h->TC, C_pad = h->C_pad;
    const bool have_cols = h->C > 0;

    // which a5 path: 0 auto, 1 product form only, 2 series + guard + fallback at any size, 3 series only
    const int opt = g_opt[NQS_OPT_A5_PATH].load();
    const bool series_ok = have_cols && N <= SR_MAX_N && series_gemm_smem_bytes(h->NB, N) <= 227 * 1024;
    const bool big = (double)B * h->C * M >= 268435456.0;  // 2^28 (sample, column, hidden unit) triples
    bool use_series = series_ok && (opt == 2 || opt == 3 || (opt == 0 && big));  // the refusal latch below may clear it
    const bool use_product = have_cols && !(use_series && opt == 3);

    // small problems: a1 .. a6 in one launch (nqs_small.cuh) when the tables of a CTA fit in shared memory
    if (opt == 0 && !use_series && !keep_tp && g_opt[NQS_OPT_SMALL_PATH].load() == 0) {
        if (small_smem_bytes(N, M, h->C, 4) <= SMALL_SMEM_MAX) {
            // samples per CTA: the batch spread over a whole number of waves of one CTA per SM, as far as the CTA's
            // shared memory allows
            int SB = 4;
            for (int waves = 1;; ++waves) {
                SB = (int)round_up((B + (long long)D->sms * waves - 1) / ((long long)D->sms * waves), 4);
                if (SB <= SM_MAX_SB && small_smem_bytes(N, M, h->C, SB) <= SMALL_SMEM_MAX) break;
            }
            const size_t smem = small_smem_bytes(N, M, h->C, SB);
            NQS_TRY(ensure_smem(D, small_eloc_kernel, smem));
            SmallParams sp;
            sp.spins = d_spins;
            sp.B = B;
            sp.N = N;
            sp.M = M;
            sp.C = h->C;
            sp.a = (const float2*)d_a;
            sp.b = (const float2*)d_b;
            sp.W = (const float2*)d_W;
            sp.H = h->dev;
            sp.eloc = (float2*)d_eloc;
            sp.logpsi = (float2*)d_logpsi;
            sp.SB = SB;
            const long long blocks = (B + SB - 1) / SB;
            if (blocks > 0x7fffffffll) return fail(NQS_ERR_UNSUPPORTED, "B exceeds the grid limit");
            for (int k = 0; k <= 5; ++k) NQS_PROF(k, st);
            small_eloc_kernel<<<(unsigned)blocks, small_threads(h->C, SB), smem, st>>>(sp);
            NQS_LAUNCHED();
            NQS_PROF(6, st);
            if (D->last_tag.exchange(3) != 3) {
                NQS_CUDA(cudaMemsetAsync(D->status, 0, 2 * sizeof(int), st));
                NQS_CUDA(cudaMemcpyAsync(D->status + 2, D->tags + 3, sizeof(int), cudaMemcpyDeviceToDevice, st));
            }
            NQS_PROF(7, st);
            g_prof_valid = g_prof_on;
            mark_use(h, st);
            return NQS_OK;
        }
    }

    // refusal latch (automatic mode only): what the most recent finished series attempt of this handle reported is
    // read from pinned memory -- no synchronisation, so it may lag by the calls still in flight.  A refusal sends the
    // next skip_len calls to the product form alone (no series operands, no GEMM, no guard); then one call probes again.
    int latch_seq = 0;
    volatile int* latch_rec = nullptr;
    if (opt == 0 && use_series && h->latch_slot >= 0 && g_opt[NQS_OPT_SERIES_LATCH].load() == 0) {
        std::lock_guard<std::mutex> lk(h->use_mu);
        volatile int* L = D->latch_host + 4 * h->latch_slot;
        const int seq = L[0];
        const int flag = L[1];
        const bool own = h->seq_first != 0 && (unsigned)(seq - h->seq_first) <= (unsigned)(h->seq_last - h->seq_first);
        if (own && seq != h->seq_seen) {
            h->seq_seen = seq;
            if (flag) {
                h->skip_left = h->skip_len;
                h->skip_len = h->skip_len * 2 < LATCH_SKIP_MAX ? h->skip_len * 2 : LATCH_SKIP_MAX;
            } else {
                h->skip_left = 0;
                h->skip_len = LATCH_SKIP0;
            }
        }
        if (h->skip_left > 0) {
            --h->skip_left;
            use_series = false;
        } else {
            latch_seq = g_latch_seq.fetch_add(1) + 1;
            if (latch_seq == 0) latch_seq = g_latch_seq.fetch_add(1) + 1;  // 0 means "none"
            if (!h->seq_first) h->seq_first = latch_seq;
            h->seq_last = latch_seq;
            latch_rec = D->latch_dev + 4 * h->latch_slot;
        }
    }

    // the tensor-core theta kernel writes the series planes itself; tanh(theta) is then only needed by the
    // product form (in a gated second pass if the guard fails) or by the caller (keep_tp)
    const bool fused_pack = use_series && theta_use_mma(N);
    Scratch S(D, st);
    float4 *tp = nullptr, *tab = nullptr, *rho = nullptr;
    float2* partial = nullptr;
    if (use_product || keep_tp || (use_series && !fused_pack)) NQS_TRY(S.get(&tp, (size_t)M_pad * nPairsPad));
    NQS_PROF(0, st);
    if (use_product) {
        NQS_TRY(S.get(&tab, (size_t)nTiles * M_pad * TC));
        NQS_TRY(S.get(&rho, (size_t)C_pad));
        NQS_TRY(S.get(&partial, (size_t)B * nTiles));
    }
    // series operands that do not depend on the samples
    const bool wide = use_series && h->NBw > 0 && g_opt[NQS_OPT_SERIES_WIDE].load() != 1;
    const int NB = wide ? h->NBw : h->NB, nNT = wide ? h->nNTw : h->nNT, nJC = M_pad / 16;
    uint4 *sA = nullptr, *sB = nullptr;
    SeriesCol* scols = nullptr;
    SeriesTerms* sterms = nullptr;
    float4 *rown = nullptr, *spartial = nullptr;
    float* rowmax = nullptr;
    double2* lp_part = nullptr;
    int nS = 1;
    int* status = nullptr;
    if (use_series) {
        NQS_TRY(S.get(&sA, (size_t)(B_pad / SR_M) * nJC * SR_PLANES * SR_A_PLANE_U4));
        NQS_TRY(S.get(&sB, (size_t)nNT * nJC * SR_PLANES * 2 * NB));
        NQS_TRY(S.get(&scols, (size_t)nNT * NB));
        NQS_TRY(S.get(&sterms, (size_t)nNT * NB));
        nS = fused_pack && !keep_tp && g_opt[NQS_OPT_THETA_SPLIT].load() != 1 ? theta_split(B_pad / TM_M, M_pad / TH_JT, D->sms) : 1;
        NQS_TRY(S.get(&rown, (size_t)B_pad * nS));
        NQS_TRY(S.get(&rowmax, (size_t)B_pad * nS));
        if (nS > 1 && d_logpsi) NQS_TRY(S.get(&lp_part, (size_t)B_pad * nS));
        NQS_TRY(S.get(&spartial, (size_t)B * nNT));
        NQS_TRY(S.get(&status, 4));
        NQS_CUDA(cudaMemsetAsync(status, 0, 4 * sizeof(int), st));
        series_table_kernel<<<(unsigned)(nNT * NB), 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad,
                                                                  h->C, NB, h->dev, sB, wide ? 1 : 0, scols,
                                                                  sterms);
        NQS_LAUNCHED();
    }
    NQS_PROF(1, st);
    // tanh(theta) itself: now if the caller keeps it or the product form runs unconditionally; with the fused
    // series planes it is otherwise produced only in the gated second pass after the guard
    const bool tp_now = keep_tp || !use_series || !fused_pack;
    if (have_cols || d_logpsi || keep_tp) {
        ThetaOut o;
        o.logpsi = d_logpsi;
        o.tp = tp_now ? tp : nullptr;
        if (fused_pack) o.sA = sA, o.rown = rown, o.rowmax = rowmax, o.S = nS, o.lp_part = lp_part, o.sA_wide = wide;
        NQS_TRY(launch_theta(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
    }
    NQS_PROF(2, st);
    if (use_series && !fused_pack) {
        series_pack_kernel<<<(unsigned)(B_pad / SR_M), 256, 0, st>>>(tp, nPairsPad, M_pad, sA, wide ? 1 : 0, rown,
                                                                             rowmax);
        NQS_LAUNCHED();
    }
    NQS_PROF(3, st);
    if (use_series) {
        const size_t smem = series_gemm_smem_bytes(NB, N, wide);
        if (wide) NQS_TRY(ensure_smem(D, series_gemm_kernel<true>, smem));
        else NQS_TRY(ensure_smem(D, series_gemm_kernel<false>, smem));
        float2* even = nullptr;
        if (wide) NQS_TRY(S.get(&even, (size_t)(B_pad / SR_M) * nNT * NB * SR_M));
        SeriesGemmParams gp;
        gp.A_packed = sA;
        gp.B_packed = sB;
        gp.nMT = B_pad / SR_M;
        gp.cols = scols;
        gp.terms = sterms;
        gp.rown = rown;
        gp.rowmax = rowmax;
        gp.nS = nS;
        gp.rows = B_pad;
        gp.spins = d_spins;
        gp.B = B;
        gp.N = N;
        gp.nJC = nJC;
        gp.NB = NB;
        gp.nNT = nNT;
        gp.H = h->dev;
        gp.partial = spartial;
        gp.even = even;
#ifdef NQS_SERIES_TIMELINE
        gp.timeline = g_series_timeline;
#endif
        const long long blocks = (B_pad / SR_M) * nNT;
        if (blocks > 0x7fffffffll) return fail(NQS_ERR_UNSUPPORTED, "B x column tiles exceeds the grid limit");
        if (wide) series_gemm_kernel<true><<<(unsigned)blocks, SR_THREADS, smem, st>>>(gp);
        else series_gemm_kernel<false><<<(unsigned)blocks, SR_THREADS, smem, st>>>(gp);
        NQS_LAUNCHED();
    }
    NQS_PROF(4, st);
    if (use_series) {
        series_guard_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(spartial, (long long)B, nNT, (float2*)d_eloc,
                                                                         status, lp_part, nS, (long long)B_pad,
                                                                         (float2*)d_logpsi);
        NQS_LAUNCHED();
    }
    NQS_PROF(5, st);
    const int* gate = (use_series && use_product) ? status : nullptr;
    const bool fused_finalize = use_product && !use_series && nTiles == 1;  // eloc_kernel writes E_loc itself
    if (use_product) {  // the product form's tables (behind the series: only if the guard failed)
        const long long total = (long long)M_pad * C_pad;
        const unsigned tgrid = (unsigned)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
        table_kernel<<<tgrid, 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad, h->C, TC, nTiles,
                                            h->dev, tab, rho, gate);
        NQS_LAUNCHED();
    }
    if (use_product && !tp_now) {  // fallback pass: tanh(theta) for the product form, only if the guard failed
        ThetaOut o;
        o.tp = tp;
        o.gate = gate;
        NQS_TRY(launch_theta(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
    }
    if (use_product) {
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
        p.status = gate;
        p.eloc_out = fused_finalize ? (float2*)d_eloc : nullptr;
        NQS_TRY(launch_eloc(D, h, p, B_pad, st));
    }
    NQS_PROF(6, st);
    if ((use_product || !use_series) && !fused_finalize) {
        finalize_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(d_spins, (long long)B, N, h->dev, partial,
                                                                     have_cols ? nTiles : 0, (float2*)d_eloc, gate);
        NQS_LAUNCHED();
    }
    // debug record of the decision (nqs_debug_last_a5): {guard flag, failed samples} of this call, path tag.
    // Product-only calls rewrite it only when the previous call on this device was not one of them.
    if (use_series) {
        series_latch_kernel<<<1, 32, 0, st>>>(status, D->status, latch_rec, latch_seq);
        NQS_LAUNCHED();
        D->last_tag.store(1);
    } else if (D->last_tag.exchange(2) != 2) {
        NQS_CUDA(cudaMemsetAsync(D->status, 0, 2 * sizeof(int), st));
        NQS_CUDA(cudaMemcpyAsync(D->status + 2, D->tags + 2, sizeof(int), cudaMemcpyDeviceToDevice, st));
    }
    NQS_PROF(7, st);
    g_prof_valid = g_prof_on;
    mark_use(h, st);
    if (keep_tp) {
        *keep_tp = tp;
        S.disown(tp);
        keeper->adopt(tp);
    }
    return NQS_OK;
}

#ifdef NQS_SMALL_TIMELINE
// development builds only (NQS_NVCC_FLAGS=-DNQS_SMALL_TIMELINE): clock64 at the phase boundaries of block 0 of the most
// recent small_eloc_kernel (start, W levels done, theta done, tables done, amplitudes done, end)
extern "C" int nqs_debug_small_timeline(long long out[8]) {
    NQS_CUDA(cudaDeviceSynchronize());
    NQS_CUDA(cudaMemcpyFromSymbol(out, g_small_stamps, 8 * sizeof(long long)));
    return NQS_OK;
}
#endif

#ifdef NQS_SERIES_TIMELINE
// development builds only (NQS_NVCC_FLAGS=-DNQS_SERIES_TIMELINE): a device buffer of [blocks][8] int64 that receives
// the clock64 stamps of every series_gemm_kernel block (start, after set-up, after the prologue, accumulators ready,
// epilogue done, end)
extern "C" int nqs_debug_series_timeline(void* d_buf) {
    g_series_timeline = (long long*)d_buf;
    return NQS_OK;
}
#endif

extern "C" int nqs_debug_last_a5(int32_t out[3], void* stream) {
    if (!out) return fail(NQS_ERR_INVALID_ARG, "out is NULL");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    cudaStream_t st = (cudaStream_t)stream;
    int v[3] = {0, 0, 0};
    NQS_CUDA(cudaMemcpyAsync(v, D->status, 3 * sizeof(int), cudaMemcpyDeviceToHost, st));
    NQS_CUDA(cudaStreamSynchronize(st));
    out[0] = v[2];  // 1 = the series path was attempted, 2 = product form only, 3 = the single-launch kernel
    out[1] = v[0];  // 1 = the guard failed (and, unless NQS_OPT_A5_PATH = 3, the product form recomputed the call)
    out[2] = v[1];  // samples whose error bound exceeded the guard threshold
    return NQS_OK;
}

extern "C" int nqs_local_energy_h(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M,
                                  const nqs_c64* d_a, const nqs_c64* d_b, const nqs_c64* d_W, nqs_c64* d_eloc,
                                  nqs_c64* d_logpsi, void* stream) {
    return local_energy_impl(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream, nullptr, nullptr);
}

extern "C" int nqs_local_energy_k(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                                  const nqs_c64* d_b, const nqs_c64* d_W, int32_t T, int32_t K, const int32_t* h_sites,
                                  const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_c64* d_eloc,
                                  nqs_c64* d_logpsi, void* stream) {
    NQS_TRY(check_common(d_spins, B, N, M, d_a, d_b, d_W));
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    HamRef h;
    NQS_TRY(cached_hamiltonian(N, T, K, h_sites, h_paulis, h_coeffs, (cudaStream_t)stream, &h));
    return nqs_local_energy_h(h.get(), d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream);
}

extern "C" int nqs_local_energy(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                                const nqs_c64* d_b, const nqs_c64* d_W, int32_t T, const int32_t* h_sites,
                                const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_c64* d_eloc,
                                nqs_c64* d_logpsi, void* stream) {
    return nqs_local_energy_k(d_spins, B, N, M, d_a, d_b, d_W, T, 2, h_sites, h_paulis, h_coeffs, d_eloc, d_logpsi,
                              stream);
}

static int enumerate_impl(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int8_t* d_sprime,
                          nqs_c64* d_mel, void* stream) {
    if (!h) return fail(NQS_ERR_INVALID_ARG, "hamiltonian handle is NULL");
    if (B < 0 || (B > 0 && (!d_spins || !d_sprime || !d_mel))) return fail(NQS_ERR_INVALID_ARG, "bad arguments");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (h->device < 0) return fail(NQS_ERR_INVALID_ARG, "handle was compiled host-only");
    if (B == 0) return NQS_OK;
    const long long total = (long long)B * (h->dev.G + 1);
    const unsigned grid = (unsigned)((total + 127) / 128 < 65535 ? (total + 127) / 128 : 65535);
    enumerate_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(d_spins, (long long)B, h->hc.N, h->dev, d_sprime,
                                                             (float2*)d_mel);
    NQS_LAUNCHED();
    mark_use(h, (cudaStream_t)stream);
    return NQS_OK;
}

extern "C" int nqs_enumerate_connected_h(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B,
                                         int8_t* d_sprime, nqs_c64* d_mel, void* stream) {
    return enumerate_impl(h, d_spins, B, d_sprime, d_mel, stream);
}

extern "C" int nqs_enumerate_connected(const int8_t* d_spins, int64_t B, int32_t N, int32_t T,
                                       const int32_t* h_sites, const uint8_t* h_paulis, const nqs_c64* h_coeffs,
                                       int8_t* d_sprime, nqs_c64* d_mel, int32_t* G_out, void* stream) {
    if (B < 0 || N <= 0) return fail(NQS_ERR_INVALID_ARG, "nqs_enumerate_connected: B < 0 or N <= 0");
    if (B == 0) {  // sizing call: no device needed
        nqs_hamiltonian* hh = nullptr;
        NQS_TRY(create_impl(N, T, 2, h_sites, h_paulis, h_coeffs, 0, nullptr, &hh));
        if (G_out) *G_out = (int32_t)hh->hc.groups.size();
        destroy_handle(hh);
        return NQS_OK;
    }
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    HamRef h;
    NQS_TRY(cached_hamiltonian(N, T, 2, h_sites, h_paulis, h_coeffs, (cudaStream_t)stream, &h));
    if (G_out) *G_out = (int32_t)h->hc.groups.size();
    return enumerate_impl(h.get(), d_spins, B, d_sprime, d_mel, stream);
}

// ----------------------------------------------------------------------------------------
// host-buffer entry points (end-to-end: H2D, kernels, D2H, synchronise)
// ----------------------------------------------------------------------------------------

// Host buffers in, host buffers out (the end-to-end leg of bench.py).  The batch goes through the device in chunks:
// the parameters and the first chunk of spins are copied, then the kernels of chunk k run on the compute stream while
// the copy stream brings chunk k + 1 -- the transfer of all but the first chunk hides behind the kernels.  Chunks are
// whole waves of the kernels (2 x SMs sample tiles of 128 = 37888 samples on a B200, at least HOST_CHUNK_MIN); every
// sample's result is independent of the chunking except that the series guard decides per chunk.
constexpr int64_t HOST_CHUNK_MIN = 32768;

static int host_streams(DeviceState* D) {
    if (D->host_comp) return NQS_OK;
    NQS_CUDA(cudaStreamCreateWithFlags(&D->host_copy, cudaStreamNonBlocking));
    NQS_CUDA(cudaStreamCreateWithFlags(&D->host_comp, cudaStreamNonBlocking));
    for (int k = 0; k <= HOST_MAX_CHUNKS; ++k) NQS_CUDA(cudaEventCreateWithFlags(&D->host_ev[k], cudaEventDisableTiming));
    return NQS_OK;
}

extern "C" int nqs_local_energy_host(const int8_t* h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* h_a,
                                     const nqs_c64* h_b, const nqs_c64* h_W, int32_t T, const int32_t* h_sites,
                                     const uint8_t* h_paulis, const nqs_c64* h_coeffs, nqs_c64* h_eloc,
                                     nqs_c64* h_logpsi) {
    NQS_TRY(check_common(h_spins, B, N, M, h_a, h_b, h_W));
    if (B > 0 && !h_eloc) return fail(NQS_ERR_INVALID_ARG, "h_eloc is NULL");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    std::lock_guard<std::mutex> host_lock(D->host_mu);
    NQS_TRY(host_streams(D));
    cudaStream_t comp = D->host_comp, copy = D->host_copy;
    HamRef h;
    NQS_TRY(cached_hamiltonian(N, T, 2, h_sites, h_paulis, h_coeffs, comp, &h));
    if (B == 0) return NQS_OK;
    // on every exit: wait for both streams (the scratch below is released in the order of `comp`)
    struct Drain {
        cudaStream_t a, b;
        ~Drain() {
            cudaStreamSynchronize(a);
            cudaStreamSynchronize(b);
        }
    };
    Scratch S(D, comp);
    Drain drain{copy, comp};
    int8_t* ds = nullptr;
    nqs_c64 *da = nullptr, *db = nullptr, *dW = nullptr, *de = nullptr, *dl = nullptr;
    NQS_TRY(S.get(&ds, (size_t)B * N));
    NQS_TRY(S.get(&da, (size_t)N));
    NQS_TRY(S.get(&db, (size_t)M));
    NQS_TRY(S.get(&dW, (size_t)M * N));
    NQS_TRY(S.get(&de, (size_t)B));
    if (h_logpsi) NQS_TRY(S.get(&dl, (size_t)B));
    // chunk boundaries: automatic = whole waves of the kernels -- 2 x SMs sample tiles of 128 fill the CTA slots of the
    // theta kernel exactly once and give the series GEMM a multiple of SMs CTAs whatever the number of column tiles; a
    // short remainder joins the chunk before it.  NQS_OPT_HOST_CHUNKS = n: n equal chunks.
    int64_t start[HOST_MAX_CHUNKS + 1];
    int nChunks = 0;
    const int forced = g_opt[NQS_OPT_HOST_CHUNKS].load();
    if (forced > 0) {
        nChunks = (int)std::min<int64_t>(forced, (B + 255) / 256);
        const int64_t per = round_up((B + nChunks - 1) / nChunks, 256);
        for (int k = 0; k <= nChunks; ++k) start[k] = std::min<int64_t>(B, k * per);
    } else {
        const int64_t unit = std::max<int64_t>(HOST_CHUNK_MIN, 2ll * D->sms * 128);
        start[0] = 0;
        while (nChunks < HOST_MAX_CHUNKS - 1 && B - start[nChunks] >= unit + unit / 4) {
            start[nChunks + 1] = start[nChunks] + unit;
            ++nChunks;
        }
        start[++nChunks] = B;
    }
    // the blocks were allocated in the order of `comp`: the copy stream may touch them after this point of it
    NQS_CUDA(cudaEventRecord(D->host_ev[HOST_MAX_CHUNKS], comp));
    NQS_CUDA(cudaStreamWaitEvent(copy, D->host_ev[HOST_MAX_CHUNKS], 0));
    NQS_CUDA(cudaMemcpyAsync(da, h_a, sizeof(nqs_c64) * N, cudaMemcpyHostToDevice, copy));
    NQS_CUDA(cudaMemcpyAsync(db, h_b, sizeof(nqs_c64) * M, cudaMemcpyHostToDevice, copy));
    NQS_CUDA(cudaMemcpyAsync(dW, h_W, sizeof(nqs_c64) * (size_t)M * N, cudaMemcpyHostToDevice, copy));
    for (int k = 0; k < nChunks; ++k) {
        const int64_t b0 = start[k], nb = start[k + 1] - b0;
        if (nb <= 0) continue;
        NQS_CUDA(cudaMemcpyAsync(ds + b0 * N, h_spins + b0 * N, (size_t)nb * N, cudaMemcpyHostToDevice, copy));
        NQS_CUDA(cudaEventRecord(D->host_ev[k], copy));
    }
    for (int k = 0; k < nChunks; ++k) {
        const int64_t b0 = start[k], nb = start[k + 1] - b0;
        if (nb <= 0) continue;
        NQS_CUDA(cudaStreamWaitEvent(comp, D->host_ev[k], 0));
        NQS_TRY(nqs_local_energy_h(h.get(), ds + b0 * N, nb, M, da, db, dW, de + b0, dl ? dl + b0 : nullptr, comp));
        NQS_CUDA(cudaMemcpyAsync(h_eloc + b0, de + b0, sizeof(nqs_c64) * nb, cudaMemcpyDeviceToHost, comp));
        if (h_logpsi) NQS_CUDA(cudaMemcpyAsync(h_logpsi + b0, dl + b0, sizeof(nqs_c64) * nb, cudaMemcpyDeviceToHost, comp));
    }
    NQS_CUDA(cudaStreamSynchronize(comp));
    return NQS_OK;
}

extern "C" int nqs_log_psi_host(const int8_t* h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* h_a,
                                const nqs_c64* h_b, const nqs_c64* h_W, nqs_c64* h_logpsi) {
    NQS_TRY(check_common(h_spins, B, N, M, h_a, h_b, h_W));
    if (B > 0 && !h_logpsi) return fail(NQS_ERR_INVALID_ARG, "h_logpsi is NULL");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (B == 0) return NQS_OK;
    std::lock_guard<std::mutex> host_lock(D->host_mu);
    NQS_TRY(host_streams(D));
    cudaStream_t st = D->host_comp;
    struct Drain {
        cudaStream_t a;
        ~Drain() { cudaStreamSynchronize(a); }
    };
    Scratch S(D, st);
    Drain drain{st};
    int8_t* ds = nullptr;
    nqs_c64 *da = nullptr, *db = nullptr, *dW = nullptr, *dl = nullptr;
    NQS_TRY(S.get(&ds, (size_t)B * N));
    NQS_TRY(S.get(&da, (size_t)N));
    NQS_TRY(S.get(&db, (size_t)M));
    NQS_TRY(S.get(&dW, (size_t)M * N));
    NQS_TRY(S.get(&dl, (size_t)B));
    NQS_CUDA(cudaMemcpyAsync(ds, h_spins, (size_t)B * N, cudaMemcpyHostToDevice, st));
    NQS_CUDA(cudaMemcpyAsync(da, h_a, sizeof(nqs_c64) * N, cudaMemcpyHostToDevice, st));
    NQS_CUDA(cudaMemcpyAsync(db, h_b, sizeof(nqs_c64) * M, cudaMemcpyHostToDevice, st));
    NQS_CUDA(cudaMemcpyAsync(dW, h_W, sizeof(nqs_c64) * (size_t)M * N, cudaMemcpyHostToDevice, st));
    NQS_TRY(nqs_log_psi(ds, B, N, M, da, db, dW, dl, st));
    NQS_CUDA(cudaMemcpyAsync(h_logpsi, dl, sizeof(nqs_c64) * B, cudaMemcpyDeviceToHost, st));
    NQS_CUDA(cudaStreamSynchronize(st));
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
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
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
        NQS_LAUNCHED();
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
static int launch_stats(DeviceState* D, const nqs_c64* d_x, const float* d_w, int64_t B, double* d_stats,
                        cudaStream_t st) {
    Scratch S(D, st);
    double* partial = nullptr;
    const int nblk = (int)((B + 255) / 256 < ST_BLOCKS ? (B + 255) / 256 : ST_BLOCKS);
    NQS_TRY(S.get(&partial, (size_t)4 * ST_BLOCKS));
    stats_partial_kernel<<<nblk, 256, 0, st>>>((const float2*)d_x, d_w, (long long)B, partial);
    NQS_LAUNCHED();
    stats_final_kernel<<<1, 32, 0, st>>>(partial, nblk, d_stats);
    NQS_LAUNCHED();
    return NQS_OK;
}

extern "C" int nqs_energy_stats(const nqs_c64* d_x, const float* d_weights, int64_t B, double* d_stats,
                                void* stream) {
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "nqs_energy_stats: B < 0");
    if (B == 0) return NQS_OK;
    if (!d_x || !d_stats) return fail(NQS_ERR_INVALID_ARG, "nqs_energy_stats: NULL pointer");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    return launch_stats(D, d_x, d_weights, B, d_stats, (cudaStream_t)stream);
}

// ----------------------------------------------------------------------------------------
// nqs_energy_stats_static (include/nqs.h): the same two kernels as nqs_energy_stats, launched in the same
// geometry, for callers that must not allocate.  The per-block partial sums do not come from the library's pool
// but from the fixed array below, which is part of the loaded module: every device that loads libnqs_b200.so
// holds these 8 KB from module load to process exit, whether or not this entry point is ever called.
//
// In host code `g_stats_static_scratch` is only a handle for the runtime, NOT a device address: handing it to a
// kernel would make the kernel read and write some unrelated location (or fault).  The address the kernels get is
// the one cudaGetSymbolAddress reports for the device that is current, looked up once per device and kept in
// g_stats_static_ptr.  This entry point deliberately stays clear of device_state() (which creates the pool and
// allocates the status block) and of Scratch: it calls no cudaMalloc*, cudaFree* or pool routine.
// ----------------------------------------------------------------------------------------
static __device__ __align__(256) double g_stats_static_scratch[4 * ST_BLOCKS];  // ST_BLOCKS records {sum w, sum w Re x, sum w Im x, sum w |x|^2}
static double* g_stats_static_ptr[MAX_DEVICES] = {};  // device address of the array, per device ordinal (g_stats_static_mu)
static std::mutex g_stats_static_mu;

// Device address of the scratch array on the CURRENT device; the first call per device does the lookup.
static int stats_static_scratch(double** out) {
    int dev = 0;
    NQS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(NQS_ERR_UNSUPPORTED, "device ordinal >= 64");
    std::lock_guard<std::mutex> lk(g_stats_static_mu);
    if (!g_stats_static_ptr[dev]) {
        void* p = nullptr;
        NQS_CUDA(cudaGetSymbolAddress(&p, g_stats_static_scratch));
        if (!p) return fail(NQS_ERR_CUDA, "nqs_energy_stats_static: cudaGetSymbolAddress returned a null address");
        g_stats_static_ptr[dev] = static_cast<double*>(p);
    }
    *out = g_stats_static_ptr[dev];
    return NQS_OK;
}

extern "C" int nqs_energy_stats_static(const nqs_c64* d_x, const float* d_weights, int64_t B, double* d_stats,
                                       void* stream) {
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "nqs_energy_stats_static: B < 0");
    if (B == 0) return NQS_OK;
    if (!d_x || !d_stats) return fail(NQS_ERR_INVALID_ARG, "nqs_energy_stats_static: NULL pointer");
    if (B > (int64_t)NQS_STATS_STATIC_MAX_B)
        return fail(NQS_ERR_UNSUPPORTED,
                    "nqs_energy_stats_static: B = " + std::to_string((long long)B) + " exceeds NQS_STATS_STATIC_MAX_B = " +
                        std::to_string((long long)NQS_STATS_STATIC_MAX_B) +
                        " (the limit of the fixed scratch array; use nqs_energy_stats for larger batches)");
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        cudaGetLastError();
        return fail(NQS_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
    }
    double* partial = nullptr;
    NQS_TRY(stats_static_scratch(&partial));
    cudaStream_t st = (cudaStream_t)stream;
    // one record per block, as in launch_stats; stats_partial_kernel writes all four sums of every record
    // 0 .. nblk-1 and stats_final_kernel reads exactly those, so nothing left behind by an earlier call is ever
    // read and nothing has to be cleared first
    const int nblk = (int)((B + 255) / 256 < ST_BLOCKS ? (B + 255) / 256 : ST_BLOCKS);
    stats_partial_kernel<<<nblk, 256, 0, st>>>((const float2*)d_x, d_weights, (long long)B, partial);
    NQS_LAUNCHED();
    stats_final_kernel<<<1, 32, 0, st>>>(partial, nblk, d_stats);
    NQS_LAUNCHED();
    return NQS_OK;
}

// F[k] = sum_b conj(O_k(s_b)) cb[b] for all K = N + M + M N parameters: the exact int8 contraction over the
// samples of nqs_forces.cuh.  tp = tanh(theta) pair records, cb [B_pad] (0 for the padding samples).
// spT_out != NULL: the transposed int8 spins it packs ([nIT][K16][128] uint4) are handed to `keeper`.
static int force_contract(DeviceState* D, const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const float4* tp,
                          const float2* cb, nqs_c64* d_F, cudaStream_t st, uint4** spT_out, Scratch* keeper) {
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;
    const int K16 = (int)(B_pad / 16);
    const int nIT = (N + 1 + TM_M - 1) / TM_M, nJT = (M + 1 + TM_JT - 1) / TM_JT;
    Scratch S(D, st);
    int* gexp = nullptr;
    uint4 *A_packed = nullptr, *B_packed = nullptr;
    NQS_TRY(S.get(&gexp, (size_t)nJT * TM_JT));
    NQS_TRY(S.get(&A_packed, (size_t)nIT * K16 * TM_M));
    NQS_TRY(S.get(&B_packed, (size_t)nJT * K16 * TM_N));
    force_gscale_kernel<<<(unsigned)(nJT * TM_JT), 256, 0, st>>>(tp, nPairsPad, cb, M, gexp);
    NQS_LAUNCHED();
    force_pack_g_kernel<<<(unsigned)D->sms * 8, 256, 0, st>>>(tp, nPairsPad, cb, M, K16, nJT, gexp, B_packed);
    NQS_LAUNCHED();
    force_pack_spins_kernel<<<(unsigned)D->sms * 8, 256, 0, st>>>(d_spins, (long long)B, N, K16, nIT, A_packed);
    NQS_LAUNCHED();
    NQS_TRY(ensure_smem(D, force_mma_kernel, FM_SMEM));
    ForceMmaParams p;
    p.A_packed = A_packed;
    p.B_packed = B_packed;
    p.gexp = gexp;
    p.N = N;
    p.M = M;
    p.K16 = K16;
    p.F = (float2*)d_F;
    force_mma_kernel<<<dim3((unsigned)nIT, (unsigned)nJT), FM_THREADS, FM_SMEM, st>>>(p);
    NQS_LAUNCHED();
    if (spT_out) {
        *spT_out = A_packed;
        S.disown(A_packed);
        keeper->adopt(A_packed);
    }
    return NQS_OK;
}

// tp_in != NULL: tanh(theta) of this batch from local_energy_impl (owned by the caller's Scratch)
static int forces_impl(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                       const nqs_c64* d_b, const nqs_c64* d_W, const nqs_c64* d_eloc, const float* d_weights,
                       nqs_c64* d_F, double* d_stats, void* stream, float4* tp_in) {
    NQS_TRY(check_common(d_spins, B, N, M, d_a, d_b, d_W));
    if (B == 0) return NQS_OK;
    if (!d_eloc || !d_F) return fail(NQS_ERR_INVALID_ARG, "nqs_forces: NULL d_eloc / d_F");
    if (B > (1ll << 25)) return fail(NQS_ERR_UNSUPPORTED, "nqs_forces: B > 2^25 (int32 accumulation range)");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    cudaStream_t st = (cudaStream_t)stream;
    const int M_pad = (int)round_up(M, KJ);
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;

    Scratch S(D, st);
    float4* tp = tp_in;
    float2* cb = nullptr;
    double* stats = nullptr;
    if (!tp) NQS_TRY(S.get(&tp, (size_t)M_pad * nPairsPad));
    NQS_TRY(S.get(&cb, (size_t)B_pad));
    NQS_TRY(S.get(&stats, 4));
    NQS_TRY(launch_stats(D, d_eloc, d_weights, B, stats, st));
    if (d_stats) NQS_CUDA(cudaMemcpyAsync(d_stats, stats, sizeof(double) * 4, cudaMemcpyDeviceToDevice, st));
    force_coef_kernel<<<(unsigned)((B_pad + 255) / 256), 256, 0, st>>>((const float2*)d_eloc, d_weights, (long long)B,
                                                                       B_pad, stats, cb);
    NQS_LAUNCHED();
    if (!tp_in) {
        ThetaOut o;
        o.tp = tp;
        NQS_TRY(launch_theta(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
    }
    return force_contract(D, d_spins, B, N, M, tp, cb, d_F, st, nullptr, nullptr);
}

// S = <<O* O>>_c (nqs_fisher.cuh).  tp_in != NULL: tanh(theta) of this batch (owned by the caller's Scratch).
static int fisher_impl(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a, const nqs_c64* d_b,
                       const nqs_c64* d_W, const float* d_weights, nqs_c64* d_S, nqs_c64* d_Obar, void* stream,
                       float4* tp_in) {
    NQS_TRY(check_common(d_spins, B, N, M, d_a, d_b, d_W));
    if (B == 0) return NQS_OK;
    if (!d_S) return fail(NQS_ERR_INVALID_ARG, "nqs_fisher: NULL d_S");
    const long long K = (long long)N + M + (long long)M * N;
    if (K > FS_MAX_K) return fail(NQS_ERR_UNSUPPORTED, "nqs_fisher: more than 8192 parameters (S would exceed 512 MB)");
    if (B > (1ll << 25)) return fail(NQS_ERR_UNSUPPORTED, "nqs_fisher: B > 2^25");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    cudaStream_t st = (cudaStream_t)stream;
    const int M_pad = (int)round_up(M, KJ);
    const long long B_pad = round_up(B, 256);
    const long long nPairsPad = B_pad / 2;
    const int K16 = (int)(B_pad / 16);
    const int nKT = (int)((K + FS_T - 1) / FS_T);

    Scratch S(D, st);
    float4* tp = tp_in;
    float2 *cb = nullptr, *Fc = nullptr;
    float* sw = nullptr;
    double* stats = nullptr;
    uint4 *spT = nullptr, *X = nullptr;
    if (!tp) NQS_TRY(S.get(&tp, (size_t)M_pad * nPairsPad));
    NQS_TRY(S.get(&cb, (size_t)B_pad));
    NQS_TRY(S.get(&sw, (size_t)B_pad));
    NQS_TRY(S.get(&stats, 4));
    NQS_TRY(S.get(&Fc, (size_t)K));
    NQS_TRY(S.get(&X, (size_t)nKT * K16 * FS_PLANES * FS_PLANE_U4));
    NQS_TRY(launch_stats(D, nullptr, d_weights, B, stats, st));
    fisher_mean_coef_kernel<<<(unsigned)((B_pad + 255) / 256), 256, 0, st>>>(d_weights, (long long)B, B_pad, stats, cb, sw);
    NQS_LAUNCHED();
    if (!tp_in) {
        ThetaOut o;
        o.tp = tp;
        NQS_TRY(launch_theta(D, d_spins, B, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
    }
    NQS_TRY(force_contract(D, d_spins, B, N, M, tp, cb, (nqs_c64*)Fc, st, &spT, &S));
    // power-of-two operand scale: |X| ~ |O - <O>| / sqrt(B) is brought to O(1) (exactly removed in the epilogue)
    int e = 0;
    (void)frexpf(sqrtf((float)B), &e);
    float scale = ldexpf(4.f, e);
    if (scale > 16384.f) scale = 16384.f;
    const long long nB8 = B_pad / 8;
    fisher_pack_kernel<<<(unsigned)D->sms * 16, 256, 0, st>>>(tp, nPairsPad, spT, K16, sw, Fc, N, M, (int)K, nKT, nB8, scale, X);
    NQS_LAUNCHED();
    NQS_TRY(ensure_smem(D, fisher_gemm_kernel, FS_SMEM));
    FisherGemmParams p;
    p.X_packed = X;
    p.nBC = K16;
    p.K = (int)K;
    p.nKT = nKT;
    p.inv_scale2 = 1.f / (scale * scale);
    p.S = (float2*)d_S;
    p.Obar = (float2*)d_Obar;
    p.Fc = Fc;
    fisher_gemm_kernel<<<(unsigned)(nKT * (nKT + 1) / 2), FS_THREADS, FS_SMEM, st>>>(p);
    NQS_LAUNCHED();
    return NQS_OK;
}

extern "C" int nqs_fisher(const int8_t* d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64* d_a,
                          const nqs_c64* d_b, const nqs_c64* d_W, const float* d_weights, nqs_c64* d_S,
                          nqs_c64* d_Obar, void* stream) {
    return fisher_impl(d_spins, B, N, M, d_a, d_b, d_W, d_weights, d_S, d_Obar, stream, nullptr);
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
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "nqs_local_energy_forces_h: B < 0");
    if (B == 0) return NQS_OK;
    if (!d_F) return fail(NQS_ERR_INVALID_ARG, "nqs_local_energy_forces_h: NULL d_F");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    Scratch keeper(D, (cudaStream_t)stream);
    float4* tp = nullptr;
    NQS_TRY(local_energy_impl(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream, &tp, &keeper));
    return forces_impl(d_spins, B, h->hc.N, M, d_a, d_b, d_W, d_eloc, d_weights, d_F, d_stats, stream, tp);
}

// Algorithm 1 lines 6-9 in one call: E_loc, statistics, force vector F and Fisher matrix S of one batch.
extern "C" int nqs_vmc_step_h(const nqs_hamiltonian* h, const int8_t* d_spins, int64_t B, int32_t M, const nqs_c64* d_a,
                              const nqs_c64* d_b, const nqs_c64* d_W, const float* d_weights, nqs_c64* d_eloc,
                              nqs_c64* d_logpsi, nqs_c64* d_F, nqs_c64* d_S, nqs_c64* d_Obar, double* d_stats,
                              void* stream) {
    if (B < 0) return fail(NQS_ERR_INVALID_ARG, "nqs_vmc_step_h: B < 0");
    if (B == 0) return NQS_OK;
    if (!d_F || !d_S) return fail(NQS_ERR_INVALID_ARG, "nqs_vmc_step_h: NULL d_F / d_S");
    if (!h) return fail(NQS_ERR_INVALID_ARG, "hamiltonian handle is NULL");
    const long long K = (long long)h->hc.N + M + (long long)M * h->hc.N;
    if (K > FS_MAX_K) return fail(NQS_ERR_UNSUPPORTED, "nqs_vmc_step_h: more than 8192 parameters");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    Scratch keeper(D, (cudaStream_t)stream);
    float4* tp = nullptr;
    NQS_TRY(local_energy_impl(h, d_spins, B, M, d_a, d_b, d_W, d_eloc, d_logpsi, stream, &tp, &keeper));
    NQS_TRY(forces_impl(d_spins, B, h->hc.N, M, d_a, d_b, d_W, d_eloc, d_weights, d_F, d_stats, stream, tp));
    return fisher_impl(d_spins, B, h->hc.N, M, d_a, d_b, d_W, d_weights, d_S, d_Obar, stream, tp);
}

// ----------------------------------------------------------------------------------------
// Metropolis chains
// ----------------------------------------------------------------------------------------
template <int CPB>
static int launch_metropolis_t(DeviceState* D, const MetroParams& p, size_t smem, cudaStream_t st) {
    NQS_TRY(ensure_smem(D, metropolis_kernel<CPB>, smem));
    metropolis_kernel<CPB><<<(unsigned)((p.C + CPB - 1) / CPB), CPB * 32, smem, st>>>(p);
    NQS_LAUNCHED();
    return NQS_OK;
}

static int metropolis_impl(int8_t* d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64* d_a, const nqs_c64* d_b,
                           const nqs_c64* d_W, int32_t S, const int32_t* d_sites, const float* d_u,
                           int32_t* d_accepted, uint8_t* d_decisions, void* stream) {
    NQS_TRY(check_common(d_spins, C, N, M, d_a, d_b, d_W));
    if (S < 0 || (S > 0 && C > 0 && (!d_sites || !d_u)))
        return fail(NQS_ERR_INVALID_ARG, "nqs_metropolis: S < 0 or NULL sites / u");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (C == 0) return NQS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    NQS_TRY(validate_spins(D, d_spins, C, N, st));
    const int M_pad = (int)round_up(M, KJ);
    const long long C_pad = round_up(C, 256);
    const long long nPairsPad = C_pad / 2;
    int cpb = 16;
    while (cpb > 2 && metropolis_smem_bytes(cpb, N, M_pad) > 220 * 1024) cpb >>= 1;
    const size_t smem = metropolis_smem_bytes(cpb, N, M_pad);
    if (smem > 220 * 1024)
        return fail(NQS_ERR_UNSUPPORTED, "nqs_metropolis: M too large for the shared-memory chain state");

    Scratch Sc(D, st);
    float4 *tp = nullptr, *Gp = nullptr, *Gm = nullptr;
    float* lk2 = nullptr;
    NQS_TRY(Sc.get(&tp, (size_t)M_pad * nPairsPad));
    NQS_TRY(Sc.get(&Gp, (size_t)N * (M_pad / 2)));
    NQS_TRY(Sc.get(&Gm, (size_t)N * (M_pad / 2)));
    NQS_TRY(Sc.get(&lk2, (size_t)N));
    site_table_kernel<<<(unsigned)N, 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad, Gp, Gm, lk2);
    NQS_LAUNCHED();
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
    // chunks of two sweeps; theta is recomputed from the current spins before each chunk
    const int chunk = 2 * N;
    for (int s0 = 0; s0 == 0 || s0 < S; s0 += chunk) {
        ThetaOut o;
        o.tp = tp;
        o.raw = true;
        NQS_TRY(launch_theta(D, d_spins, C, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
        p.S = S - s0 < chunk ? S - s0 : chunk;
        p.sites = d_sites + (long long)s0 * C;
        p.u = d_u + (long long)s0 * C;
        p.decisions = d_decisions ? d_decisions + (long long)s0 * C : nullptr;
        p.accumulate = s0 > 0;
        switch (cpb) {
            case 16: NQS_TRY(launch_metropolis_t<16>(D, p, smem, st)); break;
            case 8: NQS_TRY(launch_metropolis_t<8>(D, p, smem, st)); break;
            case 4: NQS_TRY(launch_metropolis_t<4>(D, p, smem, st)); break;
            default: NQS_TRY(launch_metropolis_t<2>(D, p, smem, st)); break;
        }
    }
    return NQS_OK;
}

template <int PPL>
static int launch_metropolis_shared_t(DeviceState* D, const MetroSharedParams& p, cudaStream_t st) {
    using Cfg = MetroSharedCfg<PPL>;
    const size_t smem = metropolis_shared_smem_bytes(Cfg::WARPS, p.N, p.M_pad);
    NQS_TRY(ensure_smem(D, metropolis_shared_kernel<PPL>, smem));
    metropolis_shared_kernel<PPL><<<(unsigned)((p.C + Cfg::WARPS - 1) / Cfg::WARPS), Cfg::NT, smem, st>>>(p);
    NQS_LAUNCHED();
    return NQS_OK;
}

extern "C" int nqs_metropolis_shared(int8_t* d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64* d_a,
                                     const nqs_c64* d_b, const nqs_c64* d_W, int32_t S, const int32_t* d_sites,
                                     const float* d_u, int32_t* d_accepted, uint8_t* d_decisions, void* stream) {
    NQS_TRY(check_common(d_spins, C, N, M, d_a, d_b, d_W));
    if (S < 0 || (S > 0 && C > 0 && (!d_sites || !d_u)))
        return fail(NQS_ERR_INVALID_ARG, "nqs_metropolis_shared: S < 0 or NULL sites / u");
    DeviceState* D = nullptr;
    NQS_TRY(device_state(&D));
    if (C == 0) return NQS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    NQS_TRY(validate_spins(D, d_spins, C, N, st));
    const int M_pad = (int)round_up(M, KJ);
    const int ppl_need = (M_pad / 2 + 31) / 32;
    if (ppl_need > 32)
        return fail(NQS_ERR_UNSUPPORTED, "nqs_metropolis_shared: M > 2048 (the chain state lives in registers)");
    {   // the ring of table rows, the chains' spins and the per-site data must fit the 227 KB a CTA may opt into
        const int warps = ppl_need <= 1 ? MetroSharedCfg<1>::WARPS : ppl_need <= 2 ? MetroSharedCfg<2>::WARPS
                        : ppl_need <= 4 ? MetroSharedCfg<4>::WARPS : ppl_need <= 8 ? MetroSharedCfg<8>::WARPS
                        : ppl_need <= 13 ? MetroSharedCfg<13>::WARPS : ppl_need <= 16 ? MetroSharedCfg<16>::WARPS
                        : ppl_need <= 25 ? MetroSharedCfg<25>::WARPS : MetroSharedCfg<32>::WARPS;
        const size_t need = metropolis_shared_smem_bytes(warps, N, M_pad);
        if (need > 227 * 1024)
            return fail(NQS_ERR_UNSUPPORTED, "nqs_metropolis_shared: N = " + std::to_string(N) + ", M = " + std::to_string(M) +
                                                 " need " + std::to_string(need) + " bytes of shared memory per block (limit 232448); use nqs_metropolis");
    }
    const long long C_pad = round_up(C, 256);
    const long long nPairsPad = C_pad / 2;
    Scratch Sc(D, st);
    float4 *tp = nullptr, *Gp = nullptr, *Gm = nullptr;
    float* lk2 = nullptr;
    NQS_TRY(Sc.get(&tp, (size_t)M_pad * nPairsPad));
    NQS_TRY(Sc.get(&Gp, (size_t)N * (M_pad / 2)));
    NQS_TRY(Sc.get(&Gm, (size_t)N * (M_pad / 2)));
    NQS_TRY(Sc.get(&lk2, (size_t)N));
    site_table_kernel<<<(unsigned)N, 256, 0, st>>>((const float2*)d_W, (const float2*)d_a, N, M, M_pad, Gp, Gm, lk2);
    NQS_LAUNCHED();
    MetroSharedParams p;
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
    const int chunk = 2 * N;  // theta is recomputed from the current spins every two sweeps
    for (int s0 = 0; s0 == 0 || s0 < S; s0 += chunk) {
        ThetaOut o;
        o.tp = tp;
        o.raw = true;
        NQS_TRY(launch_theta(D, d_spins, C, N, M, M_pad, d_a, d_b, d_W, nPairsPad, o, st));
        p.S = S - s0 < chunk ? S - s0 : chunk;
        p.sites = d_sites + s0;
        p.u = d_u + (long long)s0 * C;
        p.decisions = d_decisions ? d_decisions + (long long)s0 * C : nullptr;
        p.accumulate = s0 > 0;
        if (ppl_need <= 1) NQS_TRY(launch_metropolis_shared_t<1>(D, p, st));
        else if (ppl_need <= 2) NQS_TRY(launch_metropolis_shared_t<2>(D, p, st));
        else if (ppl_need <= 4) NQS_TRY(launch_metropolis_shared_t<4>(D, p, st));
        else if (ppl_need <= 8) NQS_TRY(launch_metropolis_shared_t<8>(D, p, st));
        else if (ppl_need <= 13) NQS_TRY(launch_metropolis_shared_t<13>(D, p, st));
        else if (ppl_need <= 16) NQS_TRY(launch_metropolis_shared_t<16>(D, p, st));
        else if (ppl_need <= 25) NQS_TRY(launch_metropolis_shared_t<25>(D, p, st));
        else NQS_TRY(launch_metropolis_shared_t<32>(D, p, st));
    }
    return NQS_OK;
}

extern "C" int nqs_metropolis(int8_t* d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64* d_a,
                              const nqs_c64* d_b, const nqs_c64* d_W, int32_t S, const int32_t* d_sites,
                              const float* d_u, int32_t* d_accepted, void* stream) {
    return metropolis_impl(d_spins, C, N, M, d_a, d_b, d_W, S, d_sites, d_u, d_accepted, nullptr, stream);
}

extern "C" int nqs_metropolis_trace(int8_t* d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64* d_a,
                                    const nqs_c64* d_b, const nqs_c64* d_W, int32_t S, const int32_t* d_sites,
                                    const float* d_u, int32_t* d_accepted, uint8_t* d_decisions, void* stream) {
    return metropolis_impl(d_spins, C, N, M, d_a, d_b, d_W, S, d_sites, d_u, d_accepted, d_decisions, stream);
}
