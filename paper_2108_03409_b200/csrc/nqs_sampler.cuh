// single-spin-flip Metropolis sampling of |psi(s)|^2, many chains in lock-step
// (PAPER.md:70 Metropolis-Hastings; :341 sweeps; :490-494 chains advanced in sync on one device).
//
// A chain's state is E_j = exp(2 theta_j) for every hidden unit.  For the proposal "flip site i" of a
// chain with spin sigma = s_i, theta_j -> theta_j - 2 sigma W_ji, and with G_ji(sigma) = exp(4 sigma W_ji)
//   cosh(theta_j - 2 sigma W_ji) / cosh(theta_j) = exp(-2 sigma W_ji) (E_j + G_ji(sigma)) / (E_j + 1),
//   psi(s')/psi(s) = exp(-2 sigma (a_i + sum_j W_ji)) prod_j (E_j + G_ji(sigma)) / (E_j + 1),
// and an accepted move updates the state IN PLACE by one complex multiplication,
//   E_j <- E_j G_ji(-sigma)          (no division, no transcendental in the loop).
// Only |psi(s')/psi(s)|^2 is needed, so numerator and denominator are real products of squared
// moduli, accumulated as sums of log2 (range-safe) and reduced over the warp with shuffles.
// Why E and not tanh(theta) with the addition theorem (the first version of this kernel, 15 % faster
// at config 5, failed the shape fuzz by drift at sigma = 0.25; DESIGN.md section 9 has the record): for a saturated unit (|Re theta| >~ 4)
// tanh(theta) = +-1 - tiny cannot hold theta to float32 accuracy, and the loss shows up as an O(0.1)
// error in log |ratio|^2 once later flips bring the unit back; E_j keeps a RELATIVE error of 1 ulp
// per update, i.e. an ABSOLUTE error of 6e-8 per update in theta.  Range: |E + 1|^2 must stay finite,
// i.e. |Re theta| < 22; the acceptance test multiplies per-pair RATIOS |E + G|^2 / |E + 1|^2, never the
// two squared moduli separately.
//
// One warp owns one chain for the whole call; the chain's E (M complex numbers) and spins live in
// shared memory, the tables exp(+-4 W)^T [N][M_pad/2] (2 x 5 MB at config 5) are read from L2.  The
// random numbers (proposal site, uniform u) are inputs.  The host splits a call into chunks of two
// sweeps (2 N steps) and recomputes theta from the spins with the a2 kernel before each chunk.
//
// Hidden units are handled in PAIRS (j0, j1) = (2 jp, 2 jp + 1) riding in the two halves of packed
// FFMA2 operands: records are float4 (re_j0, re_j1, im_j0, im_j1) for E and for the tables.
#pragma once
#include "nqs_device.cuh"

namespace nqs {

// One block per site i: Gp[i][jp] = exp(+4 W_ji), Gm[i][jp] = exp(-4 W_ji) for the pair jp (1 for the
// padding j >= M: (E + 1)/(E + 1) = 1) and lk2[i] = -4 log2(e) Re(a_i + sum_j W_ji), so that
// log2 |exp(-2 sigma (a_i + sum_j W_ji))|^2 = sigma lk2[i].
__global__ void __launch_bounds__(256) site_table_kernel(const float2* __restrict__ W, const float2* __restrict__ a,
                                                         int N, int M, int M_pad, float4* __restrict__ Gp,
                                                         float4* __restrict__ Gm, float* __restrict__ lk2) {
    const int i = blockIdx.x;
    __shared__ double sh[256];
    double acc = 0.0;
    for (int jp = threadIdx.x; jp < M_pad / 2; jp += 256) {
        float pr[2] = {1.f, 1.f}, pi[2] = {0.f, 0.f}, mr[2] = {1.f, 1.f}, mi[2] = {0.f, 0.f};
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int j = 2 * jp + h;
            if (j < M) {
                const float2 w = W[(long long)j * N + i];
                float sn, cs;
                sincosf(4.f * w.y, &sn, &cs);
                const float ep = expf(4.f * w.x), em = expf(-4.f * w.x);
                pr[h] = ep * cs, pi[h] = ep * sn;
                mr[h] = em * cs, mi[h] = -em * sn;
                acc += (double)w.x;
            }
        }
        Gp[(long long)i * (M_pad / 2) + jp] = make_float4(pr[0], pr[1], pi[0], pi[1]);
        Gm[(long long)i * (M_pad / 2) + jp] = make_float4(mr[0], mr[1], mi[0], mi[1]);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) lk2[i] = (float)(-4.0 * 1.4426950408889634 * (sh[0] + (double)a[i].x));
}

// MUFU.RCP (1 ulp) and MUFU.LG2 (absolute error 2^-22) instead of the correctly rounded routines: the sum of the
// 32 lanes' logarithms is needed to ~1e-5 (the decision margin of the parity rule is 2e-4), not to the last bit
__device__ __forceinline__ float fast_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

struct MetroParams {
    int8_t* spins;           // [C][N] in / out
    long long C;
    int N, M, M_pad, S;
    const float4* tp;        // [M_pad][nPairsPad]: theta of the start states (raw), two chains per record
    long long nPairsPad;
    const float4* Gp;        // [N][M_pad / 2]  exp(+4 W)
    const float4* Gm;        // [N][M_pad / 2]  exp(-4 W)
    const float* lk2;        // [N]
    const int* sites;        // [S][C]
    const float* u;          // [S][C]
    int* accepted;           // [C] or nullptr
    int accumulate;          // add to accepted[] instead of overwriting it
    uint8_t* decisions;      // [S][C] or nullptr: 1 = the proposal of step t was accepted (nqs_metropolis_trace)
};

__host__ __device__ inline size_t metropolis_smem_bytes(int cpb, int N, int M_pad) {
    return (size_t)cpb * ((size_t)M_pad * sizeof(float2) + (size_t)((N + 15) / 16 * 16));
}

constexpr int MT_UNROLL = 5;  // pairs per lane whose loads are issued together (config 5: 25 = 5 x 5)

template <int CPB>
__global__ void __launch_bounds__(CPB * 32, 1) metropolis_kernel(const MetroParams p) {
    extern __shared__ __align__(16) unsigned char mt_smem[];
    float4* const E_all = reinterpret_cast<float4*>(mt_smem);
    const int N_pad = (p.N + 15) / 16 * 16;
    const int MP = p.M_pad / 2;  // hidden-unit pairs (padding pairs: theta = 0, E = 1, G = 1: factor 1)
    int8_t* const s_all = reinterpret_cast<int8_t*>(mt_smem + (size_t)CPB * p.M_pad * sizeof(float2));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long c0 = (long long)blockIdx.x * CPB;

    // E = exp(2 theta); the block's CPB chains are CPB/2 consecutive records of every tp row
    for (int idx = tid; idx < MP * (CPB / 2); idx += CPB * 32) {
        const int jp = idx / (CPB / 2), pr = idx % (CPB / 2);
        const float4 r0 = p.tp[(long long)(2 * jp) * p.nPairsPad + c0 / 2 + pr];      // (xA, xB, yA, yB) of unit 2 jp
        const float4 r1 = p.tp[(long long)(2 * jp + 1) * p.nPairsPad + c0 / 2 + pr];  // of unit 2 jp + 1
        float sn, cs;
        float4 eA, eB;
        float m;
        m = expf(2.f * r0.x), sincosf(2.f * r0.z, &sn, &cs), eA.x = m * cs, eA.z = m * sn;
        m = expf(2.f * r1.x), sincosf(2.f * r1.z, &sn, &cs), eA.y = m * cs, eA.w = m * sn;
        m = expf(2.f * r0.y), sincosf(2.f * r0.w, &sn, &cs), eB.x = m * cs, eB.z = m * sn;
        m = expf(2.f * r1.y), sincosf(2.f * r1.w, &sn, &cs), eB.y = m * cs, eB.w = m * sn;
        E_all[(size_t)(2 * pr) * MP + jp] = eA;
        E_all[(size_t)(2 * pr + 1) * MP + jp] = eB;
    }
    for (int idx = tid; idx < CPB * p.N; idx += CPB * 32) {
        const int w = idx / p.N, i = idx % p.N;
        s_all[w * N_pad + i] = (c0 + w < p.C) ? p.spins[(c0 + w) * p.N + i] : (int8_t)1;
    }
    __syncthreads();

    const long long c = c0 + warp;
    if (c >= p.C) return;
    float4* const E_s = E_all + (size_t)warp * MP;
    int8_t* const s_s = s_all + warp * N_pad;
    const int nFull = MP / (32 * MT_UNROLL);  // groups of 32 x MT_UNROLL pairs with no ragged lane
    const float4 one4 = make_float4(1.f, 1.f, 0.f, 0.f);
    int acc = 0;
    bool bad = false;
    for (int step = 0; step < p.S; ++step) {
        int site = 0;
        float ul = 0.f;
        if (lane == 0) {
            site = p.sites[(long long)step * p.C + c];
            ul = p.u[(long long)step * p.C + c];
        }
        site = __shfl_sync(0xffffffffu, site, 0);
        ul = __shfl_sync(0xffffffffu, ul, 0);
        const int sgi = s_s[site];
        const float4* const Gfwd = (sgi > 0 ? p.Gp : p.Gm) + (long long)site * MP;  // G(sigma)
        const float4* const Gbwd = (sgi > 0 ? p.Gm : p.Gp) + (long long)site * MP;  // G(-sigma)
        // pass 1: sum_j log2 |E_j + G_j|^2 - log2 |E_j + 1|^2
        float lg = 0.f;
        auto pass1 = [&](int jp0, bool ragged) {
            float4 E[MT_UNROLL], G[MT_UNROLL];
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                const int jp = jp0 + 32 * k;
                const bool live = !ragged || jp < MP;
                G[k] = live ? Gfwd[jp] : one4;
                E[k] = live ? E_s[jp] : one4;
            }
            // per pair the RATIO |E + G|^2 / |E + 1|^2 (O(1)); the two squared moduli are each ~ e^{4 |Re theta|}
            // and a product of them overflows float32 for saturated units
            float2 q = make_float2(1.f, 1.f);
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                const float2 er = make_float2(E[k].x, E[k].y), ei = make_float2(E[k].z, E[k].w);
                const float2 nr = __fadd2_rn(er, make_float2(G[k].x, G[k].y)), ni = __fadd2_rn(ei, make_float2(G[k].z, G[k].w));
                const float2 dr = __fadd2_rn(er, bc2(1.f));
                const float2 n2 = __ffma2_rn(nr, nr, __fmul2_rn(ni, ni));
                const float2 d2 = __ffma2_rn(dr, dr, __fmul2_rn(ei, ei));
                q = __fmul2_rn(q, __fmul2_rn(n2, make_float2(fast_rcp(d2.x), fast_rcp(d2.y))));
            }
            lg += __log2f(q.x * q.y);
        };
        for (int g = 0; g < nFull; ++g) pass1(g * 32 * MT_UNROLL + lane, false);
        if (nFull * 32 * MT_UNROLL < MP) pass1(nFull * 32 * MT_UNROLL + lane, true);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lg += __shfl_xor_sync(0xffffffffu, lg, o);
        const float lk = p.lk2[site];
        bad |= !(lg <= 3.0e38f);  // NaN / +inf: a hidden unit left the float32 range of exp(2 theta); -inf is psi(s') = 0, a plain rejection
        const bool accept = log2f(ul) < (sgi > 0 ? lk : -lk) + lg;  // u == 0: -inf, always accepted
        if (lane == 0 && p.decisions) p.decisions[(long long)step * p.C + c] = accept ? 1 : 0;
        if (accept) {
            // pass 2: E_j <- E_j G_j(-sigma)
            auto pass2 = [&](int jp0, bool ragged) {
                float4 E[MT_UNROLL], G[MT_UNROLL];
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    const int jp = jp0 + 32 * k;
                    const bool live = !ragged || jp < MP;
                    G[k] = live ? Gbwd[jp] : one4;
                    E[k] = live ? E_s[jp] : one4;
                }
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    const float2 er = make_float2(E[k].x, E[k].y), ei = make_float2(E[k].z, E[k].w);
                    const float2 gr = make_float2(G[k].x, G[k].y), gi = make_float2(G[k].z, G[k].w);
                    const float2 outr = __ffma2_rn(neg2(ei), gi, __fmul2_rn(er, gr));
                    const float2 outi = __ffma2_rn(ei, gr, __fmul2_rn(er, gi));
                    const int jp = jp0 + 32 * k;
                    if (!ragged || jp < MP) E_s[jp] = make_float4(outr.x, outr.y, outi.x, outi.y);
                }
            };
            for (int g = 0; g < nFull; ++g) pass2(g * 32 * MT_UNROLL + lane, false);
            if (nFull * 32 * MT_UNROLL < MP) pass2(nFull * 32 * MT_UNROLL + lane, true);
            if (lane == 0) s_s[site] = (int8_t)(-sgi);
            ++acc;
        }
        __syncwarp();
    }
    for (int i = lane; i < p.N; i += 32) p.spins[c * p.N + i] = s_s[i];
    if (lane == 0 && p.accepted) {
        const int prev = p.accumulate ? p.accepted[c] : 0;
        p.accepted[c] = (bad || prev < 0) ? -1 : prev + acc;  // -1: the chain's state overflowed (|Re theta| >~ 22)
    }
}

// ---------------------------------------------------------------------------------------
// Shared-site variant (nqs_metropolis_shared): at step t EVERY chain proposes the same site sites[t].
// metropolis_kernel above is bound by the L2 -> SM stream of table rows (one 8 M-byte row of exp(+-4W)^T per chain
// and proposal: 655 GB per sweep at config 5, profiles/r2_ncu_summary.md).  With a common site the two rows
// exp(+4W)[site], exp(-4W)[site] are fetched ONCE per CTA and step by a bulk copy into a double-buffered shared
// memory stage (the copy for step t + 1 overlaps step t), and the chain state E_j = exp(2 theta_j) moves from
// shared memory into REGISTERS: lane l of the chain's warp owns the hidden-unit pairs l, l + 32, ... (PPL of them),
// so a proposal reads only the staged row from shared memory.  Same arithmetic and acceptance rule as above.
// ---------------------------------------------------------------------------------------
struct MetroSharedParams {
    int8_t* spins;           // [C][N] in / out
    long long C;
    int N, M, M_pad, S;
    const float4* tp;        // [M_pad][nPairsPad]: theta of the start states (raw)
    long long nPairsPad;
    const float4* Gp;        // [N][M_pad / 2]  exp(+4 W)
    const float4* Gm;        // [N][M_pad / 2]  exp(-4 W)
    const float* lk2;        // [N]
    const int* sites;        // [S]
    const float* u;          // [S][C]
    int* accepted;           // [C] or nullptr
    int accumulate;
    uint8_t* decisions;      // [S][C] or nullptr
};

template <int PPL>
struct MetroSharedCfg {
    static constexpr int WARPS = PPL > 25 ? 8 : 12;  // register budget: 4 PPL state registers per lane
    static constexpr int NT = WARPS * 32;
};
constexpr int MS_BUFS = 4;  // row buffers: the copy for step t + 3 is in flight while step t computes
// rows, the chains' spins, lk2[N], the site schedule of the launch (at most 2 N steps), barriers
__host__ __device__ inline size_t metropolis_shared_smem_bytes(int warps, int N, int M_pad) {
    return 128 + (size_t)MS_BUFS * 2 * (M_pad / 2) * sizeof(float4) + (size_t)warps * ((N + 15) / 16 * 16) +
           (size_t)3 * N * 4;
}

template <int PPL>
__global__ void __launch_bounds__(MetroSharedCfg<PPL>::NT, 1) metropolis_shared_kernel(const MetroSharedParams p) {
    constexpr int WARPS = MetroSharedCfg<PPL>::WARPS;
    extern __shared__ __align__(128) unsigned char ms_smem[];
    const int MP = p.M_pad / 2;
    const uint32_t row_bytes = (uint32_t)MP * 16u;
    uint64_t* const full = reinterpret_cast<uint64_t*>(ms_smem);     // [MS_BUFS] barriers in the first 128 bytes
    float4* const rows = reinterpret_cast<float4*>(ms_smem + 128);  // [MS_BUFS][Gp row | Gm row][MP]
    const int N_pad = (p.N + 15) / 16 * 16;
    int8_t* const s_all = reinterpret_cast<int8_t*>(ms_smem + 128 + (size_t)MS_BUFS * 2 * row_bytes);
    float* const lk_s = reinterpret_cast<float*>(s_all + (size_t)WARPS * N_pad);  // [N]
    int* const site_s = reinterpret_cast<int*>(lk_s + p.N);                       // [S <= 2 N]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long c = (long long)blockIdx.x * WARPS + warp;
    const bool live_chain = c < p.C;

    if (tid == 0) {
        for (int q = 0; q < MS_BUFS; ++q) mbar_init(&full[q], 1);
        fence_mbar_init();
    }
    for (int i = tid; i < p.N; i += WARPS * 32) lk_s[i] = p.lk2[i];
    for (int t = tid; t < p.S; t += WARPS * 32) site_s[t] = p.sites[t];
    auto stage = [&](int t) {  // thread 0: rows of step t -> buffer t % MS_BUFS
        const int site = site_s[t];
        float4* dst = rows + (size_t)(t % MS_BUFS) * 2 * MP;
        mbar_expect_tx(&full[t % MS_BUFS], 2 * row_bytes);
        bulk_g2s(dst, p.Gp + (long long)site * MP, row_bytes, &full[t % MS_BUFS]);
        bulk_g2s(dst + MP, p.Gm + (long long)site * MP, row_bytes, &full[t % MS_BUFS]);
    };
    // chain state: E = exp(2 theta) of the pairs this lane owns
    float4 E[PPL];
    const float4 one4 = make_float4(1.f, 1.f, 0.f, 0.f);
#pragma unroll
    for (int k = 0; k < PPL; ++k) {
        const int jp = lane + 32 * k;
        E[k] = one4;
        if (live_chain && jp < MP) {
            const float4 r0 = p.tp[(long long)(2 * jp) * p.nPairsPad + (c >> 1)];      // (xA, xB, yA, yB) of unit 2 jp
            const float4 r1 = p.tp[(long long)(2 * jp + 1) * p.nPairsPad + (c >> 1)];  // of unit 2 jp + 1
            const bool hi = c & 1;
            const float x0 = hi ? r0.y : r0.x, y0 = hi ? r0.w : r0.z, x1 = hi ? r1.y : r1.x, y1 = hi ? r1.w : r1.z;
            float sn, cs, m;
            m = expf(2.f * x0), sincosf(2.f * y0, &sn, &cs), E[k].x = m * cs, E[k].z = m * sn;
            m = expf(2.f * x1), sincosf(2.f * y1, &sn, &cs), E[k].y = m * cs, E[k].w = m * sn;
        }
    }
    int8_t* const s_s = s_all + warp * N_pad;
    for (int i = lane; i < p.N; i += 32) s_s[i] = live_chain ? p.spins[c * p.N + i] : (int8_t)1;
    __syncthreads();
    if (tid == 0)
        for (int t = 0; t < MS_BUFS - 1 && t < p.S; ++t) stage(t);

    int acc = 0;
    bool bad = false;
    float u_next = (live_chain && p.S > 0) ? p.u[c] : 2.f;  // the uniform of a step is fetched one step ahead
    for (int step = 0; step < p.S; ++step) {
        __syncthreads();  // every warp has finished step - 1: its row buffer may be overwritten
        if (tid == 0 && step + MS_BUFS - 1 < p.S) {
            fence_proxy_async();
            stage(step + MS_BUFS - 1);
        }
        const float ul = u_next;
        if (live_chain && step + 1 < p.S) u_next = p.u[(long long)(step + 1) * p.C + c];
        mbar_wait(&full[step % MS_BUFS], (uint32_t)((step / MS_BUFS) & 1));
        const int site = site_s[step];
        const int sgi = s_s[site];
        const float4* const buf = rows + (size_t)(step % MS_BUFS) * 2 * MP;
        const float4* const Gfwd = sgi > 0 ? buf : buf + MP;  // G(sigma)
        const float4* const Gbwd = sgi > 0 ? buf + MP : buf;  // G(-sigma)
        // pass 1: sum_j log2 |E_j + G_j|^2 - log2 |E_j + 1|^2, ratios multiplied in groups of up to five pairs
        float lg = 0.f;
        float2 q = make_float2(1.f, 1.f);
#pragma unroll
        for (int k = 0; k < PPL; ++k) {
            const int jp = lane + 32 * k;
            const float4 G = jp < MP ? Gfwd[jp] : one4;
            const float2 er = make_float2(E[k].x, E[k].y), ei = make_float2(E[k].z, E[k].w);
            const float2 nr = __fadd2_rn(er, make_float2(G.x, G.y)), ni = __fadd2_rn(ei, make_float2(G.z, G.w));
            const float2 dr = __fadd2_rn(er, bc2(1.f));
            const float2 n2 = __ffma2_rn(nr, nr, __fmul2_rn(ni, ni));
            const float2 d2 = __ffma2_rn(dr, dr, __fmul2_rn(ei, ei));
            q = __fmul2_rn(q, __fmul2_rn(n2, make_float2(fast_rcp(d2.x), fast_rcp(d2.y))));
            if (k % MT_UNROLL == MT_UNROLL - 1 || k == PPL - 1) {
                lg += __log2f(q.x * q.y);
                q = make_float2(1.f, 1.f);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lg += __shfl_xor_sync(0xffffffffu, lg, o);
        const float lk = lk_s[site];
        bad |= !(lg <= 3.0e38f);  // NaN / +inf: a hidden unit left the float32 range of exp(2 theta); -inf is psi(s') = 0, a plain rejection
        const bool accept = live_chain && (log2f(ul) < (sgi > 0 ? lk : -lk) + lg);  // u == 0: -inf, always accepted
        if (lane == 0 && live_chain && p.decisions) p.decisions[(long long)step * p.C + c] = accept ? 1 : 0;
        if (accept) {
            // pass 2: E_j <- E_j G_j(-sigma)
#pragma unroll
            for (int k = 0; k < PPL; ++k) {
                const int jp = lane + 32 * k;
                const float4 G = jp < MP ? Gbwd[jp] : one4;
                const float2 er = make_float2(E[k].x, E[k].y), ei = make_float2(E[k].z, E[k].w);
                const float2 gr = make_float2(G.x, G.y), gi = make_float2(G.z, G.w);
                const float2 outr = __ffma2_rn(neg2(ei), gi, __fmul2_rn(er, gr));
                const float2 outi = __ffma2_rn(ei, gr, __fmul2_rn(er, gi));
                E[k] = make_float4(outr.x, outr.y, outi.x, outi.y);
            }
            if (lane == 0) s_s[site] = (int8_t)(-sgi);
            ++acc;
        }
        __syncwarp();
    }
    if (live_chain) {
        for (int i = lane; i < p.N; i += 32) p.spins[c * p.N + i] = s_s[i];
        if (lane == 0 && p.accepted) {
            const int prev = p.accumulate ? p.accepted[c] : 0;
            p.accepted[c] = (bad || prev < 0) ? -1 : prev + acc;  // -1: the chain's state overflowed
        }
    }
}

}  // namespace nqs
