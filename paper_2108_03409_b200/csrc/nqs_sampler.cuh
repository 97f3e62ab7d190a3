// single-spin-flip Metropolis sampling of |psi(s)|^2, many chains in lock-step
// (PAPER.md:70 Metropolis-Hastings; :341 sweeps; :490-494 chains advanced in sync on one device).
//
// For a proposal "flip site i" of a chain with spin sigma = s_i the one-site ratio identity (R) gives
//   psi(s')/psi(s) = exp(-2 sigma a_i) prod_j cosh(2 W_ji) * prod_j D_j,   D_j = 1 - sigma t_j T_ji,
// t_j = tanh theta_j, T_ji = tanh 2 W_ji, and, by the addition theorem of tanh, an accepted move
// updates the chain's state IN PLACE without any transcendental:
//   t_j <- tanh(theta_j - 2 sigma W_ji) = (t_j - sigma T_ji) / D_j.
// Only |psi(s')/psi(s)|^2 is needed, so the product over hidden units is a real product of |D_j|^2,
// accumulated as a sum of log2 (range-safe) and reduced over the warp with shuffles.
//
// One warp owns one chain for the whole call; the chain's t (M complex numbers) and spins live in
// shared memory, T^T [N][M_pad] (5 MB at config 5) is read from L2.  The random numbers (proposal
// site, uniform u) are inputs.  The rational update is a Moebius map: it does not damp rounding
// errors, so the host splits a call into chunks of two sweeps (2 N steps) and recomputes t from
// the spins with the a2/a3 kernels before each chunk, which bounds the drift.
#pragma once
#include "nqs_device.cuh"

namespace nqs {

// Hidden units are handled in PAIRS (j0, j1) = (2 jp, 2 jp + 1) riding in the two halves of packed
// FFMA2 operands: records are float4 (re_j0, re_j1, im_j0, im_j1), for t in shared memory and for
// T^T in global memory, so one 16-byte load per operand feeds two hidden units.

// One block per site i: TT[i][jp] = tanh(2 W_ji) for the pair jp (0 for the padding j >= M) and
// lk2[i] = log2(e) * (Re L_i - 2 Re a_i, Re L_i + 2 Re a_i),  L_i = sum_j log cosh(2 W_ji):
// log2 |exp(-2 sigma a_i) prod_j cosh 2 W_ji|^2 / 2 for sigma = +1 (x) and -1 (y).
__global__ void __launch_bounds__(256) site_table_kernel(const float2* __restrict__ W, const float2* __restrict__ a,
                                                         int N, int M, int M_pad, float4* __restrict__ TT,
                                                         float2* __restrict__ lk2) {
    const int i = blockIdx.x;
    __shared__ double sh[256];
    double acc = 0.0;
    for (int jp = threadIdx.x; jp < M_pad / 2; jp += 256) {
        float tr[2] = {0.f, 0.f}, ti[2] = {0.f, 0.f};
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int j = 2 * jp + h;
            if (j < M) {
                const float2 w = W[(long long)j * N + i];
                float lr, li;
                lncosh_tanh(2.f * w.x, 2.f * w.y, lr, li, tr[h], ti[h]);
                acc += (double)lr;
            }
        }
        TT[(long long)i * (M_pad / 2) + jp] = make_float4(tr[0], tr[1], ti[0], ti[1]);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double L = sh[0], ar = (double)a[i].x, l2e = 1.4426950408889634;
        lk2[i] = make_float2((float)(l2e * (L - 2.0 * ar)), (float)(l2e * (L + 2.0 * ar)));
    }
}

struct MetroParams {
    int8_t* spins;           // [C][N] in / out
    long long C;
    int N, M, M_pad, S;
    const float4* tp;        // [M_pad][nPairsPad]: tanh theta of the start states, two chains per record
    long long nPairsPad;
    const float4* TT;        // [N][M_pad / 2]
    const float2* lk2;       // [N]
    const int* sites;        // [S][C]
    const float* u;          // [S][C]
    int* accepted;           // [C] or nullptr
    int accumulate;          // add to accepted[] instead of overwriting it
};

__host__ __device__ inline size_t metropolis_smem_bytes(int cpb, int N, int M_pad) {
    return (size_t)cpb * ((size_t)M_pad * sizeof(float2) + (size_t)((N + 15) / 16 * 16));
}

constexpr int MT_UNROLL = 5;  // pairs per lane whose loads are issued together (config 5: 25 = 5 x 5)

// D = 1 - sigma t T for a pair of hidden units; returns |D|^2 per half
__device__ __forceinline__ float2 metro_D(const float4 t, const float4 T, const float nsg, float2& Dr, float2& Di) {
    const float2 tr = make_float2(t.x, t.y), ti = make_float2(t.z, t.w);
    const float2 Tr = make_float2(T.x, T.y), Ti = make_float2(T.z, T.w);
    const float2 xr = __ffma2_rn(neg2(ti), Ti, __fmul2_rn(tr, Tr));
    const float2 xi = __ffma2_rn(ti, Tr, __fmul2_rn(tr, Ti));
    Dr = __ffma2_rn(bc2(nsg), xr, bc2(1.f));
    Di = __fmul2_rn(bc2(nsg), xi);
    return __ffma2_rn(Dr, Dr, __fmul2_rn(Di, Di));
}

template <int CPB>
__global__ void __launch_bounds__(CPB * 32, 1) metropolis_kernel(const MetroParams p) {
    extern __shared__ __align__(16) unsigned char mt_smem[];
    float4* const t_all = reinterpret_cast<float4*>(mt_smem);
    const int N_pad = (p.N + 15) / 16 * 16;
    const int MP = p.M_pad / 2;  // hidden-unit pairs (padding pairs hold t = 0, T = 0: D = 1)
    int8_t* const s_all = reinterpret_cast<int8_t*>(mt_smem + (size_t)CPB * p.M_pad * sizeof(float2));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long c0 = (long long)blockIdx.x * CPB;

    // the block's CPB chains are CPB/2 consecutive records of every tp row
    for (int idx = tid; idx < MP * (CPB / 2); idx += CPB * 32) {
        const int jp = idx / (CPB / 2), pr = idx % (CPB / 2);
        const float4 r0 = p.tp[(long long)(2 * jp) * p.nPairsPad + c0 / 2 + pr];
        const float4 r1 = p.tp[(long long)(2 * jp + 1) * p.nPairsPad + c0 / 2 + pr];
        t_all[(size_t)(2 * pr) * MP + jp] = make_float4(r0.x, r1.x, r0.z, r1.z);
        t_all[(size_t)(2 * pr + 1) * MP + jp] = make_float4(r0.y, r1.y, r0.w, r1.w);
    }
    for (int idx = tid; idx < CPB * p.N; idx += CPB * 32) {
        const int w = idx / p.N, i = idx % p.N;
        s_all[w * N_pad + i] = (c0 + w < p.C) ? p.spins[(c0 + w) * p.N + i] : (int8_t)1;
    }
    __syncthreads();

    const long long c = c0 + warp;
    if (c >= p.C) return;
    float4* const t_s = t_all + (size_t)warp * MP;
    int8_t* const s_s = s_all + warp * N_pad;
    const int nFull = MP / (32 * MT_UNROLL);  // groups of 32 x MT_UNROLL pairs with no ragged lane
    int acc = 0;
    for (int step = 0; step < p.S; ++step) {
        int site = 0;
        float ul = 0.f;
        if (lane == 0) {
            site = p.sites[(long long)step * p.C + c];
            ul = p.u[(long long)step * p.C + c];
        }
        site = __shfl_sync(0xffffffffu, site, 0);
        ul = __shfl_sync(0xffffffffu, ul, 0);
        const float sg = (float)s_s[site], nsg = -sg;
        const float4* const Trow = p.TT + (long long)site * MP;
        // pass 1: log2 prod_j |D_j|^2 (real product per lane, log2 per group, shuffle sum)
        float lg = 0.f;
        auto pass1 = [&](int jp0, bool ragged) {
            float4 t[MT_UNROLL], T[MT_UNROLL];
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                const int jp = jp0 + 32 * k;
                const bool live = !ragged || jp < MP;
                T[k] = live ? Trow[jp] : make_float4(0.f, 0.f, 0.f, 0.f);
                t[k] = live ? t_s[jp] : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            float2 q = make_float2(1.f, 1.f);
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                float2 Dr, Di;
                q = __fmul2_rn(q, metro_D(t[k], T[k], nsg, Dr, Di));
            }
            lg += log2f(q.x * q.y);
        };
        for (int g = 0; g < nFull; ++g) pass1(g * 32 * MT_UNROLL + lane, false);
        if (nFull * 32 * MT_UNROLL < MP) pass1(nFull * 32 * MT_UNROLL + lane, true);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lg += __shfl_xor_sync(0xffffffffu, lg, o);
        const float2 lk = p.lk2[site];
        const bool accept = log2f(ul) < 2.f * (sg > 0.f ? lk.x : lk.y) + lg;  // u == 0: -inf, always accepted
        if (accept) {
            // pass 2: t_j <- (t_j - sigma T_j) / D_j
            auto pass2 = [&](int jp0, bool ragged) {
                float4 t[MT_UNROLL], T[MT_UNROLL];
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    const int jp = jp0 + 32 * k;
                    const bool live = !ragged || jp < MP;
                    T[k] = live ? Trow[jp] : make_float4(0.f, 0.f, 0.f, 0.f);
                    t[k] = live ? t_s[jp] : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    float2 Dr, Di;
                    const float2 d2 = metro_D(t[k], T[k], nsg, Dr, Di);
                    const float2 inv = make_float2(__frcp_rn(d2.x), __frcp_rn(d2.y));
                    const float2 nr = __ffma2_rn(bc2(nsg), make_float2(T[k].x, T[k].y), make_float2(t[k].x, t[k].y));
                    const float2 ni = __ffma2_rn(bc2(nsg), make_float2(T[k].z, T[k].w), make_float2(t[k].z, t[k].w));
                    const float2 outr = __fmul2_rn(__ffma2_rn(nr, Dr, __fmul2_rn(ni, Di)), inv);
                    const float2 outi = __fmul2_rn(__ffma2_rn(ni, Dr, __fmul2_rn(neg2(nr), Di)), inv);
                    const int jp = jp0 + 32 * k;
                    if (!ragged || jp < MP) t_s[jp] = make_float4(outr.x, outr.y, outi.x, outi.y);
                }
            };
            for (int g = 0; g < nFull; ++g) pass2(g * 32 * MT_UNROLL + lane, false);
            if (nFull * 32 * MT_UNROLL < MP) pass2(nFull * 32 * MT_UNROLL + lane, true);
            if (lane == 0) s_s[site] = (int8_t)(-(int)sg);
            ++acc;
        }
        __syncwarp();
    }
    for (int i = lane; i < p.N; i += 32) p.spins[c * p.N + i] = s_s[i];
    if (lane == 0 && p.accepted) p.accepted[c] = p.accumulate ? p.accepted[c] + acc : acc;
}

}  // namespace nqs
