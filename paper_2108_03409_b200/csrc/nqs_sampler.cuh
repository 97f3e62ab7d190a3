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

// One block per site i: TT[i][j] = tanh(2 W_ji) (0 for the padding j >= M) and
// lk2[i] = log2(e) * (Re L_i - 2 Re a_i, Re L_i + 2 Re a_i),  L_i = sum_j log cosh(2 W_ji):
// log2 |exp(-2 sigma a_i) prod_j cosh 2 W_ji|^2 / 2 for sigma = +1 (x) and -1 (y).
__global__ void __launch_bounds__(256) site_table_kernel(const float2* __restrict__ W, const float2* __restrict__ a,
                                                         int N, int M, int M_pad, float2* __restrict__ TT,
                                                         float2* __restrict__ lk2) {
    const int i = blockIdx.x;
    __shared__ double sh[256];
    double acc = 0.0;
    for (int j = threadIdx.x; j < M_pad; j += 256) {
        float2 t = make_float2(0.f, 0.f);
        if (j < M) {
            const float2 w = W[(long long)j * N + i];
            float lr, li;
            lncosh_tanh(2.f * w.x, 2.f * w.y, lr, li, t.x, t.y);
            acc += (double)lr;
        }
        TT[(long long)i * M_pad + j] = t;
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
    const float2* TT;        // [N][M_pad]
    const float2* lk2;       // [N]
    const int* sites;        // [S][C]
    const float* u;          // [S][C]
    int* accepted;           // [C] or nullptr
    int accumulate;          // add to accepted[] instead of overwriting it
};

__host__ __device__ inline size_t metropolis_smem_bytes(int cpb, int N, int M_pad) {
    return (size_t)cpb * ((size_t)M_pad * sizeof(float2) + (size_t)((N + 15) / 16 * 16));
}

constexpr int MT_UNROLL = 8;

template <int CPB>
__global__ void __launch_bounds__(CPB * 32) metropolis_kernel(const MetroParams p) {
    extern __shared__ __align__(16) unsigned char mt_smem[];
    float2* const t_all = reinterpret_cast<float2*>(mt_smem);
    const int N_pad = (p.N + 15) / 16 * 16;
    int8_t* const s_all = reinterpret_cast<int8_t*>(mt_smem + (size_t)CPB * p.M_pad * sizeof(float2));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long c0 = (long long)blockIdx.x * CPB;

    // the block's CPB chains are CPB/2 consecutive records of every tp row
    for (int idx = tid; idx < p.M_pad * (CPB / 2); idx += CPB * 32) {
        const int j = idx / (CPB / 2), pr = idx % (CPB / 2);
        const float4 r = p.tp[(long long)j * p.nPairsPad + c0 / 2 + pr];
        t_all[(size_t)(2 * pr) * p.M_pad + j] = make_float2(r.x, r.z);
        t_all[(size_t)(2 * pr + 1) * p.M_pad + j] = make_float2(r.y, r.w);
    }
    for (int idx = tid; idx < CPB * p.N; idx += CPB * 32) {
        const int w = idx / p.N, i = idx % p.N;
        s_all[w * N_pad + i] = (c0 + w < p.C) ? p.spins[(c0 + w) * p.N + i] : (int8_t)1;
    }
    __syncthreads();

    const long long c = c0 + warp;
    if (c >= p.C) return;
    float2* const t_s = t_all + (size_t)warp * p.M_pad;
    int8_t* const s_s = s_all + warp * N_pad;
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
        const float sg = (float)s_s[site];
        const float2* const Trow = p.TT + (long long)site * p.M_pad;
        // pass 1: log2 prod_j |D_j|^2, eight hidden units per lane at a time (loads issued together)
        float lg = 0.f;
        for (int j0 = lane; j0 < p.M; j0 += 32 * MT_UNROLL) {
            float2 t[MT_UNROLL], T[MT_UNROLL];
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                const int j = j0 + 32 * k;
                const bool live = j < p.M;  // t = T = 0 gives D = 1
                T[k] = live ? Trow[j] : make_float2(0.f, 0.f);
                t[k] = live ? t_s[j] : make_float2(0.f, 0.f);
            }
            float q = 1.f;
#pragma unroll
            for (int k = 0; k < MT_UNROLL; ++k) {
                const float xr = fmaf(t[k].x, T[k].x, -t[k].y * T[k].y), xi = fmaf(t[k].x, T[k].y, t[k].y * T[k].x);
                const float Dr = fmaf(-sg, xr, 1.f), Di = -sg * xi;
                q *= fmaf(Dr, Dr, Di * Di);
            }
            lg += log2f(q);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lg += __shfl_xor_sync(0xffffffffu, lg, o);
        const float2 lk = p.lk2[site];
        const bool accept = log2f(ul) < 2.f * (sg > 0.f ? lk.x : lk.y) + lg;  // u == 0: -inf, always accepted
        if (accept) {
            // pass 2: t_j <- (t_j - sigma T_j) / D_j
            for (int j0 = lane; j0 < p.M; j0 += 32 * MT_UNROLL) {
                float2 t[MT_UNROLL], T[MT_UNROLL];
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    const int j = j0 + 32 * k;
                    const bool live = j < p.M;
                    T[k] = live ? Trow[j] : make_float2(0.f, 0.f);
                    t[k] = live ? t_s[j] : make_float2(0.f, 0.f);
                }
#pragma unroll
                for (int k = 0; k < MT_UNROLL; ++k) {
                    const float xr = fmaf(t[k].x, T[k].x, -t[k].y * T[k].y), xi = fmaf(t[k].x, T[k].y, t[k].y * T[k].x);
                    const float Dr = fmaf(-sg, xr, 1.f), Di = -sg * xi;
                    const float inv = __frcp_rn(fmaf(Dr, Dr, Di * Di));
                    const float nr = fmaf(-sg, T[k].x, t[k].x), ni = fmaf(-sg, T[k].y, t[k].y);
                    if (j0 + 32 * k < p.M)
                        t_s[j0 + 32 * k] = make_float2(fmaf(nr, Dr, ni * Di) * inv, fmaf(ni, Dr, -nr * Di) * inv);
                }
            }
            if (lane == 0) s_s[site] = (int8_t)(-(int)sg);
            ++acc;
        }
        __syncwarp();
    }
    for (int i = lane; i < p.N; i += 32) p.spins[c * p.N + i] = s_s[i];
    if (lane == 0 && p.accepted) p.accepted[c] = p.accumulate ? p.accepted[c] + acc : acc;
}

}  // namespace nqs
