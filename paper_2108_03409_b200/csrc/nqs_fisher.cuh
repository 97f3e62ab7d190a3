// the quantum Fisher matrix (Eq. 10-11; Algorithm 1 line 9;
// jVMC's get_global_covariance, :515)
//   S_{k,k'} = << O_k^* O_k' >>_c = sum_b w_b (O_k(s_b) - <O_k>)^* (O_k'(s_b) - <O_k'>) / sum_b w_b
// for the RBM's logarithmic derivatives O_{a_i} = s_i, O_{b_j} = tanh theta_j, O_{W_ji} = tanh theta_j s_i (Eq. 8).
// With X[k, b] = sqrt(w_b / sum w) (O_k(s_b) - <O_k>) this is the Hermitian rank-B update S = conj(X) X^T: a
// dense contraction over the samples, run on the tensor cores as FP16 tcgen05.mma (kind::f16) with FP32
// accumulators in TMEM.  X is split error-free into two FP16 parts (hi + lo; products hi.hi + hi.lo + lo.hi:
// 22 bits), complex arithmetic is four real MMAs per product (conj(A) B: re = Ar Br + Ai Bi, im = Ar Bi - Ai Br,
// the minus sign by the negate-A bit).  <O_k> comes from the exact int8 contraction of nqs_forces.cuh with the
// coefficient vector w_b / sum w.  Only the tiles of the upper triangle are computed; the epilogue writes the
// mirror image conjugated.
//
//
// Accumulation.  The tensor cores add the 16 products of an MMA step to the FP32 accumulator with the addends
// aligned to the accumulator and truncated, so a long chain of same-sign terms (the diagonal of S: sum_b |X|^2)
// drifts low in proportion to its length (measured: 2.6e-4 relative after 1024 steps at config 2).  The chain
// is therefore kept short: TMEM holds TWO accumulator sets used alternately for groups of FS_GROUP = 8 steps
// (128 samples); while the MMAs fill one set, sixteen epilogue warps drain the other into float32 registers
// with ordinary round-to-nearest additions (64 values per thread), and S is written from the registers.
//
//   fisher_pack_kernel   X planes (hi.re hi.im lo.re lo.im) in the UMMA shared-memory image
//   fisher_gemm_kernel   one CTA per tile pair (kt <= kt') of 128 x 128 parameters, K = samples
#pragma once
#include <cuda_fp16.h>

#include "nqs_device.cuh"
#include "nqs_series.cuh"
#include "nqs_theta_mma.cuh"

namespace nqs {

constexpr int FS_T = 128;                       // parameters per tile (UMMA M and N)
constexpr int FS_PLANES = 4;                    // hi.re hi.im lo.re lo.im
constexpr int FS_PLANE_U4 = 2 * FS_T;           // uint4 per plane: [slab 2][row 128][16 bytes]
constexpr int FS_TILE_STAGE_BYTES = FS_PLANES * FS_PLANE_U4 * 16;  // 16 KB: one tile, 16 samples
constexpr int FS_STAGES = 6;
constexpr size_t FS_SMEM = (size_t)FS_STAGES * 2 * FS_TILE_STAGE_BYTES + 256;
constexpr int FS_EPI_WARPS = 16;                // TMEM lane group (warp % 4) x column quarter (warp / 4)
constexpr int FS_THREADS = 64 + 32 * FS_EPI_WARPS;  // producer, MMA issuer, epilogue warps
constexpr int FS_GROUP = 8;                     // sample chunks (of 16) per accumulation group, see fisher_gemm_kernel
constexpr int FS_MAX_K = 8192;                  // parameters (S is K x K complex64: 512 MB at the limit)

// coefficient vector of the mean: c_b = w_b / sum w (real), 0 for the padding samples.  stats[3] = sum w.
__global__ void fisher_mean_coef_kernel(const float* __restrict__ w, long long B, long long B_pad,
                                        const double* __restrict__ stats, float2* __restrict__ cb,
                                        float* __restrict__ sw) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B_pad) return;
    float c = 0.f;
    if (b < B) c = (float)((w ? (double)w[b] : 1.0) / stats[3]);
    cb[b] = make_float2(c, 0.f);
    sw[b] = sqrtf(c);
}

// X planes.  thread <-> (parameter k, 8 consecutive samples); consecutive threads take consecutive k, so the
// 16-byte stores of a warp are contiguous.  X_packed[ktile][bchunk16][plane][slab 2][row 128][8 halves].
// Fc = sum_b conj(O_k) w_b / sum w (from the force contraction), i.e. <O_k> = conj(Fc[k]).
// spT = the force kernels' transposed spins: spT[(itile * K16 + b16) * 128 + irow] = 16 samples of site i.
__global__ void __launch_bounds__(256) fisher_pack_kernel(const float4* __restrict__ tp, long long nPairsPad,
                                                          const uint4* __restrict__ spT, int K16s,
                                                          const float* __restrict__ sw, const float2* __restrict__ Fc,
                                                          int N, int M, int K, int nKT, long long nB8, float scale,
                                                          uint4* __restrict__ X_packed) {
    const long long total = (long long)nKT * FS_T * nB8;
    const long long nBC = nB8 / 2;
    for (long long idx = blockIdx.x * 256ll + threadIdx.x; idx < total; idx += (long long)gridDim.x * 256) {
        const int k = (int)(idx % ((long long)nKT * FS_T));
        const long long b8 = idx / ((long long)nKT * FS_T);
        float2 x[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) x[q] = make_float2(0.f, 0.f);
        if (k < K) {
            const float2 fc = Fc[k];
            const float obr = fc.x, obi = -fc.y;  // <O_k>
            // which block: a (k < N), b (N <= k < N + M), W (k = N + M + j N + i)
            int i = -1, j = -1;
            if (k < N) i = k;
            else if (k < N + M) j = k - N;
            else {
                j = (k - N - M) / N;
                i = (k - N - M) % N;
            }
            unsigned sp[2] = {0x01010101u, 0x01010101u};  // 8 spins of site i (or +1 for the b block)
            if (i >= 0) {
                const uint4 v = spT[((long long)(i / TM_M) * K16s + (b8 >> 1)) * TM_M + (i % TM_M)];
                sp[0] = (b8 & 1) ? v.z : v.x;
                sp[1] = (b8 & 1) ? v.w : v.y;
            }
            float4 t4[4];
            if (j >= 0) {
#pragma unroll
                for (int q = 0; q < 4; ++q) t4[q] = tp[(long long)j * nPairsPad + b8 * 4 + q];
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float s = (float)(int8_t)((sp[q >> 2] >> (8 * (q & 3))) & 0xff);
                float orr = s, oi = 0.f;
                if (j >= 0) {
                    const float4 t = t4[q >> 1];
                    const float tr = (q & 1) ? t.y : t.x, ti = (q & 1) ? t.w : t.z;
                    orr = tr * s;
                    oi = ti * s;
                }
                const float wq = sw[b8 * 8 + q] * scale;  // 0 for the padding samples
                x[q] = make_float2((orr - obr) * wq, (oi - obi) * wq);
            }
        }
        float hr[8], hi[8], lr[8], li[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            hr[q] = __half2float(__float2half_rn(x[q].x));
            hi[q] = __half2float(__float2half_rn(x[q].y));
            lr[q] = x[q].x - hr[q];
            li[q] = x[q].y - hi[q];
        }
        const int kt = k / FS_T, row = k % FS_T;
        uint4* dst = X_packed + (((long long)kt * nBC + (b8 >> 1)) * FS_PLANES) * FS_PLANE_U4 + (b8 & 1) * FS_T + row;
        dst[0 * FS_PLANE_U4] = make_uint4(pack_h2(hr[0], hr[1]), pack_h2(hr[2], hr[3]), pack_h2(hr[4], hr[5]), pack_h2(hr[6], hr[7]));
        dst[1 * FS_PLANE_U4] = make_uint4(pack_h2(hi[0], hi[1]), pack_h2(hi[2], hi[3]), pack_h2(hi[4], hi[5]), pack_h2(hi[6], hi[7]));
        dst[2 * FS_PLANE_U4] = make_uint4(pack_h2(lr[0], lr[1]), pack_h2(lr[2], lr[3]), pack_h2(lr[4], lr[5]), pack_h2(lr[6], lr[7]));
        dst[3 * FS_PLANE_U4] = make_uint4(pack_h2(li[0], li[1]), pack_h2(li[2], li[3]), pack_h2(li[4], li[5]), pack_h2(li[6], li[7]));
    }
}

struct FisherGemmParams {
    const uint4* X_packed;   // [nKT][nBC][4][256]
    long long nBC;           // sample chunks of 16
    int K, nKT;
    float inv_scale2;
    float2* S;               // [K][K] row-major
    float2* Obar;            // [K] or nullptr (written by the diagonal tiles from Fc)
    const float2* Fc;
};

__global__ void __launch_bounds__(FS_THREADS, 1) fisher_gemm_kernel(const FisherGemmParams p) {
    extern __shared__ __align__(128) unsigned char fs_smem[];
    constexpr uint32_t STAGE = 2 * FS_TILE_STAGE_BYTES;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(fs_smem + (size_t)FS_STAGES * STAGE);
    uint64_t* const full = bars;
    uint64_t* const empty = bars + FS_STAGES;
    uint64_t* const t_full = bars + 2 * FS_STAGES;       // [2]
    uint64_t* const t_empty = bars + 2 * FS_STAGES + 2;  // [2]
    uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * FS_STAGES + 4);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // tile pair of the upper triangle: blockIdx.x = kt' (kt' + 1) / 2 + kt, kt <= kt'
    int ktp = (int)((sqrtf(8.f * (float)blockIdx.x + 1.f) - 1.f) * 0.5f);
    while ((ktp + 1) * (ktp + 2) / 2 <= (int)blockIdx.x) ++ktp;
    while (ktp * (ktp + 1) / 2 > (int)blockIdx.x) --ktp;
    const int kt = (int)blockIdx.x - ktp * (ktp + 1) / 2;
    const long long nBC = p.nBC;
    const long long nGroups = (nBC + FS_GROUP - 1) / FS_GROUP;

    if (tid == 0) {
        for (int s = 0; s < FS_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&t_full[s], 1);
            mbar_init(&t_empty[s], FS_EPI_WARPS);
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            const uint4* gA = p.X_packed + (long long)kt * nBC * FS_PLANES * FS_PLANE_U4;
            const uint4* gB = p.X_packed + (long long)ktp * nBC * FS_PLANES * FS_PLANE_U4;
            for (long long kc = 0; kc < nBC; ++kc) {
                const int s = (int)(kc % FS_STAGES);
                mbar_wait(&empty[s], (uint32_t)(((kc / FS_STAGES) & 1) ^ 1));
                unsigned char* const st = fs_smem + (size_t)s * STAGE;
                mbar_expect_tx(&full[s], STAGE);
                bulk_g2s(st, gA + kc * FS_PLANES * FS_PLANE_U4, FS_TILE_STAGE_BYTES, &full[s]);
                bulk_g2s(st + FS_TILE_STAGE_BYTES, gB + kc * FS_PLANES * FS_PLANE_U4, FS_TILE_STAGE_BYTES, &full[s]);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t s0 = smem_u32(fs_smem);
            const uint32_t idesc = series_idesc(FS_T);
            long long kc = 0;
            for (long long g = 0; g < nGroups; ++g) {
                const int set = (int)(g & 1);
                mbar_wait(&t_empty[set], (uint32_t)(((g >> 1) & 1) ^ 1));
                tc_fence_after();
                const uint32_t d_re = tmem_base + (uint32_t)set * 256u, d_im = d_re + FS_T;
                const long long kend = (kc + FS_GROUP < nBC) ? kc + FS_GROUP : nBC;
                for (bool first = true; kc < kend; ++kc, first = false) {
                    const int s = (int)(kc % FS_STAGES);
                    mbar_wait(&full[s], (uint32_t)((kc / FS_STAGES) & 1));
                    tc_fence_after();
                    const uint32_t sa = s0 + (uint32_t)s * STAGE, sb = sa + FS_TILE_STAGE_BYTES;
                    auto A = [&](int pl) { return umma_desc(sa + (uint32_t)pl * 4096u, 2048u, 128u); };
                    auto Bd = [&](int pl) { return umma_desc(sb + (uint32_t)pl * 4096u, 2048u, 128u); };
                    // conj(a) b for parts (pa, pa + 1 = re, im) x (pb, pb + 1)
                    auto cprod = [&](int pa, int pb, uint32_t acc) {
                        umma_f16(d_re, A(pa), Bd(pb), idesc, acc);
                        umma_f16(d_re, A(pa + 1), Bd(pb + 1), idesc, 1u);
                        umma_f16(d_im, A(pa), Bd(pb + 1), idesc, acc);
                        umma_f16(d_im, A(pa + 1), Bd(pb), idesc | SR_IDESC_NEG_A, 1u);
                    };
                    cprod(0, 0, first ? 0u : 1u);  // hi . hi
                    cprod(0, 2, 1u);               // hi . lo
                    cprod(2, 0, 1u);               // lo . hi
                    tc_commit(&empty[s]);
                }
                tc_commit(&t_full[set]);
            }
        }
    } else {
        const int ew = warp - 2;
        const int lane_grp = warp & 3, quarter = ew >> 2;  // warps 2..17: (warp & 3) covers all four lane groups
        const int row = lane_grp * 32 + lane;
        const int k = kt * FS_T + row;
        if (kt == ktp && quarter == 0 && p.Obar && k < p.K) {
            const float2 fc = p.Fc[k];
            p.Obar[k] = make_float2(fc.x, -fc.y);
        }
        float accr[32], acci[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) accr[q] = 0.f, acci[q] = 0.f;
        for (long long g = 0; g < nGroups; ++g) {
            const int set = (int)(g & 1);
            mbar_wait(&t_full[set], (uint32_t)((g >> 1) & 1));
            tc_fence_after();
            const uint32_t tb = tmem_base + ((uint32_t)(lane_grp * 32) << 16) + (uint32_t)set * 256u + (uint32_t)quarter * 32u;
            int vr[32], vi[32];
            tmem_ld32_nowait(tb, vr);
            tmem_ld32_nowait(tb + FS_T, vi);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&t_empty[set]);
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                accr[q] += __int_as_float(vr[q]);
                acci[q] += __int_as_float(vi[q]);
            }
        }
        if (k < p.K) {
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                const int kp = ktp * FS_T + quarter * 32 + q;
                if (kp >= p.K || kp < k) continue;  // diagonal tile: the lower part is the mirror of the upper one
                const float2 v = make_float2(accr[q] * p.inv_scale2, kp == k ? 0.f : acci[q] * p.inv_scale2);
                p.S[(long long)k * p.K + kp] = v;
                if (kp != k) p.S[(long long)kp * p.K + k] = make_float2(v.x, -v.y);  // Hermitian mirror
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
}

}  // namespace nqs
