// batch statistics of E_loc (Eq. 5) and the
// force vector F_k = <<E_loc O_k^*>>^c (Eq. 16, :134-138; Eq. 7-8, :81-93) for the RBM of Eq. 38,
//   O_{a_i} = s_i,   O_{b_j} = tanh theta_j,   O_{W_ji} = tanh theta_j s_i.
// With c_b = w_b (E_b - mean E) / sum w  (centred: <<AB>>^c = <<A (B - <<B>>)>>) all three blocks are
// ONE dense contraction over the samples,
//   F[j', i'] = sum_b G[b, j'] S[b, i'],   G[b, j] = conj(t_bj) c_b,  G[b, M] = c_b,
//                                          S[b, i] = s_bi,            S[b, N] = 1,
// (row M = the a-part, column N = the b-part, the rest = the W-part), run on the tensor cores as
// an EXACT integer GEMM like a2: S is +-1 / 0 / 1 in int8, G is split per hidden unit into four
// balanced base-128 digits of a 28-bit fixed-point value; the int8 MMAs accumulate exactly in
// int32 (|sum| <= 64 B <= 2^31 for B <= 2^25), so the result is independent of the summation
// order and deterministic.
//
//   A = S^T     [128 sites]  x [K = samples] int8, K-major core-matrix layout
//   B = digits  [256 = 32 hidden x (re, im) x 4 digits] x [K] int8, same layout
//   D = A B^T   [128 lanes] x [256 columns] int32 in TMEM
// One CTA per (site tile, hidden tile); both operands stream through a ring of bulk copies.
#pragma once
#include <climits>

#include "nqs_device.cuh"
#include "nqs_theta_mma.cuh"

namespace nqs {

constexpr int FM_STAGES = 6;
constexpr int FM_A_STAGE_BYTES = TM_A_K16_BYTES * (TM_KC / 16);   //  8 KB: 64 samples x 128 sites
constexpr int FM_B_STAGE_BYTES = TM_B_STAGE_BYTES;                // 16 KB: 64 samples x 256 columns
constexpr int FM_STAGE_BYTES = FM_A_STAGE_BYTES + FM_B_STAGE_BYTES;
constexpr size_t FM_SMEM = (size_t)FM_STAGES * FM_STAGE_BYTES + 256;
constexpr int ST_BLOCKS = 256;

// ---------------------------------------------------------------------------------------
// Eq. 5: sums in double, fixed order (deterministic).  partial[blk] = {sum w, sum w Re E, sum w Im E,
// sum w |E|^2}; stats = {Re mean, Im mean, variance = <<|E|^2>> - |mean|^2, sum w}.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) stats_partial_kernel(const float2* __restrict__ x, const float* __restrict__ w,
                                                            long long B, double* __restrict__ partial) {
    __shared__ double sh[4][256];
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    for (long long b = blockIdx.x * 256ll + threadIdx.x; b < B; b += (long long)gridDim.x * 256) {
        const float2 e = x ? x[b] : make_float2(0.f, 0.f);  // x == nullptr: only the sum of the weights
        const double wb = w ? (double)w[b] : 1.0, er = e.x, ei = e.y;
        s0 += wb;
        s1 += wb * er;
        s2 += wb * ei;
        s3 += wb * (er * er + ei * ei);
    }
    sh[0][threadIdx.x] = s0, sh[1][threadIdx.x] = s1, sh[2][threadIdx.x] = s2, sh[3][threadIdx.x] = s3;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 4) partial[blockIdx.x * 4 + threadIdx.x] = sh[threadIdx.x][0];
}

// one warp: lane l adds the partials l, l + 32, ... in that order, lane 0 then adds the 32 lane sums in lane order
// (a fixed order: deterministic; the 1024 dependent loads of a single thread took 40 us)
__global__ void stats_final_kernel(const double* __restrict__ partial, int nblk, double* __restrict__ stats) {
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    const int lane = threadIdx.x;
    double s[4] = {0, 0, 0, 0};
    for (int k = lane; k < nblk; k += 32)
        for (int q = 0; q < 4; ++q) s[q] += partial[k * 4 + q];
    double t[4] = {0, 0, 0, 0};
    for (int l = 0; l < 32; ++l)
        for (int q = 0; q < 4; ++q) t[q] += __shfl_sync(0xffffffffu, s[q], l);
    if (lane != 0) return;
    const double mr = t[1] / t[0], mi = t[2] / t[0];
    stats[0] = mr;
    stats[1] = mi;
    stats[2] = t[3] / t[0] - (mr * mr + mi * mi);
    stats[3] = t[0];
}

// c_b = w_b (E_b - mean) / sum w as float2; 0 for the padding samples b >= B
__global__ void force_coef_kernel(const float2* __restrict__ eloc, const float* __restrict__ w, long long B,
                                  long long B_pad, const double* __restrict__ stats, float2* __restrict__ cb) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B_pad) return;
    float2 c = make_float2(0.f, 0.f);
    if (b < B) {
        const double f = (w ? (double)w[b] : 1.0) / stats[3];
        c = make_float2((float)(f * ((double)eloc[b].x - stats[0])), (float)(f * ((double)eloc[b].y - stats[1])));
    }
    cb[b] = c;
}

// G[b, j] = conj(t_bj) c_b for the two samples of a pair (j == M: the constant row, G = c_b)
__device__ __forceinline__ void force_g_pair(const float4 t, const float2 c0, const float2 c1, bool ones, float2& g0,
                                             float2& g1) {
    if (ones) {
        g0 = c0;
        g1 = c1;
    } else {  // (tr - i ti)(cr + i ci)
        g0 = make_float2(fmaf(t.x, c0.x, t.z * c0.y), fmaf(t.x, c0.y, -t.z * c0.x));
        g1 = make_float2(fmaf(t.y, c1.x, t.w * c1.y), fmaf(t.y, c1.y, -t.w * c1.x));
    }
}

// One block per row j' in [0, nJT*32): power-of-two scale from max_b max(|Re G|, |Im G|).
// gexp[j'] = e with max = f 2^e, f in [0.5, 1); INT_MIN marks an all-zero (or padding) row.
__global__ void __launch_bounds__(256) force_gscale_kernel(const float4* __restrict__ tp, long long nPairsPad,
                                                           const float2* __restrict__ cb, int M,
                                                           int* __restrict__ gexp) {
    const int j = blockIdx.x;
    __shared__ float smax[8];
    float mx = 0.f;
    if (j <= M)
        for (long long pr = threadIdx.x; pr < nPairsPad; pr += 256) {
            const float4 t = (j < M) ? tp[(long long)j * nPairsPad + pr] : make_float4(0.f, 0.f, 0.f, 0.f);
            float2 g0, g1;
            force_g_pair(t, cb[2 * pr], cb[2 * pr + 1], j == M, g0, g1);
            mx = fmaxf(mx, fmaxf(fmaxf(fabsf(g0.x), fabsf(g0.y)), fmaxf(fabsf(g1.x), fabsf(g1.y))));
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0) smax[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) mx = fmaxf(mx, smax[k]);
        int e = INT_MIN;
        if (mx > 0.f && isfinite(mx)) (void)frexpf(mx, &e);
        gexp[j] = e;
    }
}

// B operand: thread <-> (row j', k16 = 16 consecutive samples), consecutive threads <-> consecutive j'.  G 2^(27-e) rounded to an integer Q,
// |Q| <= 2^27, digits d0..d3: Q = d0 + 128 d1 + 128^2 d2 + 128^3 d3, d0..d2 in [-64, 63].
// B_packed[jtile][k16][n = 8*jl + 4*part + digit][16 bytes]: a thread writes one 128-byte line.
__global__ void __launch_bounds__(256) force_pack_g_kernel(const float4* __restrict__ tp, long long nPairsPad,
                                                           const float2* __restrict__ cb, int M, int K16, int nJT,
                                                           const int* __restrict__ gexp,
                                                           uint4* __restrict__ B_packed) {
    const long long total = (long long)nJT * TM_JT * K16;
    for (long long idx = blockIdx.x * 256ll + threadIdx.x; idx < total; idx += (long long)gridDim.x * 256) {
        // lanes <-> 32 consecutive hidden units of one 16-sample slab: a warp writes one contiguous 4 KB block of
        // B_packed and reads whole 128-byte lines of tp (each lane its own), the coefficients by broadcast
        const int nJ = nJT * TM_JT;
        const int j = (int)(idx % nJ);
        const int k16 = (int)(idx / nJ);
        const int e = gexp[j];
        unsigned d[2][4][4];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int l = 0; l < 4; ++l)
#pragma unroll
                for (int q = 0; q < 4; ++q) d[p][l][q] = 0u;
        if (j <= M && e != INT_MIN) {
#pragma unroll
            for (int pp = 0; pp < 8; ++pp) {
                const long long pr = (long long)k16 * 8 + pp;
                const float4 t = (j < M) ? tp[(long long)j * nPairsPad + pr] : make_float4(0.f, 0.f, 0.f, 0.f);
                float2 g[2];
                force_g_pair(t, cb[2 * pr], cb[2 * pr + 1], j == M, g[0], g[1]);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int k = 2 * pp + h;
#pragma unroll
                    for (int p = 0; p < 2; ++p) {
                        int Q = __float2int_rn(ldexpf(p ? g[h].y : g[h].x, 27 - e));
#pragma unroll
                        for (int l = 0; l < 3; ++l) {
                            const int dl = ((Q + 64) & 127) - 64;
                            Q = (Q - dl) >> 7;
                            d[p][l][k >> 2] |= (unsigned)(uint8_t)(int8_t)dl << (8 * (k & 3));
                        }
                        d[p][3][k >> 2] |= (unsigned)(uint8_t)(int8_t)Q << (8 * (k & 3));
                    }
                }
            }
        }
        const int jt = j / TM_JT, jl = j % TM_JT;
        uint4* dst = B_packed + ((long long)jt * K16 + k16) * TM_N + jl * 8;
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int l = 0; l < 4; ++l) dst[p * 4 + l] = make_uint4(d[p][l][0], d[p][l][1], d[p][l][2], d[p][l][3]);
    }
}

// A operand = S^T: A_packed[itile][k16][row i'][16 bytes] = S[16 k16 .. 16 k16 + 15][i'];
// i' < N: the spin, i' == N: 1 (the b-part column), else 0; samples b >= B: 0.
__global__ void __launch_bounds__(256) force_pack_spins_kernel(const int8_t* __restrict__ spins, long long B, int N,
                                                               int K16, int nIT, uint4* __restrict__ A_packed) {
    const long long total = (long long)nIT * K16 * TM_M;
    for (long long idx = blockIdx.x * 256ll + threadIdx.x; idx < total; idx += (long long)gridDim.x * 256) {
        const int row = (int)(idx % TM_M);
        const int k16 = (int)((idx / TM_M) % K16);
        const int it = (int)(idx / ((long long)TM_M * K16));
        const int i = it * TM_M + row;
        unsigned w[4] = {0, 0, 0, 0};
        if (i <= N) {
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const long long b = (long long)k16 * 16 + k;
                if (b < B) {
                    const int8_t v = (i < N) ? spins[b * N + i] : (int8_t)1;
                    w[k >> 2] |= (unsigned)(uint8_t)v << (8 * (k & 3));
                }
            }
        }
        A_packed[idx] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// ---------------------------------------------------------------------------------------
// the GEMM: one CTA per (site tile, hidden tile).  Warp 0 = bulk-copy producer, warp 1 = TMEM
// allocator + MMA issuer (one elected lane), warps 2..5 = epilogue (one TMEM lane group each).
// ---------------------------------------------------------------------------------------
struct ForceMmaParams {
    const uint4* A_packed;   // [nIT][K16][128]
    const uint4* B_packed;   // [nJT][K16][256]
    const int* gexp;         // [nJT*32]
    int N, M, K16;
    float2* F;               // [N + M + M*N]: a-part, b-part, W-part (row-major [M,N])
};
constexpr int FM_THREADS = 192;

__global__ void __launch_bounds__(FM_THREADS, 1) force_mma_kernel(const ForceMmaParams p) {
    extern __shared__ __align__(128) unsigned char fm_smem[];
    uint64_t* const bars = reinterpret_cast<uint64_t*>(fm_smem + (size_t)FM_STAGES * FM_STAGE_BYTES);
    uint64_t* const full = bars;
    uint64_t* const empty = bars + FM_STAGES;
    uint64_t* const t_full = bars + 2 * FM_STAGES;
    uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * FM_STAGES + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int it = blockIdx.x, jt = blockIdx.y;
    const int K16 = p.K16;
    const int nKC = K16 / (TM_KC / 16);

    if (tid == 0) {
        for (int s = 0; s < FM_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        mbar_init(t_full, 1);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, TM_N);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            const uint4* gA = p.A_packed + (long long)it * K16 * TM_M;
            const uint4* gB = p.B_packed + (long long)jt * K16 * TM_N;
            for (int kc = 0; kc < nKC; ++kc) {
                const int s = kc % FM_STAGES;
                mbar_wait(&empty[s], ((kc / FM_STAGES) & 1) ^ 1);
                unsigned char* const st = fm_smem + (size_t)s * FM_STAGE_BYTES;
                mbar_expect_tx(&full[s], FM_STAGE_BYTES);
                bulk_g2s(st, gA + (long long)kc * (TM_KC / 16) * TM_M, FM_A_STAGE_BYTES, &full[s]);
                bulk_g2s(st + FM_A_STAGE_BYTES, gB + (long long)kc * (TM_KC / 16) * TM_N, FM_B_STAGE_BYTES, &full[s]);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t s0 = smem_u32(fm_smem);
            for (int kc = 0; kc < nKC; ++kc) {
                const int s = kc % FM_STAGES;
                mbar_wait(&full[s], (kc / FM_STAGES) & 1);
                tc_fence_after();
                const uint32_t sa = s0 + (uint32_t)s * FM_STAGE_BYTES, sb = sa + FM_A_STAGE_BYTES;
#pragma unroll
                for (int ks = 0; ks < TM_KC / 32; ++ks) {
                    const uint64_t ad = umma_desc(sa + (uint32_t)(ks * 2) * TM_A_K16_BYTES, TM_A_K16_BYTES, 128);
                    const uint64_t bd = umma_desc(sb + (uint32_t)(ks * 2) * TM_B_K16_BYTES, TM_B_K16_BYTES, 128);
                    umma_i8(tmem_base, ad, bd, TM_IDESC, (kc | ks) ? 1u : 0u);
                }
                tc_commit(&empty[s]);  // frees the stage once these MMAs have read it
            }
            tc_commit(t_full);
        }
    } else {
        const int lane_grp = warp & 3;
        const int i = it * TM_M + lane_grp * 32 + lane;
        mbar_wait(t_full, 0);
        tc_fence_after();
#pragma unroll 1
        for (int q = 0; q < 8; ++q) {  // 4 hidden units per TMEM load
            int v[32];
            tmem_ld32(tmem_base + ((uint32_t)(lane_grp * 32) << 16) + (uint32_t)(q * 32), v);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int j = jt * TM_JT + q * 4 + u;
                if (j > p.M || i > p.N || (j == p.M && i == p.N)) continue;
                const int e = p.gexp[j];
                float2 f = make_float2(0.f, 0.f);
                if (e != INT_MIN) {
                    const int* w = &v[u * 8];
                    const double re = (((double)w[3] * 128.0 + (double)w[2]) * 128.0 + (double)w[1]) * 128.0 + (double)w[0];
                    const double im = (((double)w[7] * 128.0 + (double)w[6]) * 128.0 + (double)w[5]) * 128.0 + (double)w[4];
                    f = make_float2((float)ldexp(re, e - 27), (float)ldexp(im, e - 27));
                }
                long long k;
                if (j == p.M) k = i;                                   // a-part: sum_b c_b s_bi
                else if (i == p.N) k = (long long)p.N + j;             // b-part: sum_b conj(t_bj) c_b
                else k = (long long)p.N + p.M + (long long)j * p.N + i;
                p.F[k] = f;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, TM_N);
    }
}

}  // namespace nqs
