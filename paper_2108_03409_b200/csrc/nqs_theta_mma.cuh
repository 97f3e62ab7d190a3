// a2 on the 5th-generation tensor cores (tcgen05, sm_100a): theta = b + W s as an EXACT integer GEMM.
//
// theta[b, j] = b_j + sum_i W_ji s_bi  (Eq. 30 / Eq. 38) is a dense
// [B, N] x [N, 2M] contraction with s = +-1 exactly representable in int8.  W is split per hidden
// unit into four balanced base-128 digits of a 28-bit fixed-point value (error-compensated split:
// the four int8 GEMMs accumulate exactly in int32, so the only error is the 2^-28 * max_i |W_ji|
// quantisation -- below float32's own rounding of W -- and there is no accumulation-order or
// tensor-core truncation error at all).  north_star: "tensor cores only if an error-compensated
// split meets tolerance".
//
//   A = spins   [128 samples] x [K]  int8, K-major, canonical no-swizzle core-matrix layout
//   B = digits  [256 = 32 hidden x (re, im) x 4 digits] x [K] int8, K-major, same layout
//   D = A B^T   [128 lanes] x [256 columns] int32 in TMEM  (tcgen05.mma.cta_group::1.kind::i8)
//
// Both operands are pre-packed in global memory in exactly the shared-memory image the MMA wants
// ([k16][row][16 bytes]), so every pipeline stage is ONE contiguous cp.async.bulk (TMA engine).
// CTA = 128 samples (TM_THREADS = 320: warp 0 = bulk-copy producer, warp 1 = TMEM allocator + MMA issuer with one
// elected lane, warps 2..9 = epilogue: tcgen05.ld -> theta -> log cosh, tanh -> log psi, tp / series planes).  A CTA
// loops over its hidden tiles of TH_JT = 16 units (the constants further down; TM_JT = 32 below is the tile of the
// force / Fisher kernels that share this file's operand layout) with two accumulator sets in TMEM, so the MMAs of the
// next tile overlap the epilogue of the current one; two CTAs per SM share the 512 TMEM columns.  On the series path
// the hidden tiles of a sample tile may be split over 1, 2, 4 or 8 CTAs (NQS_OPT_THETA_SPLIT): log psi and the row norms
// are then partial sums combined in a fixed order by series_guard_kernel / series_gemm_kernel.
#pragma once
#include <cuda_fp16.h>

#include "nqs_device.cuh"

namespace nqs {

constexpr int TM_M = 128;       // samples per CTA (UMMA M)
constexpr int TM_JT = 32;       // hidden units per accumulator tile
constexpr int TM_N = 256;       // accumulator columns = TM_JT * 2 * 4
constexpr int TM_KC = 64;       // K bytes per B stage (two K=32 MMAs)
constexpr int TM_STAGES = 3;
constexpr int TM_A_K16_BYTES = TM_M * 16;   // one 16-byte K slab of the A tile
constexpr int TM_B_K16_BYTES = TM_N * 16;
constexpr int TM_B_STAGE_BYTES = TM_B_K16_BYTES * (TM_KC / 16);
constexpr int TM_THREADS = 320;
constexpr int TM_MAX_KPAD = 512;

// theta_mma_kernel itself works on tiles of 16 hidden units (128 accumulator columns) and keeps TWO accumulator
// sets in TMEM, so that the MMAs of tile nt + 1 run while the epilogue warps are still on tile nt
constexpr int TH_JT = 16;       // hidden units per accumulator tile
constexpr int TH_N = 128;       // accumulator columns = TH_JT * 2 * 4
constexpr int TH_STAGES = 6;
constexpr int TH_B_K16_BYTES = TH_N * 16;
constexpr int TH_B_STAGE_BYTES = TH_B_K16_BYTES * (TM_KC / 16);  // 8 KB

__host__ __device__ inline size_t theta_mma_smem_bytes(int K_pad) {
    return (size_t)(K_pad / 16) * TM_A_K16_BYTES + (size_t)TH_STAGES * TH_B_STAGE_BYTES + 256;
}

// ---------------------------------------------------------------------------------------
// operand packing
// ---------------------------------------------------------------------------------------
// A_packed[mtile][k16][row 0..127][16 bytes] = spins[mtile*128 + row][16*k16 .. +16), zero padded
__global__ void pack_spins_kernel(const int8_t* __restrict__ spins, long long B, int N, int K16, long long nMT,
                                  uint4* __restrict__ A_packed, const int* __restrict__ gate) {
    if (gate && !(gate[0] & 1)) return;
    const long long total = nMT * K16 * TM_M;
    const bool vec = (N % 16 == 0) && ((reinterpret_cast<uintptr_t>(spins) & 15) == 0);
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(idx % TM_M);
        const int k16 = (int)((idx / TM_M) % K16);
        const long long mt = idx / ((long long)TM_M * K16);
        const long long b = mt * TM_M + row;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (b < B) {
            const int i0 = k16 * 16;
            if (vec && i0 + 16 <= N) {
                v = *reinterpret_cast<const uint4*>(spins + b * N + i0);
            } else {
                unsigned w[4] = {0, 0, 0, 0};
                for (int k = 0; k < 16; ++k)
                    if (i0 + k < N) w[k >> 2] |= (unsigned)(uint8_t)spins[b * N + i0 + k] << (8 * (k & 3));
                v = make_uint4(w[0], w[1], w[2], w[3]);
            }
        }
        A_packed[idx] = v;
    }
}

// One block per hidden unit j (padded to nNT*32): power-of-two scale from the row maximum, then
// W_ji * 2^(27-e) rounded to an integer Q, |Q| <= 2^27, written as digits d0..d3 in [-64, 64]:
//   Q = d0 + 128 d1 + 128^2 d2 + 128^3 d3.
// B_packed[ntile16][k16][n = 8*jl + 4*part + digit][16 bytes] (tiles of TH_JT = 16 units);  scale[j] = 2^(e-27).
__global__ void __launch_bounds__(128) pack_w_kernel(const float2* __restrict__ W, int N, int M, int K16,
                                                     uint4* __restrict__ B_packed, float* __restrict__ scale,
                                                     const int* __restrict__ gate) {
    if (gate && !(gate[0] & 1)) return;
    const int j = blockIdx.x;
    const int tid = threadIdx.x;
    __shared__ float smax[4];
    float mx = 0.f;
    if (j < M)
        for (int i = tid; i < N; i += 128) {
            const float2 w = W[(long long)j * N + i];
            mx = fmaxf(mx, fmaxf(fabsf(w.x), fabsf(w.y)));
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((tid & 31) == 0) smax[tid >> 5] = mx;
    __syncthreads();
    mx = fmaxf(fmaxf(smax[0], smax[1]), fmaxf(smax[2], smax[3]));
    int e = 0;
    if (mx > 0.f) (void)frexpf(mx, &e);  // mx = f * 2^e, f in [0.5, 1)
    if (tid == 0) scale[j] = (mx > 0.f && j < M) ? ldexpf(1.f, e - 27) : 0.f;
    const int nt = j / TH_JT, jl = j % TH_JT;
    for (int item = tid; item < 2 * K16; item += 128) {
        const int part = item & 1, k16 = item >> 1;
        unsigned d[4][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
        if (j < M && mx > 0.f) {
            for (int k = 0; k < 16; ++k) {
                const int i = k16 * 16 + k;
                if (i < N) {
                    const float2 w = W[(long long)j * N + i];
                    int Q = __float2int_rn(ldexpf(part ? w.y : w.x, 27 - e));
#pragma unroll
                    for (int l = 0; l < 3; ++l) {
                        const int dl = ((Q + 64) & 127) - 64;
                        Q = (Q - dl) >> 7;
                        d[l][k >> 2] |= (unsigned)(uint8_t)(int8_t)dl << (8 * (k & 3));
                    }
                    d[3][k >> 2] |= (unsigned)(uint8_t)(int8_t)Q << (8 * (k & 3));
                }
            }
        }
        uint4* dst = B_packed + ((long long)nt * K16 + k16) * TH_N + jl * 8 + part * 4;
#pragma unroll
        for (int l = 0; l < 4; ++l) dst[l] = make_uint4(d[l][0], d[l][1], d[l][2], d[l][3]);
    }
}

// ---------------------------------------------------------------------------------------
// tcgen05 / TMEM PTX wrappers
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t* slot, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, int8 x int8 -> int32
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}
// K-major, no swizzle: 8-row x 16-byte core matrices; LBO = byte step between the two 16-byte K slabs
// of one K=32 MMA, SBO = byte step between 8-row groups; descriptor version 1 (Blackwell).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46);
}
constexpr uint32_t TM_IDESC = (2u << 4) /* D = S32 */ | (1u << 7) /* A = INT8 */ | (1u << 10) /* B = INT8 */ |
                              ((uint32_t)(TM_N >> 3) << 17) | ((uint32_t)(TM_M >> 4) << 24);
constexpr uint32_t TH_IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TH_N >> 3) << 17) | ((uint32_t)(TM_M >> 4) << 24);

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, int (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, int (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------
// Series operands of the a5 GEMM (nqs_series.cuh), written straight from the epilogue when sA != nullptr:
//   sA[mtile][jchunk16][plane 8][slab 2][row 128][8 halves]   planes: 16 t (hi.re hi.im lo.re lo.im), 16 t^2 (re im),
//   16 t^3 (re im);   rown[b] = (n2t, n4t, n6t, n8t), nPt = sqrt(sum_j |t_bj|^P);   rowmax[b] = max_j |t_bj|
constexpr float TM_SERIES_SA = 16.f;  // == SR_SA of nqs_series.cuh (static_assert there)

// Index (in planes) of plane pl (0 .. 7: hi.re hi.im lo.re lo.im sq.re sq.im cu.re cu.im) of chunk jc of tile `tile` in a
// packed operand array of nTiles x nJC chunks.  Narrow layout: eight planes per chunk, contiguous.  Wide layout (column
// tiles of up to 224, nqs_series.cuh): the six planes of the ODD pass per chunk, contiguous, and behind all of them the
// two square planes of every chunk, contiguous over the chunks of a tile -- one bulk copy fetches three chunks of them.
__host__ __device__ inline long long series_plane_index(bool wide, long long tile, int jc, int pl, long long nTiles, int nJC) {
    if (!wide) return (tile * nJC + jc) * 8 + pl;
    if (pl == 4 || pl == 5) return nTiles * nJC * 6 + (tile * nJC + jc) * 2 + (pl - 4);
    return (tile * nJC + jc) * 6 + (pl < 4 ? pl : pl - 2);
}

struct ThetaMmaParams {
    const uint4* A_packed;   // [nMT][K16][128]
    const uint4* B_packed;   // [nNT][K16][256]
    const float* scale;      // [nNT*32]
    const float2* bvec;      // [M]
    const float2* a;         // [N]
    const int8_t* spins;     // [B][N]
    long long B;
    int N, M, M_pad, K16, nNT;
    float4* tp;              // [M_pad][nPairsPad] or nullptr
    long long nPairsPad;
    float2* logpsi;          // [B] or nullptr
    int raw_theta;           // 1: tp receives theta itself instead of tanh(theta) (nqs_metropolis)
    uint4* sA;               // series operand planes or nullptr
    int sA_wide;             // their layout (series_plane_index)
    long long sA_tiles;      // sample tiles in sA
    float4* rown;            // [rows] (with sA)
    float* rowmax;           // [rows] (with sA)
    const int* gate;         // nullptr, or: run only if (gate[0] & 1) -- the series guard failed (fallback pass)
    // S > 1 (series path only): the hidden-unit tiles of a sample tile are split over S CTAs (grid = sample tiles x S)
    // so that the grid is a near-whole number of waves of the 2 x 148 CTA slots; every CTA then leaves PARTIAL sums
    //   lp_part[js][b] = (Re, Im) of its share of log psi (float64; the visible bias a.s rides in js = 0)
    //   rown[js][b]    = (sum |t|^2, sum |t|^4, sum |t|^6, sum |t|^8) (no square root),  rowmax[js][b] = max |t|^2
    // which series_gemm_kernel / series_guard_kernel combine in a fixed order.
    int S;
    double2* lp_part;        // [S][rows] (S > 1)
    long long rows;          // padded number of rows = stride of the partial arrays
};

__device__ __forceinline__ unsigned tm_pack_h2(float2 v) {
    const __half2 h = __float22half2_rn(v);
    return *reinterpret_cast<const unsigned*>(&h);
}
__device__ __forceinline__ float2 tm_unpack_h2(unsigned u) { return __half22float2(*reinterpret_cast<const __half2*>(&u)); }

__global__ void __launch_bounds__(TM_THREADS, 2) theta_mma_kernel(const ThetaMmaParams p) {
    extern __shared__ __align__(128) unsigned char tm_smem[];
    if (p.gate && !(p.gate[0] & 1)) return;
    const int K16 = p.K16;
    unsigned char* const sA = tm_smem;
    unsigned char* const sB = tm_smem + (size_t)K16 * TM_A_K16_BYTES;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(sB + (size_t)TH_STAGES * TH_B_STAGE_BYTES);
    uint64_t* const a_full = bars;
    uint64_t* const b_full = bars + 1;
    uint64_t* const b_empty = bars + 1 + TH_STAGES;
    uint64_t* const t_full = bars + 1 + 2 * TH_STAGES;   // [2]: one per accumulator set
    uint64_t* const t_empty = bars + 3 + 2 * TH_STAGES;  // [2]
    uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(bars + 5 + 2 * TH_STAGES);
    double* const lp_x = reinterpret_cast<double*>(sB);           // reused after the main loop: [128][2]
    float* const nrm_x = reinterpret_cast<float*>(lp_x + 2 * TM_M);  // [128][5]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int S = p.S, js = (int)(blockIdx.x % S);
    const long long mt = blockIdx.x / S;
    const int nt0 = (int)((long long)p.nNT * js / S), nt1 = (int)((long long)p.nNT * (js + 1) / S);  // this CTA's unit tiles
    const int nKC = K16 / (TM_KC / 16);

    if (tid == 0) {
        mbar_init(a_full, 1);
        for (int s = 0; s < TH_STAGES; ++s) {
            mbar_init(&b_full[s], 1);
            mbar_init(&b_empty[s], 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&t_full[s], 1);
            mbar_init(&t_empty[s], 8);
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, 2 * TH_N);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            const uint32_t a_bytes = (uint32_t)K16 * TM_A_K16_BYTES;
            mbar_expect_tx(a_full, a_bytes);
            bulk_g2s(sA, p.A_packed + mt * (long long)K16 * TM_M, a_bytes, a_full);
            int it = 0;
            for (int nt = nt0; nt < nt1; ++nt)
                for (int kc = 0; kc < nKC; ++kc, ++it) {
                    const int s = it % TH_STAGES;
                    mbar_wait(&b_empty[s], ((it / TH_STAGES) & 1) ^ 1);
                    mbar_expect_tx(&b_full[s], TH_B_STAGE_BYTES);
                    bulk_g2s(sB + (size_t)s * TH_B_STAGE_BYTES,
                             p.B_packed + ((long long)nt * K16 + kc * (TM_KC / 16)) * TH_N, TH_B_STAGE_BYTES,
                             &b_full[s]);
                }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            mbar_wait(a_full, 0);
            const uint32_t sA_u = smem_u32(sA), sB_u = smem_u32(sB);
            int it = 0;
            for (int nt = nt0; nt < nt1; ++nt) {
                const int ln = nt - nt0, set = ln & 1;
                mbar_wait(&t_empty[set], ((ln >> 1) & 1) ^ 1);
                tc_fence_after();
                for (int kc = 0; kc < nKC; ++kc, ++it) {
                    const int s = it % TH_STAGES;
                    mbar_wait(&b_full[s], (it / TH_STAGES) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int ks = 0; ks < TM_KC / 32; ++ks) {
                        const uint64_t ad = umma_desc(sA_u + (uint32_t)(kc * (TM_KC / 16) + ks * 2) * TM_A_K16_BYTES,
                                                      TM_A_K16_BYTES, 128);
                        const uint64_t bd = umma_desc(sB_u + (uint32_t)s * TH_B_STAGE_BYTES + (uint32_t)(ks * 2) * TH_B_K16_BYTES,
                                                      TH_B_K16_BYTES, 128);
                        umma_i8(tmem_base + (uint32_t)set * TH_N, ad, bd, TH_IDESC, (kc | ks) ? 1u : 0u);
                    }
                    tc_commit(&b_empty[s]);  // frees the stage once these MMAs have read it
                }
                tc_commit(&t_full[set]);
            }
        }
    } else {
        // ---------------- epilogue: 8 warps; TMEM lanes 32*(warp%4).., column half (warp-2)/4 = 8 hidden units
        const int ew = warp - 2;
        const int lane_grp = warp & 3, half = ew >> 2;
        const int row = lane_grp * 32 + lane;
        const long long b = mt * TM_M + row;
        const long long pair = b >> 1;
        const bool odd = lane & 1;
        const int nJC = p.M_pad / 16;
        double lpr = 0.0, lpi = 0.0;
        float2 n2 = make_float2(0.f, 0.f), n4 = n2, n6 = n2, n8 = n2;  // the two halves of a unit pair accumulate apart
        float tmx = 0.f;
        for (int nt = nt0; nt < nt1; ++nt) {
            // scale and bias of this warp's 8 hidden units: lane u (mod 8) holds unit u, fetched before the
            // accumulator wait and handed round by shuffles
            const int ln = nt - nt0, set = ln & 1;
            const int jmine = nt * TH_JT + half * 8 + (lane & 7);
            const float my_sc = p.scale[jmine];
            const float2 my_b = jmine < p.M ? p.bvec[jmine] : make_float2(0.f, 0.f);
            mbar_wait(&t_full[set], (ln >> 1) & 1);
            tc_fence_after();
            {   // 8 hidden units per warp and tile = one 16-byte slab of every series plane
                int v0[32], v1[32];
                const uint32_t col = (uint32_t)(set * TH_N + half * 64);
                tmem_ld32_nowait(tmem_base + ((uint32_t)(lane_grp * 32) << 16) + col, v0);
                tmem_ld32_nowait(tmem_base + ((uint32_t)(lane_grp * 32) << 16) + col + 32, v1);
                tmem_ld_wait();
                tc_fence_before();  // the accumulators are in registers: hand the set back to the MMA issuer
                __syncwarp();
                if (lane == 0) mbar_arrive(&t_empty[set]);
                const int jbase = nt * TH_JT + half * 8;
                float2 tr[4], ti[4];
                float lsr = 0.f, lsi = 0.f;
#pragma unroll
                for (int pq = 0; pq < 4; ++pq) {  // unit pair (jbase + 2 pq, + 1)
                    float2 thr, thi;
                    bool live[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int u = 2 * pq + h;
                        const int j = jbase + u;
                        live[h] = j < p.M;
                        const int src = u;
                        const float sc = __shfl_sync(0xffffffffu, my_sc, src);
                        const float2 bj = make_float2(__shfl_sync(0xffffffffu, my_b.x, src), __shfl_sync(0xffffffffu, my_b.y, src));
                        const int* w = (u < 4) ? &v0[u * 8] : &v1[(u - 4) * 8];
                        const float hr = (float)(w[3] * 128 + w[2]), lr_ = (float)(w[1] * 128 + w[0]);
                        const float hi_ = (float)(w[7] * 128 + w[6]), li_ = (float)(w[5] * 128 + w[4]);
                        const float re = fmaf(hr * 16384.f, sc, fmaf(lr_, sc, bj.x));
                        const float im = fmaf(hi_ * 16384.f, sc, fmaf(li_, sc, bj.y));
                        if (h == 0) thr.x = re, thi.x = im;
                        else thr.y = re, thi.y = im;
                    }
                    if (p.raw_theta) {
                        tr[pq] = make_float2(live[0] ? thr.x : 0.f, live[1] ? thr.y : 0.f);
                        ti[pq] = make_float2(live[0] ? thi.x : 0.f, live[1] ? thi.y : 0.f);
                        continue;
                    }
                    float2 lr, li;
                    lncosh_tanh2(thr, thi, lr, li, tr[pq], ti[pq]);
                    if (live[0]) lsr += lr.x, lsi += li.x;
                    else tr[pq].x = 0.f, ti[pq].x = 0.f;
                    if (live[1]) lsr += lr.y, lsi += li.y;
                    else tr[pq].y = 0.f, ti[pq].y = 0.f;
                }
                lpr += (double)lsr;  // eight small float32 terms first, then float64 across the M / 8 groups
                lpi += (double)lsi;
                if (p.tp) {
#pragma unroll
                    for (int pq = 0; pq < 4; ++pq) {
                        // even lane writes unit 2 pq (needs the odd lane's values), odd lane writes 2 pq + 1
                        const float sr = odd ? tr[pq].x : tr[pq].y, si = odd ? ti[pq].x : ti[pq].y;
                        const float rr = __shfl_xor_sync(0xffffffffu, sr, 1), ri = __shfl_xor_sync(0xffffffffu, si, 1);
                        const int j = jbase + 2 * pq + (odd ? 1 : 0);
                        const float4 rec = odd ? make_float4(rr, tr[pq].y, ri, ti[pq].y)
                                               : make_float4(tr[pq].x, rr, ti[pq].x, ri);
                        if (j < p.M_pad) p.tp[(long long)j * p.nPairsPad + pair] = rec;
                    }
                }
                if (p.sA && jbase < p.M_pad) {
                    unsigned wd[8][4];
#pragma unroll
                    for (int pq = 0; pq < 4; ++pq) {
                        const float2 r = tr[pq], i = ti[pq];
                        const float2 m2 = __ffma2_rn(r, r, __fmul2_rn(i, i));
                        const float2 m4 = __fmul2_rn(m2, m2);
                        n2 = __fadd2_rn(n2, m2);
                        n4 = __fadd2_rn(n4, m4);
                        n6 = __ffma2_rn(m4, m2, n6);
                        n8 = __ffma2_rn(m4, m4, n8);
                        tmx = fmaxf(tmx, fmaxf(m2.x, m2.y));
                        const float2 sr = __fmul2_rn(r, bc2(TM_SERIES_SA)), si = __fmul2_rn(i, bc2(TM_SERIES_SA));
                        wd[0][pq] = tm_pack_h2(sr);
                        wd[1][pq] = tm_pack_h2(si);
                        wd[2][pq] = tm_pack_h2(__fadd2_rn(sr, neg2(tm_unpack_h2(wd[0][pq]))));
                        wd[3][pq] = tm_pack_h2(__fadd2_rn(si, neg2(tm_unpack_h2(wd[1][pq]))));
                        const float2 qr = __ffma2_rn(r, r, neg2(__fmul2_rn(i, i))), qi = __fmul2_rn(__fadd2_rn(r, r), i);
                        wd[4][pq] = tm_pack_h2(__fmul2_rn(qr, bc2(TM_SERIES_SA)));
                        wd[5][pq] = tm_pack_h2(__fmul2_rn(qi, bc2(TM_SERIES_SA)));
                        const float2 cr = __ffma2_rn(sr, qr, neg2(__fmul2_rn(si, qi))), ci = __ffma2_rn(sr, qi, __fmul2_rn(si, qr));
                        wd[6][pq] = tm_pack_h2(cr);
                        wd[7][pq] = tm_pack_h2(ci);
                    }
                    // planes 0 .. 3 (hi, lo) and 6, 7 (cube) from `dm`, planes 4, 5 (square) from `dq` (series_plane_index)
                    const bool wide = p.sA_wide != 0;
                    uint4* const dst = p.sA + ((jbase >> 3) & 1) * TM_M + row;
                    uint4* const dm = dst + series_plane_index(wide, mt, jbase >> 4, 0, p.sA_tiles, nJC) * (2 * TM_M);
                    uint4* const dq = dst + series_plane_index(wide, mt, jbase >> 4, 4, p.sA_tiles, nJC) * (2 * TM_M);
                    uint4* const dc = dm + (wide ? 4 : 6) * (2 * TM_M);
#pragma unroll
                    for (int pl = 0; pl < 4; ++pl) dm[pl * 2 * TM_M] = make_uint4(wd[pl][0], wd[pl][1], wd[pl][2], wd[pl][3]);
#pragma unroll
                    for (int pl = 0; pl < 2; ++pl) {
                        dq[pl * 2 * TM_M] = make_uint4(wd[4 + pl][0], wd[4 + pl][1], wd[4 + pl][2], wd[4 + pl][3]);
                        dc[pl * 2 * TM_M] = make_uint4(wd[6 + pl][0], wd[6 + pl][1], wd[6 + pl][2], wd[6 + pl][3]);
                    }
                }
            }
        }
        // visible bias, split between the two column halves of a row
        if (b < p.B && p.logpsi && js == 0) {
            float ar = 0.f, ai = 0.f;
            const int i_lo = half ? p.N / 2 : 0, i_hi = half ? p.N : p.N / 2;
            for (int i = i_lo; i < i_hi; ++i) {
                const float s = (float)p.spins[b * p.N + i];
                const float2 av = p.a[i];
                ar = fmaf(av.x, s, ar);
                ai = fmaf(av.y, s, ai);
            }
            lpr += (double)ar;
            lpi += (double)ai;
        }
        // all MMAs have completed (t_full of the last tile was observed): the B stages are dead
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (half == 1) {
            lp_x[2 * row] = lpr;
            lp_x[2 * row + 1] = lpi;
            nrm_x[5 * row + 0] = n2.x + n2.y;
            nrm_x[5 * row + 1] = n4.x + n4.y;
            nrm_x[5 * row + 2] = n6.x + n6.y;
            nrm_x[5 * row + 3] = n8.x + n8.y;
            nrm_x[5 * row + 4] = tmx;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (half == 0 && S > 1) {  // partial sums of this CTA's share of the hidden units
            const long long o = (long long)js * p.rows + b;
            if (p.logpsi) p.lp_part[o] = make_double2(lpr + lp_x[2 * row], lpi + lp_x[2 * row + 1]);
            if (p.sA) {
                p.rown[o] = make_float4(n2.x + n2.y + nrm_x[5 * row + 0], n4.x + n4.y + nrm_x[5 * row + 1],
                                        n6.x + n6.y + nrm_x[5 * row + 2], n8.x + n8.y + nrm_x[5 * row + 3]);
                p.rowmax[o] = fmaxf(tmx, nrm_x[5 * row + 4]);
            }
        } else if (half == 0) {
            if (b < p.B && p.logpsi)
                p.logpsi[b] = make_float2((float)(lpr + lp_x[2 * row]), (float)(lpi + lp_x[2 * row + 1]));
            if (p.sA) {
                p.rown[b] = make_float4(sqrtf(n2.x + n2.y + nrm_x[5 * row + 0]), sqrtf(n4.x + n4.y + nrm_x[5 * row + 1]),
                                        sqrtf(n6.x + n6.y + nrm_x[5 * row + 2]), sqrtf(n8.x + n8.y + nrm_x[5 * row + 3]));
                p.rowmax[b] = sqrtf(fmaxf(tmx, nrm_x[5 * row + 4]));
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 2 * TH_N);
    }
}

}  // namespace nqs
