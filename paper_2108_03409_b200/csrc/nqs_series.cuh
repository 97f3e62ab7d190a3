// a5 on the 5th-generation tensor cores (Algorithm 1 line 7, PAPER.md:181-183,
// the call sequence at :464-469): the connected amplitudes as a guarded series of dense contractions.
//
// Ratio identity R:  psi(s')/psi(s) = rho_c(sigma) prod_j (C_jc - sigma t_bj S_jc)
//                                   = rho_c(sigma) kappa_c prod_j (1 - sigma t_bj T_jc),
// with C = cosh 2V, S = sinh 2V, T = tanh 2V = S/C, kappa_c = prod_j C_jc, t = tanh theta.  Hence
//   log R_bc = log kappa_c - 2 sigma A_c - sigma ODD_bc - EVEN_bc,
//   ODD_bc  = sum_{k odd}  (1/k) sum_j t_bj^k T_jc^k,      EVEN_bc = sum_{k even} (1/k) sum_j t_bj^k T_jc^k
// (log(1 - x) = -sum_k x^k / k, |x| < 1).  Truncated at k = 3, every k is a complex [B, M] x [M, C] GEMM
// of element-wise powers.  The GEMMs run as FP16 tcgen05.mma (kind::f16) with FP32 accumulators in
// TMEM; the k = 1 operands are split error-free into two FP16 parts each (hi + lo, three products
// hi.hi + hi.lo + lo.hi: 22 bits), k = 2 and k = 3 need one FP16 part (they are corrections of relative
// size |x| and |x|^2).  Complex arithmetic = four real MMAs per product, the minus sign of Re by the
// negate-A bit of the instruction descriptor.  5 products x 4 = 20 MMAs (M = 128, N = NB, K = 16) per
// 16 hidden units; all odd-k products accumulate into one pair (re, im) of TMEM column ranges and the
// even-k product into a second one, so an accumulator tile is 4 NB <= 512 TMEM columns (NB <= 128).  Hamiltonians
// with more than 128 table columns take column tiles of NB <= 224 instead, with ONE pair in TMEM at a time and two
// passes over the hidden units (series_gemm_kernel<true>): fewer operand bytes into the SM per MAC, which is what
// bounds the narrow kernel's main loop.
//
// The series is only valid where |t T| is small.  The kernel evaluates, per sample, a bound on the
// error it made (truncation + FP16 operand rounding, from row norms of t and column norms of T by
// Cauchy-Schwarz; DESIGN.md section 12 derives it) weighted with |m_bc R_bc|; series_guard_kernel
// compares it with 0.5e-4 max(1, |E_loc|) and raises a device flag if ANY sample fails, in which case
// the FP32 product-form eloc_kernel (which always follows in the stream and exits at once otherwise)
// recomputes the whole call.  No host synchronisation is involved in the decision.
//
// Kernels:  series_table_kernel  T^k planes (FP16, UMMA smem image), log kappa, column norms
//           series_pack_kernel   t^k planes (FP16, UMMA smem image) from tanh(theta), row norms
//           series_gemm_kernel   the GEMMs + fused epilogue exp / matrix element / reduction over c
//           series_guard_kernel  E_loc = diagonal + partial sums, guard decision
#pragma once
#include <cuda_fp16.h>

#include <type_traits>

#include "nqs_device.cuh"
#include "nqs_theta_mma.cuh"

namespace nqs {

constexpr int SR_M = 128;                 // samples per CTA (UMMA M)
constexpr int SR_PLANES = 8;              // hi.re hi.im lo.re lo.im sq.re sq.im cu.re cu.im
constexpr int SR_A_PLANE_U4 = 2 * SR_M;   // uint4 per A plane: [slab 2][row 128][16 bytes]
constexpr int SR_A_STAGE_BYTES = SR_PLANES * SR_A_PLANE_U4 * 16;  // 32 KB
constexpr int SR_STAGES = 3;
constexpr int SR_EPI_PARTS = 4;           // epilogue warps per TMEM lane group: each takes a quarter of the tile's columns
constexpr int SR_EPI_WARPS = 4 * SR_EPI_PARTS;
constexpr int SR_EPI_THREADS = 32 * SR_EPI_WARPS;
constexpr int SR_EPI_COLS = 8;            // columns per TMEM load batch
constexpr int SR_THREADS = 64 + 32 * SR_EPI_WARPS;  // producer, MMA issuer, epilogue warps
constexpr int SR_MAX_N = 2048;            // sites (bit-packed spins of the tile live in shared memory)
// power-of-two operand scales (keep the FP16 parts normal; removed exactly in the epilogue)
constexpr float SR_SA = 16.f;             // every t plane
constexpr float SR_SB1 = 64.f;            // T and T^3/3 planes  -> ODD  is scaled by 2^10
constexpr float SR_SB2 = 2048.f;          // T^2/2 plane         -> EVEN is scaled by 2^15
static_assert(SR_SA == TM_SERIES_SA, "theta_mma_kernel writes the t planes with this scale");
constexpr float SR_INV_ODD = 1.f / (SR_SA * SR_SB1);
constexpr float SR_INV_EVEN = 1.f / (SR_SA * SR_SB2);
constexpr float SR_GUARD_FRACTION = 0.5f; // of the tolerance 1e-4 max(1, |E_loc|)

// per table column, written by series_table_kernel (64 bytes)
struct __align__(16) SeriesCol {
    float lkr, lki;      // log kappa_c = sum_j log cosh 2 V_jc
    float a2r, a2i;      // 2 A_c,  A = a_i + p a_k
    float k0, k1, k2, k3;  // guard: delta_bc = k0 + n2t k1 + n4t k2 + n6t k3 + n8t k4
    float k4, tmax;      // tmax = max_j |T_jc|
    int site, sitek;     // first / second flip site (sitek = -1: single flip)
    int par, group;      // bit q: relative sign of flip site q + 1 is -1; flip group (-1: padding column)
    int sx, count;       // third | fourth << 16 flip site (0xffff: none); number of terms of the group, with
                         // SR_GENERIC_TERMS set when they are not (all) inline in SeriesTerms
};
constexpr int SR_GENERIC_TERMS = 1 << 30;
// the column's matrix element is m0 + sigma m1 with constants m0, m1 whenever the column applies: at most two inline terms
// whose Z factors sit on the column's own (one or two) flip sites -- the X_i of a transverse field, the XX + YY of a
// Heisenberg bond (s_k = +/- s_i is fixed by the column's relative sign) -- or a padding column (0).  SeriesTerms then
// holds m0 as a constant term and m1 as a term on s[site]; a tile of such columns takes a shorter epilogue.
constexpr int SR_AFFINE = 1 << 29;
constexpr int SR_COUNT_MASK = SR_AFFINE - 1;
static_assert(sizeof(SeriesCol) == 64, "SeriesCol layout");
// the first two terms of the column's group, element = c * s[z0] * s[z1] (z = -1: factor 1); an absent term has c = 0
struct __align__(16) SeriesTerms {
    int z0a, z1a;
    float cra, cia;
    int z0b, z1b;
    float crb, cib;
};
static_assert(sizeof(SeriesTerms) == 32, "SeriesTerms layout");

__host__ __device__ inline int series_bits_stride(int N) { return (N + 31) / 32 | 1; }  // odd: conflict-free rows
// wide = false: a stage holds all eight planes of both operands (32 KB + 256 NB bytes), NB <= 128.
// wide = true : column tiles of NB <= 224 with the (re, im) accumulators of ONE of the two series sums in TMEM at a time: a
//               stage holds six planes (hi, lo, cube: 24 KB + 192 NB bytes); the partial sums of the column parts reuse
//               the first stage at the end.
constexpr int SR_WIDE_PLANES = 6;
constexpr int SR_WIDE_MAX_NB = 224;
__host__ __device__ inline size_t series_gemm_smem_bytes(int NB, int N, bool wide = false) {
    const size_t fixed = (size_t)NB * (sizeof(SeriesCol) + sizeof(SeriesTerms)) + (size_t)SR_M * series_bits_stride(N) * 4 + 256;
    if (wide) return (size_t)SR_STAGES * (SR_WIDE_PLANES * SR_A_PLANE_U4 * 16 + 192 * NB) + fixed;
    return (size_t)SR_STAGES * (SR_A_STAGE_BYTES + 256 * NB) + fixed + (size_t)(SR_EPI_PARTS - 1) * SR_M * 16;
}

__device__ __forceinline__ unsigned pack_h2(float a, float b) {
    const __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<const unsigned*>(&h);
}

// ---------------------------------------------------------------------------------------
// B operand + per-column data.  One block per (padded) column c, thread <-> 8 consecutive hidden units.
// B_packed[ntile][jchunk16][plane][slab 2][row NB][8 halves]  (one contiguous 256 NB-byte block per stage)
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) series_table_kernel(const float2* __restrict__ W, const float2* __restrict__ a,
                                                           int N, int M, int M_pad, int C, int NB, DevHam H,
                                                           uint4* __restrict__ B_packed, int wide,
                                                           SeriesCol* __restrict__ cols,
                                                           SeriesTerms* __restrict__ terms) {
    const int c = blockIdx.x, tid = threadIdx.x;
    const int nt = c / NB, cl = c % NB;
    const int nJC = M_pad / 16;
    const bool live_col = c < C;
    double lkr = 0.0, lki = 0.0;
    float n2 = 0.f, n4 = 0.f, n6 = 0.f, n8 = 0.f, tmx = 0.f;
    for (int j8 = tid; j8 < M_pad / 8; j8 += 256) {
        float v[SR_PLANES][8];
#pragma unroll
        for (int q2 = 0; q2 < 8; q2 += 2) {
            // log cosh 2V and T = tanh 2V of two hidden units at a time (packed Taylor series for |2V|^2 < 0.36, the
            // closed form otherwise: nqs_device.cuh)
            const int j0 = j8 * 8 + q2;
            const bool l0 = live_col && j0 < M, l1 = live_col && j0 + 1 < M;
            const float2 w0 = l0 ? column_sum(H, c, W + (long long)j0 * N) : make_float2(0.f, 0.f);
            const float2 w1 = l1 ? column_sum(H, c, W + (long long)(j0 + 1) * N) : make_float2(0.f, 0.f);
            float2 lr2, li2, Tr2, Ti2;
            lncosh_tanh2(make_float2(2.f * w0.x, 2.f * w1.x), make_float2(2.f * w0.y, 2.f * w1.y), lr2, li2, Tr2, Ti2);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int q = q2 + h;
                const bool lv = h ? l1 : l0;
                const float Tr = lv ? (h ? Tr2.y : Tr2.x) : 0.f, Ti = lv ? (h ? Ti2.y : Ti2.x) : 0.f;
                if (lv) {
                    lkr += (double)(h ? lr2.y : lr2.x);
                    lki += (double)(h ? li2.y : li2.x);
                    const float m2 = fmaf(Tr, Tr, Ti * Ti);
                    n2 += m2;
                    n4 = fmaf(m2, m2, n4);
                    n6 = fmaf(m2 * m2, m2, n6);
                    n8 = fmaf(m2 * m2, m2 * m2, n8);
                    tmx = fmaxf(tmx, m2);
                }
                const float sr = Tr * SR_SB1, si = Ti * SR_SB1;
                v[0][q] = __half2float(__float2half_rn(sr));
                v[1][q] = __half2float(__float2half_rn(si));
                v[2][q] = sr - v[0][q];
                v[3][q] = si - v[1][q];
                const float T2r = fmaf(Tr, Tr, -Ti * Ti), T2i = 2.f * Tr * Ti;
                v[4][q] = 0.5f * SR_SB2 * T2r;
                v[5][q] = 0.5f * SR_SB2 * T2i;
                v[6][q] = (SR_SB1 / 3.f) * fmaf(Tr, T2r, -Ti * T2i);
                v[7][q] = (SR_SB1 / 3.f) * fmaf(Tr, T2i, Ti * T2r);
            }
        }
        const int jc = j8 >> 1, slab = j8 & 1;
        uint4* const dst = B_packed + slab * NB + cl;
        const int nNT = gridDim.x / NB;
#pragma unroll
        for (int pl = 0; pl < SR_PLANES; ++pl)
            dst[series_plane_index(wide != 0, nt, jc, pl, nNT, nJC) * (2 * NB)] = make_uint4(pack_h2(v[pl][0], v[pl][1]), pack_h2(v[pl][2], v[pl][3]),
                                                     pack_h2(v[pl][4], v[pl][5]), pack_h2(v[pl][6], v[pl][7]));
    }
    // block reduction in a fixed order (deterministic)
    __shared__ double sd[2][256];
    __shared__ float sf[5][256];
    sd[0][tid] = lkr, sd[1][tid] = lki;
    sf[0][tid] = n2, sf[1][tid] = n4, sf[2][tid] = n6, sf[3][tid] = n8, sf[4][tid] = tmx;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) {
            sd[0][tid] += sd[0][tid + o];
            sd[1][tid] += sd[1][tid + o];
#pragma unroll
            for (int q = 0; q < 4; ++q) sf[q][tid] += sf[q][tid + o];
            sf[4][tid] = fmaxf(sf[4][tid], sf[4][tid + o]);
        }
        __syncthreads();
    }
    if (tid == 0) {
        SeriesCol r;
        r.lkr = (float)sd[0][0];
        r.lki = (float)sd[1][0];
        const float2 A = live_col ? column_sum(H, c, a) : make_float2(0.f, 0.f);
        r.a2r = 2.f * A.x;
        r.a2i = 2.f * A.y;
        // guard coefficients; u16 = 2^-21 (hi + lo split), u = 2^-10 (one FP16 part,
        // both operands), eta = absolute rounding floor of the scaled FP16 subnormals; factor 2 = re / im slack
        const float n2T = sqrtf(sf[0][0]), n4T = sqrtf(sf[1][0]), n6T = sqrtf(sf[2][0]), n8T = sqrtf(sf[3][0]);
        const float sqM = sqrtf((float)M);
        r.k0 = 2.f * sqM * 1.8626451e-9f * n2T;                              // 2^-29 sum_j |T_j|
        r.k1 = 2.f * (4.7683716e-7f * n2T + sqM * 4.6566129e-10f);           // 2^-21 n2T + 2^-31 sqrt(M)
        r.k2 = 9.765625e-4f * n4T;                                           // 2 . 2^-10 . 1/2
        r.k3 = (2.f / 3.f) * 9.765625e-4f * n6T;                             // 2 . 2^-10 . 1/3
        r.k4 = 0.5f * n8T;                                                   // truncation: 1/(4 (1 - X)), X <= 1/2
        r.tmax = sqrtf(sf[4][0]);
        r.site = live_col ? H.col_i[c] : 0;
        r.sitek = live_col ? H.col_k[c] : -1;
        r.par = 0;
        r.sx = 0xffffffff;
        if (live_col) {
            const int s2 = H.col_s2[c], s3 = H.col_s3[c];
            r.par = (H.col_p[c] < 0 ? 1 : 0) | (H.col_p2[c] < 0 ? 2 : 0) | (H.col_p3[c] < 0 ? 4 : 0);
            r.sx = (s2 >= 0 ? s2 : 0xffff) | ((s3 >= 0 ? s3 : 0xffff) << 16);
        }
        r.group = live_col ? H.col_group[c] : -1;
        const int first = r.group >= 0 ? H.grp_first[r.group] : 0;
        int count = r.group >= 0 ? H.grp_count[r.group] : 0;
        // inline fast path: at most two terms, none with more than two z factors
        bool generic = count > 2;
        if (H.has_zx)
            for (int u = 0; u < count; ++u) generic |= H.gt_zx_off[first + u + 1] > H.gt_zx_off[first + u];
        SeriesTerms t2 = {-1, -1, 0.f, 0.f, -1, -1, 0.f, 0.f};
        if (!generic && count >= 1) {
            const float2 cc = H.gt_c[first];
            t2.z0a = H.gt_z0[first], t2.z1a = H.gt_z1[first], t2.cra = cc.x, t2.cia = cc.y;
        }
        if (!generic && count >= 2) {
            const float2 cc = H.gt_c[first + 1];
            t2.z0b = H.gt_z0[first + 1], t2.z1b = H.gt_z1[first + 1], t2.crb = cc.x, t2.cib = cc.y;
        }
        bool affine = !generic && r.sx == (int)0xffffffff;
        if (affine) {
            const float psign = (r.par & 1) ? -1.f : 1.f;
            float m0r = 0.f, m0i = 0.f, m1r = 0.f, m1i = 0.f;
            const int zs[2][2] = {{t2.z0a, t2.z1a}, {t2.z0b, t2.z1b}};
            const float cs[2][2] = {{t2.cra, t2.cia}, {t2.crb, t2.cib}};
            for (int u = 0; u < 2; ++u) {
                int ni = 0, nk = 0;
                for (int q = 0; q < 2; ++q) {
                    const int z = zs[u][q];
                    if (z < 0) continue;
                    if (z == r.site) ++ni;
                    else if (r.sitek >= 0 && z == r.sitek) ++nk;
                    else affine = false;
                }
                const float f = (nk & 1) ? psign : 1.f;  // s_k = psign s_i where the column applies
                if ((ni + nk) & 1) m1r = fmaf(cs[u][0], f, m1r), m1i = fmaf(cs[u][1], f, m1i);
                else m0r = fmaf(cs[u][0], f, m0r), m0i = fmaf(cs[u][1], f, m0i);
            }
            if (affine) t2 = {-1, -1, m0r, m0i, r.site, -1, m1r, m1i};
        }
        r.count = count | (generic ? SR_GENERIC_TERMS : 0) | (affine ? SR_AFFINE : 0);
        cols[c] = r;
        terms[c] = t2;
    }
}

// ---------------------------------------------------------------------------------------
// A operand + row norms.  One block per 128-sample tile; thread <-> (pair of samples, 8 hidden units).
// A_packed[mtile][jchunk16][plane][slab 2][row 128][8 halves]  (32 KB contiguous per stage)
// rown[b] = (n2t, n4t, n6t, n8t), nPt = sqrt(sum_j |t_bj|^P);  rowmax[b] = max_j |t_bj|
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) series_pack_kernel(const float4* __restrict__ tp, long long nPairsPad, int M_pad,
                                                          uint4* __restrict__ A_packed, int wide, float4* __restrict__ rown,
                                                          float* __restrict__ rowmax) {
    const int tid = threadIdx.x, pl = tid & 63, jsub = tid >> 6;
    const long long mt = blockIdx.x;
    const long long pair = mt * 64 + pl;
    const int nJC = M_pad / 16;
    float acc[2][5] = {{0.f, 0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f, 0.f}};
    for (int j8 = jsub; j8 < M_pad / 8; j8 += 4) {
        float4 t[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) t[q] = tp[(long long)(j8 * 8 + q) * nPairsPad + pair];
        uint4* const dst = A_packed + (j8 & 1) * SR_M + 2 * pl;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float v[SR_PLANES][8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float tr = h ? t[q].y : t[q].x, ti = h ? t[q].w : t[q].z;
                const float m2 = fmaf(tr, tr, ti * ti);
                acc[h][0] += m2;
                acc[h][1] = fmaf(m2, m2, acc[h][1]);
                acc[h][2] = fmaf(m2 * m2, m2, acc[h][2]);
                acc[h][3] = fmaf(m2 * m2, m2 * m2, acc[h][3]);
                acc[h][4] = fmaxf(acc[h][4], m2);
                const float sr = tr * SR_SA, si = ti * SR_SA;
                v[0][q] = __half2float(__float2half_rn(sr));
                v[1][q] = __half2float(__float2half_rn(si));
                v[2][q] = sr - v[0][q];
                v[3][q] = si - v[1][q];
                const float t2r = fmaf(tr, tr, -ti * ti), t2i = 2.f * tr * ti;
                v[4][q] = SR_SA * t2r;
                v[5][q] = SR_SA * t2i;
                v[6][q] = SR_SA * fmaf(tr, t2r, -ti * t2i);
                v[7][q] = SR_SA * fmaf(tr, t2i, ti * t2r);
            }
#pragma unroll
            for (int p = 0; p < SR_PLANES; ++p)
                dst[series_plane_index(wide != 0, mt, j8 >> 1, p, gridDim.x, nJC) * SR_A_PLANE_U4 + h] = make_uint4(pack_h2(v[p][0], v[p][1]), pack_h2(v[p][2], v[p][3]),
                                                        pack_h2(v[p][4], v[p][5]), pack_h2(v[p][6], v[p][7]));
        }
    }
    __shared__ float sh[4][128][5];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int q = 0; q < 5; ++q) sh[jsub][2 * pl + h][q] = acc[h][q];
    __syncthreads();
    if (tid < 128) {
        float s[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) s[q] = sh[0][tid][q];
        for (int k = 1; k < 4; ++k) {
#pragma unroll
            for (int q = 0; q < 4; ++q) s[q] += sh[k][tid][q];
            s[4] = fmaxf(s[4], sh[k][tid][4]);
        }
        const long long b = mt * SR_M + tid;
        rown[b] = make_float4(sqrtf(s[0]), sqrtf(s[1]), sqrtf(s[2]), sqrtf(s[3]));
        rowmax[b] = sqrtf(s[4]);
    }
}

// ---------------------------------------------------------------------------------------
// tcgen05 kind::f16 wrappers (descriptors: umma_desc of nqs_theta_mma.cuh; the byte layout of a K = 16
// FP16 step equals that of a K = 32 INT8 step: two 16-byte slabs)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}
// no register of v may be touched before tcgen05.wait::ld (the load is asynchronous)
__device__ __forceinline__ void tmem_ld8_nowait(uint32_t taddr, float (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(r[k]);
}
// D = F32, A = B = F16, K-major both, N >> 3 at bit 17, M >> 4 at bit 24; bit 13 negates A
__host__ __device__ inline uint32_t series_idesc(int NB) {
    return (1u << 4) | ((uint32_t)(NB >> 3) << 17) | ((uint32_t)(SR_M >> 4) << 24);
}
constexpr uint32_t SR_IDESC_NEG_A = 1u << 13;

// spin of site i from a bit-packed row (bit = 1 <=> spin +1)
__device__ __forceinline__ float spin_from_bits(const uint32_t* __restrict__ bits, int i) {
    return ((bits[i >> 5] >> (i & 31)) & 1u) ? 1.f : -1.f;
}

struct SeriesGemmParams {
    const uint4* A_packed;   // [nMT][nJC][8][256];  WIDE: the wide layout of series_plane_index (planes of 256 uint4)
    const uint4* B_packed;   // [nNT][nJC][8][2 NB]; WIDE: the same with planes of 2 NB uint4
    long long nMT;           // sample tiles in A_packed
    const SeriesCol* cols;   // [nNT * NB]
    const SeriesTerms* terms;  // [nNT * NB]
    const float4* rown;      // [B_pad] (n2t, n4t, n6t, n8t);  nS > 1: [nS][B_pad] partial sums of |t|^P (theta kernel split
    const float* rowmax;     // [B_pad] max |t|;                over nS CTAs per sample tile): combined here
    int nS;                  // number of partials (1: final values)
    long long rows;          // B_pad: stride of the partials
    const int8_t* spins;     // [B][N]
    long long B;
    int N, nJC, NB, nNT;
    DevHam H;
    float4* partial;         // [B][nNT]: (Re, Im of sum_c m R [+ diagonal in tile 0], guard eps, 0)
    float2* even;            // WIDE: [nMT][nNT][NB][128 rows] scratch for the EVEN sums (written and read back by the same thread)
#ifdef NQS_SERIES_TIMELINE
    long long* timeline;     // [blocks][8] clock64 stamps of the first epilogue thread (development builds only)
#endif
};
#ifdef NQS_SERIES_TIMELINE
#define NQS_STAMP(k) stamp[k] = clock64()
#else
#define NQS_STAMP(k)
#endif

// WIDE = false: all four accumulator ranges (ODD.re, ODD.im, EVEN.re, EVEN.im) of a tile of NB <= 128 columns in TMEM,
//               20 MMAs per chunk of 16 hidden units, 32 KB + 256 NB bytes of operands per chunk.
// WIDE = true : tiles of NB <= 224 columns.  What bounds the main loop is the operand bytes an SM takes in per MMA
//               cycle (~45 B/clk), i.e. (128 + NB) / (128 NB): a tile twice as wide needs 1.6 x
//               fewer bytes per MAC, but its four accumulator ranges no longer fit in the 512 TMEM columns.  So the
//               kernel makes two passes over the hidden units: pass A accumulates EVEN (4 MMAs per chunk on the t^2 /
//               T^2 planes) and the epilogue threads move it to a global scratch array (each thread writes and later
//               reads back only its own (row, columns): L2-resident, no fence); pass B accumulates ODD (16 MMAs per chunk)
//               into the same TMEM columns and the epilogue proceeds as before.  Every accumulator element sees the
//               same addends in the same order as in the narrow kernel: bit-identical E_loc.
template <bool WIDE>
__global__ void __launch_bounds__(SR_THREADS, 1) series_gemm_kernel(const SeriesGemmParams p) {
    extern __shared__ __align__(128) unsigned char sr_smem[];
    const int NB = p.NB;
    constexpr uint32_t A_STAGE = WIDE ? SR_WIDE_PLANES * SR_A_PLANE_U4 * 16 : SR_A_STAGE_BYTES;
    const uint32_t b_plane = 32u * NB, b_lbo = 16u * NB;
    const uint32_t b_stage_bytes = (WIDE ? SR_WIDE_PLANES : SR_PLANES) * b_plane, stage_bytes = A_STAGE + b_stage_bytes;
    SeriesCol* const scol = reinterpret_cast<SeriesCol*>(sr_smem + (size_t)SR_STAGES * stage_bytes);
    SeriesTerms* const sterm = reinterpret_cast<SeriesTerms*>(scol + NB);
    // [parts - 1][128] partial sums of the other column parts; WIDE: over the first stage (dead after the last MMA)
    float4* const sred = WIDE ? reinterpret_cast<float4*>(sr_smem) : reinterpret_cast<float4*>(sterm + NB);
    uint32_t* const sbits = WIDE ? reinterpret_cast<uint32_t*>(sterm + NB)
                                 : reinterpret_cast<uint32_t*>(reinterpret_cast<float4*>(sterm + NB) + (SR_EPI_PARTS - 1) * SR_M);
    const int bstride = series_bits_stride(p.N);
    uint64_t* const bars = reinterpret_cast<uint64_t*>(sbits + (size_t)SR_M * bstride + (((size_t)SR_M * bstride) & 1));
    uint64_t* const full = bars;
    uint64_t* const empty = bars + SR_STAGES;
    uint64_t* const t_full = bars + 2 * SR_STAGES;
    uint64_t* const t_free = bars + 2 * SR_STAGES + 1;  // WIDE: the EVEN sums have left TMEM
    uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * SR_STAGES + 2);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
#ifdef NQS_SERIES_TIMELINE
    long long stamp[6] = {0, 0, 0, 0, 0, 0};
#endif
    NQS_STAMP(0);
    const int nt = blockIdx.x % p.nNT;
    const long long mt = blockIdx.x / p.nNT;
    const int nJC = p.nJC;

    if (tid == 0) {
        for (int s = 0; s < SR_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        mbar_init(t_full, 1);
        mbar_init(t_free, SR_EPI_WARPS);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    NQS_STAMP(1);

    if (warp == 0) {
        if (lane == 0) {
            const uint4* gA = p.A_packed + mt * (long long)nJC * SR_PLANES * SR_A_PLANE_U4;
            const uint4* gB = p.B_packed + (long long)nt * nJC * SR_PLANES * (2 * NB);
            const uint32_t a_plane = SR_A_PLANE_U4 * 16;
            if (WIDE) {
                // pass A: the square planes of three chunks per stage (contiguous in the wide layout); pass B: the six
                // planes hi, lo, cube of one chunk per stage.  Two bulk copies per stage either way.
                const unsigned char* const baseA = reinterpret_cast<const unsigned char*>(p.A_packed);
                const unsigned char* const baseB = reinterpret_cast<const unsigned char*>(p.B_packed);
                const int nA = (nJC + 2) / 3;
                for (int it = 0; it < nA + nJC; ++it) {
                    const int s = it % SR_STAGES;
                    mbar_wait(&empty[s], ((it / SR_STAGES) & 1) ^ 1);
                    unsigned char* const stA = sr_smem + (size_t)s * stage_bytes;
                    unsigned char* const stB = stA + A_STAGE;
                    if (it < nA) {
                        const int kc = 3 * it, nc = min(3, nJC - kc);
                        mbar_expect_tx(&full[s], (uint32_t)nc * 2 * (a_plane + b_plane));
                        bulk_g2s(stA, baseA + series_plane_index(true, mt, kc, 4, p.nMT, nJC) * a_plane, (uint32_t)nc * 2 * a_plane, &full[s]);
                        bulk_g2s(stB, baseB + series_plane_index(true, nt, kc, 4, p.nNT, nJC) * b_plane, (uint32_t)nc * 2 * b_plane, &full[s]);
                    } else {
                        const int kc = it - nA;
                        mbar_expect_tx(&full[s], 6 * (a_plane + b_plane));
                        bulk_g2s(stA, baseA + series_plane_index(true, mt, kc, 0, p.nMT, nJC) * a_plane, 6 * a_plane, &full[s]);
                        bulk_g2s(stB, baseB + series_plane_index(true, nt, kc, 0, p.nNT, nJC) * b_plane, 6 * b_plane, &full[s]);
                    }
                }
            } else {
                for (int kc = 0; kc < nJC; ++kc) {
                    const int s = kc % SR_STAGES;
                    mbar_wait(&empty[s], ((kc / SR_STAGES) & 1) ^ 1);
                    unsigned char* const st = sr_smem + (size_t)s * stage_bytes;
                    mbar_expect_tx(&full[s], stage_bytes);
                    bulk_g2s(st, gA + (long long)kc * SR_PLANES * SR_A_PLANE_U4, SR_A_STAGE_BYTES, &full[s]);
                    bulk_g2s(st + SR_A_STAGE_BYTES, gB + (long long)kc * SR_PLANES * (2 * NB), b_stage_bytes, &full[s]);
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t s0 = smem_u32(sr_smem);
            const uint32_t idesc = series_idesc(NB);
            // accumulator column ranges: ODD.re, ODD.im, EVEN.re, EVEN.im (WIDE: EVEN first, then ODD, in the same columns)
            const uint32_t d_or = tmem_base, d_oi = tmem_base + NB;
            const uint32_t d_er = WIDE ? d_or : tmem_base + 2 * NB, d_ei = WIDE ? d_oi : tmem_base + 3 * NB;
            uint32_t sa = 0, sb = 0;
            auto A = [&](int pl) { return umma_desc(sa + (uint32_t)pl * 4096u, 2048u, 128u); };
            auto Bd = [&](int pl) { return umma_desc(sb + (uint32_t)pl * b_plane, b_lbo, 128u); };
            // one complex product (a.re, a.im = planes pa, pa + 1) x (b.re, b.im = planes pb, pb + 1)
            auto cprod = [&](int pa, int pb, uint32_t dre, uint32_t dim, uint32_t first) {
                umma_f16(dre, A(pa), Bd(pb), idesc, first);
                umma_f16(dre, A(pa + 1), Bd(pb + 1), idesc | SR_IDESC_NEG_A, 1u);
                umma_f16(dim, A(pa), Bd(pb + 1), idesc, first);
                umma_f16(dim, A(pa + 1), Bd(pb), idesc, 1u);
            };
            if (WIDE) {
                const int nA = (nJC + 2) / 3;
                for (int it = 0; it < nA + nJC; ++it) {
                    const int s = it % SR_STAGES;
                    if (it == nA) {  // EVEN is complete: hand it to the epilogue warps, wait until it has left TMEM
                        tc_commit(t_full);
                        mbar_wait(t_free, 0);
                    }
                    mbar_wait(&full[s], (it / SR_STAGES) & 1);
                    tc_fence_after();
                    sa = s0 + (uint32_t)s * stage_bytes, sb = sa + A_STAGE;
                    if (it < nA) {
                        const int nc = min(3, nJC - 3 * it);
                        for (int u = 0; u < nc; ++u)
                            cprod(2 * u, 2 * u, d_er, d_ei, (it | u) ? 1u : 0u);   // t^2 T^2 / 2 of chunk 3 it + u
                    } else {
                        const uint32_t first = it > nA ? 1u : 0u;
                        cprod(0, 0, d_or, d_oi, first);   // t.hi T.hi
                        cprod(0, 2, d_or, d_oi, 1u);      // t.hi T.lo
                        cprod(2, 0, d_or, d_oi, 1u);      // t.lo T.hi
                        cprod(4, 4, d_or, d_oi, 1u);      // t^3 T^3 / 3  (stage slots 4, 5)
                    }
                    tc_commit(&empty[s]);
                }
            } else {
                for (int kc = 0; kc < nJC; ++kc) {
                    const int s = kc % SR_STAGES;
                    mbar_wait(&full[s], (kc / SR_STAGES) & 1);
                    tc_fence_after();
                    sa = s0 + (uint32_t)s * stage_bytes, sb = sa + A_STAGE;
                    const uint32_t first = kc ? 1u : 0u;
                    cprod(0, 0, d_or, d_oi, first);   // t.hi T.hi
                    cprod(0, 2, d_or, d_oi, 1u);      // t.hi T.lo
                    cprod(2, 0, d_or, d_oi, 1u);      // t.lo T.hi
                    cprod(6, 6, d_or, d_oi, 1u);      // t^3 T^3 / 3
                    cprod(4, 4, d_er, d_ei, first);   // t^2 T^2 / 2
                    tc_commit(&empty[s]);
                }
            }
            tc_commit(t_full);
        }
    } else {
        // ---------------- epilogue warps: TMEM lane group = warp % 4, column part = (warp - 2) / 4
        const int lane_grp = warp & 3, part = (warp - 2) >> 2;
        const int row = lane_grp * 32 + lane;
        const long long b = mt * SR_M + row;
        // while the MMAs run: column records -> smem (part 1), bit-packed spins of the own row (part 0)
        if (part == 1) {
            const int et = tid - 64 - 128;
            for (int idx = et; idx < NB * 4; idx += 128)
                reinterpret_cast<uint4*>(scol)[idx] = reinterpret_cast<const uint4*>(p.cols + (long long)nt * NB)[idx];
            for (int idx = et; idx < NB * 2; idx += 128)
                reinterpret_cast<uint4*>(sterm)[idx] = reinterpret_cast<const uint4*>(p.terms + (long long)nt * NB)[idx];
        } else if (part == 0) {
            uint32_t* const wbits = sbits + (size_t)row * bstride;
            const int nW = (p.N + 31) / 32;
            if (b >= p.B) {
                for (int w = 0; w < nW; ++w) wbits[w] = 0u;
            } else {
                const int8_t* const srow = p.spins + b * p.N;
                auto nib = [](uint32_t x) {  // 4 spins (bytes +1 / -1) -> 4 bits, bit k = (byte k > 0)
                    const uint32_t y = (~x >> 7) & 0x01010101u;
                    return (y & 1u) | ((y >> 7) & 2u) | ((y >> 14) & 4u) | ((y >> 21) & 8u);
                };
                if ((p.N & 15) == 0 && (reinterpret_cast<uintptr_t>(p.spins) & 15) == 0) {
                    const uint4* const v = reinterpret_cast<const uint4*>(srow);
                    const int nV = p.N / 16;
#pragma unroll 4
                    for (int w = 0; w < nW; ++w) {
                        const uint4 lo = v[2 * w];
                        const uint4 hi = (2 * w + 1 < nV) ? v[2 * w + 1] : make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
                        wbits[w] = nib(lo.x) | (nib(lo.y) << 4) | (nib(lo.z) << 8) | (nib(lo.w) << 12) | (nib(hi.x) << 16) |
                                   (nib(hi.y) << 20) | (nib(hi.z) << 24) | (nib(hi.w) << 28);
                    }
                } else {
                    for (int w = 0; w < nW; ++w) {
                        uint32_t word = 0u;
                        const int i1 = min(32, p.N - 32 * w);
                        for (int i = 0; i < i1; ++i) word |= (srow[32 * w + i] > 0 ? 1u : 0u) << i;
                        wbits[w] = word;
                    }
                }
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(SR_EPI_THREADS) : "memory");  // records and bits visible to the epilogue warps
        const uint32_t* const mybits = sbits + (size_t)row * bstride;
        auto spin_or_one = [&](int z) { return z >= 0 ? spin_from_bits(mybits, z) : 1.f; };
        float er_acc = 0.f, ei_acc = 0.f, eps = 0.f;
        if (nt == 0 && !p.H.has_zx) {
            // diagonal terms (empty flip set): d = sum_t c_t s[z0] s[z1].  The parts split the list into contiguous
            // quarters; a warp fetches 32 terms at a time (one per lane, coalesced) and hands them round by shuffles
            const int per = (p.H.Td + SR_EPI_PARTS - 1) / SR_EPI_PARTS;
            const int t0 = part * per, t1 = min(p.H.Td, t0 + per);
            for (int tb = t0; tb < t1; tb += 32) {
                const int tl = tb + lane;
                const int z0l = tl < t1 ? p.H.diag_z0[tl] : -1, z1l = tl < t1 ? p.H.diag_z1[tl] : -1;
                const float2 cl = tl < t1 ? p.H.diag_c[tl] : make_float2(0.f, 0.f);
                const int n = min(32, t1 - tb);
                for (int u = 0; u < n; ++u) {
                    const int z0 = __shfl_sync(0xffffffffu, z0l, u), z1 = __shfl_sync(0xffffffffu, z1l, u);
                    const float cx = __shfl_sync(0xffffffffu, cl.x, u), cy = __shfl_sync(0xffffffffu, cl.y, u);
                    const float f = spin_or_one(z0) * spin_or_one(z1);
                    er_acc = fmaf(cx, f, er_acc);
                    ei_acc = fmaf(cy, f, ei_acc);
                }
            }
        } else if (nt == 0) {  // terms with more than two Z factors (k-site strings): the general list
            for (int t = part; t < p.H.Td; t += SR_EPI_PARTS) {
                float f = spin_or_one(p.H.diag_z0[t]) * spin_or_one(p.H.diag_z1[t]);
                for (int x = p.H.diag_zx_off[t]; x < p.H.diag_zx_off[t + 1]; ++x) f *= spin_from_bits(mybits, p.H.diag_zx[x]);
                const float2 cc = p.H.diag_c[t];
                er_acc = fmaf(cc.x, f, er_acc);
                ei_acc = fmaf(cc.y, f, ei_acc);
            }
        }
        NQS_STAMP(2);
        float4 rn = p.rown[b];
        float rmax = p.rowmax[b];
        if (p.nS > 1) {  // fixed order: deterministic
            for (int k = 1; k < p.nS; ++k) {
                const float4 o = p.rown[k * p.rows + b];
                rn.x += o.x, rn.y += o.y, rn.z += o.z, rn.w += o.w;
                rmax = fmaxf(rmax, p.rowmax[k * p.rows + b]);
            }
            rn = make_float4(sqrtf(rn.x), sqrtf(rn.y), sqrtf(rn.z), sqrtf(rn.w));
            rmax = sqrtf(rmax);
        }
        const int nBatch = NB / SR_EPI_COLS;
        const int b_lo = nBatch * part / SR_EPI_PARTS, b_hi = nBatch * (part + 1) / SR_EPI_PARTS;
        const uint32_t tbase = tmem_base + ((uint32_t)(lane_grp * 32) << 16);
        // WIDE: this thread's slice of the EVEN scratch, [column][row] so that a warp's stores and loads coalesce
        float2* const even = WIDE ? p.even + ((mt * p.nNT + nt) * (long long)NB) * SR_M + row : nullptr;
        if (WIDE) {
            mbar_wait_sleep(t_full, 0, 256);  // pass A: EVEN is in TMEM
            tc_fence_after();
#pragma unroll 1
            for (int bt = b_lo; bt < b_hi; ++bt) {
                const int c0 = bt * SR_EPI_COLS;
                float ver[SR_EPI_COLS], vei[SR_EPI_COLS];
                tmem_ld8_nowait(tbase + (uint32_t)c0, ver);
                tmem_ld8_nowait(tbase + (uint32_t)(NB + c0), vei);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int q = 0; q < SR_EPI_COLS; ++q) even[(long long)(c0 + q) * SR_M] = make_float2(ver[q], vei[q]);
            }
            tc_fence_before();  // the loads have completed: the columns may be overwritten by pass B
            __syncwarp();
            if (lane == 0) mbar_arrive(t_free);
        }
        mbar_wait_sleep(t_full, WIDE ? 1u : 0u, 256);
        NQS_STAMP(3);
        tc_fence_after();
        // are all columns of the tile affine (warp-uniform: the records are the same for every row)?
        bool tile_affine = true;
        for (int c = lane; c < NB; c += 32) tile_affine = tile_affine && (scol[c].count & SR_AFFINE);
        tile_affine = __all_sync(0xffffffffu, tile_affine);
        auto columns = [&](auto affine_tag) {
        constexpr bool AFFINE = decltype(affine_tag)::value;
#pragma unroll 1
        for (int bt = b_lo; bt < b_hi; ++bt) {
            const int c0 = bt * SR_EPI_COLS;
            float vor[SR_EPI_COLS], voi[SR_EPI_COLS], ver[SR_EPI_COLS], vei[SR_EPI_COLS];
            tmem_ld8_nowait(tbase + (uint32_t)c0, vor);
            tmem_ld8_nowait(tbase + (uint32_t)(NB + c0), voi);
            if (WIDE) {
#pragma unroll
                for (int q = 0; q < SR_EPI_COLS; ++q) {
                    const float2 ev = even[(long long)(c0 + q) * SR_M];
                    ver[q] = ev.x, vei[q] = ev.y;
                }
            } else {
                tmem_ld8_nowait(tbase + (uint32_t)(2 * NB + c0), ver);
                tmem_ld8_nowait(tbase + (uint32_t)(3 * NB + c0), vei);
            }
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            // branch-free per column, so that the columns of a batch overlap in the pipeline
#pragma unroll
            for (int q = 0; q < SR_EPI_COLS; ++q) {
                const SeriesCol cr = scol[c0 + q];
                const SeriesTerms tm = sterm[c0 + q];
                const float si = spin_from_bits(mybits, cr.site);
                // the column applies iff every further flip site q has s_q s_i equal to the column's relative sign
                bool active = cr.group >= 0;
                if (cr.sitek >= 0) {
                    active = active && (si * spin_from_bits(mybits, cr.sitek) == ((cr.par & 1) ? -1.f : 1.f));
                    if (!AFFINE) {
                        const int s2 = cr.sx & 0xffff, s3 = (cr.sx >> 16) & 0xffff;
                        if (s2 != 0xffff) active = active && (si * spin_from_bits(mybits, s2) == ((cr.par & 2) ? -1.f : 1.f));
                        if (s3 != 0xffff) active = active && (si * spin_from_bits(mybits, s3) == ((cr.par & 4) ? -1.f : 1.f));
                    }
                }
                // summed matrix element of the group (Eq. 39): two inline terms, or (rare) the general list
                float mr = fmaf(tm.crb, si, tm.cra), mi = fmaf(tm.cib, si, tm.cia);  // AFFINE: m0 + sigma m1
                if (!AFFINE) {
                    const float fa = spin_or_one(tm.z0a) * spin_or_one(tm.z1a), fb = spin_or_one(tm.z0b) * spin_or_one(tm.z1b);
                    mr = fmaf(tm.cra, fa, tm.crb * fb), mi = fmaf(tm.cia, fa, tm.cib * fb);
                }
                if (!AFFINE && (cr.count & SR_GENERIC_TERMS)) {
                    const int first = p.H.grp_first[cr.group], count = cr.count & SR_COUNT_MASK;
                    for (int u = 0; u < count; ++u) {
                        float f = spin_or_one(p.H.gt_z0[first + u]) * spin_or_one(p.H.gt_z1[first + u]);
                        if (p.H.has_zx)
                            for (int x = p.H.gt_zx_off[first + u]; x < p.H.gt_zx_off[first + u + 1]; ++x)
                                f *= spin_from_bits(mybits, p.H.gt_zx[x]);
                        const float2 cc = p.H.gt_c[first + u];
                        mr = fmaf(cc.x, f, mr);
                        mi = fmaf(cc.y, f, mi);
                    }
                }
                const bool live = active && (mr != 0.f || mi != 0.f);
                mr = live ? mr : 0.f;
                mi = live ? mi : 0.f;
                // log R = log kappa - sigma (2 A + ODD) - EVEN   (R = 1 for a dead column: nothing to overflow)
                const float zr = live ? cr.lkr - si * fmaf(SR_INV_ODD, vor[q], cr.a2r) - SR_INV_EVEN * ver[q] : 0.f;
                float zi = live ? cr.lki - si * fmaf(SR_INV_ODD, voi[q], cr.a2i) - SR_INV_EVEN * vei[q] : 0.f;
                const float kk = rintf(zi * 0.15915494309189535f);
                zi = fmaf(-kk, 6.2831855f, zi);
                zi = fmaf(-kk, -1.7484555e-7f, zi);
                float sn, cs;
                __sincosf(zi, &sn, &cs);
                const float mag = expf(zr);
                const float Rr = mag * cs, Ri = mag * sn;
                er_acc += mr * Rr - mi * Ri;
                ei_acc += mr * Ri + mi * Rr;
                // guard: |m R| (k0 + n2t k1 + n4t k2 + n6t k3 + n8t k4), valid while max |t| max |T| <= 1/2
                const float delta = fmaf(rn.x, cr.k1, fmaf(rn.y, cr.k2, fmaf(rn.z, cr.k3, fmaf(rn.w, cr.k4, cr.k0))));
                const float wgt = (fabsf(mr) + fabsf(mi)) * mag;
                const float bound = (rmax * cr.tmax <= 0.5f) ? wgt * delta : __int_as_float(0x7f800000);
                eps += live ? bound : 0.f;
            }
        }
        };
        if (tile_affine) columns(std::true_type{});
        else columns(std::false_type{});
        NQS_STAMP(4);
        // the other column parts hand their sums to part 0, which owns the row's output (fixed order: deterministic)
        if (part > 0) sred[(part - 1) * SR_M + row] = make_float4(er_acc, ei_acc, eps, 0.f);
        asm volatile("bar.sync 1, %0;" ::"n"(SR_EPI_THREADS) : "memory");
        if (part == 0 && b < p.B) {
#pragma unroll
            for (int q = 0; q < SR_EPI_PARTS - 1; ++q) {
                const float4 o = sred[q * SR_M + row];
                er_acc += o.x, ei_acc += o.y, eps += o.z;
            }
            p.partial[b * p.nNT + nt] = make_float4(er_acc, ei_acc, eps, 0.f);
        }
    }
#ifdef NQS_SERIES_TIMELINE
    if (p.timeline && tid == 64) {
        NQS_STAMP(5);
        for (int k = 0; k < 6; ++k) p.timeline[(long long)blockIdx.x * 8 + k] = stamp[k];
    }
#endif
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
}

// E_loc = sum of the column tiles' partial sums (the diagonal rides in tile 0); guard: the call fails as a
// whole if any sample's error bound exceeds SR_GUARD_FRACTION * 1e-4 * max(1, |E_loc|) (or is NaN).
// status[0] |= 1 when the guard fails (read by eloc_kernel / finalize_kernel), status[1] counts the samples.
// nS > 1: log psi = sum of the theta kernel's nS partial sums (float64, fixed order).
__global__ void series_guard_kernel(const float4* __restrict__ partial, long long B, int nNT, float2* __restrict__ eloc,
                                    int* __restrict__ status, const double2* __restrict__ lp_part, int nS,
                                    long long rows, float2* __restrict__ logpsi) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B) return;
    if (nS > 1 && logpsi) {
        double lr = 0.0, li = 0.0;
        for (int k = 0; k < nS; ++k) {
            const double2 v = lp_part[k * rows + b];
            lr += v.x, li += v.y;
        }
        logpsi[b] = make_float2((float)lr, (float)li);
    }
    float er = 0.f, ei = 0.f, eps = 0.f;
    for (int t = 0; t < nNT; ++t) {
        const float4 v = partial[b * nNT + t];
        er += v.x;
        ei += v.y;
        eps += v.z;
    }
    eloc[b] = make_float2(er, ei);
    const float mod = sqrtf(er * er + ei * ei);
    const bool ok = eps <= SR_GUARD_FRACTION * 1e-4f * fmaxf(1.f, mod);  // false for NaN
    if (!ok) {
        atomicOr(&status[0], 1);
        atomicAdd(&status[1], 1);
    }
}

// End of a series call: the debug record of the device ({guard flag, samples over, path tag 1}, nqs_debug_last_a5) and,
// for calls in automatic mode, the refusal latch of the handle: a record in pinned host memory the NEXT call reads
// without synchronising -- {sequence number of this call, guard flag, samples over}; the sequence number is written
// last, behind a system-wide fence, so a reader that sees it sees the flag of the same call.
__global__ void series_latch_kernel(const int* __restrict__ status, int* __restrict__ dstatus, volatile int* latch,
                                    int seq) {
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    const int flag = status[0], over = status[1];
    dstatus[0] = flag;
    dstatus[1] = over;
    dstatus[2] = 1;
    if (latch) {
        latch[1] = flag;
        latch[2] = over;
        __threadfence_system();
        latch[0] = seq;
    }
}

}  // namespace nqs
