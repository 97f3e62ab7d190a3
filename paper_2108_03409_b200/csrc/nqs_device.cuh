// Device-side data structures and math helpers shared by the kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nqs {

// Device image of the compiled Hamiltonian (see nqs_hamiltonian.h).  All pointers are device
// pointers into one allocation owned by the nqs_hamiltonian handle.
struct DevHam {
    int N, G, C, Td, Tg;
    const int* diag_z0;
    const int* diag_z1;
    const float2* diag_c;
    const int* grp_f0;
    const int* grp_f1;
    const int* grp_first;
    const int* grp_count;
    const int* gt_z0;
    const int* gt_z1;
    const float2* gt_c;
    // columns, padded to C_pad entries (col_group = -1 marks padding)
    const int* col_i;
    const int* col_k;
    const int* col_p;
    const int* col_group;
    // k-site Pauli strings: third / fourth flip site of a group and of a column (-1: none)
    // with the column's relative signs, and the z sites of a term beyond the first two (has_zx: any at all)
    const int* grp_f2;
    const int* grp_f3;
    const int* col_s2;
    const int* col_p2;
    const int* col_s3;
    const int* col_p3;
    int has_zx;
    const int* diag_zx_off;
    const int* diag_zx;
    const int* gt_zx_off;
    const int* gt_zx;
};

__device__ __forceinline__ float2 bc2(float x) { return make_float2(x, x); }
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }

// Summed matrix element of flip group g for the configuration `srow` (Eq. 39):
// m = sum_{t in g} c'_t * s[z0_t] * s[z1_t]   (c' carries (-i)^{n_Y}; z = -1 means factor 1).
__device__ __forceinline__ float2 group_element(const DevHam& H, const int8_t* __restrict__ srow, int g) {
    const int first = H.grp_first[g], count = H.grp_count[g];
    float mr = 0.f, mi = 0.f;
    for (int q = 0; q < count; ++q) {
        const int z0 = H.gt_z0[first + q], z1 = H.gt_z1[first + q];
        float f = 1.f;
        if (z0 >= 0) f *= (float)srow[z0];
        if (z1 >= 0) f *= (float)srow[z1];
        if (H.has_zx)
            for (int x = H.gt_zx_off[first + q]; x < H.gt_zx_off[first + q + 1]; ++x) f *= (float)srow[H.gt_zx[x]];
        const float2 c = H.gt_c[first + q];
        mr = fmaf(c.x, f, mr);
        mi = fmaf(c.y, f, mi);
    }
    return make_float2(mr, mi);
}

// Is column c (flip sites ci [, ck, s2, s3] with relative signs cp, p2, p3) the one that applies to `srow`?
__device__ __forceinline__ bool column_active(const DevHam& H, const int8_t* __restrict__ srow, int c, int si) {
    const int ck = H.col_k[c];
    if (ck < 0) return true;
    if ((int)srow[ck] * si != H.col_p[c]) return false;
    const int s2 = H.col_s2[c];
    if (s2 < 0) return true;
    if ((int)srow[s2] * si != H.col_p2[c]) return false;
    const int s3 = H.col_s3[c];
    return s3 < 0 || (int)srow[s3] * si == H.col_p3[c];
}

// V_j = W[j, i] + p W[j, k] + p2 W[j, s2] + p3 W[j, s3] of a column (absent sites: -1), likewise for the bias a
__device__ __forceinline__ float2 column_sum(const DevHam& H, int c, const float2* __restrict__ row) {
    float2 v = row[H.col_i[c]];
    const int k = H.col_k[c];
    if (k >= 0) {
        const float p = (float)H.col_p[c];
        v.x = fmaf(p, row[k].x, v.x);
        v.y = fmaf(p, row[k].y, v.y);
        const int s2 = H.col_s2[c];
        if (s2 >= 0) {
            const float p2 = (float)H.col_p2[c];
            v.x = fmaf(p2, row[s2].x, v.x);
            v.y = fmaf(p2, row[s2].y, v.y);
            const int s3 = H.col_s3[c];
            if (s3 >= 0) {
                const float p3 = (float)H.col_p3[c];
                v.x = fmaf(p3, row[s3].x, v.x);
                v.y = fmaf(p3, row[s3].y, v.y);
            }
        }
    }
    return v;
}

// Sum of the diagonal terms (empty flip set): d = sum_t c_t * s[z0] * s[z1].
__device__ __forceinline__ float2 diagonal_element(const DevHam& H, const int8_t* __restrict__ srow) {
    float dr = 0.f, di = 0.f;
    for (int t = 0; t < H.Td; ++t) {
        const int z0 = H.diag_z0[t], z1 = H.diag_z1[t];
        float f = 1.f;
        if (z0 >= 0) f *= (float)srow[z0];
        if (z1 >= 0) f *= (float)srow[z1];
        if (H.has_zx)
            for (int x = H.diag_zx_off[t]; x < H.diag_zx_off[t + 1]; ++x) f *= (float)srow[H.diag_zx[x]];
        const float2 c = H.diag_c[t];
        dr = fmaf(c.x, f, dr);
        di = fmaf(c.y, f, di);
    }
    return make_float2(dr, di);
}

// log cosh z and tanh z for z = x + i y, float32, written for accuracy at small |z| (the
// log psi tolerance is 1e-5 absolute on a sum of M terms) and stability at large |x|.
//   |cosh z|^2 = cosh^2 x - sin^2 y = 1 + (sinh^2 x - sin^2 y)
//   arg cosh z = atan2(tanh x sin y, cos y)            (principal value per hidden unit, Q6)
//   tanh z     = [tanh x + i sin y cos y sech^2 x] / (cos^2 y + tanh^2 x sin^2 y)
__device__ __forceinline__ void lncosh_tanh(float x, float y, float& lr, float& li, float& tr, float& ti) {
    const float ax = fabsf(x);
    float s, c;
    sincosf(y, &s, &c);
    float th, sech2;
    if (ax < 4.0f) {
        const float sh = sinhf(x);
        const float ch2 = fmaf(sh, sh, 1.0f);
        th = sh * rsqrtf(ch2);
        sech2 = 1.0f / ch2;
        // |cosh z|^2 = 1 + (sinh^2 x - sin^2 y) = sinh^2 x + cos^2 y: the first form keeps relative
        // accuracy at small |z|, the second near the zeros of cosh (y -> pi/2, x -> 0)
        const float s2 = s * s;
        lr = (s2 > 0.5f) ? 0.5f * logf(fmaf(sh, sh, c * c)) : 0.5f * log1pf(fmaf(sh, sh, -s2));
    } else {
        const float q = expf(-2.0f * ax);  // <= 3.4e-4
        const float d = 1.0f + q;
        th = copysignf((1.0f - q) / d, x);
        sech2 = 4.0f * q / (d * d);
        const float cos2y2 = 2.0f * (c * c - s * s);
        lr = ax - 0.69314718055994531f + 0.5f * log1pf(q * (cos2y2 + q));
    }
    li = atan2f(th * s, c);
    const float D = fmaf(c, c, th * th * s * s);
    const float inv = 1.0f / D;
    tr = th * inv;
    ti = s * c * sech2 * inv;
}

// The same for TWO arguments at once, (x.x + i y.x) and (x.y + i y.y), on packed FFMA2 operands.  Small |z|
// (|z|^2 < 0.36, every hidden unit of the five configurations): Taylor series in w = z^2,
//   log cosh z = w (1/2 - w/12 + w^2/45 - ...)  (8 terms),   tanh z = z (1 - w/3 + 2 w^2/15 - ...)  (9 terms),
// pure FMA, no cancellation: absolute error <= 3e-8 on log cosh (unbiased: 3e-7 on a sum of 1600 units against the
// 1e-5 tolerance of log psi), relative error <= 1.2e-7 on tanh (float32 emulation over the full range, round 2).
// Anything else (|z|^2 >= 0.36, NaN) takes lncosh_tanh above, lane by lane.
__device__ __forceinline__ void lncosh_tanh2(float2 x, float2 y, float2& lr, float2& li, float2& tr, float2& ti) {
    const float2 yy = __fmul2_rn(y, y);
    const float2 wr = __ffma2_rn(x, x, neg2(yy));
    const float2 wi = __fmul2_rn(__fadd2_rn(x, x), y);
    const float2 nwi = neg2(wi);
    // Horner in w with real coefficients: (pr, pi) <- (pr, pi) w + c
    float2 pr, pi, nr;
#define NQS_HORNER(c)                              \
    nr = __ffma2_rn(pr, wr, bc2(c));               \
    nr = __ffma2_rn(pi, nwi, nr);                  \
    pi = __ffma2_rn(pi, wr, __fmul2_rn(pr, wi));   \
    pr = nr;
    pr = __ffma2_rn(bc2(-9.09896491907074e-05f), wr, bc2(2.565805740408915e-04f));
    pi = __fmul2_rn(bc2(-9.09896491907074e-05f), wi);
    NQS_HORNER(-7.386029608251831e-04f)
    NQS_HORNER(2.1869488536155205e-03f)
    NQS_HORNER(-6.746031746031746e-03f)
    NQS_HORNER(2.2222222222222223e-02f)
    NQS_HORNER(-8.333333333333333e-02f)
    NQS_HORNER(0.5f)
    lr = __ffma2_rn(pi, nwi, __fmul2_rn(pr, wr));
    li = __ffma2_rn(pi, wr, __fmul2_rn(pr, wi));
    pr = __ffma2_rn(bc2(5.90027440945586e-04f), wr, bc2(-1.4558343870513183e-03f));
    pi = __fmul2_rn(bc2(5.90027440945586e-04f), wi);
    NQS_HORNER(3.592128036572481e-03f)
    NQS_HORNER(-8.863235529902197e-03f)
    NQS_HORNER(2.1869488536155203e-02f)
    NQS_HORNER(-5.396825396825397e-02f)
    NQS_HORNER(0.13333333333333333f)
    NQS_HORNER(-0.3333333333333333f)
    NQS_HORNER(1.0f)
#undef NQS_HORNER
    tr = __ffma2_rn(pi, neg2(y), __fmul2_rn(pr, x));
    ti = __ffma2_rn(pi, x, __fmul2_rn(pr, y));
    const float m0 = fmaf(x.x, x.x, yy.x), m1 = fmaf(x.y, x.y, yy.y);
    if (!(m0 < 0.36f && m1 < 0.36f)) {  // rare: one branch for the pair
        if (!(m0 < 0.36f)) lncosh_tanh(x.x, y.x, lr.x, li.x, tr.x, ti.x);
        if (!(m1 < 0.36f)) lncosh_tanh(x.y, y.y, lr.y, li.y, tr.y, ti.y);
    }
}

// ---- mbarrier / bulk-copy (TMA engine, non-tensor) helpers: PTX for sm_90+/sm_100a ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// the same for warps that wait through a whole main loop: sleep between polls instead of spinning
__device__ __forceinline__ void mbar_wait_sleep(uint64_t* bar, uint32_t parity, uint32_t ns) {
    uint32_t done = 0;
    while (true) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (done) break;
        __nanosleep(ns);
    }
}
// global -> shared bulk copy, completion signalled on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

}  // namespace nqs
