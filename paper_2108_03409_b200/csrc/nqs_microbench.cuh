// Pipe-rate micro-benchmarks behind nqs_microbench() (include/nqs.h): the on-box FP32 / MUFU peaks
// that SURVEY.md 8(d)(ii) asks the roofline to be quoted against, and the register-only ceiling of
// the a5 inner-loop body.  Pure register kernels: no memory traffic inside the timed loop.
#pragma once
#include <cuda_runtime.h>

namespace nqs {

enum { MB_FFMA = 0, MB_FFMA2 = 1, MB_BODY_PACKED = 2, MB_BODY_SCALAR = 3, MB_MUFU_EX2 = 4, MB_KINDS = 5 };

// lane-operations one thread performs per loop iteration, by kind
__host__ __device__ constexpr int mb_ops_per_iter(int kind) {
    return kind == MB_FFMA ? 16 : kind == MB_FFMA2 ? 16 : kind == MB_MUFU_EX2 ? 8 : 64;
}

template <int KIND>
__global__ void __launch_bounds__(320, 2) microbench_kernel(float* out, int iters, float a0, float b0) {
    float2 acc[8], x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        acc[i] = make_float2(1.f + i, 2.f + threadIdx.x);
        x[i] = make_float2(a0 + i * 1e-3f, a0 - i * 1e-3f);
    }
    const float2 m = make_float2(b0, b0 * 0.5f);
    const float4 e = make_float4(1.f, a0, b0, a0 * b0);  // (Cr, Ci, Sr, Si)
    float2 Pr[4], Pi[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        Pr[i] = make_float2(1.f, 1.f);
        Pi[i] = make_float2(0.f, 0.f);
    }
    for (int it = 0; it < iters; ++it) {
        if (KIND == MB_FFMA) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                acc[i].x = fmaf(acc[i].x, m.x, x[i].x);
                acc[i].y = fmaf(acc[i].y, m.y, x[i].y);
            }
        } else if (KIND == MB_FFMA2) {
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] = __ffma2_rn(acc[i], make_float2(e.z, e.z), make_float2(e.x, e.x));
        } else if (KIND == MB_MUFU_EX2) {
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i].x = exp2f(acc[i].x) * 0.25f;  // MUFU.EX2 + 1 FMUL
        } else {
            // the a5 body for 4 sample pairs: r = C + u S, P <- P r (8 packed / 16 scalar FMA-pipe ops)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const float2 ur = x[r], ui = x[r + 4];
                float2 rr, ri, nr, ni;
                if (KIND == MB_BODY_PACKED) {
                    rr = __ffma2_rn(ur, make_float2(e.z, e.z), make_float2(e.x, e.x));
                    rr = __ffma2_rn(ui, make_float2(-e.w, -e.w), rr);
                    ri = __ffma2_rn(ur, make_float2(e.w, e.w), make_float2(e.y, e.y));
                    ri = __ffma2_rn(ui, make_float2(e.z, e.z), ri);
                    nr = __fmul2_rn(Pr[r], rr);
                    nr = __ffma2_rn(make_float2(-Pi[r].x, -Pi[r].y), ri, nr);
                    ni = __fmul2_rn(Pr[r], ri);
                    ni = __ffma2_rn(Pi[r], rr, ni);
                } else {
                    rr.x = fmaf(ur.x, e.z, e.x), rr.y = fmaf(ur.y, e.z, e.x);
                    rr.x = fmaf(ui.x, -e.w, rr.x), rr.y = fmaf(ui.y, -e.w, rr.y);
                    ri.x = fmaf(ur.x, e.w, e.y), ri.y = fmaf(ur.y, e.w, e.y);
                    ri.x = fmaf(ui.x, e.z, ri.x), ri.y = fmaf(ui.y, e.z, ri.y);
                    nr.x = Pr[r].x * rr.x, nr.y = Pr[r].y * rr.y;
                    nr.x = fmaf(-Pi[r].x, ri.x, nr.x), nr.y = fmaf(-Pi[r].y, ri.y, nr.y);
                    ni.x = Pr[r].x * ri.x, ni.y = Pr[r].y * ri.y;
                    ni.x = fmaf(Pi[r].x, rr.x, ni.x), ni.y = fmaf(Pi[r].y, rr.y, ni.y);
                }
                Pr[r] = nr;
                Pi[r] = ni;
                x[r].x += 1e-7f;  // keeps r loop-variant (1 extra FADD per 8 packed ops)
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i].x + acc[i].y;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += Pr[i].x + Pr[i].y + Pi[i].x + Pi[i].y;
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace nqs
