// Small problems in ONE launch (SURVEY.md 7.1 "Small G"; steps a1 .. a6 of DESIGN.md section 1): below the size
// where the tensor-core path pays (B x columns x M < 2^28), a call used to be five launches of a few microseconds
// each whose latencies added up (configs 1 and 2: 0.10 / 0.14 ms).  Here one CTA owns SB samples and does, in
// shared memory and in this order,
//   theta = b + W s        W split into two float32 levels whose sums are exact / round at 2^-36 (s = +/-1), packed FFMA2,
//                          thread <-> (sample, 4 hidden units at a time)
//   log psi, t = tanh      lncosh_tanh per hidden unit, float64 partial sums over j in a fixed order
//   tables                 C = cosh 2V, S = sinh 2V per (hidden unit, column), rho = exp(-/+ 2A) per column (every CTA
//                          recomputes them: columns x M entries, a few percent of the CTA's work at SB = 128)
//   connected amplitudes   product form  R = rho prod_j (C_j - sigma t_j S_j)  (ratio identity R of nqs_kernels.cuh),
//                          thread <-> (two pairs of samples on packed FFMA2 operands, column), exponent pulled out
//                          every 16 hidden units
//   E_loc                  diagonal + sum over the columns in column order (deterministic)
// Same readings as the large kernels: a column applies when its relative signs match (Q4), an element that is
// exactly zero is skipped (Q5), psi(s) = 0 gives IEEE inf / NaN (Q7).
#pragma once
#include "nqs_device.cuh"

namespace nqs {

constexpr int SM_MAX_THREADS = 640;  // threads per CTA: chosen per call (small_threads)
constexpr int SM_MAX_SB = 128;

struct SmallParams {
    const int8_t* spins;   // [B][N]
    long long B;
    int N, M, C;
    const float2* a;       // [N]
    const float2* b;       // [M]
    const float2* W;       // [M][N]
    DevHam H;
    float2* eloc;          // [B]
    float2* logpsi;        // [B] or nullptr
    int SB;                // samples per CTA: a multiple of 4, at most SM_MAX_SB
};

__host__ __device__ inline int small_tstride(int M) { return M | 1; }                // float4 (a pair of samples) per row of t
__host__ __device__ inline int small_sstride(int N) { return (N + 3) / 4 * 4 + 4; }  // bytes per row of spins
__host__ __device__ inline size_t small_smem_bytes(int N, int M, int C, int SB) {
    const size_t region = (size_t)M * (size_t)(C > N ? C : N) * 16;  // W levels [M][N] float4, then tables [M][C] float4
    return region + (size_t)C * 16 + (size_t)(SB / 2) * small_tstride(M) * 16 + (size_t)SB * C * 8 +
           (size_t)SM_MAX_THREADS * 16 + (size_t)SB * small_sstride(N) + 64;
}
// threads per CTA: the (4 samples, column) items of the amplitude phase in as few whole rounds as possible
__host__ __device__ inline int small_threads(int C, int SB) {
    const int items = (SB / 4) * (C > 0 ? C : 1);
    const int rounds = (items + SM_MAX_THREADS - 1) / SM_MAX_THREADS;
    int T = ((items + rounds - 1) / rounds + 31) / 32 * 32;
    if (T < SB) T = (SB + 31) / 32 * 32;  // at least one thread per sample
    return T < 128 ? 128 : T;
}

#ifdef NQS_SMALL_TIMELINE
__device__ long long g_small_stamps[8];
#define NQS_SSTAMP(k) if (blockIdx.x == 0 && threadIdx.x == 0) g_small_stamps[k] = clock64()
#else
#define NQS_SSTAMP(k)
#endif

__global__ void __launch_bounds__(SM_MAX_THREADS) small_eloc_kernel(const SmallParams p) {
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int SM_THREADS = blockDim.x;
    const int N = p.N, M = p.M, C = p.C, SB = p.SB, JL = SM_THREADS / SB;
    const int ts = small_tstride(M), ss = small_sstride(N);
    float4* const tab = reinterpret_cast<float4*>(sm_raw);                // [M][C]  (Cr, Ci, Sr, Si) -- after theta
    float4* const wlv = tab;                                              // [M][N]  (Wh.re, Wh.im, Wl.re, Wl.im) -- before
    float4* const rho = tab + (size_t)M * (C > N ? C : N);                // [C]
    float4* const t_s = rho + C;                                          // [SB / 2][ts]  (tr0, tr1, ti0, ti1)
    float2* const contrib = reinterpret_cast<float2*>(t_s + (size_t)(SB / 2) * ts);  // [SB][C]
    double* const lp = reinterpret_cast<double*>(contrib + (size_t)SB * C);  // [SB][JL][2]
    int8_t* const sp = reinterpret_cast<int8_t*>(lp + (size_t)SB * JL * 2);  // [SB][ss]
    const int tid = threadIdx.x;
    const long long b0 = (long long)blockIdx.x * SB;

    NQS_SSTAMP(0);
    // spins of the CTA's samples (rows past the batch repeat the last sample; nothing of them is stored)
    for (int idx = tid; idx < SB * N; idx += SM_THREADS) {
        const int r = idx / N, i = idx - r * N;
        const long long b = b0 + r < p.B ? b0 + r : p.B - 1;
        sp[r * ss + i] = p.spins[b * N + i];
    }
    // W in two float32 levels per hidden unit: Wh on a grid of 2^-k with |Wh| 2^k <= 2^11 (every partial sum of
    // +/- Wh is then exact in float32 for N <= 8192), Wl = W - Wh exactly (|Wl| <= 2^-12 max|W_j|: its sums round at
    // 2^-36 of the row scale).  theta = b + sum Wh s + sum Wl s is what the int8 tensor-core kernel computes to 2^-28.
    for (int jw = (tid >> 5) * 4; jw < M; jw += SM_THREADS / 8) {  // eight threads per row, four rows per warp
        const int l8 = tid & 7, j = jw + ((tid & 31) >> 3);
        const float2* const wrow = p.W + (long long)(j < M ? j : jw) * N;
        float mx = 0.f;
        for (int i = l8; i < N; i += 8) mx = fmaxf(mx, fmaxf(fabsf(wrow[i].x), fabsf(wrow[i].y)));
        for (int o = 4; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o, 8));
        // a row below 2^-100 keeps e = 0 like an all-zero row (Wh = 0, Wl = W: the sums of such values need no split);
        // 2^(11 - e) would otherwise overflow to inf for max|W_j| < ~2^-116 and inf * 0 = NaN poison theta
        int e = 0;
        if (mx > 7.8e-31f && mx < 3.0e38f) (void)frexpf(mx, &e);  // mx = f 2^e, f in [0.5, 1)
        const float up = ldexpf(1.f, 11 - e), dn = ldexpf(1.f, e - 11);
        for (int i = l8; i < N && j < M; i += 8) {
            const float2 w = wrow[i];
            const float hr = rintf(w.x * up) * dn, hi = rintf(w.y * up) * dn;
            wlv[j * N + i] = make_float4(hr, hi, w.x - hr, w.y - hi);
        }
    }
    __syncthreads();
    NQS_SSTAMP(1);

    // a2 + a3: thread <-> (sample r, hidden units jl, jl + JL, ...), four hidden units at a time
    {
        const int r = tid % SB, jl = tid / SB;  // threads beyond SB * JL idle in this phase
        const int8_t* const srow = sp + r * ss;
        float* const tdst = reinterpret_cast<float*>(t_s + (size_t)(r >> 1) * ts) + (r & 1);
        double lr = 0.0, li = 0.0;
        for (int j0 = jl; j0 < M && jl < JL; j0 += 4 * JL) {
            float2 ah[4], al[4];
            int wo[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                ah[u] = al[u] = make_float2(0.f, 0.f);
                const int j = j0 + u * JL;
                wo[u] = (j < M ? j : j0) * N;
            }
#pragma unroll 4
            for (int i = 0; i < N; ++i) {
                const float2 s2 = bc2((float)srow[i]);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float4 w = wlv[wo[u] + i];
                    ah[u] = __ffma2_rn(s2, make_float2(w.x, w.y), ah[u]);
                    al[u] = __ffma2_rn(s2, make_float2(w.z, w.w), al[u]);
                }
            }
            // log cosh and tanh of the four units, two at a time (packed Taylor series for |theta|^2 < 0.36, the stable
            // closed form lane by lane otherwise: nqs_device.cuh)
#pragma unroll
            for (int u = 0; u < 4; u += 2) {
                const int ja = j0 + u * JL, jb = ja + JL;
                const float2 ba = ja < M ? p.b[ja] : make_float2(0.f, 0.f), bb = jb < M ? p.b[jb] : make_float2(0.f, 0.f);
                const float2 xr = make_float2(ah[u].x + (al[u].x + ba.x), ah[u + 1].x + (al[u + 1].x + bb.x));
                const float2 xi = make_float2(ah[u].y + (al[u].y + ba.y), ah[u + 1].y + (al[u + 1].y + bb.y));
                float2 l_r, l_i, t_r, t_i;
                lncosh_tanh2(xr, xi, l_r, l_i, t_r, t_i);
                if (ja < M) {
                    lr += (double)l_r.x;
                    li += (double)l_i.x;
                    tdst[4 * ja] = t_r.x;
                    tdst[4 * ja + 2] = t_i.x;
                }
                if (jb < M) {
                    lr += (double)l_r.y;
                    li += (double)l_i.y;
                    tdst[4 * jb] = t_r.y;
                    tdst[4 * jb + 2] = t_i.y;
                }
            }
        }
        if (jl < JL) {
            lp[(r * JL + jl) * 2] = lr;
            lp[(r * JL + jl) * 2 + 1] = li;
        }
    }
    __syncthreads();
    NQS_SSTAMP(2);

    // a1: tables (over the W levels, which are dead now)
    for (int idx = tid; idx < M * C; idx += SM_THREADS) {
        const int j = idx / C, c = idx - j * C;
        const float2 v = column_sum(p.H, c, p.W + (long long)j * N);
        const float x = 2.f * v.x, y = 2.f * v.y;
        float sy, cy;
        sincosf(y, &sy, &cy);
        const float sh = sinhf(x), ch = coshf(x);
        tab[idx] = make_float4(ch * cy, sh * sy, sh * cy, ch * sy);
    }
    for (int c = tid; c < C; c += SM_THREADS) {
        const float2 A = column_sum(p.H, c, p.a);
        float sy, cy;
        sincosf(2.f * A.y, &sy, &cy);
        const float em = expf(-2.f * A.x), ep = expf(2.f * A.x);
        rho[c] = make_float4(em * cy, -em * sy, ep * cy, ep * sy);
    }
    __syncthreads();
    NQS_SSTAMP(3);

    // a4 + a5: thread <-> (samples 4 q .. 4 q + 3 = two pairs on packed FFMA2 operands, column c)
    const int nItems = (SB / 4) * C;
    for (int item = tid; item < nItems; item += SM_THREADS) {
        const int q4 = item / C, c = item - q4 * C;
        const int site = p.H.col_i[c];
        float2 Pr[2], Pi[2], sg[2];
        int2 ex[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            ex[h] = make_int2(0, 0);
            Pr[h] = make_float2(1.f, 1.f), Pi[h] = make_float2(0.f, 0.f);
            sg[h] = make_float2((float)sp[(4 * q4 + 2 * h) * ss + site], (float)sp[(4 * q4 + 2 * h + 1) * ss + site]);
        }
        const float4* const trow = t_s + (size_t)(2 * q4) * ts;
        for (int j0 = 0; j0 < M; j0 += 16) {
            const int j1 = min(M, j0 + 16);
#pragma unroll 4
            for (int j = j0; j < j1; ++j) {
                const float4 e = tab[j * C + c];
                const float2 Cr = bc2(e.x), Ci = bc2(e.y), Sr = bc2(e.z), Si = bc2(e.w);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float4 t = trow[h * ts + j];
                    const float2 ur = __fmul2_rn(sg[h], make_float2(t.x, t.y));   // sigma t
                    const float2 ui = __fmul2_rn(sg[h], make_float2(t.z, t.w));
                    const float2 fr = __ffma2_rn(neg2(ur), Sr, __ffma2_rn(ui, Si, Cr));       // C - sigma t S
                    const float2 fi = __ffma2_rn(neg2(ur), Si, __ffma2_rn(neg2(ui), Sr, Ci));
                    const float2 nr = __ffma2_rn(neg2(Pi[h]), fi, __fmul2_rn(Pr[h], fr));
                    Pi[h] = __ffma2_rn(Pi[h], fr, __fmul2_rn(Pr[h], fi));
                    Pr[h] = nr;
                }
            }
            // range safety: pull the exponent out when a running product leaves [2^-40, 2^40]
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float m0 = fmaxf(fabsf(Pr[h].x), fabsf(Pi[h].x)), m1 = fmaxf(fabsf(Pr[h].y), fabsf(Pi[h].y));
                if (m0 > 1.0995116e12f || (m0 < 9.094947e-13f && m0 > 0.f)) {
                    int e2;
                    (void)frexpf(m0, &e2);
                    Pr[h].x = ldexpf(Pr[h].x, -e2);
                    Pi[h].x = ldexpf(Pi[h].x, -e2);
                    ex[h].x += e2;
                }
                if (m1 > 1.0995116e12f || (m1 < 9.094947e-13f && m1 > 0.f)) {
                    int e2;
                    (void)frexpf(m1, &e2);
                    Pr[h].y = ldexpf(Pr[h].y, -e2);
                    Pi[h].y = ldexpf(Pi[h].y, -e2);
                    ex[h].y += e2;
                }
            }
        }
        const int g = p.H.col_group[c];
        const float4 rh = rho[c];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int r = 4 * q4 + q;
            const int8_t* const srow = sp + r * ss;
            const int si = srow[site];
            const float pr = (q & 1) ? Pr[q >> 1].y : Pr[q >> 1].x, pi = (q & 1) ? Pi[q >> 1].y : Pi[q >> 1].x;
            float cr = 0.f, ci = 0.f;
            if (g >= 0 && column_active(p.H, srow, c, si)) {
                const float2 m = group_element(p.H, srow, g);
                if (m.x != 0.f || m.y != 0.f) {
                    const float rr = si > 0 ? rh.x : rh.z, ri = si > 0 ? rh.y : rh.w;
                    const float vr = m.x * rr - m.y * ri, vi = m.x * ri + m.y * rr;
                    const int e2 = (q & 1) ? ex[q >> 1].y : ex[q >> 1].x;
                    cr = ldexpf(vr * pr - vi * pi, e2);
                    ci = ldexpf(vr * pi + vi * pr, e2);
                }
            }
            contrib[r * C + c] = make_float2(cr, ci);
        }
    }
    __syncthreads();
    NQS_SSTAMP(4);

    // a6 (+ the visible bias of log psi): four adjacent lanes per sample, each a quarter of the diagonal terms, of the
    // columns and of the sites; the four partial sums are added in lane order (fixed: deterministic)
    for (int base = 0; base < 4 * SB; base += SM_THREADS) {
        const int item = base + tid;
        const bool on = item < 4 * SB;                      // whole warps stay in the loop for the shuffles
        const int r = on ? item >> 2 : 0, q4 = item & 3;
        const long long b = b0 + r;
        const int8_t* const srow = sp + r * ss;
        float er = 0.f, ei = 0.f, ar = 0.f, ai = 0.f;
        if (on) {
            for (int t = q4; t < p.H.Td; t += 4) {
                const int z0 = p.H.diag_z0[t], z1 = p.H.diag_z1[t];
                float f = 1.f;
                if (z0 >= 0) f *= (float)srow[z0];
                if (z1 >= 0) f *= (float)srow[z1];
                if (p.H.has_zx)
                    for (int x = p.H.diag_zx_off[t]; x < p.H.diag_zx_off[t + 1]; ++x) f *= (float)srow[p.H.diag_zx[x]];
                const float2 cc = p.H.diag_c[t];
                er = fmaf(cc.x, f, er);
                ei = fmaf(cc.y, f, ei);
            }
            for (int c = q4; c < C; c += 4) {
                er += contrib[r * C + c].x;
                ei += contrib[r * C + c].y;
            }
            if (p.logpsi)
                for (int i = q4; i < N; i += 4) {
                    const float sv = (float)srow[i];
                    const float2 av = p.a[i];
                    ar = fmaf(av.x, sv, ar);
                    ai = fmaf(av.y, sv, ai);
                }
        }
        const int l0 = (tid & 31) & ~3;
        float sr = 0.f, si = 0.f, br = 0.f, bi = 0.f;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            sr += __shfl_sync(0xffffffffu, er, l0 + k);
            si += __shfl_sync(0xffffffffu, ei, l0 + k);
            br += __shfl_sync(0xffffffffu, ar, l0 + k);
            bi += __shfl_sync(0xffffffffu, ai, l0 + k);
        }
        if (on && q4 == 0 && b < p.B) {
            p.eloc[b] = make_float2(sr, si);
            if (p.logpsi) {
                double lr = 0.0, li = 0.0;
                for (int k = 0; k < JL; ++k) {
                    lr += lp[(r * JL + k) * 2];
                    li += lp[(r * JL + k) * 2 + 1];
                }
                p.logpsi[b] = make_float2((float)(lr + (double)br), (float)(li + (double)bi));
            }
        }
    }
    __syncthreads();
    NQS_SSTAMP(5);
}

}  // namespace nqs
