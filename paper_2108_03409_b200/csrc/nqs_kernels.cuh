// CUDA kernels of the local-energy hot path (sm_100a).  Steps a1..a6 of DESIGN.md:
//   a1 table_kernel      per-call parameter tables  C = cosh 2V, S = sinh 2V, rho = exp(-/+ 2A)
//   a2 theta_kernel      theta = b + W s  (FP32 SIMT, FFMA2), fused with
//   a3                   log psi = a.s + sum_j log cosh theta_j  and  t = tanh theta
//   a4 group_element()   device-side enumerator of connected configurations (nqs_device.cuh)
//   a5 eloc_kernel       connected amplitudes, product form
//                           psi(s')/psi(s) = rho * prod_j (C_j - sigma t_j S_j)
//   a6 eloc_kernel epilogue + finalize_kernel   E_loc = d + sum_g m_g R_g
// Ratio identity (addition theorem): cosh(theta - delta)/cosh(theta) = cosh delta - tanh theta sinh delta
// with delta_j = 2 sigma V_j, V_j = W_ji (+/- W_jk for a pair flip), sigma = s_i.
#pragma once
#include "nqs_device.cuh"

namespace nqs {

// ----------------------------------------------------------------------------------------
// a1: parameter tables.  tab layout [tile][M_pad][TC] float4 = (Cr, Ci, Sr, Si); rows j >= M and
// padded columns hold (1,0,0,0) so they multiply the running product by 1.
// rho[c] = (exp(-2A).re, exp(-2A).im, exp(+2A).re, exp(+2A).im), A = a_i + p a_k.
// ----------------------------------------------------------------------------------------
__global__ void table_kernel(const float2* __restrict__ W, const float2* __restrict__ a, int N, int M, int M_pad,
                             int C, int TC, int nTiles, DevHam H,
                             float4* __restrict__ tab, float4* __restrict__ rho, const int* __restrict__ gate) {
    if (gate && !(gate[0] & 1)) return;  // fallback pass: only if the series guard failed
    const int C_pad = nTiles * TC;
    const long long total = (long long)M_pad * C_pad;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(idx % C_pad);
        const int j = (int)(idx / C_pad);
        float4 e = make_float4(1.f, 0.f, 0.f, 0.f);
        if (c < C && j < M) {
            const float2 v = column_sum(H, c, W + (long long)j * N);
            const float x = 2.f * v.x, y = 2.f * v.y;
            float sy, cy;
            sincosf(y, &sy, &cy);
            const float sh = sinhf(x), ch = coshf(x);
            e = make_float4(ch * cy, sh * sy, sh * cy, ch * sy);
        }
        const int tile = c / TC, cl = c % TC;
        tab[((long long)tile * M_pad + j) * TC + cl] = e;
        if (j == 0) {
            float4 r = make_float4(1.f, 0.f, 1.f, 0.f);
            if (c < C) {
                const float2 A = column_sum(H, c, a);
                float sy, cy;
                sincosf(2.f * A.y, &sy, &cy);
                const float em = expf(-2.f * A.x), ep = expf(2.f * A.x);
                r = make_float4(em * cy, -em * sy, ep * cy, ep * sy);
            }
            rho[c] = r;
        }
    }
}

// ----------------------------------------------------------------------------------------
// a2 + a3: theta contraction, log psi, tanh(theta).
// Block = 256 threads, tile = 64 samples x 64 hidden units, loops over all hidden tiles so that
// log psi needs no cross-block reduction.  Thread (tb, tj) owns samples 4 tb .. 4 tb + 3 and hidden
// units tj + 16 q.  theta accumulators are (re, im) pairs updated with packed FFMA2.
// Output tp[j][pair] = (tr_b0, tr_b1, ti_b0, ti_b1) for pair = (b0, b0 + 1), written as whole
// 512-byte rows through a shared-memory transpose.
// ----------------------------------------------------------------------------------------
constexpr int TH_KI = 32;
constexpr size_t TH_SMEM = (sizeof(float) + sizeof(float2)) * TH_KI * 64 + sizeof(float4) * 64 * 33;

__global__ void __launch_bounds__(256) theta_kernel(const int8_t* __restrict__ spins, long long B, int N, int M,
                                                    int M_pad, const float2* __restrict__ a,
                                                    const float2* __restrict__ bvec, const float2* __restrict__ W,
                                                    float4* __restrict__ tp, long long nPairsPad,
                                                    float2* __restrict__ logpsi, int raw_theta,
                                                    const int* __restrict__ gate) {
    extern __shared__ __align__(16) unsigned char th_smem[];
    if (gate && !(gate[0] & 1)) return;
    float(*sS)[64] = reinterpret_cast<float(*)[64]>(th_smem);
    float2(*sW)[64] = reinterpret_cast<float2(*)[64]>(th_smem + sizeof(float) * TH_KI * 64);
    float4(*sT)[33] = reinterpret_cast<float4(*)[33]>(th_smem + (sizeof(float) + sizeof(float2)) * TH_KI * 64);

    const int tid = threadIdx.x;
    const int tb = tid >> 4, tj = tid & 15;
    const long long b0 = (long long)blockIdx.x * 64;
    double lpr[4] = {0, 0, 0, 0}, lpi[4] = {0, 0, 0, 0};

    const int nJT = (M_pad + 63) / 64;
    for (int jt = 0; jt < nJT; ++jt) {
        const int j0 = jt * 64;
        float2 acc[4][4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int j = j0 + tj + 16 * q;
            const float2 bj = (j < M) ? bvec[j] : make_float2(0.f, 0.f);
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[e][q] = bj;
        }
        for (int i0 = 0; i0 < N; i0 += TH_KI) {
            __syncthreads();
            {   // spins tile [64 samples][32 sites] -> sS[site][sample] as float
                const int sm = tid >> 2, ib = (tid & 3) * 8;
                const long long b = b0 + sm;
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int i = i0 + ib + k;
                    float v = 0.f;
                    if (b < B && i < N) v = (float)spins[b * N + i];
                    sS[ib + k][sm] = v;
                }
                // W tile [64 hidden][32 sites] -> sW[site][hidden]
                const int j = j0 + sm;
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int i = i0 + ib + k;
                    float2 v = make_float2(0.f, 0.f);
                    if (j < M && i < N) v = W[(long long)j * N + i];
                    sW[ib + k][sm] = v;
                }
            }
            __syncthreads();
#pragma unroll 8
            for (int i = 0; i < TH_KI; ++i) {
                const float4 s4 = *reinterpret_cast<const float4*>(&sS[i][tb * 4]);
                float2 w[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) w[q] = sW[i][tj + 16 * q];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    acc[0][q] = __ffma2_rn(bc2(s4.x), w[q], acc[0][q]);
                    acc[1][q] = __ffma2_rn(bc2(s4.y), w[q], acc[1][q]);
                    acc[2][q] = __ffma2_rn(bc2(s4.z), w[q], acc[2][q]);
                    acc[3][q] = __ffma2_rn(bc2(s4.w), w[q], acc[3][q]);
                }
            }
        }
        // epilogue of this hidden tile: log cosh, tanh
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int jl = tj + 16 * q;
            const bool live = (j0 + jl) < M;
            float tr[4], ti[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (raw_theta) {  // tp receives theta itself (nqs_metropolis)
                    tr[e] = live ? acc[e][q].x : 0.f;
                    ti[e] = live ? acc[e][q].y : 0.f;
                    continue;
                }
                float lr, li;
                lncosh_tanh(acc[e][q].x, acc[e][q].y, lr, li, tr[e], ti[e]);
                if (live) {
                    lpr[e] += (double)lr;
                    lpi[e] += (double)li;
                } else {
                    tr[e] = 0.f;
                    ti[e] = 0.f;
                }
            }
            if (tp) {
                sT[jl][tb * 2 + 0] = make_float4(tr[0], tr[1], ti[0], ti[1]);
                sT[jl][tb * 2 + 1] = make_float4(tr[2], tr[3], ti[2], ti[3]);
            }
        }
        if (tp) {
            __syncthreads();
            const long long pair0 = b0 >> 1;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int idx = tid + 256 * k;
                const int jl = idx >> 5, pl = idx & 31;
                if (j0 + jl < M_pad) tp[(long long)(j0 + jl) * nPairsPad + pair0 + pl] = sT[jl][pl];
            }
        }
    }
    // visible bias: sum_i a_i s_i, sites i = tj, tj + 16, ...
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long b = b0 + tb * 4 + e;
        if (b < B) {
            float ar = 0.f, ai = 0.f;
            for (int i = tj; i < N; i += 16) {
                const float s = (float)spins[b * N + i];
                const float2 av = a[i];
                ar = fmaf(av.x, s, ar);
                ai = fmaf(av.y, s, ai);
            }
            lpr[e] += (double)ar;
            lpi[e] += (double)ai;
        }
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) {
            lpr[e] += __shfl_xor_sync(0xffffffffu, lpr[e], o);
            lpi[e] += __shfl_xor_sync(0xffffffffu, lpi[e], o);
        }
        if (tj == 0 && b < B && logpsi) logpsi[b] = make_float2((float)lpr[e], (float)lpi[e]);
    }
}

// ----------------------------------------------------------------------------------------
// a5 (+ a4, a6): connected amplitudes in product form.
//
// Block tile: TB = 32 WS samples x TC = 16 WC table columns, WC*WS warps.  In a warp the 16 lanes
// lc own 16 consecutive columns and the two half-warps ls own two interleaved sets of 8 sample
// PAIRS; the two samples of a pair ride in the two halves of packed FFMA2 operands.  The sign
// sigma of (sample, column) is never applied arithmetically: shared memory holds, for every
// (j, pair), the four sign variants (+-t_b0, +-t_b1) and each thread reads the variant its two
// signs select (a per-(thread, pair) byte offset computed once per tile).  Per (pair, column, j):
// one 16-byte shared load + 8 packed FMA-pipe instructions = 8 FP32 FMA per (sample, column, j).
//
// Shared memory per stage:  rec [KJ][4 variants][TBP + 2] float4  (TBP = 16 WS pairs; +2 pads the
// variant stride by 8 banks so the <= 8 distinct addresses of a warp read hit distinct banks) and
// tab [KJ][TC] float4 filled by ONE bulk copy (cp.async.bulk, mbarrier completion) per chunk.
// ----------------------------------------------------------------------------------------
struct ElocParams {
    const float4* tp;       // [M_pad][nPairsPad]
    long long nPairsPad;
    const float4* tab;      // [nTiles][M_pad][TC]
    const float4* rho;      // [C_pad]
    const int8_t* spins;    // [B][N]
    long long B;
    int N, M_pad, nTiles;
    DevHam H;
    float2* partial;        // [B][nTiles]
    const int* status;      // nullptr, or the guard word of the series path: run only if (status[0] & 1)
    float2* eloc_out;       // [B] or nullptr: with a single column tile the kernel also adds the diagonal and writes E_loc
};

template <int WC, int WS, int KJ>
struct ElocCfg {
    static constexpr int NW = WC * WS, NT = NW * 32;
    static constexpr int TB = 32 * WS, TBP = 16 * WS, TC = 16 * WC;
    static constexpr int RSTR = TBP + 2;                       // float4 per variant row
    static constexpr int REC_F4 = KJ * 4 * RSTR;               // float4 per stage
    static constexpr int TAB_F4 = KJ * TC;
    static constexpr int STAGE_F4 = REC_F4 + TAB_F4;
    static constexpr int ITEMS = (KJ * TBP + NT - 1) / NT;     // record items per thread per chunk
    static constexpr size_t SMEM = (size_t)2 * STAGE_F4 * 16 + 64;
};

template <int WC, int WS, int KJ>
__global__ void __launch_bounds__(WC * WS * 32, (WC * WS <= 10) ? 2 : 1) eloc_kernel(const ElocParams p) {
    using Cfg = ElocCfg<WC, WS, KJ>;
    constexpr int NT = Cfg::NT, TBP = Cfg::TBP, TC = Cfg::TC, RSTR = Cfg::RSTR;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* const stage0 = reinterpret_cast<float4*>(smem_raw);
    uint64_t* const mbar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)2 * Cfg::STAGE_F4 * 16);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wc = warp % WC, ws = warp / WC;
    const int lc = lane & 15, ls = lane >> 4;
    if (p.status && !(p.status[0] & 1)) return;  // the tensor-core series path passed its guard (nqs_series.cuh)
    const int tile = (int)(blockIdx.x % (unsigned)p.nTiles);  // 1-D grid, column tile fastest
    const long long pair0 = (long long)(blockIdx.x / (unsigned)p.nTiles) * TBP;
    const int c = tile * TC + wc * 16 + lc;
    const int nChunks = p.M_pad / KJ;
    const float4* const tab_tile = p.tab + (long long)tile * p.M_pad * TC;
    constexpr uint32_t TAB_BYTES = Cfg::TAB_F4 * 16;

    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&mbar[0], TAB_BYTES);
        bulk_g2s(stage0 + Cfg::REC_F4, tab_tile, TAB_BYTES, &mbar[0]);
    }

    // a4 (part 1): signs.  sigma = spin at the column's first flip site; u = -sigma t, so the
    // variant bit of a sample is (sigma > 0).  off[r] = float4 offset inside a rec row block.
    const int site = p.H.col_i[c];
    int off[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int pl = ws * 16 + 2 * r + ls;
        const long long bA = 2 * (pair0 + pl), bB = bA + 1;
        const int sA = (bA < p.B) ? (int)p.spins[bA * p.N + site] : 1;
        const int sB = (bB < p.B) ? (int)p.spins[bB * p.N + site] : 1;
        const int v = (sA > 0 ? 1 : 0) + (sB > 0 ? 2 : 0);
        off[r] = v * RSTR + pl;
    }

    // record staging: item = (jj, pl), lanes <-> consecutive pairs
    float4 pre[Cfg::ITEMS];
    auto load_items = [&](int chunk) {
#pragma unroll
        for (int k = 0; k < Cfg::ITEMS; ++k) {
            const int idx = tid + k * NT;
            const int jj = idx / TBP, pl = idx % TBP;
            if (idx < KJ * TBP) pre[k] = p.tp[(long long)(chunk * KJ + jj) * p.nPairsPad + pair0 + pl];
        }
    };
    auto store_items = [&](float4* rec) {
#pragma unroll
        for (int k = 0; k < Cfg::ITEMS; ++k) {
            const int idx = tid + k * NT;
            const int jj = idx / TBP, pl = idx % TBP;
            if (idx < KJ * TBP) {
                const float4 t = pre[k];  // (tr0, tr1, ti0, ti1)
                float4* row = rec + jj * 4 * RSTR + pl;
                row[0 * RSTR] = make_float4(t.x, t.y, t.z, t.w);      // sigma0 < 0, sigma1 < 0 : u = +t
                row[1 * RSTR] = make_float4(-t.x, t.y, -t.z, t.w);    // sigma0 > 0
                row[2 * RSTR] = make_float4(t.x, -t.y, t.z, -t.w);    // sigma1 > 0
                row[3 * RSTR] = make_float4(-t.x, -t.y, -t.z, -t.w);  // both > 0
            }
        }
    };
    load_items(0);
    store_items(stage0);
    __syncthreads();

    float2 Pr[8], Pi[8];
    int exA[8], exB[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        Pr[r] = make_float2(1.f, 1.f);
        Pi[r] = make_float2(0.f, 0.f);
        exA[r] = 0;
        exB[r] = 0;
    }

    for (int chunk = 0; chunk < nChunks; ++chunk) {
        const int s = chunk & 1;
        float4* const rec = stage0 + (size_t)s * Cfg::STAGE_F4;
        const float4* const tabs = rec + Cfg::REC_F4;
        float4* const rec_next = stage0 + (size_t)(s ^ 1) * Cfg::STAGE_F4;
        const bool more = (chunk + 1) < nChunks;
        if (more) {
            load_items(chunk + 1);
            if (tid == 0) {
                fence_proxy_async();  // earlier generic-proxy reads of this buffer vs the async write
                mbar_expect_tx(&mbar[s ^ 1], TAB_BYTES);
                bulk_g2s(rec_next + Cfg::REC_F4, tab_tile + (long long)(chunk + 1) * KJ * TC, TAB_BYTES, &mbar[s ^ 1]);
            }
        }
        mbar_wait(&mbar[s], (chunk >> 1) & 1);

#pragma unroll
        for (int jj = 0; jj < KJ; ++jj) {
            const float4 e = tabs[jj * TC + wc * 16 + lc];  // Cr Ci Sr Si
            const float4* const rrow = rec + jj * 4 * RSTR;
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const float4 u = rrow[off[r]];
                const float2 ur = make_float2(u.x, u.y), ui = make_float2(u.z, u.w);
                float2 rr = __ffma2_rn(ur, bc2(e.z), bc2(e.x));
                rr = __ffma2_rn(ui, bc2(-e.w), rr);
                float2 ri = __ffma2_rn(ur, bc2(e.w), bc2(e.y));
                ri = __ffma2_rn(ui, bc2(e.z), ri);
                float2 nr = __fmul2_rn(Pr[r], rr);
                nr = __ffma2_rn(neg2(Pi[r]), ri, nr);
                float2 ni = __fmul2_rn(Pr[r], ri);
                ni = __ffma2_rn(Pi[r], rr, ni);
                Pr[r] = nr;
                Pi[r] = ni;
            }
        }
        // range safety: pull the exponent out when a running product leaves [2^-40, 2^40]
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const float mA = fmaxf(fabsf(Pr[r].x), fabsf(Pi[r].x));
            const float mB = fmaxf(fabsf(Pr[r].y), fabsf(Pi[r].y));
            if (mA > 1.0995116e12f || (mA < 9.094947e-13f && mA > 0.f)) {
                int ex;
                (void)frexpf(mA, &ex);
                Pr[r].x = ldexpf(Pr[r].x, -ex);
                Pi[r].x = ldexpf(Pi[r].x, -ex);
                exA[r] += ex;
            }
            if (mB > 1.0995116e12f || (mB < 9.094947e-13f && mB > 0.f)) {
                int ex;
                (void)frexpf(mB, &ex);
                Pr[r].y = ldexpf(Pr[r].y, -ex);
                Pi[r].y = ldexpf(Pi[r].y, -ex);
                exB[r] += ex;
            }
        }
        if (more) store_items(rec_next);
        __syncthreads();
    }

    // a4 (part 2) + a6: matrix elements, rho, reduction over the block's columns.  Everything that depends on the
    // column only is fetched once; the per-sample part is branch-free (inline terms) so that the loads of the 16
    // samples a thread owns are in flight together -- on small problems this epilogue is the critical path.
    float2* const accs = reinterpret_cast<float2*>(smem_raw);  // [TB][WC], stages are dead now
    const int g = p.H.col_group[c];
    const float4 rho = p.rho[c];
    const int ck = p.H.col_k[c], cs2 = p.H.col_s2[c], cs3 = p.H.col_s3[c];
    const int pk = p.H.col_p[c], p2 = p.H.col_p2[c], p3 = p.H.col_p3[c];
    const int first = g >= 0 ? p.H.grp_first[g] : 0, count = g >= 0 ? p.H.grp_count[g] : 0;
    bool generic = count > 2;  // inline: at most two terms, none with more than two z factors
    if (p.H.has_zx)
        for (int u = 0; u < count; ++u) generic |= p.H.gt_zx_off[first + u + 1] > p.H.gt_zx_off[first + u];
    int z0a = -1, z1a = -1, z0b = -1, z1b = -1;
    float2 ca = make_float2(0.f, 0.f), cb = ca;
    if (!generic && count >= 1) z0a = p.H.gt_z0[first], z1a = p.H.gt_z1[first], ca = p.H.gt_c[first];
    if (!generic && count >= 2) z0b = p.H.gt_z0[first + 1], z1b = p.H.gt_z1[first + 1], cb = p.H.gt_c[first + 1];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int pl = ws * 16 + 2 * r + ls;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long b = 2 * (pair0 + pl) + h;
            const bool live_b = g >= 0 && b < p.B;
            const int8_t* srow = p.spins + (b < p.B ? b : p.B - 1) * p.N;
            auto spin_or = [&](int z, int dflt) { return z >= 0 ? (int)srow[z] : dflt; };
            const int si = srow[site];
            const bool active = live_b && spin_or(ck, si * pk) * si == pk && spin_or(cs2, si * p2) * si == p2 &&
                                spin_or(cs3, si * p3) * si == p3;
            const float fa = (float)(spin_or(z0a, 1) * spin_or(z1a, 1)), fb = (float)(spin_or(z0b, 1) * spin_or(z1b, 1));
            float2 m = make_float2(fmaf(ca.x, fa, cb.x * fb), fmaf(ca.y, fa, cb.y * fb));
            if (generic && active) m = group_element(p.H, srow, g);
            float cr = 0.f, ci = 0.f;
            if (active && (m.x != 0.f || m.y != 0.f)) {
                const float rr = si > 0 ? rho.x : rho.z, ri = si > 0 ? rho.y : rho.w;
                const float vr = m.x * rr - m.y * ri, vi = m.x * ri + m.y * rr;
                const float pr = h ? Pr[r].y : Pr[r].x, pi = h ? Pi[r].y : Pi[r].x;
                const int ex = h ? exB[r] : exA[r];
                cr = ldexpf(vr * pr - vi * pi, ex);
                ci = ldexpf(vr * pi + vi * pr, ex);
            }
#pragma unroll
            for (int o = 1; o < 16; o <<= 1) {
                cr += __shfl_xor_sync(0xffffffffu, cr, o);
                ci += __shfl_xor_sync(0xffffffffu, ci, o);
            }
            if (lc == 0) accs[(2 * pl + h) * WC + wc] = make_float2(cr, ci);
        }
    }
    __syncthreads();
    for (int sl = tid; sl < Cfg::TB; sl += NT) {
        const long long b = 2 * pair0 + sl;
        if (b < p.B) {
            float sr = 0.f, si = 0.f;
#pragma unroll
            for (int w = 0; w < WC; ++w) {
                sr += accs[sl * WC + w].x;
                si += accs[sl * WC + w].y;
            }
            if (p.eloc_out) {  // single column tile: a6 finishes here (diagonal + off-diagonal sum), no finalize launch
                const float2 d = diagonal_element(p.H, p.spins + b * p.N);
                p.eloc_out[b] = make_float2(d.x + sr, d.y + si);
            } else {
                p.partial[b * p.nTiles + tile] = make_float2(sr, si);
            }
        }
    }
}

// a6: E_loc = diagonal + sum over column tiles of the partial sums (fixed order: deterministic)
__global__ void finalize_kernel(const int8_t* __restrict__ spins, long long B, int N, DevHam H,
                                const float2* __restrict__ partial, int nTiles, float2* __restrict__ eloc,
                                const int* __restrict__ status) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B) return;
    if (status && !(status[0] & 1)) return;  // series_guard_kernel already wrote E_loc
    float2 d = diagonal_element(H, spins + b * N);
    for (int t = 0; t < nTiles; ++t) {
        const float2 v = partial[b * nTiles + t];
        d.x += v.x;
        d.y += v.y;
    }
    eloc[b] = d;
}

// Test/debug: materialise Eq. 39 per flip group (slot 0 = diagonal).
__global__ void enumerate_kernel(const int8_t* __restrict__ spins, long long B, int N, DevHam H,
                                 int8_t* __restrict__ sprime, float2* __restrict__ mel) {
    const long long total = B * (long long)(H.G + 1);
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long b = idx / (H.G + 1);
        const int slot = (int)(idx % (H.G + 1));
        const int8_t* srow = spins + b * N;
        int8_t* out = sprime + idx * N;
        for (int i = 0; i < N; ++i) out[i] = srow[i];
        if (slot == 0) {
            mel[idx] = diagonal_element(H, srow);
        } else {
            const int g = slot - 1;
            const int f0 = H.grp_f0[g], f1 = H.grp_f1[g], f2 = H.grp_f2[g], f3 = H.grp_f3[g];
            out[f0] = (int8_t)(-srow[f0]);
            if (f1 >= 0) out[f1] = (int8_t)(-srow[f1]);
            if (f2 >= 0) out[f2] = (int8_t)(-srow[f2]);
            if (f3 >= 0) out[f3] = (int8_t)(-srow[f3]);
            mel[idx] = group_element(H, srow, g);
        }
    }
}

}  // namespace nqs
