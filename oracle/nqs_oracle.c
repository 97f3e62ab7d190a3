/*
 * oracle/nqs_oracle.c -- float64 CPU oracle for the batched RBM local energy.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under paper_2108_03409_b200/ (the product) may include,
 * link, import or call this file; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs use it.  It shares no code, header, table or helper
 * with the CUDA path.  Plain, slow, written to be checked against the paper by eye.
 *
 * What it computes (citations are /root/reference/PAPER.md line numbers):
 *   log psi(s) = sum_i a_i s_i + sum_j log cosh(b_j + sum_i W_ji s_i)      Eq. 38, :385-390
 *                (index reading Q1 of DESIGN.md: j hidden, i visible, W is [M,N])
 *   E_loc(s)   = sum_s' <s|H|s'> psi(s') / psi(s)                           Eq. 4,  :63-68, :89
 *   H          = sum_t c_t P_t,  P_t a product of Pauli matrices on distinct sites (a "Pauli
 *                string": K slots per term, K = 2 for the five configurations, any K for the
 *                k-site strings of SURVEY.md 8(f) item 4 / PAPER.md:473 "tensor products of
 *                branch-free operators"); its action on a basis configuration is the map of
 *                s -> (s', <s|P_t|s'>) ("branch-free": one non-zero per row).   Eq. 39, :418-426
 *
 * Inputs are the SAME BYTES the GPU gets (int8 spins, complex64 parameters); they are
 * promoted exactly to double.  All arithmetic is double / double complex.
 *
 * Two modes:
 *   definition mode  oracle_local_energy_definition(): Algorithm 1 lines 6-8 (:163-194,
 *       :464-469) literally -- every term in list order, no grouping, s' built explicitly,
 *       log psi(s') recomputed from scratch with log cosh = clog(ccosh(.)) from libm.
 *       This is the parity authority.
 *   fast mode        oracle_local_energy_fast(): same float64 arithmetic, but terms are grouped
 *       by flip set and theta' = theta - 2 sum_{i in F} W_:,i s_i is used with differences of
 *       a stable log cosh (formula F1 below).  Pinned to definition mode (pin P8) and used for
 *       full-batch parity and as the timed CPU baseline.
 *
 * Parity pins: see tests/test_oracle_pins.py (P1 dense H brute force, P2 Eq. 2-3 identity,
 * P3 zero parameters closed form, P4 product eigenstate, P5 singlet, P6 spin-flip symmetry,
 * P7 Pfeuty closed form for the dense-H builder, P8 definition<->fast, P9 log cosh special
 * cases; PF1 log-derivatives against finite differences of log psi, PF2 force vector against
 * finite differences of the dense <H>, PF3 mean / variance against numpy and Eq. 3; PM1 the
 * Metropolis rule against the dense psi, PM2 its stationary distribution |psi|^2).
 * No function here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

enum { P_I = 0, P_X = 1, P_Y = 2, P_Z = 3 };

/* complex64 (interleaved float re, im) element k -> double complex, exact promotion */
static inline cplx c64(const float *p, int64_t k) { return (double)p[2 * k] + I * (double)p[2 * k + 1]; }

/* ---------------------------------------------------------------------------------------
 * log cosh
 * ------------------------------------------------------------------------------------- */

/* Definition: the principal complex logarithm of cosh z, straight from libm. */
static inline cplx lncosh_def(cplx z) { return clog(ccosh(z)); }

/* F1 (reading Q6): z = x + iy, sgn = sign(x) (+1 at 0), u = |x|, yt = sgn*y,
 * q = exp(-2u), D = 1 + 2 q cos 2yt + q^2 = |1 + q e^{2 i yt}|^2.  Since cosh z = cosh(sgn z)
 * = e^{u + i yt} (1 + q e^{-2 i yt}) / 2 ... written out:
 *   Re = u - ln 2 + (1/2) log D,   Im = yt + atan2(-q sin 2yt, 1 + q cos 2yt).
 * Never overflows.  Im is an unwrapped phase: equal to the principal value when |y| < pi/2,
 * else it differs by a multiple of 2 pi. */
static inline cplx lncosh_stable(cplx z) {
    double x = creal(z), y = cimag(z);
    double sgn = (x < 0.0) ? -1.0 : 1.0;
    double u = fabs(x), yt = sgn * y;
    double q = exp(-2.0 * u);
    double c = cos(2.0 * yt), s = sin(2.0 * yt);
    double D = 1.0 + 2.0 * q * c + q * q;
    return (u - M_LN2 + 0.5 * log(D)) + I * (yt + atan2(-q * s, 1.0 + q * c));
}

/* exported pointwise for pin P9: mode 0 = definition, 1 = F1 */
void oracle_lncosh(const double *z_re_im, int64_t n, int mode, double *out_re_im) {
    for (int64_t k = 0; k < n; ++k) {
        cplx z = z_re_im[2 * k] + I * z_re_im[2 * k + 1];
        cplx r = mode ? lncosh_stable(z) : lncosh_def(z);
        out_re_im[2 * k] = creal(r);
        out_re_im[2 * k + 1] = cimag(r);
    }
}

/* ---------------------------------------------------------------------------------------
 * log psi, Eq. 38
 * ------------------------------------------------------------------------------------- */
static cplx log_psi_one(const int8_t *s, int N, int M, const float *a, const float *b, const float *W,
                        int stable) {
    cplx acc = 0.0;
    for (int i = 0; i < N; ++i) acc += c64(a, i) * (double)s[i];
    for (int j = 0; j < M; ++j) {
        cplx theta = c64(b, j);
        for (int i = 0; i < N; ++i) theta += c64(W, (int64_t)j * N + i) * (double)s[i];
        acc += stable ? lncosh_stable(theta) : lncosh_def(theta);
    }
    return acc;
}

/* spins [B,N] int8, a [N], b [M], W [M,N] complex64; out [B] complex128 (re, im doubles).
 * mode 0: log cosh by definition; mode 1: F1. */
void oracle_log_psi(const int8_t *spins, int64_t B, int N, int M, const float *a, const float *b,
                    const float *W, int mode, double *out_logpsi) {
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < B; ++n) {
        cplx lp = log_psi_one(spins + n * N, N, M, a, b, W, mode);
        out_logpsi[2 * n] = creal(lp);
        out_logpsi[2 * n + 1] = cimag(lp);
    }
}

/* ---------------------------------------------------------------------------------------
 * matrix element of one Pauli on one site, row convention (reading Q3):
 *   <s|X_k|s'> = 1,  <s|Y_k|s'> = -i s_k  (s' = s with site k flipped),
 *   <s|Z_k|s>  = s_k, identity = 1.   s_k is the spin of the ROW configuration s.
 * ------------------------------------------------------------------------------------- */
static inline cplx pauli_factor(int p, int sk, int *flips) {
    switch (p) {
    case P_X: *flips = 1; return 1.0;
    case P_Y: *flips = 1; return -I * (double)sk;
    case P_Z: *flips = 0; return (double)sk;
    default:  *flips = 0; return 1.0;
    }
}

/* ---------------------------------------------------------------------------------------
 * definition mode: Eq. 4 + Eq. 39 + Eq. 38, term by term (Algorithm 1 lines 6-8)
 * ------------------------------------------------------------------------------------- */
void oracle_local_energy_definition(const int8_t *spins, int64_t B, int N, int M, const float *a,
                                    const float *b, const float *W, int T, int K, const int32_t *sites,
                                    const uint8_t *paulis, const float *coeffs, double *out_eloc,
                                    double *out_logpsi) { /* sites, paulis: [T,K] */
#pragma omp parallel
    {
        int8_t *sp = (int8_t *)malloc((size_t)N);
#pragma omp for schedule(dynamic, 1)
        for (int64_t n = 0; n < B; ++n) {
            const int8_t *s = spins + n * N;
            cplx lp = log_psi_one(s, N, M, a, b, W, 0);
            cplx E = 0.0;
            for (int t = 0; t < T; ++t) {
                cplx m = c64(coeffs, t);
                memcpy(sp, s, (size_t)N);
                for (int k = 0; k < K; ++k) {
                    int site = sites[(int64_t)K * t + k];
                    if (site < 0) continue; /* unused slot */
                    int flips = 0;
                    m *= pauli_factor(paulis[(int64_t)K * t + k], s[site], &flips);
                    if (flips) sp[site] = (int8_t)(-sp[site]);
                }
                if (m == 0.0) continue; /* "non-zero matrix elements", :458 (reading Q5) */
                cplx lpp = log_psi_one(sp, N, M, a, b, W, 0);
                E += m * cexp(lpp - lp);
            }
            out_eloc[2 * n] = creal(E);
            out_eloc[2 * n + 1] = cimag(E);
            if (out_logpsi) {
                out_logpsi[2 * n] = creal(lp);
                out_logpsi[2 * n + 1] = cimag(lp);
            }
        }
        free(sp);
    }
}

/* ---------------------------------------------------------------------------------------
 * fast mode: flip grouping + low-rank theta update, same float64 arithmetic
 * ------------------------------------------------------------------------------------- */
#define ORACLE_MAX_SLOTS 16
typedef struct { int nf; int f[ORACLE_MAX_SLOTS]; int first, count; } group_t; /* sorted flip set; nf = 0: diagonal */

/* the flip set of term t: the sites carrying X or Y, sorted */
static int key_of(const int32_t *sites, const uint8_t *paulis, int K, int t, int *f) {
    int nf = 0;
    for (int k = 0; k < K; ++k) {
        int site = sites[(int64_t)K * t + k];
        int p = paulis[(int64_t)K * t + k];
        if (site >= 0 && (p == P_X || p == P_Y)) f[nf++] = site;
    }
    for (int i = 1; i < nf; ++i) /* insertion sort */
        for (int j = i; j > 0 && f[j - 1] > f[j]; --j) { int tmp = f[j]; f[j] = f[j - 1]; f[j - 1] = tmp; }
    return nf;
}

void oracle_local_energy_fast(const int8_t *spins, int64_t B, int N, int M, const float *a,
                              const float *b, const float *W, int T, int K, const int32_t *sites,
                              const uint8_t *paulis, const float *coeffs, double *out_eloc,
                              double *out_logpsi) { /* sites, paulis: [T,K], K <= ORACLE_MAX_SLOTS */
    /* group terms by flip set: order[] lists term ids group by group (O(T^2), T is small) */
    int *order = (int *)malloc(sizeof(int) * (size_t)(T > 0 ? T : 1));
    group_t *groups = (group_t *)malloc(sizeof(group_t) * (size_t)(T > 0 ? T : 1));
    char *done = (char *)calloc((size_t)(T > 0 ? T : 1), 1);
    int G = 0, pos = 0;
    for (int t = 0; t < T; ++t) {
        if (done[t]) continue;
        groups[G].nf = key_of(sites, paulis, K, t, groups[G].f);
        groups[G].first = pos; groups[G].count = 0;
        for (int u = t; u < T; ++u) {
            int g[ORACLE_MAX_SLOTS];
            if (done[u]) continue;
            int ng = key_of(sites, paulis, K, u, g);
            if (ng == groups[G].nf && memcmp(g, groups[G].f, sizeof(int) * (size_t)ng) == 0) {
                order[pos++] = u; done[u] = 1; groups[G].count++;
            }
        }
        ++G;
    }

#pragma omp parallel
    {
        cplx *theta = (cplx *)malloc(sizeof(cplx) * (size_t)(M > 0 ? M : 1));
        cplx *L = (cplx *)malloc(sizeof(cplx) * (size_t)(M > 0 ? M : 1));
#pragma omp for schedule(dynamic, 1)
        for (int64_t n = 0; n < B; ++n) {
            const int8_t *s = spins + n * N;
            cplx lp = 0.0;
            for (int i = 0; i < N; ++i) lp += c64(a, i) * (double)s[i];
            for (int j = 0; j < M; ++j) {
                cplx th = c64(b, j);
                for (int i = 0; i < N; ++i) th += c64(W, (int64_t)j * N + i) * (double)s[i];
                theta[j] = th;
                L[j] = lncosh_stable(th);
                lp += L[j];
            }
            cplx E = 0.0;
            for (int g = 0; g < G; ++g) {
                /* summed matrix element of the group's terms (they all reach the same s') */
                cplx m = 0.0;
                for (int q = 0; q < groups[g].count; ++q) {
                    int t = order[groups[g].first + q];
                    cplx mt = c64(coeffs, t);
                    for (int k = 0; k < K; ++k) {
                        int site = sites[(int64_t)K * t + k];
                        if (site < 0) continue;
                        int flips;
                        mt *= pauli_factor(paulis[(int64_t)K * t + k], s[site], &flips);
                    }
                    m += mt;
                }
                if (groups[g].nf == 0) { E += m; continue; } /* diagonal: s' = s, ratio 1 */
                if (m == 0.0) continue;
                cplx dlog = 0.0;
                for (int q = 0; q < groups[g].nf; ++q) {
                    int f = groups[g].f[q];
                    dlog += -2.0 * c64(a, f) * (double)s[f];
                }
                for (int j = 0; j < M; ++j) {
                    cplx thp = theta[j];
                    for (int q = 0; q < groups[g].nf; ++q) {
                        int f = groups[g].f[q];
                        thp -= 2.0 * c64(W, (int64_t)j * N + f) * (double)s[f];
                    }
                    dlog += lncosh_stable(thp) - L[j];
                }
                E += m * cexp(dlog);
            }
            out_eloc[2 * n] = creal(E);
            out_eloc[2 * n + 1] = cimag(E);
            if (out_logpsi) {
                out_logpsi[2 * n] = creal(lp);
                out_logpsi[2 * n + 1] = cimag(lp);
            }
        }
        free(theta);
        free(L);
    }
    free(order);
    free(groups);
    free(done);
}

/* ---------------------------------------------------------------------------------------
 * Eq. 39 as data: connected configurations and matrix elements, term by term (no grouping).
 * sprime [B,T,N] int8, mel [B,T] complex128.  Used to check the GPU enumerator.
 * ------------------------------------------------------------------------------------- */
void oracle_connected(const int8_t *spins, int64_t B, int N, int T, int K, const int32_t *sites,
                      const uint8_t *paulis, const float *coeffs, int8_t *sprime, double *mel) {
    for (int64_t n = 0; n < B; ++n) {
        const int8_t *s = spins + n * N;
        for (int t = 0; t < T; ++t) {
            int8_t *sp = sprime + ((n * T) + t) * N;
            memcpy(sp, s, (size_t)N);
            cplx m = c64(coeffs, t);
            for (int k = 0; k < K; ++k) {
                int site = sites[(int64_t)K * t + k];
                if (site < 0) continue;
                int flips = 0;
                m *= pauli_factor(paulis[(int64_t)K * t + k], s[site], &flips);
                if (flips) sp[site] = (int8_t)(-sp[site]);
            }
            mel[2 * (n * T + t)] = creal(m);
            mel[2 * (n * T + t) + 1] = cimag(m);
        }
    }
}

/* ---------------------------------------------------------------------------------------
 * batch statistics, logarithmic derivatives, force vector.
 * Parameter order k = 0..K-1, K = N + M + M*N:  a_i (k = i), b_j (k = N + j),
 * W_ji (k = N + M + j*N + i).  Weights w_b >= 0 are optional (NULL = uniform): with
 * w_b = p(s_b) over the full basis they turn the sample mean of Eq. 5 into the exact
 * expectation of Eq. 3.  They are normalised by their own sum.
 * ------------------------------------------------------------------------------------- */

/* Eq. 5 (:70-73) / Eq. 3: mean = sum_b w_b x_b / sum_b w_b and the variance
 * <<|x - mean|^2>> (:511-515 get_global_mean / get_global_variance).
 * x [B] complex128; out = {Re mean, Im mean, variance, sum of weights}. */
void oracle_mean_variance(const double *x_re_im, const double *w, int64_t B, double out[4]) {
    double sw = 0.0;
    cplx sx = 0.0;
    for (int64_t n = 0; n < B; ++n) {
        const double wn = w ? w[n] : 1.0;
        sw += wn;
        sx += wn * (x_re_im[2 * n] + I * x_re_im[2 * n + 1]);
    }
    const cplx mean = sx / sw;
    double var = 0.0;
    for (int64_t n = 0; n < B; ++n) {
        const double wn = w ? w[n] : 1.0;
        const cplx d = (x_re_im[2 * n] + I * x_re_im[2 * n + 1]) - mean;
        var += wn * (creal(d) * creal(d) + cimag(d) * cimag(d));
    }
    out[0] = creal(mean);
    out[1] = cimag(mean);
    out[2] = var / sw;
    out[3] = sw;
}

/* Eq. 8 (:93): O_k(s) = d log psi(s) / d theta_k for the RBM of Eq. 38 (complex derivative,
 * holomorphic ansatz :126, :299):  O_{a_i} = s_i,  O_{b_j} = tanh(theta_j),
 * O_{W_ji} = tanh(theta_j) s_i,  theta_j = b_j + sum_i W_ji s_i.  tanh from libm (ctanh). */
static void log_derivatives_one(const int8_t *s, int N, int M, const float *b, const float *W, cplx *O) {
    for (int i = 0; i < N; ++i) O[i] = (double)s[i];
    for (int j = 0; j < M; ++j) {
        cplx theta = c64(b, j);
        for (int i = 0; i < N; ++i) theta += c64(W, (int64_t)j * N + i) * (double)s[i];
        const cplx t = ctanh(theta);
        O[N + j] = t;
        for (int i = 0; i < N; ++i) O[N + M + (int64_t)j * N + i] = t * (double)s[i];
    }
}

/* out_O [B,K] complex128 (small inputs only: B*K*16 bytes) */
void oracle_log_derivatives(const int8_t *spins, int64_t B, int N, int M, const float *a, const float *b,
                            const float *W, double *out_O) {
    (void)a;
    const int64_t K = (int64_t)N + M + (int64_t)M * N;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < B; ++n) log_derivatives_one(spins + n * N, N, M, b, W, (cplx *)(out_O + 2 * n * K));
}

/* Eq. 16 (:134-138), Eq. 7 (:81-89): F_k = <<E_loc O_k^*>>^c = <<O_k^* E_loc>> - <<O_k^*>> <<E_loc>>,
 * the connected correlation written out as its two terms.  eloc [B] complex128 is an INPUT
 * (any estimator values).  out_F [K] complex128.  Never materialises O [B,K]. */
void oracle_forces(const int8_t *spins, int64_t B, int N, int M, const float *a, const float *b, const float *W,
                   const double *eloc_re_im, const double *w, double *out_F) {
    (void)a;
    const int64_t K = (int64_t)N + M + (int64_t)M * N;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    cplx *OE = calloc((size_t)K * nthreads, sizeof(cplx)); /* per-thread sum_b w_b O_k^* E_b */
    cplx *Oc = calloc((size_t)K * nthreads, sizeof(cplx)); /* per-thread sum_b w_b O_k^*     */
    cplx *Ebar = calloc((size_t)nthreads, sizeof(cplx));
    double *Wsum = calloc((size_t)nthreads, sizeof(double));
#pragma omp parallel
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        cplx *O = malloc((size_t)K * sizeof(cplx));
        cplx *oe = OE + (size_t)tid * K, *oc = Oc + (size_t)tid * K;
#pragma omp for schedule(static)
        for (int64_t n = 0; n < B; ++n) {
            const double wn = w ? w[n] : 1.0;
            const cplx E = eloc_re_im[2 * n] + I * eloc_re_im[2 * n + 1];
            log_derivatives_one(spins + n * N, N, M, b, W, O);
            for (int64_t k = 0; k < K; ++k) {
                oe[k] += wn * conj(O[k]) * E;
                oc[k] += wn * conj(O[k]);
            }
            Ebar[tid] += wn * E;
            Wsum[tid] += wn;
        }
        free(O);
    }
    cplx E = 0.0;
    double sw = 0.0;
    for (int t = 0; t < nthreads; ++t) {
        E += Ebar[t];
        sw += Wsum[t];
    }
    E /= sw;
    for (int64_t k = 0; k < K; ++k) {
        cplx oe = 0.0, oc = 0.0;
        for (int t = 0; t < nthreads; ++t) {
            oe += OE[(size_t)t * K + k];
            oc += Oc[(size_t)t * K + k];
        }
        const cplx F = oe / sw - (oc / sw) * E;
        out_F[2 * k] = creal(F);
        out_F[2 * k + 1] = cimag(F);
    }
    free(OE);
    free(Oc);
    free(Ebar);
    free(Wsum);
}

/* ---------------------------------------------------------------------------------------
 * Metropolis sampling of p(s) = |psi(s)|^2 / <psi|psi> with single-spin-flip
 * proposals, many independent chains (PAPER.md:70 Metropolis-Hastings; :341 one sweep = one
 * proposal per degree of freedom; :490-494 chains run in sync).  The random numbers are INPUTS
 * (proposal site and a uniform number per chain and step), so this function is deterministic.
 *
 * For chain c and step t:  s' = s with site sites[t,c] flipped;  the move is accepted iff
 *     u[t,c] < |psi(s') / psi(s)|^2          (Metropolis: min(1, p(s')/p(s)), symmetric proposal)
 * evaluated in logarithms, log u < 2 Re(log psi(s') - log psi(s)), with log psi(s') recomputed FROM
 * SCRATCH by Eq. 38 at every proposal (no incremental update).  u = 0 always accepts.
 *
 * spins [C,N] int8 in/out; sites [S,C] int32; u [S,C] float32 in [0,1); accepted [C] int32 out;
 * min_margin [C] float64 out = min over the steps of |2 Re dlogpsi - log u|: how far the closest
 * decision of the chain was from a tie (a float32 implementation can only be asked to reproduce
 * chains whose margin exceeds its rounding error).
 * decisions [S,C] uint8 out or NULL: 1 = the proposal of step t was accepted; margins [S,C] float64 out or
 * NULL: the same |2 Re dlogpsi - log u| per step (the trace behind min_margin: where a float32 chain and
 * this one first part ways, the margin AT THAT STEP says whether the parting was a legitimate near-tie).
 * ------------------------------------------------------------------------------------- */
void oracle_metropolis(int8_t *spins, int64_t C, int N, int M, const float *a, const float *b, const float *W,
                       int S, const int32_t *sites, const float *u, int32_t *accepted, double *min_margin,
                       uint8_t *decisions, double *margins) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t c = 0; c < C; ++c) {
        int8_t *s = spins + c * N;
        cplx lp = log_psi_one(s, N, M, a, b, W, 1);
        int acc = 0;
        double mm = INFINITY;
        for (int t = 0; t < S; ++t) {
            const int site = sites[(int64_t)t * C + c];
            const double ut = (double)u[(int64_t)t * C + c];
            s[site] = (int8_t)(-s[site]);
            const cplx lp_new = log_psi_one(s, N, M, a, b, W, 1);
            const double log_ratio = 2.0 * creal(lp_new - lp);
            const double log_u = ut > 0.0 ? log(ut) : -INFINITY;
            const double margin = fabs(log_ratio - log_u);
            if (margin < mm) mm = margin;
            if (margins) margins[(int64_t)t * C + c] = margin;
            if (decisions) decisions[(int64_t)t * C + c] = (uint8_t)(log_u < log_ratio);
            if (log_u < log_ratio) {
                lp = lp_new;
                ++acc;
            } else {
                s[site] = (int8_t)(-s[site]);
            }
        }
        accepted[c] = acc;
        min_margin[c] = mm;
    }
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
