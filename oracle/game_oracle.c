/*
 * game_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU oracle for the GAME hot path of
 * arXiv:1211.5481 ("Genetic Algorithm Modeling with GPU Parallel Computing
 * Technology"): population fitness over a knowledge base + one GA generation.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant generator with paper_1211_5481_b200/csrc (the CUDA
 * path); neither side includes or imports the other.
 *
 * Every function cites the passage it follows: "PAPER.md:<line>" is the paper
 * text, "SURVEY §8(c) R<n>" is the reading of the paper fixed in SURVEY.md /
 * DESIGN.md where the paper is silent (DESIGN.md lists every such reading).
 *
 * Arithmetic: fitness in IEEE binary64 on the (double) of the float32 inputs,
 * loops in the order the definition states (no blocking, no reordering).  The
 * GA operators are integer work plus a handful of individually rounded
 * binary32 operations (no FMA contraction: build with -ffp-contract=off, no
 * -ffast-math), so that they can be reproduced bit for bit.
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, brute force, library
 * routines, Random123 known-answer vectors, GA invariants).  Unpinned: the
 * *quality* of the GA on the paper's NGC1399 data set --
 * the data set is not available; out of scope.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define EXP_CHEBYSHEV 0
#define EXP_TRIG 1
#define ACT_IDENTITY 0
#define ACT_SIGMOID 1
#define ACT_TANH 2

/* ---- shapes -------------------------------------------------------------
 * PAPER.md:75-77 eq.(5) gives NUM_genes = B*d+1 for coefficients shared by all
 * features; BASELINE.json fixes per-feature coefficients (DESIGN.md reading
 * D1): G = N*d+1 (Chebyshev, B=1) or N*2d+1 (polytrigo, B=2).
 */
int oracle_num_genes(int N, int d, int family)
{
    int expansion = family & 0xff;
    int shared = (family >> 16) & 1;    /* PAPER.md:52-55 eq.(2) literally: coefficients shared by all features */
    if (N < 1 || d < 1 || (family >> 17) != 0) return -1;
    if (expansion == EXP_CHEBYSHEV) return (shared ? 1 : N) * d + 1;
    if (expansion == EXP_TRIG) return (shared ? 1 : N) * 2 * d + 1;
    return -1;
}

/* PAPER.md:71-77 eq.(4),(5): the paper's own shape rule (shared coefficients).
 * Used only as a pin of the worked example PAPER.md:84-89 (N=11,d=3,B=2 ->
 * 23 chromosomes x 7 genes). */
void oracle_paper_shapes(int N, int d, int B, int *num_chromosomes, int *num_genes)
{
    *num_chromosomes = B * N + 1;
    *num_genes = B * d + 1;
}

/* ---- expansion phi(x)  (eq.(1), 79-82 eq.(6))
 * phi[0] = 1 (the a_0 of eq.(2)).
 * Chebyshev: phi[1+i*d+(j-1)] = T_j(x_i), recurrence T_0=1, T_1=x,
 *            T_{j+1} = 2x T_j - T_{j-1}.
 * Trig:      phi[1+i*2K+(k-1)] = cos(k x_i), phi[1+i*2K+K+(k-1)] = sin(k x_i),
 *            k=1..K, per-feature block [cos 1..K, sin 1..K] mirroring the
 *            paper's gene order [a_1..a_3, b_1..b_3]; libm.
 */
void oracle_expand(int N, int d, int family, const float *x, double *phi)
{
    int expansion = family & 0xff;
    if ((family >> 16) & 1) {
        /* Shared coefficients, the paper's own form (eq.(2), 75-77 eq.(5), 84-89 eq.(7)):
         * Out = a_0 + sum_j a_j sum_i g_j(f_i), so the expansion term of gene j is the SUM over the features --
         * the per-pattern sums of cosines and sines that the paper precomputes once.
         * Gene order [a_0, a_1..a_d] (Chebyshev) or [a_0, a_1..a_d, b_1..b_d] (trig). */
        int G = oracle_num_genes(N, d, family);
        phi[0] = 1.0;
        for (int g = 1; g < G; ++g) phi[g] = 0.0;
        for (int i = 0; i < N; ++i) {
            double xi = (double)x[i];
            if (expansion == EXP_CHEBYSHEV) {
                double tjm1 = 1.0, tj = xi;
                for (int j = 1; j <= d; ++j) {
                    phi[j] += tj;
                    double tn = 2.0 * xi * tj - tjm1;
                    tjm1 = tj;
                    tj = tn;
                }
            } else {
                for (int k = 1; k <= d; ++k) {
                    phi[k] += cos((double)k * xi);
                    phi[d + k] += sin((double)k * xi);
                }
            }
        }
        return;
    }
    phi[0] = 1.0;
    if (expansion == EXP_CHEBYSHEV) {
        for (int i = 0; i < N; ++i) {
            double xi = (double)x[i];
            double tjm1 = 1.0, tj = xi;
            for (int j = 1; j <= d; ++j) {
                phi[1 + i * d + (j - 1)] = tj;
                double tn = 2.0 * xi * tj - tjm1;
                tjm1 = tj;
                tj = tn;
            }
        }
    } else {
        int K = d;
        for (int i = 0; i < N; ++i) {
            double xi = (double)x[i];
            for (int k = 1; k <= K; ++k) {
                phi[1 + i * 2 * K + (k - 1)] = cos((double)k * xi);
                phi[1 + i * 2 * K + K + (k - 1)] = sin((double)k * xi);
            }
        }
    }
}

static double activation(int act, double z)
{
    if (act == ACT_SIGMOID) return 1.0 / (1.0 + exp(-z));
    if (act == ACT_TANH) return tanh(z);
    return z;
}

/* ---- model output of one chromosome on one pattern
 * PAPER.md:52-55 eq.(2) (with per-feature coefficients, D1) + activation (D2). */
double oracle_output(int N, int d, int family, const float *x, const float *w)
{
    int G = oracle_num_genes(N, d, family);
    double *phi = (double *)malloc(sizeof(double) * (size_t)G);
    oracle_expand(N, d, family, x, phi);
    double z = 0.0;
    for (int g = 0; g < G; ++g) z += (double)w[g] * phi[g];
    free(phi);
    return activation((family >> 8) & 0xff, z);
}

/* ---- fitness  (eq.(3): E_k=(t_k-Out)^2, MSE)
 * F[m] = (1/P) sum_p (act(sum_g W[m][g] phi_g(x_p)) - t_p)^2, g ascending,
 * p ascending, all in double.  Lower is better (D4).
 * Returns the un-normalised sum in SSE (if not NULL) and the mean in F.
 */
int oracle_eval_fitness(int64_t P, int N, int d, int M, int family,
                        const float *X, const float *t, const float *W,
                        double *F, double *SSE)
{
    int G = oracle_num_genes(N, d, family);
    int act = (family >> 8) & 0xff;
    if (G < 0 || P < 1 || M < 1 || act > ACT_TANH) return -1;
    double *phi = (double *)malloc(sizeof(double) * (size_t)G);
    double *S = (double *)calloc((size_t)M, sizeof(double));
    if (!phi || !S) { free(phi); free(S); return -2; }
    for (int64_t p = 0; p < P; ++p) {
        oracle_expand(N, d, family, X + p * N, phi);
        double tp = (double)t[p];
        for (int m = 0; m < M; ++m) {
            const float *w = W + (size_t)m * G;
            double z = 0.0;
            for (int g = 0; g < G; ++g) z += (double)w[g] * phi[g];
            double e = activation(act, z) - tp;
            S[m] += e * e;
        }
    }
    for (int m = 0; m < M; ++m) {
        if (SSE) SSE[m] = S[m];
        F[m] = S[m] / (double)P;
    }
    free(phi);
    free(S);
    return 0;
}

/* ---- Philox4x32-10  (Salmon, Moraes, Dror, Shaw, SC'11)
 * PAPER.md:101 offloads random-chromosome generation to the GPU in bulk; the
 * build replaces the pool by a counter-based generator (BASELINE.json).
 */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { TAG_INIT = 0, TAG_SELECT = 1, TAG_CROSS = 2, TAG_MUTATE = 3 };

/* counter = (index, chromosome, generation, tag), key = (seed lo, seed hi). R4 */
static void draw(uint64_t seed, uint32_t index, uint32_t chrom, uint32_t gen, uint32_t tag,
                 uint32_t out[4])
{
    uint32_t ctr[4] = { index, chrom, gen, tag };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    oracle_philox4x32_10(ctr, key, out);
}

/* R4 integer maps */
uint32_t oracle_index(uint32_t w, uint32_t n) { return (uint32_t)(((uint64_t)w * n) >> 32); }

uint64_t oracle_bernoulli_threshold(double p)
{
    if (!(p > 0.0)) return 0;
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)floor(p * 4294967296.0);
}

/* ---- deterministic N(0,1)
 * Box-Muller on 23+26 bits with Taylor-series log / sin / cos; only binary32
 * + - * / sqrt, each rounded once.  -2 ln u1 and the cosine are exposed for
 * the accuracy pins.
 */
float oracle_neg2ln_u1(uint32_t a)
{
    float u1 = (float)((a >> 9) + 1u) * 0x1p-23f;      /* (0,1], exact */
    uint32_t bits;
    memcpy(&bits, &u1, 4);
    int e = (int)(bits >> 23) - 127;
    uint32_t fb = (bits & 0x007FFFFFu) | 0x3F800000u;
    float f;
    memcpy(&f, &fb, 4);                                 /* [1,2) */
    if (f > 0x1.6a09e6p+0f) { f = f * 0.5f; e += 1; }  /* (0.7071, 1.4142] */
    float num = f - 1.0f;
    float den = f + 1.0f;
    float s = num / den;
    float s2 = s * s;
    float p = 0x1.c71c72p-4f;                           /* 1/9 */
    p = p * s2; p = p + 0x1.24924ap-3f;                 /* 1/7 */
    p = p * s2; p = p + 0x1.99999ap-3f;                 /* 1/5 */
    p = p * s2; p = p + 0x1.555556p-2f;                 /* 1/3 */
    p = p * s2; p = p + 1.0f;
    float el = (float)e * 0x1.62e430p-1f;               /* e * ln 2 */
    float two_s = 2.0f * s;
    float sp = two_s * p;
    float ln = el + sp;
    return -2.0f * ln;
}

/* cos((q + frac) * pi/2) with q = b>>30 and frac = ((b>>6) & 0xFFFFFF) / 2^24 */
float oracle_cos_angle(uint32_t b)
{
    uint32_t q = b >> 30;
    float frac = (float)((b >> 6) & 0xFFFFFFu) * 0x1p-24f;
    float x = frac * 0x1.921fb6p+0f;                    /* * pi/2 */
    float x2 = x * x;
    float p = -0x1.93974ap-37f;                         /* -1/14! */
    p = p * x2; p = p + 0x1.1eed8ep-29f;                /*  1/12! */
    p = p * x2; p = p - 0x1.27e4fcp-22f;                /* -1/10! */
    p = p * x2; p = p + 0x1.a01a02p-16f;                /*  1/8!  */
    p = p * x2; p = p - 0x1.6c16c2p-10f;                /* -1/6!  */
    p = p * x2; p = p + 0x1.555556p-5f;                 /*  1/4!  */
    p = p * x2; p = p - 0.5f;
    p = p * x2; p = p + 1.0f;
    float cosx = p;
    float r = 0x1.612462p-33f;                          /*  1/13! */
    r = r * x2; r = r - 0x1.ae6456p-26f;                /* -1/11! */
    r = r * x2; r = r + 0x1.71de3ap-19f;                /*  1/9!  */
    r = r * x2; r = r - 0x1.a01a02p-13f;                /* -1/7!  */
    r = r * x2; r = r + 0x1.111112p-7f;                 /*  1/5!  */
    r = r * x2; r = r - 0x1.555556p-3f;                 /* -1/3!  */
    r = r * x2; r = r + 1.0f;
    float sinx = x * r;
    if (q == 0) return cosx;
    if (q == 1) return -sinx;
    if (q == 2) return -cosx;
    return sinx;
}

float oracle_gauss(uint32_t a, uint32_t b)
{
    float t = oracle_neg2ln_u1(a);
    float r = sqrtf(t);
    float c = oracle_cos_angle(b);
    return r * c;
}

/* ---- population init  (PAPER.md:66,89 genes random in [-1,+1])
 * gene g of chromosome m: call counter (g>>2, m, 0, TAG_INIT), word g&3,
 * w = float(word>>8) * 2^-23 - 1  in [-1,1), exact.
 */
void oracle_init_population(int M, int G, uint64_t seed, float *W)
{
    for (int m = 0; m < M; ++m)
        for (int g = 0; g < G; ++g) {
            uint32_t r[4];
            draw(seed, (uint32_t)(g >> 2), (uint32_t)m, 0u, TAG_INIT, r);
            W[(size_t)m * G + g] = (float)(r[g & 3] >> 8) * 0x1p-23f - 1.0f;
        }
}

/* ---- order on chromosomes  (R7.1): a < b iff key(F[a]) < key(F[b]) or
 * (equal and a < b); key(NaN) = +inf.  Lower fitness (MSE) is better (D4). */
static float fit_key(float f) { return isnan(f) ? INFINITY : f; }

static int precedes(const float *F, int a, int b)
{
    float ka = fit_key(F[a]), kb = fit_key(F[b]);
    if (ka < kb) return 1;
    if (ka > kb) return 0;
    return a < b;
}

int oracle_best_index(int M, const float *F)
{
    int best = 0;
    for (int m = 1; m < M; ++m)
        if (precedes(F, m, best)) best = m;
    return best;
}

/* ---- one GA generation  ("crossover, genetic
 * mutation, roulette/ranking, elitism", PAPER.md:134-136 rates and elitism;
 * operators defined by BASELINE.json: tournament, single-point, Gaussian).
 */
int oracle_step(int M, int G, int E, int k, double p_cross, double p_mut, float sigma,
                uint64_t seed, uint32_t gen, const float *W, const float *F, float *Wnext)
{
    if (M < 1 || G < 1 || E < 0 || E >= M || k < 1) return -1;
    /* 1. elitism: the E first chromosomes in the order, copied unchanged */
    char *taken = (char *)calloc((size_t)M, 1);
    if (!taken) return -2;
    for (int s = 0; s < E; ++s) {
        int best = -1;
        for (int m = 0; m < M; ++m) {
            if (taken[m]) continue;
            if (best < 0 || precedes(F, m, best)) best = m;
        }
        taken[best] = 1;
        memcpy(Wnext + (size_t)s * G, W + (size_t)best * G, sizeof(float) * (size_t)G);
    }
    free(taken);
    uint64_t Tc = oracle_bernoulli_threshold(p_cross);
    uint64_t Tm = oracle_bernoulli_threshold(p_mut);
    for (int c = E; c < M; ++c) {
        /* 2. tournaments: entrants 0..k-1 -> parent A, k..2k-1 -> parent B */
        int parent[2] = { -1, -1 };
        for (int e = 0; e < 2 * k; ++e) {
            uint32_t r[4];
            draw(seed, (uint32_t)(e >> 2), (uint32_t)c, gen, TAG_SELECT, r);
            int idx = (int)oracle_index(r[e & 3], (uint32_t)M);
            int side = e < k ? 0 : 1;
            if (parent[side] < 0 || precedes(F, idx, parent[side])) parent[side] = idx;
        }
        const float *A = W + (size_t)parent[0] * G;
        const float *B = W + (size_t)parent[1] * G;
        float *child = Wnext + (size_t)c * G;
        /* 3. single-point crossover, one child per slot */
        uint32_t rc[4];
        draw(seed, 0u, (uint32_t)c, gen, TAG_CROSS, rc);
        int q = G;                                  /* no crossover: child = A */
        if ((uint64_t)rc[0] < Tc && G >= 2) q = 1 + (int)oracle_index(rc[1], (uint32_t)(G - 1));
        for (int g = 0; g < G; ++g) child[g] = g < q ? A[g] : B[g];
        /* 4. per-gene Gaussian mutation, no clamping (D6) */
        for (int g = 0; g < G; ++g) {
            uint32_t rm[4];
            draw(seed, (uint32_t)g, (uint32_t)c, gen, TAG_MUTATE, rm);
            if ((uint64_t)rm[0] < Tm) {
                float z = oracle_gauss(rm[1], rm[2]);
                float delta = sigma * z;
                child[g] = child[g] + delta;
            }
        }
    }
    return 0;
}

/* ---- run  ("replicated as many times as it is the
 * training iteration number").  best[g] = fitness of the first chromosome in
 * the order of generation gen0+g, g = 0..n; population g+1 = step(population g,
 * (float)F_g, seed, gen0+g).  W is updated in place to the final population,
 * F32 receives the final fitness.
 */
int oracle_run(int64_t P, int N, int d, int M, int family, const float *X, const float *t,
               int E, int k, double p_cross, double p_mut, float sigma,
               uint64_t seed, uint32_t gen0, uint32_t n_gens, float *W, float *F32, float *best)
{
    int G = oracle_num_genes(N, d, family);
    if (G < 0) return -1;
    double *F = (double *)malloc(sizeof(double) * (size_t)M);
    float *Wn = (float *)malloc(sizeof(float) * (size_t)M * G);
    if (!F || !Wn) { free(F); free(Wn); return -2; }
    int rc = 0;
    for (uint32_t g = 0; g <= n_gens; ++g) {
        rc = oracle_eval_fitness(P, N, d, M, family, X, t, W, F, NULL);
        if (rc) break;
        for (int m = 0; m < M; ++m) F32[m] = (float)F[m];
        if (best) best[g] = F32[oracle_best_index(M, F32)];
        if (g == n_gens) break;
        rc = oracle_step(M, G, E, k, p_cross, p_mut, sigma, seed, gen0 + g, W, F32, Wn);
        if (rc) break;
        memcpy(W, Wn, sizeof(float) * (size_t)M * G);
    }
    free(F);
    free(Wn);
    return rc;
}

/* ---- batch views of the scalar samplers (same arithmetic, for the pins) ---- */
void oracle_neg2ln_u1_many(int64_t n, const uint32_t *a, float *out)
{
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_neg2ln_u1(a[i]);
}

void oracle_cos_angle_many(int64_t n, const uint32_t *b, float *out)
{
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_cos_angle(b[i]);
}

void oracle_gauss_many(int64_t n, const uint32_t *a, const uint32_t *b, float *out)
{
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_gauss(a[i], b[i]);
}

/* ---- test / validation use case  ("test" and "run" apply a trained chromosome to patterns;
 * PAPER.md:91 "crispy" classification).  y[q] = act(sum_g w[g] phi_g(x_q)) -- eq.(2) with D1/D2 -- for one
 * chromosome over Q patterns, and the confusion counts of the thresholded outputs against 0/1 targets:
 * counts = {TP, FP, TN, FN} with predicted class = (y > threshold), true class = (t > 0.5). */
void oracle_predict(int64_t Q, int N, int d, int family, const float *X, const float *w, double *y)
{
    for (int64_t q = 0; q < Q; ++q) y[q] = oracle_output(N, d, family, X + q * N, w);
}

void oracle_confusion(int64_t Q, const double *y, const float *t, double threshold, int64_t counts[4])
{
    counts[0] = counts[1] = counts[2] = counts[3] = 0;
    for (int64_t q = 0; q < Q; ++q) {
        int pred = y[q] > threshold, truth = t[q] > 0.5f;
        if (pred && truth) counts[0]++;
        else if (pred && !truth) counts[1]++;
        else if (!pred && !truth) counts[2]++;
        else counts[3]++;
    }
}

/* ---- run with the paper's stop rule  ("until the maximum number of iterations or the learning error
 * threshold", "MSE error threshold 0.001").  As oracle_run, but generation g's population is final as
 * soon as its best fitness <= threshold (a NaN best never stops).  Returns the number of GA steps performed in
 * *gens_done (0..max_gens); best[0..*gens_done] are written, W/F32 hold the final population and its fitness. */
int oracle_run_until(int64_t P, int N, int d, int M, int family, const float *X, const float *t,
                     int E, int k, double p_cross, double p_mut, float sigma,
                     uint64_t seed, uint32_t gen0, uint32_t max_gens, float threshold,
                     float *W, float *F32, float *best, uint32_t *gens_done)
{
    int G = oracle_num_genes(N, d, family);
    if (G < 0) return -1;
    double *F = (double *)malloc(sizeof(double) * (size_t)M);
    float *Wn = (float *)malloc(sizeof(float) * (size_t)M * G);
    if (!F || !Wn) { free(F); free(Wn); return -2; }
    int rc = 0;
    uint32_t g = 0;
    for (;; ++g) {
        rc = oracle_eval_fitness(P, N, d, M, family, X, t, W, F, NULL);
        if (rc) break;
        for (int m = 0; m < M; ++m) F32[m] = (float)F[m];
        float b = F32[oracle_best_index(M, F32)];
        if (best) best[g] = b;
        if (b <= threshold || g == max_gens) break;
        rc = oracle_step(M, G, E, k, p_cross, p_mut, sigma, seed, gen0 + g, W, F32, Wn);
        if (rc) break;
        memcpy(W, Wn, sizeof(float) * (size_t)M * G);
    }
    *gens_done = g;
    free(F);
    free(Wn);
    return rc;
}

/* ---- the paper's own selection methods  ("roulette/ranking", "selection: RANKING and
 * ROULETTE"; the paper does not define them: DESIGN.md reading R10).  Both pick parent A and parent B of child slot c
 * independently from words w0 and w1 of ONE Philox call with counter (0, c, gen, TAG_SELECT); everything is integer
 * arithmetic so that a GPU can reproduce it bit for bit.
 *
 * RANKING (linear ranking): chromosomes ordered by `precedes` (rank 0 = best); rank r has weight M - r, total
 *   T = M (M + 1) / 2;  u = floor(w * T / 2^32);  the selected rank is the smallest r with
 *   C(r) = (r + 1) M - r (r + 1) / 2 > u;  the parent is the chromosome holding that rank.
 * ROULETTE (fitness-proportionate on the paper's fitness 1 - error): weight_i =
 *   floor(clamp(1 - key(F_i), 0, 1) * 2^32) evaluated in double (NaN / +inf fitness -> 0), T = sum of weights;
 *   u = floor(w * T / 2^32);  the parent is the smallest index i whose prefix sum exceeds u;  T = 0 -> uniform index.
 */
enum { SEL_TOURNAMENT = 0, SEL_RANKING = 1, SEL_ROULETTE = 2 };

uint64_t oracle_roulette_weight(float f)
{
    float key = fit_key(f);
    double v = 1.0 - (double)key;
    if (!(v > 0.0)) return 0;
    if (v >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)floor(v * 4294967296.0);
}

int oracle_rank_from_word(uint32_t w, int M)
{
    uint64_t T = (uint64_t)M * (uint64_t)(M + 1) / 2;
    uint64_t u = (uint64_t)(((unsigned __int128)w * T) >> 32);
    for (int r = 0; r < M; ++r) {
        uint64_t C = (uint64_t)(r + 1) * (uint64_t)M - (uint64_t)r * (uint64_t)(r + 1) / 2;
        if (C > u) return r;
    }
    return M - 1;
}

int oracle_roulette_from_word(uint32_t w, int M, const uint64_t *weight)
{
    uint64_t T = 0;
    for (int i = 0; i < M; ++i) T += weight[i];
    if (T == 0) return (int)oracle_index(w, (uint32_t)M);
    uint64_t u = (uint64_t)(((unsigned __int128)w * T) >> 32);
    uint64_t acc = 0;
    for (int i = 0; i < M; ++i) {
        acc += weight[i];
        if (acc > u) return i;
    }
    return M - 1;
}

/* One generation as oracle_step, with the selection method chosen by `selection` (crossover, mutation, elitism and
 * their draws are unchanged; `k` is only used by SEL_TOURNAMENT). */
int oracle_step_sel(int M, int G, int E, int k, int selection, double p_cross, double p_mut, float sigma,
                    uint64_t seed, uint32_t gen, const float *W, const float *F, float *Wnext)
{
    if (selection == SEL_TOURNAMENT) return oracle_step(M, G, E, k, p_cross, p_mut, sigma, seed, gen, W, F, Wnext);
    if (M < 1 || G < 1 || E < 0 || E >= M || selection > SEL_ROULETTE) return -1;
    int *by_rank = (int *)malloc(sizeof(int) * (size_t)M);
    uint64_t *weight = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)M);
    if (!by_rank || !weight) { free(by_rank); free(weight); return -2; }
    for (int m = 0; m < M; ++m) {
        int r = 0;
        for (int j = 0; j < M; ++j) r += precedes(F, j, m);
        by_rank[r] = m;
        weight[m] = oracle_roulette_weight(F[m]);
    }
    for (int s = 0; s < E; ++s)
        memcpy(Wnext + (size_t)s * G, W + (size_t)by_rank[s] * G, sizeof(float) * (size_t)G);
    uint64_t Tc = oracle_bernoulli_threshold(p_cross);
    uint64_t Tm = oracle_bernoulli_threshold(p_mut);
    for (int c = E; c < M; ++c) {
        uint32_t r[4];
        draw(seed, 0u, (uint32_t)c, gen, TAG_SELECT, r);
        int parent[2];
        for (int s = 0; s < 2; ++s)
            parent[s] = selection == SEL_RANKING ? by_rank[oracle_rank_from_word(r[s], M)]
                                                 : oracle_roulette_from_word(r[s], M, weight);
        const float *A = W + (size_t)parent[0] * G;
        const float *B = W + (size_t)parent[1] * G;
        float *child = Wnext + (size_t)c * G;
        uint32_t rc[4];
        draw(seed, 0u, (uint32_t)c, gen, TAG_CROSS, rc);
        int q = G;
        if ((uint64_t)rc[0] < Tc && G >= 2) q = 1 + (int)oracle_index(rc[1], (uint32_t)(G - 1));
        for (int g = 0; g < G; ++g) child[g] = g < q ? A[g] : B[g];
        for (int g = 0; g < G; ++g) {
            uint32_t rm[4];
            draw(seed, (uint32_t)g, (uint32_t)c, gen, TAG_MUTATE, rm);
            if ((uint64_t)rm[0] < Tm) {
                float z = oracle_gauss(rm[1], rm[2]);
                float delta = sigma * z;
                child[g] = child[g] + delta;
            }
        }
    }
    free(by_rank);
    free(weight);
    return 0;
}


/* ---- random replacement  ("a variable number of chromosomes are randomly generated to replace older
 * individuals"; reading R12).  After a generation step the last R child slots M-R..M-1 (never elite slots:
 * R <= M - E) are overwritten by fresh random chromosomes, genes uniform in [-1,1) exactly as at initialisation but
 * drawn with counter (g>>2, c, gen, TAG_IMMIGRANT = 4), word g&3. */
enum { TAG_IMMIGRANT = 4 };

int oracle_immigrate(int M, int G, int E, int R, uint64_t seed, uint32_t gen, float *Wnext)
{
    if (R < 0 || R > M - E) return -1;
    for (int c = M - R; c < M; ++c)
        for (int g = 0; g < G; ++g) {
            uint32_t r[4];
            draw(seed, (uint32_t)(g >> 2), (uint32_t)c, gen, TAG_IMMIGRANT, r);
            Wnext[(size_t)c * G + g] = (float)(r[g & 3] >> 8) * 0x1p-23f - 1.0f;
        }
    return 0;
}


/* ---- RMSE  ("the MSE or the RMSE may be used"): F_rmse[m] = sqrt((1/P) sum_p (y - t)^2), in double. */
int oracle_eval_rmse(int64_t P, int N, int d, int M, int family, const float *X, const float *t, const float *W, double *F)
{
    int rc = oracle_eval_fitness(P, N, d, M, family, X, t, W, F, NULL);
    if (rc) return rc;
    for (int m = 0; m < M; ++m) F[m] = sqrt(F[m]);
    return 0;
}
