/*
 * game_oracle.c -- fp64 CPU oracle for the GAME fitness / GA hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this.  It shares no code
 * (no headers, helpers, tables, constants) with paper_1304_0597_b200/csrc; the product
 * never calls it and has no CPU fallback.
 *
 * Written from /root/reference/PAPER.md (Cavuoti et al., arXiv:1304.0597); "L<n>" below
 * are PAPER.md line numbers.  Where the paper is silent or garbled the reading is the one
 * listed in DESIGN.md section 3 (G1..G22, R0..R6, taken from SURVEY.md 8(c)).
 *
 * Two halves:
 *   fitness      -- the plain definition: eq. 1-2 / eq. 8-9 (L52-L58, L95-L103) expansion,
 *                   dot product with the chromosome, activation (DESIGN G4), per-pattern
 *                   error eq. 3 / eq. 10 (L62, L113; DESIGN G5), mean eq. 4-5 (L71-L75).
 *                   fp64, ascending loops, no blocking, no BLAS.
 *   GA operators -- an algorithm, followed step by step (L217-L220, L144-L148, L282-L291),
 *                   every random decision in integer arithmetic on Philox4x32-10 words.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Chebyshev/trig closed forms, discrete
 * orthogonality, the paper's worked MSE/TMSE example (L109, L118), numpy float64 GEMM for
 * the identity+MSE case, least squares optimum, planted chromosome, tied-gene reduction
 * (eq. 9 as printed), row replication (L326), hand-written brute force, Philox against
 * torch's ATen philox_engine, tournament closed-form distribution, crossover / mutation /
 * elitism invariants; exact hand-worked values (rational arithmetic, ATen's Philox words) for
 * interior roulette weights and the normal-mode initial gene (tests/test_oracle_exact_pins.py);
 * the whole pin suite also runs against an -fsanitize=address,undefined build
 * (tests/test_oracle_sanitized.py).  The roulette weight RULE R4 (DESIGN G14) is this build's
 * choice -- the paper gives none ("parity unpinned" against the paper); its implementation here
 * is pinned exactly to that rule.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libgame_oracle.so game_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { FAM_TRIG = 0, FAM_CHEB = 1, FAM_TRIG_TIED = 2, FAM_POLY_TIED = 3 };
enum { ACT_SIGMOID = 0, ACT_IDENTITY = 1 };
enum { ERR_MSE = 0, ERR_TMSE = 1, ERR_RMSE = 2 };
enum { SEL_TOURNAMENT = 0, SEL_ROULETTE = 1 };
enum { INIT_UNIFORM_PM1 = 0, INIT_NORMAL_PM1 = 1, INIT_UNIFORM_01 = 2 };
enum { ELITE_COPIES_OF_BEST = 0, ELITE_TOP_E = 1 };
enum { TAG_INIT = 0, TAG_SELECT = 1, TAG_XOVER = 2, TAG_MUTATE = 3 };

typedef struct {
    int P, tournament_size, elitism, elite_mode, selection, init_mode;
    float p_crossover, p_mutation, stop_error;
} oracle_ga_params;

typedef struct {
    int generations_run;
    int stopped_on_error;
    float best_error;
    int best_index;
} oracle_result;

/* ---- threads (cpu_baseline reports the count it actually used) ------------------------- */
int oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

/* ---- a1: feature expansion -------------------------------------------------------------
 * Gene / term index k = i*B + m, feature-major, block order [a_0, a_1..a_d, b_1..b_d] (L105).
 * TRIG (eq. 8-9): B = 2d+1; m=0 -> 1; m=1..d -> cos(m x); m=d+1..2d -> sin((m-d) x),
 *   radians, argument m*x with no pi factor, as printed.
 * CHEB (eq. 1 with g^j = T_j, DESIGN G7): B = d+1; T_0 = 1, T_1 = x, T_{m+1} = 2x T_m - T_{m-1}.
 */
int oracle_num_terms(int family, int degree, int F)
{
    if (F < 1 || degree < 1) return -1;
    if (family == FAM_TRIG) return F * (2 * degree + 1);
    if (family == FAM_CHEB) return F * (degree + 1);
    if (family == FAM_TRIG_TIED) return 2 * degree + 1;   /* eq. 7 with B = 2: the paper's own chromosome (L105) */
    if (family == FAM_POLY_TIED) return degree + 1;       /* eq. 7 with B = 1, g(x) = x (L89) */
    return -1;
}

/* Paper-literal models: ONE coefficient set shared by every feature (eq. 2 and eq. 9 as printed, L57, L100-L103):
 *   TRIG_TIED: Out = a_0 + sum_m a_m sum_i cos(m f_i) + sum_m b_m sum_i sin(m f_i), genes [a_0, a_1..a_d, b_1..b_d];
 *              the per-pattern sums of cosines and sines are the paper's two precomputed vectors (L254).
 *   POLY_TIED: Out = a_0 + sum_j a_j sum_i f_i^j (eq. 2 with g(x) = x, powers), genes [a_0..a_d].
 * The constant a_0 appears once, not once per feature. */
static void expand_row_tied(int family, int d, int F, const float *x, double *phi)
{
    int K = family == FAM_TRIG_TIED ? 2 * d + 1 : d + 1;
    for (int k = 0; k < K; ++k) phi[k] = 0.0;
    phi[0] = 1.0;
    for (int i = 0; i < F; ++i) {
        double xi = (double)x[i];
        if (family == FAM_TRIG_TIED) {
            for (int m = 1; m <= d; ++m) { phi[m] += cos((double)m * xi); phi[d + m] += sin((double)m * xi); }
        } else {
            double pw = 1.0;
            for (int j = 1; j <= d; ++j) { pw *= xi; phi[j] += pw; }
        }
    }
}

static void expand_row(int family, int d, int F, const float *x, double *phi)
{
    if (family == FAM_TRIG_TIED || family == FAM_POLY_TIED) { expand_row_tied(family, d, F, x, phi); return; }
    for (int i = 0; i < F; ++i) {
        double xi = (double)x[i];
        if (family == FAM_TRIG) {
            int B = 2 * d + 1;
            phi[i * B + 0] = 1.0;
            for (int m = 1; m <= d; ++m) phi[i * B + m] = cos((double)m * xi);
            for (int m = 1; m <= d; ++m) phi[i * B + d + m] = sin((double)m * xi);
        } else {
            int B = d + 1;
            double tm1 = 1.0, t0 = xi;
            phi[i * B + 0] = 1.0;
            if (d >= 1) phi[i * B + 1] = xi;
            for (int m = 2; m <= d; ++m) {
                double t1 = 2.0 * xi * t0 - tm1;
                phi[i * B + m] = t1;
                tm1 = t0;
                t0 = t1;
            }
        }
    }
}

void oracle_expand(int family, int degree, int F, const float *X, long long N, double *E)
{
    int K = oracle_num_terms(family, degree, F);
    for (long long n = 0; n < N; ++n) expand_row(family, degree, F, X + n * F, E + n * K);
}

/* ---- a3: activation (DESIGN G4): logistic 1/(1+e^-z), or identity (paper-literal eq. 2) -- */
static double activate(int act, double z)
{
    if (act == ACT_SIGMOID) return 1.0 / (1.0 + exp(-z));
    return z;
}

/* forward pass of ONE chromosome on N patterns: z = sum_k E[n][k] c[k] (eq. 2 / eq. 9), y = act(z) */
void oracle_forward(int family, int degree, int F, int act, const float *X, long long N,
                    const float *genes, double *z_out, double *y_out)
{
    int K = oracle_num_terms(family, degree, F);
    double *phi = (double *)malloc(sizeof(double) * (size_t)K);
    for (long long n = 0; n < N; ++n) {
        expand_row(family, degree, F, X + n * F, phi);
        double z = 0.0;
        for (int k = 0; k < K; ++k) z += phi[k] * (double)genes[k];
        if (z_out) z_out[n] = z;
        if (y_out) y_out[n] = activate(act, z);
    }
    free(phi);
}

/* ---- test / run use cases (L127-L129) and the figures of merit of L301 ----------------------------------
 * A pattern is classified GC (class 1) when act(z) > cut, and IS a GC when its target > 0.5.
 * counts = {TP, FP, TN, FN}.  L301: accuracy = "fraction of patterns which are correctly classified
 * (either GCs or non-GCs) with respect to the total" = (TP+TN)/N; completeness = "fraction of GCs which are
 * correctly classified as such" = TP/(TP+FN); contamination = "fraction of non-GC objects which are
 * erroneously classified as GCs" = FP/(FP+TN), read literally (DESIGN G23).  An empty denominator gives 0.
 * near (optional) counts the patterns with |act(z) - cut| <= delta: a lower-precision implementation may
 * legitimately classify those the other way. */
void oracle_classify(int family, int degree, int F, int act, const float *X, const float *t, long long N,
                     const float *genes, double cut, long long counts[4], double fom[3], long long *near,
                     double delta)
{
    int K = oracle_num_terms(family, degree, F);
    double *phi = (double *)malloc(sizeof(double) * (size_t)K);
    long long tp = 0, fp = 0, tn = 0, fn = 0, nr = 0;
    for (long long n = 0; n < N; ++n) {
        expand_row(family, degree, F, X + n * F, phi);
        double z = 0.0;
        for (int k = 0; k < K; ++k) z += phi[k] * (double)genes[k];
        double y = activate(act, z);
        int pred = y > cut, truth = (double)t[n] > 0.5;
        if (pred && truth) ++tp;
        else if (pred && !truth) ++fp;
        else if (!pred && !truth) ++tn;
        else ++fn;
        if (fabs(y - cut) <= delta) ++nr;
    }
    free(phi);
    counts[0] = tp; counts[1] = fp; counts[2] = tn; counts[3] = fn;
    if (fom) {
        fom[0] = N > 0 ? (double)(tp + tn) / (double)N : 0.0;
        fom[1] = tp + fn > 0 ? (double)tp / (double)(tp + fn) : 0.0;
        fom[2] = fp + tn > 0 ? (double)fp / (double)(fp + tn) : 0.0;
    }
    if (near) *near = nr;
}

/* ---- a1..a5: fitness of every chromosome -------------------------------------------------
 * fit[p] = (1/N) sum_n e(t_n - act(z[n][p]))  (eq. 4); RMSE = sqrt (eq. 5).
 * e(r) = r^2 (eq. 3); TMSE (eq. 10, read per DESIGN G5 from the worked example
 * L109/L118): e = r^2 if |r| > R else 0, still averaged over all N.
 * near[p] (optional) = #{n : ||r| - R| <= delta}: how many patterns sit within delta of the TMSE
 * discontinuity, so a test can widen its tolerance by near*(R+delta)^2/N.
 * The expansion is computed once (the paper's own hoisting, L254) and the contraction is the
 * plain triple loop; OpenMP only splits the chromosome loop, the order inside one chromosome
 * is ascending n, ascending k.
 */
int oracle_fitness(int family, int degree, int F, int act, int err, double R, const float *X,
                   const float *t, long long N, const float *pop, int P, double *fit,
                   long long *near, double delta)
{
    int K = oracle_num_terms(family, degree, F);
    if (K < 0 || N < 1 || P < 1) return 1;
    double *E = (double *)malloc(sizeof(double) * (size_t)N * (size_t)K);
    if (!E) return 2;
    oracle_expand(family, degree, F, X, N, E);
#pragma omp parallel for schedule(dynamic, 1)
    for (int p = 0; p < P; ++p) {
        const float *c = pop + (size_t)p * K;
        double acc = 0.0;
        long long cnt = 0;
        for (long long n = 0; n < N; ++n) {
            const double *phi = E + (size_t)n * K;
            double z = 0.0;
            for (int k = 0; k < K; ++k) z += phi[k] * (double)c[k];
            double y = activate(act, z);
            double r = (double)t[n] - y;
            double e = r * r;
            if (err == ERR_TMSE) {
                if (fabs(r) <= R) e = 0.0;
                if (fabs(fabs(r) - R) <= delta) ++cnt;
            }
            acc += e;
        }
        double f = acc / (double)N;
        if (err == ERR_RMSE) f = sqrt(f);
        fit[p] = f;
        if (near) near[p] = cnt;
    }
    free(E);
    return 0;
}

/* ---- Philox4x32-10 (Salmon et al. 2011), counter-based: out = f(key, counter) --------------
 * DESIGN R-rules: key = (seed lo, seed hi); counter = (primary, secondary, generation, tag). */
void oracle_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
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

static void draw(uint64_t seed, uint32_t a, uint32_t b, uint32_t g, uint32_t tag, uint32_t w[4])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { a, b, g, tag };
    oracle_philox4x32_10(key, ctr, w);
}

/* ---- R0 helpers: integer -> decision / float, all exact ------------------------------------ */
uint32_t oracle_idx(uint32_t w, uint32_t n) { return (uint32_t)(((uint64_t)w * (uint64_t)n) >> 32); }

/* thr(p): p >= 1 -> always; else floor(p * 2^32) computed in double (p is a float, so exact) */
uint32_t oracle_thr(float p, int *always)
{
    if (p >= 1.0f) { *always = 1; return 0xFFFFFFFFu; }
    *always = 0;
    if (!(p > 0.0f)) return 0u;
    return (uint32_t)floor((double)p * 4294967296.0);
}

static int hit(uint32_t w, float p)
{
    int always;
    uint32_t th = oracle_thr(p, &always);
    return always || (w < th);
}

float oracle_upm1(uint32_t w) { return (float)((int32_t)(w >> 8) - 8388608) * 0x1p-23f; }
float oracle_u01(uint32_t w) { return (float)(w >> 8) * 0x1p-24f; }

/* ---- a12: initial population (L133-L142; DESIGN G13, R1, R2) ------------------------------- */
float oracle_init_gene(int mode, uint64_t seed, int p, int k)
{
    uint32_t w[4];
    if (mode == INIT_NORMAL_PM1) {
        /* Irwin-Hall: 12 uniform 24-bit integers; Z = (S - 6(2^24-1)) 2^-24 ~ N(0,1); gene = clamp(Z/3) */
        uint32_t S = 0;
        for (uint32_t j = 0; j < 3; ++j) {
            draw(seed, (uint32_t)k, (uint32_t)p, j, TAG_INIT, w);
            for (int i = 0; i < 4; ++i) S += (w[i] >> 8);
        }
        float v = (float)((int32_t)S - (int32_t)(6u * 16777215u));
        volatile float prod = v * 0x1.555556p-26f; /* fl(2^-24 / 3), one IEEE multiply */
        float gne = prod;
        if (gne < -1.0f) gne = -1.0f;
        if (gne > 1.0f) gne = 1.0f;
        return gne;
    }
    draw(seed, (uint32_t)k, (uint32_t)p, 0u, TAG_INIT, w);
    return mode == INIT_UNIFORM_01 ? oracle_u01(w[0]) : oracle_upm1(w[0]);
}

void oracle_init_population(int mode, uint64_t seed, int P, int K, float *pop)
{
    for (int p = 0; p < P; ++p)
        for (int k = 0; k < K; ++k) pop[(size_t)p * K + k] = oracle_init_gene(mode, seed, p, k);
}

/* ---- a6: rank (L218 "find and sort the best chromosomes"; DESIGN G12, G20) -----------------
 * ascending error, ties by index, NaN counts as +inf.  Insertion sort: P <= ~1e4 in tests. */
static int before(const float *fit, int a, int b)
{
    float fa = isnan(fit[a]) ? INFINITY : fit[a];
    float fb = isnan(fit[b]) ? INFINITY : fit[b];
    if (fa < fb) return 1;
    if (fb < fa) return 0;
    return a < b;
}

void oracle_rank(const float *fit, int P, int *order)
{
    /* bottom-up merge sort on indices with the (fit, index) total order: stable and exact */
    int *tmp = (int *)malloc(sizeof(int) * (size_t)P);
    for (int i = 0; i < P; ++i) order[i] = i;
    for (int w = 1; w < P; w *= 2) {
        for (int lo = 0; lo < P; lo += 2 * w) {
            int mid = lo + w < P ? lo + w : P, hi = lo + 2 * w < P ? lo + 2 * w : P;
            int i = lo, j = mid, o = lo;
            while (i < mid && j < hi) tmp[o++] = before(fit, order[j], order[i]) ? order[j++] : order[i++];
            while (i < mid) tmp[o++] = order[i++];
            while (j < hi) tmp[o++] = order[j++];
        }
        memcpy(order, tmp, sizeof(int) * (size_t)P);
    }
    free(tmp);
}

/* ---- a9: selection ------------------------------------------------------------------------- */
/* R3 tournament by rank (L147 "ranking", L290 tournament size; DESIGN G14): t rank draws with
 * replacement, the best (smallest) rank wins. */
static int select_tournament(const oracle_ga_params *gp, uint64_t seed, uint32_t g, uint32_t slot,
                             const int *order)
{
    uint32_t w[4];
    uint32_t best = 0xFFFFFFFFu;
    for (int j = 0; j < gp->tournament_size; ++j) {
        if ((j & 3) == 0) draw(seed, (uint32_t)(j >> 2), slot, g, TAG_SELECT, w);
        uint32_t r = oracle_idx(w[j & 3], (uint32_t)gp->P);
        if (r < best) best = r;
    }
    return order[best];
}

/* R4 roulette (L147; weight formula is DESIGN G14's choice -- parity unpinned by the paper):
 * w_r = floor(((f_max - f_r)/(f_max - f_min)) * 2^24) + 1 on the fp32 fitness bits. */
void oracle_roulette_weights(const float *fit, const int *order, int P, uint32_t *wts)
{
    float fmax = -INFINITY, fmin = INFINITY;
    int nfinite = 0;
    for (int r = 0; r < P; ++r) {
        float f = fit[order[r]];
        if (isfinite(f)) { ++nfinite; if (f > fmax) fmax = f; if (f < fmin) fmin = f; }
    }
    volatile float b = fmax - fmin;
    for (int r = 0; r < P; ++r) {
        float f = fit[order[r]];
        if (nfinite == 0) { wts[r] = 1u; continue; }
        if (!isfinite(f)) { wts[r] = 0u; continue; }
        if (!(b > 0.0f)) { wts[r] = 1u; continue; }
        volatile float a = fmax - f;
        volatile float q = a / b;               /* IEEE fp32 divide */
        wts[r] = (uint32_t)(q * 16777216.0f) + 1u; /* exact scale by 2^24, truncation */
    }
}

static int select_roulette(const oracle_ga_params *gp, uint64_t seed, uint32_t g, uint32_t slot,
                           const int *order, const uint32_t *wts)
{
    uint32_t w[4];
    draw(seed, 0u, slot, g, TAG_SELECT, w);
    uint64_t total = 0;
    for (int r = 0; r < gp->P; ++r) total += wts[r];
    uint64_t u = ((uint64_t)w[0] << 32) | (uint64_t)w[1];
    uint64_t T = (uint64_t)(((unsigned __int128)u * (unsigned __int128)total) >> 64);
    uint64_t pre = 0;
    for (int r = 0; r < gp->P; ++r) {
        pre += wts[r];
        if (pre > T) return order[r];
    }
    return order[gp->P - 1];
}

/* ---- a8..a11: one generation of operators, from a given rank order -------------------------
 * steps 4-6 of DESIGN 3.3: elitism (L148, L291; G17), selection (R3/R4),
 * single-point crossover per pair with probability p_c (L288; G15, R5), per-gene mutation with
 * probability p_m on non-elite children (L289, L226; G16, R6).
 * dbg_parents[2*q+s], dbg_do[q], dbg_cut[q] (optional) expose the decisions to the tests. */
void oracle_ga_step(const oracle_ga_params *gp, uint64_t seed, uint32_t g, int K, const int *order,
                    const float *fit, const float *pop, float *next, int *dbg_parents, int *dbg_do,
                    int *dbg_cut)
{
    const int P = gp->P, e = gp->elitism;
    uint32_t *wts = NULL;
    if (gp->selection == SEL_ROULETTE) {
        wts = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)P);
        oracle_roulette_weights(fit, order, P, wts);
    }
    /* 4. elites */
    for (int j = 0; j < e; ++j) {
        int src = gp->elite_mode == ELITE_TOP_E ? order[j] : order[0];
        memcpy(next + (size_t)j * K, pop + (size_t)src * K, sizeof(float) * (size_t)K);
    }
    /* 5. children in pairs */
    int npairs = (P - e + 1) / 2;
    for (int q = 0; q < npairs; ++q) {
        int par[2];
        for (int s = 0; s < 2; ++s)
            par[s] = gp->selection == SEL_ROULETTE
                         ? select_roulette(gp, seed, g, (uint32_t)(2 * q + s), order, wts)
                         : select_tournament(gp, seed, g, (uint32_t)(2 * q + s), order);
        uint32_t w[4];
        draw(seed, 0u, (uint32_t)q, g, TAG_XOVER, w);
        int doit = (K >= 2) && hit(w[0], gp->p_crossover);
        int cut = K >= 2 ? 1 + (int)oracle_idx(w[1], (uint32_t)(K - 1)) : 0;
        if (dbg_parents) { dbg_parents[2 * q] = par[0]; dbg_parents[2 * q + 1] = par[1]; }
        if (dbg_do) dbg_do[q] = doit;
        if (dbg_cut) dbg_cut[q] = cut;
        const float *pa = pop + (size_t)par[0] * K, *pb = pop + (size_t)par[1] * K;
        for (int s = 0; s < 2; ++s) {
            int slot = e + 2 * q + s;
            if (slot >= P) break; /* odd child count: last B dropped (G19) */
            float *ch = next + (size_t)slot * K;
            for (int k = 0; k < K; ++k) {
                int from_a = doit ? ((k < cut) == (s == 0)) : (s == 0);
                ch[k] = from_a ? pa[k] : pb[k];
            }
        }
    }
    /* 6. mutation over slots e..P-1 */
    for (int s = e; s < P; ++s)
        for (int k = 0; k < K; ++k) {
            uint32_t w[4];
            draw(seed, (uint32_t)k, (uint32_t)s, g, TAG_MUTATE, w);
            if (hit(w[0], gp->p_mutation)) next[(size_t)s * K + k] = oracle_upm1(w[1]);
        }
    free(wts);
}

/* ---- the training loop (L217-L220; DESIGN G18) ---------------------------------------------
 * [init if !have_pop] ; G x (fitness, rank, stop test, operators) ; final fitness + rank.
 * *gen_io is the absolute generation counter (continues across calls, DESIGN P22).
 * best_hist (optional, length generations+1) receives the best error seen at each evaluation. */
int oracle_evolve(int family, int degree, int F, int act, int err, double R, const float *X,
                  const float *t, long long N, const oracle_ga_params *gp, uint64_t seed,
                  int generations, float *pop, int have_pop, uint32_t *gen_io, float *fit_out,
                  int *order_out, oracle_result *res, float *best_hist)
{
    const int P = gp->P;
    const int K = oracle_num_terms(family, degree, F);
    if (K < 0 || P < 2) return 1;
    if (!have_pop) oracle_init_population(gp->init_mode, seed, P, K, pop);
    double *fit64 = (double *)malloc(sizeof(double) * (size_t)P);
    float *next = (float *)malloc(sizeof(float) * (size_t)P * (size_t)K);
    int run = 0, stopped = 0;
    for (;;) {
        oracle_fitness(family, degree, F, act, err, R, X, t, N, pop, P, fit64, NULL, 0.0);
        for (int p = 0; p < P; ++p) fit_out[p] = (float)fit64[p];
        oracle_rank(fit_out, P, order_out);
        if (best_hist) best_hist[run] = fit_out[order_out[0]];
        if (gp->stop_error >= 0.0f && fit_out[order_out[0]] <= gp->stop_error) { stopped = 1; break; }
        if (run == generations) break;
        oracle_ga_step(gp, seed, *gen_io, K, order_out, fit_out, pop, next, NULL, NULL, NULL);
        memcpy(pop, next, sizeof(float) * (size_t)P * (size_t)K);
        ++*gen_io;
        ++run;
    }
    if (res) {
        res->generations_run = run;
        res->stopped_on_error = stopped;
        res->best_error = fit_out[order_out[0]];
        res->best_index = order_out[0];
    }
    free(fit64);
    free(next);
    return 0;
}
