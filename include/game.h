/*
 * game.h -- C ABI of libgame_b200: the GAME (Genetic Algorithm Model Experiment) fitness / GA
 * hot path of Cavuoti et al., arXiv:1304.0597, as hand-written sm_100a CUDA kernels.
 *
 * Citations "L<n>" are line numbers of the paper text; "DESIGN Gx/Rx" are the
 * readings listed in DESIGN.md section 3 for what the paper leaves open.
 *
 * Notation (BASELINE.json's): N patterns, F features, d degree, K terms = genes per chromosome,
 * P chromosomes, G generations.  K = F*(2d+1) for GAME_TRIG, F*(d+1) for GAME_CHEB.
 *
 * Conventions
 *  - Every function returns 0 (GAME_OK) or a positive error code; game_last_error() gives the text.
 *    No exceptions, no exit(), no global state (no environment variables are read; every setting lives
 *    in the context), no CPU fallback: without a CUDA device every compute call fails with GAME_ERR_CUDA.
 *  - A context belongs to the CUDA device that was current when game_create ran; every call makes that
 *    device current for its duration and restores the caller's, so contexts on several GPUs can be
 *    driven from one thread.
 *  - Pointer arguments are marked DEV (CUDA device memory, caller-owned, must stay valid until the
 *    context's stream has consumed them) or HOST (ordinary or pinned host memory).  The library
 *    never frees or keeps caller memory; game_load* copies / re-lays what it needs.
 *  - Calls enqueue work on the context's stream and return without waiting, except where noted.
 *  - A context is not thread-safe; use one per thread.
 *  - Fitness values are ERRORS: lower is better (the paper says "maximum fitness", L131, while
 *    minimising eq. 3-5; DESIGN G12).
 */
#ifndef GAME_B200_H
#define GAME_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct game_ctx game_ctx; /* opaque */

enum { GAME_OK = 0, GAME_ERR_INVALID_ARG = 1, GAME_ERR_NOT_LOADED = 2, GAME_ERR_ALLOC = 3,
       GAME_ERR_CUDA = 4, GAME_ERR_UNSUPPORTED = 5, GAME_ERR_NONFINITE_INPUT = 6 };

/* Expansion family.  TRIG / CHEB: one coefficient per (feature, term), K = F(2d+1) / F(d+1) (eq. 8-9 L95-L103 /
 * eq. 1 with g^j = T_j; DESIGN G1).  TRIG_TIED / POLY_TIED: the paper-literal models, one coefficient set shared
 * by all features acting on per-pattern sums over features (eq. 9 / eq. 2 as printed, L57, L100-L105, L254):
 * K = 2d+1 genes [a_0, a_1..a_d, b_1..b_d] on (1, sum_i cos(m f_i), sum_i sin(m f_i)); K = d+1 genes on sum_i f_i^j. */
enum { GAME_TRIG = 0, GAME_CHEB = 1, GAME_TRIG_TIED = 2, GAME_POLY_TIED = 3 };
enum { GAME_ACT_SIGMOID = 0, GAME_ACT_IDENTITY = 1 };  /* DESIGN G4; identity is the paper-literal eq. 2 */
enum { GAME_ERR_MSE = 0, GAME_ERR_TMSE = 1, GAME_ERR_RMSE = 2 };   /* eq. 4, eq. 10, eq. 5 (L71-L75, L113) */
enum { GAME_SEL_TOURNAMENT = 0, GAME_SEL_ROULETTE = 1 };           /* L147, L290; DESIGN G14 */
enum { GAME_INIT_UNIFORM_PM1 = 0, GAME_INIT_NORMAL_PM1 = 1, GAME_INIT_UNIFORM_01 = 2 }; /* L133-L142; DESIGN G13 */
enum { GAME_ELITE_COPIES_OF_BEST = 0, GAME_ELITE_TOP_E = 1 };      /* L148; DESIGN G17 */
/* Fitness kernel choice.  FP32: FFMA contraction, |rel err| <= 1e-5 class.  TENSOR: tcgen05 fp16-input /
 * fp32-accumulate MMA (same 11-bit significand as TF32), 1e-3 class.  AUTO picks by problem shape. */
enum { GAME_PATH_AUTO = 0, GAME_PATH_FP32 = 1, GAME_PATH_TENSOR = 2, GAME_PATH_TENSOR_SPLIT = 3 };
enum { GAME_EXPAND_AUTO = 0, GAME_EXPAND_MATERIALIZED = 1, GAME_EXPAND_REGENERATED = 2 };
/* GA parameters (L275-L291).  Probabilities are per parent pair (crossover, DESIGN G15) and per gene
 * (mutation, DESIGN G16).  stop_error < 0 disables the error-threshold stop (L219, L287). */
typedef struct {
    int   P;                /* population size, >= 2 */
    int   tournament_size;  /* >= 1 (L290) */
    int   elitism;          /* 0 <= elitism < P (L291) */
    int   elite_mode;       /* GAME_ELITE_* */
    int   selection;        /* GAME_SEL_* */
    int   init_mode;        /* GAME_INIT_* */
    float p_crossover;      /* [0,1] (L288) */
    float p_mutation;       /* [0,1] (L289) */
    float stop_error;       /* stop when best error <= stop_error; < 0: never */
} game_ga_params;

typedef struct {
    int   generations_run;   /* evolution steps performed by this call */
    int   stopped_on_error;  /* 1 if the last evaluation met stop_error */
    float best_error;        /* error of the best chromosome of the returned population */
    int   best_index;        /* its row in the population */
} game_result;

/* Create a context for one problem shape.  1 <= degree <= 32, F >= 1.  HOST out pointer.
 * The model: Out(pat) = sum_i G(f_i), G a degree-d expansion of feature f_i (eq. 1-2). */
int game_create(int family, int degree, int F, game_ctx **out);
void game_destroy(game_ctx *ctx);   /* synchronises the stream, frees all device memory */

/* K, the number of terms / genes per chromosome (eq. 7 generalised per feature, DESIGN G1). */
int game_num_terms(const game_ctx *ctx);
/* Absolute generation counter: number of evolution steps applied to the current population. */
long long game_generation(const game_ctx *ctx);
const char *game_last_error(const game_ctx *ctx);   /* HOST string owned by the context */

/* cuda_stream is a cudaStream_t (0 = legacy default stream).  Takes effect for later calls. */
int game_set_stream(game_ctx *ctx, void *cuda_stream);
int game_set_activation(game_ctx *ctx, int act);                 /* default GAME_ACT_SIGMOID */
int game_set_error(game_ctx *ctx, int err_type, float tmse_R);   /* default MSE; R in (0,1) for TMSE (L116) */
/* Which kernels evaluate a2-a5, i.e. the arithmetic and the tolerance class of the returned fitness (north_star (2)):
 *   GAME_PATH_FP32          fp32 FFMA contraction, fp32 epilogue: |fit - exact| <= 1e-5 |exact| + 1e-7;
 *   GAME_PATH_TENSOR        tcgen05 tensor cores, fp16 operands (TF32's 11-bit significand), fp32 accumulate:
 *                           1e-3 |exact| + 1e-5;  needs max|E| <= 2 (else GAME_ERR_UNSUPPORTED);
 *   GAME_PATH_TENSOR_SPLIT  tensor cores on split operands: E and the genes are each an fp16 hi + lo pair and the three
 *                           products hi.hi + hi.lo + lo.hi run as one fp16 contraction over 3K terms, fp32 accumulate,
 *                           ex2 + rcp logistic: the FP32 path's class (1e-5 |exact| + 1e-7; measured 3e-7 .. 9e-7).
 *                           Per-feature families with max|E| <= 1024;
 *   GAME_PATH_AUTO          (default) N >= 16384: TENSOR;  smaller datasets: TENSOR_SPLIT;  FP32 where the tensor paths'
 *                           conditions fail (tied families, large |E|). */
int game_set_path(game_ctx *ctx, int path);
/* Which path the next fitness call will take for population size P (one of the three above), or -1 if the requested
 * one is unavailable for the loaded dataset. */
int game_resolved_path(const game_ctx *ctx, int P);
/* a1, TENSOR path only: where the fused fitness kernel takes the expansion from (north_star (1)).
 *   GAME_EXPAND_MATERIALIZED  streams the fp16 expansion matrix built once by game_load (L254's hoisting);
 *   GAME_EXPAND_REGENERATED   recomputes each 256-pattern tile of it from X inside the kernel, straight into shared
 *                             memory, with the population's fp16 copy resident there.  Available for the per-feature
 *                             families when P <= 256, F <= 32 and K (padded to 64 per 8 features) <= 576, and for the
 *                             trigonometric family only when max|X| <= pi; otherwise the fitness call fails with
 *                             GAME_ERR_UNSUPPORTED;
 *   GAME_EXPAND_AUTO          (default) the faster of the two as measured on B200: regenerated
 *                             where it is available AND the contraction has >= 8 k-blocks of 64 terms, more than 24
 *                             features, the launch >= 2000 tiles of 256 patterns and P > 32; materialised otherwise.
 * game_resolved_expansion: which of the two a TENSOR-path fitness call on P chromosomes will use, or -1 if the
 * requested one is unavailable. */
int game_set_expansion(game_ctx *ctx, int mode);
int game_resolved_expansion(const game_ctx *ctx, int P);
/* Pattern-sharded runs: the number of patterns of the WHOLE problem (all shards).  GAME_PATH_AUTO then picks the path from
 * it instead of this context's own N, so every shard evaluates in the same tolerance class.  0 = unset. */
int game_set_global_patterns(game_ctx *ctx, long long N_total);

/* a0 + a1: load the dataset and expand it (L254: "calculate the time consuming trigonometric functions
 * only once").  X is N x F row-major fp32, targets N fp32.  Builds the device-resident expansion
 * matrix E (fp32 K x N for the FP32 path, fp16 N x K for the TENSOR path) and rejects NaN/Inf inputs
 * with GAME_ERR_NONFINITE_INPUT (this check synchronises the stream).  X and targets may be freed once
 * the stream has passed this call.  game_load: DEV pointers.  game_load_host: HOST pointers, copied with
 * cudaMemcpyAsync on the context's stream. */
int game_load(game_ctx *ctx, const float *X, const float *targets, long long N);
int game_load_host(game_ctx *ctx, const float *X, const float *targets, long long N);

/* a1-a5: out[p] = error of chromosome p over all N patterns (eq. 2-5, eq. 9-10):
 *   z = sum_k E[n][k] pop[p][k];  y = act(z);  r = t_n - y;  e = r^2 (TMSE: 0 if |r| <= R);
 *   out[p] = mean_n e  (RMSE: sqrt).
 * pop is P x K row-major fp32, out is P fp32.  Asynchronous.  The N x P matrix z never reaches HBM.
 * game_fitness: DEV pointers.  game_fitness_host: HOST pointers; copies pop in, runs, copies out back
 * and synchronises the stream before returning.  Populations of >= 2048 chromosomes on large datasets go up in two (>= 1 MB) or four (>= 8 MB)
 * chunks on a copy stream of the context's own (ordered after the work already on the context's stream), each chunk's
 * kernels starting when it has landed -- pass pinned memory for the upload to overlap; the result is bit-identical to
 * one call (a chromosome's fitness does not depend on its row or on the rest of the population). */
int game_fitness(game_ctx *ctx, const float *pop, int P, float *out);
int game_fitness_host(game_ctx *ctx, const float *pop, int P, float *out);


/* Pattern-sharded evaluation (the paper's future work (iii), L421): when the patterns are split over
 * several contexts -- one per GPU -- each evaluates its shard and the per-chromosome error totals are added across
 * shards (one all-reduce of P doubles per generation) before eq. 4's mean is taken.
 * game_fitness_sums: a1-a5 without the mean: sums[p] = sum over THIS context's patterns of e (eq. 3 / eq. 10), fp64,
 *   in a fixed order.  pop DEV P x K (or NULL: the context's own population, P ignored), sums DEV P doubles.
 *   accumulate != 0: sums[p] += this context's totals (out-of-core evaluation: the chunks of one dataset pass through
 *   the context one after the other and their totals add up in the library, in call order).  Asynchronous on the
 *   context's stream.
 * game_advance: the rest of one generation from the (summed) totals: fit = sums / N_total (root for RMSE), rank (a6),
 *   stop test (a7) and, if apply_operators != 0 and the stop test did not fire, a8-a11 on the context's population
 *   (generation counter + 1).  Every shard calls it with the same totals, seed and parameters and so holds the same
 *   population afterwards, bit for bit (the random numbers are counter-based).  With one shard and N_total = N it
 *   reproduces game_evolve(1) exactly.  sums DEV P doubles.
 *   res != NULL (HOST): synchronises the stream and reports this call (and any asynchronous ones before it).
 *   res == NULL: ASYNCHRONOUS -- nothing waits on the host; the generation counter and the stop flag live on the device
 *   (once the stop test has fired, later asynchronous calls leave the population unchanged), and game_sync collects them.
 * game_sync: synchronises the stream and closes a run of asynchronous game_advance calls: res (HOST, may be NULL) gets
 *   the generations applied since the run began, whether the stop test fired, and the best error / index of the last
 *   evaluation.  Every other call that needs the host-side generation counter does this implicitly.  With NO run open
 *   (no asynchronous game_advance since the last collection) there is nothing to report: res is filled with zeros, and its
 *   best_error / best_index then carry no information (they are not a perfect fit at row 0).
 * An asynchronous run may mix evaluation-only calls (apply_operators == 0, e.g. to log the fitness) with stepping ones:
 *   the operators' random draws are keyed on the number of steps APPLIED, so the trajectory is the one game_evolve gives. */
int game_fitness_sums(game_ctx *ctx, const float *pop, int P, double *sums, int accumulate);
int game_advance(game_ctx *ctx, const double *sums, long long N_total, unsigned long long seed, const game_ga_params *params,
                 int apply_operators, game_result *res);
int game_sync(game_ctx *ctx, game_result *res);
/* Forward pass of ONE chromosome (the paper's test / run use cases, L127-L129): z_out[n] = Out(pat_n),
 * y_out[n] = act(z), over the patterns of the LOADED dataset -- to apply a trained chromosome to other data (a test or
 * run set), game_load that data (into this or a second context of the same family / degree / F) and call this.
 * genes: K fp32, z_out / y_out: N fp32, either may be NULL.  DEV pointers. fp32. */
int game_predict(game_ctx *ctx, const float *genes, float *z_out, float *y_out);
/* The same forward pass on CALLER-SUPPLIED patterns (a trained chromosome applied to a test / run
 * set, L127-L129) without a game_load: X_new is N_new x F row-major fp32 (DEV), expanded on the fly (a1: fp64 term,
 * rounded once to fp32 -- the values game_load would store), z accumulated in fp32 in ascending gene order, so the
 * result equals game_load(X_new) + game_predict bit for bit.  No dataset needs to be loaded; the loaded one, if any,
 * is untouched.  genes K fp32, z_out / y_out N_new fp32 (either may be NULL), all DEV.  Rejects nothing: a NaN
 * feature gives a NaN output for that pattern.  Asynchronous. */
int game_predict_new(game_ctx *ctx, const float *genes, const float *X_new, long long N_new, float *z_out, float *y_out);

/* Figures of merit of a trained chromosome on the loaded dataset (L301).  A pattern is classified as class 1
 * when act(z) > cut and belongs to class 1 when its target > 0.5.  counts (DEV, 4 x int64) = {TP, FP, TN, FN};
 * fom (DEV, 3 x double) = {accuracy (TP+TN)/N, completeness TP/(TP+FN), contamination FP/(FP+TN)}, 0 for an
 * empty denominator.  genes: K fp32 DEV.  fp32 forward pass.  Asynchronous. */
int game_classify(game_ctx *ctx, const float *genes, float cut, long long *counts, double *fom);

/* Install a population (P x K fp32, DEV) instead of the random initial one; resets nothing else.  Measures max|gene|
 * (synchronises the stream): NaN / Inf genes are rejected with GAME_ERR_NONFINITE_INPUT; a population with
 * |gene| > 65504 cannot be an fp16 operand, so GAME_PATH_AUTO evaluates it on the FP32 path and an explicitly requested
 * tensor path fails with GAME_ERR_UNSUPPORTED (nothing is clamped silently).  game_fitness on a caller-supplied
 * population is asynchronous and cannot reject: there a chromosome holding such a gene evaluates to NaN on the tensor
 * paths (and ranks last); game_fitness_host checks and returns GAME_ERR_UNSUPPORTED. */
int game_set_population(game_ctx *ctx, const float *pop, int P);
/* Number of chromosomes of the installed / evolved population, 0 if there is none yet. */
int game_population_size(const game_ctx *ctx);
/* Set the absolute generation counter (checkpoint resume; Philox draws are keyed on it). */
int game_set_generation(game_ctx *ctx, long long generation);

/* The training loop (L217-L220):  [random initial population if none is set, a12]  then up to
 * `generations` x ( fitness a1-a5, rank a6, stop test a7, elitism a8, selection a9, crossover a10,
 * mutation a11 ), then one more fitness + rank so the returned fitness belongs to the returned
 * population (DESIGN G18).  All random decisions come from Philox4x32-10 keyed on
 * (seed; index, index, absolute generation, purpose) -- DESIGN R0-R6 -- so stepping one generation at
 * a time equals one long call, and a CPU implementation of the same rules draws identical numbers.
 * Runs entirely on the device; synchronises the stream before filling *res (HOST, may be NULL).
 * params is a HOST pointer.  params->P must match an installed population, if any. */
int game_evolve(game_ctx *ctx, int generations, unsigned long long seed, const game_ga_params *params,
                game_result *res);

/* Copy out the current population (P x K), its fitness (P) and rank order (P int32, order[0] = best).
 * Any pointer may be NULL.  fit / order are valid after game_evolve.  DEV pointers; asynchronous. */
int game_get_population(game_ctx *ctx, float *pop, float *fit, int *order);
/* HOST pointers; synchronises. */
int game_get_population_host(game_ctx *ctx, float *pop, float *fit, int *order);

/* Individual operators, exposed so each can be checked bit for bit (all DEV pointers, asynchronous):
 * game_rank: order = argsort of (fit, index) ascending, NaN last (a6, DESIGN G20).
 * game_ga_step: next (P x K) from pop (P x K), order and fit for absolute generation `generation`
 *   (a8-a11; fit is read only by roulette selection).
 * game_init_population: a12. */
int game_rank(game_ctx *ctx, const float *fit, int P, int *order);
int game_ga_step(game_ctx *ctx, const game_ga_params *params, unsigned long long seed, long long generation,
                 const int *order, const float *fit, const float *pop, float *next);
int game_init_population(game_ctx *ctx, int init_mode, unsigned long long seed, int P, float *pop);

/* Raw Philox4x32-10 words for n counters (ctr: n x 4 uint32, out: n x 4 uint32, DEV): lets a test
 * compare the device generator with an independent implementation word for word. */
int game_philox(game_ctx *ctx, unsigned long long seed, const unsigned int *ctr, int n, unsigned int *out);

/* game_rank without any device-memory allocation (a6: the "sort by fitness" of the training loop, L217-L220; same key
 * and tie rule as game_rank, DESIGN G20).
 *
 * For callers that cannot allocate on the GPU: game_rank takes its P ints of counting scratch from the driver's
 * stream-ordered allocator on every call, which is not an option in a process whose device memory is wholly owned by
 * another component (a framework's caching allocator, a serving engine that reserved all of HBM at start-up), in a
 * latency-critical loop that must stay off the driver's allocation path, or in a service that forbids driver
 * allocations after set-up so that running out of memory can only happen at start.  This entry point needs no context
 * and calls no cudaMalloc / cudaFree / allocating library routine: its scratch is an array of
 * GAME_RANK_STATIC_MAX_P ints (256 KiB) built into the library image.  Every GPU that loads libgame_b200.so holds that
 * array until the process exits, used or not; hence the modest limit.
 *
 *   fit    DEV  P fp32 errors (lower is better; NaN ranks last, -0 == +0, equal errors by ascending index)
 *   order  DEV  P int32, written: order[0] = index of the best chromosome ... order[P-1] = the worst
 *   cuda_stream  a cudaStream_t of the CURRENT device (0 = legacy default stream); the work is enqueued on it and
 *          the call returns without waiting.  fit and order stay the caller's and must live until the stream has
 *          passed this call.
 * Runs on the device that is current in the calling thread.  The FIRST call on each device also looks up the device
 * address of the built-in array (once per device; a cheap host-side query, no allocation): make that first call
 * during set-up, before any stream capture is begun.
 * 1 <= P <= GAME_RANK_STATIC_MAX_P, else GAME_ERR_INVALID_ARG (use game_rank for larger populations); NULL pointers
 * likewise; CUDA failures give GAME_ERR_CUDA.  game_rank_static_error() returns the text of the calling thread's last
 * failure (HOST string owned by the library, "" after a success).
 * All calls on one GPU share the one array and find in it what the previous call left: each call clears the part it
 * uses first, on its stream.  Calls that can OVERLAP on the same GPU -- different streams with no ordering between
 * them, or several threads -- race on that array and give wrong orders: keep them on one stream or order them with
 * events. */
#define GAME_RANK_STATIC_MAX_P 65536
int game_rank_static(const float *fit, int P, int *order, void *cuda_stream);
const char *game_rank_static_error(void);

/* Measurement aids (kernel timing, launch counter, pipe micro-benchmarks, launch-configuration knobs) are NOT part of this
 * API: they are declared in game_bench.h, which this header does not include. */

#ifdef __cplusplus
}
#endif
#endif
