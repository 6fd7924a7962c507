// The C ABI of libgame_b200 (include/game.h): context management, argument validation and the
// host-side sequencing of the kernels.  No arithmetic of the method happens on the host.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "game_internal.cuh"

namespace game {

int fail(game_ctx *ctx, int code, const char *what)
{
    if (ctx) ctx->msg = what;
    return code;
}

int cuda_fail(game_ctx *ctx, cudaError_t e, const char *where)
{
    if (ctx) {
        ctx->msg = std::string("CUDA error: ") + cudaGetErrorString(e) + " at " + where;
    }
    return e == cudaErrorMemoryAllocation ? GAME_ERR_ALLOC : GAME_ERR_CUDA;
}

template <typename T>
static void dfree(T *&p)
{
    if (p) cudaFree(p);
    p = nullptr;
}

static void free_dataset(game_ctx *c)
{
    dfree(c->X); dfree(c->t); dfree(c->ET); dfree(c->E16); dfree(c->E16s);
    c->N = 0; c->tensor_ok = false; c->split_ok = false; c->have_fit = false;
}

static void free_population(game_ctx *c)
{
    dfree(c->pop); dfree(c->pop_next); dfree(c->fit); dfree(c->order); dfree(c->rank);
    dfree(c->rw); dfree(c->rprefix);
    c->pop_cap = 0; c->have_pop = false; c->have_fit = false; c->P = 0;
}

static int ensure_population(game_ctx *c, int P)
{
    if ((size_t)P <= c->pop_cap) return GAME_OK;
    free_population(c);
    size_t n = (size_t)P * c->K;
    GAME_CUDA(c, cudaMalloc(&c->pop, n * sizeof(float)));
    GAME_CUDA(c, cudaMalloc(&c->pop_next, n * sizeof(float)));
    GAME_CUDA(c, cudaMalloc(&c->fit, (size_t)P * sizeof(float)));
    GAME_CUDA(c, cudaMalloc(&c->order, (size_t)P * sizeof(int)));
    GAME_CUDA(c, cudaMalloc(&c->rank, (size_t)P * sizeof(int)));
    GAME_CUDA(c, cudaMemsetAsync(c->rank, 0, (size_t)P * sizeof(int), c->stream));   // rank kernels keep it zeroed
    GAME_CUDA(c, cudaMalloc(&c->rw, (size_t)P * sizeof(unsigned int)));
    GAME_CUDA(c, cudaMalloc(&c->rprefix, (size_t)P * sizeof(unsigned long long)));
    c->pop_cap = P;
    return GAME_OK;
}

static int ensure_scratch(game_ctx *c, int P)
{
    size_t need = fitness_partial_floats(c, P);
    if (need > c->partial_cap) {
        dfree(c->partial);
        GAME_CUDA(c, cudaMalloc(&c->partial, need * sizeof(float)));
        c->partial_cap = need;
    }
    size_t need2 = (size_t)FIN_SPLIT * ((P + 255) / 256) * 256;
    if (need2 > c->fin2_cap) {
        dfree(c->fin2);
        GAME_CUDA(c, cudaMalloc(&c->fin2, need2 * sizeof(double)));
        c->fin2_cap = need2;
    }
    size_t need16 = (size_t)((P + 255) / 256) * 256 * (size_t)c->Kpad;
    if (c->tensor_ok && need16 > c->c16_cap) {
        dfree(c->C16);
        GAME_CUDA(c, cudaMalloc(&c->C16, need16 * sizeof(__half)));
        GAME_CUDA(c, cudaMemsetAsync(c->C16, 0, need16 * sizeof(__half), c->stream));
        c->c16_cap = need16; c->c16_src = nullptr;
    }
    if (c->split_ok && c->path != GAME_PATH_FP32 && c->path != GAME_PATH_TENSOR && 3 * need16 > c->c16s_cap) {   // AUTO or SPLIT may need it
        dfree(c->C16s);
        GAME_CUDA(c, cudaMalloc(&c->C16s, 3 * need16 * sizeof(__half)));
        GAME_CUDA(c, cudaMemsetAsync(c->C16s, 0, 3 * need16 * sizeof(__half), c->stream));
        c->c16s_cap = 3 * need16; c->c16_src = nullptr;
    }
    return GAME_OK;
}

// own: the population evaluated is the context's own (installed or evolved), whose gene range is known
static int resolve_path(const game_ctx *c, int P, bool own = false)
{
    (void)P;
    // genes beyond the finite fp16 range cannot be tensor-path operands (game_set_population measured them)
    const bool genes_ok = !own || c->pop_maxabs <= 65504.0f;
    bool can_tensor = tensor_path_built() && c->tensor_ok && genes_ok;
    if (c->path == GAME_PATH_FP32) return GAME_PATH_FP32;
    if (c->path == GAME_PATH_TENSOR) return can_tensor ? GAME_PATH_TENSOR : -1;
    const bool can_split = tensor_path_built() && c->split_ok && genes_ok;
    if (c->path == GAME_PATH_TENSOR_SPLIT) return can_split ? GAME_PATH_TENSOR_SPLIT : -1;
    // AUTO: the tensor cores wherever they can be used -- measured on B200 they beat the FFMA kernels at every population
    // size down to P = 8 (N = 2e5, K = 544: 0.05 / 0.14 ms against 0.43 ms; config 1 in the loop: 60.6k against 48.5k
    // generations/s).  Large datasets take the one-pass fp16 form (1e-3 class), small ones -- where a generation is a few
    // microseconds either way -- the split form, which stays in the FP32 path's 1e-5 class.  The FFMA kernels remain for
    // what the tensor paths cannot take (tied families, |E| > 2) and for GAME_PATH_FP32.
    // (a pattern shard decides from the GLOBAL N, game_set_global_patterns, so that all shards share one tolerance class)
    if (can_tensor && (c->N_global > 0 ? c->N_global : c->N) >= 16384) return GAME_PATH_TENSOR;
    if (can_split) return GAME_PATH_TENSOR_SPLIT;
    return GAME_PATH_FP32;
}

static int run_fitness(game_ctx *c, const float *pop, int P, float *out, const DevState *state, PartialInfo *defer = nullptr)
{
    int rc = ensure_scratch(c, P);
    if (rc) return rc;
    int path = resolve_path(c, P, pop == c->pop);
    if (path < 0) return fail(c, GAME_ERR_UNSUPPORTED, "tensor path unavailable for this dataset / population (|E| or |gene| exceeds the fp16 range, or a tied family)");
    if (path == GAME_PATH_TENSOR) return launch_fitness_tensor(c, pop, P, out, state, defer, false);
    if (path == GAME_PATH_TENSOR_SPLIT) return launch_fitness_tensor(c, pop, P, out, state, defer, true);
    return launch_fitness_fp32(c, pop, P, out, state, defer);
}

static int validate_params(game_ctx *c, const game_ga_params *g)
{
    if (!g) return fail(c, GAME_ERR_INVALID_ARG, "params is NULL");
    if (g->P < 2) return fail(c, GAME_ERR_INVALID_ARG, "P must be >= 2");
    if (g->tournament_size < 1) return fail(c, GAME_ERR_INVALID_ARG, "tournament_size must be >= 1");
    if (g->elitism < 0 || g->elitism >= g->P) return fail(c, GAME_ERR_INVALID_ARG, "need 0 <= elitism < P");
    if (g->elite_mode != GAME_ELITE_COPIES_OF_BEST && g->elite_mode != GAME_ELITE_TOP_E)
        return fail(c, GAME_ERR_INVALID_ARG, "bad elite_mode");
    if (g->selection != GAME_SEL_TOURNAMENT && g->selection != GAME_SEL_ROULETTE)
        return fail(c, GAME_ERR_INVALID_ARG, "bad selection");
    if (g->init_mode < 0 || g->init_mode > 2) return fail(c, GAME_ERR_INVALID_ARG, "bad init_mode");
    if (!(g->p_crossover >= 0.f && g->p_crossover <= 1.f) || !(g->p_mutation >= 0.f && g->p_mutation <= 1.f))
        return fail(c, GAME_ERR_INVALID_ARG, "probabilities must be in [0,1]");
    return GAME_OK;
}

// close a run of asynchronous game_advance calls: the device-side counters become the host's
static int close_loop(game_ctx *c, game_result *res)
{
    DevState h{};
    GAME_CUDA(c, cudaMemcpyAsync(&h, c->state, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->loop_open) {
        c->generation += h.gens_run;
        c->loop_open = false;
        // once the stop test has fired the population no longer moves: fit / order describe it
        if (h.stopped || h.stop_request) c->have_fit = true;
    } else {
        h = DevState{};
    }
    if (res) {
        res->generations_run = h.gens_run;
        res->stopped_on_error = (h.stopped || h.stop_request) ? 1 : 0;
        res->best_error = h.best_error;
        res->best_index = h.best_index;
    }
    return GAME_OK;
}
#define GAME_CLOSE_LOOP(c) do { if ((c)->loop_open) { int rc__ = close_loop(c, nullptr); if (rc__) return rc__; } } while (0)

static int load_common(game_ctx *c, const float *X, const float *targets, long long N)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!X || !targets || N < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_load: X, targets must be non-NULL and N >= 1");
    free_dataset(c);                              // also drops have_fit: fit / order described the previous dataset
    dfree(c->partial); c->partial_cap = 0;
    c->c16_src = nullptr;
    // c->N stays 0 (nothing loaded) until everything below has succeeded; every failure frees what was built
    const int n_slabs = (int)((N + SLAB - 1) / SLAB);
    c->n_slabs = n_slabs;
    c->Npad = (long long)n_slabs * SLAB;
    c->Npad256 = ((N + 255) / 256) * 256;
    int *flag = nullptr;
    int h[3] = {0, 0, 0};
    auto body = [&]() -> int {
        GAME_CUDA(c, cudaMalloc(&c->X, (size_t)N * c->F * sizeof(float)));
        GAME_CUDA(c, cudaMalloc(&c->t, (size_t)c->Npad256 * sizeof(float)));
        GAME_CUDA(c, cudaMalloc(&flag, 3 * sizeof(int)));      // [0] non-finite input, [1] max|E| bits, [2] max|X| bits
        GAME_CUDA(c, cudaMemsetAsync(flag, 0, 3 * sizeof(int), c->stream));
        GAME_CUDA(c, cudaMemsetAsync(c->t, 0, (size_t)c->Npad256 * sizeof(float), c->stream));
        GAME_CUDA(c, cudaMemcpyAsync(c->X, X, (size_t)N * c->F * sizeof(float), cudaMemcpyDefault, c->stream));
        GAME_CUDA(c, cudaMemcpyAsync(c->t, targets, (size_t)N * sizeof(float), cudaMemcpyDefault, c->stream));
        c->N = N;                                 // the expansion launchers read it; withdrawn again on failure
        int rc = launch_check_finite(c, c->X, N * c->F, c->t, N, flag);
        if (rc) return rc;
        // The fp16 tile-blocked expansion of the tensor paths (E16) also measures max|E|, which decides whether those paths are
        // offered.  Where that maximum is known without looking -- |cos|, |sin| <= 1 always; |T_m(x)| <= 1 for |x| <= 1 -- E16 is
        // built on FIRST USE instead (tensor_ensure_E16): a run whose fitness calls all regenerate the expansion in the kernel
        // (config 4, and every chunk of the out-of-core driver at such shapes) never pays for the matrix or its 2 N Kpad bytes.
        // The fp32 term-major expansion (ET) is built on first use by the FFMA kernels / game_predict / game_classify (ensure_ET).
        GAME_CUDA(c, cudaMemcpyAsync(h, flag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
        GAME_CUDA(c, cudaStreamSynchronize(c->stream));
        if (h[0]) return fail(c, GAME_ERR_NONFINITE_INPUT, "game_load: X or targets contain NaN/Inf");
        memcpy(&c->x_maxabs, &h[2], sizeof(float));
        const bool bounded = c->family == GAME_TRIG || (c->family == GAME_CHEB && c->x_maxabs <= 1.0f);
        if (!bounded) {
            size_t n16 = (size_t)c->Npad256 * c->Kpad;
            GAME_CUDA(c, cudaMalloc(&c->E16, n16 * sizeof(__half)));
            GAME_CUDA(c, cudaMemsetAsync(c->E16, 0, n16 * sizeof(__half), c->stream));
            rc = launch_expand_fp16(c, reinterpret_cast<float *>(flag + 1));
            if (rc) return rc;
            GAME_CUDA(c, cudaMemcpyAsync(h, flag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
            GAME_CUDA(c, cudaStreamSynchronize(c->stream));
        } else {
            const float one = 1.0f;
            memcpy(&h[1], &one, sizeof(float));
        }
        float mx;
        memcpy(&mx, &h[1], sizeof(float));
        // fp16 rounding is relative: sums over features (tied families) of magnitude ~F would carry an absolute
        // error ~F*2^-11 into z, outside the 1e-3 class, so the tensor path is offered for |E| <= 2 only
        // ... and the tile-blocked expansion is addressed with 32-bit TMA row coordinates (the split form has 3x the rows)
        const bool rows_ok = (double)c->Npad256 * (3.0 * c->Kpad / TC_KBLK) < 2147483647.0;
        c->tensor_ok = mx <= 2.0f && rows_ok;
        // the split form keeps ~22 bits of every value whatever its magnitude (hi + lo), so it only needs the values well
        // inside fp16's range and above its subnormals' grain: |E| <= 1024 (e.g. Chebyshev terms of unnormalised features)
        c->split_ok = mx <= 1024.0f && rows_ok && tc_permuted(c->family);
        if (c->tensor_ok && c->E16) return tensor_prepare(c);
        if (!c->tensor_ok) dfree(c->E16);
        return GAME_OK;
    };
    const int rc = body();
    if (flag) cudaFree(flag);
    if (rc) {
        cudaStreamSynchronize(c->stream);         // nothing may still be writing what is freed
        free_dataset(c);
    }
    return rc;
}

}  // namespace game

using namespace game;

extern "C" {

int game_create(int family, int degree, int F, game_ctx **out)
{
    if (!out) return GAME_ERR_INVALID_ARG;
    *out = nullptr;
    if (family < GAME_TRIG || family > GAME_POLY_TIED || degree < 1 || degree > 32 || F < 1) return GAME_ERR_INVALID_ARG;
    game_ctx *c = new (std::nothrow) game_ctx();
    if (!c) return GAME_ERR_ALLOC;
    c->family = family; c->degree = degree; c->F = F;
    c->K = family == GAME_TRIG ? F * (2 * degree + 1) : family == GAME_CHEB ? F * (degree + 1)
         : family == GAME_TRIG_TIED ? 2 * degree + 1 : degree + 1;
    c->Kpad = ((tc_num_positions(family, degree, F, c->K) + TC_KBLK - 1) / TC_KBLK) * TC_KBLK;
    for (int &t : c->tune) t = -1;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    c->device = dev;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaMalloc(&c->state, sizeof(DevState) + 16);
    if (e == cudaSuccess) e = cudaMemset(c->state, 0, sizeof(DevState) + 16);
    c->ticket = reinterpret_cast<unsigned int *>(c->state + 1);
    if (e != cudaSuccess) {       // no CPU fallback: without a device there is no context
        cudaGetLastError();
        delete c;
        return GAME_ERR_CUDA;
    }
    *out = c;
    return GAME_OK;
}

void game_destroy(game_ctx *c)
{
    if (!c) return;
    DeviceGuard dg(c);
    cudaStreamSynchronize(c->stream);
    free_dataset(c);
    free_population(c);
    dfree(c->partial); dfree(c->fin2); dfree(c->C16); dfree(c->C16s); dfree(c->stage_pop); dfree(c->stage_fit); dfree(c->state);
    dfree(c->gbar);
    free(c->tmap_E); free(c->tmap_C); free(c->tmap_Es);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (cudaEvent_t e : c->copy_ev) if (e) cudaEventDestroy(e);
    delete c;
}

int game_num_terms(const game_ctx *c) { return c ? c->K : -1; }
long long game_generation(const game_ctx *cc)
{
    if (!cc) return -1;
    game_ctx *c = const_cast<game_ctx *>(cc);
    if (c->loop_open) { DeviceGuard dg(c); if (close_loop(c, nullptr)) return -1; }   // asynchronous advances pending
    return c->generation;
}
int game_population_size(const game_ctx *c) { return (c && c->have_pop) ? c->P : 0; }
const char *game_last_error(const game_ctx *c) { return c ? c->msg.c_str() : "null context"; }
long long game_launch_count(const game_ctx *c) { return c ? c->launches : -1; }

int game_set_stream(game_ctx *c, void *s)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    c->stream = (cudaStream_t)s;
    return GAME_OK;
}

int game_set_activation(game_ctx *c, int act)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (act != GAME_ACT_SIGMOID && act != GAME_ACT_IDENTITY) return fail(c, GAME_ERR_INVALID_ARG, "bad activation");
    c->act = act;
    c->have_fit = false;
    return GAME_OK;
}

int game_set_error(game_ctx *c, int err, float R)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (err != GAME_ERR_MSE && err != GAME_ERR_TMSE && err != GAME_ERR_RMSE) return fail(c, GAME_ERR_INVALID_ARG, "bad error type");
    if (err == GAME_ERR_TMSE && !(R > 0.f && R < 1.f)) return fail(c, GAME_ERR_INVALID_ARG, "TMSE threshold R must be in (0,1)");
    c->err = err; c->R = R;
    c->have_fit = false;
    return GAME_OK;
}

int game_set_path(game_ctx *c, int path)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (path < GAME_PATH_AUTO || path > GAME_PATH_TENSOR_SPLIT) return fail(c, GAME_ERR_INVALID_ARG, "bad path");
    c->path = path;
    return GAME_OK;
}

int game_resolved_path(const game_ctx *c, int P) { return c ? resolve_path(c, P, c->have_pop && P == c->P) : -1; }

int game_set_tuning(game_ctx *c, int knob, int value)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (knob < 0 || knob >= GAME_TUNE_COUNT_) return fail(c, GAME_ERR_INVALID_ARG, "game_set_tuning: unknown knob");
    static const int lo[GAME_TUNE_COUNT_] = {0, 1, 0, 0, 0, 0, 0, 0}, hi[GAME_TUNE_COUNT_] = {1, 2, 2, 1, 1, 1, 2, 8};
    if (value != -1 && (value < lo[knob] || value > hi[knob] || (knob == GAME_TUNE_SIGMOID && value == 1)))
        return fail(c, GAME_ERR_INVALID_ARG, "game_set_tuning: value out of range for this knob");
    c->tune[knob] = value;
    return GAME_OK;
}

int game_set_global_patterns(game_ctx *c, long long N_total)
{
    if (!c || N_total < 0) return GAME_ERR_INVALID_ARG;
    c->N_global = N_total;
    return GAME_OK;
}

int game_set_expansion(game_ctx *c, int mode)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (mode < GAME_EXPAND_AUTO || mode > GAME_EXPAND_REGENERATED) return fail(c, GAME_ERR_INVALID_ARG, "bad expansion mode");
    c->expand_mode = mode;
    return GAME_OK;
}

int game_resolved_expansion(const game_ctx *c, int P) { return (c && c->N && P >= 1) ? tensor_expansion(c, P) : -1; }

int game_load(game_ctx *c, const float *X, const float *t, long long N) { DeviceGuard dg(c); return load_common(c, X, t, N); }
int game_load_host(game_ctx *c, const float *X, const float *t, long long N) { DeviceGuard dg(c); return load_common(c, X, t, N); }

int game_fitness(game_ctx *c, const float *pop, int P, float *out)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_fitness before game_load");
    if (!pop || !out || P < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_fitness: pop/out NULL or P < 1");
    DeviceGuard dg(c);
    return run_fitness(c, pop, P, out, nullptr);
}

int game_fitness_host(game_ctx *c, const float *pop, int P, float *out)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_fitness_host before game_load");
    if (!pop || !out || P < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_fitness_host: pop/out NULL or P < 1");
    DeviceGuard dg(c);
    if ((size_t)P > c->stage_cap) {
        dfree(c->stage_pop); dfree(c->stage_fit);
        c->stage_cap = 0;
        GAME_CUDA(c, cudaMalloc(&c->stage_pop, (size_t)P * c->K * sizeof(float)));
        GAME_CUDA(c, cudaMalloc(&c->stage_fit, ((size_t)P + 2) * sizeof(float)));     // + the two gene-range words
        c->stage_cap = P;
    }
    int *range = reinterpret_cast<int *>(c->stage_fit + P);
    // Large populations go up in chunks on a copy stream, each chunk's kernels starting as soon as it has landed: the
    // upload (27 MB at config 5, ~1.1 ms over PCIe) hides behind the evaluation of the chunks before it.  A chromosome's
    // fitness does not depend on its row or on the rest of the population (DESIGN P20), so the chunks give the bits one call
    // would; they are used only when a chunk takes the same path and launch configuration class as the whole population.
    // How many chunks: every chunk repeats the small launches of a call, so a 1.8 MB population (config 3) goes up in two
    // (242 us per call against 270 in one piece; four measured slower than one there), 8 MB and more in four.
    const size_t pop_bytes = (size_t)P * c->K * sizeof(float);
    const int want = pop_bytes >= ((size_t)8 << 20) ? 4 : pop_bytes >= ((size_t)1 << 20) ? 2 : 1;
    const int Pc = (((P + want - 1) / want + 255) / 256) * 256;
    // (a chunk must also be well above one wave of tiles, or the tensor path would switch to its half-size tiles for it)
    // The same must hold for the ragged LAST chunk (it can be as short as one row, which would run single CTAs, the resident
    // tile or half tiles, and could resolve AUTO's expansion differently): a tail that fails the test is folded into the
    // chunk before it.
    auto same_class = [&](int n) {
        return n >= 1024 && resolve_path(c, n) == resolve_path(c, P) &&
               (c->Npad256 / 256) * (long long)(n / 128) >= 2LL * c->sm_count &&
               (resolve_path(c, P) != GAME_PATH_TENSOR || tensor_expansion(c, n) == tensor_expansion(c, P));
    };
    int cstart[8], ccount[8], nch = 0;
    for (int p0 = 0; p0 < P && nch < 8; p0 += Pc, ++nch) { cstart[nch] = p0; ccount[nch] = P - p0 < Pc ? P - p0 : Pc; }
    if (nch >= 2 && !same_class(ccount[nch - 1])) { ccount[nch - 2] += ccount[nch - 1]; --nch; }
    const bool chunked = want > 1 && P >= 2048 && nch >= 2 && same_class(Pc);
    int rc = GAME_OK;
    if (!chunked) {
        GAME_CUDA(c, cudaMemcpyAsync(c->stage_pop, pop, (size_t)P * c->K * sizeof(float), cudaMemcpyHostToDevice, c->stream));
        GAME_CUDA(c, cudaMemsetAsync(range, 0, 2 * sizeof(int), c->stream));
        rc = launch_max_abs(c, c->stage_pop, (long long)P * c->K, range);
        if (!rc) rc = run_fitness(c, c->stage_pop, P, c->stage_fit, nullptr);
    } else {
        if (!c->copy_stream) {
            GAME_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
            for (cudaEvent_t &e : c->copy_ev) GAME_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        }
        GAME_CUDA(c, cudaEventRecord(c->copy_ev[0], c->stream));            // earlier work on the context's stream may still read the staging area
        GAME_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->copy_ev[0], 0));
        for (int i = 0; i < nch; ++i) {
            const int p0 = cstart[i], n = ccount[i];
            GAME_CUDA(c, cudaMemcpyAsync(c->stage_pop + (size_t)p0 * c->K, pop + (size_t)p0 * c->K, (size_t)n * c->K * sizeof(float),
                                         cudaMemcpyHostToDevice, c->copy_stream));
            GAME_CUDA(c, cudaEventRecord(c->copy_ev[1 + i], c->copy_stream));
        }
        GAME_CUDA(c, cudaMemsetAsync(range, 0, 2 * sizeof(int), c->stream));
        for (int i = 0; i < nch && !rc; ++i) {
            const int p0 = cstart[i], n = ccount[i];
            GAME_CUDA(c, cudaStreamWaitEvent(c->stream, c->copy_ev[1 + i], 0));
            rc = launch_max_abs(c, c->stage_pop + (size_t)p0 * c->K, (long long)n * c->K, range);
            if (!rc) rc = run_fitness(c, c->stage_pop + (size_t)p0 * c->K, n, c->stage_fit + p0, nullptr);
        }
    }
    if (rc) return rc;
    int hr[2] = {0, 0};
    GAME_CUDA(c, cudaMemcpyAsync(out, c->stage_fit, (size_t)P * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    GAME_CUDA(c, cudaMemcpyAsync(hr, range, sizeof(hr), cudaMemcpyDeviceToHost, c->stream));
    GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    float mx;
    memcpy(&mx, &hr[1], sizeof(float));
    if ((hr[0] || mx > 65504.0f) && resolve_path(c, P) != GAME_PATH_FP32)
        return fail(c, GAME_ERR_UNSUPPORTED, "game_fitness_host: genes outside the finite fp16 range (|gene| > 65504 or NaN/Inf) "
                                             "cannot be evaluated on a tensor path; use GAME_PATH_FP32");
    return GAME_OK;
}

int game_fitness_sums(game_ctx *c, const float *pop, int P, double *sums, int accumulate)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_fitness_sums before game_load");
    DeviceGuard dg(c);
    if (!pop) {                                   // the context's own population
        if (!c->have_pop) return fail(c, GAME_ERR_NOT_LOADED, "game_fitness_sums: no population yet");
        pop = c->pop; P = c->P;
    }
    if (!sums || P < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_fitness_sums: sums NULL or P < 1");
    PartialInfo pi{};
    int rc = run_fitness(c, pop, P, nullptr, nullptr, &pi);
    if (rc) return rc;
    return launch_finalize(c, pi.n_chunks, pi.Ppad, P, nullptr, nullptr, sums, accumulate != 0);
}

int game_advance(game_ctx *c, const double *sums, long long N_total, unsigned long long seed, const game_ga_params *gp,
                 int apply_operators, game_result *res)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    int rc = validate_params(c, gp);
    if (rc) return rc;
    if (!c->have_pop || c->P != gp->P) return fail(c, GAME_ERR_NOT_LOADED, "game_advance: no population of params->P chromosomes installed");
    if (!sums || N_total < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_advance: sums NULL or N_total < 1");
    DeviceGuard dg(c);
    const int P = gp->P;
    if (!c->loop_open) {
        // a run of advances shares ONE device-side state: evaluations done, generations applied and the stop flag live
        // there, so an asynchronous call needs nothing from the host (ga_step_kernel derives its generation index from
        // gen_base_open + evals_done - 1, as the game_evolve loop does)
        GAME_CUDA(c, cudaMemsetAsync(c->state, 0, sizeof(DevState), c->stream));
        c->gen_base_open = (unsigned int)c->generation;
        c->noop_evals_open = 0;
        c->loop_open = true;
    }
    rc = launch_fit_from_sums(c, sums, P, N_total, c->fit, c->state);                              // a5 tail
    if (!rc) rc = launch_rank(c, c->fit, P, c->rank, c->order, c->state, gp->stop_error, true);    // a6, a7
    if (rc) return rc;
    if (apply_operators) {                                                                          // a8-a11
        const int path = resolve_path(c, P, true);
        // the operators also write the next fitness call's fp16 copy: size it for THIS population first (the sums may come
        // from elsewhere, so no fitness call of this context need have seen P chromosomes yet)
        if (c->N > 0) { rc = ensure_scratch(c, P); if (rc) return rc; }
        C16Sink sink = tensor_sink(c, path == GAME_PATH_TENSOR_SPLIT);
        const size_t need16 = (size_t)((P + 255) / 256) * 256 * (size_t)c->Kpad;
        const bool sink_fits = sink.split ? c->c16s_cap >= 3 * need16 : c->c16_cap >= need16;
        const bool with_sink = (path == GAME_PATH_TENSOR || path == GAME_PATH_TENSOR_SPLIT) && sink.ptr != nullptr && sink_fits && c->N > 0;
        // generation key of the operators = gen_base + (evaluations done - 1) on the device; evaluation-only calls inside this
        // run (apply_operators == 0) count as evaluations but apply nothing, so the base steps back by their number
        rc = launch_ga_step(c, gp, seed, c->gen_base_open - c->noop_evals_open, c->order, c->fit, c->pop, c->pop_next, c->state, c->rw,
                            c->rprefix, with_sink ? &sink : nullptr);
        if (rc) return rc;
        float *tmp = c->pop; c->pop = c->pop_next; c->pop_next = tmp;
        c->c16_src = with_sink ? c->pop : nullptr; c->c16_split = sink.split; c->c16_scale = sink.scale;
        c->have_fit = false;       // (if the stop test fired the population did not move, but the host cannot know yet)
    } else {
        c->have_fit = true;
        ++c->noop_evals_open;
    }
    if (!res) return GAME_OK;      // asynchronous: game_sync (or any call that needs the counters) collects later
    return close_loop(c, res);
}

int game_sync(game_ctx *c, game_result *res)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    DeviceGuard dg(c);
    return close_loop(c, res);
}

int game_predict(game_ctx *c, const float *genes, float *z_out, float *y_out)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_predict before game_load");
    if (!genes) return fail(c, GAME_ERR_INVALID_ARG, "game_predict: genes is NULL");
    DeviceGuard dg(c);
    return launch_predict(c, genes, z_out, y_out);
}

int game_predict_new(game_ctx *c, const float *genes, const float *X_new, long long N_new, float *z_out, float *y_out)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!genes || !X_new || N_new < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_predict_new: genes / X_new NULL or N_new < 1");
    DeviceGuard dg(c);
    return launch_predict_new(c, genes, X_new, N_new, z_out, y_out);
}

int game_classify(game_ctx *c, const float *genes, float cut, long long *counts, double *fom)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_classify before game_load");
    if (!genes || !counts || !fom) return fail(c, GAME_ERR_INVALID_ARG, "game_classify: NULL pointer");
    DeviceGuard dg(c);
    return launch_classify(c, genes, cut, counts, fom, c->ticket);
}

int game_set_population(game_ctx *c, const float *pop, int P)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!pop || P < 2) return fail(c, GAME_ERR_INVALID_ARG, "game_set_population: pop NULL or P < 2");
    DeviceGuard dg(c);
    GAME_CLOSE_LOOP(c);
    int rc;
    if ((size_t)P > c->pop_cap && c->have_pop) {
        // growing means reallocating, which frees the installed population: check the newcomer in a buffer of its own first,
        // so that a rejected one (NaN / Inf genes, genes too large for the requested tensor path) leaves the old one in place
        float *probe = nullptr;
        const size_t n = (size_t)P * c->K;
        GAME_CUDA(c, cudaMalloc(&probe, (n + 2) * sizeof(float)));
        int *prange = reinterpret_cast<int *>(probe + n);
        int hp[2] = {0, 0};
        cudaError_t e = cudaMemcpyAsync(probe, pop, n * sizeof(float), cudaMemcpyDefault, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(prange, 0, 2 * sizeof(int), c->stream);
        rc = e == cudaSuccess ? launch_max_abs(c, probe, (long long)n, prange) : cuda_fail(c, e, "game_set_population: staging copy");
        if (!rc) {
            e = cudaMemcpyAsync(hp, prange, sizeof(hp), cudaMemcpyDeviceToHost, c->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
            if (e != cudaSuccess) rc = cuda_fail(c, e, "game_set_population: staging check");
        }
        cudaFree(probe);
        if (rc) return rc;
        float pmx;
        memcpy(&pmx, &hp[1], sizeof(float));
        if (hp[0]) return fail(c, GAME_ERR_NONFINITE_INPUT, "game_set_population: genes contain NaN/Inf");
        if (pmx > 65504.0f && (c->path == GAME_PATH_TENSOR || c->path == GAME_PATH_TENSOR_SPLIT))
            return fail(c, GAME_ERR_UNSUPPORTED, "game_set_population: |gene| > 65504 cannot be an fp16 operand of the requested tensor path; "
                                                 "use GAME_PATH_FP32 or GAME_PATH_AUTO");
    }
    rc = ensure_population(c, P);
    if (rc) return rc;
    // gene range first (into the spare buffer): a rejected population leaves the installed one untouched
    int *range = reinterpret_cast<int *>(c->rank);          // P >= 2 ints, zero between uses (the rank kernels keep it so)
    GAME_CUDA(c, cudaMemcpyAsync(c->pop_next, pop, (size_t)P * c->K * sizeof(float), cudaMemcpyDefault, c->stream));
    rc = launch_max_abs(c, c->pop_next, (long long)P * c->K, range);
    if (rc) return rc;
    int hr[2] = {0, 0};
    GAME_CUDA(c, cudaMemcpyAsync(hr, range, sizeof(hr), cudaMemcpyDeviceToHost, c->stream));
    GAME_CUDA(c, cudaMemsetAsync(range, 0, 2 * sizeof(int), c->stream));
    GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    if (hr[0]) return fail(c, GAME_ERR_NONFINITE_INPUT, "game_set_population: genes contain NaN/Inf");
    float mx;
    memcpy(&mx, &hr[1], sizeof(float));
    if (mx > 65504.0f && (c->path == GAME_PATH_TENSOR || c->path == GAME_PATH_TENSOR_SPLIT))
        return fail(c, GAME_ERR_UNSUPPORTED, "game_set_population: |gene| > 65504 cannot be an fp16 operand of the requested tensor path; "
                                             "use GAME_PATH_FP32 or GAME_PATH_AUTO");
    float *tmp = c->pop; c->pop = c->pop_next; c->pop_next = tmp;
    c->pop_maxabs = mx;
    c->P = P; c->have_pop = true; c->have_fit = false; c->c16_src = nullptr;
    return GAME_OK;
}

int game_set_generation(game_ctx *c, long long g)
{
    if (!c || g < 0) return GAME_ERR_INVALID_ARG;
    DeviceGuard dg(c);
    GAME_CLOSE_LOOP(c);
    c->generation = g;
    return GAME_OK;
}

int game_evolve(game_ctx *c, int generations, unsigned long long seed, const game_ga_params *gp, game_result *res)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->N) return fail(c, GAME_ERR_NOT_LOADED, "game_evolve before game_load");
    int rc = validate_params(c, gp);
    if (rc) return rc;
    if (generations < 0) return fail(c, GAME_ERR_INVALID_ARG, "generations < 0");
    if (c->have_pop && c->P != gp->P) return fail(c, GAME_ERR_INVALID_ARG, "params->P differs from the installed population");
    DeviceGuard dg(c);
    GAME_CLOSE_LOOP(c);
    const int P = gp->P;
    if (!c->have_pop) {
        rc = ensure_population(c, P);
        if (rc) return rc;
        rc = launch_init_population(c, gp->init_mode, seed, P, c->pop);     // a12
        if (rc) return rc;
        c->P = P; c->have_pop = true; c->c16_src = nullptr; c->pop_maxabs = 1.0f;
    }
    if (resolve_path(c, P, true) < 0)
        return fail(c, GAME_ERR_UNSUPPORTED, "tensor path unavailable for this dataset / population (|E| or |gene| exceeds the fp16 range, or a tied family)");
    GAME_CUDA(c, cudaMemsetAsync(c->state, 0, sizeof(DevState), c->stream));
    DevState h{};
    {
        // Sub-wave problems (configs 1-2): the whole loop -- fitness tiles, rank, stop test, operators, `generations` times,
        // plus the final evaluation -- as ONE persistent cooperative kernel with grid barriers between the phases
        // (evolve_persistent.cu).  Bit-identical to the launch-per-kernel path below.
        const int path0 = resolve_path(c, P, true);
        const bool ran_persistent = persistent_eligible(c, gp, path0);
        if (ran_persistent) {
            const bool split = path0 == GAME_PATH_TENSOR_SPLIT;
            rc = ensure_scratch(c, P);
            if (!rc) rc = tensor_refresh_c16(c, c->pop, P, split, nullptr);
            if (!rc) rc = launch_evolve_persistent(c, gp, seed, generations, path0);
            if (rc > 0) return rc;
        }
        // (rc == PERSISTENT_UNAVAILABLE: the cooperative grid cannot be co-resident on this device right now; nothing ran, and
        // the launch-per-kernel loop below gives the same bits)
        if (ran_persistent && rc == GAME_OK) {
            const bool split = path0 == GAME_PATH_TENSOR_SPLIT;
            GAME_CUDA(c, cudaMemcpyAsync(&h, c->state, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
            GAME_CUDA(c, cudaStreamSynchronize(c->stream));
            if (h.gens_run & 1) { float *tmp = c->pop; c->pop = c->pop_next; c->pop_next = tmp; }
            const C16Sink sink = tensor_sink(c, split);
            c->c16_src = c->pop; c->c16_split = sink.split; c->c16_scale = sink.scale;     // the operators kept the fp16 copy current
            c->generation += h.gens_run;
            c->have_fit = true;
            if (res) {
                res->generations_run = h.gens_run;
                res->stopped_on_error = (h.stopped || h.stop_request) ? 1 : 0;
                res->best_error = h.best_error;
                res->best_index = h.best_index;
            }
            return GAME_OK;
        }
        rc = GAME_OK;
    }
    const bool can_stop = gp->stop_error >= 0.f;
    const unsigned int gen_base = (unsigned int)c->generation;      // the device adds its own evaluation counter
    auto evaluate = [&]() -> int {                                   // a1-a5, then a5 tail + a6 + a7
        PartialInfo pi{};
        int r = run_fitness(c, c->pop, P, c->fit, c->state, &pi);
        if (r) return r;
        return launch_post(c, pi, P, c->fit, c->rank, c->order, c->state, gp->stop_error);
    };
    auto generation = [&]() -> int {
        int r = evaluate();
        if (r) return r;
        // a8-a11; on the tensor paths the operators also write the fp16 copy the next evaluation contracts against
        const int path = resolve_path(c, P, true);
        C16Sink sink = tensor_sink(c, path == GAME_PATH_TENSOR_SPLIT);
        const bool with_sink = (path == GAME_PATH_TENSOR || path == GAME_PATH_TENSOR_SPLIT) && sink.ptr != nullptr;
        r = launch_ga_step(c, gp, seed, gen_base, c->order, c->fit, c->pop, c->pop_next, c->state, c->rw, c->rprefix,
                           with_sink ? &sink : nullptr);
        if (r) return r;
        float *tmp = c->pop; c->pop = c->pop_next; c->pop_next = tmp;
        c->c16_src = with_sink ? c->pop : nullptr; c->c16_split = sink.split; c->c16_scale = sink.scale;
        return GAME_OK;
    };
    auto stopped_now = [&](bool &stop) -> int {                      // poll the device-side stop flag
        GAME_CUDA(c, cudaMemcpyAsync(&h, c->state, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
        GAME_CUDA(c, cudaStreamSynchronize(c->stream));
        stop = h.stopped || h.stop_request;
        return GAME_OK;
    };
    int g = 0;
    bool stop = false;
    const bool capturable = c->stream != nullptr && c->stream != cudaStreamLegacy && c->stream != cudaStreamPerThread;
    if (generations >= 8 && !c->timing && capturable) {
        // Launch-latency matters for small problems: capture TWO generations (the population buffers swap
        // back after two) into a CUDA graph and replay it.  Nothing in the captured kernels depends on host
        // arguments that change per generation: the generation index and the stop flag live on the device.
        rc = generation();                     // outside the graph: sets kernel attributes, sizes scratch
        if (rc) return rc;
        g = 1;
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        const long long before = c->launches;
        GAME_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        rc = generation();
        if (!rc) rc = generation();
        cudaError_t ce = cudaStreamEndCapture(c->stream, &graph);
        const long long per_graph = c->launches - before;
        c->launches = before;
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (ce != cudaSuccess) return cuda_fail(c, ce, "cudaStreamEndCapture");
        ce = cudaGraphInstantiate(&exec, graph, 0);
        if (ce != cudaSuccess) { cudaGraphDestroy(graph); return cuda_fail(c, ce, "cudaGraphInstantiate"); }
        for (int rep = 0; g + 2 <= generations && !stop; ++rep) {
            ce = cudaGraphLaunch(exec, c->stream);
            if (ce != cudaSuccess) break;
            c->launches += per_graph;
            g += 2;
            if (can_stop && (rep & 15) == 15) { rc = stopped_now(stop); if (rc) break; }
        }
        cudaGraphExecDestroy(exec);
        cudaGraphDestroy(graph);
        if (ce != cudaSuccess) return cuda_fail(c, ce, "cudaGraphLaunch");
        if (rc) return rc;
    }
    for (; g < generations && !stop; ++g) {
        rc = generation();
        if (rc) return rc;
        if (can_stop && (g & 31) == 31) { rc = stopped_now(stop); if (rc) return rc; }
    }
    rc = evaluate();                           // the returned fitness belongs to the returned population (G18)
    if (rc) return rc;
    GAME_CUDA(c, cudaMemcpyAsync(&h, c->state, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    c->generation += h.gens_run;
    c->have_fit = true;
    if (res) {
        res->generations_run = h.gens_run;
        res->stopped_on_error = (h.stopped || h.stop_request) ? 1 : 0;
        res->best_error = h.best_error;
        res->best_index = h.best_index;
    }
    return GAME_OK;
}

static int get_population(game_ctx *c, float *pop, float *fit, int *order, bool sync)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!c->have_pop) return fail(c, GAME_ERR_NOT_LOADED, "no population yet");
    DeviceGuard dg(c);
    GAME_CLOSE_LOOP(c);
    if ((fit || order) && !c->have_fit) return fail(c, GAME_ERR_NOT_LOADED, "fitness / order are only valid after game_evolve");
    if (pop) GAME_CUDA(c, cudaMemcpyAsync(pop, c->pop, (size_t)c->P * c->K * sizeof(float), cudaMemcpyDefault, c->stream));
    if (fit) GAME_CUDA(c, cudaMemcpyAsync(fit, c->fit, (size_t)c->P * sizeof(float), cudaMemcpyDefault, c->stream));
    if (order) GAME_CUDA(c, cudaMemcpyAsync(order, c->order, (size_t)c->P * sizeof(int), cudaMemcpyDefault, c->stream));
    if (sync) GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    return GAME_OK;
}

int game_get_population(game_ctx *c, float *pop, float *fit, int *order) { return get_population(c, pop, fit, order, false); }
int game_get_population_host(game_ctx *c, float *pop, float *fit, int *order) { return get_population(c, pop, fit, order, true); }

int game_rank(game_ctx *c, const float *fit, int P, int *order)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!fit || !order || P < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_rank: NULL pointer or P < 1");
    DeviceGuard dg(c);
    int *scratch = nullptr;
    GAME_CUDA(c, cudaMallocAsync(&scratch, (size_t)P * sizeof(int), c->stream));
    GAME_CUDA(c, cudaMemsetAsync(scratch, 0, (size_t)P * sizeof(int), c->stream));
    int rc = launch_rank(c, fit, P, scratch, order, nullptr, -1.f, false);
    cudaFreeAsync(scratch, c->stream);
    return rc;
}

int game_ga_step(game_ctx *c, const game_ga_params *gp, unsigned long long seed, long long generation, const int *order,
                 const float *fit, const float *pop, float *next)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    int rc = validate_params(c, gp);
    if (rc) return rc;
    if (!order || !pop || !next || generation < 0) return fail(c, GAME_ERR_INVALID_ARG, "game_ga_step: NULL pointer or generation < 0");
    if (gp->selection == GAME_SEL_ROULETTE && !fit) return fail(c, GAME_ERR_INVALID_ARG, "roulette selection needs fit");
    DeviceGuard dg(c);
    unsigned int *rw = nullptr;
    unsigned long long *rp = nullptr;
    if (gp->selection == GAME_SEL_ROULETTE) {
        GAME_CUDA(c, cudaMallocAsync(&rw, (size_t)gp->P * sizeof(unsigned int), c->stream));
        GAME_CUDA(c, cudaMallocAsync(&rp, (size_t)gp->P * sizeof(unsigned long long), c->stream));
    }
    rc = launch_ga_step(c, gp, seed, (unsigned int)generation, order, fit, pop, next, nullptr, rw, rp);
    if (rw) cudaFreeAsync(rw, c->stream);
    if (rp) cudaFreeAsync(rp, c->stream);
    return rc;
}

int game_init_population(game_ctx *c, int mode, unsigned long long seed, int P, float *pop)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!pop || P < 1 || mode < 0 || mode > 2) return fail(c, GAME_ERR_INVALID_ARG, "game_init_population: bad argument");
    DeviceGuard dg(c);
    return launch_init_population(c, mode, seed, P, pop);
}

int game_set_kernel_timing(game_ctx *c, int enabled)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    c->timing = enabled != 0;
    return GAME_OK;
}

int game_get_kernel_timing(game_ctx *c, double *total_ms, long long *launches)
{
    if (!c || !total_ms || !launches) return GAME_ERR_INVALID_ARG;
    DeviceGuard dg(c);
    GAME_CUDA(c, cudaStreamSynchronize(c->stream));
    double tot = 0.0;
    for (size_t i = 0; i + 1 < c->ev.size(); i += 2) {
        float ms = 0.f;
        GAME_CUDA(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        tot += ms;
    }
    *total_ms = tot;
    *launches = (long long)(c->ev.size() / 2);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    return GAME_OK;
}

int game_philox(game_ctx *c, unsigned long long seed, const unsigned int *ctr, int n, unsigned int *out)
{
    if (!c) return GAME_ERR_INVALID_ARG;
    if (!ctr || !out || n < 1) return fail(c, GAME_ERR_INVALID_ARG, "game_philox: bad argument");
    DeviceGuard dg(c);
    return launch_philox(c, seed, ctr, n, out);
}

}  // extern "C"
