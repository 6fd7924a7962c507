// Internal declarations shared by the translation units of libgame_b200 (not part of the ABI).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/game.h"
#include "../../include/game_bench.h"   // measurement aids (tuning knobs, kernel timing, micro-benchmarks): not product API

namespace game {

constexpr int SLAB = 128;        // patterns per n-slab: unit of the per-chromosome partial sums
constexpr int FIN_SPLIT = 64;     // CTAs along the slab axis in the two-pass final reduction
constexpr int TC_KBLK = 64;      // fp16 elements per 128-byte swizzled smem row (tensor path k-block)

// Device-resident loop state, so a generation needs no host round trip.
struct DevState {
    int stopped;          // the loop has stopped: later kernels of the loop become no-ops
    int stop_request;     // written by the stop test (a7) inside rank_scatter_kernel; the next ga_step_kernel promotes
                          // it to `stopped`, so no kernel ever tests a flag that its own launch may be writing
    int gens_run;         // evolution steps actually applied
    int evals_done;       // fitness + rank evaluations completed; ga_step derives its generation index from it,
                          // so a captured CUDA graph of the loop needs no per-generation host arguments
    float best_error;
    int best_index;
};

// where a fitness launch left its per-slab sums, when the caller fuses the final reduction with the rank
struct PartialInfo { int n_chunks, Ppad; };

// rank key: (error, index) ascending, NaN as +inf, -0 as +0 (DESIGN G20)
__device__ __forceinline__ unsigned int sort_key(float f)
{
    if (f != f) f = __int_as_float(0x7f800000);
    f += 0.0f;
    unsigned int u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// ---- term order of the TENSOR path's operands ---------------------------------------------------------------
// A contraction does not care in which order its terms are stored as long as both operands agree, so E16 and C16
// use an order that an in-kernel generator can stream: features in groups of 8, one 8-wide chunk (16 bytes of fp16 =
// one swizzle chunk) per (term type, group), the 8 lanes of the chunk being the group's features, TERM TYPE MAJOR:
//     position = (tau * G + i / 8) * 8 + (i % 8),      G = ceil(F / 8) groups, tau = 0 .. T-1 (T = 2d+1 or d+1)
// tau: Chebyshev T_0..T_d in order; trigonometric 1, cos x, sin x, cos 2x, sin 2x, ...  A k-block (8 chunks) is thus a
// fixed run of consecutive term types for ALL groups, so generator threads that each own (pattern row, group) advance
// their recurrences in step, one chunk per term type, with no per-chunk bookkeeping (round 1's group-major order had
// 17 chunks per group straddling k-blocks: ~37 instructions per chunk in one in-order warp).  Features are padded to
// a multiple of 8 (zero genes).  The tied families keep their natural order.  The ABI's order (L105) is untouched:
// only the fp16 copies are permuted, by pop_to_f16_kernel / ga_step_kernel and the expansion kernels.
__host__ __device__ inline bool tc_permuted(int family) { return family == GAME_TRIG || family == GAME_CHEB; }
__host__ __device__ inline int tc_terms_per_feature(int family, int d) { return family == GAME_TRIG ? 2 * d + 1 : d + 1; }
__host__ __device__ inline int tc_num_positions(int family, int d, int F, int K)
{
    return tc_permuted(family) ? ((F + 7) / 8) * 8 * tc_terms_per_feature(family, d) : K;
}
// m = index inside the feature's block in the ABI's order [a_0, a_1..a_d, b_1..b_d]; F = number of features
__host__ __device__ inline int tc_position(int family, int d, int F, int i, int m)
{
    const int G = (F + 7) >> 3;
    const int tau = family == GAME_TRIG ? (m == 0 ? 0 : (m <= d ? 2 * m - 1 : 2 * (m - d))) : m;
    return (tau * G + (i >> 3)) * 8 + (i & 7);
}

// ---- programmatic dependent launch (PDL) -----------------------------------------------------------------------
// The kernels of one generation form a chain of small dependent launches; with the programmatic-stream-serialization
// attribute the next kernel's CTAs are scheduled while the previous kernel drains, and wait (griddepcontrol.wait) only
// where they first touch what the predecessor wrote.  pdl_wait() returns once every prerequisite grid has COMPLETED and
// its writes are visible, so it is always safe; pdl_trigger() lets the dependents be scheduled early.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Where (and how) the tensor paths keep their fp16 copy of a population: written by pop_to_f16_kernel, or directly by
// ga_step_kernel while it builds the next generation (one launch and one pass over the genes less per generation).
struct C16Sink {
    __half *ptr;         // nullptr: no copy wanted
    int Kpad, family, d, F, split;
    float scale;         // 1, or 0.5 for the tanh logistic (exact)
};
// gene k (ABI order) of chromosome p -> its fp16 position(s): round to nearest even.  A gene outside the finite fp16
// range (|gene| > 65504, Inf, NaN) cannot be an operand of the tensor paths: it is stored as NaN, so THAT chromosome's
// fitness comes out NaN (ranked last) instead of being silently clamped; game_set_population / game_fitness_host
// reject such populations up front (GAME_ERR_UNSUPPORTED) or route AUTO to the FP32 path.
// split: rows of 3 Kpad positions [hi | lo | hi], hi = fp16(c), lo = fp16(c - hi) (see expand_kernel)
__device__ __forceinline__ void c16_store(const C16Sink &s, int p, int k, float gene)
{
    const float v = fabsf(gene) <= 65504.f ? gene * s.scale : __int_as_float(0x7fc00000);
    int pos = k;
    if (tc_permuted(s.family)) {              // ABI order k = i*B + m  ->  the tensor path's term order
        const int B = tc_terms_per_feature(s.family, s.d);
        pos = tc_position(s.family, s.d, s.F, k / B, k % B);
    }
    if (!s.split) {
        s.ptr[(long long)p * s.Kpad + pos] = __float2half_rn(v);
    } else {
        __half *row = s.ptr + (long long)p * 3 * s.Kpad;
        const __half hi = __float2half_rn(v);
        row[pos] = hi; row[s.Kpad + pos] = __float2half_rn(v - __half2float(hi)); row[2 * s.Kpad + pos] = hi;
    }
}

struct FitnessCfg {
    int act, err;
    float R;
};

}  // namespace game

struct game_ctx {
    int family = 0, degree = 0, F = 0, K = 0;
    int act = GAME_ACT_SIGMOID, err = GAME_ERR_MSE, path = GAME_PATH_AUTO, expand_mode = GAME_EXPAND_AUTO;
    float R = 0.f;
    cudaStream_t stream = 0;
    int sm_count = 148;
    int device = 0;                                  // the CUDA device this context lives on (current at game_create)
    int tune[GAME_TUNE_COUNT_];                       // game_set_tuning knobs, -1 = automatic
    std::unordered_map<const void *, int> smem_attr;  // kernels whose dynamic-smem opt-in was raised ON THIS DEVICE
    long long N_global = 0;                           // pattern-sharded runs: the global N the AUTO path choice uses

    // dataset (a0/a1)
    long long N = 0, Npad = 0;
    int n_slabs = 0;
    float *X = nullptr;        // N x F copy (kept for game_predict-style regeneration)
    float *t = nullptr;        // Npad, zero padded
    float *ET = nullptr;       // K x Npad fp32, term-major (FP32 path, predict / classify), zero padded; built on first use
    __half *E16 = nullptr;     // Npad256 x Kpad fp16, pattern-major (TENSOR path), zero padded
    __half *E16s = nullptr;    // Npad256 x 3 Kpad fp16: [hi | hi | lo] halves of E (TENSOR_SPLIT path), built on first use
    long long Npad256 = 0;
    int Kpad = 0;              // K rounded up to TC_KBLK
    bool tensor_ok = false;    // E16 built and all |E| <= 2 (TENSOR path)
    bool split_ok = false;     // |E| within the range where the fp16 hi + lo split is exact enough (TENSOR_SPLIT path)
    float x_maxabs = 0.f;      // max |X| of the loaded dataset

    // population / loop state
    int P = 0;
    bool have_pop = false, have_fit = false;
    float pop_maxabs = 0.f;                  // max |gene| of an installed population (game_set_population); evolution keeps it <= max(this, 1)
    long long generation = 0;
    bool loop_open = false;                  // asynchronous game_advance calls pending: DevState counts since gen_base_open
    unsigned int gen_base_open = 0;
    unsigned int noop_evals_open = 0;        // evaluation-only game_advance calls (apply_operators == 0) since the run opened
    float *pop = nullptr, *pop_next = nullptr, *fit = nullptr;
    int *order = nullptr, *rank = nullptr;
    unsigned int *rw = nullptr;              // roulette weights
    unsigned long long *rprefix = nullptr;   // roulette inclusive prefix sums
    size_t pop_cap = 0;                      // capacity in chromosomes of the buffers above
    game::DevState *state = nullptr;
    unsigned int *gbar = nullptr;            // grid-barrier counter of the persistent loop kernel
    unsigned int *ticket = nullptr;          // last-CTA ticket for classify_kernel (lives behind `state`)

    // scratch
    float *partial = nullptr;  // n_chunks x Ppad per-chunk error sums
    size_t partial_cap = 0;
    double *fin2 = nullptr;    // FIN_SPLIT x Ppad partial totals of the two-pass final reduction
    size_t fin2_cap = 0;
    __half *C16 = nullptr;     // Ppad128 x Kpad fp16 population copy (TENSOR path)
    size_t c16_cap = 0;
    __half *C16s = nullptr;    // Ppad x 3 Kpad fp16 [hi | lo | hi] population copy (TENSOR_SPLIT path); padding stays zero
    size_t c16s_cap = 0;
    const float *c16_src = nullptr;   // the fp32 population the fp16 copy currently mirrors (nullptr: none), and how
    int c16_split = 0;
    float c16_scale = 0.f;
    float *stage_pop = nullptr, *stage_fit = nullptr;   // device staging for *_host calls
    size_t stage_cap = 0;
    cudaStream_t copy_stream = nullptr;                 // game_fitness_host on large populations: uploads run here, a chunk ahead of the kernels
    cudaEvent_t copy_ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // [0] entry (context stream), [1..4] chunk uploaded
    void *tmap_E = nullptr, *tmap_C = nullptr;          // host copies of CUtensorMap (TENSOR path)
    void *tmap_Es = nullptr;                            // the same for E16s

    long long launches = 0;
    bool timing = false;
    std::vector<cudaEvent_t> ev;     // start/stop pairs recorded around the dominant kernel
    std::string msg;
};

namespace game {

int fail(game_ctx *ctx, int code, const char *what);
int cuda_fail(game_ctx *ctx, cudaError_t e, const char *where);

#define GAME_CUDA(ctx, call)                                                   \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return game::cuda_fail(ctx, e__, #call);       \
    } while (0)
#define GAME_LAUNCHED(ctx)                                                     \
    do {                                                                       \
        ++(ctx)->launches;                                                     \
        cudaError_t e__ = cudaGetLastError();                                  \
        if (e__ != cudaSuccess) return game::cuda_fail(ctx, e__, "kernel launch"); \
    } while (0)

// brackets the dominant kernel with events when ctx->timing is on
struct KernelTimer {
    game_ctx *c;
    explicit KernelTimer(game_ctx *ctx) : c(ctx)
    {
        if (!c->timing) return;
        cudaEvent_t a, b;
        cudaEventCreate(&a); cudaEventCreate(&b);
        c->ev.push_back(a); c->ev.push_back(b);
        cudaEventRecord(a, c->stream);
    }
    ~KernelTimer() { if (c->timing) cudaEventRecord(c->ev.back(), c->stream); }
};

inline bool pdl_enabled(const game_ctx *c) { return c->tune[GAME_TUNE_PDL] != 0; }   // GAME_TUNE_PDL = 0 turns the attribute off

// Makes the context's device current for the duration of an ABI call (a context belongs to the device that was current
// at game_create; callers may hold contexts on several GPUs in one process) and restores the caller's device afterwards.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const game_ctx *c)
    {
        int cur = -1;
        if (c && cudaGetDevice(&cur) == cudaSuccess && cur != c->device) { prev = cur; cudaSetDevice(c->device); }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Opt a kernel in to `bytes` of dynamic shared memory.  The attribute is per DEVICE (and per function), so the record of
// what has been raised lives in the context -- which is bound to one device -- not in a process-wide static.
inline cudaError_t ensure_smem_attr(game_ctx *c, const void *func, int bytes)
{
    int &have = c->smem_attr[func];
    if (bytes <= have) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

// kernel<<<grid, block, smem, ctx->stream>>>(args...) with the PDL attribute
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, const game_ctx *ctx, Args &&...args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl_enabled(ctx) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// expand.cu
int launch_check_finite(game_ctx *ctx, const float *X, long long nX, const float *t, long long nT, int *flag_dev);
int launch_expand_fp32(game_ctx *ctx);      // X -> ET
int ensure_ET(game_ctx *ctx);               // allocate + build ET on first use (FP32 path, predict, classify)
int launch_max_abs(game_ctx *ctx, const float *v, long long n, int *flag2_dev);   // flag2[0] |= non-finite, flag2[1] = max|v| bits
int launch_predict_new(game_ctx *ctx, const float *genes, const float *X_new, long long N_new, float *z_out, float *y_out);
int launch_expand_fp16(game_ctx *ctx, float *maxabs_dev);   // X -> E16
int launch_expand_split(game_ctx *ctx);                     // X -> E16s
int launch_predict(game_ctx *ctx, const float *genes, float *z_out, float *y_out);
int launch_classify(game_ctx *ctx, const float *genes, float cut, long long *counts, double *fom, unsigned int *ticket);

// fitness_fp32.cu
size_t fitness_partial_floats(const game_ctx *ctx, int P);
int launch_fitness_fp32(game_ctx *ctx, const float *pop, int P, float *out, const DevState *state, PartialInfo *defer);
int launch_finalize(game_ctx *ctx, int n_chunks, int Ppad, int P, float *out, const DevState *state, double *sums = nullptr,
                    bool accumulate = false);
int launch_fit_from_sums(game_ctx *ctx, const double *sums, int P, long long N_total, float *out, const DevState *state);
// a5 tail + a6 + a7 in one go: final reduction of the slab sums, rank, stop test (single CTA when small)
int launch_post(game_ctx *ctx, PartialInfo pi, int P, float *fit, int *rank_scratch, int *order, DevState *state,
                float stop_error);

// fitness_tc.cu
bool tensor_path_built();
int tensor_prepare(game_ctx *ctx);                               // tensor maps etc. after load
int tensor_ensure_E16(game_ctx *ctx);                            // build the materialised fp16 expansion if game_load deferred it
int tensor_expansion(const game_ctx *ctx, int P);                // GAME_EXPAND_MATERIALIZED / _REGENERATED, or -1
int launch_fitness_tensor(game_ctx *ctx, const float *pop, int P, float *out, const DevState *state, PartialInfo *defer,
                          bool split = false);
int tensor_prepare_split(game_ctx *ctx);                         // E16s + its tensor maps, on first use
int tensor_refresh_c16(game_ctx *ctx, const float *pop, int P, bool split, const DevState *state);   // the fp16 copy mirrors `pop`
int tensor_encode_population_map(game_ctx *ctx, bool split, int Ppad);                               // ctx->tmap_C for C16 / C16s

// evolve_persistent.cu: the whole loop as one cooperative kernel, for sub-wave problems
bool persistent_eligible(const game_ctx *ctx, const game_ga_params *gp, int path);
// returns GAME_OK, an error code (> 0), or PERSISTENT_UNAVAILABLE when the cooperative grid cannot be co-resident on the
// device as it is now (nothing was launched: the caller runs the launch-per-kernel loop instead)
constexpr int PERSISTENT_UNAVAILABLE = -1;
int launch_evolve_persistent(game_ctx *ctx, const game_ga_params *gp, unsigned long long seed, int generations, int path);

// ga.cu
int launch_init_population(game_ctx *ctx, int mode, unsigned long long seed, int P, float *pop);
int launch_rank(game_ctx *ctx, const float *fit, int P, int *rank_scratch, int *order, DevState *state,
                float stop_error, bool update_state);
// generation index = gen_base (+ state->evals_done - 1 when state is given: the loop's device-side counter)
int launch_ga_step(game_ctx *ctx, const game_ga_params *gp, unsigned long long seed, unsigned int gen_base,
                   const int *order, const float *fit, const float *pop, float *next, DevState *state,
                   unsigned int *rw, unsigned long long *rprefix, const C16Sink *sink = nullptr);
// the sink a TENSOR / TENSOR_SPLIT fitness call on this context would read (ptr == nullptr when buffers are missing)
C16Sink tensor_sink(const game_ctx *ctx, bool split);
int launch_philox(game_ctx *ctx, unsigned long long seed, const unsigned int *ctr, int n, unsigned int *out);

}  // namespace game
