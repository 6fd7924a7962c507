// a6-a12: the GA-operator kernels -- rank, stop test, elitism, selection, crossover, mutation and the
// initial population.  The paper runs these on the host
// (L357, and lists moving them to the GPU as future work, L421); here they are device kernels so a
// generation never leaves the GPU.  Every random decision is integer arithmetic on Philox4x32-10 words
// keyed on (seed; primary, secondary, absolute generation, purpose) -- DESIGN R0-R6 -- so that a CPU
// implementation of the same rules reproduces the population bit for bit.
#include "ga_device.cuh"

namespace game {

// ---- a12: initial population (R1, R2) ---------------------------------------------------------------
__global__ void init_population_kernel(int mode, unsigned long long seed, int P, int K, float *__restrict__ pop)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= (long long)P * K) return;
    uint32_t p = (uint32_t)(i / K), k = (uint32_t)(i % K);
    float g;
    if (mode == GAME_INIT_NORMAL_PM1) {
        uint32_t S = 0;
#pragma unroll
        for (uint32_t j = 0; j < 3; ++j) {
            W4 w = draw(seed, k, p, j, TAG_INIT);
            S += (w.x >> 8) + (w.y >> 8) + (w.z >> 8) + (w.w >> 8);
        }
        float v = (float)((int)S - (int)(6u * 16777215u));
        g = __fmul_rn(v, __int_as_float(0x32AAAAAB));       // fl(2^-24 / 3)
        g = fminf(fmaxf(g, -1.0f), 1.0f);
    } else {
        W4 w = draw(seed, k, p, 0u, TAG_INIT);
        g = mode == GAME_INIT_UNIFORM_01 ? u01(w.x) : upm1(w.x);
    }
    pop[i] = g;
}

int launch_init_population(game_ctx *ctx, int mode, unsigned long long seed, int P, float *pop)
{
    long long n = (long long)P * ctx->K;
    init_population_kernel<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(mode, seed, P, ctx->K, pop);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// ---- a6: rank by counting.  key = (error, index) ascending, NaN as +inf, -0 as +0 (DESIGN G20) --------
// (Measured and dropped: ONE launch with all P keys in every CTA's shared memory and eight lanes per chromosome -- the tail of a
// generation grew from 30 to 45 us on config 3 (P = 4096) and from 100 to 121 us on config 5: 128-256 CTAs each staging
// every key cost more than the launch they saved.)
constexpr int RANK_T = 128, RANK_Q = 256;   // chromosomes per CTA x keys per CTA: (P/128) x (P/256) CTAs

__global__ void rank_count_kernel(const float *__restrict__ fit, int P, int *__restrict__ rank, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    __shared__ unsigned long long keys[RANK_Q];
    int p = blockIdx.x * RANK_T + threadIdx.x;
    int q0 = blockIdx.y * RANK_Q;
    for (int i = threadIdx.x; i < RANK_Q; i += RANK_T) {
        int q = q0 + i;
        keys[i] = q < P ? (((unsigned long long)sort_key(fit[q]) << 32) | (unsigned)q) : ~0ull;
    }
    __syncthreads();
    if (p >= P) return;
    unsigned long long mine = ((unsigned long long)sort_key(fit[p]) << 32) | (unsigned)p;
    int cnt = 0;
#pragma unroll 8
    for (int i = 0; i < RANK_Q; ++i) cnt += keys[i] < mine;
    if (gridDim.y == 1) rank[p] = cnt;
    else if (cnt) atomicAdd(&rank[p], cnt);      // integer: order-independent, exact; buffer is zero on entry
}

// order[rank[p]] = p, plus a7: record the best and apply the stop test (L219, L287; DESIGN G18)
__global__ void rank_scatter_kernel(const float *__restrict__ fit, int P, int *__restrict__ rank,
                                    int *__restrict__ order, DevState *state, float stop_error, int update_state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    int r = rank[p];
    rank[p] = 0;                                 // leave the scratch zeroed for the next call's atomics
    order[r] = p;
    if (r == 0 && update_state) {
        float f = fit[p];
        state->best_error = f;
        state->best_index = p;
        state->evals_done += 1;
        if (stop_error >= 0.0f && f <= stop_error) state->stop_request = 1;
    }
}

int launch_rank(game_ctx *ctx, const float *fit, int P, int *rank_scratch, int *order, DevState *state,
                float stop_error, bool update_state)
{
    dim3 grid((P + RANK_T - 1) / RANK_T, (P + RANK_Q - 1) / RANK_Q);
    GAME_CUDA(ctx, launch_pdl(rank_count_kernel, grid, dim3(RANK_T), 0, ctx, fit, P, rank_scratch, state));
    ++ctx->launches;
    GAME_CUDA(ctx, launch_pdl(rank_scatter_kernel, dim3((P + 255) / 256), dim3(256), 0, ctx, fit, P, rank_scratch, order, state,
                              stop_error, update_state ? 1 : 0));
    ++ctx->launches;
    return GAME_OK;
}

// ---- R4: roulette weights and their inclusive prefix sums, in rank order (single CTA) -----------------
__global__ void roulette_kernel(const float *__restrict__ fit, const int *__restrict__ order, int P,
                                unsigned int *__restrict__ wts, unsigned long long *__restrict__ prefix,
                                const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    __shared__ float smax[32], smin[32];
    __shared__ int scnt[32];
    __shared__ unsigned long long csum[1024];
    const int T = blockDim.x, tid = threadIdx.x;
    float fmx = -INFINITY, fmn = INFINITY;
    int nf = 0;
    for (int r = tid; r < P; r += T) {
        float f = fit[order[r]];
        if (isfinite(f)) { ++nf; fmx = fmaxf(fmx, f); fmn = fminf(fmn, f); }
    }
    for (int o = 16; o; o >>= 1) {
        fmx = fmaxf(fmx, __shfl_xor_sync(0xffffffffu, fmx, o));
        fmn = fminf(fmn, __shfl_xor_sync(0xffffffffu, fmn, o));
        nf += __shfl_xor_sync(0xffffffffu, nf, o);
    }
    if ((tid & 31) == 0) { smax[tid >> 5] = fmx; smin[tid >> 5] = fmn; scnt[tid >> 5] = nf; }
    __syncthreads();
    fmx = -INFINITY; fmn = INFINITY; nf = 0;
    for (int w = 0; w < (T >> 5); ++w) { fmx = fmaxf(fmx, smax[w]); fmn = fminf(fmn, smin[w]); nf += scnt[w]; }
    const float b = __fsub_rn(fmx, fmn);
    // contiguous chunk per thread
    const int per = (P + T - 1) / T;
    const int lo = tid * per, hi = min(lo + per, P);
    unsigned long long s = 0;
    for (int r = lo; r < hi; ++r) {
        float f = fit[order[r]];
        unsigned int w;
        if (nf == 0) w = 1u;
        else if (!isfinite(f)) w = 0u;
        else if (!(b > 0.0f)) w = 1u;
        else w = (unsigned int)__fmul_rn(__fdiv_rn(__fsub_rn(fmx, f), b), 16777216.0f) + 1u;
        wts[r] = w;
        s += w;
    }
    csum[tid] = s;
    __syncthreads();
    if (tid == 0) {
        unsigned long long run = 0;
        for (int i = 0; i < T; ++i) { unsigned long long v = csum[i]; csum[i] = run; run += v; }
    }
    __syncthreads();
    unsigned long long run = csum[tid];
    for (int r = lo; r < hi; ++r) { run += wts[r]; prefix[r] = run; }
}

// ---- a8-a11: one CTA per elite slot or per child pair (StepArgs, select_parent: ga_device.cuh) ----------
__global__ void ga_step_kernel(StepArgs a, const int *__restrict__ order, const float *__restrict__ pop,
                               float *__restrict__ next, const unsigned long long *__restrict__ prefix,
                               DevState *state, int *dbg)
{
    const int K = a.K;
    pdl_wait();
    pdl_trigger();
    if (state) a.gen += (uint32_t)(state->evals_done - 1);     // written by the rank step of THIS generation, stable here
    const bool stopped = state && (state->stopped | state->stop_request);
    if (stopped && threadIdx.x == 0) state->stopped = 1;      // promote (every CTA writes the same value)
    if (blockIdx.x < a.e) {                         // a8 elitism (L148, L291; DESIGN G17)
        int j = blockIdx.x;
        int src = stopped ? j : (a.elite_mode == GAME_ELITE_TOP_E ? order[j] : order[0]);
        for (int k = threadIdx.x; k < K; k += blockDim.x) {
            const float v = pop[(long long)src * K + k];
            next[(long long)j * K + k] = v;
            if (a.sink.ptr) c16_store(a.sink, j, k, v);
        }
        return;
    }
    const int q = blockIdx.x - a.e;
    const int sA = a.e + 2 * q, sB = sA + 1;
    if (stopped) {                                  // loop already stopped: carry the population over unchanged
        for (int k = threadIdx.x; k < K; k += blockDim.x) {
            const float vA = pop[(long long)sA * K + k];
            next[(long long)sA * K + k] = vA;
            if (a.sink.ptr) c16_store(a.sink, sA, k, vA);
            if (sB < a.P) {
                const float vB = pop[(long long)sB * K + k];
                next[(long long)sB * K + k] = vB;
                if (a.sink.ptr) c16_store(a.sink, sB, k, vB);
            }
        }
        return;
    }
    __shared__ int sh[4];
    if (threadIdx.x < 2) sh[threadIdx.x] = select_parent(a, (uint32_t)(2 * q + threadIdx.x), order, prefix);   // a9
    if (threadIdx.x == 2) {                          // a10 decision (R5)
        W4 w = draw(a.seed, 0u, (uint32_t)q, a.gen, TAG_XOVER);
        sh[2] = (K >= 2) && hit(w.x, a.pc);
        sh[3] = K >= 2 ? 1 + (int)idx_of(w.y, (uint32_t)(K - 1)) : 0;
    }
    __syncthreads();
    const int pa = sh[0], pb = sh[1], doit = sh[2], cut = sh[3];
    if (dbg && threadIdx.x == 0) { dbg[4 * q] = pa; dbg[4 * q + 1] = pb; dbg[4 * q + 2] = doit; dbg[4 * q + 3] = cut; }
    if (q == 0 && threadIdx.x == 0 && state) state->gens_run += 1;
    const float *ra = pop + (long long)pa * K, *rb = pop + (long long)pb * K;
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        float ga = ra[k], gb = rb[k];
        bool head = doit ? (k < cut) : true;
        float cA = head ? ga : gb;                  // A = pa[0:c] | pb[c:K]
        float cB = head ? gb : ga;                  // B = pb[0:c] | pa[c:K]
        W4 w = draw(a.seed, (uint32_t)k, (uint32_t)sA, a.gen, TAG_MUTATE);       // a11 (R6)
        if (hit(w.x, a.pm)) cA = upm1(w.y);
        next[(long long)sA * K + k] = cA;
        if (a.sink.ptr) c16_store(a.sink, sA, k, cA);
        if (sB < a.P) {
            W4 v = draw(a.seed, (uint32_t)k, (uint32_t)sB, a.gen, TAG_MUTATE);
            if (hit(v.x, a.pm)) cB = upm1(v.y);
            next[(long long)sB * K + k] = cB;
            if (a.sink.ptr) c16_store(a.sink, sB, k, cB);
        }
    }
}

void fill_step_args(const game_ctx *ctx, const game_ga_params *gp, unsigned long long seed, unsigned int gen_base, StepArgs *out)
{
    StepArgs &a = *out;
    a.sink.ptr = nullptr;
    a.P = gp->P; a.K = ctx->K; a.e = gp->elitism; a.elite_mode = gp->elite_mode; a.selection = gp->selection;
    a.tsize = gp->tournament_size; a.npairs = (gp->P - gp->elitism + 1) / 2;
    a.pc = host_thr(gp->p_crossover); a.pm = host_thr(gp->p_mutation);
    a.seed = seed; a.gen = gen_base;
}

int launch_ga_step(game_ctx *ctx, const game_ga_params *gp, unsigned long long seed, unsigned int gen_base,
                   const int *order, const float *fit, const float *pop, float *next, DevState *state,
                   unsigned int *rw, unsigned long long *rprefix, const C16Sink *sink)
{
    StepArgs a;
    fill_step_args(ctx, gp, seed, gen_base, &a);
    if (sink) a.sink = *sink;
    if (gp->selection == GAME_SEL_ROULETTE) {
        GAME_CUDA(ctx, launch_pdl(roulette_kernel, dim3(1), dim3(1024), 0, ctx, fit, order, gp->P, rw, rprefix, state));
        ++ctx->launches;
    }
    int threads = ctx->K >= 512 ? 256 : ctx->K >= 128 ? 128 : 64;
    GAME_CUDA(ctx, launch_pdl(ga_step_kernel, dim3(a.e + a.npairs), dim3(threads), 0, ctx, a, order, pop, next, rprefix, state,
                              (int *)nullptr));
    ++ctx->launches;
    return GAME_OK;
}

// ---- raw Philox words for tests -----------------------------------------------------------------------
__global__ void philox_kernel(unsigned long long seed, const uint32_t *__restrict__ ctr, int n, uint32_t *__restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    W4 w = draw(seed, ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    out[4 * i] = w.x; out[4 * i + 1] = w.y; out[4 * i + 2] = w.z; out[4 * i + 3] = w.w;
}

int launch_philox(game_ctx *ctx, unsigned long long seed, const unsigned int *ctr, int n, unsigned int *out)
{
    philox_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(seed, ctr, n, out);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

}  // namespace game
