// a2-a5, FP32 path: z = E.C^T on the FFMA pipe with the activation, error and per-chromosome
// reduction fused in the epilogue (eq. 2-5, eq. 9-10).
// The N x P matrix z lives only in registers.
//
// Tiling: one CTA = 128 patterns (one SLAB) x 128 chromosomes, 256 threads, 8x8 outputs per thread,
// k-chunks of 16 staged in shared memory with register prefetch of the next chunk.  A CTA walks
// `slabs_per_cta` consecutive slabs and keeps the per-chromosome error sums in registers, then writes
// one row of `partial[chunk][p]`; finalize_kernel adds the rows in fixed order in fp64.  No float
// atomics anywhere: the result is run-to-run reproducible and independent of where a chromosome sits
// in the population (DESIGN P20: the elite's fitness must not change when its row moves).
#include "game_internal.cuh"

namespace game {

constexpr int BN = 128, BP = 128, BK = 16, NT = 256;

__device__ __forceinline__ float act_err(float z, float t, bool valid, int act, int err, float R)
{
    float y = act == GAME_ACT_SIGMOID ? __fdividef(1.0f, 1.0f + __expf(-z)) : z;
    float r = t - y;
    float e = r * r;
    if (err == GAME_ERR_TMSE && !(fabsf(r) > R)) e = 0.f;
    return valid ? e : 0.f;
}

__global__ void __launch_bounds__(NT, 2)
fitness_fp32_kernel(const float *__restrict__ ET, long long Npad, long long N, int K,
                    const float *__restrict__ pop, int P, const float *__restrict__ tgt,
                    int n_slabs, int slabs_per_cta, FitnessCfg cfg, float *__restrict__ partial, int Ppad,
                    const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    __shared__ __align__(16) float As[BK][BN];        // E chunk: [k][n]
    __shared__ __align__(16) float Bs[BK][BP + 4];    // C chunk: [k][p], padded against store conflicts
    __shared__ float red[16][BP];

    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int p0 = blockIdx.y * BP;
    const int chunk = blockIdx.x;
    const int slab_lo = chunk * slabs_per_cta;
    const int slab_hi = min(slab_lo + slabs_per_cta, n_slabs);

    float colsum[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) colsum[j] = 0.f;

    const int nk = (K + BK - 1) / BK;
    for (int slab = slab_lo; slab < slab_hi; ++slab) {
        const long long n0 = (long long)slab * BN;
        float acc[8][8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

        float4 ra[2];
        float rb[8];
        auto gload = [&](int kc) {
            const int k0 = kc * BK;
#pragma unroll
            for (int v = 0; v < 2; ++v) {     // 16 rows x 32 float4
                int idx = tid + v * NT;
                int kr = idx >> 5, c4 = idx & 31;
                int k = k0 + kr;
                ra[v] = k < K ? *reinterpret_cast<const float4 *>(ET + (long long)k * Npad + n0 + c4 * 4)
                              : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int v = 0; v < 8; ++v) {     // 128 rows x 16 k, 16 consecutive k per row segment
                int idx = tid + v * NT;
                int pr = idx >> 4, kk = idx & 15;
                int p = p0 + pr, k = k0 + kk;
                rb[v] = (p < P && k < K) ? pop[(long long)p * K + k] : 0.f;
            }
        };
        auto sstore = [&]() {
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                int idx = tid + v * NT;
                int kr = idx >> 5, c4 = idx & 31;
                *reinterpret_cast<float4 *>(&As[kr][c4 * 4]) = ra[v];
            }
#pragma unroll
            for (int v = 0; v < 8; ++v) {
                int idx = tid + v * NT;
                int pr = idx >> 4, kk = idx & 15;
                Bs[kk][pr] = rb[v];
            }
        };

        gload(0);
        for (int kc = 0; kc < nk; ++kc) {
            __syncthreads();          // previous chunk fully consumed
            sstore();
            __syncthreads();
            if (kc + 1 < nk) gload(kc + 1);
#pragma unroll
            for (int kk = 0; kk < BK; ++kk) {
                float4 a0 = *reinterpret_cast<const float4 *>(&As[kk][ty * 4]);
                float4 a1 = *reinterpret_cast<const float4 *>(&As[kk][64 + ty * 4]);
                float4 b0 = *reinterpret_cast<const float4 *>(&Bs[kk][tx * 4]);
                float4 b1 = *reinterpret_cast<const float4 *>(&Bs[kk][64 + tx * 4]);
                float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
                float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
            }
        }
        // epilogue for this slab: activation, error, sum over this thread's 8 patterns
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            long long n = n0 + (i < 4 ? ty * 4 + i : 64 + ty * 4 + (i - 4));
            bool valid = n < N;
            float t = tgt[n];       // tgt is padded to Npad
#pragma unroll
            for (int j = 0; j < 8; ++j) colsum[j] += act_err(acc[i][j], t, valid, cfg.act, cfg.err, cfg.R);
        }
    }
    // fixed-order reduction over the 16 thread rows
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 8; ++j) red[ty][(j < 4 ? tx * 4 + j : 64 + tx * 4 + (j - 4))] = colsum[j];
    __syncthreads();
    if (tid < BP) {
        float s = 0.f;
#pragma unroll
        for (int r = 0; r < 16; ++r) s += red[r][tid];
        partial[(long long)chunk * Ppad + p0 + tid] = s;
    }
}

// Small problems (configs 1-2) are launch-latency bound, so the tail of a generation is ONE single-CTA kernel:
// a5 final reduction (same summation order as finalize_kernel, so the bits agree), a6 rank by counting
// over shared-memory keys, a7 best / stop test.  One thread per chromosome; used for P <= 256, n_chunks*P <= 8192
// (beyond that the multi-CTA rank is faster than one CTA's P^2 compares).
constexpr int POST_SMALL_FLOATS = 8192;

__global__ void __launch_bounds__(256, 1)
post_small_kernel(const float *__restrict__ partial, int n_chunks, int Ppad, int P, long long N, int err,
                  float *__restrict__ fit, int *__restrict__ order, DevState *state, float stop_error)
{
    pdl_wait();
    pdl_trigger();
    if (state->stopped) return;            // single CTA: the flag this kernel may set is stop_request, read by later launches
    __shared__ unsigned long long keys[256];
    __shared__ float part[POST_SMALL_FLOATS];
    const int p = threadIdx.x;
    for (int i = p; i < n_chunks * P; i += blockDim.x)        // all slab sums in flight at once, then summed in order
        part[i] = partial[(long long)(i / P) * Ppad + (i % P)];
    __syncthreads();
    unsigned long long mine = ~0ull;
    float f = 0.f;
    if (p < P) {
        double tot = 0.0;
        for (int r = 0; r < 32; ++r) {
            double s = 0.0;
            for (int ch = r; ch < n_chunks; ch += 32) s += (double)part[ch * P + p];
            tot += s;
        }
        double v = tot / (double)N;
        if (err == GAME_ERR_RMSE) v = sqrt(v);
        f = (float)v;
        fit[p] = f;
        mine = ((unsigned long long)sort_key(f) << 32) | (unsigned)p;
    }
    keys[p] = mine;
    __syncthreads();
    if (p >= P) return;
    int cnt = 0;
#pragma unroll 8
    for (int q = 0; q < P; ++q) cnt += keys[q] < mine;
    order[cnt] = p;
    if (cnt == 0) {
        state->best_error = f;
        state->best_index = p;
        state->evals_done += 1;
        if (stop_error >= 0.0f && f <= stop_error) state->stop_request = 1;
    }
}

// The same tail for small populations over MANY slabs (config 4: 256 chromosomes x 3907 tiles): the slab axis is totalled by
// finalize_split_kernel's FIN_SPLIT CTAs, and this single CTA adds those totals in finalize_merge_kernel's order, ranks and
// tests -- one launch instead of three (merge, rank count, rank scatter) in every generation.
__global__ void __launch_bounds__(256, 1)
post_merge_small_kernel(const double *__restrict__ fin2, int Ppad, int P, long long N, int err,
                        float *__restrict__ fit, int *__restrict__ order, DevState *state, float stop_error)
{
    pdl_wait();
    pdl_trigger();
    if (state->stopped) return;
    __shared__ unsigned long long keys[256];
    const int p = threadIdx.x;
    unsigned long long mine = ~0ull;
    float f = 0.f;
    if (p < P) {
        double tot = 0.0;
        for (int y = 0; y < FIN_SPLIT; ++y) tot += fin2[(long long)y * Ppad + p];
        double v = tot / (double)N;
        if (err == GAME_ERR_RMSE) v = sqrt(v);
        f = (float)v;
        fit[p] = f;
        mine = ((unsigned long long)sort_key(f) << 32) | (unsigned)p;
    }
    keys[p] = mine;
    __syncthreads();
    if (p >= P) return;
    int cnt = 0;
#pragma unroll 8
    for (int q = 0; q < P; ++q) cnt += keys[q] < mine;
    order[cnt] = p;
    if (cnt == 0) {
        state->best_error = f;
        state->best_index = p;
        state->evals_done += 1;
        if (stop_error >= 0.0f && f <= stop_error) state->stop_request = 1;
    }
}

__global__ void finalize_split_kernel(const float *__restrict__ partial, int n_chunks, int Ppad, int P, double *__restrict__ fin2,
                                      const DevState *state);

int launch_post(game_ctx *ctx, PartialInfo pi, int P, float *fit, int *rank_scratch, int *order, DevState *state,
                float stop_error)
{
    if (P <= 256 && (long long)pi.n_chunks * P <= POST_SMALL_FLOATS) {
        GAME_CUDA(ctx, launch_pdl(post_small_kernel, dim3(1), dim3(256), 0, ctx, ctx->partial, pi.n_chunks, pi.Ppad, P, ctx->N,
                                  ctx->err, fit, order, state, stop_error));
        ++ctx->launches;
        return GAME_OK;
    }
    if (P <= 256 && pi.n_chunks >= 1024) {            // the two-pass reduction's first pass, then merge + rank + stop test in one CTA
        GAME_CUDA(ctx, launch_pdl(finalize_split_kernel, dim3((P + 31) / 32, FIN_SPLIT), dim3(32, 32), 0, ctx, ctx->partial, pi.n_chunks, pi.Ppad, P,
                                  ctx->fin2, (const DevState *)state));
        GAME_CUDA(ctx, launch_pdl(post_merge_small_kernel, dim3(1), dim3(256), 0, ctx, (const double *)ctx->fin2, pi.Ppad, P, ctx->N, ctx->err,
                                  fit, order, state, stop_error));
        ctx->launches += 2;
        return GAME_OK;
    }
    // (a fused multi-CTA finalize + rank kernel for mid-size populations was measured on config 2: 22.7 vs 19.7 us per
    // generation -- inside the captured graph three small kernels cost less than one with serial phases)
    int rc = launch_finalize(ctx, pi.n_chunks, pi.Ppad, P, fit, state);
    if (rc) return rc;
    return launch_rank(ctx, fit, P, rank_scratch, order, state, stop_error, true);
}

// fit[p] = (sum over chunks, ascending, in fp64) / N; RMSE takes the root (eq. 4-5).
// With `sums` set the fp64 total itself is written instead (game_fitness_sums: the pattern-sharded exchange adds the
// totals of all shards before the mean is taken).
__global__ void finalize_kernel(const float *__restrict__ partial, int n_chunks, int Ppad, int P, long long N,
                                int err, float *__restrict__ out, double *__restrict__ sums, int accumulate, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    __shared__ double red[32][33];
    int c = threadIdx.x, r = threadIdx.y;
    int p = blockIdx.x * 32 + c;
    double s = 0.0;
    if (p < P)
        for (int ch = r; ch < n_chunks; ch += 32) s += (double)partial[(long long)ch * Ppad + p];
    red[r][c] = s;
    __syncthreads();
    if (r == 0 && p < P) {
        double tot = 0.0;
        for (int q = 0; q < 32; ++q) tot += red[q][c];
        if (sums) { sums[p] = accumulate ? sums[p] + tot : tot; return; }
        double f = tot / (double)N;
        if (err == GAME_ERR_RMSE) f = sqrt(f);
        out[p] = (float)f;
    }
}

// Many slabs, few chromosomes (config 4: 7814 x 256): one CTA per 32 chromosomes would leave the GPU idle, so the
// slab axis is split over FIN_SPLIT CTAs that each total a contiguous range in fp64, and a second tiny kernel adds
// the FIN_SPLIT totals in ascending order.  Fixed order again: reproducible, and the same for every caller.
__global__ void finalize_split_kernel(const float *__restrict__ partial, int n_chunks, int Ppad, int P,
                                      double *__restrict__ fin2, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    __shared__ double red[32][33];
    const int c = threadIdx.x, r = threadIdx.y;
    const int p = blockIdx.x * 32 + c;
    const int len = (n_chunks + FIN_SPLIT - 1) / FIN_SPLIT;
    const int lo = blockIdx.y * len, hi = min(lo + len, n_chunks);
    double s = 0.0;
    if (p < P)
        for (int ch = lo + r; ch < hi; ch += 32) s += (double)partial[(long long)ch * Ppad + p];
    red[r][c] = s;
    __syncthreads();
    if (r == 0 && p < P) {
        double tot = 0.0;
        for (int q = 0; q < 32; ++q) tot += red[q][c];
        fin2[(long long)blockIdx.y * Ppad + p] = tot;
    }
}

__global__ void finalize_merge_kernel(const double *__restrict__ fin2, int Ppad, int P, long long N, int err,
                                      float *__restrict__ out, double *__restrict__ sums, int accumulate, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double tot = 0.0;
    for (int y = 0; y < FIN_SPLIT; ++y) tot += fin2[(long long)y * Ppad + p];
    if (sums) { sums[p] = accumulate ? sums[p] + tot : tot; return; }
    double f = tot / (double)N;
    if (err == GAME_ERR_RMSE) f = sqrt(f);
    out[p] = (float)f;
}

// ---- small problems (configs 1-2): latency, not throughput, decides ------------------------------------
// The 128x128 tile above needs ~20 us per CTA whatever P is; when the whole grid is under two waves a
// finer decomposition finishes sooner.  One CTA = one 128-pattern slab x 32 chromosomes, one THREAD = one
// pattern: it streams its column of the term-major expansion (coalesced across the warp) against the 32
// chromosomes staged in shared memory (broadcast reads), keeps 32 dot products in registers, applies the
// activation and error, and the 32 per-pattern errors are summed over the slab's patterns by a fixed
// butterfly (31 shuffles) and a 4-warp shared-memory pass.  Same partial[slab][p] layout as the big kernel.
constexpr int SP = 32, SKC = 128;

constexpr int SMALL_SMEM = SKC * SLAB * 4 + SKC * (SP + 4) * 4;      // E chunk [128][128] + C chunk [128][36]

__global__ void __launch_bounds__(128)
fitness_small_kernel(const float *__restrict__ ET, long long Npad, long long N, int K, const float *__restrict__ pop,
                     int P, const float *__restrict__ tgt, int n_slabs, int spc, int kcap, FitnessCfg cfg,
                     float *__restrict__ partial, int Ppad, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    extern __shared__ __align__(16) float small_smem[];
    float (*Es)[SLAB] = reinterpret_cast<float (*)[SLAB]>(small_smem);                       // [k][n], as in ET
    float (*Cs)[SP + 4] = reinterpret_cast<float (*)[SP + 4]>(small_smem + kcap * SLAB);     // [k][p]; +4: transposed
    __shared__ float red[4][SP];                                                             // stores 4-way, not 32-way
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int p0 = blockIdx.y * SP;
    const bool one_chunk = K <= kcap;          // then the chromosomes are staged once for all of this CTA's slabs
    auto stage_C = [&](int k0, int kc) {       // Cs[k][p] <- pop[p0+p][k0+k] (zero-filled outside), k fastest
        for (int i = tid; i < kcap * SP; i += 128) {
            const int pp = i / kcap, kk = i % kcap;
            const bool in = p0 + pp < P && kk < kc;
            const float *src = in ? pop + (long long)(p0 + pp) * K + k0 + kk : pop;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&Cs[kk][pp]);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(in ? 4 : 0) : "memory");
        }
    };
    if (one_chunk) stage_C(0, K);
    float esum[SP];
#pragma unroll
    for (int j = 0; j < SP; ++j) esum[j] = 0.f;
    const int slab_hi = min((int)(blockIdx.x + 1) * spc, n_slabs);
    for (int slab = blockIdx.x * spc; slab < slab_hi; ++slab) {
        const long long n0 = (long long)slab * SLAB;
        const long long n = n0 + tid;
        float acc[SP];
#pragma unroll
        for (int j = 0; j < SP; ++j) acc[j] = 0.f;
        for (int k0 = 0; k0 < K; k0 += kcap) {
            const int kc = min(kcap, K - k0);
            __syncthreads();
            // the whole E chunk in flight at once (cp.async, 16 B per request): one memory latency, not kc of them
            for (int i = tid; i < kc * (SLAB / 4); i += 128) {
                const int kk = i / (SLAB / 4), c4 = i % (SLAB / 4);
                const float *src = ET + (long long)(k0 + kk) * Npad + n0 + c4 * 4;
                const unsigned dst = (unsigned)__cvta_generic_to_shared(&Es[kk][c4 * 4]);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
            }
            if (!one_chunk) stage_C(k0, kc);
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
#pragma unroll 4
            for (int kk = 0; kk < kc; ++kk) {
                const float e = Es[kk][tid];
#pragma unroll
                for (int j = 0; j < SP; j += 4) {
                    const float4 c4 = *reinterpret_cast<const float4 *>(&Cs[kk][j]);
                    acc[j] = fmaf(e, c4.x, acc[j]);
                    acc[j + 1] = fmaf(e, c4.y, acc[j + 1]);
                    acc[j + 2] = fmaf(e, c4.z, acc[j + 2]);
                    acc[j + 3] = fmaf(e, c4.w, acc[j + 3]);
                }
            }
        }
        const bool valid = n < N;
        const float t = tgt[n];
#pragma unroll
        for (int j = 0; j < SP; ++j) esum[j] += act_err(acc[j], t, valid, cfg.act, cfg.err, cfg.R);
    }
    float (&acc)[SP] = esum;
    // butterfly: after the step with offset o each lane holds half as many columns, summed over lane pairs;
    // a + b is commutative, so every chromosome sees the same fixed tree whatever its column (DESIGN P20)
#pragma unroll
    for (int o = 16, w = SP / 2; o >= 1; o >>= 1, w >>= 1) {
        const bool upper = (lane & o) != 0;
#pragma unroll
        for (int j = 0; j < w; ++j) {
            float keep = upper ? acc[j + w] : acc[j];
            float send = upper ? acc[j] : acc[j + w];
            acc[j] = keep + __shfl_xor_sync(0xffffffffu, send, o);
        }
    }
    // lane l now owns column bitrev-free index: the kept halves follow the lane bits, i.e. column == lane
    red[warp][lane] = acc[0];
    __syncthreads();
    if (tid < SP) partial[(long long)blockIdx.x * Ppad + p0 + tid] = red[0][tid] + red[1][tid] + red[2][tid] + red[3][tid];
}

static int pick_slabs_per_cta(const game_ctx *ctx, int P)
{
    // enough CTAs for >= ~4 waves at 2 CTAs/SM, but no more partial rows than needed
    long long ptiles = (P + BP - 1) / BP;
    long long want = (long long)ctx->sm_count * 8;
    long long s = (ctx->n_slabs * ptiles) / want;
    if (s < 1) s = 1;
    if (s > 16) s = 16;
    return (int)s;
}

size_t fitness_partial_floats(const game_ctx *ctx, int P)
{
    size_t Ppad = (size_t)((P + 255) / 256) * 256;
    return (size_t)(ctx->n_slabs + 2) * Ppad;     // worst case: one row per slab (tensor path pads N to 256)
}

// fit[p] = sums[p] / N_total (root for RMSE): the tail of a5 after the shards' totals have been added
__global__ void fit_from_sums_kernel(const double *__restrict__ sums, int P, long long N_total, int err, float *__restrict__ out,
                                     const DevState *state)
{
    if (state && state->stopped) return;          // the loop has stopped: fit / order keep describing the final population
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double f = sums[p] / (double)N_total;
    if (err == GAME_ERR_RMSE) f = sqrt(f);
    out[p] = (float)f;
}

int launch_fit_from_sums(game_ctx *ctx, const double *sums, int P, long long N_total, float *out, const DevState *state)
{
    fit_from_sums_kernel<<<(P + 255) / 256, 256, 0, ctx->stream>>>(sums, P, N_total, ctx->err, out, state);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

int launch_finalize(game_ctx *ctx, int n_chunks, int Ppad, int P, float *out, const DevState *state, double *sums, bool accumulate)
{
    const int acc = accumulate ? 1 : 0;
    dim3 block(32, 32);
    if (n_chunks >= 1024 && (P + 31) / 32 < 2 * ctx->sm_count) {
        dim3 grid((P + 31) / 32, FIN_SPLIT);
        GAME_CUDA(ctx, launch_pdl(finalize_split_kernel, grid, block, 0, ctx, ctx->partial, n_chunks, Ppad, P, ctx->fin2, state));
        ++ctx->launches;
        GAME_CUDA(ctx, launch_pdl(finalize_merge_kernel, dim3((P + 255) / 256), dim3(256), 0, ctx, ctx->fin2, Ppad, P, ctx->N,
                                  ctx->err, out, sums, acc, state));
        ++ctx->launches;
        return GAME_OK;
    }
    GAME_CUDA(ctx, launch_pdl(finalize_kernel, dim3((P + 31) / 32), block, 0, ctx, ctx->partial, n_chunks, Ppad, P, ctx->N,
                              ctx->err, out, sums, acc, state));
    ++ctx->launches;
    return GAME_OK;
}

int launch_fitness_fp32(game_ctx *ctx, const float *pop, int P, float *out, const DevState *state, PartialInfo *defer)
{
    int rce = ensure_ET(ctx);             // the fp32 expansion is built on first use
    if (rce) return rce;
    int Ppad = ((P + 255) / 256) * 256;
    FitnessCfg cfg{ctx->act, ctx->err, ctx->R};
    // under two waves of big tiles, or so few chromosomes that a 128-wide tile would mostly compute padding
    if ((long long)ctx->n_slabs * ((P + BP - 1) / BP) < 2LL * ctx->sm_count || P <= 2 * SP) {
        const int ptiles = (P + SP - 1) / SP;
        long long spc_ll = ((long long)ctx->n_slabs * ptiles) / ((long long)ctx->sm_count * 32);
        const int spc = (int)(spc_ll < 1 ? 1 : spc_ll > 64 ? 64 : spc_ll);
        const int n_chunks = (ctx->n_slabs + spc - 1) / spc;
        const int kcap = ctx->K < SKC ? ctx->K : SKC;
        const int smem = kcap * (SLAB + SP + 4) * 4;
        dim3 grid((unsigned)n_chunks, (unsigned)ptiles);
        GAME_CUDA(ctx, ensure_smem_attr(ctx, (const void *)fitness_small_kernel, SMALL_SMEM));
        {
            KernelTimer timer(ctx);
            GAME_CUDA(ctx, launch_pdl(fitness_small_kernel, grid, dim3(128), (size_t)smem, ctx, ctx->ET, ctx->Npad, ctx->N, ctx->K,
                                      pop, P, ctx->t, ctx->n_slabs, spc, kcap, cfg, ctx->partial, Ppad, state));
        }
        ++ctx->launches;
        if (defer) { defer->n_chunks = n_chunks; defer->Ppad = Ppad; return GAME_OK; }
        return launch_finalize(ctx, n_chunks, Ppad, P, out, state);
    }
    int spc = pick_slabs_per_cta(ctx, P);
    int n_chunks = (ctx->n_slabs + spc - 1) / spc;
    dim3 grid((unsigned)n_chunks, (unsigned)((P + BP - 1) / BP));
    {
        KernelTimer timer(ctx);
        GAME_CUDA(ctx, launch_pdl(fitness_fp32_kernel, grid, dim3(NT), 0, ctx, ctx->ET, ctx->Npad, ctx->N, ctx->K, pop, P, ctx->t,
                                  ctx->n_slabs, spc, cfg, ctx->partial, Ppad, state));
    }
    ++ctx->launches;
    if (defer) { defer->n_chunks = n_chunks; defer->Ppad = Ppad; return GAME_OK; }
    return launch_finalize(ctx, n_chunks, Ppad, P, out, state);
}

}  // namespace game
