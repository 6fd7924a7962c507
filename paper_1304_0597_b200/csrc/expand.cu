// a0/a1: dataset checks and feature expansion (eq. 8-9; Chebyshev per DESIGN G7),
// computed ONCE per game_load as the paper does (L254).  Terms are evaluated in fp64 on the device and
// rounded once to the storage type, so E is the correctly rounded expansion to within an ulp.
#include "game_internal.cuh"

namespace game {

// flag[0] |= 1 when X (a) or the targets (b) hold a NaN/Inf; flag[2] = max |X| as float bits (the in-kernel
// generator's fast sincos is only offered for |x| <= pi)
__global__ void check_finite_kernel(const float *__restrict__ a, long long na, const float *__restrict__ b,
                                    long long nb, int *flag)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    bool bad = false;
    float mx = 0.f;
    for (long long j = i; j < na; j += stride) { const float v = a[j]; bad |= !isfinite(v); mx = fmaxf(mx, fabsf(v)); }
    for (long long j = i; j < nb; j += stride) bad |= !isfinite(b[j]);
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1);
    for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.f && mx < INFINITY) atomicMax(flag + 2, __float_as_int(mx));   // non-negative floats order as ints
}

int launch_check_finite(game_ctx *ctx, const float *X, long long nX, const float *t, long long nT, int *flag_dev)
{
    long long n = nX > nT ? nX : nT;
    int blocks = (int)((n + 255) / 256);
    if (blocks > ctx->sm_count * 8) blocks = ctx->sm_count * 8;
    if (blocks < 1) blocks = 1;
    check_finite_kernel<<<blocks, 256, 0, ctx->stream>>>(X, nX, t, nT, flag_dev);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// flag2[0] |= 1 when v holds a NaN/Inf; flag2[1] = max |v| over the finite values, as float bits (game_set_population,
// game_fitness_host: is every gene inside the fp16 range the tensor paths need?)
__global__ void max_abs_kernel(const float *__restrict__ v, long long n, int *flag2)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    bool bad = false;
    float mx = 0.f;
    for (long long j = i; j < n; j += stride) { const float x = v[j]; if (isfinite(x)) mx = fmaxf(mx, fabsf(x)); else bad = true; }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag2, 1);
    for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.f) atomicMax(flag2 + 1, __float_as_int(mx));
}

int launch_max_abs(game_ctx *ctx, const float *v, long long n, int *flag2_dev)
{
    int blocks = (int)((n + 255) / 256);
    if (blocks > ctx->sm_count * 8) blocks = ctx->sm_count * 8;
    if (blocks < 1) blocks = 1;
    max_abs_kernel<<<blocks, 256, 0, ctx->stream>>>(v, n, flag2_dev);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// One thread per (feature i, pattern n); n is the fastest thread index so the term-major stores
// ET[k][n] are coalesced.  Term index k = i*B + m, block order [1, cos 1..d, sin 1..d] / [T_0..T_d].
// split != 0 (TENSOR_SPLIT path): E is written as three fp16 k-ranges [hi | hi | lo] of ld/3 positions each, hi = fp16(E),
// lo = fp16(E - hi), so that against genes laid out [hi | lo | hi] one fp16 contraction over 3K terms yields
// E_hi C_hi + E_hi C_lo + E_lo C_hi = E C to ~2^-22 relative.
template <typename OutT, bool PATTERN_MAJOR>
__global__ void expand_kernel(const float *__restrict__ X, long long N, int F, int family, int d,
                              OutT *__restrict__ E, long long ld, float *maxabs, int split = 0)
{
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int i = blockIdx.y;
    float local_max = 0.f;
    if (n < N) {
        double x = (double)X[n * F + i];
        int B = family == GAME_TRIG ? 2 * d + 1 : d + 1;
        int k0 = i * B;
        auto put = [&](int m, double v) {      // m: index inside feature i's block, ABI order
            float f = (float)v;
            local_max = fmaxf(local_max, fabsf(f));
            if (PATTERN_MAJOR) {
                // TENSOR path: permuted term order (tc_position), tile-blocked [n/256][k/64][256][64] so that every
                // TMA box is one contiguous 32 KB run
                const long long k = tc_position(family, d, F, i, m);
                auto at = [&](long long kk) -> OutT & { return E[(((n >> 8) * (ld >> 6) + (kk >> 6)) << 14) + ((n & 255) << 6) + (kk & 63)]; };
                if (!split) {
                    at(k) = (OutT)f;
                } else {
                    const long long third = ld / 3;
                    const OutT hi = (OutT)f;
                    at(k) = hi; at(third + k) = hi; at(2 * third + k) = (OutT)(f - (float)hi);
                }
            } else {
                E[(long long)(k0 + m) * ld + n] = (OutT)f;
            }
        };
        put(0, 1.0);
        if (family == GAME_TRIG) {
            for (int m = 1; m <= d; ++m) {
                double s, c;
                sincos((double)m * x, &s, &c);
                put(m, c);
                put(d + m, s);
            }
        } else {
            double tm1 = 1.0, t0 = x;
            if (d >= 1) put(1, x);
            for (int m = 2; m <= d; ++m) {
                double t1 = 2.0 * x * t0 - tm1;
                put(m, t1);
                tm1 = t0;
                t0 = t1;
            }
        }
    }
    if (maxabs) {
        for (int o = 16; o; o >>= 1) local_max = fmaxf(local_max, __shfl_xor_sync(0xffffffffu, local_max, o));
        if ((threadIdx.x & 31) == 0 && local_max > 0.f)
            atomicMax((int *)maxabs, __float_as_int(local_max));   // non-negative floats order as ints
    }
}

// Paper-literal tied families (eq. 2 / eq. 9 as printed, L57, L100-L103): one coefficient set for all features,
// so a term is a per-pattern SUM over features -- the "sums of sines and cosines ... stored in two vectors"
// the paper precomputes (L254).  One thread per pattern, fp64 sums in ascending feature order.
template <typename OutT, bool PATTERN_MAJOR>
__global__ void expand_tied_kernel(const float *__restrict__ X, long long N, int F, int family, int d,
                                   OutT *__restrict__ E, long long ld, float *maxabs)
{
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    float local_max = 0.f;
    if (n < N) {
        double sum[65];
        const int K = family == GAME_TRIG_TIED ? 2 * d + 1 : d + 1;
        for (int k = 0; k < K; ++k) sum[k] = 0.0;
        sum[0] = 1.0;
        for (int i = 0; i < F; ++i) {
            double x = (double)X[n * F + i];
            if (family == GAME_TRIG_TIED) {
                for (int m = 1; m <= d; ++m) {
                    double s, c;
                    sincos((double)m * x, &s, &c);
                    sum[m] += c;
                    sum[d + m] += s;
                }
            } else {
                double pw = 1.0;
                for (int j = 1; j <= d; ++j) { pw *= x; sum[j] += pw; }
            }
        }
        for (int k = 0; k < K; ++k) {
            float f = (float)sum[k];
            local_max = fmaxf(local_max, fabsf(f));
            if (PATTERN_MAJOR) E[(((n >> 8) * (ld >> 6) + (k >> 6)) << 14) + ((n & 255) << 6) + (k & 63)] = (OutT)f;
            else E[(long long)k * ld + n] = (OutT)f;
        }
    }
    if (maxabs) {
        for (int o = 16; o; o >>= 1) local_max = fmaxf(local_max, __shfl_xor_sync(0xffffffffu, local_max, o));
        if ((threadIdx.x & 31) == 0 && local_max > 0.f) atomicMax((int *)maxabs, __float_as_int(local_max));
    }
}

static bool tied(const game_ctx *ctx) { return ctx->family == GAME_TRIG_TIED || ctx->family == GAME_POLY_TIED; }

int launch_expand_fp32(game_ctx *ctx)
{
    if (tied(ctx)) {
        expand_tied_kernel<float, false><<<(unsigned)((ctx->N + 127) / 128), 128, 0, ctx->stream>>>(
            ctx->X, ctx->N, ctx->F, ctx->family, ctx->degree, ctx->ET, ctx->Npad, nullptr);
        GAME_LAUNCHED(ctx);
        return GAME_OK;
    }
    dim3 grid((unsigned)((ctx->N + 255) / 256), (unsigned)ctx->F);
    expand_kernel<float, false><<<grid, 256, 0, ctx->stream>>>(ctx->X, ctx->N, ctx->F, ctx->family, ctx->degree,
                                                                ctx->ET, ctx->Npad, nullptr);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// The fp32 term-major expansion serves the FFMA kernels, game_predict and game_classify only; the tensor paths never
// read it.  It is therefore built on first use (config 4: 2.2 GB and one fp64 sincos per term that a run on the tensor
// path never needs; the out-of-core driver reloads a chunk per generation and would pay it every time).
int ensure_ET(game_ctx *ctx)
{
    if (ctx->ET) return GAME_OK;
    const size_t bytes = (size_t)ctx->K * ctx->Npad * sizeof(float);
    GAME_CUDA(ctx, cudaMalloc(&ctx->ET, bytes));
    cudaError_t e = cudaMemsetAsync(ctx->ET, 0, bytes, ctx->stream);
    int rc = e == cudaSuccess ? launch_expand_fp32(ctx) : cuda_fail(ctx, e, "cudaMemsetAsync(ET)");
    if (rc) { cudaFree(ctx->ET); ctx->ET = nullptr; }
    return rc;
}

int launch_expand_split(game_ctx *ctx)
{
    dim3 grid((unsigned)((ctx->N + 255) / 256), (unsigned)ctx->F);
    expand_kernel<__half, true><<<grid, 256, 0, ctx->stream>>>(ctx->X, ctx->N, ctx->F, ctx->family, ctx->degree,
                                                                ctx->E16s, 3LL * ctx->Kpad, nullptr, 1);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

int launch_expand_fp16(game_ctx *ctx, float *maxabs_dev)
{
    if (tied(ctx)) {
        expand_tied_kernel<__half, true><<<(unsigned)((ctx->N + 127) / 128), 128, 0, ctx->stream>>>(
            ctx->X, ctx->N, ctx->F, ctx->family, ctx->degree, ctx->E16, ctx->Kpad, maxabs_dev);
        GAME_LAUNCHED(ctx);
        return GAME_OK;
    }
    dim3 grid((unsigned)((ctx->N + 255) / 256), (unsigned)ctx->F);
    expand_kernel<__half, true><<<grid, 256, 0, ctx->stream>>>(ctx->X, ctx->N, ctx->F, ctx->family, ctx->degree,
                                                                ctx->E16, ctx->Kpad, maxabs_dev);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// Forward pass of one chromosome (the paper's test / run use cases, L127-L129): thread per pattern,
// coalesced reads of the term-major expansion, fp32 accumulate in ascending k.
__global__ void predict_kernel(const float *__restrict__ ET, long long Npad, long long N, int K,
                               const float *__restrict__ genes, int act, float *z_out, float *y_out)
{
    extern __shared__ float g[];
    for (int k = threadIdx.x; k < K; k += blockDim.x) g[k] = genes[k];
    __syncthreads();
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    float z = 0.f;
    for (int k = 0; k < K; ++k) z = fmaf(ET[(long long)k * Npad + n], g[k], z);
    if (z_out) z_out[n] = z;
    if (y_out) y_out[n] = act == GAME_ACT_SIGMOID ? 1.0f / (1.0f + expf(-z)) : z;
}

// Figures of merit of the test / run use cases: forward pass as above, class = act(z) > cut,
// truth = target > 0.5, counts {TP, FP, TN, FN} by integer atomics (exact, order-independent), then
// accuracy (TP+TN)/N, completeness TP/(TP+FN), contamination FP/(FP+TN) (DESIGN G23) by the last CTA.
__global__ void classify_kernel(const float *__restrict__ ET, long long Npad, long long N, int K,
                                const float *__restrict__ genes, const float *__restrict__ tgt, int act, float cut,
                                unsigned long long *counts, double *fom, unsigned int *ticket)
{
    extern __shared__ float g[];
    __shared__ unsigned int sc[4];
    for (int k = threadIdx.x; k < K; k += blockDim.x) g[k] = genes[k];
    if (threadIdx.x < 4) sc[threadIdx.x] = 0;
    __syncthreads();
    long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n < N) {
        float z = 0.f;
        for (int k = 0; k < K; ++k) z = fmaf(ET[(long long)k * Npad + n], g[k], z);
        float y = act == GAME_ACT_SIGMOID ? 1.0f / (1.0f + expf(-z)) : z;
        bool pred = y > cut, truth = tgt[n] > 0.5f;
        atomicAdd(&sc[pred ? (truth ? 0 : 1) : (truth ? 3 : 2)], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 4 && sc[threadIdx.x]) atomicAdd(&counts[threadIdx.x], (unsigned long long)sc[threadIdx.x]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(ticket, 1u) == gridDim.x - 1) {      // last CTA: every count has landed
        __threadfence();
        volatile unsigned long long *c = counts;
        double tp = (double)c[0], fp = (double)c[1], tn = (double)c[2], fn = (double)c[3];
        fom[0] = N > 0 ? (tp + tn) / (double)N : 0.0;
        fom[1] = tp + fn > 0 ? tp / (tp + fn) : 0.0;
        fom[2] = fp + tn > 0 ? fp / (fp + tn) : 0.0;
        *ticket = 0;
    }
}

int launch_classify(game_ctx *ctx, const float *genes, float cut, long long *counts, double *fom, unsigned int *ticket)
{
    int rce = ensure_ET(ctx);
    if (rce) return rce;
    GAME_CUDA(ctx, cudaMemsetAsync(counts, 0, 4 * sizeof(long long), ctx->stream));
    int blocks = (int)((ctx->N + 255) / 256);
    classify_kernel<<<blocks, 256, ctx->K * sizeof(float), ctx->stream>>>(ctx->ET, ctx->Npad, ctx->N, ctx->K, genes, ctx->t,
                                                                         ctx->act, cut, (unsigned long long *)counts, fom,
                                                                         ticket);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

int launch_predict(game_ctx *ctx, const float *genes, float *z_out, float *y_out)
{
    int rce = ensure_ET(ctx);
    if (rce) return rce;
    int blocks = (int)((ctx->N + 255) / 256);
    predict_kernel<<<blocks, 256, ctx->K * sizeof(float), ctx->stream>>>(ctx->ET, ctx->Npad, ctx->N, ctx->K, genes,
                                                                        ctx->act, z_out, y_out);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

// game_predict_new: the forward pass on caller-supplied patterns, expansion on the fly (no dataset load).  One thread
// per pattern; every term is computed exactly as expand_kernel / expand_tied_kernel compute it (fp64, one rounding to
// fp32) and accumulated in ascending ABI gene order k = i*B + m, so the bits equal game_load(X_new) + game_predict.
__global__ void predict_new_kernel(const float *__restrict__ X, long long N, int F, int family, int d, int K,
                                   const float *__restrict__ genes, int act, float *z_out, float *y_out)
{
    extern __shared__ float g[];
    for (int k = threadIdx.x; k < K; k += blockDim.x) g[k] = genes[k];
    __syncthreads();
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    float z = 0.f;
    if (family == GAME_TRIG_TIED || family == GAME_POLY_TIED) {
        double sum[65];
        for (int k = 0; k < K; ++k) sum[k] = 0.0;
        sum[0] = 1.0;
        for (int i = 0; i < F; ++i) {
            const double x = (double)X[n * F + i];
            if (family == GAME_TRIG_TIED) {
                for (int m = 1; m <= d; ++m) {
                    double s, c;
                    sincos((double)m * x, &s, &c);
                    sum[m] += c;
                    sum[d + m] += s;
                }
            } else {
                double pw = 1.0;
                for (int j = 1; j <= d; ++j) { pw *= x; sum[j] += pw; }
            }
        }
        for (int k = 0; k < K; ++k) z = fmaf((float)sum[k], g[k], z);
    } else {
        const int B = family == GAME_TRIG ? 2 * d + 1 : d + 1;
        for (int i = 0; i < F; ++i) {
            const double x = (double)X[n * F + i];
            const float *gi = g + i * B;
            z = fmaf(1.0f, gi[0], z);
            if (family == GAME_TRIG) {
                // ABI order inside the block is [1, cos 1..d, sin 1..d]: the sines wait in a local array so that the
                // accumulation order stays ascending in k while sincos is called exactly as expand_kernel calls it
                float sn[32];
                for (int m = 1; m <= d; ++m) {
                    double sv, cv;
                    sincos((double)m * x, &sv, &cv);
                    sn[m - 1] = (float)sv;
                    z = fmaf((float)cv, gi[m], z);
                }
                for (int m = 1; m <= d; ++m) z = fmaf(sn[m - 1], gi[d + m], z);
            } else {
                double tm1 = 1.0, t0 = x;
                z = fmaf((float)x, gi[1], z);
                for (int m = 2; m <= d; ++m) {
                    const double t1 = 2.0 * x * t0 - tm1;
                    z = fmaf((float)t1, gi[m], z);
                    tm1 = t0;
                    t0 = t1;
                }
            }
        }
    }
    if (z_out) z_out[n] = z;
    if (y_out) y_out[n] = act == GAME_ACT_SIGMOID ? 1.0f / (1.0f + expf(-z)) : z;
}

int launch_predict_new(game_ctx *ctx, const float *genes, const float *X_new, long long N_new, float *z_out, float *y_out)
{
    const int blocks = (int)((N_new + 127) / 128);
    predict_new_kernel<<<blocks, 128, ctx->K * sizeof(float), ctx->stream>>>(X_new, N_new, ctx->F, ctx->family, ctx->degree,
                                                                            ctx->K, genes, ctx->act, z_out, y_out);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

}  // namespace game
