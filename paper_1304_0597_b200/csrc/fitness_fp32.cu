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

// fit[p] = (sum over chunks, ascending, in fp64) / N; RMSE takes the root (eq. 4-5).
__global__ void finalize_kernel(const float *__restrict__ partial, int n_chunks, int Ppad, int P, long long N,
                                int err, float *__restrict__ out, const DevState *state)
{
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
        double f = tot / (double)N;
        if (err == GAME_ERR_RMSE) f = sqrt(f);
        out[p] = (float)f;
    }
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

int launch_finalize(game_ctx *ctx, int n_chunks, int Ppad, int P, float *out, const DevState *state)
{
    dim3 block(32, 32);
    finalize_kernel<<<(P + 31) / 32, block, 0, ctx->stream>>>(ctx->partial, n_chunks, Ppad, P, ctx->N, ctx->err, out,
                                                               state);
    GAME_LAUNCHED(ctx);
    return GAME_OK;
}

int launch_fitness_fp32(game_ctx *ctx, const float *pop, int P, float *out, const DevState *state)
{
    int Ppad = ((P + 255) / 256) * 256;
    int spc = pick_slabs_per_cta(ctx, P);
    int n_chunks = (ctx->n_slabs + spc - 1) / spc;
    dim3 grid((unsigned)n_chunks, (unsigned)((P + BP - 1) / BP));
    FitnessCfg cfg{ctx->act, ctx->err, ctx->R};
    {
        KernelTimer timer(ctx);
        fitness_fp32_kernel<<<grid, NT, 0, ctx->stream>>>(ctx->ET, ctx->Npad, ctx->N, ctx->K, pop, P, ctx->t,
                                                          ctx->n_slabs, spc, cfg, ctx->partial, Ppad, state);
    }
    GAME_LAUNCHED(ctx);
    return launch_finalize(ctx, n_chunks, Ppad, P, out, state);
}

}  // namespace game
