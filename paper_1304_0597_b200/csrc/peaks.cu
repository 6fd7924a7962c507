// Micro-benchmarks behind the "alu" roofline denominators ("SM count, lane counts, FFMA and MUFU peaks are
// nominal and must be replaced by micro-benchmarks on the box"): register-only loops, one CTA per SM, timed with CUDA
// events on the context's stream.  bench.py --peaks runs them and bench.py's "alu" bounds quote what they measure.
//   GAME_PEAK_FFMA       fp32 FMA pipe, scalar FFMA                         -> FMA/s   (x2 = flop/s)
//   GAME_PEAK_FFMA2      the same pipe through the packed FFMA2 instruction -> FMA/s
//   GAME_PEAK_TANH       special-function unit, tanh.approx.f32             -> op/s
//   GAME_PEAK_EX2        ... ex2.approx.ftz.f32                             -> op/s
//   GAME_PEAK_TANH_MIX   tanh.approx.f32 interleaved with `param` independent FFMA per tanh in the same warps
//                        (the fused epilogue's situation)                   -> tanh/s
#include "game_internal.cuh"

namespace game {

template <int OP> __device__ __forceinline__ float sfu(float x)
{
    float y;
    if (OP == 0) asm volatile("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    else asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int OP> __global__ void peak_sfu_kernel(float *out, int iters)
{
    float v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = threadIdx.x * 0.001f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = sfu<OP>(v[i]);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void peak_ffma_kernel(float *out, int iters, float a, float b)
{
    float v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = threadIdx.x * 0.001f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = fmaf(v[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void peak_ffma2_kernel(float *out, int iters, float a, float b)
{
    float2 v[8];
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = make_float2(threadIdx.x * 0.001f + i, threadIdx.x * 0.002f + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __ffma2_rn(v[i], a2, b2);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i].x + v[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int NF> __global__ void peak_mix_kernel(float *out, int iters, float a, float b)
{
    float v[16], w[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) { v[i] = threadIdx.x * 0.001f + i; w[i] = v[i] + 1.f; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            v[i] = sfu<0>(v[i]);
#pragma unroll
            for (int j = 0; j < NF; ++j) w[(i + j) & 15] = fmaf(w[(i + j) & 15], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i] + w[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace game

using namespace game;

extern "C" int game_microbench(game_ctx *c, int kind, int param, double *ops_per_s, double *ms_out)
{
    if (!c || !ops_per_s) return GAME_ERR_INVALID_ARG;
    if (kind < GAME_PEAK_FFMA || kind > GAME_PEAK_TANH_MIX) return fail(c, GAME_ERR_INVALID_ARG, "game_microbench: unknown kind");
    if (kind == GAME_PEAK_TANH_MIX && (param < 0 || param > 8)) return fail(c, GAME_ERR_INVALID_ARG, "game_microbench: 0 <= FMA per tanh <= 8");
    DeviceGuard dg(c);
    const int warps = 16, threads = warps * 32, blocks = c->sm_count, iters = 20000;
    float *out = nullptr;
    GAME_CUDA(c, cudaMalloc(&out, (size_t)blocks * threads * sizeof(float)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto launch = [&](int it) {
        switch (kind) {
        case GAME_PEAK_FFMA: peak_ffma_kernel<<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
        case GAME_PEAK_FFMA2: peak_ffma2_kernel<<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
        case GAME_PEAK_TANH: peak_sfu_kernel<0><<<blocks, threads, 0, c->stream>>>(out, it); break;
        case GAME_PEAK_EX2: peak_sfu_kernel<1><<<blocks, threads, 0, c->stream>>>(out, it); break;
        default:
            switch (param) {
            case 0: peak_mix_kernel<0><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 1: peak_mix_kernel<1><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 2: peak_mix_kernel<2><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 3: peak_mix_kernel<3><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 4: peak_mix_kernel<4><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 5: peak_mix_kernel<5><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 6: peak_mix_kernel<6><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            case 7: peak_mix_kernel<7><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            default: peak_mix_kernel<8><<<blocks, threads, 0, c->stream>>>(out, it, 1.0001f, 0.5f); break;
            }
        }
    };
    launch(200);                                   // warm-up
    cudaEventRecord(e0, c->stream);
    launch(iters);
    cudaEventRecord(e1, c->stream);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    c->launches += 2;
    if (e != cudaSuccess) return cuda_fail(c, e, "game_microbench");
    *ops_per_s = (double)blocks * threads * 16.0 * iters / (ms * 1e-3);     // 16 FMA (8 FFMA2) / 16 special-function ops per thread and iteration
    if (ms_out) *ms_out = ms;
    return GAME_OK;
}
