// game_rank_static: the rank step (a6; "sort the population by fitness", DESIGN G20) for callers
// that must not allocate device memory.
//
// Who this is for.  game_rank borrows P ints of counting scratch from the stream-ordered allocator on every call
// (cudaMallocAsync / cudaFreeAsync).  Some hosts of this library cannot afford that:
//   - a process in which another component owns the device's memory (a framework's caching allocator or a serving
//     engine that reserved the whole of HBM up front): a driver allocation there can fail, or evict what that
//     component keeps cached;
//   - a latency-critical loop that may not take the driver's allocation path at all (its locks, a possible device-wide
//     synchronisation when a pool has to grow or trim) between two kernels;
//   - code that runs after set-up under a "no driver allocations from here on" rule, as long-running services often
//     impose so that an out-of-memory can only happen at start-up.
// For them the scratch lives in the library image itself: one file-scope __device__ array of GAME_RANK_STATIC_MAX_P
// ints (256 KiB).  Every GPU that loads libgame_b200.so carries that array from module load until the process exits,
// whether or not this entry point is ever called -- which is why the limit is modest.
//
// What follows from sharing ONE array per device:
//   - the array holds whatever the previous call left in it, so each call first clears the P ints it is going to
//     count into (a cudaMemsetAsync on the caller's stream -- no allocation);
//   - two calls whose kernels can overlap on the same GPU (different streams without an ordering between them,
//     several host threads) would count into the same ints and corrupt each other: callers must order them;
//   - nothing here touches game_rank or any context: the kernels below are this file's own copies of the counting
//     rank, reading the same sort_key() as every other rank in the library, so the order they give is the same.
//
// The array's NAME is only meaningful in device code.  On the host, `g_rank_scratch` is a stand-in symbol of the
// host image, not a device address, so the host side asks the runtime for the real address once per device
// (cudaGetSymbolAddress with that device current) and hands that pointer to the kernels.
#include "game_internal.cuh"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace {

constexpr int MAXP = GAME_RANK_STATIC_MAX_P;
constexpr int MAX_DEVICES = 64;
constexpr int RS_T = 128, RS_Q = 256;      // chromosomes per CTA x keys per CTA, as in ga.cu's rank

static __device__ __align__(256) int g_rank_scratch[MAXP];

std::mutex g_mu;
int *g_scratch_addr[MAX_DEVICES];          // device address of g_rank_scratch on each device, nullptr until set up
thread_local char g_err[256];

int rs_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

// cnt[p] += number of keys in this CTA's slab of RS_Q chromosomes that sort before chromosome p's key.
// key = (sort_key(error), index): NaN as +inf, -0 as +0, ties broken by the lower index (DESIGN G20).
__global__ void rank_static_count_kernel(const float *__restrict__ fit, int P, int *__restrict__ cnt)
{
    __shared__ unsigned long long keys[RS_Q];
    const int p = blockIdx.x * RS_T + threadIdx.x;
    const int q0 = blockIdx.y * RS_Q;
    for (int i = threadIdx.x; i < RS_Q; i += RS_T) {
        const int q = q0 + i;
        keys[i] = q < P ? (((unsigned long long)game::sort_key(fit[q]) << 32) | (unsigned)q) : ~0ull;
    }
    __syncthreads();
    if (p >= P) return;
    const unsigned long long mine = ((unsigned long long)game::sort_key(fit[p]) << 32) | (unsigned)p;
    int c = 0;
#pragma unroll 8
    for (int i = 0; i < RS_Q; ++i) c += keys[i] < mine;
    if (c) atomicAdd(&cnt[p], c);              // integer adds: exact in any order; cnt was cleared by this call
}

__global__ void rank_static_scatter_kernel(int P, const int *__restrict__ cnt, int *__restrict__ order)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < P) order[cnt[p]] = p;              // the keys are distinct, so cnt is a permutation of 0..P-1
}

// Device address of the static scratch on the CURRENT device; looked up once per device.
int scratch_for_current_device(int **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return rs_fail(GAME_ERR_CUDA, "game_rank_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES)
        return rs_fail(GAME_ERR_UNSUPPORTED, "game_rank_static: device ordinal %d is beyond the %d this entry point tracks", dev, MAX_DEVICES);
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_addr[dev]) {
        int *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_rank_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return rs_fail(GAME_ERR_CUDA, "game_rank_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return GAME_OK;
}

}  // namespace

extern "C" int game_rank_static(const float *fit, int P, int *order, void *cuda_stream)
{
    g_err[0] = 0;
    if (!fit || !order) return rs_fail(GAME_ERR_INVALID_ARG, "game_rank_static: NULL pointer");
    if (P < 1) return rs_fail(GAME_ERR_INVALID_ARG, "game_rank_static: P = %d, need P >= 1", P);
    if (P > MAXP)
        return rs_fail(GAME_ERR_INVALID_ARG, "game_rank_static: P = %d exceeds GAME_RANK_STATIC_MAX_P = %d, the size of the "
                       "library's built-in scratch; use game_rank (which allocates) for larger populations", P, MAXP);
    int *cnt = nullptr;
    int rc = scratch_for_current_device(&cnt);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemsetAsync(cnt, 0, (size_t)P * sizeof(int), s);
    if (e != cudaSuccess) return rs_fail(GAME_ERR_CUDA, "game_rank_static: clearing the scratch: %s", cudaGetErrorString(e));
    dim3 grid((P + RS_T - 1) / RS_T, (P + RS_Q - 1) / RS_Q);
    rank_static_count_kernel<<<grid, RS_T, 0, s>>>(fit, P, cnt);
    e = cudaGetLastError();
    if (e != cudaSuccess) return rs_fail(GAME_ERR_CUDA, "game_rank_static: count kernel launch: %s", cudaGetErrorString(e));
    rank_static_scatter_kernel<<<(P + 255) / 256, 256, 0, s>>>(P, cnt, order);
    e = cudaGetLastError();
    if (e != cudaSuccess) return rs_fail(GAME_ERR_CUDA, "game_rank_static: scatter kernel launch: %s", cudaGetErrorString(e));
    return GAME_OK;
}

extern "C" const char *game_rank_static_error(void) { return g_err; }
