// Device-side pieces of the GA operators shared by ga.cu and evolve_persistent.cu: the counter-based generator and the
// exact integer -> decision / float mappings (DESIGN R0-R6), the operator arguments and parent selection (a9).
#pragma once
#include "game_internal.cuh"

namespace game {

enum { TAG_INIT = 0, TAG_SELECT = 1, TAG_XOVER = 2, TAG_MUTATE = 3 };

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011): ten rounds of two 32x32->64 multiplies ---------
struct W4 { uint32_t x, y, z, w; };

__device__ __forceinline__ W4 philox(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += W0; k1 += W1;
    }
    return W4{c0, c1, c2, c3};
}

__device__ __forceinline__ W4 draw(unsigned long long seed, uint32_t a, uint32_t b, uint32_t g, uint32_t tag)
{
    return philox((uint32_t)seed, (uint32_t)(seed >> 32), a, b, g, tag);
}

// ---- R0: integer -> decision / float, exact ---------------------------------------------------------
__device__ __forceinline__ uint32_t idx_of(uint32_t w, uint32_t n) { return __umulhi(w, n); }
__device__ __forceinline__ float upm1(uint32_t w) { return (float)((int)(w >> 8) - 8388608) * 1.1920928955078125e-7f; }
__device__ __forceinline__ float u01(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-8f; }

struct Thr { uint32_t thr; int always; };
inline Thr host_thr(float p)      // floor(p * 2^32) in double: p is a float, so the product is exact
{
    Thr t;
    if (p >= 1.0f) { t.always = 1; t.thr = 0xFFFFFFFFu; return t; }
    t.always = 0;
    t.thr = p > 0.0f ? (uint32_t)((double)p * 4294967296.0) : 0u;
    return t;
}
__device__ __forceinline__ bool hit(uint32_t w, Thr t) { return t.always || w < t.thr; }

// ---- a8-a11: one CTA per elite slot or per child pair -------------------------------------------------
struct StepArgs {
    int P, K, e, elite_mode, selection, tsize, npairs;
    Thr pc, pm;
    unsigned long long seed;
    uint32_t gen;
    C16Sink sink;        // the next fitness call's fp16 copy of `next`, written alongside (ptr == nullptr: none)
};

__device__ __forceinline__ int select_parent(const StepArgs &a, uint32_t slot, const int *__restrict__ order,
                             const unsigned long long *__restrict__ prefix)
{
    if (a.selection == GAME_SEL_ROULETTE) {
        W4 w = draw(a.seed, 0u, slot, a.gen, TAG_SELECT);
        unsigned long long total = prefix[a.P - 1];
        unsigned long long u = ((unsigned long long)w.x << 32) | w.y;
        unsigned long long T = __umul64hi(u, total);
        int lo = 0, hi = a.P - 1;                  // first r with prefix[r] > T
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (prefix[mid] > T) hi = mid; else lo = mid + 1;
        }
        return order[lo];
    }
    uint32_t best = 0xFFFFFFFFu;
    W4 w{0, 0, 0, 0};
    for (int j = 0; j < a.tsize; ++j) {
        if ((j & 3) == 0) w = draw(a.seed, (uint32_t)(j >> 2), slot, a.gen, TAG_SELECT);
        uint32_t word = (j & 3) == 0 ? w.x : (j & 3) == 1 ? w.y : (j & 3) == 2 ? w.z : w.w;
        best = min(best, idx_of(word, (uint32_t)a.P));
    }
    return order[best];
}

// host: the operator arguments of one generation from the ABI's parameters (sink left empty)
void fill_step_args(const game_ctx *ctx, const game_ga_params *gp, unsigned long long seed, unsigned int gen_base, StepArgs *out);

}  // namespace game
