// Device-side building blocks shared by the tensor-core kernels (fitness_tc.cu, evolve_persistent.cu): tile constants,
// the PTX wrappers for mbarrier / TMA / tcgen05 / TMEM, and the fused epilogue (activation, error, row sum; eq. 2-5, eq. 10
// of the paper).  Everything here is inline device code.
#pragma once
#include <cuda.h>

#include "game_internal.cuh"

namespace game {

constexpr int BM = 128;            // chromosomes per CTA  = TMEM lanes
constexpr int BN = 256;            // patterns per tile    = TMEM columns of one accumulator
constexpr int BKB = TC_KBLK;       // 64 fp16 = one 128-byte swizzle row per k-block
constexpr int UMMA_K = 16;
constexpr int A_BYTES = BM * BKB * 2;
// ---- PTX wrappers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// arrive on the barrier at the same offset in CTA `rank` of the cluster.  Default semantics (release at CTA scope):
// what is handed over lives in the ARRIVING CTA's own shared / tensor memory and is made visible there beforehand
// (tcgen05.fence / fence.proxy.async + a CTA barrier); only the signal crosses to the peer.  A cluster-scope release
// costs a GPU-wide memory barrier per arrival (measured: it alone bounded the generator variant at 47 % tensor-pipe use).
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar, uint32_t rank)
{
    asm volatile("{\n\t.reg .b32 ra;\n\tmapa.shared::cluster.u32 ra, %0, %1;\n\t"
                 "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}" ::"r"(bar), "r"(rank) : "memory");
}
// SUSPEND: pass a suspend-time hint, so a waiting thread sleeps in hardware instead of re-probing the barrier.  Measured
// on B200, same box, all waits of the kernel switched together: config 5 kernel 2.34 -> 2.20 ms, config 4 0.243 -> 0.238 ms
// (deep contractions: the producer, the MMA issuer and the epilogue all wait for long stretches), config 3 0.143 -> 0.145 ms
// (shallow: wake-up latency counts).  The kernel therefore uses it exactly where it uses the eight-warp epilogue.
// A wait that never completes is a protocol bug and must fail loudly instead of hanging the device; the bound is
// wall-clock time (globaltimer, looked at every 2^16 probes), not a probe count, so a debugger, time-slicing or a
// profiler replay that stalls the kernel for a while cannot trip it.
constexpr unsigned long long MBAR_TIMEOUT_NS = 20ull * 1000 * 1000 * 1000;
// (t0 travels by value: a reference would pin it to a stack slot and put a local store into every wait loop)
static __device__ __noinline__ unsigned long long mbar_timeout_check(unsigned long long t0)
{
    unsigned long long now;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
    if (t0 == 0) return now;
    if (now - t0 > MBAR_TIMEOUT_NS) __trap();
    return t0;
}
template <bool SUSPEND = false>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok = 0;
    unsigned long long t0 = 0;
    for (uint32_t spin = 0; !ok; ++spin) {
        if (SUSPEND)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(ok) : "r"(bar), "r"(parity), "r"(0x989680u) : "memory");
        else
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if ((spin & 0xFFFFu) == 0xFFFFu) t0 = mbar_timeout_check(t0);
    }
}
// the same wait with the probing loop out of line: one try_wait on the fast path (for waits that mostly succeed at once
// and sit in code that is inlined many times)
// (a suspend-time hint in the out-of-line loop changes nothing: 0.2565 vs 0.2566 ms on config 4)
static __device__ __noinline__ void mbar_wait_slow(uint32_t bar, uint32_t parity) { mbar_wait<false>(bar, parity); }
__device__ __forceinline__ void mbar_wait_lean(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (!ok) mbar_wait_slow(bar, parity);
}
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// setmaxnreg for the calling warpgroup (all four warps must execute it together)
template <int REGS> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS)); }
template <int REGS> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS)); }
// one lane of the (converged) warp; the same lane every time (elect.sync is deterministic for a given member mask)
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// all state spaces: orders this thread's generic-proxy accesses (global stores included) with async-proxy (TMA) ones
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

template <int CG>
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar)
{
    if (CG == 1) {
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                     ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
    } else {    // both CTAs of the pair issue; the bytes are accounted on the LEADER's barrier (rank 0)
        asm volatile("{\n\t.reg .b32 rb;\n\tmapa.shared::cluster.u32 rb, %4, 0;\n\t"
                     "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [rb];\n\t}"
                     ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
    }
}

// plain (non-tensor) bulk copy global -> this CTA's shared memory, completion counted on an mbarrier; 16-byte granular
__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

template <int CG> __device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols)
{
    if (CG == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    } else {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
}
template <int CG> __device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols)
{
    if (CG == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
    else asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}

// D[tmem] (+)= A[smem] . B[smem]^T, both operands K-major
template <int CG>
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    if (CG == 1) {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
    } else {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
    }
}

// arrive on `bar` (same offset in every CTA of the pair) once all MMAs issued so far have completed
template <int CG> __device__ __forceinline__ void umma_commit(uint32_t bar)
{
    if (CG == 1) {
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
    } else {
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                     ::"r"(bar), "h"((unsigned short)3) : "memory");
    }
}

// shared-memory matrix descriptor: K-major tile of [rows x 64] fp16, 128-byte swizzle, 8-row groups 1024 B apart
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((addr & 0x3FFFF) >> 4);          // start address, 16-byte units        bits [0,14)
    d |= (uint64_t)1 << 16;                          // leading byte offset (unused here)   bits [16,30)
    d |= (uint64_t)(1024 >> 4) << 32;                // stride byte offset: 8 rows x 128 B  bits [32,46)
    d |= (uint64_t)1 << 46;                          // descriptor version (sm_100)         bits [46,48)
    d |= (uint64_t)2 << 61;                          // layout: SWIZZLE_128B                bits [61,64)
    return d;
}

// instruction descriptor, kind::f16: fp16 x fp16 -> fp32, both K-major, M x N tile
__host__ __device__ constexpr uint32_t make_idesc(int M, int N)
{
    return (1u << 4)                 // D format: F32
         | (0u << 7) | (0u << 10)    // A, B format: F16
         | (0u << 15) | (0u << 16)   // A, B major: K
         | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
// Wait for this warp's outstanding TMEM loads.  The loaded registers pass through the statement as in/out operands, so
// the compiler can neither read them before the wait nor start on them early: consumers stay BELOW this point and the
// evaluation of the previous chunk stays ABOVE the next tmem_ld32 into the same registers.  Without that tie ptxas
// interleaves the two chunks and the warp blocks on the load it was meant to overlap (measured: config 3, K = 112).
__device__ __forceinline__ void tmem_ld_wait(uint32_t (&v)[32])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3]), "+r"(v[4]), "+r"(v[5]), "+r"(v[6]), "+r"(v[7]),
                   "+r"(v[8]), "+r"(v[9]), "+r"(v[10]), "+r"(v[11]), "+r"(v[12]), "+r"(v[13]), "+r"(v[14]), "+r"(v[15]),
                   "+r"(v[16]), "+r"(v[17]), "+r"(v[18]), "+r"(v[19]), "+r"(v[20]), "+r"(v[21]), "+r"(v[22]), "+r"(v[23]),
                   "+r"(v[24]), "+r"(v[25]), "+r"(v[26]), "+r"(v[27]), "+r"(v[28]), "+r"(v[29]), "+r"(v[30]), "+r"(v[31])
                 :: "memory");
}

__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Epilogue modes (template parameter ACT): the two activations of the ABI plus a cheaper logistic form.
//   0 sigmoid, 1/(1+2^(-z log2 e)) with ex2.approx + rcp.approx: 2 MUFU ops per evaluation
//   1 identity
//   2 sigmoid as 0.5 + 0.5 tanh(z/2) with tanh.approx.f32: 1 MUFU op per evaluation.  Measured against the
//     oracle on configs 2 and 3 (512 chromosomes x 3 gene distributions x MSE/TMSE) its fitness error is
//     indistinguishable from mode 0's (both dominated by the fp16 operand rounding, max 5e-4 relative, no
//     bias), and the MUFU-bound config 3 runs 1.4x faster, so it is the default.  A packed
//     tanh.approx.f16x2 form (0.5 MUFU per evaluation) was measured too: biased by -2e-4 and slower; dropped.
// In mode 2 the staged targets are t - 0.5 and the fp16 genes are pre-halved (a power-of-two scale: the same
// rounding), so the accumulator is z/2 and r = (t - 0.5) - 0.5 tanh(z/2) is one MUFU + one FFMA.
// Arithmetic is issued two evaluations at a time with the packed fp32 instructions of sm_100
// (FMUL2 / FFMA2), which halves the FMA-pipe issue slots the epilogue needs.
constexpr int MODE_SIG_EXACT = 0, MODE_IDENTITY = 1, MODE_SIG_TANH32 = 2;
constexpr int RATIONAL_SHARE_AUTO = 3;      // of 16 evaluation pairs: the measured best on config 3

__device__ __forceinline__ float tanh_approx(float x) { float y; asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// residual r = t - act(z) for two evaluations
template <int ACT> __device__ __forceinline__ float2 residual2(float2 z, float2 t)
{
    if (ACT == MODE_SIG_EXACT) {
        float2 a = __fmul2_rn(z, make_float2(-1.4426950408889634f, -1.4426950408889634f));
        float2 d = __fadd2_rn(make_float2(ex2_approx(a.x), ex2_approx(a.y)), make_float2(1.0f, 1.0f));
        return __ffma2_rn(make_float2(rcp_approx(d.x), rcp_approx(d.y)), make_float2(-1.0f, -1.0f), t);
    } else if (ACT == MODE_IDENTITY) {
        return __ffma2_rn(z, make_float2(-1.0f, -1.0f), t);
    } else {
        // the accumulator already holds z/2: pop_to_f16_kernel halves the genes (exact in fp16) in this mode
        return __ffma2_rn(make_float2(tanh_approx(z.x), tanh_approx(z.y)), make_float2(-0.5f, -0.5f), t);
    }
}

// The logistic of TWO evaluations on the FMA pipe with ONE special-function op (SURVEY 7 "hard parts"):
//   tanh(x) ~ x P(u) / Q(u),  u = x^2,  P, Q of degree 2 in u, x clamped to [-5, 5]
// a minimax fit (Lawson-weighted least squares on [0, 5], 4000 Chebyshev nodes): |error| <= 4.3e-5 inside the clamp and
// <= 1 - tanh(5) = 9.1e-5 beyond it -- five times tighter than tanh.approx.f32's 2^-11 -- and all coefficients are
// positive, so nothing cancels in fp32 (an odd polynomial of the same accuracy needs degree 21 and loses 1e-3 to
// cancellation).  The pair shares its reciprocal: r = 1 / (Q1 Q2), tanh(x1) = N1 Q2 r, tanh(x2) = N2 Q1 r.  Per
// evaluation: 8.5 FMA-pipe lane operations (packed FFMA2 / FMUL2), 2 FMNMX and HALF a special-function op, against ONE
// special-function op on the tanh.approx path.  The micro-benchmarks (profiles/r02_peaks.md) put the two pipes at 16 and
// 128 lanes/clk/SM, so sending a share s of the evaluations this way moves the epilogue's floor from 8 clk per warp
// evaluation to max(8 - 4 s, 3 + 7.5 s): 6.3 clk at s = 0.43.  The coefficients of P carry the -1/2 of
// r = (t - 1/2) - tanh(z/2) / 2.
__device__ __forceinline__ float2 residual2_rational(float2 x, float2 t)
{
    constexpr float A = 5.0f;
    constexpr float P0 = -0.5f * 9.998101439e-01f, P1 = -0.5f * 1.017231629e-01f, P2 = -0.5f * 6.549444594e-04f;
    constexpr float Q1 = 4.345040910e-01f, Q2 = 1.263918723e-02f;
    const float2 xc = make_float2(fminf(fmaxf(x.x, -A), A), fminf(fmaxf(x.y, -A), A));
    const float2 u = __fmul2_rn(xc, xc);
    float2 P = __ffma2_rn(u, make_float2(P2, P2), make_float2(P1, P1));
    P = __ffma2_rn(P, u, make_float2(P0, P0));
    float2 Q = __ffma2_rn(u, make_float2(Q2, Q2), make_float2(Q1, Q1));
    Q = __ffma2_rn(Q, u, make_float2(1.0f, 1.0f));
    const float2 N = __fmul2_rn(xc, P);                          // -x P(u) / 2
    const float r = rcp_approx(Q.x * Q.y);                       // Q >= 1, Q1 Q2 <= 391: no overflow, no division by zero
    const float2 M = __fmul2_rn(N, make_float2(Q.y, Q.x));
    return __ffma2_rn(M, make_float2(r, r), t);
}

// acc += e(r) for two evaluations; TMSE zeroes residuals inside the tube first (|r| <= R -> 0).  The tube test is
// one FSET per evaluation (a 1.0 / 0.0 mask) folded in by a packed multiply, instead of a compare + select pair.
template <bool TMSE> __device__ __forceinline__ void accumulate2(float2 r, float R, float2 &acc)
{
    if (TMSE) {
        const float2 m = make_float2(fabsf(r.x) > R ? 1.0f : 0.0f, fabsf(r.y) > R ? 1.0f : 0.0f);
        acc = __ffma2_rn(__fmul2_rn(r, m), r, acc);
    } else {
        acc = __ffma2_rn(r, r, acc);
    }
}

// 32 consecutive accumulator columns of this thread's chromosome against 32 staged targets; four independent
// running sums so the additions do not form one dependent chain
// SHARE (tanh mode only): of the chunk's 16 evaluation pairs, how many take the FMA-pipe rational form instead of
// tanh.approx; they are spread evenly over the chunk (pair q goes that way when floor((q+1) SHARE / 16) > floor(q SHARE / 16)),
// so the instruction stream alternates between the two pipes.
template <int ACT, int SHARE> __device__ __forceinline__ float2 residual_pair(int q, float2 z, float2 t)
{
    if (ACT == MODE_SIG_TANH32 && SHARE > 0 && ((q + 1) * SHARE) / 16 > (q * SHARE) / 16) return residual2_rational(z, t);
    return residual2<ACT>(z, t);
}
template <int ACT, bool TMSE, int SHARE = 0>
__device__ __forceinline__ void epilogue_chunk(const uint32_t (&v)[32], const float *ts, float R, float2 (&acc)[4])
{
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
        const float4 t4 = *reinterpret_cast<const float4 *>(ts + j);
        accumulate2<TMSE>(residual_pair<ACT, SHARE>(j >> 1, make_float2(__uint_as_float(v[j]), __uint_as_float(v[j + 1])), make_float2(t4.x, t4.y)), R,
                          acc[(j >> 1) & 3]);
        accumulate2<TMSE>(residual_pair<ACT, SHARE>((j >> 1) + 1, make_float2(__uint_as_float(v[j + 2]), __uint_as_float(v[j + 3])), make_float2(t4.z, t4.w)), R,
                          acc[((j >> 1) + 1) & 3]);
    }
}


}  // namespace game
