// a2-a5, TENSOR path: the N x K x P contraction on the 5th-generation tensor cores (tcgen05.mma,
// kind::f16: fp16 operands -- the same 11-bit significand as TF32 at twice the rate and half the bytes --
// fp32 accumulate in TMEM) with the activation, error and per-chromosome reduction fused in the epilogue
// (eq. 2-5, eq. 9-10).  z never leaves the SM.
//
// Orientation: chromosomes sit on the MMA's M axis (TMEM lanes), patterns on its N axis (TMEM columns),
// so an epilogue thread owns ONE chromosome, walks its row of the accumulator and sums the errors of the
// tile's patterns in a register: no shuffles, targets are a shared-memory broadcast.
//
// Persistent, warp-specialised CTAs (one per SM, or one CTA pair per two SMs with cta_group::2):
//   warp 0      TMA producer: 128B-swizzled [rows x 64] fp16 boxes of C (A operand) and E (B operand)
//               into a ring of shared-memory stages, completion on mbarriers
//   warp 1      TMEM allocator and the MMA issuer (the whole warp walks the loop, one elected lane issues);
//               tcgen05.commit frees stages and publishes finished accumulators
//   warps 2-9   epilogue: tcgen05.ld the accumulator (two 128x256 fp32 buffers = all 512 TMEM columns, so
//               the epilogue of tile i overlaps the MMAs of tile i+1), sigmoid, error, row sum, one
//               coalesced store per warp into partial[slab][p]
// (The regenerated variant, SRC_GEN, lays its roles out by warpgroup instead: {TMA, MMA, relay, idle}, two epilogue
// warpgroups, four generator warpgroups -- 896 threads, registers moved between the groups with setmaxnreg.)
// Tiles are ordered chromosome-block fastest so CTAs running together share the same E tile out of L2.
// finalize_kernel (fitness_fp32.cu) then adds the slabs in fixed order: no float atomics, bit-reproducible,
// and a chromosome's result does not depend on its row (DESIGN P20).
#include "tc_common.cuh"

namespace game {

constexpr int WARP_TMA = 0, WARP_MMA = 1, WARP_EPI0 = 2;      // warp roles; the epilogue warps follow (EW = 8 or 16 of them)
// Where the B operand (the expansion tile) comes from:
//   SRC_TMA  streamed from the materialised E16 in HBM, together with the A (population) tile, through a TMA ring
//   SRC_GEN  regenerated from X inside the kernel by sixteen generator warps writing 128B-swizzled k-blocks straight
//            into shared memory, with the whole population tile RESIDENT in shared memory (small populations:
//            one CTA pair covers all chromosomes, so every expansion value is generated exactly once per launch)
//   SRC_RES  the resident population tile of SRC_GEN, with the B halves streamed from E16 by TMA into the same ring
//            (isolates what residency alone buys: a third of the L2 -> SM traffic of SRC_TMA at P = 256)
constexpr int SRC_TMA = 0, SRC_GEN = 1, SRC_RES = 2;
constexpr int GEN_WARPS = 16;           // generator threads: (pattern row of this CTA's 128-row B half, feature group)
constexpr int GEN_GROUPS = GEN_WARPS / 4; // feature groups (of 8) the generator covers: F <= 32
constexpr int GEN_EW = 8;               // epilogue warps of the generator variant (four were the bottleneck once the generator was fast: 0.257 vs 0.222 ms)
constexpr int GEN_STAGES = 4;           // B k-block stages of the generator ring
constexpr int GEN_B_BYTES = 128 * BKB * 2;
constexpr int GEN_THREADS = 128 + 32 * GEN_EW + 32 * GEN_WARPS;      // warpgroups: {TMA, MMA, relay, idle}, 2 x epilogue, 4 x generators
// setmaxnreg: an 896-thread CTA starts at 72 registers per thread; the first warpgroup hands registers to the epilogue.
// Measured on config 4: 40 / 88 / 72 (first warpgroup / epilogue / generators) 0.217 ms; 40 / 104 / 64 (generators spill)
// 0.269 ms; one epilogue warpgroup on 768 threads, 56 / 128 / 72: 0.257 ms.
constexpr int GEN_REGS_START = 72, GEN_REGS_LOW = 40, GEN_REGS_GEN = 72, GEN_REGS_EPI = 88;
static_assert((GEN_STAGES & (GEN_STAGES - 1)) == 0, "ring slot = k-block count mod GEN_STAGES");
static_assert(128 * GEN_REGS_LOW + 32 * GEN_WARPS * GEN_REGS_GEN + 32 * GEN_EW * GEN_REGS_EPI <= GEN_REGS_START * GEN_THREADS, "register pool of the CTA");
static_assert(GEN_REGS_START * GEN_THREADS <= 65536, "register file");
constexpr int GEN_BAR0 = 2;             // named barriers 2.. : one per generator stage (0 = CTA, 1 = epilogue)
constexpr int MAX_STAGES = 6;           // barrier slots are laid out for the deepest ring
constexpr int TC_TAIL_BYTES = 256 /*barriers*/ + 3 * BN * 4 /*targets: [3][BN], or [team][2][BN]*/ + 2 * 4 * BM * 4 /*column-block error sums of two tiles*/;

template <int CG> struct Cfg {
    static constexpr int BNL = BN / CG;                 // pattern rows this CTA stages
    static constexpr int B_BYTES = BNL * BKB * 2;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int STAGES = CG == 1 ? 4 : 6;
    static constexpr int SMEM = STAGES * STAGE_BYTES + 1024 /*align*/ + TC_TAIL_BYTES;
};


// ---- a1 inside the kernel: the generator warps of the SRC_GEN variant ---------------------------------------
// 512 generator threads per CTA: thread (row, g) owns feature group g (eight features, four packed pairs) of one pattern
// row of this CTA's half of the 256-pattern tile.  It writes the group's chunks, 16 bytes (8 fp16 = one swizzle chunk) at
// a time, into the B ring exactly where a 128B-swizzled TMA box would have put them: chunk j of row r of a k-block lives at
// r*128 + ((j ^ (r & 7)) << 4).  With the term-type-major order of game_internal.cuh's tc_position() chunk c = tau * G + g,
// so the thread's chunks lie G <= 4 apart: they come in ascending k-block order as it steps its recurrences, every thread
// owns a chunk of every k-block, and all generator threads move from stage to stage together, one step at a time.
//   Chebyshev (G7, G9):  T_{-1} = x, T_0 = 1, T_{m+1} = 2x T_m - T_{m-1}
//   trigonometric (eq. 8-9):  the constant term is cos 0x; cos / sin mx = 2 cos x . cos / sin (m-1)x - cos / sin (m-2)x
//   started from cos(-x), cos 0x and sin(-x), sin 0x -- no special cases inside the loops
// in fp32 (packed FFMA2; the recurrences' error grows like m^2 eps / 2: 3e-5 at m = 32, far below fp16's 2^-11), rounded
// once to fp16.  The new value of a recurrence overwrites the older one in place (ping-pong, no register moves).  Rows
// beyond N generate zeros (their start values are 0), matching the zero padding of the materialised E16.
// A stage is published by the async-proxy fence + a (non-blocking) arrival on the stage's named barrier; the relay warp
// completes that barrier and performs the one mbarrier arrival per CTA and stage.
__device__ __forceinline__ uint32_t pack_half2(float2 v)
{
    __half2 h = __floats2half2_rn(v.x, v.y);
    return *reinterpret_cast<uint32_t *>(&h);
}
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }

template <int FAMILY>
__device__ __forceinline__ void generate_expansion(const float *__restrict__ X, int F, int d, long long N, int k_blocks,
                                                   int pair, int n_pairs, int total_tiles, int cta_rank, int gt,
                                                   uint32_t bring, uint32_t bar0)
{
    const int g = gt >> 7, row = gt & 127;             // g is warp-uniform
    int G = (F + 7) >> 3;
    if (g >= G) return;                                // fewer feature groups than generator warpgroups
    const int T = tc_terms_per_feature(FAMILY, d);
    int bar_count = 128 * G + 32;                      // the active generator warps + the relay warp
    const int nchunks = k_blocks * 8;
    // this row of ring slot 0, with the row's swizzle term folded in: chunk j lives at (row address) ^ (j << 4)
    uint32_t my_row = (bring + (uint32_t)row * 128u) ^ ((uint32_t)(row & 7) << 4);
    uint32_t empty0 = bar0 + 8u * MAX_STAGES;
    // (opaque to the compiler from here on: it would otherwise re-derive them from special registers at every use)
    asm volatile("" : "+r"(my_row), "+r"(empty0), "+r"(G), "+r"(bar_count));
    const bool vec = (F & 3) == 0;
    uint32_t it = 0;                                   // k-blocks published so far: ring slot it % 4, phase (it / 4) & 1
    int c_end = 8;                                     // first chunk of the NEXT k-block of the tile
    uint32_t dst = my_row;
    mbar_wait(empty0, 1);                              // stage 0 starts free

    auto advance = [&]() {                             // publish the stage being written, move on to the next k-block
        fence_proxy_async();                           // generic-proxy stores -> visible to the tensor core's async proxy
        asm volatile("bar.arrive %0, %1;" ::"r"(GEN_BAR0 + (it & (GEN_STAGES - 1))), "r"(bar_count) : "memory");
        ++it;
        const uint32_t s = it & (GEN_STAGES - 1);
        dst = my_row + s * GEN_B_BYTES;
        mbar_wait_lean(empty0 + 8u * s, ((it / GEN_STAGES) & 1u) ^ 1u);     // the MMAs that read this slot last have retired
    };
    auto put = [&](int c, const float2 (&v)[4]) {      // chunk c of this thread's row
        if (c >= c_end) { advance(); c_end += 8; }
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                     ::"r"(dst ^ (((uint32_t)c << 4) & 0x70u)), "r"(pack_half2(v[0])), "r"(pack_half2(v[1])),
                       "r"(pack_half2(v[2])), "r"(pack_half2(v[3])) : "memory");
    };
    auto load_x = [&](int tile, float (&x)[8]) {       // this thread's features of its pattern (0 outside)
        const long long n = (long long)tile * BN + cta_rank * 128 + row;
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 0.f;
        if (tile >= total_tiles || n >= N) return;
        const float *xr = X + n * F + g * 8;
        if (vec) {
#pragma unroll
            for (int h = 0; h < 2; ++h)
                if (g * 8 + 4 * h < F) {
                    const float4 v = __ldg(reinterpret_cast<const float4 *>(xr) + h);
                    x[4 * h] = v.x; x[4 * h + 1] = v.y; x[4 * h + 2] = v.z; x[4 * h + 3] = v.w;
                }
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) if (g * 8 + j < F) x[j] = __ldg(xr + j);
        }
    };

    float xn[8];
    load_x(pair, xn);
    for (int tile = pair; tile < total_tiles; tile += n_pairs) {
        const long long n = (long long)tile * BN + cta_rank * 128 + row;
        const float one = n < N ? 1.f : 0.f;
        const float2 one2 = make_float2(one, one);
        int c = g;                                     // chunk of (tau, g): tau * G + g
        if (FAMILY == GAME_CHEB) {
            float2 ta[4], tb[4], x2[4];                // T_tau and T_{tau-1} (alternating), 2x
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float2 x = make_float2(xn[2 * j], xn[2 * j + 1]);
                ta[j] = one2; tb[j] = __fmul2_rn(x, one2); x2[j] = __fadd2_rn(x, x);
            }
            load_x(tile + n_pairs, xn);                // the next tile's features travel while this one is generated
            for (int tau = 0; tau <= d; tau += 2) {
                put(c, ta); c += G;
#pragma unroll
                for (int j = 0; j < 4; ++j) tb[j] = __ffma2_rn(x2[j], ta[j], neg2(tb[j]));
                if (tau + 1 <= d) {
                    put(c, tb); c += G;
#pragma unroll
                    for (int j = 0; j < 4; ++j) ta[j] = __ffma2_rn(x2[j], tb[j], neg2(ta[j]));
                }
            }
        } else {
            float2 C2[4], ca[4], cb[4], sa[4], sb[4];  // 2 cos x; cos (m-1)x / (m-2)x and sin (m-1)x / (m-2)x (alternating)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float2 Cv, Sv;
                __sincosf(xn[2 * j], &Sv.x, &Cv.x);                    // |x| <= pi is checked at load for this variant
                __sincosf(xn[2 * j + 1], &Sv.y, &Cv.y);
                C2[j] = __fadd2_rn(Cv, Cv);
                ca[j] = one2; cb[j] = __fmul2_rn(Cv, one2);                       // cos 0x, cos(-x)
                sa[j] = make_float2(0.f, 0.f); sb[j] = neg2(__fmul2_rn(Sv, one2)); // sin 0x, sin(-x)
            }
            load_x(tile + n_pairs, xn);
            put(c, ca); c += G;                        // tau = 0: the constant term
            for (int m = 1; m <= d; m += 2) {
#pragma unroll
                for (int j = 0; j < 4; ++j) cb[j] = __ffma2_rn(C2[j], ca[j], neg2(cb[j]));
                put(c, cb); c += G;                    // tau = 2m - 1: cos mx
#pragma unroll
                for (int j = 0; j < 4; ++j) sb[j] = __ffma2_rn(C2[j], sa[j], neg2(sb[j]));
                put(c, sb); c += G;                    // tau = 2m: sin mx
                if (m + 1 <= d) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) ca[j] = __ffma2_rn(C2[j], cb[j], neg2(ca[j]));
                    put(c, ca); c += G;
#pragma unroll
                    for (int j = 0; j < 4; ++j) sa[j] = __ffma2_rn(C2[j], sb[j], neg2(sa[j]));
                    put(c, sa); c += G;
                }
            }
        }
        const float2 zeros[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        for (; c < nchunks; c += G) put(c, zeros);     // K padded up to whole k-blocks (c = T * G + g here)
        advance();                                     // publish the tile's last k-block; on to the next tile's first stage
        c_end = 8;
    }
    (void)T;
}

// ---- the kernel -----------------------------------------------------------------------------------------
// BNT: patterns per tile, 256 or (SRC_TMA, single CTAs, team epilogue only) 128: problems of less than one wave of
// 256-pattern tiles finish sooner on twice as many half-size tiles (configs 1-2).
// SHARE: see epilogue_chunk.  k_last: UMMA k-steps (of 16 terms) that hold real terms in the LAST k-block -- the
// padding steps beyond them would multiply zeros (config 3: K = 112 = 7 steps, not 8) and are not issued.
template <int CG, int ACT, bool TMSE, int EW, int SRC, int FAMILY, bool TEAMS, int BNT = BN, int SHARE = 0>
__global__ void __launch_bounds__(SRC == SRC_GEN ? GEN_THREADS : 64 + 32 * EW, 1)
fitness_tc_kernel(const __grid_constant__ CUtensorMap tmC, const __grid_constant__ CUtensorMap tmE,
                  int n_tiles, int m_blocks, int k_blocks, long long N, const float *__restrict__ tgt, float R,
                  float *__restrict__ partial, int Ppad, const DevState *state,
                  const float *__restrict__ X, int F, int degree, int k_last, int kb_range)
{
    using C = Cfg<CG>;
    static_assert(SRC == SRC_TMA || CG == 2, "the generator variant runs as CTA pairs");
    static_assert(BNT == BN || (BNT == 128 && SRC == SRC_TMA && CG == 1 && TEAMS), "half-size tiles: streamed, single CTA, team epilogue");
    constexpr bool RESIDENT_A = SRC != SRC_TMA;
    constexpr bool SUSP = !TEAMS;                                          // see mbar_wait
    constexpr int B_BYTES_K = (BNT / CG) * BKB * 2;                        // B k-block bytes this CTA stages
    constexpr int STAGE_BYTES_K = A_BYTES + B_BYTES_K;
    constexpr int NSTAGES = RESIDENT_A ? GEN_STAGES : (STAGE_BYTES_K <= 32768 ? 6 : 4);
    static_assert(BNT != BN || (STAGE_BYTES_K == C::STAGE_BYTES && NSTAGES == (RESIDENT_A ? GEN_STAGES : C::STAGES)), "Cfg<CG> describes the full-size tile");
    // SRC_GEN: roles are laid out by warpgroup so that setmaxnreg can move registers between them
    constexpr int EPI0 = SRC == SRC_GEN ? 4 : WARP_EPI0;
    constexpr int WARP_GEN0 = EPI0 + EW, WARP_RELAY = 2;
    static_assert(SRC != SRC_GEN || EW == GEN_EW, "generator variant: whole epilogue warpgroups");
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - smem_u32(smem_raw));
    // operand area: SRC_TMA a ring of (A, B) k-block stages; SRC_GEN the resident A tile (k_blocks blocks) + a B ring
    const uint32_t ring_bytes = RESIDENT_A ? (uint32_t)(k_blocks * A_BYTES + GEN_STAGES * GEN_B_BYTES)
                                               : (uint32_t)(NSTAGES * STAGE_BYTES_K);
    const uint32_t bar0 = base + ring_bytes;
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (MAX_STAGES + s); };
    auto tfull_bar = [&](int a) { return bar0 + 8u * (2 * MAX_STAGES + a); };
    auto tempty_bar = [&](int a) { return bar0 + 8u * (2 * MAX_STAGES + 2 + a); };
    const uint32_t afull_bar = bar0 + 8u * (2 * MAX_STAGES + 4);      // SRC_GEN: the resident A tile has landed
    const uint32_t tmem_slot = bar0 + 8u * (2 * MAX_STAGES + 5);
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + ring_bytes + 8 * (2 * MAX_STAGES + 5));
    float *tgt_s = reinterpret_cast<float *>(gbase + ring_bytes + 256);   // [3][BN] (TEAMS: [2 teams][2][BN], reaching into sum_s)
    float *sum_s = tgt_s + 3 * BN;                                        // [2][4][BM]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t cta_rank = 0;
    if (CG == 2) asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(cta_rank));
    const int pair = blockIdx.x / CG, n_pairs = gridDim.x / CG;
    const int total_tiles = n_tiles * m_blocks;
    const int my_tiles = pair < total_tiles ? (total_tiles - pair + n_pairs - 1) / n_pairs : 0;     // this CTA (pair) takes tiles pair, pair + n_pairs, ...

    if (threadIdx.x == 0) {
        // SRC_GEN: a B stage is full when the generator warps of BOTH CTAs have published their half
        for (int s = 0; s < NSTAGES; ++s) { mbar_init(full_bar(s), SRC == SRC_GEN ? CG : 1); mbar_init(empty_bar(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), CG * (TEAMS ? 4 : EW) /* the epilogue warps (per CTA) that drain one accumulator */); }
        mbar_init(afull_bar, 1);
        fence_barrier_init();
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmC) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmE) : "memory");
    }
    if (warp == WARP_MMA) tmem_alloc<CG>(tmem_slot, 512);
    tc_fence_before();
    if (CG == 2) { asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory"); }
    else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;

    // Everything above touched only this CTA's own shared / tensor memory, so under programmatic dependent launch it
    // overlaps the tail of the previous kernel; from here on the kernel reads what its predecessors wrote.
    pdl_wait();
    const bool stopped = state && state->stopped;      // uniform across the grid: the loop has stopped, nothing to do

    // SRC_GEN lays the roles out by warpgroup and moves registers between them (setmaxnreg, inside the role branches so
    // that each one dominates its code): a 768-thread CTA starts with 80 registers per thread; the epilogue needs more
    // (two 32-register accumulator chunks in flight), the first warpgroup (TMA, MMA, relay) and the generators fewer
    if (SRC == SRC_GEN && warp >= WARP_GEN0) {
        // ===== generator warps (a1 inside the kernel) =====
        if (GEN_REGS_GEN < GEN_REGS_START) setmaxnreg_dec<GEN_REGS_GEN>();
        if (!stopped)
            generate_expansion<FAMILY>(X, F, degree, N, k_blocks, pair, n_pairs, total_tiles, (int)cta_rank,
                                       threadIdx.x - 32 * WARP_GEN0, base + k_blocks * A_BYTES, bar0);
    } else if (warp < EPI0) {
        if (SRC == SRC_GEN) setmaxnreg_dec<GEN_REGS_LOW>();
        if (stopped) {
        } else if (warp == WARP_TMA) {
            // ===== TMA producer =====
            if (lane == 0 && RESIDENT_A) {
                // the population tile is loaded ONCE and stays: block kb of this CTA's 128 chromosomes at base + kb * A_BYTES
                if (cta_rank == 0) mbar_expect_tx(afull_bar, (uint32_t)(CG * k_blocks * A_BYTES));
                for (int kb = 0; kb < k_blocks; ++kb)
                    tma_load_2d<CG>(base + kb * A_BYTES, &tmC, kb * BKB, (int)cta_rank * BM, afull_bar);
            }
            if (SRC == SRC_GEN) {
            } else if (SRC == SRC_RES) {
                if (lane == 0) {                                  // stream this CTA's 128-pattern half of every B k-block
                    int s = 0; uint32_t ph = 0;
                    for (int tile = pair; tile < total_tiles; tile += n_pairs) {
                        const int rowE = tile * k_blocks * BN + (int)cta_rank * 128;
                        for (int kb = 0; kb < k_blocks; ++kb) {
                            mbar_wait<SUSP>(empty_bar(s), ph ^ 1);
                            if (cta_rank == 0) mbar_expect_tx(full_bar(s), CG * GEN_B_BYTES);
                            tma_load_2d<CG>(base + k_blocks * A_BYTES + s * GEN_B_BYTES, &tmE, 0, rowE + kb * BN, full_bar(s));
                            if (++s == NSTAGES) { s = 0; ph ^= 1; }
                        }
                    }
                }
            } else if (lane == 0) {
                int s = 0; uint32_t ph = 0;
                for (int tile = pair; tile < total_tiles; tile += n_pairs) {
                    const int n_tile = tile / m_blocks, m_blk = tile % m_blocks;
                    const int rowC = (m_blk * CG + (int)cta_rank) * BM;
                    // E16 is tile-blocked [n/256][kb][256][64]: this tile's (and this CTA's) rows inside the 256-row block
                    const int n_first = n_tile * BNT + (int)cta_rank * (BNT / CG);
                    const int rowE = (n_first >> 8) * k_blocks * BN + (n_first & 255);
                    for (int kb = 0; kb < k_blocks; ++kb) {
                        mbar_wait<SUSP>(empty_bar(s), ph ^ 1);
                        const uint32_t sa = base + s * STAGE_BYTES_K, sb = sa + A_BYTES;
                        if (CG == 1 || cta_rank == 0) mbar_expect_tx(full_bar(s), CG * STAGE_BYTES_K);
                        tma_load_2d<CG>(sa, &tmC, kb * BKB, rowC, full_bar(s));
                        tma_load_2d<CG>(sb, &tmE, 0, rowE + kb * BN, full_bar(s));
                        if (++s == NSTAGES) { s = 0; ph ^= 1; }
                    }
                }
            }
        } else if (warp == WARP_MMA) {
            // ===== MMA issuer (leader CTA only when paired) =====
            // The whole warp walks the loop, so the ring position, the phases and the descriptors are warp-uniform values
            // (kept in uniform registers); one elected lane issues the MMAs and their commits.  (Running the loop in a
            // lane-0 branch instead made every tcgen05.mma cost ~25 instructions of vector -> uniform register traffic.)
            if (cta_rank == 0) {
                constexpr uint32_t idesc = make_idesc(BM * CG, BNT);
                int s = 0; uint32_t ph = 0;
                int acc = 0; uint32_t aph = 0;
                if (RESIDENT_A) mbar_wait<SUSP>(afull_bar, 0);          // resident population tile of both CTAs
                for (int t = 0; t < my_tiles; ++t) {
                    mbar_wait<SUSP>(tempty_bar(acc), aph ^ 1);          // epilogue has drained this accumulator
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BNT);
                    int kr = 0;                                         // k-block inside the current K range (wrap counter)
                    for (int kb = 0; kb < k_blocks; ++kb) {
                        mbar_wait<SUSP>(full_bar(s), ph);               // operands have landed (SRC_GEN: were generated)
                        tc_fence_after();
                        const uint32_t sa = RESIDENT_A ? base + kb * A_BYTES : base + s * STAGE_BYTES_K;
                        const uint32_t sb = RESIDENT_A ? base + k_blocks * A_BYTES + s * GEN_B_BYTES : sa + A_BYTES;
                        const uint64_t adesc = make_smem_desc(sa), bdesc = make_smem_desc(sb);
                        const bool last = kb + 1 == k_blocks;
                        // the last k-block of a K range stops at its real k-steps: padding steps would multiply zeros.  A wrap
                        // counter, NOT (kb + 1) % kb_range: the integer division by a run-time value sat on the issue path of
                        // every k-block and cost config 5 7 % (2.17 vs 2.01 ms, same box: profiles/r03_ab_cfg5.md)
                        const bool range_end = ++kr == kb_range;
                        if (range_end) kr = 0;
                        const int nk = range_end ? k_last : BKB / UMMA_K;
                        if (elect_one()) {
    #pragma unroll
                            for (int k = 0; k < BKB / UMMA_K; ++k) {
                                // advance 16 fp16 = 32 bytes inside the swizzle row: +2 in 16-byte units
                                if (k < nk) umma_f16<CG>(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) != 0);
                            }
                            umma_commit<CG>(empty_bar(s));            // stage reusable when these MMAs retire
                            if (last) umma_commit<CG>(tfull_bar(acc));  // accumulator complete
                        }
                        __syncwarp();
                        if (++s == NSTAGES) { s = 0; ph ^= 1; }
                    }
                    if (++acc == 2) { acc = 0; aph ^= 1; }
                }
            }
        } else if (SRC == SRC_GEN && warp == WARP_RELAY) {
            // ===== relay: the generators never stall on the hand-over -- each thread makes its stores visible to the async
            // proxy and arrives (non-blocking) on the stage's named barrier; this warp completes that barrier and performs
            // the one mbarrier arrival per CTA and stage on the leader's barrier =====
            const int G = (F + 7) >> 3;
            const int bar_count = 128 * (G < GEN_GROUPS ? G : GEN_GROUPS) + 32;
            int s = 0;
            for (int t = 0; t < my_tiles; ++t)
                for (int kb = 0; kb < k_blocks; ++kb) {
                    asm volatile("bar.sync %0, %1;" ::"r"(GEN_BAR0 + s), "r"(bar_count) : "memory");
                    if (lane == 0) {
                        if (cta_rank == 0) mbar_arrive(full_bar(s)); else mbar_arrive_cluster(full_bar(s), 0);
                    }
                    if (++s == GEN_STAGES) s = 0;
                }
        }
    } else {
        if (SRC == SRC_GEN) setmaxnreg_inc<GEN_REGS_EPI>();
        if (stopped) {
        } else if (TEAMS) {
            // ===== epilogue warps: two independent teams of four =====
            // Warp w may touch TMEM lanes 32*(w%4).., so four warps cover a tile's 128 chromosomes.  Team g (warps 4g..4g+3)
            // owns accumulator g and takes every other tile of this CTA's sequence: a thread walks ALL 256 pattern columns of
            // its chromosome, so the error sum of a tile is finished in registers (no cross-warp combine) and `partial` gets
            // one row per 256 patterns.  The two warps that share a scheduler belong to different teams and therefore to
            // different tiles at different stages: while one team waits for its accumulator's next MMA the other keeps the
            // special-function unit busy, which two warps marching through the same tile in lockstep could not.
            // Inside a tile the TMEM load of the next 32-column chunk is in flight while the current one is evaluated.
            // Targets are staged per team through two buffers (the team's one barrier per tile separates writer and
            // readers); the next tile's target is fetched a tile ahead.  Patterns beyond N carry the target that makes their
            // residual exactly zero (their expansion rows are zero, so z = 0): no masked code path.
            static_assert(!TEAMS || EW == 8, "two teams of four warps");
            constexpr int NCH = BNT / 32;               // 32-column chunks per tile: 8 (4 for half-size tiles)
            const int ew = warp - EPI0;
            const int team = ew >> 2;
            const int quarter = warp & 3;               // TMEM lane quarter this warp may touch
            const int tt = (ew & 3) * 32 + lane;        // thread index inside the team, 0..127
            constexpr float tbias = ACT == MODE_SIG_TANH32 ? 0.5f : 0.f;           // staged target = t - tbias
            constexpr float tneutral = ACT == MODE_SIG_EXACT ? 0.5f : 0.f;         // staged target of a padding pattern
            // raw targets of this thread's two patterns in `tile` (tneutral + tbias for a padding pattern); the bias comes
            // off when the values are staged one tile later, so nothing waits on the loads where they are issued
            auto fetch_targets = [&](int tile, float &t0v, float &t1v) {
                const long long n = (long long)(tile / m_blocks) * BNT + tt;
                t0v = n < N ? tgt[n] : tneutral + tbias;
                t1v = (BNT > 128 && n + 128 < N) ? tgt[n + 128] : tneutral + tbias;
            };
            auto team_barrier = [&]() { asm volatile("bar.sync %0, 128;" ::"r"(1 + team) : "memory"); };
            const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(team * BNT);
            const uint32_t tfull_b = tfull_bar(team), tempty_b = tempty_bar(team);
            const int row = quarter * 32 + lane;        // chromosome row inside the 128-row block
            const int step = 2 * n_pairs;
            uint32_t aph = 0; int tb = 0;
            uint32_t va[32], vb[32];
            float tn0 = 0.f, tn1 = 0.f;
            if (pair + team * n_pairs < total_tiles) fetch_targets(pair + team * n_pairs, tn0, tn1);
            for (int tile = pair + team * n_pairs; tile < total_tiles; tile += step) {
                const int n_tile = tile / m_blocks, m_blk = tile % m_blocks;
                float *ts = tgt_s + (team * 2 + tb) * BNT;
                ts[tt] = tn0 - tbias;
                if (BNT > 128) ts[tt + 128] = tn1 - tbias;
                if (tile + step < total_tiles) fetch_targets(tile + step, tn0, tn1);
                team_barrier();
                mbar_wait<SUSP>(tfull_b, aph);
                tc_fence_after();
                tmem_ld32(lane_addr, va);
                float2 acc2[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
    #pragma unroll
                for (int c = 0; c < NCH; ++c) {
                    uint32_t (&cur)[32] = (c & 1) ? vb : va;
                    uint32_t (&nxt)[32] = (c & 1) ? va : vb;
                    tmem_ld_wait(cur);
                    if (c + 1 < NCH) {
                        tmem_ld32(lane_addr + 32 * (c + 1), nxt);
                    } else {
                        // every TMEM read of this accumulator has completed: hand it back to the MMA warp right away
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) {
                            if (CG == 1) mbar_arrive(tempty_b);
                            else mbar_arrive_cluster(tempty_b, 0);
                        }
                    }
                    epilogue_chunk<ACT, TMSE, SHARE>(cur, ts + 32 * c, R, acc2);
                }
                partial[(long long)n_tile * Ppad + (m_blk * CG + (int)cta_rank) * BM + row] =
                    ((acc2[0].x + acc2[0].y) + (acc2[1].x + acc2[1].y)) + ((acc2[2].x + acc2[2].y) + (acc2[3].x + acc2[3].y));
                tb ^= 1;
                aph ^= 1;
            }
        } else {
            // ===== epilogue warps =====
            // EW warps: warp w may touch TMEM lanes 32*(w%4).., so four warps cover the 128 chromosomes and EW/4 such
            // groups split the tile's 256 pattern columns.  16 warps (4 per scheduler) keep the MUFU pipe fed where the
            // epilogue is the bound (shallow K); 8 leave more registers per thread.
            constexpr int NCB = EW / 4;                 // column blocks per tile
            constexpr int CBW = BN / NCB;               // columns per block: 128 or 64
            constexpr int NCH = CBW / 32;               // 32-column chunks per tile and warp: 4 or 2 (even)
            const int ew = warp - EPI0;
            const int quarter = warp & 3;               // TMEM lane quarter this warp may touch
            const int cb = ew >> 2;                     // which column block of the 256-column tile
            const int et = threadIdx.x - 32 * EPI0;
            // One continuous stream of 32-column chunks: the TMEM load of the next chunk -- the next TILE's first chunk
            // included -- is in flight while the current one is evaluated.  Targets are staged one tile ahead in a ring
            // of three buffers: the buffer written during tile i was last read in tile i-2, and the one barrier per tile
            // separates the two.  Patterns beyond N carry the target that makes their residual exactly zero (their
            // expansion rows are zero, so z = 0): no masked code path.  The column blocks' sums of a tile meet in shared
            // memory and are added in fixed order by block 0's warps one tile later: one partial row per 256 patterns.
            constexpr float tbias = ACT == MODE_SIG_TANH32 ? 0.5f : 0.f;           // staged target = t - tbias
            constexpr float tneutral = ACT == MODE_SIG_EXACT ? 0.5f : 0.f;         // staged target of a padding pattern
            // raw target of this thread's pattern in `tile` (tneutral + tbias for a padding pattern); the bias comes
            // off when the value is staged one tile later, so nothing waits on the load where it is issued
            constexpr int TPT = BN / (32 * EW) > 0 ? BN / (32 * EW) : 1;            // targets each epilogue thread stages per tile
            auto fetch_target = [&](int tile, int u) -> float {
                const int col = et + u * 32 * EW;
                const long long n = (long long)(tile / m_blocks) * BN + col;
                return (col < BN && n < N) ? tgt[n] : tneutral + tbias;
            };
            auto epi_barrier = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(32 * EW) : "memory"); };
            const int row = quarter * 32 + lane;        // chromosome row inside the 128-row block
            long long prev_off = -1;                    // where the previous tile's sum goes in `partial`
            auto flush = [&](int buf) {                 // block 0's warps: add the tile's column-block sums, ascending
                if (cb == 0 && prev_off >= 0) {
                    const float *ss = sum_s + buf * 4 * BM + row;
                    float s = ss[0];
    #pragma unroll
                    for (int j = 1; j < NCB; ++j) s += ss[j * BM];
                    partial[prev_off] = s;
                }
            };
            const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(cb * CBW);
            int acc = 0; uint32_t aph = 0; int tb = 0, sb = 0;
            uint32_t va[32], vb[32];
            float t_next[TPT];
#pragma unroll
            for (int u = 0; u < TPT; ++u) t_next[u] = 0.f;
            if (pair < total_tiles) {
#pragma unroll
                for (int u = 0; u < TPT; ++u) {
                    if (et + u * 32 * EW < BN) tgt_s[et + u * 32 * EW] = fetch_target(pair, u) - tbias;
                    if (pair + n_pairs < total_tiles) t_next[u] = fetch_target(pair + n_pairs, u);
                }
                epi_barrier();
                mbar_wait<SUSP>(tfull_bar(0), 0);
                tc_fence_after();
                tmem_ld32(lane_addr, va);
            }
            for (int tile = pair; tile < total_tiles; tile += n_pairs) {
                const int n_tile = tile / m_blocks, m_blk = tile % m_blocks;
                const bool has_next = tile + n_pairs < total_tiles;
                const uint32_t t0 = lane_addr + (uint32_t)(acc * BN);
                const float *ts = tgt_s + tb * BN + cb * CBW;
                const int tbn = tb == 2 ? 0 : tb + 1;
                float2 acc2[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
    #pragma unroll
                for (int c = 0; c < NCH; ++c) {
                    uint32_t (&cur)[32] = (c & 1) ? vb : va;
                    uint32_t (&nxt)[32] = (c & 1) ? va : vb;
                    tmem_ld_wait(cur);
                    if (c + 1 < NCH) {
                        tmem_ld32(t0 + 32 * (c + 1), nxt);
                    } else {
                        // every TMEM read of this tile's accumulator has completed: hand it back to the MMA warp
                        // BEFORE waiting for the next one
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) {
                            if (CG == 1) mbar_arrive(tempty_bar(acc));
                            else mbar_arrive_cluster(tempty_bar(acc), 0);
                        }
#pragma unroll
                        for (int u = 0; u < TPT; ++u) {
                            if (has_next && et + u * 32 * EW < BN) tgt_s[tbn * BN + et + u * 32 * EW] = t_next[u] - tbias;
                            if (tile + 2 * n_pairs < total_tiles) t_next[u] = fetch_target(tile + 2 * n_pairs, u);
                        }
                        epi_barrier();
                        flush(sb ^ 1);
                        if (has_next) {                   // uniform over the CTA's epilogue warps
                            mbar_wait<SUSP>(tfull_bar(acc ^ 1), acc ? aph ^ 1 : aph);
                            tc_fence_after();
                            tmem_ld32(lane_addr + (uint32_t)((acc ^ 1) * BN), nxt);
                        }
                    }
                    epilogue_chunk<ACT, TMSE>(cur, ts + 32 * c, R, acc2);
                }
                sum_s[(sb * 4 + cb) * BM + row] = ((acc2[0].x + acc2[0].y) + (acc2[1].x + acc2[1].y)) + ((acc2[2].x + acc2[2].y) + (acc2[3].x + acc2[3].y));
                prev_off = (long long)n_tile * Ppad + (m_blk * CG + (int)cta_rank) * BM + row;
                tb = tbn;
                sb ^= 1;
                if (++acc == 2) { acc = 0; aph ^= 1; }
            }
            if (pair < total_tiles) {
                epi_barrier();
                flush(sb ^ 1);
            }
        }
    }

    // teardown: everyone done with TMEM before it is released
    pdl_trigger();
    tc_fence_before();
    if (CG == 2) { asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory"); }
    else __syncthreads();
    if (warp == WARP_MMA) { __syncwarp(); tc_fence_after(); tmem_dealloc<CG>(tmem_base, 512); }
}

// pop fp32 [P][K] -> the fp16 copy described by `sink` (c16_store)
__global__ void pop_to_f16_kernel(const float *__restrict__ pop, int P, int K, C16Sink sink, const DevState *state)
{
    pdl_wait();
    pdl_trigger();
    if (state && state->stopped) return;
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= (long long)P * K) return;
    c16_store(sink, (int)(i / K), (int)(i % K), pop[i]);
}

// ---- host side ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// [rows][row_elems] fp16 row-major, boxes of [box_rows][64], 128-byte swizzle
static int encode_map(game_ctx *ctx, CUtensorMap *m, void *ptr, long long rows, int Kpad, int box_rows)
{
    EncodeTiledFn enc = get_encode();
    if (!enc) return fail(ctx, GAME_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[2] = {(cuuint64_t)Kpad, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)Kpad * 2};
    cuuint32_t box[2] = {(cuuint32_t)BKB, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, GAME_ERR_CUDA, "cuTensorMapEncodeTiled failed");
    return GAME_OK;
}

bool tensor_path_built() { return true; }

// CTA pairs (cta_group::2, 256 chromosomes x 256 patterns per pair) halve the E-tile bytes each SM stages;
// measured on B200 they win for deep contractions over wide populations (config 5: 1500 vs 1442 TFLOP/s)
// and lose where the pair leaves too few chromosome blocks (config 4) or K is shallow (config 3).
// game_set_tuning(GAME_TUNE_CTA_GROUP, 1|2) overrides, for measurement.
static int cta_group(const game_ctx *ctx, int Ppad, int Kp)
{
    const int forced = ctx->tune[GAME_TUNE_CTA_GROUP];
    if (forced == 1 || forced == 2) return forced;
    return (Kp >= 512 && Ppad >= 1024) ? 2 : 1;
}

// Which logistic form the epilogue uses: mode 2 unless game_set_tuning(GAME_TUNE_SIGMOID, 0) (measurement knob).
static int sigmoid_mode(const game_ctx *ctx)
{
    return ctx->tune[GAME_TUNE_SIGMOID] == 0 ? MODE_SIG_EXACT : MODE_SIG_TANH32;
}

C16Sink tensor_sink(const game_ctx *ctx, bool split)
{
    const int mode = ctx->act == GAME_ACT_IDENTITY ? MODE_IDENTITY : (split ? MODE_SIG_EXACT : sigmoid_mode(ctx));
    C16Sink s;
    s.ptr = split ? ctx->C16s : ctx->C16;
    s.Kpad = ctx->Kpad; s.family = ctx->family; s.d = ctx->degree; s.F = ctx->F; s.split = split ? 1 : 0;
    s.scale = mode == MODE_SIG_TANH32 ? 0.5f : 1.0f;
    return s;
}

int tensor_prepare(game_ctx *ctx)
{
    if (!ctx->tmap_E) ctx->tmap_E = aligned_alloc(64, 2 * sizeof(CUtensorMap));    // [0]: 256-row boxes, [1]: 128-row
    if (!ctx->tmap_C) ctx->tmap_C = aligned_alloc(64, sizeof(CUtensorMap));
    if (!ctx->tmap_E || !ctx->tmap_C) return fail(ctx, GAME_ERR_ALLOC, "tensor map allocation failed");
    for (int cg = 1; cg <= 2; ++cg) {
        // E16 viewed as [(Npad256/256) * (Kpad/64) * 256][64]: one 128-byte row per (pattern, k-block)
        int rc = encode_map(ctx, (CUtensorMap *)ctx->tmap_E + (cg - 1), ctx->E16, ctx->Npad256 * (ctx->Kpad / BKB), BKB, BN / cg);
        if (rc) return rc;
    }
    return GAME_OK;
}

// the materialised fp16 expansion and its tensor maps, where game_load left them for the first call that needs them
int tensor_ensure_E16(game_ctx *ctx)
{
    if (ctx->E16) return GAME_OK;
    const size_t n16 = (size_t)ctx->Npad256 * ctx->Kpad;
    GAME_CUDA(ctx, cudaMalloc(&ctx->E16, n16 * sizeof(__half)));
    GAME_CUDA(ctx, cudaMemsetAsync(ctx->E16, 0, n16 * sizeof(__half), ctx->stream));
    int rc = launch_expand_fp16(ctx, nullptr);
    return rc ? rc : tensor_prepare(ctx);
}

// TENSOR_SPLIT path: the [hi | hi | lo] expansion and its tensor maps, built on the first call that needs them
int tensor_prepare_split(game_ctx *ctx)
{
    if (ctx->E16s) return GAME_OK;
    const size_t n16 = (size_t)ctx->Npad256 * 3 * ctx->Kpad;
    GAME_CUDA(ctx, cudaMalloc(&ctx->E16s, n16 * sizeof(__half)));
    GAME_CUDA(ctx, cudaMemsetAsync(ctx->E16s, 0, n16 * sizeof(__half), ctx->stream));
    int rc = launch_expand_split(ctx);
    if (rc) return rc;
    if (!ctx->tmap_Es) ctx->tmap_Es = aligned_alloc(64, 2 * sizeof(CUtensorMap));
    if (!ctx->tmap_C) ctx->tmap_C = aligned_alloc(64, sizeof(CUtensorMap));           // (the TENSOR path may be unavailable)
    if (!ctx->tmap_Es || !ctx->tmap_C) return fail(ctx, GAME_ERR_ALLOC, "tensor map allocation failed");
    for (int cg = 1; cg <= 2; ++cg) {
        rc = encode_map(ctx, (CUtensorMap *)ctx->tmap_Es + (cg - 1), ctx->E16s, ctx->Npad256 * (3 * ctx->Kpad / BKB), BKB, BN / cg);
        if (rc) return rc;
    }
    return GAME_OK;
}

template <int CG, int ACT, bool TMSE, int EW, int SRC, int FAMILY, bool TEAMS = false, int BNT = BN, int SHARE = 0>
static int launch_variant(game_ctx *ctx, int n_tiles, int m_blocks, int Ppad, const DevState *state, bool split = false)
{
    using C = Cfg<CG>;
    auto kern = fitness_tc_kernel<CG, ACT, TMSE, EW, SRC, FAMILY, TEAMS, BNT, SHARE>;
    const int k_blocks = (split ? 3 : 1) * ctx->Kpad / BKB;
    // real terms in the last k-block of a K range, in UMMA k-steps of 16 (the split form has three ranges that end in the same
    // padding; the generator variant still writes whole k-blocks, the MMAs just do not read the padding: config 4, K = 544,
    // issues 34 instead of 36 MMAs per tile: 0.2338 vs 0.2361 ms, same box)
    const int npos = tc_num_positions(ctx->family, ctx->degree, ctx->F, ctx->K);
    const int k_last = (npos - (ctx->Kpad - BKB) + UMMA_K - 1) / UMMA_K;
    const int kb_range = ctx->Kpad / BKB;                    // k-blocks per K range
    // (the generator variant takes no expansion map: the population's stands in for the unused argument)
    const CUtensorMap *maps_E = (const CUtensorMap *)(SRC == SRC_GEN ? ctx->tmap_C : split ? ctx->tmap_Es : ctx->tmap_E);
    const int smem = SRC != SRC_TMA ? k_blocks * A_BYTES + GEN_STAGES * GEN_B_BYTES + 1024 + TC_TAIL_BYTES
                   : BNT == BN    ? C::SMEM
                                  : 6 * (A_BYTES + BNT * BKB * 2) + 1024 + TC_TAIL_BYTES;
    GAME_CUDA(ctx, ensure_smem_attr(ctx, (const void *)kern, smem));
    long long total = (long long)n_tiles * m_blocks;
    int pairs = ctx->sm_count / CG;
    if (pairs > total) pairs = (int)total;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(pairs * CG));
    cfg.blockDim = dim3(SRC == SRC_GEN ? GEN_THREADS : 64 + 32 * EW);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl_enabled(ctx) ? 2 : 1;
    KernelTimer timer(ctx);
    GAME_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, *(const CUtensorMap *)ctx->tmap_C, maps_E[SRC == SRC_GEN ? 0 : BNT / CG == 128 ? 1 : 0], n_tiles,
                                      m_blocks, k_blocks, ctx->N, (const float *)ctx->t, ctx->R, ctx->partial, Ppad, state,
                                      (const float *)ctx->X, ctx->F, ctx->degree, k_last, kb_range));
    return GAME_OK;
}

// north_star (1): materialise E or regenerate it in the kernel, by measured cost.  The generator variant needs the
// whole population in ONE CTA pair (Ppad = 256) and its fp16 copy resident in shared memory beside the B ring, i.e.
// exactly the shapes where streaming the materialised E16 could limit the kernel (bytes of E16 per flop ~ 1/P).
// Measured on B200, same box, kernel ms materialised / regenerated (DESIGN.md section 7 has the table):
//   trig d=8 F=32 (K=544) N=1e6: P=256 0.226 / 0.217, P=128 0.215 / 0.211, P=20 0.205 / 0.208; N=2e5 0.052 / 0.056
//   cheb d=16 F=32 (K=544) N=1e6 P=256 0.228 / 0.215;  K=272 (F=16) 0.128 / 0.147;  K=160 (d=2) 0.100 / 0.146
// so AUTO regenerates deep contractions (>= 8 k-blocks) over all four feature groups on datasets of >= 2000 tiles per
// launch (the matrix no longer fits in L2 and the start-up -- resident population tile, first features -- is amortised)
// for P > 32, and streams the materialised matrix everywhere else.  The trigonometric generator uses the fast sincos,
// accurate on |x| <= pi only (checked against the dataset at load).
int tensor_expansion(const game_ctx *ctx, int P)
{
    const int Ppad = ((P + 255) / 256) * 256;
    const int k_blocks = ctx->Kpad / BKB;
    const bool can = tc_permuted(ctx->family) && Ppad == 256 && ctx->X != nullptr && ctx->F <= 8 * GEN_GROUPS &&
                     k_blocks * A_BYTES + GEN_STAGES * GEN_B_BYTES + 1024 + TC_TAIL_BYTES <= 227 * 1024 &&
                     (ctx->family != GAME_TRIG || ctx->x_maxabs <= 3.14159f);
    if (ctx->expand_mode == GAME_EXPAND_REGENERATED) return can ? GAME_EXPAND_REGENERATED : -1;
    if (ctx->expand_mode == GAME_EXPAND_MATERIALIZED) return GAME_EXPAND_MATERIALIZED;
    const bool pays = k_blocks >= 8 && ctx->F > 8 * (GEN_GROUPS - 1) && ctx->Npad256 / BN >= 2000 && P > 32;
    return can && pays ? GAME_EXPAND_REGENERATED : GAME_EXPAND_MATERIALIZED;
}

// make the fp16 operand copy (C16 / C16s) mirror `pop`, unless the GA operators already wrote it while building `pop`
int tensor_refresh_c16(game_ctx *ctx, const float *pop, int P, bool split, const DevState *state)
{
    const C16Sink sink = tensor_sink(ctx, split);
    if (ctx->c16_src == pop && ctx->c16_split == sink.split && ctx->c16_scale == sink.scale) return GAME_OK;
    const long long n = (long long)P * ctx->K;
    GAME_CUDA(ctx, launch_pdl(pop_to_f16_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, ctx, pop, P, ctx->K, sink, state));
    ++ctx->launches;
    ctx->c16_src = nullptr;               // an external population: nothing to remember
    return GAME_OK;
}

int tensor_encode_population_map(game_ctx *ctx, bool split, int Ppad)
{
    if (!ctx->tmap_C) ctx->tmap_C = aligned_alloc(64, sizeof(CUtensorMap));
    if (!ctx->tmap_C) return fail(ctx, GAME_ERR_ALLOC, "tensor map allocation failed");
    return encode_map(ctx, (CUtensorMap *)ctx->tmap_C, split ? ctx->C16s : ctx->C16, Ppad, (split ? 3 : 1) * ctx->Kpad, BM);
}

int launch_fitness_tensor(game_ctx *ctx, const float *pop, int P, float *out, const DevState *state, PartialInfo *defer, bool split)
{
    const int Ppad = ((P + 255) / 256) * 256;
    if (split) {
        int rcs = tensor_prepare_split(ctx);
        if (rcs) return rcs;
    }
    const int Kp = (split ? 3 : 1) * ctx->Kpad;              // contraction depth the kernel sees
    const int expansion = split ? GAME_EXPAND_MATERIALIZED : tensor_expansion(ctx, P);
    if (expansion < 0) return fail(ctx, GAME_ERR_UNSUPPORTED, "regenerated expansion unavailable for this shape (needs P <= 256, K <= 576 after padding, trig: max|X| <= pi)");
    if (!split && expansion != GAME_EXPAND_REGENERATED) {
        int rce = tensor_ensure_E16(ctx);
        if (rce) return rce;
    }
    // Small populations (one CTA pair covers all chromosomes): keep the fp16 population tile RESIDENT in shared memory and
    // stream only the expansion (SRC_RES) -- a third of SRC_TMA's L2 -> SM traffic.  Config 4, same box: 0.229 vs 0.263 ms,
    // identical bits; the kernel then runs at 5.1 TB/s of HBM reads (78 % of the measured peak).
    // game_set_tuning(GAME_TUNE_RESIDENT, 0) turns it off, for measurement.
    const bool resident_ok = ctx->tune[GAME_TUNE_RESIDENT] != 0;
    const bool fits = (Kp / BKB) * A_BYTES + GEN_STAGES * GEN_B_BYTES + 1024 + TC_TAIL_BYTES <= 227 * 1024;
    const long long tiles256 = (long long)(ctx->Npad256 / BN) * ((P + BM - 1) / BM);     // 128-chromosome x 256-pattern tiles
    const bool resident_only = expansion != GAME_EXPAND_REGENERATED && resident_ok && Ppad == 256 && fits && Kp >= 256 &&
                               tiles256 >= ctx->sm_count;
    const int src = expansion == GAME_EXPAND_REGENERATED ? SRC_GEN : (resident_only ? SRC_RES : SRC_TMA);
    const int cg = src != SRC_TMA ? 2 : cta_group(ctx, Ppad, Kp);
    // Which epilogue: for shallow contractions (the MMAs of a tile take less time than its epilogue) two independent
    // teams of four warps, one per accumulator, so the warps sharing a scheduler are in different stages of different
    // tiles (config 3, same box: 0.139 vs 0.150 ms); for deep ones all eight warps on one tile, which hands the
    // accumulator back sooner (configs 4, 5: the team form loses 1-2 % there).  GAME_TUNE_TEAMS = 0|1 overrides.
    const int teams_forced = ctx->tune[GAME_TUNE_TEAMS];
    const bool teams = teams_forced < 0 ? Kp <= 256 : teams_forced == 1;
    // Less than one wave of 256-pattern tiles (configs 1-2): twice as many 128-pattern tiles on single CTAs finish sooner.
    // GAME_TUNE_HALF_TILES = 0|1 overrides, for measurement.
    const int half_forced = ctx->tune[GAME_TUNE_HALF_TILES];
    const bool half_tiles = src == SRC_TMA && (half_forced < 0 ? tiles256 < ctx->sm_count : half_forced == 1);
    const int n_tiles = (int)(ctx->Npad256 / (half_tiles ? 128 : BN));
    const int m_blocks = half_tiles ? (P + BM - 1) / BM : Ppad / (BM * cg);
    const bool tmse = ctx->err == GAME_ERR_TMSE;
    // the split path is the 1e-5 tolerance class: its logistic is the ex2 + rcp form (2^-22), not tanh.approx (2^-11)
    const int mode = ctx->act == GAME_ACT_IDENTITY ? MODE_IDENTITY : (split ? MODE_SIG_EXACT : sigmoid_mode(ctx));
    // a share of the logistics on the FMA pipe (shallow contractions, where the special-function unit binds): pairs of 16
    // per 32-column chunk; GAME_TUNE_RATIONAL_SHARE = 0 turns it off.  Only the measured best share (RATIONAL_SHARE_AUTO
    // of every 16 pairs) is built: the sweep over 4..8 that found it lives in DESIGN.md section 7, not in the library.
    const int share_req = ctx->tune[GAME_TUNE_RATIONAL_SHARE];
    const int share = (mode != MODE_SIG_TANH32 || !teams || cg != 1 || half_tiles || share_req == 0) ? 0 : RATIONAL_SHARE_AUTO;
    int rc = tensor_refresh_c16(ctx, pop, P, split, state);
    if (!rc) rc = tensor_encode_population_map(ctx, split, Ppad);
    if (rc) return rc;
#define GAME_TC_SHARE(M, T, S) launch_variant<1, M, T, 8, SRC_TMA, GAME_TRIG, true, BN, (M == MODE_SIG_TANH32 ? S : 0)>(ctx, n_tiles, m_blocks, Ppad, state, split)
#define GAME_TC_EW(CGV, M, T)                                                                              \
    rc = half_tiles ? launch_variant<1, M, T, 8, SRC_TMA, GAME_TRIG, true, 128>(ctx, n_tiles, m_blocks, Ppad, state, split)  \
       : (teams && CGV == 1 && share > 0) ? GAME_TC_SHARE(M, T, RATIONAL_SHARE_AUTO)                                          \
       : teams ? launch_variant<CGV, M, T, 8, SRC_TMA, GAME_TRIG, true>(ctx, n_tiles, m_blocks, Ppad, state, split)           \
               : launch_variant<CGV, M, T, 8, SRC_TMA, GAME_TRIG, false>(ctx, n_tiles, m_blocks, Ppad, state, split)
#define GAME_TC_GEN(M, T)                                                                                  \
    rc = resident_only ? launch_variant<2, M, T, 8, SRC_RES, GAME_TRIG>(ctx, n_tiles, 1, Ppad, state, split) \
       : ctx->family == GAME_TRIG ? launch_variant<2, M, T, GEN_EW, SRC_GEN, GAME_TRIG>(ctx, n_tiles, 1, Ppad, state) \
                                  : launch_variant<2, M, T, GEN_EW, SRC_GEN, GAME_CHEB>(ctx, n_tiles, 1, Ppad, state)
#define GAME_TC_MODE(CGV, M)                                                                               \
    if (src != SRC_TMA) { if (tmse) { GAME_TC_GEN(M, true); } else { GAME_TC_GEN(M, false); } }            \
    else if (tmse) { GAME_TC_EW(CGV, M, true); } else { GAME_TC_EW(CGV, M, false); }
#define GAME_TC_DISPATCH(CGV)                                                                              \
    switch (mode) {                                                                                        \
    case MODE_IDENTITY: GAME_TC_MODE(CGV, MODE_IDENTITY); break;                                           \
    case MODE_SIG_TANH32: GAME_TC_MODE(CGV, MODE_SIG_TANH32); break;                                       \
    default: GAME_TC_MODE(CGV, MODE_SIG_EXACT); break;                                                     \
    }
    if (cg == 2 || src != SRC_TMA) { GAME_TC_DISPATCH(2); } else { GAME_TC_DISPATCH(1); }
#undef GAME_TC_DISPATCH
#undef GAME_TC_MODE
#undef GAME_TC_GEN
#undef GAME_TC_EW
#undef GAME_TC_SHARE
    if (rc) return rc;
    ++ctx->launches;
    if (defer) { defer->n_chunks = n_tiles; defer->Ppad = Ppad; return GAME_OK; }     // one partial row per 256-pattern tile
    return launch_finalize(ctx, n_tiles, Ppad, P, out, state);
}

}  // namespace game

