// The whole training loop (fitness, sort, stop test, operators, repeat) as ONE persistent cooperative
// kernel, for problems of less than one wave of tiles (configs 1-2): there a generation is a few microseconds of work and
// five dependent launches cost more than they compute (SURVEY section 7 "tiny configs").
//
// One CTA per 128-chromosome x 128-pattern tile, all co-resident (cooperative launch), looping on the device:
//   phase A  a1-a5   the CTA's tile of z = E . C^T on the tensor cores (tcgen05, fp32 accumulate in TMEM) with the fused
//                    activation / error / row-sum epilogue -> partial[n_tile][p].  The expansion tile (B operand) is
//                    loaded ONCE and stays resident in shared memory for the whole run; the population tile (A operand)
//                    is fetched whole by TMA every generation (all k-blocks in flight at once).
//   -- grid barrier --
//   phase B  a5-a7   final reduction over the pattern tiles in the launch path's fixed order (fp64), rank by counting on
//                    (error, index) keys, best / stop test.  Up to 256 chromosomes every CTA ranks the whole population
//                    itself (no further barrier); beyond, each CTA ranks a slice and a second grid barrier publishes `order`.
//   phase C  a8-a11  elitism, tournament selection, crossover, mutation for the CTA's share of the children, from the same
//                    Philox counters as ga_step_kernel; also writes the next generation's fp16 operand copy.
//   -- grid barrier --
// Small populations (one chromosome block, P K <= PERS_LOCAL_GENES: config 1, the paper's own shape) keep the WHOLE
// population in every CTA's shared memory: each CTA applies the operators to all children itself (same counters, same
// bits), writes the fp16 operand tile where a TMA box would have put it, and CTA 0 mirrors the result to global memory --
// no population traffic, no population load in phase A and no second grid barrier (the tile sums alternate between two
// buffers so that a CTA one phase ahead cannot overwrite what a slower one still reads).
// The arithmetic of every phase is the launch path's, operation for operation (same MMA shapes and k order, the same
// epilogue code, the same summation order, the same integer decisions), so a run through this kernel is bit-identical
// to stepping the multi-launch path one generation at a time; tests/test_gpu_parity.py holds it to that.
#include "ga_device.cuh"
#include "tc_common.cuh"

namespace game {
constexpr int PERS_TMEM_COLS = 128;

constexpr int PERS_THREADS = 512;       // warp 0 TMA producer, warp 1 MMA issuer, warps 2-5 epilogue; all 16 warps in phases B, C (256 threads: phase C 5.6k vs 8.4k clk on config 1)
constexpr int PERS_TILE_N = 128;        // patterns per tile: the half-size tiles the launch path uses below one wave
constexpr int PERS_KB_BYTES = 128 * BKB * 2;
constexpr int PERS_LOCAL_RANK = 256;    // up to this many chromosomes every CTA ranks the whole population itself
constexpr int PERS_MAX_P = 2048;        // sort keys of the whole population live in shared memory
constexpr int PERS_LOCAL_GENES = 4096;  // local-population mode: every CTA rebuilds all P K genes itself (two Philox calls per gene)

struct PersistArgs {
    int n_tiles, m_blocks, k_blocks, kb1, split, k_last, P, Ppad, generations, err;
    int local;                          // local-population mode (see the header)
    long long N;
    const float *tgt;
    float R, stop_error;
    float *partial, *fit;
    int *order;
    float *pop_a, *pop_b;               // the population ping-pong: evaluation e reads (e even ? pop_a : pop_b)
    DevState *state;
    unsigned int *gbar;                 // grid barrier counter, zero at launch
    StepArgs step;                      // seed, generation base, thresholds, the fp16 sink
};

// all CTAs of the (co-resident) grid: monotonic counter, release on arrival, acquire on the poll
__device__ __forceinline__ void grid_barrier(unsigned int *ctr, unsigned int &target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        // one fence on each side and relaxed accesses in between: an acquire load in the polling loop would pay an L1
        // invalidation per probe (measured: 3.3 us per barrier with release-red + acquire-poll)
        target += gridDim.x;
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned int v;
        unsigned long long t0 = 0;
        for (uint32_t spin = 1;; ++spin) {
            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
            if ((int)(v - target) >= 0) break;
            if ((spin & 0xFFFFu) == 0) t0 = mbar_timeout_check(t0);
        }
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
}

template <int ACT, bool TMSE>
__global__ void __launch_bounds__(PERS_THREADS, 1)
evolve_persistent_kernel(const __grid_constant__ CUtensorMap tmC, const __grid_constant__ CUtensorMap tmE,
                         const __grid_constant__ PersistArgs a)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - smem_u32(smem_raw));
    const int k_blocks = a.k_blocks, P = a.P, K = a.step.K;
    // Both operands are RESIDENT: the expansion tile for the whole run, the population tile for one generation.  The split
    // form's K axis is E = [hi | hi | lo] against C = [hi | lo | hi] (three ranges of kb1 k-blocks): only 2 kb1 DISTINCT
    // blocks per operand exist, so the repeated range is not stored twice -- the MMAs of range 1 of E (range 2 of C) read
    // the blocks of range 0 again.  That is what lets both tiles of the split form fit (12 x 16 KB at K = 99) and ALL of
    // a generation's population k-blocks be in flight at once: one L2 round trip per generation instead of one per ring turn.
    const int kb1 = a.kb1, nres = a.split ? 2 * kb1 : kb1;                  // distinct k-blocks per operand
    const uint32_t baseB = base, baseA = base + (uint32_t)nres * PERS_KB_BYTES;
    const uint32_t bar0 = baseA + (uint32_t)nres * PERS_KB_BYTES;
    const uint32_t afull_bar = bar0, bfull_bar = bar0 + 8u, tfull_bar = bar0 + 16u, tmem_slot = bar0 + 24u, sfull_bar = bar0 + 32u;
    uint8_t *tail = gbase + 2 * nres * PERS_KB_BYTES;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(tail + 24);
    float *tgt_s = reinterpret_cast<float *>(tail + 128);                                       // [128]
    unsigned long long *keys = reinterpret_cast<unsigned long long *>(tail + 128 + 512);        // [P]
    float *fit_s = reinterpret_cast<float *>(keys + P);                                         // [P]
    int *order_s = reinterpret_cast<int *>(fit_s + P);                                          // [P] (local rank only)
    // local-population mode: the population twice (this generation's and the next one's genes) and a staging area of its own
    // for the tile sums (the population tile, which serves as staging area otherwise, now lives across the phases)
    const uint32_t local_off = (uint32_t)(128 + 512 + P * 16 + 15) & ~15u;                     // 16-byte aligned, behind order_s
    float *pop_s0 = reinterpret_cast<float *>(tail + local_off);                                // [P K]
    float *pop_s1 = pop_s0 + ((P * K + 3) & ~3);                                                // [P K]
    float *stage_local = pop_s1 + ((P * K + 3) & ~3);                                           // [n_tiles][P4]
    __shared__ int sh[8];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
    const int tile = blockIdx.x, n_tile = tile / a.m_blocks, m_blk = tile % a.m_blocks;
    const bool local_rank = P <= PERS_LOCAL_RANK;

    if (tid == 0) {
        mbar_init(afull_bar, 1);
        mbar_init(bfull_bar, 1);
        mbar_init(tfull_bar, 1);
        mbar_init(sfull_bar, 1);
        fence_barrier_init();
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmC) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmE) : "memory");
    }
    if (warp == 1) tmem_alloc<1>(tmem_slot, PERS_TMEM_COLS);
    // the tile's targets, staged once: t - tbias, and for a padding pattern the value that makes its residual exactly zero
    // (its expansion row is zero, so z = 0) -- the launch path's rule (fitness_tc_kernel, team epilogue)
    constexpr float tbias = ACT == MODE_SIG_TANH32 ? 0.5f : 0.f;
    constexpr float tneutral = ACT == MODE_SIG_EXACT ? 0.5f : 0.f;
    if (tid < PERS_TILE_N) {
        const long long n = (long long)n_tile * PERS_TILE_N + tid;
        tgt_s[tid] = (n < a.N ? a.tgt[n] : tneutral + tbias) - tbias;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;

    if (warp == 0 && lane == 0) {      // the expansion tile: resident for the whole run
        const int n_first = n_tile * PERS_TILE_N;
        const int rowE = (n_first >> 8) * k_blocks * BN + (n_first & 255);      // E16 is tile-blocked [n/256][kb][256][64]
        mbar_expect_tx(bfull_bar, (uint32_t)(nres * PERS_KB_BYTES));
        for (int j = 0; j < nres; ++j) {                                       // split: ranges 0 (hi) and 2 (lo)
            const int kb = j < kb1 ? j : j + kb1;
            tma_load_2d<1>(baseB + j * PERS_KB_BYTES, &tmE, 0, rowE + kb * BN, bfull_bar);
        }
    }

    // local-population mode: gene k of chromosome p goes to the CTA's fp32 copy and, as fp16 (c16_store's rounding and
    // positions), to the operand tile at the 128B-swizzled address a TMA box of C16 / C16s would have filled; CTA 0 mirrors
    // both to global memory, so the context's population and fp16 copy are what the launch path would have left
    const C16Sink &sink = a.step.sink;
    const int Bterms = tc_terms_per_feature(sink.family, sink.d);
    struct GeneSlot { uint32_t blk_off, chunk; int pos; };       // where gene k lives: operand-tile block + in-row bytes, swizzle chunk, position
    auto gene_slot = [&](int k) {
        const int pos = tc_position(sink.family, sink.d, sink.F, k / Bterms, k % Bterms);
        return GeneSlot{(uint32_t)(nres + (pos >> 6)) * PERS_KB_BYTES + ((uint32_t)pos & 7u) * 2u, ((uint32_t)pos & 63u) >> 3, pos};
    };
    auto store_gene = [&](const GeneSlot &g, float *pop_dst_s, float *pop_dst_g, int p, int k, float gene) {   // pop_dst_g: global mirror (or null)
        pop_dst_s[p * K + k] = gene;
        const float v = fabsf(gene) <= 65504.f ? gene * sink.scale : __int_as_float(0x7fc00000);
        uint8_t *blk = gbase + g.blk_off + (uint32_t)p * 128u + ((g.chunk ^ ((uint32_t)p & 7u)) << 4);
        const __half hi = __float2half_rn(v);
        const __half lo = __float2half_rn(v - __half2float(hi));
        *reinterpret_cast<__half *>(blk) = hi;
        if (a.split) *reinterpret_cast<__half *>(blk + (size_t)kb1 * PERS_KB_BYTES) = lo;
        if (pop_dst_g) {                                 // what c16_store would have written
            pop_dst_g[(long long)p * K + k] = gene;
            if (!a.split) sink.ptr[(long long)p * sink.Kpad + g.pos] = hi;
            else { __half *row = sink.ptr + (long long)p * 3 * sink.Kpad; row[g.pos] = hi; row[sink.Kpad + g.pos] = lo; row[2 * sink.Kpad + g.pos] = hi; }
        }
    };
    auto put_gene = [&](float *pop_dst_s, float *pop_dst_g, int p, int k, float gene) { store_gene(gene_slot(k), pop_dst_s, pop_dst_g, p, k, gene); };
    if (a.local) {
        uint4 *at = reinterpret_cast<uint4 *>(gbase + (size_t)nres * PERS_KB_BYTES);
        for (int i = tid; i < nres * PERS_KB_BYTES / 16; i += PERS_THREADS) at[i] = make_uint4(0u, 0u, 0u, 0u);   // rows >= P, padding positions
        __syncthreads();
        for (int i = tid; i < P * K; i += PERS_THREADS) put_gene(pop_s0, nullptr, i / K, i % K, __ldcg(a.pop_a + i));   // (global memory already holds both)
        fence_proxy_async();               // generic-proxy stores of the operand tile -> the tensor core's async-proxy reads
        __syncthreads();
    }
    float *pop_cur_s = pop_s0, *pop_next_s = pop_s1;

    unsigned int bar_target = 0;
    uint32_t sph = 0;                                    // staging barrier phase
    int applied = 0, evals = 0, stopped = 0;
    float best_f = 0.f; int best_p = 0;
    const float *pop_cur = a.pop_a;
    float *pop_next = a.pop_b;

    for (int e = 0;; ++e) {
        // local mode has one grid barrier per generation: the tile sums alternate between two buffers (see the header)
        float *partial_e = a.partial + (a.local && (e & 1) ? (long long)a.n_tiles * a.Ppad : 0);
        // ================= phase A: this CTA's tile of the fused fitness =================
        if (warp == 0) {
            if (lane == 0 && !a.local) {
                fence_proxy_async_all();                 // the genes were written by other CTAs' generic stores (phase C)
                mbar_expect_tx(afull_bar, (uint32_t)(nres * PERS_KB_BYTES));
                for (int j = 0; j < nres; ++j)           // split: ranges 0 (hi) and 1 (lo); range 2 repeats range 0
                    tma_load_2d<1>(baseA + j * PERS_KB_BYTES, &tmC, j * BKB, m_blk * BM, afull_bar);
            }
        } else if (warp == 1) {
            // the whole warp walks the loop (descriptors stay warp-uniform), one elected lane issues -- see fitness_tc.cu
            constexpr uint32_t idesc = make_idesc(BM, PERS_TILE_N);
            if (e == 0) mbar_wait(bfull_bar, 0);
            if (!a.local) mbar_wait(afull_bar, (uint32_t)(e & 1));      // (local mode: the tile was written before the CTA barrier)
            tc_fence_after();
            int kr = 0;                                  // k-block inside the current K range (wrap counter: no division on the issue path)
            for (int kb = 0; kb < k_blocks; ++kb) {      // the launch path's k order, whatever block the data sits in
                const int ja = kb < nres ? kb : kb - nres, jb = kb < kb1 ? kb : kb - kb1;
                const uint64_t adesc = make_smem_desc(baseA + ja * PERS_KB_BYTES), bdesc = make_smem_desc(baseB + jb * PERS_KB_BYTES);
                const bool range_end = ++kr == kb1;
                if (range_end) kr = 0;
                const int nk = range_end ? a.k_last : BKB / UMMA_K;               // the last block of each K range ends in padding
                if (elect_one()) {
#pragma unroll
                    for (int k = 0; k < BKB / UMMA_K; ++k)
                        if (k < nk) umma_f16<1>(tmem_base, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) != 0);
                    if (kb + 1 == k_blocks) umma_commit<1>(tfull_bar);
                }
                __syncwarp();
            }
        } else if (warp < 6) {
            // one thread per chromosome walks the tile's 128 pattern columns in four 32-column chunks, the TMEM load of the
            // next chunk in flight while the current one is evaluated: the launch path's team epilogue at BNT = 128
            const int quarter = warp & 3;
            const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
            uint32_t va[32], vb[32];
            mbar_wait(tfull_bar, (uint32_t)(e & 1));
            tc_fence_after();
            tmem_ld32(lane_addr, va);
            float2 acc2[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
            for (int c = 0; c < PERS_TILE_N / 32; ++c) {
                uint32_t (&cur)[32] = (c & 1) ? vb : va;
                uint32_t (&nxt)[32] = (c & 1) ? va : vb;
                tmem_ld_wait(cur);
                if (c + 1 < PERS_TILE_N / 32) tmem_ld32(lane_addr + 32 * (c + 1), nxt);
                epilogue_chunk<ACT, TMSE>(cur, tgt_s + 32 * c, a.R, acc2);
            }
            tc_fence_before();                           // the next generation's MMAs overwrite the accumulator after the barrier
            partial_e[(long long)n_tile * a.Ppad + m_blk * BM + quarter * 32 + lane] =
                ((acc2[0].x + acc2[0].y) + (acc2[1].x + acc2[1].y)) + ((acc2[2].x + acc2[2].y) + (acc2[3].x + acc2[3].y));
        }
        grid_barrier(a.gbar, bar_target);
        ++evals;

        // ================= phase B: a5 tail, a6 rank, a7 stop test =================
        // The tile sums are pulled into shared memory by bulk asynchronous copies -- one per pattern tile, all in flight at
        // once (the population tile's area is idle between the phases and serves as the staging buffer) -- so the reduction
        // costs ONE L2 round trip instead of one per addend.
        {
            float *stage = a.local ? stage_local : reinterpret_cast<float *>(gbase + nres * PERS_KB_BYTES);
            const uint32_t stage_addr = a.local ? smem_u32(stage_local) : baseA;
            const int P4 = (P + 3) & ~3;
            const int cp = a.local ? P4 : min(P4, (nres * PERS_KB_BYTES / 4 / a.n_tiles) & ~3);      // chromosomes per pass (n_tiles <= 148: >= 24)
            for (int p0 = 0; p0 < P; p0 += cp) {
                const int np4 = min(cp, P4 - p0);                                     // a multiple of 4: 16-byte rows
                if (a.n_tiles * np4 <= 8 * PERS_THREADS) {
                    // few values (config 1: 17 x 20): eight independent plain loads per thread beat the bulk copy's set-up
                    float v[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int i = u * PERS_THREADS + tid, ch = i / np4, pp = i - ch * np4;
                        v[u] = i < a.n_tiles * np4 ? __ldcg(partial_e + (long long)ch * a.Ppad + p0 + pp) : 0.f;
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (u * PERS_THREADS + tid < a.n_tiles * np4) stage[u * PERS_THREADS + tid] = v[u];
                    __syncthreads();
                } else {
                    if (tid == 0) {
                        fence_proxy_async_all();       // other CTAs' generic stores -> this thread's async-proxy reads
                        mbar_expect_tx(sfull_bar, (uint32_t)(a.n_tiles * np4 * 4));
                        for (int ch = 0; ch < a.n_tiles; ++ch)
                            bulk_load(stage_addr + (uint32_t)(ch * np4 * 4), partial_e + (long long)ch * a.Ppad + p0, (uint32_t)(np4 * 4), sfull_bar);
                    }
                    mbar_wait(sfull_bar, sph);
                    sph ^= 1;
                }
                for (int pp = tid; pp < np4 && p0 + pp < P; pp += PERS_THREADS) {
                    // the fixed order of finalize_kernel / post_small_kernel: 32 interleaved fp64 sub-totals, added ascending
                    const int p = p0 + pp;
                    double tot = 0.0;
                    if (a.n_tiles <= 32) {
                        // every sub-total has at most one addend and the empty ones add +0.0 to a non-negative total: the
                        // same bits from one ascending pass (the tile sums are sums of squares, never -0.0)
                        for (int ch = 0; ch < a.n_tiles; ++ch) tot += (double)stage[ch * np4 + pp];
                    } else {
                        for (int r = 0; r < 32; ++r) {
                            double sub = 0.0;
                            for (int ch = r; ch < a.n_tiles; ch += 32) sub += (double)stage[ch * np4 + pp];
                            tot += sub;
                        }
                    }
                    double v = tot / (double)a.N;
                    if (a.err == GAME_ERR_RMSE) v = sqrt(v);
                    const float f = (float)v;
                    keys[p] = ((unsigned long long)sort_key(f) << 32) | (unsigned)p;
                    fit_s[p] = f;
                    if (blockIdx.x == 0) a.fit[p] = f;
                }
                __syncthreads();                       // the staging area is rewritten by the next pass / the next phase A
            }
            fence_proxy_async();          // generic reads of the area are ordered before the TMA writes of the next phase A
        }
        if (local_rank) {
            if (tid < P) {
                const unsigned long long mine = keys[tid];
                int cnt = 0;
#pragma unroll 8
                for (int q = 0; q < P; ++q) cnt += keys[q] < mine;
                order_s[cnt] = tid;
                if (blockIdx.x == 0) a.order[cnt] = tid;
                if (cnt == 0) sh[4] = tid;
            }
            __syncthreads();
            best_p = sh[4];
        } else {
            // this CTA's slice of the chromosomes, one per warp at a time, the lanes striding over the keys
            for (int p = blockIdx.x + warp * gridDim.x; p < P; p += gridDim.x * (PERS_THREADS / 32)) {
                const unsigned long long mine = keys[p];
                int cnt = 0;
                for (int q = lane; q < P; q += 32) cnt += keys[q] < mine;
                for (int o = 16; o; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
                if (lane == 0) {
                    a.order[cnt] = p;
                    if (cnt == 0) a.state->best_index = p;
                }
            }
            grid_barrier(a.gbar, bar_target);
            best_p = __ldcg(&a.state->best_index);
        }
        best_f = fit_s[best_p];                          // every CTA holds every fitness: the same bits everywhere
        if (a.stop_error >= 0.0f && best_f <= a.stop_error) stopped = 1;
        if (stopped || e == a.generations) break;

        // ================= phase C: a8-a11 for this CTA's share of the elites and child pairs =================
        const uint32_t gen = a.step.gen + (uint32_t)e;
        const int n_items = a.step.e + a.step.npairs;
        if (a.local) {
            // every CTA builds the whole next population from its own copy.  Step 1: one thread per child pair and parent draws
            // the pair's decisions (a9 tournament, a10 cut point); step 2: one (item, gene) per thread and turn, so a thread
            // walks n_items K / 512 genes with two Philox calls each.  Nothing goes to global memory inside the loop: the final
            // population is written out once, after the last evaluation.
            int *dec_s = reinterpret_cast<int *>(stage_local);            // [3][npairs]: parents A, B, crossover word (staging area is idle)
            const int npairs = a.step.npairs;
            if (tid < 3 * npairs) {
                const int q = tid % npairs, what = tid / npairs;
                int mine;
                if (what < 2) {                          // a9 tournament by rank (R3): t rank draws, the best wins
                    uint32_t best = 0xFFFFFFFFu;
                    W4 w{0, 0, 0, 0};
                    for (int j = 0; j < a.step.tsize; ++j) {
                        if ((j & 3) == 0) w = draw(a.step.seed, (uint32_t)(j >> 2), (uint32_t)(2 * q + what), gen, TAG_SELECT);
                        const uint32_t word = (j & 3) == 0 ? w.x : (j & 3) == 1 ? w.y : (j & 3) == 2 ? w.z : w.w;
                        best = min(best, idx_of(word, (uint32_t)P));
                    }
                    mine = order_s[(int)best];
                } else {                                 // a10 decision (R5): bit 30 = apply, low bits = cut point
                    W4 w = draw(a.step.seed, 0u, (uint32_t)q, gen, TAG_XOVER);
                    const int doit = (K >= 2) && hit(w.x, a.step.pc);
                    mine = (doit << 30) | (K >= 2 ? 1 + (int)idx_of(w.y, (uint32_t)(K - 1)) : 0);
                }
                dec_s[what * npairs + q] = mine;
            }
            __syncthreads();
            // a thread keeps ONE gene index (its slot in the operand tile is computed once) and walks the items; genes beyond
            // 128 per chromosome take further turns
            const int kt = tid & 127;
            for (int k = kt; k < K; k += 128) {
              const GeneSlot gs = gene_slot(k);
              float *const mirror = nullptr;
              for (int item = tid >> 7; item < n_items; item += PERS_THREADS / 128) {
                if (item < a.step.e) {                   // a8 elitism (L148, L291; DESIGN G17)
                    const int src = a.step.elite_mode == GAME_ELITE_TOP_E ? order_s[item] : order_s[0];
                    store_gene(gs, pop_next_s, mirror, item, k, pop_cur_s[src * K + k]);
                    continue;
                }
                const int q = item - a.step.e;
                const int sA = a.step.e + 2 * q, sB = sA + 1;
                const int pa = dec_s[q], pb = dec_s[npairs + q], xo = dec_s[2 * npairs + q];
                const int doit = xo >> 30, cut = xo & 0x3fffffff;
                const float ga = pop_cur_s[pa * K + k], gb = pop_cur_s[pb * K + k];
                const bool head = doit ? (k < cut) : true;
                float cA = head ? ga : gb, cB = head ? gb : ga;      // A = pa[0:c] | pb[c:K], B = pb[0:c] | pa[c:K]
                const W4 w = draw(a.step.seed, (uint32_t)k, (uint32_t)sA, gen, TAG_MUTATE);       // a11 (R6)
                const W4 v = draw(a.step.seed, (uint32_t)k, (uint32_t)sB, gen, TAG_MUTATE);
                if (hit(w.x, a.step.pm)) cA = upm1(w.y);
                if (hit(v.x, a.step.pm)) cB = upm1(v.y);
                store_gene(gs, pop_next_s, mirror, sA, k, cA);
                if (sB < P) store_gene(gs, pop_next_s, mirror, sB, k, cB);
              }
            }
            ++applied;
            fence_proxy_async();                         // the operand tile just written is read by the tensor core next
            __syncthreads();
            { float *t = pop_cur_s; pop_cur_s = pop_next_s; pop_next_s = t; }
            const float *t = pop_cur; pop_cur = pop_next; pop_next = const_cast<float *>(t);
            continue;
        }
        // This CTA's share of the items (item = blockIdx.x + j gridDim.x), in two steps like the local form.  Step 1: one thread
        // per item and decision (elite source; the pair's two parents by a9 tournament; its a10 cut point), so the dependent
        // rank -> index loads of all of them are in flight at once.  Step 2: one (item, gene) per thread and turn: the parents'
        // genes, two Philox calls, the children and their fp16 copies -- a gene per thread instead of a warp per pair.
        {
            const int nj = blockIdx.x < n_items ? (n_items - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
            int *dec_s = reinterpret_cast<int *>(gbase + nres * PERS_KB_BYTES);          // [3][nj] (the population tile's area is idle)
            auto rank_to_index = [&](int r) { return local_rank ? order_s[r] : __ldcg(a.order + r); };
            for (int u = tid; u < 3 * nj; u += PERS_THREADS) {
                const int j = u % nj, what = u / nj, item = blockIdx.x + j * gridDim.x;
                int mine = 0;
                if (item < a.step.e) {                   // a8 elitism (L148, L291; DESIGN G17)
                    if (what == 0) mine = a.step.elite_mode == GAME_ELITE_TOP_E ? rank_to_index(item) : rank_to_index(0);
                } else if (what < 2) {                   // a9 tournament by rank (R3): t rank draws, the best wins
                    const int q = item - a.step.e;
                    uint32_t best = 0xFFFFFFFFu;
                    W4 w{0, 0, 0, 0};
                    for (int i = 0; i < a.step.tsize; ++i) {
                        if ((i & 3) == 0) w = draw(a.step.seed, (uint32_t)(i >> 2), (uint32_t)(2 * q + what), gen, TAG_SELECT);
                        const uint32_t word = (i & 3) == 0 ? w.x : (i & 3) == 1 ? w.y : (i & 3) == 2 ? w.z : w.w;
                        best = min(best, idx_of(word, (uint32_t)P));
                    }
                    mine = rank_to_index((int)best);
                } else {                                 // a10 decision (R5): bit 30 = apply, low bits = cut point
                    W4 w = draw(a.step.seed, 0u, (uint32_t)(item - a.step.e), gen, TAG_XOVER);
                    const int doit = (K >= 2) && hit(w.x, a.step.pc);
                    mine = (doit << 30) | (K >= 2 ? 1 + (int)idx_of(w.y, (uint32_t)(K - 1)) : 0);
                }
                dec_s[what * nj + j] = mine;
            }
            __syncthreads();
            for (int k = tid & 127; k < K; k += 128) {
                for (int j = tid >> 7; j < nj; j += PERS_THREADS / 128) {
                    const int item = blockIdx.x + j * gridDim.x;
                    if (item < a.step.e) {
                        const float v = __ldcg(pop_cur + (long long)dec_s[j] * K + k);
                        pop_next[(long long)item * K + k] = v;
                        if (a.step.sink.ptr) c16_store(a.step.sink, item, k, v);
                        continue;
                    }
                    const int q = item - a.step.e;
                    const int sA = a.step.e + 2 * q, sB = sA + 1;
                    const int pa = dec_s[j], pb = dec_s[nj + j], xo = dec_s[2 * nj + j];
                    const int doit = xo >> 30, cut = xo & 0x3fffffff;
                    const float ga = __ldcg(pop_cur + (long long)pa * K + k), gb = __ldcg(pop_cur + (long long)pb * K + k);
                    const bool head = doit ? (k < cut) : true;
                    float cA = head ? ga : gb;           // A = pa[0:c] | pb[c:K]
                    float cB = head ? gb : ga;           // B = pb[0:c] | pa[c:K]
                    const W4 w = draw(a.step.seed, (uint32_t)k, (uint32_t)sA, gen, TAG_MUTATE);       // a11 (R6)
                    const W4 v = draw(a.step.seed, (uint32_t)k, (uint32_t)sB, gen, TAG_MUTATE);
                    if (hit(w.x, a.step.pm)) cA = upm1(w.y);
                    if (hit(v.x, a.step.pm)) cB = upm1(v.y);
                    pop_next[(long long)sA * K + k] = cA;
                    if (a.step.sink.ptr) c16_store(a.step.sink, sA, k, cA);
                    if (sB < P) {
                        pop_next[(long long)sB * K + k] = cB;
                        if (a.step.sink.ptr) c16_store(a.step.sink, sB, k, cB);
                    }
                }
            }
        }
        ++applied;
        fence_proxy_async_all();                         // the fp16 genes just stored are read by TMA (async proxy) next
        grid_barrier(a.gbar, bar_target);
        const float *t = pop_cur; pop_cur = pop_next; pop_next = const_cast<float *>(t);
    }

    if (a.local) {
        // the population the loop ended on (this CTA's copy is everyone's) goes to the buffer the launch path would have left
        // it in, with its fp16 copy; the CTAs share the writing
        float *out = const_cast<float *>(pop_cur);
        for (int i = blockIdx.x * PERS_THREADS + tid; i < P * K; i += gridDim.x * PERS_THREADS) {
            const float gene = pop_cur_s[i];
            out[i] = gene;
            c16_store(sink, i / K, i % K, gene);
        }
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.state->stopped = stopped;
        a.state->stop_request = stopped;
        a.state->gens_run = applied;
        a.state->evals_done = evals;
        a.state->best_error = best_f;
        a.state->best_index = best_p;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) { __syncwarp(); tc_fence_after(); tmem_dealloc<1>(tmem_base, PERS_TMEM_COLS); }
}


// local-population mode (see the header): one chromosome block and few enough genes for every CTA to rebuild them all.
// GAME_TUNE_PERSISTENT = 2 keeps the shared-population form, for measurement.
static bool persistent_local(const game_ctx *c, int P)
{
    return c->tune[GAME_TUNE_PERSISTENT] != 2 && P <= BM && (long long)P * c->K <= PERS_LOCAL_GENES;
}

static size_t persistent_smem_bytes(const game_ctx *c, int path, int P)
{
    const int kb1 = c->Kpad / BKB, nres = path == GAME_PATH_TENSOR_SPLIT ? 2 * kb1 : kb1;
    size_t bytes = (size_t)2 * nres * PERS_KB_BYTES + 1024 + 128 + 512 + (size_t)P * 16 + 64;
    if (persistent_local(c, P)) {
        const size_t n_tiles = (size_t)((c->N + PERS_TILE_N - 1) / PERS_TILE_N);
        bytes += 16 + 2 * (((size_t)P * c->K + 3) & ~(size_t)3) * 4 + (n_tiles < 2 ? 2 : n_tiles) * ((P + 3) & ~3) * 4;   // (the staging area also holds phase C's 3 P / 2 decisions)
    }
    return bytes;
}

// can game_evolve run this population / dataset through the persistent kernel?
bool persistent_eligible(const game_ctx *c, const game_ga_params *gp, int path)
{
    if (c->tune[GAME_TUNE_PERSISTENT] == 0 || c->timing) return false;
    if (path != GAME_PATH_TENSOR && path != GAME_PATH_TENSOR_SPLIT) return false;
    if (!tc_permuted(c->family) || gp->selection != GAME_SEL_TOURNAMENT) return false;
    if (c->expand_mode == GAME_EXPAND_REGENERATED) return false;
    const int P = gp->P;
    if (P > PERS_MAX_P) return false;
    const long long tiles = ((c->N + PERS_TILE_N - 1) / PERS_TILE_N) * ((P + BM - 1) / BM);
    if (tiles > c->sm_count) return false;                                   // one tile per CTA, all co-resident
    if (persistent_smem_bytes(c, path, P) > 227 * 1024) return false;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device) != cudaSuccess || !coop) return false;
    return true;
}

template <int ACT, bool TMSE>
static int launch_persistent_variant(game_ctx *c, const CUtensorMap &tmC, const CUtensorMap &tmE, const PersistArgs &a, int grid, int smem)
{
    auto kern = evolve_persistent_kernel<ACT, TMSE>;
    GAME_CUDA(c, ensure_smem_attr(c, (const void *)kern, smem));
    // a cooperative grid must be co-resident: ask how many CTAs of THIS variant fit (a shared-memory carve-out or a
    // partitioned GPU can leave fewer than one per SM) and let the caller take the launch-per-kernel path if not
    int per_sm = 0;
    GAME_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, PERS_THREADS, (size_t)smem));
    if ((long long)per_sm * c->sm_count < grid) return PERSISTENT_UNAVAILABLE;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(PERS_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaError_t le = cudaLaunchKernelEx(&cfg, kern, tmC, tmE, a);
    if (le == cudaErrorCooperativeLaunchTooLarge) {      // SMs taken by someone else (MPS / green-context partition, a resident kernel)
        cudaGetLastError();
        return PERSISTENT_UNAVAILABLE;
    }
    GAME_CUDA(c, le);
    ++c->launches;
    return GAME_OK;
}

// `generations` evolution steps + the final evaluation on the context's population (c->pop, fp16 copy up to date);
// leaves the result in c->state / c->fit / c->order; the caller swaps the population buffers if an odd number was applied
int launch_evolve_persistent(game_ctx *c, const game_ga_params *gp, unsigned long long seed, int generations, int path)
{
    const bool split = path == GAME_PATH_TENSOR_SPLIT;
    const int P = gp->P;
    if (split) {
        int rcs = tensor_prepare_split(c);
        if (rcs) return rcs;
    } else {
        int rce = tensor_ensure_E16(c);
        if (rce) return rce;
    }
    if (!c->gbar) GAME_CUDA(c, cudaMalloc(&c->gbar, sizeof(unsigned int)));
    GAME_CUDA(c, cudaMemsetAsync(c->gbar, 0, sizeof(unsigned int), c->stream));
    PersistArgs a{};
    a.n_tiles = (int)((c->N + PERS_TILE_N - 1) / PERS_TILE_N);
    a.m_blocks = (P + BM - 1) / BM;
    a.k_blocks = (split ? 3 : 1) * c->Kpad / BKB;
    a.kb1 = c->Kpad / BKB; a.split = split ? 1 : 0;
    const int npos = tc_num_positions(c->family, c->degree, c->F, c->K);
    a.k_last = (npos - (c->Kpad - BKB) + UMMA_K - 1) / UMMA_K;      // real k-steps in the last k-block of a K range (split: three ranges)
    a.P = P; a.Ppad = ((P + 255) / 256) * 256; a.generations = generations; a.err = c->err;
    a.N = c->N; a.tgt = c->t; a.R = c->R; a.stop_error = gp->stop_error;
    a.local = persistent_local(c, P) ? 1 : 0;
    if (a.local) {                              // two buffers of tile sums (one grid barrier per generation)
        const size_t need = (size_t)2 * a.n_tiles * a.Ppad;
        if (need > c->partial_cap) {
            if (c->partial) { cudaFree(c->partial); c->partial = nullptr; c->partial_cap = 0; }
            GAME_CUDA(c, cudaMalloc(&c->partial, need * sizeof(float)));
            c->partial_cap = need;
        }
    }
    a.partial = c->partial; a.fit = c->fit; a.order = c->order;
    a.pop_a = c->pop; a.pop_b = c->pop_next;
    a.state = c->state; a.gbar = c->gbar;
    fill_step_args(c, gp, seed, (unsigned int)c->generation, &a.step);
    a.step.sink = tensor_sink(c, split);
    const int mode = c->act == GAME_ACT_IDENTITY ? MODE_IDENTITY : (int)(a.step.sink.scale == 0.5f ? MODE_SIG_TANH32 : MODE_SIG_EXACT);
    int rc = tensor_encode_population_map(c, split, a.Ppad);
    if (rc) return rc;
    const CUtensorMap &tmC = *(const CUtensorMap *)c->tmap_C;
    const CUtensorMap &tmE = ((const CUtensorMap *)(split ? c->tmap_Es : c->tmap_E))[1];        // 128-row boxes
    const int grid = a.n_tiles * a.m_blocks;
    const int smem = (int)persistent_smem_bytes(c, path, P);
    const bool tmse = c->err == GAME_ERR_TMSE;
    switch (mode) {
    case MODE_IDENTITY: return tmse ? launch_persistent_variant<MODE_IDENTITY, true>(c, tmC, tmE, a, grid, smem)
                                    : launch_persistent_variant<MODE_IDENTITY, false>(c, tmC, tmE, a, grid, smem);
    case MODE_SIG_TANH32: return tmse ? launch_persistent_variant<MODE_SIG_TANH32, true>(c, tmC, tmE, a, grid, smem)
                                      : launch_persistent_variant<MODE_SIG_TANH32, false>(c, tmC, tmE, a, grid, smem);
    default: return tmse ? launch_persistent_variant<MODE_SIG_EXACT, true>(c, tmC, tmE, a, grid, smem)
                         : launch_persistent_variant<MODE_SIG_EXACT, false>(c, tmC, tmE, a, grid, smem);
    }
}

}  // namespace game
