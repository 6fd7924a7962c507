/*
 * game_bench.h -- measurement aids of libgame_b200.  NOT part of the product API (include/game.h, which does not include
 * this file): bench.py, the profiles and a few tests use them to time the dominant kernel, count launches, measure the
 * pipe peaks the "alu" rooflines are quoted against and switch launch configurations for A/B runs.  None of
 * them changes what is computed beyond the tolerance class stated in game.h.  Same conventions as game.h (return codes,
 * DEV / HOST pointers, game_last_error).
 */
#ifndef GAME_B200_BENCH_H
#define GAME_B200_BENCH_H

#include "game.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Launch-configuration knobs of game_set_tuning: measurement aids, none changes what is computed beyond the stated
 * tolerance class.  value -1 restores the automatic choice.
 *   GAME_TUNE_PDL          1/0  programmatic dependent launch between the kernels of a generation (auto: 1)
 *   GAME_TUNE_CTA_GROUP    1/2  single CTAs or cta_group::2 pairs in the tensor kernel (auto: by shape)
 *   GAME_TUNE_SIGMOID      0 ex2+rcp logistic, 2 tanh.approx logistic (TENSOR path; auto: 2)
 *   GAME_TUNE_RESIDENT     1/0  resident population tile for P <= 256 (auto: 1)
 *   GAME_TUNE_TEAMS        1/0  two-team epilogue (auto: contraction depth <= 256)
 *   GAME_TUNE_HALF_TILES   1/0  128-pattern tiles for sub-wave problems (auto: by shape)
 *   GAME_TUNE_PERSISTENT   1/0  one persistent cooperative kernel per game_evolve for sub-wave problems (auto: by shape)
 *                          2 = the persistent kernel without its local-population form (every CTA holding the whole population)
 *   GAME_TUNE_RATIONAL_SHARE  0 = every tanh logistic on the special-function unit; 1..8 (or auto) = 3 of every 16
 *                          evaluation PAIRS on the FMA pipe by a rational form with one shared reciprocal (team epilogue,
 *                          single CTAs) -- the measured best of the sweep in DESIGN.md section 7, the only share built */
enum { GAME_TUNE_PDL = 0, GAME_TUNE_CTA_GROUP = 1, GAME_TUNE_SIGMOID = 2, GAME_TUNE_RESIDENT = 3, GAME_TUNE_TEAMS = 4,
       GAME_TUNE_HALF_TILES = 5, GAME_TUNE_PERSISTENT = 6, GAME_TUNE_RATIONAL_SHARE = 7, GAME_TUNE_COUNT_ = 8 };

/* Launch-configuration knob (GAME_TUNE_*), per context; unknown knobs / values give GAME_ERR_INVALID_ARG. */
int game_set_tuning(game_ctx *ctx, int knob, int value);

/* Number of kernels this context has launched since creation (bench.py reports it). */
long long game_launch_count(const game_ctx *ctx);

/* Measurement aid: while enabled, every launch of the dominant kernel (the fused contraction +
 * epilogue of game_fitness / game_evolve) is bracketed by CUDA events on the context's stream.
 * game_get_kernel_timing synchronises the stream, returns the summed duration in milliseconds and the
 * number of launches since the last call, and resets both.  HOST out pointers.  While enabled, game_evolve
 * issues its kernels one by one instead of replaying a captured CUDA graph (events cannot be timed inside one). */
int game_set_kernel_timing(game_ctx *ctx, int enabled);
int game_get_kernel_timing(game_ctx *ctx, double *total_ms, long long *launches);

/* Measurement aid: register-only micro-benchmarks of the pipes the "alu" rooflines are quoted against, one
 * CTA per SM, timed with CUDA events on the context's stream; synchronises.  kind = GAME_PEAK_*; param = FMA instructions
 * per tanh for GAME_PEAK_TANH_MIX (0..8), ignored otherwise.  *ops_per_s (HOST) = fused multiply-adds (FFMA, FFMA2: count
 * both lanes) or special-function results per second over the whole GPU; *ms (HOST, may be NULL) = the timed launch. */
enum { GAME_PEAK_FFMA = 0, GAME_PEAK_FFMA2 = 1, GAME_PEAK_TANH = 2, GAME_PEAK_EX2 = 3, GAME_PEAK_TANH_MIX = 4 };
int game_microbench(game_ctx *ctx, int kind, int param, double *ops_per_s, double *ms);

#ifdef __cplusplus
}
#endif
#endif
