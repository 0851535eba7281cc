/* include/mhd_bench.h — measurement plumbing of libmhd used by bench.py and the profiling runs.  NOT part of the method
 * or of the product boundary (include/mhd.h): nothing here changes what the library computes. */
#ifndef MHD_BENCH_H
#define MHD_BENCH_H

#include "mhd.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement helper for the bench (not part of the method): fp64 instructions per second of a register-only DFMA
 * kernel on the current device = the issue ceiling of the fp64 pipe ("measure it with an FMA
 * micro-benchmark"); flop/s of pure-FMA code is twice that. */
int mhd_probe_fp64(mhd_ctx *ctx, double *instr_per_s);

/* Milliseconds and launches accumulated per kernel family since the last reset; names[i] are static strings.
 * Timing uses CUDA events on the bound stream and is only collected while enabled (adds synchronisation). */
int mhd_profile_enable(mhd_ctx *ctx, int on);
int mhd_profile_get(mhd_ctx *ctx, int max_entries, const char **names, double *ms, long long *launches);

#ifdef __cplusplus
}
#endif
#endif /* MHD_BENCH_H */
