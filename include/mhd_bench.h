/* include/mhd_bench.h — measurement plumbing of libmhd used by bench.py and the profiling runs.  NOT part of the method
 * or of the product boundary (include/mhd.h): nothing here changes what the library computes. */
#ifndef MHD_BENCH_H
#define MHD_BENCH_H

#include "mhd.h"

#ifdef __cplusplus
extern "C" {
#endif

/* A/B switches for mhd_set_option(): alternative kernels that were built, are parity-tested and measured SLOWER than the
 * defaults on B200 (DESIGN.md section 6 has the numbers).  They exist so that the measurements can be repeated; they are
 * not part of the method's interface. */
/* Option ids 7 and 10 belonged to switches of earlier revisions (columns per strided tile, L2 slab loop) and stay reserved:
 * mhd_set_option() refuses them with MHD_ERR_INVALID_ARG instead of giving an old caller's value a new meaning. */
#define MHD_OPT_FUSE_ASSEMBLE 14 /* sweep S5 (in-core contexts, default equation set, N = 64..512) as ONE launch: the forward z
                                pass runs in thread-block clusters — 1: 16 CTAs, one per product field; 2: 8 CTAs, two
                                fields each — that keep the transformed rows in shared memory and assemble R^ and the
                                explicit update from each other's tiles (distributed shared memory).  Bitwise the
                                two-launch result; measured slower on B200, so the default is
                                0: forward z pass and assembly as two launches.  Where the device cannot co-schedule
                                the cluster (cudaOccupancyMaxActiveClusters = 0 or an error) the two launches run
                                whatever the option says                                                       */

#define MHD_OPT_TMA 13 /* 1: the in-core y / z passes (N = 128, 256, 512; all but the pass that builds J^ on load) run as a
                          persistent pipeline fed by the tensor-memory accelerator (cp.async.bulk.tensor into a ring of
                          shared-memory tiles, mbarrier completion); 0 (default): every CTA loads its tile into registers
                          itself — measured faster at every size.  Same results to roundoff
                          (bitwise at N = 128, 256, where both use the same butterfly plan)                         */

/* Measurement helper for the bench (not part of the method): fp64 instructions per second of a register-only DFMA
 * kernel on the current device = the issue ceiling of the fp64 pipe ("measure it with an FMA
 * micro-benchmark"); flop/s of pure-FMA code is twice that. */
int mhd_probe_fp64(mhd_ctx *ctx, double *instr_per_s);

/* Milliseconds and launches accumulated per kernel family since the last reset; names[i] are static strings.
 * Timing uses CUDA events on the bound stream and is only collected while enabled (adds synchronisation). */
int mhd_profile_enable(mhd_ctx *ctx, int on);
int mhd_profile_get(mhd_ctx *ctx, int max_entries, const char **names, double *ms, long long *launches);

/* Launches of the alternative kernels so far, so that an A/B test can tell that the path it asked for really ran and did
 * not quietly fall back to the default (no tensor maps, an ineligible pass, clusters unavailable):
 * which = MHD_OPT_TMA: strided passes run by the TMA pipeline; which = MHD_OPT_FUSE_ASSEMBLE: one-launch S5 sweeps.
 * Returns -1 for any other `which`. */
long long mhd_alt_launch_count(const mhd_ctx *ctx, int which);

#ifdef __cplusplus
}
#endif
#endif /* MHD_BENCH_H */
