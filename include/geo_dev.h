/* geo_dev.h -- DEVELOPMENT / MEASUREMENT helpers of libgeo.  NOT part of the operation's boundary (SURVEY 8(b)
 * lists neither): nothing here integrates a geodesic.  bench.py uses them to report the launch geometry and to
 * measure the FP64 FMA ceiling of the machine it runs on (MEASURED_PEAKS.json has no FP64 entry; SURVEY 8(d) asks
 * for a register-only DFMA microbenchmark beside the nominal peak). */
#ifndef GEO_DEV_H_
#define GEO_DEV_H_

#include "geo.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Launch geometry the next geo_integrate call on this ctx would use for (n, flags, snapshot_every):
 * info = { grid, block size, registers per thread, resident CTAs per SM }. */
int geo_launch_info(geo_ctx *ctx, int64_t n, int32_t flags, int64_t snapshot_every, int32_t info[4]);

/* Runs a register-only chain of dependence-free FP64 FMAs (`iters` x 64 DFMA per thread over a full-chip grid)
 * on `cuda_stream` and writes the number of FMAs executed to *n_fma (host).  Times nothing itself: the caller
 * brackets it with CUDA events.  `sink` is a device buffer of >= 8 bytes. */
int geo_probe_dfma(geo_ctx *ctx, int64_t iters, double *sink, double *n_fma, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GEO_DEV_H_ */
