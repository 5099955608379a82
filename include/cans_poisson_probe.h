/*
 * cans_poisson_probe.h -- measurement probes exported by libcans_poisson.so for bench.py.  They are bench tooling, not part
 * of the projection API (include/cans_poisson.h): the denominators that kernel numbers are read against.
 */
#ifndef CANS_POISSON_PROBE_H
#define CANS_POISSON_PROBE_H

#include "cans_poisson.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Both synchronise the stream.
 *   cans_probe_fp64_fma   FP64 FMA instructions per second of the current device (independent chains on every SM): the
 *                         measured peak of the plain FP64 pipe.
 *   cans_probe_tile_copy  duration (ms) of a bare in-place TMA copy -- tile in, tile out, no arithmetic, data unchanged --
 *                         of the field p (DEVICE, nx*ny*nz doubles) with exactly the tiles of the z solve (which = 0:
 *                         16 / 32 / 8 columns x nz rows) or of the TMA-fed y transforms (which = 1: 16 doubles x ny rows,
 *                         ny = 512, 768 only): the HBM ceiling of that access pattern.  which = 2: the z view with tiles of
 *                         32 columns x 256 rows -- the same plane-strided rows, twice as wide (every row of a z tile lies
 *                         in another 2 MB page: the rate follows the bytes moved per row).
 *                         2*8*N bytes move per call.
 */
int cans_probe_fp64_fma(double* fma_per_s, void* stream);
int cans_probe_tile_copy(cans_poisson_plan* plan, double* p, int which, float* ms, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CANS_POISSON_PROBE_H */
