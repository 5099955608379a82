// probes.cuh -- launchers of the measurement probes (probes.cu), called by the cans_probe_* entry points.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace cans {

// tile t of a 2-D tensor map: nbox boxes of box_rows x box_cols doubles at (c0, c1) = ((t % m0) * s0, (t / m0) * s1 + q * box_rows)
struct TileCopyShape {
    long ntiles, m0;
    int s0, s1, nbox, box_rows, box_cols;
};

// FP64 FMA instructions per second of the whole device (8 independent chains per thread, 2048 threads per SM); synchronises
cudaError_t probe_fp64_fma(int num_sms, double* fma_per_s, cudaStream_t st);
// duration of one in-place TMA copy of every tile (the data is rewritten unchanged); synchronises
cudaError_t probe_tile_copy(const CUtensorMap* tmap, const TileCopyShape& sh, int num_sms, float* ms, cudaStream_t st);

}  // namespace cans
