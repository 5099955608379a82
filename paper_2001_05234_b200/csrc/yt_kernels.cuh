// yt_kernels.cuh -- host-callable launcher of the TMA-fed y transforms (defined in yt_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include "yt_pass.cuh"
#include "xy_kernels.cuh"

namespace cans {

// op: OP_Y_FWD, OP_Y_INV, or OP_CONFIGURE at plan time; tw = W_N^(p k1) table [R1][32] of the plan; tmap = the tensor map of
// the whole field a.p (yt_make_tensor_map; a.p 16-byte aligned, a.nx / 2 a multiple of YT_COLS); the launch covers planes
// [a.k0, a.k0 + a.nk) with at most max_ctas persistent CTAs.  Returns false if length n has no TMA-fed kernel.
bool yt_launch(int n, int op, const XYArgs& a, const cplx* tw, const CUtensorMap* tmap, int max_ctas, cudaStream_t st,
               cudaError_t* err);
cudaError_t yt_make_tensor_map(CUtensorMap* tmap, const double* p, int nx, int ny, int nz);

}  // namespace cans
