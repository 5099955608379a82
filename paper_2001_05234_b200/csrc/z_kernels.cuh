// z_kernels.cuh -- host-callable launchers of the z-solve kernels (defined in z_solve.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "z_pass.cuh"

namespace cans {

constexpr int Z_MROWS = 16;   // rows per thread in the z solve

// columns per CTA for a given segment count (threads = TC * nseg <= 512)
inline int z_tc_for(int nseg) { return nseg <= 16 ? 32 : (nseg <= 32 ? 16 : 8); }

// dynamic shared memory of the solve kernel (two tile buffers + tables; the periodic-z kernel parks its correction vector
// in the tile's own staging buffer and needs no more); host arithmetic only
size_t z_solve_smem_bytes(int nseg);
constexpr size_t Z_SMEM_LIMIT = 227u * 1024u;
// plan time: opt in to the dynamic shared memory of the solve kernel and compute the persistent grid
cudaError_t z_solve_configure(int nseg, int cyclic, int num_sms, int* grid_out, size_t* smem_out);   // cudaErrorInvalidConfiguration: the tile buffers do not fit
// TMA boxes covering the padded column exactly: nbox boxes of box_rows (<= 256) rows
void z_boxes(int nseg, int* nbox, int* box_rows);
// tensor map of the (nz, nx*ny) view of the field p, boxes of z_tc_for(nseg) columns
cudaError_t z_make_tensor_map(CUtensorMap* tmap, const double* p, long ncols, int nz, int nseg);
// enqueue the solve (a.ticket must point at a zeroed counter; tmap from z_make_tensor_map for a.p)
cudaError_t z_solve_launch(const ZArgs& a, int grid, size_t smem, const CUtensorMap* tmap, cudaStream_t st);
// fill rstart / r00 for the shift a.alpha (enqueued on st: at plan time for alpha = 0, again whenever a Helmholtz solve
// changes the shift)
cudaError_t z_setup_launch(const ZArgs& a, double* rstart, double* r00, cudaStream_t st);

}  // namespace cans
