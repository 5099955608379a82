// xy_group_a.cu -- instantiates the x/y transform kernels for the lengths of CANS_FFT_SIZES_A
// (fft_sizes.h); the split into four files only lets them compile in parallel.
#include "fft_sizes.h"
#include "xy_kernels.cuh"

namespace cans {

bool launch_xy_group_a(int n, int op, const XYArgs& a, cudaStream_t st, cudaError_t* err) {
    switch (n) {
#define CANS_CASE(N, R1, R2, R3, NFX, NTX, TXC, NTY) \
        case N: *err = launch_xy<FftPlan<N, R1, R2, R3>, NFX, NTX, TXC, NTY>(op, a, st); return true;
        CANS_FFT_SIZES_A(CANS_CASE)
#undef CANS_CASE
        default: return false;
    }
}

}  // namespace cans
