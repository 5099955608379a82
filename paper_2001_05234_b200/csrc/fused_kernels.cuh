// fused_kernels.cuh -- instantiation helper of the fused pass-A / pass-C kernels (fused_pass.cuh):
// one translation unit per nx (fused_x*.cu, compiled in parallel), each covering every fused ny.
#pragma once
#include "fft_sizes.h"
#include "fused_pass.cuh"

namespace cans {

// radices of a transform length: the single table of fft_sizes.h (the plan's twiddle tables use the same)
template <int N> struct PlanOf;
#define CANS_PLANOF(N, R1, R2, R3, NFX, NTX, TXC, NTY) \
    template <> struct PlanOf<N> { typedef FftPlan<N, R1, R2, R3> type; };
CANS_FFT_SIZES(CANS_PLANOF)
#undef CANS_PLANOF

template <int NX>
bool fused_dispatch_nx(int ny, int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem,
                       cudaStream_t st, cudaError_t* err) {
    typedef typename PlanOf<NX>::type PX;
    constexpr int NFX = fused_nfx(NX);
    switch (ny) {
#define CANS_FY(NY) \
        case NY: *err = fused_run<PX, typename PlanOf<NY>::type, NFX, fused_txc(NY), FUSED_NT>( \
                            what, a, num_sms, grid, smem, st); return true;
        CANS_FY(256) CANS_FY(384) CANS_FY(512) CANS_FY(768) CANS_FY(1024)
#undef CANS_FY
        default: return false;
    }
}

#define CANS_FUSED_DECL(NX) \
    bool fused_dispatch_##NX(int ny, int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem, \
                             cudaStream_t st, cudaError_t* err);
CANS_FUSED_DECL(256) CANS_FUSED_DECL(384) CANS_FUSED_DECL(512) CANS_FUSED_DECL(768) CANS_FUSED_DECL(1024)

#define CANS_FUSED_DEFINE(NX) \
    bool fused_dispatch_##NX(int ny, int what, const FusedArgs* a, int num_sms, int* grid, size_t* smem, \
                             cudaStream_t st, cudaError_t* err) { \
        return fused_dispatch_nx<NX>(ny, what, a, num_sms, grid, smem, st, err); \
    }

}  // namespace cans
