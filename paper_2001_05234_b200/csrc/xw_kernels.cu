// xw_kernels.cu -- __global__ wrappers and launcher of the warp-per-line x transforms (xw_pass.cuh).
#include "xw_kernels.cuh"

namespace cans {

extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <int N, int R1, int MODE>   // MODE: 0 forward, 1 forward + divergence, 2 inverse
__global__ void __launch_bounds__(XW_WARPS * 32, 2) xw_kernel(const XYArgs a, const cplx* __restrict__ tw, long npairs) {
    typedef XWPass<N, R1> W;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    cplx* buf = reinterpret_cast<cplx*>(cans_dyn_smem) + warp * W::BUF;
    const long pr = (long)blockIdx.x * XW_WARPS + warp;
    if (pr >= npairs) return;                           // whole warp leaves: no CTA barrier is used
    const int hp = a.ny >> 1;
    const int kl = (int)(pr / hp);
    const int k = a.k0 + kl;
    const int j = 2 * (int)(pr - (long)kl * hp);
    const size_t ro = ((size_t)k * a.ny + j) * (size_t)a.nx;
    if (MODE == 2) W::inverse(a, tw, buf, ro, lane);
    else W::template forward<MODE == 1>(a, tw, buf, ro, j, k, lane);
}

template <int N, int R1>
static cudaError_t xw_launch_n(int op, const XYArgs& a, const cplx* tw, cudaStream_t st) {
    const size_t smem = sizeof(cplx) * (size_t)XW_WARPS * XWPass<N, R1>::BUF;
    if (op == OP_CONFIGURE) {
        cudaError_t e = cudaFuncSetAttribute(xw_kernel<N, R1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xw_kernel<N, R1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xw_kernel<N, R1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    }
    const long npairs = (long)(a.ny / 2) * a.nk;
    const unsigned grid = (unsigned)((npairs + XW_WARPS - 1) / XW_WARPS);
    if (op == OP_X_FWD) xw_kernel<N, R1, 0><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    else if (op == OP_X_FWD_DIV) xw_kernel<N, R1, 1><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    else xw_kernel<N, R1, 2><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    return cudaGetLastError();
}

bool xw_launch(int n, int op, const XYArgs& a, const cplx* tw, cudaStream_t st, cudaError_t* err) {
    switch (n) {
        case 512: *err = xw_launch_n<512, 16>(op, a, tw, st); return true;
        case 768: *err = xw_launch_n<768, 24>(op, a, tw, st); return true;
        case 1024: *err = xw_launch_n<1024, 32>(op, a, tw, st); return true;
        default: return false;
    }
}

}  // namespace cans
