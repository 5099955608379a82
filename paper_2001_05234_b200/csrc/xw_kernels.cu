// xw_kernels.cu -- __global__ wrappers and launcher of the warp-per-line x transforms (xw_pass.cuh).
#include "xw_kernels.cuh"

namespace cans {

extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <int N, int R1, int MODE, int KC>   // MODE: 0 forward, 1 forward + divergence, 2 inverse; KC: class of the boundary pair
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
    if (MODE == 2) W::template inverse<KC>(a, tw, buf, ro, lane);
    else W::template forward<MODE == 1, KC>(a, tw, buf, ro, j, k, lane);
}

template <int N, int R1, int KC>
static cudaError_t xw_launch_k(int op, const XYArgs& a, const cplx* tw, cudaStream_t st) {
    // N = 1024: at least 80 KB per CTA, i.e. two CTAs (8 warps) per SM whatever the register count -- the lean periodic
    // kernels would fit three, which measured slower there (1.25 against 1.00 ms for the x inverse of the 1024 x 768 x 512
    // grid); the shorter lines do run faster with three (512: 0.17 against 0.20 ms on 512 x 512 x 256)
    size_t smem = sizeof(cplx) * (size_t)XW_WARPS * XWPass<N, R1>::BUF;
    if (N >= 1024 && smem < 80 * 1024) smem = 80 * 1024;
    if (op == OP_CONFIGURE) {
        cudaError_t e = cudaFuncSetAttribute(xw_kernel<N, R1, 0, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xw_kernel<N, R1, 1, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(xw_kernel<N, R1, 2, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    }
    const long npairs = (long)(a.ny / 2) * a.nk;
    const unsigned grid = (unsigned)((npairs + XW_WARPS - 1) / XW_WARPS);
    if (op == OP_X_FWD) xw_kernel<N, R1, 0, KC><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    else if (op == OP_X_FWD_DIV) xw_kernel<N, R1, 1, KC><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    else xw_kernel<N, R1, 2, KC><<<grid, XW_WARPS * 32, smem, st>>>(a, tw, npairs);
    return cudaGetLastError();
}

// one kernel per class of boundary pair: 0 = PP, 1 = NN / DD, 2 = ND / DN
template <int N, int R1>
static cudaError_t xw_launch_n(int op, const XYArgs& a, const cplx* tw, cudaStream_t st) {
    if (op == OP_CONFIGURE) {                            // plan time: every class (the opt-in is per kernel)
        cudaError_t e = xw_launch_k<N, R1, 0>(op, a, tw, st);
        if (e == cudaSuccess) e = xw_launch_k<N, R1, 1>(op, a, tw, st);
        if (e == cudaSuccess) e = xw_launch_k<N, R1, 2>(op, a, tw, st);
        return e;
    }
    if (a.kind == KIND_PP) return xw_launch_k<N, R1, 0>(op, a, tw, st);
    return kind_mixed(a.kind) ? xw_launch_k<N, R1, 2>(op, a, tw, st) : xw_launch_k<N, R1, 1>(op, a, tw, st);
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
