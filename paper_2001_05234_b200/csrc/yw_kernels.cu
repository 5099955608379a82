// yw_kernels.cu -- __global__ wrappers and launcher of the warp-per-column y transforms (yw_pass.cuh).
#include "yw_kernels.cuh"

namespace cans {

extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <int N, int R1, bool INV>
__global__ void __launch_bounds__(YW_NT, 2) yw_kernel(const XYArgs a, const cplx* __restrict__ tw) {
    typedef YWPass<N, R1> W;
    cplx* tile = reinterpret_cast<cplx*>(cans_dyn_smem);
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int ctile = blockIdx.x;
    const int k = a.k0 + blockIdx.y;
    if (INV) {
        W::load_inverse(a, tile, ctile, k, tid);
        __syncthreads();
        for (int c = warp; c < YW_TXC; c += YW_WARPS) W::column_inverse(tile + c, tw, lane);
        __syncthreads();
        W::store_inverse(a, tile, ctile, k, tid);
    } else {
        W::load_forward(a, tile, ctile, k, tid);
        __syncthreads();
        for (int c = warp; c < YW_TXC; c += YW_WARPS) W::column_forward(tile + c, tw, lane);
        __syncthreads();
        W::store_forward(a, tile, ctile, k, tid);
    }
}

template <int N, int R1>
static cudaError_t yw_launch_n(int op, const XYArgs& a, const cplx* tw, cudaStream_t st) {
    const size_t smem = sizeof(cplx) * (size_t)YWPass<N, R1>::TILE;
    if (op == OP_CONFIGURE) {
        cudaError_t e = cudaFuncSetAttribute(yw_kernel<N, R1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(yw_kernel<N, R1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    }
    dim3 grid((unsigned)(a.nx / 2 / YW_TXC), (unsigned)a.nk);
    if (op == OP_Y_FWD) yw_kernel<N, R1, false><<<grid, YW_NT, smem, st>>>(a, tw);
    else yw_kernel<N, R1, true><<<grid, YW_NT, smem, st>>>(a, tw);
    return cudaGetLastError();
}

bool yw_launch(int n, int op, const XYArgs& a, const cplx* tw, cudaStream_t st, cudaError_t* err) {
    switch (n) {
        case 512: *err = yw_launch_n<512, 16>(op, a, tw, st); return true;
        case 768: *err = yw_launch_n<768, 24>(op, a, tw, st); return true;
        case 1024: *err = yw_launch_n<1024, 32>(op, a, tw, st); return true;
        default: return false;
    }
}

}  // namespace cans
