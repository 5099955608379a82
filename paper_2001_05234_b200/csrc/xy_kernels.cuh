// xy_kernels.cuh -- __global__ wrappers of the x / y transform phases and their per-size launchers.
// Included by the xy_group*.cu translation units, each of which instantiates a few transform lengths
// (split only to compile in parallel).
#pragma once
#include <cuda_runtime.h>
#include "xy_pass.cuh"

namespace cans {

// OP_CONFIGURE (plan time, on the plan's device): opt in to the dynamic shared memory of every kernel of a length
enum XYOp : int { OP_X_FWD = 0, OP_X_FWD_DIV = 1, OP_X_INV = 2, OP_Y_FWD = 3, OP_Y_INV = 4, OP_CONFIGURE = 5 };

extern __shared__ __align__(16) unsigned char cans_dyn_smem[];

template <class P, int NF, int NT, int MODE>   // MODE: 0 fwd, 1 fwd+div, 2 inv
__global__ void __launch_bounds__(NT, 2) x_pass_kernel(const XYArgs a, long npairs) {
    typedef XPass<P, NF, NT> X;
    cplx* sm = reinterpret_cast<cplx*>(cans_dyn_smem);
    const int tid = threadIdx.x;
    const long pair0 = (long)blockIdx.x * NF;
    X::load_twiddles(a, sm, tid);
    if (MODE == 2) {
        X::load_inverse(a, sm, pair0, npairs, tid);
        __syncthreads();
        X::pass3_inv(sm, tid);
        __syncthreads();
        if (P::R2 > 1) { X::pass2_inv(sm, tid); __syncthreads(); }
        X::pass1_inv(sm, tid);
        __syncthreads();
        X::store_inverse(a, sm, pair0, npairs, tid);
    } else {
        X::template load_forward<MODE == 1>(a, sm, pair0, npairs, tid);
        __syncthreads();
        X::pass1_fwd(sm, tid);
        __syncthreads();
        if (P::R2 > 1) { X::pass2_fwd(sm, tid); __syncthreads(); }
        X::pass3_fwd(sm, tid);
        __syncthreads();
        X::store_forward(a, sm, pair0, npairs, tid);
    }
}

template <class P, int TXC, int NT, bool INV>
__global__ void __launch_bounds__(NT, 2) y_pass_kernel(const XYArgs a) {
    typedef YPass<P, TXC, NT> Y;
    cplx* sm = reinterpret_cast<cplx*>(cans_dyn_smem);
    const int tid = threadIdx.x;
    const int ctile = blockIdx.x;
    const int k = a.k0 + blockIdx.y;
    Y::load_twiddles(a, sm, tid);
    if (INV) {
        Y::load_inverse(a, sm, ctile, k, tid);
        __syncthreads();
        Y::pass3_inv(sm, tid);
        __syncthreads();
        if (P::R2 > 1) { Y::pass2_inv(sm, tid); __syncthreads(); }
        Y::pass1_inv(sm, tid);
        __syncthreads();
        Y::store_inverse(a, sm, ctile, k, tid);
    } else {
        Y::load_forward(a, sm, ctile, k, tid);
        __syncthreads();
        Y::pass1_fwd(sm, tid);
        __syncthreads();
        if (P::R2 > 1) { Y::pass2_fwd(sm, tid); __syncthreads(); }
        Y::pass3_fwd(sm, tid);
        __syncthreads();
        Y::store_forward(a, sm, ctile, k, tid);
    }
}

template <class K>
static cudaError_t set_smem(K kern, size_t bytes) {
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// Launch one x/y operation for transform plan P.  Returns cudaSuccess or the launch error.
template <class P, int NFX, int NTX, int TXC, int NTY>
cudaError_t launch_xy(int op, const XYArgs& a, cudaStream_t st) {
    typedef XPass<P, NFX, NTX> X;
    typedef YPass<P, TXC, NTY> Y;
    const size_t smx = sizeof(cplx) * X::SMEM_CPLX;
    const size_t smy = sizeof(cplx) * Y::SMEM_CPLX;
    if (op == OP_CONFIGURE) {
        cudaError_t e = set_smem(x_pass_kernel<P, NFX, NTX, 0>, smx);
        if (e == cudaSuccess) e = set_smem(x_pass_kernel<P, NFX, NTX, 1>, smx);
        if (e == cudaSuccess) e = set_smem(x_pass_kernel<P, NFX, NTX, 2>, smx);
        if (e == cudaSuccess) e = set_smem(y_pass_kernel<P, TXC, NTY, false>, smy);
        if (e == cudaSuccess) e = set_smem(y_pass_kernel<P, TXC, NTY, true>, smy);
        return e;
    }
    if (op == OP_X_FWD || op == OP_X_FWD_DIV || op == OP_X_INV) {
        const long npairs = (long)(a.ny / 2) * a.nk;
        const unsigned grid = (unsigned)((npairs + NFX - 1) / NFX);
        if (op == OP_X_FWD) x_pass_kernel<P, NFX, NTX, 0><<<grid, NTX, smx, st>>>(a, npairs);
        else if (op == OP_X_FWD_DIV) x_pass_kernel<P, NFX, NTX, 1><<<grid, NTX, smx, st>>>(a, npairs);
        else x_pass_kernel<P, NFX, NTX, 2><<<grid, NTX, smx, st>>>(a, npairs);
    } else {
        dim3 grid((unsigned)(a.nx / 2 / TXC), (unsigned)a.nk);
        if (op == OP_Y_FWD) y_pass_kernel<P, TXC, NTY, false><<<grid, NTY, smy, st>>>(a);
        else y_pass_kernel<P, TXC, NTY, true><<<grid, NTY, smy, st>>>(a);
    }
    return cudaGetLastError();
}

// Each group file defines one of these: returns true if it owns transform length n (and sets *err).
bool launch_xy_group_a(int n, int op, const XYArgs& a, cudaStream_t st, cudaError_t* err);
bool launch_xy_group_b(int n, int op, const XYArgs& a, cudaStream_t st, cudaError_t* err);
bool launch_xy_group_c(int n, int op, const XYArgs& a, cudaStream_t st, cudaError_t* err);
bool launch_xy_group_d(int n, int op, const XYArgs& a, cudaStream_t st, cudaError_t* err);

}  // namespace cans
