// z_solve.cu -- pass B: persistent, cp.async double-buffered partitioned Thomas solve (z_pass.cuh).
#include "z_kernels.cuh"

namespace cans {

template <int MROWS, int TC>
__global__ void __launch_bounds__(512) z_solve_kernel(const ZArgs a) {
    extern __shared__ __align__(16) double zsm[];
    typedef ZPass<MROWS, TC> Z;
    __shared__ long s_next;
    const int tid = threadIdx.x;
    const int nthreads = blockDim.x;
    double* bufs = zsm + Z::table_doubles(a.nseg);
    const size_t tile_sz = Z::tile_doubles(a.nseg);

    if (a.singular && blockIdx.x == 0) {
        // the singular (0,0) column, staged in shared memory, solved by one thread (reading S3)
        for (int k = tid; k < a.nz; k += nthreads) bufs[k] = a.p[(size_t)k * a.ncols];
        __syncthreads();
        if (tid == 0) z_singular_column(a, bufs);
        __syncthreads();
    }
    Z::load_tables(a, zsm, tid, nthreads);
    if (tid == 0) s_next = (long)atomicAdd(a.ticket, 1u);
    __syncthreads();
    long cur = s_next;
    __syncthreads();
    if (cur >= a.ntiles) return;
    Z::prefetch_tile(a, bufs, cur, tid, nthreads);
    cp_async_commit();
    if (tid == 0) s_next = (long)atomicAdd(a.ticket, 1u);
    int b = 0;
    const int c = tid % TC;
    const int s = tid / TC;
    while (true) {
        __syncthreads();                       // s_next visible; buffer b^1 no longer read by anyone
        const long nxt = s_next;
        if (nxt < a.ntiles) Z::prefetch_tile(a, bufs + (size_t)(b ^ 1) * tile_sz, nxt, tid, nthreads);
        cp_async_commit();
        // per-thread scalars of the current tile (tables are L2/L1 resident; rstart is streamed once)
        const long col = cur * TC + c;
        double rs = 0.0, lam = 0.0;
        if (col < a.ncols) {
            rs = a.rstart[(size_t)s * a.ncols + col];
            lam = a.lamx[(int)(col % a.nx)] + a.lamy[(int)(col / a.nx)];
        }
        cp_async_wait<1>();                    // the current tile has landed (the next may still fly)
        __syncthreads();
        if (tid == 0 && nxt < a.ntiles) s_next = (long)atomicAdd(a.ticket, 1u);
        ZState<MROWS> st;
        Z::phase1(a, zsm, bufs + (size_t)b * tile_sz, st, cur, rs, lam, tid);
        __syncthreads();
        Z::phase2a(a, zsm, st, tid);
        __syncthreads();
        Z::phase2b(a, zsm, st, tid);
        __syncthreads();
        Z::phase3(a, zsm, st, tid);
        if (nxt >= a.ntiles) break;
        cur = nxt;
        b ^= 1;
    }
    cp_async_wait<0>();
}

template <int MROWS>
__global__ void z_setup_kernel(const ZArgs a, double* rstart, double* r00) {
    const long col = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (col < a.ncols) z_setup_column<MROWS>(a, rstart, r00, col);
}

template <int TC>
static cudaError_t configure_tc(int nseg, int nz, int num_sms, int* grid_out, size_t* smem_out) {
    size_t smem = sizeof(double) * ZPass<Z_MROWS, TC>::smem_doubles(nseg);
    (void)nz;
    cudaError_t e = cudaFuncSetAttribute(z_solve_kernel<Z_MROWS, TC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, z_solve_kernel<Z_MROWS, TC>, TC * nseg, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    if (per_sm > 4) per_sm = 4;
    *grid_out = per_sm * num_sms;
    *smem_out = smem;
    return cudaSuccess;
}

cudaError_t z_solve_configure(int nseg, int nz, int num_sms, int* grid_out, size_t* smem_out) {
    switch (z_tc_for(nseg)) {
        case 32: return configure_tc<32>(nseg, nz, num_sms, grid_out, smem_out);
        case 16: return configure_tc<16>(nseg, nz, num_sms, grid_out, smem_out);
        default: return configure_tc<8>(nseg, nz, num_sms, grid_out, smem_out);
    }
}

cudaError_t z_solve_launch(const ZArgs& a, int grid, size_t smem, cudaStream_t st) {
    long g = grid;
    if (g > a.ntiles) g = a.ntiles;
    if (g < 1) g = 1;
    switch (z_tc_for(a.nseg)) {
        case 32: z_solve_kernel<Z_MROWS, 32><<<(unsigned)g, 32 * a.nseg, smem, st>>>(a); break;
        case 16: z_solve_kernel<Z_MROWS, 16><<<(unsigned)g, 16 * a.nseg, smem, st>>>(a); break;
        default: z_solve_kernel<Z_MROWS, 8><<<(unsigned)g, 8 * a.nseg, smem, st>>>(a); break;
    }
    return cudaGetLastError();
}

cudaError_t z_setup_launch(const ZArgs& a, double* rstart, double* r00) {
    z_setup_kernel<Z_MROWS><<<(unsigned)((a.ncols + 127) / 128), 128>>>(a, rstart, r00);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    return e;
}

}  // namespace cans
