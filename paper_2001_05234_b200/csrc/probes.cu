// probes.cu -- measurement probes behind cans_probe_* (bench.py): the denominators the kernel numbers are read against.
//   * probe_fp64_fma: the plain FP64 pipe's FMA rate ("measure one before quoting pipe utilisation");
//   * probe_tile_copy: the HBM rate of a bare TMA copy (tile in, tile out, no arithmetic) with exactly the tile shape and
//     order the y transforms / the z solve use -- the ceiling of that access pattern, which for 128-byte row segments is
//     well below the contiguous copy rate.
#include "probes.cuh"
#include "tma_util.cuh"

namespace cans {

__global__ void __launch_bounds__(256) fp64_fma_kernel(double* sink, int iters) {
    double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-6;
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 123.456) sink[0] = s;                    // never true: keeps the chains alive
}

cudaError_t probe_fp64_fma(int num_sms, double* fma_per_s, cudaStream_t st) {
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 14, grid = num_sms * 8, threads = 256;
    fp64_fma_kernel<<<grid, threads, 0, st>>>(sink, 256);           // warm-up
    cudaEventRecord(e0, st);
    fp64_fma_kernel<<<grid, threads, 0, st>>>(sink, iters);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) *fma_per_s = 8.0 * iters * (double)grid * threads / (ms * 1e-3);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    return e;
}

// persistent CTAs, one elected thread: tile t -> boxes q at (c0, c1) = ((t % m0) * s0, (t / m0) * s1 + q * box_rows),
// two buffers, loads one tile ahead of the write-back
__global__ void __launch_bounds__(128) tile_copy_kernel(const __grid_constant__ CUtensorMap tmap, const TileCopyShape sh) {
    extern __shared__ __align__(1024) unsigned char tc_smem[];
    __shared__ __align__(8) unsigned long long bar[2];
    if (threadIdx.x == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_fence_init(); }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const unsigned box_bytes = (unsigned)(sh.box_rows * sh.box_cols * sizeof(double));
    const unsigned tile_bytes = box_bytes * (unsigned)sh.nbox;
    auto load = [&](long t, int b) {
        mbar_expect_tx(&bar[b], tile_bytes);
        for (int q = 0; q < sh.nbox; ++q)
            tma_load_2d(tc_smem + (size_t)b * tile_bytes + (size_t)q * box_bytes, &tmap, (int)((t % sh.m0) * sh.s0),
                        (int)((t / sh.m0) * sh.s1) + q * sh.box_rows, &bar[b]);
    };
    long t = blockIdx.x;
    if (t < sh.ntiles) load(t, 0);
    unsigned phases = 0u;
    int b = 0;
    for (; t < sh.ntiles; t += gridDim.x) {
        const long tn = t + gridDim.x;
        if (tn < sh.ntiles) {
            tma_store_wait_read_pending<0>();               // the write-back that last read buffer b^1 has drained
            load(tn, b ^ 1);
        }
        mbar_wait(&bar[b], (phases >> b) & 1u);
        phases ^= 1u << b;
        for (int q = 0; q < sh.nbox; ++q)
            tma_store_2d(&tmap, (int)((t % sh.m0) * sh.s0), (int)((t / sh.m0) * sh.s1) + q * sh.box_rows,
                         tc_smem + (size_t)b * tile_bytes + (size_t)q * box_bytes);
        tma_store_commit();
        b ^= 1;
    }
    tma_store_wait_all();
}

cudaError_t probe_tile_copy(const CUtensorMap* tmap, const TileCopyShape& sh, int num_sms, float* ms, cudaStream_t st) {
    const size_t smem = 2 * (size_t)sh.nbox * sh.box_rows * sh.box_cols * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(tile_copy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const unsigned grid = (unsigned)(sh.ntiles < num_sms ? sh.ntiles : num_sms);
    tile_copy_kernel<<<grid, 128, smem, st>>>(*tmap, sh);           // warm-up
    cudaEventRecord(e0, st);
    tile_copy_kernel<<<grid, 128, smem, st>>>(*tmap, sh);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return e;
}

}  // namespace cans
