// z_solve.cu -- pass B: persistent, cp.async double-buffered partitioned Thomas solve (z_pass.cuh).
#include <cuda.h>

#include "z_kernels.cuh"

namespace cans {

// ---- TMA / mbarrier primitives (sm_90+ PTX; SASS: UTMALDG, SYNCS) ----
CANS_D unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
CANS_D void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
CANS_D void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
CANS_D void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 2-D tiled load: box (TC columns x box_rows rows) at (col0, row0) of the (nz, ncols) view of the field
CANS_D void tma_load_2d(void* dst, const CUtensorMap* tmap, int col0, int row0, unsigned long long* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
        ::"r"(smem_u32(dst)), "l"(tmap), "r"(col0), "r"(row0), "r"(smem_u32(bar)) : "memory");
}

template <int MROWS, int TC>
__global__ void __launch_bounds__(512) z_solve_kernel(const ZArgs a, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(128) double zsm[];
    typedef ZPass<MROWS, TC> Z;
    __shared__ long s_next;
    __shared__ __align__(8) unsigned long long s_bar[2];
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
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        s_next = (long)atomicAdd(a.ticket, 1u);
    }
    __syncthreads();
    long cur = s_next;
    __syncthreads();
    if (cur >= a.ntiles) return;
    // one elected thread asks the TMA unit for a whole tile: rows beyond nz / columns beyond ncols are
    // zero-filled by the hardware, so ragged tiles need no special path
    const unsigned tile_bytes = (unsigned)(a.box_rows * TC * sizeof(double)) * (unsigned)a.nbox;
    auto issue_tile = [&](long tile, int bsel) {
        double* dst = bufs + (size_t)bsel * tile_sz;
        mbar_expect_tx(&s_bar[bsel], tile_bytes);
        for (int q = 0; q < a.nbox; ++q)
            tma_load_2d(dst + (size_t)q * a.box_rows * TC, &tmap, (int)(tile * TC), q * a.box_rows, &s_bar[bsel]);
    };
    if (tid == 0) {
        // the generic-proxy reads / writes of the staging area above are ordered before the async-proxy writes
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        issue_tile(cur, 0);
        s_next = (long)atomicAdd(a.ticket, 1u);
    }
    int b = 0;
    unsigned phases = 0u;                  // bit b = parity of the next completion of buffer b
    const int c = tid % TC;
    const int s = tid / TC;
    // per-thread scalars of a tile: Thomas pivot entering the segment (streamed once from the plan's
    // table) and the two eigenvalue parts of the column; fetched one tile ahead and only combined when
    // used, so their latency is hidden behind the previous tile
    auto tile_scalars = [&](long tile, double& rs, double& l1, double& l2) {
        const long col = tile * TC + c;
        rs = 0.0; l1 = 0.0; l2 = 0.0;
        if (tile < a.ntiles && col < a.ncols) {
            const int ci = (int)col;                  // ncols = nx*ny <= 2048^2 fits an int
            rs = __ldcs(a.rstart + (size_t)s * a.ncols + col);
            l1 = a.lamx[ci % a.nx];
            l2 = a.lamy[ci / a.nx];
        }
    };
    double rs, l1, l2;
    tile_scalars(cur, rs, l1, l2);
    while (true) {
        __syncthreads();                       // s_next visible; buffer b^1 no longer read by anyone
        const long nxt = s_next;
        if (tid == 0 && nxt < a.ntiles) issue_tile(nxt, b ^ 1);
        double rs_n, l1_n, l2_n;
        tile_scalars(nxt, rs_n, l1_n, l2_n);   // consumed in the next iteration
        mbar_wait(&s_bar[b], (phases >> b) & 1u);   // the current tile has landed (the next may still fly)
        phases ^= 1u << b;
        ZState<MROWS> st;
        Z::phase1(a, zsm, bufs + (size_t)b * tile_sz, st, cur, rs, l1 + l2, tid);
        __syncthreads();
        // every thread has read s_next (before the barrier above): thread 0 may now draw the ticket after next
        if (tid == 0 && nxt < a.ntiles) s_next = (long)atomicAdd(a.ticket, 1u);
        Z::phase2a(a, zsm, st, tid);
        __syncthreads();
        Z::phase2b(a, zsm, st, tid);
        __syncthreads();
        Z::phase3(a, zsm, st, tid);
        if (nxt >= a.ntiles) break;
        cur = nxt;
        rs = rs_n; l1 = l1_n; l2 = l2_n;
        b ^= 1;
    }
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static cudaError_t z_make_tensor_map(const ZArgs& a, int tc, CUtensorMap* tmap) {
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        encode = (EncodeTiledFn)fn;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)a.ncols, (cuuint64_t)a.nz};
    const cuuint64_t strides[1] = {(cuuint64_t)a.ncols * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)tc, (cuuint32_t)a.box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = encode(tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)a.p, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t z_solve_launch(const ZArgs& a_in, int grid, size_t smem, cudaStream_t st) {
    ZArgs a = a_in;
    long g = grid;
    if (g > a.ntiles) g = a.ntiles;
    if (g < 1) g = 1;
    // the padded column length nseg*MROWS is covered exactly by nbox boxes of box_rows (<= 256) rows:
    // box_rows = MROWS * (largest divisor of nseg that is <= 256/MROWS)
    int d = 256 / Z_MROWS;
    while (a.nseg % d) --d;
    a.box_rows = d * Z_MROWS;
    a.nbox = a.nseg / d;
    const int tc = z_tc_for(a.nseg);
    CUtensorMap tmap;
    cudaError_t e = z_make_tensor_map(a, tc, &tmap);
    if (e != cudaSuccess) return e;
    switch (tc) {
        case 32: z_solve_kernel<Z_MROWS, 32><<<(unsigned)g, 32 * a.nseg, smem, st>>>(a, tmap); break;
        case 16: z_solve_kernel<Z_MROWS, 16><<<(unsigned)g, 16 * a.nseg, smem, st>>>(a, tmap); break;
        default: z_solve_kernel<Z_MROWS, 8><<<(unsigned)g, 8 * a.nseg, smem, st>>>(a, tmap); break;
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
