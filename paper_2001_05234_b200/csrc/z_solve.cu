// z_solve.cu -- pass B: persistent partitioned Thomas solve (z_pass.cuh) fed by double-buffered TMA tile loads.
#include "z_kernels.cuh"
#include "tma_util.cuh"

namespace cans {

template <int MROWS, int TC, bool CYC>
__global__ void __launch_bounds__(512) z_solve_kernel(const ZArgs a, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(1024) double zsm[];
    typedef ZPass<MROWS, TC> Z;
    __shared__ long s_next;
    __shared__ __align__(8) unsigned long long s_bar[2];
    int tid = threadIdx.x;
    asm volatile("" : "+r"(tid));              // opaque: keeps the thread index in a register (the compiler otherwise re-reads
                                             // the special register ~14 times per warp and tile, a long-latency S2R each)
    const int nthreads = blockDim.x;
    double* bufs = zsm + Z::table_doubles(a.nseg);
    const size_t tile_sz = Z::tile_doubles(a.nseg);

    if (a.singular && blockIdx.x == 0) {
        // the singular (0,0) column (reading S3): staged by the CTA, swept by one thread, written back by the CTA
        const int nzp = a.nseg * MROWS;
        z_singular_stage(a, bufs, nzp, tid, nthreads);
        __syncthreads();
        if (tid == 0) z_singular_sweeps(a, bufs, nzp);
        __syncthreads();
        z_singular_store(a, bufs, nzp, tid, nthreads);
        __syncthreads();
    }
    Z::load_tables(a, zsm, tid, nthreads);
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
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
        fence_proxy_async_smem();
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
            const unsigned ci = (unsigned)col;        // ncols = nx*ny <= 2048^2 fits 32 bits
            rs = __ldcs(a.rstart + (size_t)s * a.ncols + col);
            const unsigned j = (unsigned)(((unsigned long long)ci * a.nx_magic) >> 40);     // ci / nx without the division
            l1 = a.lamx[ci - j * (unsigned)a.nx];
            l2 = a.lamy[j];
        }
    };
    double rs, l1, l2;
    tile_scalars(cur, rs, l1, l2);
    __syncthreads();                           // the first s_next is visible
    while (true) {
        // Open system: no barrier here -- s_next was rewritten behind the phase-1 barrier of the previous tile and published
        // by its phase-2 barrier; buffer b^1 was last read in that tile's phase 1, also behind that barrier.
        // Cyclic system: buffer b^1 held the previous tile's q until the end of that iteration, so the copy of the next tile
        // into it is issued behind this tile's phase-1 barrier instead (every thread has left the previous iteration).
        const long nxt = s_next;
        if (!CYC && tid == 0 && nxt < a.ntiles) issue_tile(nxt, b ^ 1);
        double rs_n, l1_n, l2_n;
        tile_scalars(nxt, rs_n, l1_n, l2_n);   // consumed in the next iteration
        ZState<MROWS> st;
        // (buffer address and eigenvalue sum are re-formed at every use: at the 128-register cap of a 512-thread CTA each
        // value kept live across the phases costs a rematerialised S2R or a spill elsewhere)
        mbar_wait(&s_bar[b], (phases >> b) & 1u);   // the current tile has landed (the next may still fly)
        phases ^= 1u << b;
        Z::template phase1<CYC>(a, zsm, bufs + (size_t)b * tile_sz, st, cur, rs, l1 + l2 + a.alpha, tid);
        __syncthreads();
        // every thread has read s_next (before the barrier above): thread 0 may now draw the ticket after next
        if (tid == 0 && nxt < a.ntiles) {
            if (CYC) issue_tile(nxt, b ^ 1);
            s_next = (long)atomicAdd(a.ticket, 1u);
        }
        Z::template phase2a<CYC>(a, zsm, st, tid);
        Z::template phase2b<CYC>(a, zsm, st, l1 + l2 + a.alpha, tid, bufs + (size_t)b * tile_sz);    // cyclic: the tile's buffer, now free, holds q
        __syncthreads();
        if (CYC) {
            Z::cyclic_scan(a, zsm, st, tid, bufs + (size_t)b * tile_sz);
            __syncthreads();
            Z::cyclic_store(a, zsm, st, l1 + l2 + a.alpha, tid, bufs + (size_t)b * tile_sz);
            fence_proxy_async_smem();           // this thread's accesses to q are ordered before the TMA refill of the buffer
        } else {
            Z::phase3(a, zsm, st, tid, bufs + (size_t)b * tile_sz);
        }
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

template <int TC, bool CYC>
static cudaError_t configure_tc(int nseg, int num_sms, int* grid_out, size_t* smem_out) {
    size_t smem = sizeof(double) * ZPass<Z_MROWS, TC>::smem_doubles(nseg);
    if (smem > Z_SMEM_LIMIT) return cudaErrorInvalidConfiguration;       // the plan checks z_solve_smem_bytes first
    cudaError_t e = cudaFuncSetAttribute(z_solve_kernel<Z_MROWS, TC, CYC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, z_solve_kernel<Z_MROWS, TC, CYC>, TC * nseg, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    if (per_sm > 4) per_sm = 4;
    *grid_out = per_sm * num_sms;
    *smem_out = smem;
    return cudaSuccess;
}

size_t z_solve_smem_bytes(int nseg) {
    switch (z_tc_for(nseg)) {
        case 32: return sizeof(double) * ZPass<Z_MROWS, 32>::smem_doubles(nseg);
        case 16: return sizeof(double) * ZPass<Z_MROWS, 16>::smem_doubles(nseg);
        default: return sizeof(double) * ZPass<Z_MROWS, 8>::smem_doubles(nseg);
    }
}

cudaError_t z_solve_configure(int nseg, int cyclic, int num_sms, int* grid_out, size_t* smem_out) {
    switch (z_tc_for(nseg)) {
        case 32: return cyclic ? configure_tc<32, true>(nseg, num_sms, grid_out, smem_out) : configure_tc<32, false>(nseg, num_sms, grid_out, smem_out);
        case 16: return cyclic ? configure_tc<16, true>(nseg, num_sms, grid_out, smem_out) : configure_tc<16, false>(nseg, num_sms, grid_out, smem_out);
        default: return cyclic ? configure_tc<8, true>(nseg, num_sms, grid_out, smem_out) : configure_tc<8, false>(nseg, num_sms, grid_out, smem_out);
    }
}

// TMA tiling of a column tile: the padded column length nzp = nseg*MROWS is covered exactly by nbox boxes of box_rows rows,
// box_rows = the largest divisor of nzp that is <= 256 (any divisor, not only whole segments: a prime segment count -- nz =
// 577..592 gives nseg = 37 -- still gets boxes of 148 rows, not 37 boxes of 16)
void z_boxes(int nseg, int* nbox, int* box_rows) {
    const int nzp = nseg * Z_MROWS;
    int br = nzp < 256 ? nzp : 256;
    while (nzp % br) --br;
    *box_rows = br;
    *nbox = nzp / br;
}

cudaError_t z_make_tensor_map(CUtensorMap* tmap, const double* p, long ncols, int nz, int nseg) {
    int nbox, box_rows;
    z_boxes(nseg, &nbox, &box_rows);
    return make_tensor_map_2d(tmap, p, (unsigned long long)ncols, (unsigned long long)nz,
                              (unsigned long long)ncols * sizeof(double), (unsigned)z_tc_for(nseg), (unsigned)box_rows,
                              CU_TENSOR_MAP_SWIZZLE_NONE);
}

cudaError_t z_solve_launch(const ZArgs& a_in, int grid, size_t smem, const CUtensorMap* tmap, cudaStream_t st) {
    ZArgs a = a_in;
    long g = grid;
    if (g > a.ntiles) g = a.ntiles;
    if (g < 1) g = 1;
    z_boxes(a.nseg, &a.nbox, &a.box_rows);
    a.nx_magic = ((1ull << 40) + (unsigned long long)a.nx - 1) / (unsigned long long)a.nx;
    const int tc = z_tc_for(a.nseg);
#define CANS_Z_LAUNCH(TC, CYC) z_solve_kernel<Z_MROWS, TC, CYC><<<(unsigned)g, TC * a.nseg, smem, st>>>(a, *tmap)
    if (a.cyclic) { if (tc == 32) CANS_Z_LAUNCH(32, true); else if (tc == 16) CANS_Z_LAUNCH(16, true); else CANS_Z_LAUNCH(8, true); }
    else { if (tc == 32) CANS_Z_LAUNCH(32, false); else if (tc == 16) CANS_Z_LAUNCH(16, false); else CANS_Z_LAUNCH(8, false); }
#undef CANS_Z_LAUNCH
    return cudaGetLastError();
}

cudaError_t z_setup_launch(const ZArgs& a, double* rstart, double* r00, cudaStream_t st) {
    z_setup_kernel<Z_MROWS><<<(unsigned)((a.ncols + 127) / 128), 128, 0, st>>>(a, rstart, r00);
    return cudaGetLastError();
}

}  // namespace cans
